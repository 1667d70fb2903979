// bf_umma_common.cuh -- pieces shared by the two tensor-core kernels (bf_umma.cu: coefficients resident,
// 2*nant <= 64; bf_umma_kblock.cu: K-blocked, any nant): the int8 -> fp16 converter and the fused
// |.|^2 + integrate epilogue (hot-path rows a4, a5).
#pragma once
#include "bf_internal.h"
#include "ptx.cuh"

namespace bfk {

constexpr int TILE_T = 256;                        // time samples per tile = UMMA N
constexpr int EPI_WARPS = 16;
constexpr int A_TILE_BYTES = BF_TILE_ROWS * 128;   // 128 rows x 64 fp16
constexpr int B_STAGE_BYTES = TILE_T * 128;        // 256 rows x 64 fp16
constexpr int RAW_STAGE_BYTES = TILE_T * 64;       // 256 time samples x 64 int8 (32 antennas x (re, im))

// int8 x4 (one 32-bit word) -> two half2, exact: 0x6400 | (x ^ 0x80) is the fp16 number 1024 + (x + 128)
__device__ __forceinline__ void cvt_i8x4_f16x4(uint32_t w, uint32_t &lo, uint32_t &hi) {
  const uint32_t u = w ^ 0x80808080u;
  const uint32_t l = __byte_perm(u, 0x64646464u, 0x5140);
  const uint32_t h = __byte_perm(u, 0x64646464u, 0x5342);
  const __half2 bias = __halves2half2(__ushort_as_half(0x6480), __ushort_as_half(0x6480));  // 1152
  __half2 a = __hsub2(*reinterpret_cast<const __half2 *>(&l), bias);
  __half2 b = __hsub2(*reinterpret_cast<const __half2 *>(&h), bias);
  lo = *reinterpret_cast<uint32_t *>(&a);
  hi = *reinterpret_cast<uint32_t *>(&b);
}

// 4+4-bit packed complex (high nibble re, low nibble im), 4 antennas in one 32-bit word
// -> four half2 (re, im), exact.  Per antenna: PRMT builds [b, 0x64, b, 0x64]; one LOP3 flips the two
// sign bits and masks the nibbles, leaving the halves 0x6400|(re_u<<4) = 1024 + 16 re_u and
// 0x6400|im_u = 1024 + im_u (re_u = re + 8, im_u = im + 8); one HFMA2 with per-half constants
// (x/16 - 72, x - 1032) gives (re, im).
__device__ __forceinline__ void cvt_i4x8_f16x8(uint32_t w, uint32_t (&h)[4]) {
  const uint32_t c64 = 0x64646464u, flip = 0x00080080u, mask = 0xFF0FFFF0u;
  const __half2 scale = __halves2half2(__ushort_as_half(0x2C00), __ushort_as_half(0x3C00));   // (1/16, 1)
  const __half2 off = __halves2half2(__ushort_as_half(0xD480), __ushort_as_half(0xE408));     // (-72, -1032)
#pragma unroll
  for (int a = 0; a < 4; ++a) {
    const uint32_t p = __byte_perm(w, c64, 0x4040 | a | (a << 8));  // [b_a, 0x64, b_a, 0x64]
    const uint32_t m = (p ^ flip) & mask;
    const __half2 r = __hfma2(*reinterpret_cast<const __half2 *>(&m), scale, off);
    h[a] = *reinterpret_cast<const uint32_t *>(&r);
  }
}

__device__ __forceinline__ void st_shared_v4(uint32_t addr, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
  asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(addr), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
}
__device__ __forceinline__ uint4 ld_shared_v4(uint32_t addr) {
  uint4 r;
  asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "r"(addr));
  return r;
}

// raw int8 stage (256 rows x 64 bytes, compact) -> fp16 operand stage (256 rows x 128 bytes, 128-byte
// swizzle).  PIECES 16-byte input pieces per thread; piece pc = tid + k*NTHREADS covers row pc/4,
// bytes 16*(pc%4)..  p_dst[k] = byte offset of its first output chunk (0xffffffff = not mine).
template <int PIECES, int NTHREADS>
__device__ __forceinline__ void convert_load(uint32_t s_raw, int tid, const uint32_t (&p_dst)[PIECES], uint4 (&x)[PIECES]) {
#pragma unroll
  for (int k = 0; k < PIECES; ++k)
    if (p_dst[k] != 0xffffffffu) x[k] = ld_shared_v4(s_raw + 16 * (tid + k * NTHREADS));
}
template <int PIECES>
__device__ __forceinline__ void convert_store(uint32_t s_dst, const uint32_t (&p_dst)[PIECES], const uint4 (&x)[PIECES]) {
#pragma unroll
  for (int k = 0; k < PIECES; ++k) {
    if (p_dst[k] != 0xffffffffu) {
      uint32_t h[8];
      cvt_i8x4_f16x4(x[k].x, h[0], h[1]);
      cvt_i8x4_f16x4(x[k].y, h[2], h[3]);
      cvt_i8x4_f16x4(x[k].z, h[4], h[5]);
      cvt_i8x4_f16x4(x[k].w, h[6], h[7]);
      st_shared_v4(s_dst + p_dst[k], h[0], h[1], h[2], h[3]);
      st_shared_v4(s_dst + (p_dst[k] ^ 16u), h[4], h[5], h[6], h[7]);
    }
  }
}

// 4-bit input: raw stage rows are nant bytes; a 16-byte piece = 16 antennas = 4 output chunks of 16 bytes
// (chunk (4q + j) ^ (t & 7) = first chunk ^ j, since 4q has its two low bits clear)
template <int PIECES>
__device__ __forceinline__ void convert_store_ci4(uint32_t s_dst, const uint32_t (&p_dst)[PIECES], const uint4 (&x)[PIECES]) {
#pragma unroll
  for (int k = 0; k < PIECES; ++k) {
    if (p_dst[k] != 0xffffffffu) {
      const uint32_t w[4] = {x[k].x, x[k].y, x[k].z, x[k].w};
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        uint32_t h[4];
        cvt_i4x8_f16x8(w[j], h);
        st_shared_v4(s_dst + (p_dst[k] ^ (uint32_t)(j << 4)), h[0], h[1], h[2], h[3]);
      }
    }
  }
}

// Epilogue of ONE accumulator tile for ONE warp of the 16: TMEM lanes 32*quad.., 64 columns starting at
// `taddr` (lane and column already folded in).  Rows: lane l < 16 is the re row, lane l+16 the im row of
// one beam.  The TMEM stage is handed back (arrive on bar_empty) as soon as this warp's last tcgen05.ld
// has landed; squaring, shuffle and store run in the shadow of the next MMAs.  `out` points at this
// lane's first output bin of the tile, `nvalid` = how many bins from there exist (tail tiles), `writer`
// = this lane holds a real beam and is a re lane.  All per-tile address arithmetic is the caller's, so
// that it can be hoisted out of the tile loop.
// NINT_T: integration length if a power of two <= 64; 0 = a larger multiple of 64: the partial sum of
// the warp's 64 columns is added atomically into the (zeroed) bin `out` points at.
template <int NINT_T>
__device__ __forceinline__ void epilogue_tile(uint32_t taddr, float *out, bool writer, int nvalid, bool vec_ok,
                                              uint32_t bar_empty, bool lane0) {
  constexpr int CPW = TILE_T / (EPI_WARPS / 4);                          // columns per warp (64)
  constexpr int NCH = CPW / 32;                                          // 32-column chunks per warp
  constexpr int SUB = (NINT_T == 0 || NINT_T > 32) ? 32 : NINT_T;        // columns per partial sum
  constexpr int NSUB = 32 / SUB;                                          // partial sums per chunk
  constexpr int CPB = NINT_T == 0 ? NCH : (NINT_T <= 32 ? 1 : NINT_T / 32);  // chunks per bin
  constexpr int NBIN = NINT_T == 0 ? 1 : CPW / NINT_T;                   // bins per warp and tile
  static_assert(NINT_T == 0 || (NINT_T <= CPW && CPW % (NINT_T == 0 ? 1 : NINT_T) == 0), "bin must not straddle epilogue warps");
  float ob[4];
  constexpr int NACC = SUB >= 8 ? 4 : (SUB >= 2 ? SUB / 2 : 1);
  float2 a[NACC];  // packed running sums of squares; live across the chunks of one bin
#pragma unroll
  for (int q = 0; q < NACC; ++q) a[q] = make_float2(0.f, 0.f);
#pragma unroll
  for (int ch = 0; ch < NCH; ++ch) {
    uint32_t v[32];
    BF_TMEM_LD_32x32b_X32(taddr + 32 * ch, v);
    tc_wait_ld();
    if (ch == NCH - 1) {  // all of this warp's columns are in registers: release the stage
      tc_fence_before();
      __syncwarp();
      if (lane0) mbar_arrive(bar_empty);
    }
#pragma unroll
    for (int s = 0; s < NSUB; ++s) {
      float sum;
      if constexpr (SUB == 1) {
        const float d = __uint_as_float(v[s]);
        sum = d * d;
      } else {
#pragma unroll
        for (int j = 0; j < SUB / 2; ++j) {
          const float2 d = make_float2(__uint_as_float(v[s * SUB + 2 * j]), __uint_as_float(v[s * SUB + 2 * j + 1]));
          a[j % NACC] = ffma2(d, d, a[j % NACC]);
        }
        if (CPB > 1 && (ch + 1) % CPB != 0) continue;  // bin continues in the next chunk
#pragma unroll
        for (int w = NACC / 2; w >= 1; w >>= 1)        // packed add tree
#pragma unroll
          for (int q = 0; q < w; ++q) a[q] = fadd2(a[q], a[q + w]);
        sum = a[0].x + a[0].y;
#pragma unroll
        for (int q = 0; q < NACC; ++q) a[q] = make_float2(0.f, 0.f);
      }
      const float tot = sum + __shfl_xor_sync(0xffffffffu, sum, 16);  // re^2 rows + im^2 rows
      if (NINT_T == 0) {
        if (writer && nvalid > 0) atomicAdd(out, tot);
      } else {
        const int jb = (ch / CPB) * NSUB + s;  // bin index inside this warp's columns (compile-time)
        if (NBIN >= 4 && vec_ok) {
          ob[jb & 3] = tot;
          if ((jb & 3) == 3 && writer && jb < nvalid)
            *reinterpret_cast<float4 *>(out + jb - 3) = make_float4(ob[0], ob[1], ob[2], ob[3]);
        } else if (writer && jb < nvalid) {
          out[jb] = tot;
        }
      }
    }
  }
}
// ANY integration length (the sizes of a real observation do not divide a tile).  The warp's 64 columns are
// the time samples t_first .. t_first + 63 of one beam row, and a bin ends after every column with (t + 1) % nint == 0.  The
// squares of each run of columns inside one bin are summed in registers and added atomically into the ZEROED power cube
// (`row` = first bin of this lane's beam), so a bin may straddle warps, tiles and CTAs.  Bin ends are a warp-uniform 64-bit
// mask, so the 64 unrolled flush sites branch uniformly; one integer division per tile.  Columns past nsamp hold finite
// garbage; nsamp % nint == 0 makes sample nsamp - 1 a bin end, so they only ever reach bins >= nbin, which are dropped.
__device__ __forceinline__ void epilogue_tile_anynint(uint32_t taddr, float *row, bool writer, int t_first, int nint, int nbin,
                                                      uint32_t bar_empty, bool lane0) {
  constexpr int CPW = TILE_T / (EPI_WARPS / 4);                          // columns per warp (64)
  constexpr int NCH = CPW / 32;
  int bin = t_first / nint;
  unsigned long long ends = 0;
  for (int k = nint - 1 - (t_first - bin * nint); k < CPW; k += nint) ends |= 1ull << k;
  float acc = 0.f;
  auto flush = [&](bool end) {   // warp-uniform call sites
    const float tot = acc + __shfl_xor_sync(0xffffffffu, acc, 16);  // re^2 rows + im^2 rows
    if (writer && bin < nbin) atomicAdd(row + bin, tot);
    acc = 0.f;
    if (end) ++bin;
  };
#pragma unroll
  for (int ch = 0; ch < NCH; ++ch) {
    uint32_t v[32];
    BF_TMEM_LD_32x32b_X32(taddr + 32 * ch, v);
    tc_wait_ld();
    if (ch == NCH - 1) {  // all of this warp's columns are in registers: release the stage
      tc_fence_before();
      __syncwarp();
      if (lane0) mbar_arrive(bar_empty);
    }
    // Groups of 8 columns.  With nint >= 16 a group holds at most ONE bin end.  A group with none before its last column
    // (all but one or two per tile at nint >= 64) is four packed FMAs into two independent sums; a group with an end inside
    // is split by selects into the part up to the end and the part after it, with a single flush between them -- 16 flush
    // sites in all, not one per column.  (Measured on a medium-sized buffer at nint 100: one dependent FMA chain with a test
    // after every column 5.2 ms, per-column walks only in the groups with an end 3.1 ms; nint 64 at compile time 0.91 ms.)
#pragma unroll
    for (int g = 0; g < 4; ++g) {
      const uint32_t e8 = (uint32_t)(ends >> (32 * ch + 8 * g)) & 0xffu;
      const bool last = ch == NCH - 1 && g == 3;                      // this warp's part of a bin ends with its columns
      if ((e8 & 0x7fu) == 0) {
        float2 a0 = make_float2(0.f, 0.f), a1 = make_float2(0.f, 0.f);
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const float2 d = make_float2(__uint_as_float(v[8 * g + 2 * j]), __uint_as_float(v[8 * g + 2 * j + 1]));
          if (j & 1) a1 = ffma2(d, d, a1);
          else a0 = ffma2(d, d, a0);
        }
        a0 = fadd2(a0, a1);
        acc += a0.x + a0.y;
        if (e8 != 0 || last) flush(e8 != 0);
      } else {
        const int je = __ffs((int)e8) - 1;                             // the end is after column je (0 .. 6) of the group
        float lo = 0.f, hi = 0.f;
#pragma unroll
        for (int j = 0; j < 8; ++j) {
          const float d = __uint_as_float(v[8 * g + j]);
          const float sq = d * d;
          lo += j <= je ? sq : 0.f;
          hi += j <= je ? 0.f : sq;
        }
        acc += lo;
        flush(true);
        acc = hi;
        if (last) flush(false);
      }
    }
  }
}
// ---- deferred tail ----------------------------------------------------------------------------------------------
// The epilogue warps are the critical chain of the resident kernel (profiles/: busy ~90 % of the time while every
// other role waits), and a fifth of that chain was the tail of each tile: add tree -> SHFL -> FADD -> STG, the FADD
// stalled on the shuffle, which queues behind the other warps' tcgen05.ld / LDS / STS in the same memory pipe.
// Here the tail of tile i is carried into tile i+1 and issued right after that tile's first tcgen05.ld, so its
// latency hides under the load.  EpiPend = the per-lane bin sums of the previous tile (re^2 and im^2 rows still
// apart), where they go, and whether this lane stores them.
template <int NINT_T>
struct EpiPend {
  static constexpr int NBIN = NINT_T == 0 ? 1 : (TILE_T / (EPI_WARPS / 4)) / NINT_T;   // bins per warp and tile
  static constexpr bool DEFER = NBIN <= 4;
  float s[DEFER ? NBIN : 1];
  float *out;
  int nvalid;
  bool writer, vec;
};
template <int NINT_T>
__device__ __forceinline__ void epi_pend_init(EpiPend<NINT_T> &pd) {
#pragma unroll
  for (int j = 0; j < (EpiPend<NINT_T>::DEFER ? EpiPend<NINT_T>::NBIN : 1); ++j) pd.s[j] = 0.f;
  pd.out = nullptr; pd.nvalid = 0; pd.writer = false; pd.vec = false;
}
// WHOLE: the pending tile is known to have all its bins (the lean loop): no per-bin bounds
template <int NINT_T, bool WHOLE = false>
__device__ __forceinline__ void epi_pend_flush(EpiPend<NINT_T> &pd) {
  constexpr int NBIN = EpiPend<NINT_T>::NBIN;
  if constexpr (EpiPend<NINT_T>::DEFER) {
    float tot[NBIN];
#pragma unroll
    for (int j = 0; j < NBIN; ++j) tot[j] = pd.s[j] + __shfl_xor_sync(0xffffffffu, pd.s[j], 16);  // re^2 rows + im^2 rows
    if constexpr (WHOLE && NINT_T != 0) {
      if (NBIN == 4 && pd.vec) {
        if (pd.writer) *reinterpret_cast<float4 *>(pd.out) = make_float4(tot[0], tot[1], tot[2], tot[3]);
      } else if (pd.writer) {
#pragma unroll
        for (int j = 0; j < NBIN; ++j) pd.out[j] = tot[j];
      }
      pd.writer = false;
      return;
    }
    if (NINT_T == 0) {
      if (pd.writer && pd.nvalid > 0) atomicAdd(pd.out, tot[0]);
    } else if (NBIN == 4 && pd.vec) {
      if (pd.writer && pd.nvalid >= 4) *reinterpret_cast<float4 *>(pd.out) = make_float4(tot[0], tot[1], tot[2], tot[3]);
      else if (pd.writer) {
#pragma unroll
        for (int j = 0; j < NBIN; ++j) if (j < pd.nvalid) pd.out[j] = tot[j];
      }
    } else if (pd.writer) {
#pragma unroll
      for (int j = 0; j < NBIN; ++j) if (j < pd.nvalid) pd.out[j] = tot[j];
    }
    pd.writer = false;
  }
}
// One accumulator tile for one warp, tail deferred (see above).  Same contract as epilogue_tile; `pd` carries the
// previous tile's tail in and this tile's tail out.  Bins of <= 8 samples (more than 4 bins per warp) fall back to
// the immediate form.
template <int NINT_T, bool WHOLE = false>
__device__ __forceinline__ void epilogue_tile_defer(uint32_t taddr, float *out, bool writer, int nvalid, bool vec_ok,
                                                    uint32_t bar_empty, bool lane0, EpiPend<NINT_T> &pd) {
  if constexpr (!EpiPend<NINT_T>::DEFER) {
    epilogue_tile<NINT_T>(taddr, out, writer, nvalid, vec_ok, bar_empty, lane0);
  } else {
    constexpr int CPW = TILE_T / (EPI_WARPS / 4);
    constexpr int NCH = CPW / 32;
    constexpr int SUB = (NINT_T == 0 || NINT_T > 32) ? 32 : NINT_T;
    constexpr int NSUB = 32 / SUB;
    constexpr int CPB = NINT_T == 0 ? NCH : (NINT_T <= 32 ? 1 : NINT_T / 32);
    constexpr int NACC = SUB >= 8 ? 4 : (SUB >= 2 ? SUB / 2 : 1);
    float2 a[NACC];
#pragma unroll
    for (int q = 0; q < NACC; ++q) a[q] = make_float2(0.f, 0.f);
    float sums[EpiPend<NINT_T>::NBIN];
#pragma unroll
    for (int ch = 0; ch < NCH; ++ch) {
      uint32_t v[32];
      BF_TMEM_LD_32x32b_X32(taddr + 32 * ch, v);
      if (ch == 0) epi_pend_flush<NINT_T, WHOLE>(pd);   // the previous tile's shuffles and stores, under this load
      tc_wait_ld();
      if (ch == NCH - 1) {  // all of this warp's columns are in registers: release the stage
        tc_fence_before();
        __syncwarp();
        if (lane0) mbar_arrive(bar_empty);
      }
#pragma unroll
      for (int s = 0; s < NSUB; ++s) {
#pragma unroll
        for (int j = 0; j < SUB / 2; ++j) {
          const float2 d = make_float2(__uint_as_float(v[s * SUB + 2 * j]), __uint_as_float(v[s * SUB + 2 * j + 1]));
          a[j % NACC] = ffma2(d, d, a[j % NACC]);
        }
        if (CPB > 1 && (ch + 1) % CPB != 0) continue;  // bin continues in the next chunk
#pragma unroll
        for (int w = NACC / 2; w >= 1; w >>= 1)        // packed add tree
#pragma unroll
          for (int q = 0; q < w; ++q) a[q] = fadd2(a[q], a[q + w]);
        sums[NINT_T == 0 ? 0 : (ch / CPB) * NSUB + s] = a[0].x + a[0].y;
#pragma unroll
        for (int q = 0; q < NACC; ++q) a[q] = make_float2(0.f, 0.f);
      }
    }
#pragma unroll
    for (int j = 0; j < EpiPend<NINT_T>::NBIN; ++j) pd.s[j] = sums[j];
    pd.out = out; pd.nvalid = nvalid; pd.writer = writer; pd.vec = vec_ok;
  }
}
// Voltage-beam epilogue ("electric-field ... beams ... output as 16-bit complex-valued
// words"): ONE accumulator tile for ONE warp -> y[beam][t] as fp16 (re, im) pairs, scaled by
// `scale`.  Lane l < 16 holds the re row, lane l + 16 the im row of one beam; 64 columns = 64 time samples.
// Per 32-column chunk: pack time pairs to half2, swap halves between the two lanes of a beam (the re lane
// keeps samples 0..15 and receives their im parts, the im lane keeps 16..31 and receives their re parts),
// interleave with two PRMT per pair, and store 64 contiguous bytes per lane.  `out` = this lane's beam at the
// warp's first column, `nvalid` = samples that exist from there (tail tiles), `vec_ok` = 16-byte stores allowed.
__device__ __forceinline__ void epilogue_beams_tile(uint32_t taddr, __half2 *out, bool beam_ok, int nvalid, bool vec_ok,
                                                    float scale, bool upper, uint32_t bar_empty, bool lane0) {
  constexpr int CPW = TILE_T / (EPI_WARPS / 4);
  constexpr int NCH = CPW / 32;
#pragma unroll
  for (int ch = 0; ch < NCH; ++ch) {
    uint32_t v[32];
    BF_TMEM_LD_32x32b_X32(taddr + 32 * ch, v);
    tc_wait_ld();
    if (ch == NCH - 1) {
      tc_fence_before();
      __syncwarp();
      if (lane0) mbar_arrive(bar_empty);
    }
    uint32_t h[16];
#pragma unroll
    for (int j = 0; j < 16; ++j) {
      const __half2 q = __floats2half2_rn(__uint_as_float(v[2 * j]) * scale, __uint_as_float(v[2 * j + 1]) * scale);
      h[j] = *reinterpret_cast<const uint32_t *>(&q);
    }
    uint32_t o[16];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const uint32_t send = upper ? h[i] : h[8 + i];
      const uint32_t mine = upper ? h[8 + i] : h[i];
      const uint32_t recv = __shfl_xor_sync(0xffffffffu, send, 16);
      const uint32_t re = upper ? recv : mine, im = upper ? mine : recv;
      o[2 * i] = __byte_perm(re, im, 0x5410);      // (re, im) of the even sample
      o[2 * i + 1] = __byte_perm(re, im, 0x7632);  // (re, im) of the odd sample
    }
    const int t0 = 32 * ch + (upper ? 16 : 0);     // first of this lane's 16 samples
    if (!beam_ok) continue;
    uint32_t *dst = reinterpret_cast<uint32_t *>(out + t0);
    if (vec_ok && t0 + 16 <= nvalid) {
#pragma unroll
      for (int k = 0; k < 4; ++k)
        *reinterpret_cast<uint4 *>(dst + 4 * k) = make_uint4(o[4 * k], o[4 * k + 1], o[4 * k + 2], o[4 * k + 3]);
    } else {
#pragma unroll
      for (int k = 0; k < 16; ++k)
        if (t0 + k < nvalid) dst[k] = o[k];
    }
  }
}
// a lane quadrant that holds only padding rows just hands the stage back
__device__ __forceinline__ void epilogue_skip(uint32_t bar_empty, bool lane0) {
  __syncwarp();
  if (lane0) mbar_arrive(bar_empty);
}

}  // namespace bfk
