// bf_umma.cu -- the fused tensor-core beamformer for small arrays (2*nant <= 64, complex int8 input):
// hot-path rows a2..a5 in ONE persistent kernel.
//
//   a2 ingest      int8 (re,im) voltages  --LDG.128-->  registers  --PRMT/HSUB2-->  fp16, written
//                  into shared memory in the 128-byte-swizzled K-major layout tcgen05.mma reads
//                  (the paper fuses its 4-bit unpack into the kernel for the same reason: a separate
//                  pass "would cancel any speed-up")
//   a3 contraction per channel D[row][t] = sum_k' A[row][k'] X'[t][k'], rows = (re, im) of 64 beams,
//                  k' = 2n+{0,1}: the N_b x N_a coefficient matrix times the antenna vectors of 256
//                  time samples as tcgen05.mma kind::f16, M=128, N=256, K=16, fp32
//                  accumulators in TMEM.  Coefficients stay resident in shared memory for all time
//                  tiles of a channel (the paper's weight reuse).
//   a4 detection   d^2 straight out of TMEM (tcgen05.ld -> FFMA2); re and im rows of a beam sit 16
//                  lanes apart in the same warp, so |y|^2 = re^2 + im^2 needs one shuffle per OUTPUT bin
//   a5 integrate   sum over nint columns in registers, fp32 store to P[chan][beam][bin]
//
// Warp roles (one CTA per SM, persistent over a contiguous range of (chan, beam group, time tile)):
//   warps 0-7   epilogue: warp w owns TMEM lanes 32*(w&3).., accumulator stage (w>>2)
//   warps 8..   ingest/convert (CONV_WARPS), also load the coefficient tiles when the channel changes
//   last warp   TMEM allocation + the single MMA-issuing thread
// Pipelines (all mbarrier based): voltage stages full/empty (convert <-> MMA), coefficient buffers
// full/empty, TMEM accumulator stages full/empty (MMA <-> epilogue).
#include "bf_internal.h"
#include "ptx.cuh"

namespace {

constexpr int TILE_T = 256;                 // time samples per tile = UMMA N
constexpr int EPI_WARPS = 8;
constexpr int A_TILE_BYTES = BF_TILE_ROWS * 128;   // 128 rows x 64 fp16
constexpr int B_STAGE_BYTES = TILE_T * 128;        // 256 rows x 64 fp16
constexpr int MAX_INPUT_PIECES = TILE_T * 4;  // 16-byte input pieces per tile at nant = 32

struct Item { int c, g, tt; };

__device__ __forceinline__ Item decode_item(long long idx, int nG, int nTt) {
  Item it;
  it.tt = (int)(idx % nTt);
  long long cg = idx / nTt;
  it.g = (int)(cg % nG);
  it.c = (int)(cg / nG);
  return it;
}
// items are walked in order: (chan, beam group, time tile) with the time tile fastest
__device__ __forceinline__ void next_item(Item &it, int nG, int nTt) {
  if (++it.tt == nTt) {
    it.tt = 0;
    if (++it.g == nG) { it.g = 0; ++it.c; }
  }
}

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

__device__ __forceinline__ void st_shared_v4(uint32_t addr, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
  asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(addr), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
}
__device__ __forceinline__ uint4 ldg_nc_v4(const void *p) {
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
               : "l"(p));
  return r;
}

// NINT_T: integration length if it is a power of two <= 256, 0 = multiple of 256 (partial sums are
// added atomically into a zeroed output).
template <int NINT_T, int GROUP, int NSTAGE, int CONV_WARPS>
__global__ void __launch_bounds__((EPI_WARPS + CONV_WARPS + 1) * 32, 1)
bf_umma_k64_kernel(const BfParams p, const long long total_items, const int nG, const int nTt, const int nks) {
  extern __shared__ uint8_t smem_raw[];
  constexpr int CONV_THREADS = CONV_WARPS * 32;
  constexpr int MMA_WARP = EPI_WARPS + CONV_WARPS;

  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t sA = smem_base;                                  // 2 buffers x GROUP tiles
  const uint32_t sB = sA + 2 * GROUP * A_TILE_BYTES;              // NSTAGE stages
  const uint32_t sBar = sB + NSTAGE * B_STAGE_BYTES;              // barriers
  const uint32_t bar_b_full = sBar, bar_b_empty = sBar + 8 * NSTAGE;
  const uint32_t bar_a_full = sBar + 16 * NSTAGE, bar_a_empty = bar_a_full + 16;
  const uint32_t bar_t_full = bar_a_full + 32, bar_t_empty = bar_t_full + 16;
  const uint32_t s_tmem = bar_t_full + 32;

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

  if (threadIdx.x == 0) {
    for (int s = 0; s < NSTAGE; ++s) { mbar_init(bar_b_full + 8 * s, CONV_WARPS); mbar_init(bar_b_empty + 8 * s, 1); }
    for (int s = 0; s < 2; ++s) {
      mbar_init(bar_a_full + 8 * s, CONV_WARPS); mbar_init(bar_a_empty + 8 * s, 1);
      mbar_init(bar_t_full + 8 * s, 1);          mbar_init(bar_t_empty + 8 * s, EPI_WARPS / 2);
    }
    fence_barrier_init();
  }
  if (warp == MMA_WARP) tmem_alloc(s_tmem, 512);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(s_tmem));

  // this CTA's contiguous item range
  const long long it0 = total_items * blockIdx.x / gridDim.x;
  const long long it1 = total_items * (blockIdx.x + 1) / gridDim.x;
  const int n_items = (int)(it1 - it0);
  const int nMt = p.nMt;

  if (warp < EPI_WARPS) {
    // =========================================================================== epilogue
    const int quad = warp & 3, grp = warp >> 2;
    const uint32_t t_lane = tmem_base + ((uint32_t)(quad * 32) << 16) + grp * TILE_T;
    constexpr int SUB = (NINT_T == 0 || NINT_T > 32) ? 32 : NINT_T;        // columns per partial sum
    constexpr int NSUB = 32 / SUB;                                          // partial sums per 32-column chunk
    constexpr int CPB = NINT_T == 0 ? 8 : (NINT_T <= 32 ? 1 : NINT_T / 32);  // chunks per bin
    constexpr int BINS_PER_TILE = NINT_T == 0 ? 1 : TILE_T / NINT_T;
    const bool vec_ok = (BINS_PER_TILE >= 4) && (p.nbin % 4 == 0) && ((reinterpret_cast<uintptr_t>(p.pow) & 15) == 0);
    int u = 0;
    Item it = decode_item(it0, nG, nTt);
    for (int i = 0; i < n_items; ++i, next_item(it, nG, nTt)) {
      const int gm = min(GROUP, nMt - it.g * GROUP);
      for (int m = 0; m < gm; ++m, ++u) {
        if ((u & 1) != grp) continue;
        mbar_wait(bar_t_full + 8 * grp, (u >> 1) & 1);
        tc_fence_after();
        const int mt = it.g * GROUP + m;
        const int beam0 = mt * BF_TILE_BEAMS + quad * 16;
        if (beam0 < p.nbeam) {  // warp-uniform: this lane quadrant holds real beams
          const int beam = beam0 + (lane & 15);
          const bool writer = (lane < 16) && (beam < p.nbeam);
          float *prow = p.pow + ((size_t)it.c * p.nbeam + beam) * p.nbin;
          const int bin0 = NINT_T == 0 ? (int)(((long long)it.tt * TILE_T) / p.nint) : it.tt * BINS_PER_TILE;
          uint32_t r[2][32];
          BF_TMEM_LD_32x32b_X32(t_lane, r[0]);
          float binacc = 0.f;
          float ob[4];
#pragma unroll
          for (int ch = 0; ch < 8; ++ch) {
            tc_wait_ld();
            if (ch + 1 < 8) { BF_TMEM_LD_32x32b_X32(t_lane + 32 * (ch + 1), r[(ch + 1) & 1]); }
            const uint32_t *v = r[ch & 1];
#pragma unroll
            for (int s = 0; s < NSUB; ++s) {
              float sum;
              if constexpr (SUB == 1) {
                const float d = __uint_as_float(v[s]);
                sum = d * d;
              } else {
                constexpr int NACC = SUB >= 8 ? 4 : SUB / 2;
                float2 a[NACC];
#pragma unroll
                for (int q = 0; q < NACC; ++q) a[q] = make_float2(0.f, 0.f);
#pragma unroll
                for (int j = 0; j < SUB / 2; ++j) {
                  const float2 d = make_float2(__uint_as_float(v[s * SUB + 2 * j]), __uint_as_float(v[s * SUB + 2 * j + 1]));
                  a[j % NACC] = ffma2(d, d, a[j % NACC]);
                }
                sum = 0.f;
#pragma unroll
                for (int q = 0; q < NACC; ++q) sum += a[q].x + a[q].y;
              }
              if (CPB > 1) {
                binacc += sum;
                if ((ch + 1) % CPB != 0) continue;
                sum = binacc;
                binacc = 0.f;
              }
              const float tot = sum + __shfl_xor_sync(0xffffffffu, sum, 16);  // re^2 rows + im^2 rows
              if (NINT_T == 0) {
                if (writer) atomicAdd(prow + bin0, tot);
              } else {
                const int jb = (ch / CPB) * NSUB + s;  // bin index inside the tile (compile-time)
                const int j = bin0 + jb;
                if (vec_ok) {
                  ob[jb & 3] = tot;
                  if ((jb & 3) == 3 && writer && j < p.nbin)
                    *reinterpret_cast<float4 *>(prow + j - 3) = make_float4(ob[0], ob[1], ob[2], ob[3]);
                } else if (writer && j < p.nbin) {
                  prow[j] = tot;
                }
              }
            }
          }
        }
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_t_empty + 8 * grp);
      }
    }
  } else if (warp < MMA_WARP) {
    // =========================================================================== ingest / convert
    constexpr int PIECES = MAX_INPUT_PIECES / CONV_THREADS;  // 16-byte input pieces per thread per tile
    const int ctid = threadIdx.x - EPI_WARPS * 32;
    const int npr = p.nant / 8;                  // 16-byte pieces per time sample (int8: 2*nant bytes)
    const int npieces = TILE_T * npr;
    const size_t row_bytes = (size_t)2 * p.nant;
    const char *volt = reinterpret_cast<const char *>(p.volt);
    // zero the stages once: K' columns beyond 2*nant must read as 0, never as stale NaN patterns
    for (int o = ctid * 16; o < NSTAGE * B_STAGE_BYTES; o += CONV_THREADS * 16) st_shared_v4(sB + o, 0, 0, 0, 0);
    asm volatile("bar.sync 1, %0;" ::"n"(CONV_THREADS) : "memory");

    // a thread converts the same pieces of every tile: row t, 16-byte piece q of that row
    int p_t[PIECES];        // time row inside the tile (TILE_T = not mine)
    uint32_t p_src[PIECES]; // byte offset inside the tile's input
    uint32_t p_dst[PIECES]; // byte offset of the first output chunk inside a stage (second chunk: ^ 16)
#pragma unroll
    for (int k = 0; k < PIECES; ++k) {
      const int pc = ctid + k * CONV_THREADS;
      const int t = pc / npr, q = pc - t * npr;
      p_t[k] = pc < npieces ? t : TILE_T;
      p_src[k] = (uint32_t)(t * row_bytes + 16 * q);
      p_dst[k] = (uint32_t)((t >> 3) * 1024 + (t & 7) * 128 + (((2 * q) ^ (t & 7)) << 4));
    }
    auto load_tile = [&](uint4 (&dst)[PIECES], const Item &it) {
      const int t_base = it.tt * TILE_T;
      const int rows = min(TILE_T, p.nsamp - t_base);
      const char *base = volt + ((size_t)it.c * p.nsamp + t_base) * row_bytes;
#pragma unroll
      for (int k = 0; k < PIECES; ++k) {
        if (p_t[k] < rows) dst[k] = ldg_nc_v4(base + p_src[k]);
        else dst[k] = make_uint4(0u, 0u, 0u, 0u);
      }
    };
    int ag = 0, prev_c = -1, prev_g = -1;
    auto convert_tile = [&](const uint4 (&src)[PIECES], const Item &it, int i) {
      if (it.c != prev_c || it.g != prev_g) {
        // new (channel, beam group): bring its coefficient tiles into the other A buffer
        prev_c = it.c; prev_g = it.g;
        const int ab = ag & 1;
        mbar_wait(bar_a_empty + 8 * ab, ((ag >> 1) & 1) ^ 1);
        const int gm = min(GROUP, nMt - it.g * GROUP);
        const char *wsrc = reinterpret_cast<const char *>(p.wop) + ((size_t)it.c * nMt + (size_t)it.g * GROUP) * A_TILE_BYTES;
        for (int pc = ctid; pc < gm * (A_TILE_BYTES / 16); pc += CONV_THREADS) {
          const int row = pc >> 3, j = pc & 7;  // row over gm*128 rows
          const uint4 w = *reinterpret_cast<const uint4 *>(wsrc + (size_t)pc * 16);
          const uint32_t dst = sA + ab * GROUP * A_TILE_BYTES + row * 128 + ((j ^ (row & 7)) << 4);
          st_shared_v4(dst, w.x, w.y, w.z, w.w);
        }
        fence_proxy_async_smem();
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_a_full + 8 * ab);
        ++ag;
      }
      const int st = i % NSTAGE;
      mbar_wait(bar_b_empty + 8 * st, ((i / NSTAGE) & 1) ^ 1);
      const uint32_t sdst = sB + st * B_STAGE_BYTES;
#pragma unroll
      for (int k = 0; k < PIECES; ++k) {
        if (p_t[k] < TILE_T) {
          uint32_t h[8];
          cvt_i8x4_f16x4(src[k].x, h[0], h[1]);
          cvt_i8x4_f16x4(src[k].y, h[2], h[3]);
          cvt_i8x4_f16x4(src[k].z, h[4], h[5]);
          cvt_i8x4_f16x4(src[k].w, h[6], h[7]);
          st_shared_v4(sdst + p_dst[k], h[0], h[1], h[2], h[3]);
          st_shared_v4(sdst + (p_dst[k] ^ 16u), h[4], h[5], h[6], h[7]);
        }
      }
      fence_proxy_async_smem();
      __syncwarp();
      if (lane == 0) mbar_arrive(bar_b_full + 8 * st);
    };
    // two register buffers, loads issued one tile ahead of their use
    uint4 bufA[PIECES], bufB[PIECES];
    Item itA = decode_item(it0, nG, nTt), itB;
    if (n_items > 0) load_tile(bufA, itA);
    for (int i = 0; i < n_items; i += 2) {
      itB = itA; next_item(itB, nG, nTt);
      if (i + 1 < n_items) load_tile(bufB, itB);
      convert_tile(bufA, itA, i);
      itA = itB; next_item(itA, nG, nTt);
      if (i + 1 < n_items) {
        if (i + 2 < n_items) load_tile(bufA, itA);
        convert_tile(bufB, itB, i + 1);
      }
    }
  } else if (lane == 0) {
    // =========================================================================== MMA issue (one thread)
    constexpr uint32_t idesc = make_idesc_f16(BF_TILE_ROWS, TILE_T);
    int ag = 0, prev_c = -1, prev_g = -1, ab = 0, u = 0;
    Item it = decode_item(it0, nG, nTt);
    for (int i = 0; i < n_items; ++i, next_item(it, nG, nTt)) {
      if (it.c != prev_c || it.g != prev_g) {
        if (ag > 0) tc_commit(bar_a_empty + 8 * ab);  // everything issued so far has left the old buffer
        prev_c = it.c; prev_g = it.g;
        ab = ag & 1;
        mbar_wait(bar_a_full + 8 * ab, (ag >> 1) & 1);
        ++ag;
      }
      const int st = i % NSTAGE;
      mbar_wait(bar_b_full + 8 * st, (i / NSTAGE) & 1);
      tc_fence_after();
      const int gm = min(GROUP, nMt - it.g * GROUP);
      const uint64_t bdesc = make_sdesc_k_sw128(sB + st * B_STAGE_BYTES);
      for (int m = 0; m < gm; ++m, ++u) {
        const int acc = u & 1;
        mbar_wait(bar_t_empty + 8 * acc, ((u >> 1) & 1) ^ 1);
        tc_fence_after();
        const uint64_t adesc = make_sdesc_k_sw128(sA + (ab * GROUP + m) * A_TILE_BYTES);
        const uint32_t d = tmem_base + acc * TILE_T;
        for (int k = 0; k < nks; ++k)  // advance 16 fp16 = 32 bytes along K inside the swizzle atom
          mma_f16_ss(d, adesc + 2 * k, bdesc + 2 * k, idesc, k > 0);
        tc_commit(bar_t_full + 8 * acc);
      }
      tc_commit(bar_b_empty + 8 * st);
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == MMA_WARP) tmem_dealloc(tmem_base, 512);
}

template <int NINT_T, int GROUP, int NSTAGE, int CONV_WARPS>
cudaError_t launch_k64(const BfParams &p, int sm_count, cudaStream_t st) {
  const int nG = (p.nMt + GROUP - 1) / GROUP;
  const int nTt = (p.nsamp + TILE_T - 1) / TILE_T;
  const long long total = (long long)p.nchan_run * nG * nTt;
  const int nks = (2 * p.nant + 15) / 16;
  const size_t smem = 1024 + 2 * GROUP * A_TILE_BYTES + NSTAGE * B_STAGE_BYTES + 256;
  auto kern = bf_umma_k64_kernel<NINT_T, GROUP, NSTAGE, CONV_WARPS>;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  if (NINT_T == 0) {
    e = cudaMemsetAsync(p.pow, 0, (size_t)p.nchan_run * p.nbeam * p.nbin * sizeof(float), st);
    if (e != cudaSuccess) return e;
  }
  const int grid = (int)(total < sm_count ? total : sm_count);
  kern<<<grid, (EPI_WARPS + CONV_WARPS + 1) * 32, smem, st>>>(p, total, nG, nTt, nks);
  return cudaGetLastError();
}

template <int NINT_T>
cudaError_t launch_k64_nint(const BfParams &p, int sm_count, cudaStream_t st) {
  if (p.nMt <= 2) return launch_k64<NINT_T, 2, 4, 8>(p, sm_count, st);
  return launch_k64<NINT_T, 4, 3, 8>(p, sm_count, st);
}

}  // namespace

bool bf_umma_supported(const bf_ctx *c, const char **why) {
  if (c->dtype != BF_CI8) { *why = "only complex int8 input so far"; return false; }
  if (c->nant % 8 != 0 || c->nant > 32) { *why = "needs nant in {8,16,24,32}"; return false; }
  const int I = c->nint;
  const bool pow2_small = I <= 256 && (I & (I - 1)) == 0;
  if (!pow2_small && I % 256 != 0) { *why = "needs nint a power of two <= 256 or a multiple of 256"; return false; }
  return true;
}

cudaError_t bf_launch_umma(const BfParams &p, int dtype, int sm_count, cudaStream_t st) {
  if (dtype != BF_CI8) return cudaErrorNotSupported;
  switch (p.nint) {
    case 1: return launch_k64_nint<1>(p, sm_count, st);
    case 2: return launch_k64_nint<2>(p, sm_count, st);
    case 4: return launch_k64_nint<4>(p, sm_count, st);
    case 8: return launch_k64_nint<8>(p, sm_count, st);
    case 16: return launch_k64_nint<16>(p, sm_count, st);
    case 32: return launch_k64_nint<32>(p, sm_count, st);
    case 64: return launch_k64_nint<64>(p, sm_count, st);
    case 128: return launch_k64_nint<128>(p, sm_count, st);
    case 256: return launch_k64_nint<256>(p, sm_count, st);
    default: return launch_k64_nint<0>(p, sm_count, st);
  }
}
