// bf_umma_i8.cu -- the fused tensor-core beamformer for FEW beams (<= 32) on small arrays (2*nant <= 64,
// complex int8 input): hot-path rows a2..a5 in the regime where the path is HBM-bound (SURVEY.md 8(d):
// below ~70 beams the input stream, not the arithmetic, sets the time).
//
// Why a second small-array kernel: in bf_umma.cu every input byte crosses shared memory four times (bulk
// copy in, LDS, STS of the fp16 image, operand read by the MMA) plus the coefficient tile's re-read -- ~900
// shared-memory clocks per 16 KiB of input, which caps that kernel at ~0.6 of the HBM roofline however few
// beams there are (profiles/r01_ncu_full_summary.md).  Here the int8 voltages are NEVER converted:
//
//   a2 ingest      TMA tensor copies (32 samples x 64 bytes, 64-byte swizzle) land the raw int8 rows in shared
//                  memory in exactly the K-major layout tcgen05.mma reads -- the paper's in-kernel unpack
//                   becomes "no unpack at all"
//   a3 contraction tcgen05.mma kind::i8 with the roles swapped: the A operand (M = 128 rows) is TIME, the B
//                  operand (N columns) is the coefficient rows, so TMEM holds only real beams:
//                  D[t][col] = sum_k' X'[t][k'] A[col][k'],  k' = 2n+{0,1}, int32 accumulators (exact).
//                  The fp64-derived weights (Eq. 1) are quantised to 15 bits as TWO int8 limbs,
//                  w = (128 hi + lo) / 16256 (|error| <= 3.1e-5, 8x finer than the fp16 operand), four
//                  columns per beam: (re hi, im hi, re lo, im lo)
//   a4 detection   one thread owns one time sample and ALL columns of it: re = 128 hi + lo (integer, exact),
//                  |y|^2 = re^2 + im^2 in fp32 -- re and im meet in the same thread, no shuffle per sample
//   a5 integrate   bins of nint <= 32 samples: transposing butterfly across the lanes of a warp (8 beams x 32
//                  lanes in 9 shuffles); nint = 32 G: the TMA places the samples so that ONE warp sees all of a
//                  bin in G consecutive tiles and keeps the running sums in registers
//
// Warp roles (one persistent CTA per SM over a contiguous range of (channel, super-tile)): warps 0-7 epilogue
// (two sets of four; set s takes the super-tiles of its parity, warp quadrant q = TMEM lanes 32q..), warp 8
// MMA issue + TMEM allocation, warp 9 (WIDE: 9 and 10) one thread each issuing TMA.  ~190 KiB of input in
// flight per SM.  All role loops keep 32-bit wrap counters: a 64-bit division per tile in the single producer
// thread was measurably on the critical path.
#include <cuda.h>

#include "bf_internal.h"
#include "bf_tmap.h"
#include "ptx.cuh"

namespace {

constexpr int L_TILE_T = 128;                              // time samples per tile = UMMA M
constexpr int L_ROW_BYTES = 64;                            // K' bytes per row (2 * 32 antennas)
constexpr int L_STAGE_BYTES = L_TILE_T * L_ROW_BYTES;      // 8 KiB
constexpr int L_BOX_ROWS = 32;                             // one TMA box = one warp's samples
constexpr int L_BOX_BYTES = L_BOX_ROWS * L_ROW_BYTES;
constexpr int L_EPI_WARPS = 8;
constexpr int L_MMA_WARP = 8, L_TMA_WARP = 9;
constexpr int L_THREADS = 10 * 32;

__host__ __device__ constexpr int ilog2(int x) { return x <= 1 ? 0 : 1 + ilog2(x >> 1); }

// Transposing butterfly: N running sums per lane, bins of 2*O lanes.  While more than one value is left each
// step halves the values (a lane keeps the half its bit selects and receives the partner's contribution to
// it); once one value is left the remaining steps are plain butterfly adds.
template <int N, int O>
struct LaneReduce {
  static __device__ __forceinline__ void run(float *p, int lane) {
    if constexpr (O >= 1) {
      if constexpr (N > 1) {
        const bool up = (lane & O) != 0;
#pragma unroll
        for (int j = 0; j < N / 2; ++j) {
          const float send = up ? p[j] : p[j + N / 2];
          const float keep = up ? p[j + N / 2] : p[j];
          p[j] = keep + __shfl_xor_sync(0xffffffffu, send, O);
        }
        LaneReduce<N / 2, O / 2>::run(p, lane);
      } else {
        p[0] += __shfl_xor_sync(0xffffffffu, p[0], O);
        LaneReduce<1, O / 2>::run(p, lane);
      }
    }
  }
};

// NCOL: accumulator columns = 4 * beam capacity (32 / 64 / 128 -> 8 / 16 / 32 beams).  LBIN: lanes per bin
// = nint for nint <= 32, else 32 (nint = 32 G, G tiles per super-tile).  NST: voltage stages.
template <int NCOL, int LBIN, int NST>
__global__ void __launch_bounds__(L_THREADS, 1)
bf_umma_i8_kernel(const BfParams p, const __grid_constant__ CUtensorMap tmap, const __grid_constant__ CUtensorMap tmap32,
                  const long long total_super,
                  const int n_super_chan, const int G, const int nks) {
  extern __shared__ uint8_t smem_raw[];
  constexpr int W_BYTES = NCOL * L_ROW_BYTES;               // one channel's coefficient rows
  constexpr int NACC = 512 / NCOL;                          // accumulator stages in TMEM
  constexpr int NCH = NCOL / 32;                            // 32-column (8-beam) chunks
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t sW = smem_base;                            // 2 coefficient buffers
  const uint32_t sA = sW + 2 * W_BYTES;                     // NST voltage stages (W_BYTES is a multiple of 1024)
  const uint32_t sBar = sA + NST * L_STAGE_BYTES;
  const uint32_t bar_a_full = sBar, bar_a_empty = bar_a_full + 8 * NST;
  const uint32_t bar_w_full = bar_a_empty + 8 * NST, bar_w_empty = bar_w_full + 16;
  const uint32_t bar_t_full = bar_w_empty + 16, bar_t_empty = bar_t_full + 8 * NACC;
  const uint32_t s_tmem = bar_t_empty + 8 * NACC;

  const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0), lane = threadIdx.x & 31;

  if (threadIdx.x == 0) {
    for (int s = 0; s < NST; ++s) { mbar_init(bar_a_full + 8 * s, 1); mbar_init(bar_a_empty + 8 * s, 1); }
    for (int s = 0; s < 2; ++s) { mbar_init(bar_w_full + 8 * s, 1); mbar_init(bar_w_empty + 8 * s, 1); }
    for (int s = 0; s < NACC; ++s) { mbar_init(bar_t_full + 8 * s, 1); mbar_init(bar_t_empty + 8 * s, 4); }
    fence_barrier_init();
  }
  if (warp == L_MMA_WARP) tmem_alloc(s_tmem, 512);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(s_tmem));
  tmem_base = __shfl_sync(0xffffffffu, tmem_base, 0);
  probe_mark(p.probe, 0);

  // this CTA's contiguous range of super-tiles (super-tile = G tiles of 128 samples = 4 bins of 32 G samples,
  // or 128 / nint bins for nint <= 32)
  const long long s0 = total_super * blockIdx.x / gridDim.x;
  const long long s1 = total_super * (blockIdx.x + 1) / gridDim.x;
  const int n_super = (int)(s1 - s0);
  const int c0 = (int)(s0 / n_super_chan), sp0 = (int)(s0 % n_super_chan);

  if (warp < L_EPI_WARPS) {
    // =========================================================================== epilogue
    const int quad = warp & 3, set = warp >> 2;
    const bool lane0 = lane == 0;
    const uint32_t t_lane = tmem_base + ((uint32_t)(quad * 32) << 16);
    constexpr int HALVINGS = ilog2(LBIN) < 3 ? ilog2(LBIN) : 3;   // 8 values per chunk: at most 3 halvings
    constexpr int NFINAL = 8 >> HALVINGS;                         // complete sums a lane ends up with, per chunk
    int beam_off = 0;                                             // first beam (inside a chunk) this lane ends up with
#pragma unroll
    for (int k = 0; k < HALVINGS; ++k)
      if (lane & (LBIN >> (k + 1))) beam_off += 8 >> (k + 1);
    const bool writer = (lane & ((LBIN >> HALVINGS) - 1)) == 0;   // one lane per (bin, beam) after the plain butterfly steps
    const int nbeam = p.nbeam, nbin = p.nbin;
    int c = c0, sp = sp0;
    int ti = 0;                                                   // tile counter of this CTA (all roles count alike)
    for (int s = 0; s < n_super; ++s) {
      if ((s & 1) == set) {
        float acc[NCH][8];
#pragma unroll
        for (int ch = 0; ch < NCH; ++ch)
#pragma unroll
          for (int i = 0; i < 8; ++i) acc[ch][i] = 0.f;
        for (int g = 0; g < G; ++g, ++ti) {
          const int a = ti & (NACC - 1);
          mbar_wait(bar_t_full + 8 * a, (uint32_t)((ti >> ilog2(NACC)) & 1));
          tc_fence_after();
#pragma unroll
          for (int ch = 0; ch < NCH; ++ch) {
            uint32_t v[32];
            BF_TMEM_LD_32x32b_X32(t_lane + a * NCOL + 32 * ch, v);
            tc_wait_ld();
            if (ch == NCH - 1) {  // all of this warp's columns are in registers: hand the accumulator back
              tc_fence_before();
              __syncwarp();
              if (lane0) mbar_arrive(bar_t_empty + 8 * a);
            }
#pragma unroll
            for (int i = 0; i < 8; ++i) {
              const int re = ((int)v[4 * i] << 7) + (int)v[4 * i + 2];       // 128 hi + lo, exact
              const int im = ((int)v[4 * i + 1] << 7) + (int)v[4 * i + 3];
              const float fr = (float)re, fi = (float)im;
              acc[ch][i] = fmaf(fr, fr, fmaf(fi, fi, acc[ch][i]));
            }
          }
        }
        // integrate across the lanes of each bin, then one lane per (bin, beam) stores
        const float sc = (float)p.i8scale[c];
        const float sc2 = sc * sc;
        const int bin = (32 / LBIN) * (4 * sp + quad) + lane / LBIN;
#pragma unroll
        for (int ch = 0; ch < NCH; ++ch) {
          LaneReduce<8, LBIN / 2>::run(acc[ch], lane);
          if (writer && bin < nbin) {
#pragma unroll
            for (int j = 0; j < NFINAL; ++j) {
              const int beam = 8 * ch + beam_off + j;
              if (beam < nbeam) p.pow[((size_t)c * nbeam + beam) * nbin + bin] = acc[ch][j] * sc2;
            }
          }
        }
      } else {
        ti += G;
      }
      if (++sp == n_super_chan) { sp = 0; ++c; }
    }
  } else if (warp == L_MMA_WARP) {
    // =========================================================================== MMA issue
    constexpr uint32_t idesc = make_idesc_i8(L_TILE_T, NCOL);
    int c = c0, sp = sp0, prev_c = -1, wi = 0, wb = 0;
    int ti = 0, st = 0;
    uint32_t st_par = 0;
    for (int s = 0; s < n_super; ++s) {
      if (c != prev_c) {
        if (wi > 0 && elect_one()) tc_commit(bar_w_empty + 8 * wb);   // my MMAs so far have left the old buffer
        prev_c = c;
        wb = wi & 1;
        mbar_wait(bar_w_full + 8 * wb, (uint32_t)((wi >> 1) & 1));
        ++wi;
      }
      const uint64_t bdesc = make_sdesc_k_sw64(sW + wb * W_BYTES);
      for (int g = 0; g < G; ++g, ++ti) {
        const int a = ti & (NACC - 1);
        mbar_wait(bar_a_full + 8 * st, st_par);
        mbar_wait(bar_t_empty + 8 * a, (uint32_t)(((ti >> ilog2(NACC)) & 1) ^ 1));
        tc_fence_after();
        if (elect_one()) {
          const uint64_t adesc = make_sdesc_k_sw64(sA + st * L_STAGE_BYTES);
          const uint32_t d = tmem_base + a * NCOL;
#pragma unroll
          for (int k = 0; k < 2; ++k)   // 32 bytes along K inside the 64-byte swizzle atom
            if (k < nks) mma_i8_ss(d, adesc + 2 * k, bdesc + 2 * k, idesc, k > 0);
          tc_commit(bar_t_full + 8 * a);
          tc_commit(bar_a_empty + 8 * st);
        }
        __syncwarp();
        if (++st == NST) { st = 0; st_par ^= 1; }
      }
      if (++sp == n_super_chan) { sp = 0; ++c; }
    }
  } else if (warp == L_TMA_WARP && lane == 0) {
    // =========================================================================== TMA producer (one thread)
    tma_prefetch_desc(&tmap);
    tma_prefetch_desc(&tmap32);
    int c = c0, sp = sp0, prev_c = -1, wi = 0;
    int st = 0;
    uint32_t st_par = 1;
    for (int s = 0; s < n_super; ++s) {
      if (c != prev_c) {
        prev_c = c;
        const int wb = wi & 1;
        mbar_wait(bar_w_empty + 8 * wb, (uint32_t)(((wi >> 1) & 1) ^ 1));
        mbar_arrive_expect_tx(bar_w_full + 8 * wb, W_BYTES);
        bulk_g2s(sW + wb * W_BYTES, reinterpret_cast<const char *>(p.wop8) + (size_t)c * W_BYTES, W_BYTES, bar_w_full + 8 * wb);
        ++wi;
      }
      for (int g = 0; g < G; ++g) {
        mbar_wait(bar_a_empty + 8 * st, st_par);
        mbar_arrive_expect_tx(bar_a_full + 8 * st, L_STAGE_BYTES);
        if (G == 1) {  // the four quadrants are contiguous: one box of 128 samples
          tma_load_3d(sA + st * L_STAGE_BYTES, &tmap, 0, L_TILE_T * sp, c, bar_a_full + 8 * st);
        } else {
#pragma unroll
          for (int q = 0; q < 4; ++q)  // warp quadrant q of this tile sees samples 32 G (4 sp + q) + 32 g ..
            tma_load_3d(sA + st * L_STAGE_BYTES + q * L_BOX_BYTES, &tmap32, 0, 32 * G * (4 * sp + q) + 32 * g, c,
                        bar_a_full + 8 * st);
        }
        if (++st == NST) { st = 0; st_par ^= 1; }
      }
      if (++sp == n_super_chan) { sp = 0; ++c; }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == L_MMA_WARP) tmem_dealloc(tmem_base, 512);
  probe_mark(p.probe, 1);
}

// ---- WIDE variant (nant = 32 exactly, nsamp even): shared-memory rows of 128 bytes = TWO samples --------------
// The TMA engine's cost is per box ROW, and 64-byte rows cap it near 11 B/clk/SM (measured) -- below the HBM
// rate.  With 32 antennas two consecutive samples are 128 contiguous bytes, so the tensor map views the
// voltages as rows of 128 bytes (128-byte swizzle) and the K extent of a row is sliced by the MMA instead:
// descriptor offsets 0 / 32 bytes contract the EVEN sample of every row into accumulator E, offsets 64 / 96
// bytes the ODD sample into accumulator O.  A tile is 128 rows = 256 samples = 16 KiB; lane r of the two
// accumulators holds samples 2r and 2r+1, so a bin of nint samples is nint/2 lanes wide.
// LBIN: lanes per bin (nint / 2 for 2 <= nint <= 64, 32 for nint = 64 G); 0 = nint 1 (two bins per lane).
constexpr int W_STAGE_BYTES = 128 * 128;

// BEAMS: voltage-beam mode (row f4): y itself as fp16 (re, im), no detection, nint ignored.
template <int NCOL, int LBIN, int NST, bool BEAMS>
__global__ void __launch_bounds__(L_THREADS + 32, 1)
bf_umma_i8w_kernel(const BfParams p, const __grid_constant__ CUtensorMap tmap, const __grid_constant__ CUtensorMap tmap32,
                   const long long total_super, const int n_super_chan, const int G) {
  extern __shared__ uint8_t smem_raw[];
  constexpr int W_BYTES = NCOL * L_ROW_BYTES;
  constexpr int NACC = 512 / (2 * NCOL);                    // accumulator PAIRS in TMEM
  constexpr int NCH = NCOL / 32;
  constexpr int LB = LBIN == 0 ? 1 : LBIN;
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t sW = smem_base;
  const uint32_t sA = sW + 2 * W_BYTES;
  const uint32_t sBar = sA + NST * W_STAGE_BYTES;
  const uint32_t bar_a_full = sBar, bar_a_empty = bar_a_full + 8 * NST;
  const uint32_t bar_w_full = bar_a_empty + 8 * NST, bar_w_empty = bar_w_full + 16;
  const uint32_t bar_t_full = bar_w_empty + 16, bar_t_empty = bar_t_full + 8 * NACC;
  const uint32_t s_tmem = bar_t_empty + 8 * NACC;

  const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0), lane = threadIdx.x & 31;

  if (threadIdx.x == 0) {
    for (int s = 0; s < NST; ++s) { mbar_init(bar_a_full + 8 * s, 1); mbar_init(bar_a_empty + 8 * s, 1); }
    for (int s = 0; s < 2; ++s) { mbar_init(bar_w_full + 8 * s, 1); mbar_init(bar_w_empty + 8 * s, 1); }
    for (int s = 0; s < NACC; ++s) { mbar_init(bar_t_full + 8 * s, 1); mbar_init(bar_t_empty + 8 * s, 4); }
    fence_barrier_init();
  }
  if (warp == L_MMA_WARP) tmem_alloc(s_tmem, 512);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(s_tmem));
  tmem_base = __shfl_sync(0xffffffffu, tmem_base, 0);
  probe_mark(p.probe, 0);

  const long long s0 = total_super * blockIdx.x / gridDim.x;
  const long long s1 = total_super * (blockIdx.x + 1) / gridDim.x;
  const int n_super = (int)(s1 - s0);
  const int c0 = (int)(s0 / n_super_chan), sp0 = (int)(s0 % n_super_chan);

  if (warp < L_EPI_WARPS) {
    // =========================================================================== epilogue
    const int quad = warp & 3, set = warp >> 2;
    const bool lane0 = lane == 0;
    const uint32_t t_lane = tmem_base + ((uint32_t)(quad * 32) << 16);
    constexpr int HALVINGS = ilog2(LB) < 3 ? ilog2(LB) : 3;
    constexpr int NFINAL = 8 >> HALVINGS;
    int beam_off = 0;
#pragma unroll
    for (int k = 0; k < HALVINGS; ++k)
      if (lane & (LB >> (k + 1))) beam_off += 8 >> (k + 1);
    const bool writer = (lane & ((LB >> HALVINGS) - 1)) == 0;
    const int nbeam = p.nbeam, nbin = p.nbin;
    // 8-byte stores (two samples per lane) need an 8-byte aligned output; nsamp is even in this variant
    const bool vec8 = ((reinterpret_cast<uintptr_t>(BEAMS ? p.beams : (void *)p.pow)) & 7) == 0;
    int c = c0, sp = sp0;
    int ti = 0;                                                   // tile counter of this CTA (all roles count alike)
    for (int s = 0; s < n_super; ++s) {
      if (BEAMS && (s & 1) == set) {
        // ---- voltage beams: lane r holds samples 2r and 2r+1 of every beam; 8 bytes per beam and lane
        const int a = ti & (NACC - 1);
        mbar_wait(bar_t_full + 8 * a, (uint32_t)((ti >> ilog2(NACC)) & 1));
        tc_fence_after();
        const float sc = (float)p.i8scale[c] * p.beam_scale;
        const int t = 2 * (32 * (4 * sp + quad) + lane);
        __half2 *yrow = reinterpret_cast<__half2 *>(p.beams) + (size_t)c * nbeam * p.nsamp + t;
#pragma unroll
        for (int ch = 0; ch < NCH; ++ch) {
          uint32_t v[32], u[32];
          BF_TMEM_LD_32x32b_X32(t_lane + a * 2 * NCOL + 32 * ch, v);
          BF_TMEM_LD_32x32b_X32(t_lane + a * 2 * NCOL + NCOL + 32 * ch, u);
          tc_wait_ld();
          if (ch == NCH - 1) {
            tc_fence_before();
            __syncwarp();
            if (lane0) mbar_arrive(bar_t_empty + 8 * a);
          }
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            const int re = ((int)v[4 * i] << 7) + (int)v[4 * i + 2];
            const int im = ((int)v[4 * i + 1] << 7) + (int)v[4 * i + 3];
            const int ro = ((int)u[4 * i] << 7) + (int)u[4 * i + 2];
            const int io = ((int)u[4 * i + 1] << 7) + (int)u[4 * i + 3];
            const __half2 ye = __floats2half2_rn((float)re * sc, (float)im * sc);
            const __half2 yo = __floats2half2_rn((float)ro * sc, (float)io * sc);
            if (8 * ch + i < nbeam && t < p.nsamp) {
              __half2 *dst = yrow + (size_t)(8 * ch + i) * p.nsamp;
              if (vec8) {
                *reinterpret_cast<uint2 *>(dst) =
                    make_uint2(*reinterpret_cast<const uint32_t *>(&ye), *reinterpret_cast<const uint32_t *>(&yo));
              } else {  // output pointer only 4-byte aligned (bf.h allows it): two scalar stores
                dst[0] = ye;
                dst[1] = yo;
              }
            }
          }
        }
        ++ti;
      } else if ((s & 1) == set) {
        float acc[NCH][8], acc1[LBIN == 0 ? NCH : 1][8];   // acc1: the odd sample's own bin when nint = 1
#pragma unroll
        for (int ch = 0; ch < NCH; ++ch)
#pragma unroll
          for (int i = 0; i < 8; ++i) acc[ch][i] = 0.f;
        for (int g = 0; g < G; ++g, ++ti) {
          const int a = ti & (NACC - 1);
          mbar_wait(bar_t_full + 8 * a, (uint32_t)((ti >> ilog2(NACC)) & 1));
          tc_fence_after();
#pragma unroll
          for (int ch = 0; ch < NCH; ++ch) {
            uint32_t v[32], u[32];
            BF_TMEM_LD_32x32b_X32(t_lane + a * 2 * NCOL + 32 * ch, v);          // even samples
            BF_TMEM_LD_32x32b_X32(t_lane + a * 2 * NCOL + NCOL + 32 * ch, u);   // odd samples
            tc_wait_ld();
            if (ch == NCH - 1) {
              tc_fence_before();
              __syncwarp();
              if (lane0) mbar_arrive(bar_t_empty + 8 * a);
            }
#pragma unroll
            for (int i = 0; i < 8; ++i) {
              const int re = ((int)v[4 * i] << 7) + (int)v[4 * i + 2];       // 128 hi + lo, exact
              const int im = ((int)v[4 * i + 1] << 7) + (int)v[4 * i + 3];
              const int ro = ((int)u[4 * i] << 7) + (int)u[4 * i + 2];
              const int io = ((int)u[4 * i + 1] << 7) + (int)u[4 * i + 3];
              const float fr = (float)re, fi = (float)im, gr = (float)ro, gi = (float)io;
              if constexpr (LBIN == 0) {
                acc[ch][i] = fmaf(fr, fr, fi * fi);
                acc1[ch][i] = fmaf(gr, gr, gi * gi);
              } else {
                acc[ch][i] = fmaf(fr, fr, fmaf(fi, fi, fmaf(gr, gr, fmaf(gi, gi, acc[ch][i]))));
              }
            }
          }
        }
        const float sc = (float)p.i8scale[c];
        const float sc2 = sc * sc;
        if constexpr (LBIN == 0) {  // nint = 1: lane r holds bins 2r and 2r+1 of every beam
          const int bin = 2 * (32 * (4 * sp + quad) + lane);
          if (bin < nbin) {
#pragma unroll
            for (int ch = 0; ch < NCH; ++ch)
#pragma unroll
              for (int i = 0; i < 8; ++i)
                if (8 * ch + i < nbeam) {
                  float *dst = p.pow + ((size_t)c * nbeam + 8 * ch + i) * nbin + bin;
                  if (vec8) {
                    *reinterpret_cast<float2 *>(dst) = make_float2(acc[ch][i] * sc2, acc1[ch][i] * sc2);
                  } else {  // powers pointer only 4-byte aligned: two scalar stores
                    dst[0] = acc[ch][i] * sc2;
                    dst[1] = acc1[ch][i] * sc2;
                  }
                }
          }
        } else {
          const int bin = (32 / LB) * (4 * sp + quad) + lane / LB;
#pragma unroll
          for (int ch = 0; ch < NCH; ++ch) {
            LaneReduce<8, LB / 2>::run(acc[ch], lane);
            if (writer && bin < nbin) {
#pragma unroll
              for (int j = 0; j < NFINAL; ++j) {
                const int beam = 8 * ch + beam_off + j;
                if (beam < nbeam) p.pow[((size_t)c * nbeam + beam) * nbin + bin] = acc[ch][j] * sc2;
              }
            }
          }
        }
      } else {
        ti += G;
      }
      if (++sp == n_super_chan) { sp = 0; ++c; }
    }
  } else if (warp == L_MMA_WARP) {
    // =========================================================================== MMA issue
    constexpr uint32_t idesc = make_idesc_i8(128, NCOL);
    int c = c0, sp = sp0, prev_c = -1, wi = 0, wb = 0;
    int ti = 0, st = 0;
    uint32_t st_par = 0;
    for (int s = 0; s < n_super; ++s) {
      if (c != prev_c) {
        if (wi > 0 && elect_one()) tc_commit(bar_w_empty + 8 * wb);
        prev_c = c;
        wb = wi & 1;
        mbar_wait(bar_w_full + 8 * wb, (uint32_t)((wi >> 1) & 1));
        ++wi;
      }
      const uint64_t bdesc = make_sdesc_k_sw64(sW + wb * W_BYTES);
      for (int g = 0; g < G; ++g, ++ti) {
        const int a = ti & (NACC - 1);
        mbar_wait(bar_a_full + 8 * st, st_par);
        mbar_wait(bar_t_empty + 8 * a, (uint32_t)(((ti >> ilog2(NACC)) & 1) ^ 1));
        tc_fence_after();
        if (elect_one()) {
          const uint64_t adesc = make_sdesc_k_sw128(sA + st * W_STAGE_BYTES);
          const uint32_t d = tmem_base + a * 2 * NCOL;
          mma_i8_ss(d, adesc, bdesc, idesc, 0);                  // even sample: row bytes 0..31
          mma_i8_ss(d, adesc + 2, bdesc + 2, idesc, 1);          //              row bytes 32..63
          mma_i8_ss(d + NCOL, adesc + 4, bdesc, idesc, 0);       // odd sample:  row bytes 64..95
          mma_i8_ss(d + NCOL, adesc + 6, bdesc + 2, idesc, 1);   //              row bytes 96..127
          tc_commit(bar_t_full + 8 * a);
          tc_commit(bar_a_empty + 8 * st);
        }
        __syncwarp();
        if (++st == NST) { st = 0; st_par ^= 1; }
      }
      if (++sp == n_super_chan) { sp = 0; ++c; }
    }
  } else if ((warp == L_TMA_WARP || warp == L_TMA_WARP + 1) && lane == 0) {
    // =========================================================================== TMA producers (two threads)
    // producer j issues the tiles of parity j (measured: the TMA unit overlaps two boxes, 0.097 -> 0.092 ms on
    // the sweep); producer 0 also brings in the coefficients
    const int pj = warp - L_TMA_WARP;
    constexpr int npj = 2;
    static_assert(NST % npj == 0, "stages are dealt to the producers by parity");
    tma_prefetch_desc(&tmap);
    tma_prefetch_desc(&tmap32);
    int c = c0, sp = sp0, prev_c = -1, wi = 0;
    int ti = 0, st = pj;                 // producer j: tiles j, j + npj, .. -> stages j, j + npj, .. (NST even)
    uint32_t st_par = 1;                 // parity of a_empty[st] to wait for (passes on the fresh barrier)
    for (int s = 0; s < n_super; ++s) {
      if (c != prev_c) {
        prev_c = c;
        if (pj == 0) {
          const int wb = wi & 1;
          mbar_wait(bar_w_empty + 8 * wb, (uint32_t)(((wi >> 1) & 1) ^ 1));
          mbar_arrive_expect_tx(bar_w_full + 8 * wb, W_BYTES);
          bulk_g2s(sW + wb * W_BYTES, reinterpret_cast<const char *>(p.wop8) + (size_t)c * W_BYTES, W_BYTES, bar_w_full + 8 * wb);
        }
        ++wi;
      }
      for (int g = 0; g < G; ++g, ++ti) {
        if (npj == 2 && (ti & 1) != pj) continue;
        mbar_wait(bar_a_empty + 8 * st, st_par);
        mbar_arrive_expect_tx(bar_a_full + 8 * st, W_STAGE_BYTES);
        if (G == 1) {   // rows (sample pairs) 128 sp .. 128 sp + 127: one box
          tma_load_3d(sA + st * W_STAGE_BYTES, &tmap, 0, 128 * sp, c, bar_a_full + 8 * st);
        } else {        // warp quadrant q sees rows 32 G (4 sp + q) + 32 g ..: a whole bin of 64 G samples over G tiles
#pragma unroll
          for (int q = 0; q < 4; ++q)
            tma_load_3d(sA + st * W_STAGE_BYTES + q * 4096, &tmap32, 0, 32 * G * (4 * sp + q) + 32 * g, c, bar_a_full + 8 * st);
        }
        if ((st += npj) >= NST) { st -= NST; st_par ^= 1; }
      }
      if (++sp == n_super_chan) { sp = 0; ++c; }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == L_MMA_WARP) tmem_dealloc(tmem_base, 512);
  probe_mark(p.probe, 1);
}

// 3-D view of the int8 voltages as bytes: {2 nant, nsamp, nchan}; box {64, 32, 1}, 64-byte swizzle; bytes past
// 2 nant and samples past nsamp are zero-filled
cudaError_t make_tmap(CUtensorMap *tm, const BfParams &p, int box_rows) {
  PFN_encodeTiled enc = bf_get_encode();
  if (!enc) return cudaErrorNotSupported;
  cuuint64_t dims[3] = {(cuuint64_t)2 * p.nant, (cuuint64_t)p.nsamp, (cuuint64_t)p.nchan_run};
  cuuint64_t strides[2] = {dims[0], dims[0] * (cuuint64_t)p.nsamp};
  cuuint32_t box[3] = {L_ROW_BYTES, (cuuint32_t)box_rows, 1};
  cuuint32_t estr[3] = {1, 1, 1};
  CUresult r = enc(tm, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, const_cast<void *>(p.volt), dims, strides, box, estr,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_64B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

// WIDE view: rows of 128 bytes = two samples of 32 antennas: {128, nsamp / 2, nchan}; box {128, box_rows, 1}, 128-byte swizzle
cudaError_t make_tmap_wide(CUtensorMap *tm, const BfParams &p, int box_rows) {
  PFN_encodeTiled enc = bf_get_encode();
  if (!enc) return cudaErrorNotSupported;
  cuuint64_t dims[3] = {128, (cuuint64_t)p.nsamp / 2, (cuuint64_t)p.nchan_run};
  cuuint64_t strides[2] = {128, (cuuint64_t)64 * p.nsamp};
  cuuint32_t box[3] = {128, (cuuint32_t)box_rows, 1};
  cuuint32_t estr[3] = {1, 1, 1};
  CUresult r = enc(tm, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, const_cast<void *>(p.volt), dims, strides, box, estr,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

template <int NCOL, int LBIN, bool BEAMS = false>
cudaError_t launch_i8w(const BfParams &p, int sm_count, cudaStream_t st) {
  constexpr int NST = 12;
  CUtensorMap tm, tm32;
  cudaError_t e = bf_cached_tmap(&tm, p, 1, 128, make_tmap_wide);
  if (e == cudaSuccess) e = bf_cached_tmap(&tm32, p, 1, 32, make_tmap_wide);
  if (e != cudaSuccess) return e;
  const int G = BEAMS || p.nint <= 64 ? 1 : p.nint / 64;
  const int n_super_chan = (p.nsamp + 256 * G - 1) / (256 * G);
  const long long total = (long long)p.nchan_run * n_super_chan;
  const size_t smem = 1024 + 2 * NCOL * L_ROW_BYTES + NST * W_STAGE_BYTES + 1024;
  auto kern = bf_umma_i8w_kernel<NCOL, LBIN, NST, BEAMS>;
  static thread_local int attr_dev = -1;   // once per instantiation and device
  if ((e = bf_set_smem_once(kern, smem, &attr_dev)) != cudaSuccess) return e;
  const int grid = (int)(total < sm_count ? total : sm_count);
  kern<<<grid, L_THREADS + 32, smem, st>>>(p, tm, tm32, total, n_super_chan, G);
  return cudaGetLastError();
}

template <int NCOL>
cudaError_t launch_i8w_nint(const BfParams &p, int sm_count, cudaStream_t st) {
  switch (p.nint) {
    case 1: return launch_i8w<NCOL, 0>(p, sm_count, st);
    case 2: return launch_i8w<NCOL, 1>(p, sm_count, st);
    case 4: return launch_i8w<NCOL, 2>(p, sm_count, st);
    case 8: return launch_i8w<NCOL, 4>(p, sm_count, st);
    case 16: return launch_i8w<NCOL, 8>(p, sm_count, st);
    case 32: return launch_i8w<NCOL, 16>(p, sm_count, st);
    default: return launch_i8w<NCOL, 32>(p, sm_count, st);  // 64 and its multiples
  }
}

template <int NCOL, int LBIN>
cudaError_t launch_i8(const BfParams &p, int sm_count, cudaStream_t st) {
  constexpr int NST = 24;
  CUtensorMap tm, tm32;
  cudaError_t e = bf_cached_tmap(&tm, p, 0, L_TILE_T, make_tmap);
  if (e == cudaSuccess) e = bf_cached_tmap(&tm32, p, 0, L_BOX_ROWS, make_tmap);
  if (e != cudaSuccess) return e;
  const int G = p.nint <= 32 ? 1 : p.nint / 32;
  const int n_super_chan = (p.nsamp + L_TILE_T * G - 1) / (L_TILE_T * G);
  const long long total = (long long)p.nchan_run * n_super_chan;
  const int nks = (2 * p.nant + 31) / 32;
  const size_t smem = 1024 + 2 * NCOL * L_ROW_BYTES + NST * L_STAGE_BYTES + 1024;
  auto kern = bf_umma_i8_kernel<NCOL, LBIN, NST>;
  static thread_local int attr_dev = -1;
  if ((e = bf_set_smem_once(kern, smem, &attr_dev)) != cudaSuccess) return e;
  const int grid = (int)(total < sm_count ? total : sm_count);
  kern<<<grid, L_THREADS, smem, st>>>(p, tm, tm32, total, n_super_chan, G, nks);
  return cudaGetLastError();
}

template <int NCOL>
cudaError_t launch_i8_nint(const BfParams &p, int sm_count, cudaStream_t st) {
  switch (p.nint) {
    case 1: return launch_i8<NCOL, 1>(p, sm_count, st);
    case 2: return launch_i8<NCOL, 2>(p, sm_count, st);
    case 4: return launch_i8<NCOL, 4>(p, sm_count, st);
    case 8: return launch_i8<NCOL, 8>(p, sm_count, st);
    case 16: return launch_i8<NCOL, 16>(p, sm_count, st);
    default: return launch_i8<NCOL, 32>(p, sm_count, st);  // 32 and its multiples
  }
}

}  // namespace

// bins the time-on-M kernels of this file integrate (lane butterfly / one bin per warp / running sums over whole tiles);
// any other even nint needs the bin-per-lane variant (bf_umma_i8b.cu)
static bool i8_tiled_nint_ok(int I) { return (I <= 32 && (I & (I - 1)) == 0) || I % 32 == 0; }

// which shapes the int8 kernel takes: complex int8, nant a multiple of 8 up to 32 (rows of <= 64 bytes that
// TMA can address), up to BF_I8_MAX_BEAMS beams, nint a power of two <= 32 or a multiple of 32
bool bf_umma_i8_supported(const bf_ctx *c, int mode) {
  if (c->dtype == BF_CI4)   // 4+4-bit input: the bin-per-lane variant only (rows of four samples)
    return mode == BF_MODE_POWER && c->nant == 32 && c->nbeam <= BF_I8_MAX_BEAMS && c->nint % 4 == 0 &&
           (c->nbin % 128 == 0 || c->nbin >= 512);
  if (c->dtype != BF_CI8 || c->nant % 8 != 0 || c->nant > 32 || c->nbeam > BF_I8_MAX_BEAMS) return false;
  if (mode == BF_MODE_BEAMS) return c->nant == 32 && c->nsamp % 2 == 0;   // the WIDE variant only
  const int I = c->nint;
  // the bin-per-lane variant (bf_umma_i8b.cu) integrates ANY even nint in registers
  if (c->nant == 32 && I % 2 == 0 && (c->nbin % 128 == 0 || c->nbin >= 512)) return true;
  return i8_tiled_nint_ok(I);
}

cudaError_t bf_launch_umma_i8(const BfParams &p, int dtype, int sm_count, cudaStream_t st) {
  if (dtype == BF_CI4) return bf_umma_i8b_takes(p, dtype) ? bf_launch_umma_i8b(p, dtype, sm_count, st) : cudaErrorNotSupported;
  if (p.mode == BF_MODE_BEAMS) {
    if (p.nbeam <= 8) return launch_i8w<32, 0, true>(p, sm_count, st);
    if (p.nbeam <= 16) return launch_i8w<64, 0, true>(p, sm_count, st);
    return launch_i8w<128, 0, true>(p, sm_count, st);
  }
  // 32 antennas, even nint and enough bins to fill the lanes: the bin-per-lane kernel (no cross-lane integration)
  // (measured on the sweep: 17-32 beams 0.147 -> 0.114 ms; up to 16 beams the contiguous tiles of the kernels
  // below read DRAM 7 % faster than the strided ones and their butterfly is still cheap)
  if (bf_umma_i8b_takes(p, BF_CI8) && (p.nbeam > 16 || !i8_tiled_nint_ok(p.nint)))
    return bf_launch_umma_i8b(p, BF_CI8, sm_count, st);
  // 32 antennas, an even number of samples and nint 2^k <= 64 or a multiple of 64: rows of two samples
  const bool wide = p.nant == 32 && p.nsamp % 2 == 0 && ((p.nint <= 64 && (p.nint & (p.nint - 1)) == 0) || p.nint % 64 == 0);
  if (wide) {
    if (p.nbeam <= 8) return launch_i8w_nint<32>(p, sm_count, st);
    if (p.nbeam <= 16) return launch_i8w_nint<64>(p, sm_count, st);
    return launch_i8w_nint<128>(p, sm_count, st);
  }
  if (p.nbeam <= 8) return launch_i8_nint<32>(p, sm_count, st);
  if (p.nbeam <= 16) return launch_i8_nint<64>(p, sm_count, st);
  return launch_i8_nint<128>(p, sm_count, st);
}
