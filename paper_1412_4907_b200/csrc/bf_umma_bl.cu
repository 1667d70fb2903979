// bf_umma_bl.cu -- the fused tensor-core beamformer for 33-64 beams on 32-antenna arrays (complex int8 input, nint even
// and >= 16): ONE OUTPUT BIN PER TMEM LANE and the converted voltages as the A operand IN TENSOR MEMORY (hot-path rows
// a2..a5).  This is the HBM-bound end of the fp16 path: at 64 beams bf_umma.cu issues 3472 instructions per 16 KiB of
// input (int8 -> fp16 through shared memory, an add tree, a shuffle and a store per bin and tile) and reaches 0.6 of the
// HBM roofline; the int8-operand kernels pay 2.5 instructions per real output and fall behind from 32 beams up.
//
//   a2 ingest      a raw tile is the TMA box {128 bytes, 1, 128 bins}: TWO samples of 128 consecutive bins (the strided
//                  tensor view of bf_umma_i8b.cu).  Convert thread r owns row r (= one bin): LDS.128 x 8 -> int8 -> fp16
//                  (exact, 0x6400 | (x ^ 0x80)) -> tcgen05.st: sample E and sample O become two A-operand tiles of 128
//                  rows x 64 fp16 = 32 TMEM columns each.  The fp16 voltages never touch shared memory.
//   a3 contraction tcgen05.mma kind::f16, A = voltages from TMEM (M = 128 bins), B = the coefficient tile from shared
//                  memory (N = 128 rows = 64 beams re + im: the SAME swizzled image bf_umma.cu uses as its A operand),
//                  K = 64: D[bin][row] = sum_k' X'[bin][k'] W[row][k'], fp32 in TMEM; three accumulator
//                  stages of 128 columns + four operand stages of 32 columns = the 512 TMEM columns.
//   a4 + a5        lane r of EVERY accumulator of a super-tile belongs to bin r, so detection and integration
//                   are one running sum per beam in the registers of the thread that owns the lane:
//                  columns (2j, 2j+1) hold re of beams (2j, 2j+1) and columns 16 + (2j, 2j+1) their im, so two FFMA2 add
//                  re^2 and im^2 of two beams into one float2 -- no add tree, no shuffle, one coalesced store per beam at
//                  the END of the super-tile.
//
// Work item = (channel, PAIR of super-tiles X, Y of 128 bins each); their raw tiles are interleaved (X.g, Y.g, X.g+1, ..),
// their accumulators alternate (X.E, Y.E, X.O, Y.O), and the two epilogue sets (eight warps each: TMEM lane quadrant x 64-column half) take the accumulators of X and of Y:
// a visit costs a warp ~500 clk of latency whatever it does (barrier wait, tcgen05.ld, arrive; measured with an event
// trace on a first form of this kernel in which every warp visited every accumulator), so each warp must see only every
// other accumulator -- and with X and Y on different bins the sets share nothing.  A persistent CTA per SM walks a
// contiguous range of items; the coefficient tile of a channel stays resident.  Warp roles: 0-15
// epilogue, 16-19 convert (one per quadrant), 20-21 MMA issue (accumulators of even / odd index), 22 TMA producer.
#include <cuda.h>

#include "bf_tmap.h"
#include "bf_umma_common.cuh"

namespace {

using namespace bfk;

constexpr int BL_ND = 3, BL_NA = 4;                    // accumulator stages (128 columns), A-operand stages (32 columns)
constexpr int BL_DCOLS = 128, BL_ACOLS = 32;
constexpr int BL_A_COL0 = BL_ND * BL_DCOLS;            // 384
constexpr int BL_RAW_BYTES = 128 * 128;                // 16 KiB: 128 bins x two samples x 32 antennas x (re, im)
constexpr int BL_EPI_WARPS = 16, BL_MMA_WARP0 = 20, BL_TMA_WARP = 22;
constexpr int BL_THREADS = 23 * 32;

// NRAW: raw stages.  IN: BF_CI8 (raw rows of 128 bytes = two samples) or BF_CI4 (the paper's 4+4-bit bytes, PAPER.md:102:
// raw rows of 64 bytes = two samples, 64-byte swizzle).  n_items = channels x super-tile pairs per channel (nSP2).
template <int NRAW, int IN>
__global__ void __launch_bounds__(BL_THREADS, 1)
bf_umma_bl_kernel(const BfParams p, const __grid_constant__ CUtensorMap tmap, const long long total_items, const int nSP2,
                  const int G) {
  extern __shared__ uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t sW = smem_base;                                  // 2 coefficient buffers (one tile = 64 beams each)
  const uint32_t sR = sW + 2 * A_TILE_BYTES;                      // NRAW raw stages
  constexpr int RAW_BYTES = IN == BF_CI4 ? BL_RAW_BYTES / 2 : BL_RAW_BYTES;
  const uint32_t sBar = sR + NRAW * BL_RAW_BYTES;
  const uint32_t bar_r_full = sBar, bar_r_empty = bar_r_full + 8 * NRAW;
  const uint32_t bar_a_full = bar_r_empty + 8 * NRAW, bar_a_empty = bar_a_full + 8 * BL_NA;
  // accumulator barriers per (epilogue set, stage): a waiter must see EVERY phase of a barrier it waits on (a parity
  // wait cannot tell phase n from phase n + 2), and a set visits only every other use of a stage
  const uint32_t bar_d_full = bar_a_empty + 8 * BL_NA, bar_d_empty = bar_d_full + 8 * 2 * BL_ND;
  const uint32_t bar_w_full = bar_d_empty + 8 * 2 * BL_ND, bar_w_empty = bar_w_full + 16;
  const uint32_t s_tmem = bar_w_empty + 16;

  const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0), lane = threadIdx.x & 31;

  if (threadIdx.x == 0) {
    for (int s = 0; s < NRAW; ++s) { mbar_init(bar_r_full + 8 * s, 1); mbar_init(bar_r_empty + 8 * s, 4); }
    for (int s = 0; s < BL_NA; ++s) { mbar_init(bar_a_full + 8 * s, 4); mbar_init(bar_a_empty + 8 * s, 1); }
    for (int s = 0; s < 2 * BL_ND; ++s) { mbar_init(bar_d_full + 8 * s, 1); mbar_init(bar_d_empty + 8 * s, BL_EPI_WARPS / 2); }
    for (int s = 0; s < 2; ++s) { mbar_init(bar_w_full + 8 * s, 1); mbar_init(bar_w_empty + 8 * s, 2); }
    fence_barrier_init();
  }
  if (warp == BL_MMA_WARP0) tmem_alloc(s_tmem, 512);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(s_tmem));
  tmem_base = __shfl_sync(0xffffffffu, tmem_base, 0);
  probe_mark(p.probe, 0);

  const long long it0 = total_items * blockIdx.x / gridDim.x;
  const long long it1 = total_items * (blockIdx.x + 1) / gridDim.x;
  const int n_items = (int)(it1 - it0);
  const int c0 = (int)(it0 / nSP2), q0 = (int)(it0 % nSP2);
  const int n_acc = 4 * G;                                         // accumulators per item: per g X.E, Y.E, X.O, Y.O

  if (warp < BL_EPI_WARPS) {
    // =========================================================================== epilogue (2 sets of 8 warps)
    const int quad = warp & 3, half = (warp >> 2) & 1, iset = warp >> 3;   // set 0: super-tile X, set 1: Y
    const bool lane0 = lane == 0;
    uint32_t t_lane = tmem_base + ((uint32_t)(quad * 32) << 16) + half * 64;
    uint32_t bfull = bar_d_full + 8 * BL_ND * iset;              // my set's "full" barriers; its "empty" ones are 6 on
    asm volatile("" : "+r"(t_lane), "+r"(bfull));                // keep in registers, do not rematerialise
    const int nbeam = p.nbeam, nbin = p.nbin;
    int c = c0, q = q0;
    uint32_t dpar = 0;                                           // bit s: parity of the next completion of MY d_full[s]
    int ds = 0;                                                  // accumulator kk of the CTA uses stage kk % 3, set kk & 1
    for (int n = 0; n < n_items; ++n) {
      const int sp = 2 * q + iset;                               // my super-tile of the pair
      const bool live = 128 * sp + 32 * quad < nbin;             // warp-uniform: this quadrant holds real bins
      float2 acc[2][8];                                          // 64 columns = beams 32 half .. 32 half + 31
#pragma unroll
      for (int g = 0; g < 2; ++g)
#pragma unroll
        for (int i = 0; i < 8; ++i) acc[g][i] = make_float2(0.f, 0.f);
      for (int k = 0; k < n_acc; ++k) {                          // n_acc is even: k & 1 == kk & 1
        if ((k & 1) == iset) {
          const uint32_t bf_s = bfull + 8 * ds;
          mbar_wait_tight(bf_s, (dpar >> ds) & 1);
          dpar ^= 1u << ds;
          tc_fence_after();
          if (live) {
            const uint32_t t_acc = t_lane + ds * BL_DCOLS;
#pragma unroll
            for (int g = 0; g < 2; ++g) {                        // two 32-column chunks = 16 beams each
              uint32_t v[32];
              BF_TMEM_LD_32x32b_X32(t_acc + 32 * g, v);
              tc_wait_ld();
              if (g == 1) {                                      // all of this warp's columns are in registers
                tc_fence_before();
                __syncwarp();
                if (lane0) mbar_arrive(bf_s + 8 * 2 * BL_ND);
              }
#pragma unroll
              for (int i = 0; i < 8; ++i) {                      // re of beams (2i, 2i+1), then their im
                const float2 re = make_float2(__uint_as_float(v[2 * i]), __uint_as_float(v[2 * i + 1]));
                const float2 im = make_float2(__uint_as_float(v[16 + 2 * i]), __uint_as_float(v[16 + 2 * i + 1]));
                acc[g][i] = ffma2(re, re, acc[g][i]);
                acc[g][i] = ffma2(im, im, acc[g][i]);
              }
            }
          } else {
            __syncwarp();
            if (lane0) mbar_arrive(bf_s + 8 * 2 * BL_ND);
          }
        }
        if (++ds == BL_ND) ds = 0;
      }
      const int bin = 128 * sp + 32 * quad + lane;
      if (live && bin < nbin) {
#pragma unroll
        for (int g = 0; g < 2; ++g) {
          const int beam0 = 32 * half + 16 * g;
          float *out = p.pow + ((size_t)c * nbeam + beam0) * nbin + bin;
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            if (beam0 + 2 * i < nbeam) out[(size_t)(2 * i) * nbin] = acc[g][i].x;
            if (beam0 + 2 * i + 1 < nbeam) out[(size_t)(2 * i + 1) * nbin] = acc[g][i].y;
          }
        }
      }
      if (++q == nSP2) { q = 0; ++c; }
    }
  } else if (warp < BL_MMA_WARP0) {
    // =========================================================================== convert (4 warps, one per quadrant)
    // thread (quad, lane) owns row r = 32 quad + lane of every raw tile: 128 bytes = samples E and O of one bin; the raw
    // tiles of X go to operand stages 0, 1, those of Y to stages 2, 3 (a second group of four warps on alternate raw
    // tiles was measured: 0.152 instead of 0.147 ms at 64 beams)
    const int quad = warp & 3;
    const int r = 32 * quad + lane;
    const uint32_t t_row = tmem_base + ((uint32_t)(quad * 32) << 16) + BL_A_COL0;
    const uint32_t row_off = IN == BF_CI4 ? (uint32_t)r * 64u : (uint32_t)r * 128u;
    const uint32_t sw = IN == BF_CI4 ? (uint32_t)((r >> 1) & 3) : (uint32_t)(r & 7);   // 64- / 128-byte swizzle of the TMA box
    int rs = 0, as = 0;
    uint32_t rpar = 0, apar = 1;
    const int n_raw = n_items * 2 * G;
    for (int i = 0; i < n_raw; ++i) {
      mbar_wait(bar_r_full + 8 * rs, rpar);
      const uint32_t src = sR + rs * BL_RAW_BYTES + row_off;
      constexpr int NX = IN == BF_CI4 ? 4 : 8;                     // 16-byte pieces per raw row
      uint4 x[NX];
#pragma unroll
      for (int j = 0; j < NX; ++j) x[j] = ld_shared_v4(src + ((j ^ sw) << 4));
#pragma unroll
      for (int h = 0; h < 2; ++h) {                                // sample E, sample O
        uint32_t o[32];
        if constexpr (IN == BF_CI4) {                              // 32 bytes = 32 antennas -> 32 half2 (re, im), exact
#pragma unroll
          for (int j = 0; j < 2; ++j) {
            const uint4 w = x[2 * h + j];
            uint32_t t[4];
            cvt_i4x8_f16x8(w.x, t); o[16 * j + 0] = t[0]; o[16 * j + 1] = t[1]; o[16 * j + 2] = t[2]; o[16 * j + 3] = t[3];
            cvt_i4x8_f16x8(w.y, t); o[16 * j + 4] = t[0]; o[16 * j + 5] = t[1]; o[16 * j + 6] = t[2]; o[16 * j + 7] = t[3];
            cvt_i4x8_f16x8(w.z, t); o[16 * j + 8] = t[0]; o[16 * j + 9] = t[1]; o[16 * j + 10] = t[2]; o[16 * j + 11] = t[3];
            cvt_i4x8_f16x8(w.w, t); o[16 * j + 12] = t[0]; o[16 * j + 13] = t[1]; o[16 * j + 14] = t[2]; o[16 * j + 15] = t[3];
          }
        } else {
#pragma unroll
          for (int j = 0; j < 4; ++j) {
            const uint4 w = x[4 * h + j];
            cvt_i8x4_f16x4(w.x, o[8 * j + 0], o[8 * j + 1]);
            cvt_i8x4_f16x4(w.y, o[8 * j + 2], o[8 * j + 3]);
            cvt_i8x4_f16x4(w.z, o[8 * j + 4], o[8 * j + 5]);
            cvt_i8x4_f16x4(w.w, o[8 * j + 6], o[8 * j + 7]);
          }
        }
        if (h == 1) {  // the raw row is in registers (both halves consumed): the stage may be refilled
          __syncwarp();
          if (lane == 0) mbar_arrive(bar_r_empty + 8 * rs);
        }
        mbar_wait(bar_a_empty + 8 * (as + h), apar);
        tc_fence_after();
        BF_TMEM_ST_32x32b_X32(t_row + (as + h) * BL_ACOLS, o);
      }
      tc_wait_st();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) {
        mbar_arrive(bar_a_full + 8 * as);
        mbar_arrive(bar_a_full + 8 * (as + 1));
      }
      if (++rs == NRAW) { rs = 0; rpar ^= 1; }
      if ((as += 2) == BL_NA) { as = 0; apar ^= 1; }
    }
  } else if (warp < BL_TMA_WARP) {
    // =========================================================================== MMA issue (2 warps)
    // accumulator kk of the CTA goes to stage kk % 3; per g the order is X.E, Y.E, X.O, Y.O (operand stages 0, 2, 1, 3), so
    // that the accumulators alternate between the two epilogue sets; warp m issues the accumulators with k & 1 == m, i.e.
    // one MMA warp feeds one epilogue set (tcgen05.mma issue is nearly blocking: see bf_umma.cu)
    const int id = warp - BL_MMA_WARP0;
    constexpr uint32_t idesc = make_idesc_f16(128, BL_DCOLS);
    constexpr uint32_t dhi = sdesc_k_sw128_hi();
    const uint32_t b_lo0 = sdesc_k_sw128_lo(sW);
    int c = c0, q = q0, prev_c = -1;
    int wg = 0, wb = 0;
    uint32_t apar = 0;                  // parity of a_full[*] to wait for: all four operand stages turn over once per g
    // Stage s is reused three accumulators later, i.e. after the OTHER set has read it: warp m waits on the other set's
    // "empty" barriers, each of them every sixth accumulator.  Bit s = parity to wait for next; the first user of a stage
    // (accumulators 0, 1, 2 -> warps 0, 1, 0) passes on the fresh barrier (parity 1).
    const uint32_t d_full_m = bar_d_full + 8 * BL_ND * id, d_empty_o = bar_d_empty + 8 * BL_ND * (1 - id);
    uint32_t dpar = id == 0 ? 5u : 2u;
    int ds = 0;
    for (int n = 0; n < n_items; ++n) {
      if (c != prev_c) {
        if (wg > 0 && elect_one()) tc_commit(bar_w_empty + 8 * wb);   // my MMAs so far have left the old buffer
        prev_c = c;
        wb = wg & 1;
        mbar_wait(bar_w_full + 8 * wb, (uint32_t)((wg >> 1) & 1));
        ++wg;
      }
      const uint32_t b_lo = b_lo0 + wb * (A_TILE_BYTES >> 4);
      for (int k = 0; k < n_acc; ++k) {
        const int as = ((k & 1) << 1) | ((k >> 1) & 1);   // X.E, Y.E, X.O, Y.O -> operand stages 0, 2, 1, 3
        if ((k & 1) == id) {
          mbar_wait(bar_a_full + 8 * as, apar);
          mbar_wait(d_empty_o + 8 * ds, (dpar >> ds) & 1);
          dpar ^= 1u << ds;
          tc_fence_after();
          if (elect_one()) {
            const uint32_t d = tmem_base + ds * BL_DCOLS;
            const uint32_t a = tmem_base + BL_A_COL0 + as * BL_ACOLS;
#pragma unroll
            for (int kk = 0; kk < 4; ++kk) {   // 16 fp16 along K: 8 TMEM columns of A, 32 bytes inside B's swizzle atom
              const uint64_t bdesc = ((uint64_t)dhi << 32) | (uint64_t)(b_lo + 2 * kk);
              mma_f16_ts(d, a + 8 * kk, bdesc, idesc, kk > 0);
            }
            tc_commit(d_full_m + 8 * ds);
            tc_commit(bar_a_empty + 8 * as);    // the A tile may be overwritten once these MMAs have read it
          }
          __syncwarp();
        }
        if (++ds == BL_ND) ds = 0;
        if ((k & 3) == 3) apar ^= 1;
      }
      if (++q == nSP2) { q = 0; ++c; }
    }
  } else if (warp == BL_TMA_WARP && lane == 0) {
    // =========================================================================== TMA producer (one thread)
    tma_prefetch_desc(&tmap);
    int c = c0, q = q0, prev_c = -1;
    int wg = 0;
    int rs = 0;
    uint32_t rpar = 1;
    for (int n = 0; n < n_items; ++n) {
      if (c != prev_c) {
        prev_c = c;
        const int wb = wg & 1;
        mbar_wait(bar_w_empty + 8 * wb, (uint32_t)(((wg >> 1) & 1) ^ 1));
        const char *wsrc = reinterpret_cast<const char *>(p.wop) + (size_t)c * p.nMt * A_TILE_BYTES;
        mbar_arrive_expect_tx(bar_w_full + 8 * wb, A_TILE_BYTES);
        bulk_g2s(sW + wb * A_TILE_BYTES, wsrc, A_TILE_BYTES, bar_w_full + 8 * wb);
        ++wg;
      }
      for (int g = 0; g < G; ++g) {
#pragma unroll
        for (int h = 0; h < 2; ++h) {   // row g of super-tile X, then of Y (bins past nbin are zero-filled)
          mbar_wait(bar_r_empty + 8 * rs, rpar);
          mbar_arrive_expect_tx(bar_r_full + 8 * rs, RAW_BYTES);
          tma_load_5d(sR + rs * BL_RAW_BYTES, &tmap, 0, 0, 128 * (2 * q + h), g, c, bar_r_full + 8 * rs);
          if (++rs == NRAW) { rs = 0; rpar ^= 1; }
        }
      }
      if (++q == nSP2) { q = 0; ++c; }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == BL_MMA_WARP0) tmem_dealloc(tmem_base, 512);
  probe_mark(p.probe, 1);
}

// 5-D view of one launch's voltages: {byte in row, 1, bin, row in bin, channel}, a row = two samples (128 bytes of int8,
// 64 bytes of 4+4-bit); box {row, 1, 128, 1, 1}: row g of 128 consecutive bins; bins past nbin are zero-filled
template <int IN>
cudaError_t bl_make_tmap(CUtensorMap *tm, const BfParams &p, int nint) {
  PFN_encodeTiled enc = bf_get_encode();
  if (!enc) return cudaErrorNotSupported;
  constexpr cuuint32_t ROW = IN == BF_CI4 ? 64 : 128;
  cuuint64_t dims[5] = {ROW, 1, (cuuint64_t)p.nbin, (cuuint64_t)(nint / 2), (cuuint64_t)p.nchan_run};
  cuuint64_t strides[4] = {ROW, (cuuint64_t)nint * (ROW / 2), ROW, (cuuint64_t)p.nsamp * (ROW / 2)};
  cuuint32_t box[5] = {ROW, 1, 128, 1, 1};
  cuuint32_t estr[5] = {1, 1, 1, 1, 1};
  CUresult r = enc(tm, CU_TENSOR_MAP_DATA_TYPE_UINT8, 5, const_cast<void *>(p.volt), dims, strides, box, estr,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, IN == BF_CI4 ? CU_TENSOR_MAP_SWIZZLE_64B : CU_TENSOR_MAP_SWIZZLE_128B,
                   CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

template <int IN>
cudaError_t launch_bl(const BfParams &p, int sm_count, cudaStream_t st) {
  constexpr int NRAW = 11;
  CUtensorMap tm;
  cudaError_t e = bf_cached_tmap(&tm, p, IN == BF_CI4 ? 31 : 30, p.nint, bl_make_tmap<IN>);
  if (e != cudaSuccess) return e;
  const int nSP2 = (p.nbin + 255) / 256;
  const long long total = (long long)p.nchan_run * nSP2;
  const size_t smem = 1024 + 2 * A_TILE_BYTES + (size_t)NRAW * BL_RAW_BYTES + 512;
  auto kern = bf_umma_bl_kernel<NRAW, IN>;
  static thread_local int attr_dev = -1;
  if ((e = bf_set_smem_once(kern, smem, &attr_dev)) != cudaSuccess) return e;
  const int grid = (int)(total < sm_count ? total : sm_count);
  kern<<<grid, BL_THREADS, smem, st>>>(p, tm, total, nSP2, p.nint / 2);
  return cudaGetLastError();
}

}  // namespace

// Shapes this kernel takes: bf_bl_shape (bf_internal.h) -- the one predicate the dispatcher, bf_kernel_name and
// bf_umma_supported share -- on a launch without the residual coefficient plane
bool bf_umma_bl_takes(const BfParams &p, int dtype) {
  return p.wop_lo == nullptr && bf_bl_shape(dtype, p.mode, p.nant, p.nbeam, p.nint, p.nbin);
}

cudaError_t bf_launch_umma_bl(const BfParams &p, int dtype, int sm_count, cudaStream_t st) {
  return dtype == BF_CI4 ? launch_bl<BF_CI4>(p, sm_count, st) : launch_bl<BF_CI8>(p, sm_count, st);
}
