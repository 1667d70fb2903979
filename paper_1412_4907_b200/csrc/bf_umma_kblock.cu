// bf_umma_kblock.cu -- the fused tensor-core beamformer for larger arrays (any nant that is a multiple
// of 8 (int8) / 4 (fp16)): hot-path rows a2..a5 with the contraction K-blocked.
//
// Per channel the contraction is a real GEMM  D[2B rows][T] = A[2B][K'] X'[T][K']^T, K' = 2*nant
// (the (re, -im)/(im, re) row expansion is described in bf_internal.h).  Neither operand
// fits in shared memory any more, so both stream in K-blocks of 64:
//   * coefficient tiles (128 rows x 64, pre-swizzled in HBM) by cp.async.bulk, two M-tiles (128 beams)
//     per stage -- every voltage K-block is used for both before it is released;
//   * voltage K-blocks (256 samples x 64) by a 3-D TMA tensor copy: fp16 input lands directly in the
//     128-byte-swizzled operand layout; int8 input lands raw and the convert warps rewrite it as fp16
//     (the paper's in-kernel unpack).
// The two accumulators (2 x 256 TMEM columns) are drained by the same fused |.|^2 + integrate
// epilogue as the small-array kernel once the last K-block has been issued.
//
// Work item = (channel, time tile, beam-group of 128 beams), beam group fastest.  Items are dealt
// round-robin to the persistent CTAs (item j -> CTA j mod grid), so at any moment the 148 CTAs work on
// ~148 consecutive items = one or two channels: that channel's coefficients and voltages stay in the
// 126 MB L2 while every CTA that needs them passes by (with contiguous ranges per CTA all channels
// would be live at once and DRAM traffic was 3-14x the algorithmic bytes).
#include <cuda.h>

#include "bf_tmap.h"
#include "bf_umma_common.cuh"

namespace {

using namespace bfk;

constexpr int KB_GROUP = 2;                        // M-tiles (of 64 beams) per item
constexpr int CONV_WARPS = 8;
constexpr int CONV_THREADS = CONV_WARPS * 32;
constexpr int MMA_WARP = EPI_WARPS + CONV_WARPS;
constexpr int TMA_WARP = MMA_WARP + 2;  // two MMA-issuing warps, one per accumulator
constexpr int NTHREADS = (EPI_WARPS + CONV_WARPS + 4) * 32;   // + 2 MMA warps + 2 producer warps
template <bool LO> constexpr int a_stage_bytes_v = (LO ? 2 : 1) * KB_GROUP * A_TILE_BYTES;   // [hi tiles][lo tiles]

struct KItem { int c, tt, g; };
__device__ __forceinline__ KItem kdecode(long long idx, int nG, int nTt) {
  KItem it;
  it.g = (int)(idx % nG);
  long long ct = idx / nG;
  it.tt = (int)(ct % nTt);
  it.c = (int)(ct / nTt);
  return it;
}

// LO: two-term coefficients (bf_internal.h, BF_LO_NINT): a coefficient stage holds the "hi" tiles followed by the "lo"
// tiles of the K-block and every voltage K-block is contracted against both.
// IN: BF_CI8 / BF_CF16 / BF_CI4 (the paper's 4+4-bit bytes: a K-block of 32 antennas is 32 raw bytes per
// sample, unpacked by the convert warps).
template <int NINT_T, int IN, int NA, int NB, int NR, bool BEAMS, bool LO>
__global__ void __launch_bounds__(NTHREADS, 1)
bf_umma_kblock_kernel(const BfParams p, const __grid_constant__ CUtensorMap tmap, const long long total_items,
                      const int nG, const int nTt) {
  extern __shared__ uint8_t smem_raw[];
  constexpr bool IS_F16 = IN == BF_CF16, IS_CI4 = IN == BF_CI4;
  constexpr int A_STAGE_BYTES = a_stage_bytes_v<LO>;
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t sA = smem_base;                              // NA stages x 2 (x 2) coefficient tiles
  const uint32_t sB = sA + NA * A_STAGE_BYTES;                // NB fp16 operand stages
  const uint32_t sR = sB + NB * B_STAGE_BYTES;                // NR raw int8 stages (int8 input only)
  const uint32_t sBar = sR + NR * RAW_STAGE_BYTES;
  const uint32_t bar_a_full = sBar, bar_a_empty = bar_a_full + 8 * NA;
  const uint32_t bar_b_full = bar_a_empty + 8 * NA, bar_b_empty = bar_b_full + 8 * NB;
  const uint32_t bar_r_full = bar_b_empty + 8 * NB, bar_r_empty = bar_r_full + 8 * (NR + 1);
  const uint32_t bar_t_full = bar_r_empty + 8 * (NR + 1), bar_t_empty = bar_t_full + 16;
  const uint32_t s_tmem = bar_t_empty + 16;

  const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0), lane = threadIdx.x & 31;

  if (threadIdx.x == 0) {
    for (int s = 0; s < NA; ++s) { mbar_init(bar_a_full + 8 * s, 1); mbar_init(bar_a_empty + 8 * s, 2); }
    for (int s = 0; s < NB; ++s) { mbar_init(bar_b_full + 8 * s, IS_F16 ? 1 : CONV_WARPS); mbar_init(bar_b_empty + 8 * s, 2); }
    for (int s = 0; s < NR; ++s) { mbar_init(bar_r_full + 8 * s, 1); mbar_init(bar_r_empty + 8 * s, CONV_WARPS); }
    for (int s = 0; s < 2; ++s) { mbar_init(bar_t_full + 8 * s, 1); mbar_init(bar_t_empty + 8 * s, EPI_WARPS); }
    fence_barrier_init();
  }
  if (warp == MMA_WARP) tmem_alloc(s_tmem, 512);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(s_tmem));
  tmem_base = __shfl_sync(0xffffffffu, tmem_base, 0);
  probe_mark(p.probe, 0);

  const long long it0 = blockIdx.x, it_step = gridDim.x;  // round-robin item assignment
  const int n_items = (int)((total_items - it0 + it_step - 1) / it_step);
  const int nMt = p.nMt, nKb = p.nKb;

  if (warp < EPI_WARPS) {
    // =========================================================================== epilogue
    constexpr int BPW = NINT_T == 0 ? 1 : 64 / NINT_T;       // bins per warp and tile
    constexpr int BPT = NINT_T == 0 ? 0 : TILE_T / NINT_T;   // bins per tile
    const int quad = warp & 3, slot = warp >> 2;
    const bool lane0 = lane == 0;
    const uint32_t t_lane = tmem_base + ((uint32_t)(quad * 32) << 16) + slot * 64;
    const int bl = quad * 16 + (lane & 15);
    const bool vec_ok = (p.nbin % 4 == 0) && ((reinterpret_cast<uintptr_t>(p.pow) & 15) == 0);
    const bool bvec_ok = BEAMS && (p.nsamp % 4 == 0) && ((reinterpret_cast<uintptr_t>(p.beams) & 15) == 0);
    uint32_t tpar = 0;  // bit m: parity of the next completion of t_full[m] (an odd last group skips m = 1)
    for (int i = 0; i < n_items; ++i) {
      const KItem it = kdecode(it0 + i * it_step, nG, nTt);
      const int gm = min(KB_GROUP, nMt - it.g * KB_GROUP);
      const int t_first = it.tt * TILE_T + slot * 64;
      for (int m = 0; m < gm; ++m) {
        mbar_wait_backoff(bar_t_full + 8 * m, (tpar >> m) & 1, 128);   // a K loop away: do not spin
        tpar ^= 1u << m;
        tc_fence_after();
        const int beam = (it.g * KB_GROUP + m) * BF_TILE_BEAMS + bl;
        if (beam - (lane & 15) >= p.nbeam) { epilogue_skip(bar_t_empty + 8 * m, lane0); continue; }
        const bool writer = (lane < 16) && (beam < p.nbeam);
        if constexpr (BEAMS) {  // voltage-beam mode (row f4): y itself, fp16 (re, im)
          __half2 *yrow = reinterpret_cast<__half2 *>(p.beams) + ((size_t)it.c * p.nbeam + beam) * p.nsamp + t_first;
          epilogue_beams_tile(t_lane + m * TILE_T, yrow, beam < p.nbeam, p.nsamp - t_first, bvec_ok, p.beam_scale,
                              lane >= 16, bar_t_empty + 8 * m, lane0);
          continue;
        }
        float *row = p.pow + ((size_t)it.c * p.nbeam + beam) * p.nbin;
        if (NINT_T == 0 && p.nint % 64 != 0) {   // any bin length >= 16 that is no power of two <= 64 and no multiple of 64
          epilogue_tile_anynint(t_lane + m * TILE_T, row, writer, t_first, p.nint, p.nbin, bar_t_empty + 8 * m, lane0);
        } else if (NINT_T == 0) {
          epilogue_tile<NINT_T>(t_lane + m * TILE_T, row + t_first / p.nint, writer, t_first < p.nsamp ? 1 : 0, false,
                                bar_t_empty + 8 * m, lane0);
        } else {
          const int bin0 = it.tt * BPT + slot * BPW;
          epilogue_tile<NINT_T>(t_lane + m * TILE_T, row + bin0, writer, p.nbin - bin0, vec_ok, bar_t_empty + 8 * m, lane0);
        }
      }
    }
  } else if (warp < MMA_WARP) {
    // =========================================================================== convert (int8 input only)
    if (!IS_F16) {
      // 16-byte input pieces per K-block: int8 rows are 64 bytes (4 pieces, 2 output chunks each), 4-bit rows 32 bytes
      // (2 pieces of 16 antennas, 4 output chunks each)
      constexpr int PPR = IS_CI4 ? 2 : 4, CPP = IS_CI4 ? 4 : 2;
      constexpr int PIECES = (TILE_T * PPR) / CONV_THREADS;
      const int ctid = threadIdx.x - EPI_WARPS * 32;
      uint32_t p_dst[PIECES];
#pragma unroll
      for (int k = 0; k < PIECES; ++k) {
        const int pc = ctid + k * CONV_THREADS;
        const int t = pc / PPR, q = pc % PPR;
        p_dst[k] = (uint32_t)((t >> 3) * 1024 + (t & 7) * 128 + (((CPP * q) ^ (t & 7)) << 4));
      }
      const long long nblk = (long long)n_items * nKb;
      int rs = 0, bs = 0;
      uint32_t rpar = 0, bpar = 1;
      for (long long j = 0; j < nblk; ++j) {
        mbar_wait(bar_r_full + 8 * rs, rpar);
        uint4 x[PIECES];
        convert_load<PIECES, CONV_THREADS>(sR + rs * RAW_STAGE_BYTES, ctid, p_dst, x);
        mbar_wait(bar_b_empty + 8 * bs, bpar);
        if constexpr (IS_CI4) convert_store_ci4<PIECES>(sB + bs * B_STAGE_BYTES, p_dst, x);
        else convert_store<PIECES>(sB + bs * B_STAGE_BYTES, p_dst, x);
        fence_proxy_async_smem();
        __syncwarp();
        if (lane == 0) {
          mbar_arrive(bar_r_empty + 8 * rs);
          mbar_arrive(bar_b_full + 8 * bs);
        }
        if (++rs == NR) { rs = 0; rpar ^= 1; }
        if (++bs == NB) { bs = 0; bpar ^= 1; }
      }
    }
  } else if (warp < TMA_WARP) {
    // =========================================================================== MMA issue (2 warps)
    // One issuing warp per accumulator (tcgen05.mma issue is nearly blocking, see bf_umma.cu): warp id
    // feeds accumulator id = M-tile id of the item's beam group, for every K-block.
    const int id = warp - MMA_WARP;
    constexpr uint32_t idesc = make_idesc_f16(BF_TILE_ROWS, TILE_T);
    const uint64_t adesc0 = make_sdesc_k_sw128(sA + id * A_TILE_BYTES);
    const uint64_t bdesc0 = make_sdesc_k_sw128(sB);
    const uint32_t d = tmem_base + id * TILE_T;
    int sa = 0, sb = 0;
    uint32_t apar = 0, bpar = 0, tpar = 1;
    for (int i = 0; i < n_items; ++i) {
      const KItem it = kdecode(it0 + i * it_step, nG, nTt);
      const int gm = min(KB_GROUP, nMt - it.g * KB_GROUP);
      const bool mine = id < gm;  // an odd last group has no second M-tile
      if (mine) { mbar_wait(bar_t_empty + 8 * id, tpar); tpar ^= 1; tc_fence_after(); }
      for (int kb = 0; kb < nKb; ++kb) {
        // Both warps take part in the hand-shake of EVERY K-block, also the warp without a tile in this item (an odd last
        // beam group): it waits for "full" and gives its own arrival to "empty".  A parity wait cannot tell completion n
        // from n + 2: a warp that skipped the barriers of a whole item would find those of its next own item satisfied by
        // an old phase, and a warp the other one arrived for could fall two completions behind and wait for ever (bf_umma.cu).
        mbar_wait(bar_a_full + 8 * sa, apar);
        mbar_wait(bar_b_full + 8 * sb, bpar);
        if (!mine && elect_one()) { mbar_arrive(bar_a_empty + 8 * sa); mbar_arrive(bar_b_empty + 8 * sb); }
        if (mine) {
          tc_fence_after();
          if (elect_one()) {
            const uint64_t bdesc = bdesc0 + (uint64_t)(sb * (B_STAGE_BYTES >> 4));
            const uint64_t adesc = adesc0 + (uint64_t)(sa * (A_STAGE_BYTES >> 4));
#pragma unroll
            for (int k = 0; k < 4; ++k) mma_f16_ss(d, adesc + 2 * k, bdesc + 2 * k, idesc, (kb | k) != 0);
            if constexpr (LO) {   // the residual term of the coefficients against the same voltage K-block
              const uint64_t ldesc = adesc + (uint64_t)(KB_GROUP * (A_TILE_BYTES >> 4));
#pragma unroll
              for (int k = 0; k < 4; ++k) mma_f16_ss(d, ldesc + 2 * k, bdesc + 2 * k, idesc, 1);
            }
            tc_commit(bar_a_empty + 8 * sa);
            tc_commit(bar_b_empty + 8 * sb);
            if (kb == nKb - 1) tc_commit(bar_t_full + 8 * id);
          }
        }
        if (++sa == NA) { sa = 0; apar ^= 1; }
        if (++sb == NB) { sb = 0; bpar ^= 1; }
      }
    }
  } else if (warp == TMA_WARP && lane == 0) {
    // =========================================================================== producer 1 of 2: coefficient tiles
    // Two producer threads, one per operand, each with its own ring: a single thread that issued all three copies of
    // a K-block and polled both "empty" barriers was itself the slowest stage of the pipeline (anything added to its
    // loop slowed the whole kernel; the tensor pipe sat at 70-74 %).
    int sa = 0;
    uint32_t apar = 1;
    for (int i = 0; i < n_items; ++i) {
      const KItem it = kdecode(it0 + i * it_step, nG, nTt);
      const int gm = min(KB_GROUP, nMt - it.g * KB_GROUP);
      const char *src = reinterpret_cast<const char *>(p.wop) + ((size_t)it.c * nMt + (size_t)(it.g * KB_GROUP)) * nKb * A_TILE_BYTES;
      const char *src_lo = LO ? reinterpret_cast<const char *>(p.wop_lo) + ((size_t)it.c * nMt + (size_t)(it.g * KB_GROUP)) * nKb * A_TILE_BYTES
                              : nullptr;
      const size_t mstep = (size_t)nKb * A_TILE_BYTES;     // from M-tile m to m + 1 at the same K-block
      for (int kb = 0; kb < nKb; ++kb, src += A_TILE_BYTES, src_lo += A_TILE_BYTES) {
        mbar_wait(bar_a_empty + 8 * sa, apar);
        mbar_arrive_expect_tx(bar_a_full + 8 * sa, (LO ? 2 : 1) * gm * A_TILE_BYTES);
        for (int m = 0; m < gm; ++m) {
          bulk_g2s(sA + sa * A_STAGE_BYTES + m * A_TILE_BYTES, src + m * mstep, A_TILE_BYTES, bar_a_full + 8 * sa);
          if constexpr (LO)
            bulk_g2s(sA + sa * A_STAGE_BYTES + (KB_GROUP + m) * A_TILE_BYTES, src_lo + m * mstep, A_TILE_BYTES, bar_a_full + 8 * sa);
        }
        if (++sa == NA) { sa = 0; apar ^= 1; }
      }
    }
  } else if (warp == TMA_WARP + 1 && lane == 0) {
    // =========================================================================== producer 2 of 2: voltage K-blocks
    tma_prefetch_desc(&tmap);
    int sv = 0;  // voltage stage (operand stage for fp16, raw stage for int8)
    uint32_t vpar = 1;
    constexpr int NV = IS_F16 ? NB : NR;
    constexpr uint32_t VBYTES = IS_F16 ? B_STAGE_BYTES : (IS_CI4 ? RAW_STAGE_BYTES / 2 : RAW_STAGE_BYTES);
    constexpr int XSTEP = IS_CI4 ? BF_KBLOCK / 2 : BF_KBLOCK;   // tensor-map elements (bytes / fp16) per K-block
    const uint32_t sV = IS_F16 ? sB : sR;
    const uint32_t bar_v_full = IS_F16 ? bar_b_full : bar_r_full, bar_v_empty = IS_F16 ? bar_b_empty : bar_r_empty;
    for (int i = 0; i < n_items; ++i) {
      const KItem it = kdecode(it0 + i * it_step, nG, nTt);
      for (int kb = 0; kb < nKb; ++kb) {
        mbar_wait(bar_v_empty + 8 * sv, vpar);
        mbar_arrive_expect_tx(bar_v_full + 8 * sv, VBYTES);
        tma_load_3d(sV + sv * (IS_F16 ? B_STAGE_BYTES : RAW_STAGE_BYTES), &tmap, kb * XSTEP, it.tt * TILE_T, it.c, bar_v_full + 8 * sv);
        if (++sv == NV) { sv = 0; vpar ^= 1; }
      }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == MMA_WARP) tmem_dealloc(tmem_base, 512);
  probe_mark(p.probe, 1);
}

// 3-D view of the voltages: {K' elements, nsamp, nchan}, box {64, 256, 1}
template <int IN>
cudaError_t make_tmap(CUtensorMap *tm, const BfParams &p, int box_rows) {
  PFN_encodeTiled enc = bf_get_encode();
  if (!enc) return cudaErrorNotSupported;
  const bool f16 = IN == BF_CF16;
  const cuuint64_t esz = f16 ? 2 : 1;
  // elements per sample row: 2 nant (re, im) values, or nant bytes for the 4+4-bit format
  cuuint64_t dims[3] = {(cuuint64_t)(IN == BF_CI4 ? p.nant : 2 * p.nant), (cuuint64_t)p.nsamp, (cuuint64_t)p.nchan_run};
  cuuint64_t strides[2] = {dims[0] * esz, dims[0] * esz * (cuuint64_t)p.nsamp};
  cuuint32_t box[3] = {(cuuint32_t)(IN == BF_CI4 ? BF_KBLOCK / 2 : BF_KBLOCK), (cuuint32_t)box_rows, 1};
  cuuint32_t estr[3] = {1, 1, 1};
  CUresult r = enc(tm, f16 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT16 : CU_TENSOR_MAP_DATA_TYPE_UINT8, 3,
                   const_cast<void *>(p.volt), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                   f16 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

template <int NINT_T, int IN, bool BEAMS = false, bool LO = false>
cudaError_t launch_kb(const BfParams &p, int dtype, int sm_count, cudaStream_t st) {
  (void)dtype;
  constexpr bool IS_F16 = IN == BF_CF16;
  constexpr int NA = LO ? 2 : 3, NB = LO ? 2 : (IS_F16 ? 3 : 2), NR = IS_F16 ? 0 : (LO ? 2 : 3);
  constexpr int A_STAGE_BYTES = a_stage_bytes_v<LO>;
  CUtensorMap tm;
  cudaError_t e = bf_cached_tmap(&tm, p, 100 + IN, TILE_T, make_tmap<IN>);
  if (e != cudaSuccess) return e;
  const int nG = (p.nMt + KB_GROUP - 1) / KB_GROUP;
  const int nTt = (p.nsamp + TILE_T - 1) / TILE_T;
  const long long total = (long long)p.nchan_run * nTt * nG;
  const size_t smem = 1024 + NA * A_STAGE_BYTES + NB * B_STAGE_BYTES + NR * RAW_STAGE_BYTES + 512;
  auto kern = bf_umma_kblock_kernel<NINT_T, IN, NA, NB, NR, BEAMS, LO>;
  static thread_local int attr_dev = -1;   // once per instantiation and device
  if ((e = bf_set_smem_once(kern, smem, &attr_dev)) != cudaSuccess) return e;
  if (NINT_T == 0 && !BEAMS) {
    e = cudaMemsetAsync(p.pow, 0, (size_t)p.nchan_run * p.nbeam * p.nbin * sizeof(float), st);
    if (e != cudaSuccess) return e;
  }
  const int grid = (int)(total < sm_count ? total : sm_count);
  kern<<<grid, NTHREADS, smem, st>>>(p, tm, total, nG, nTt);
  return cudaGetLastError();
}

template <int IN>
cudaError_t launch_kb_nint(const BfParams &p, int dtype, int sm_count, cudaStream_t st) {
  if (p.mode == BF_MODE_BEAMS) return launch_kb<64, IN, true>(p, dtype, sm_count, st);
  if (p.wop_lo != nullptr) {   // short bins: two-term coefficients
    switch (p.nint) {
      case 1: return launch_kb<1, IN, false, true>(p, dtype, sm_count, st);
      case 2: return launch_kb<2, IN, false, true>(p, dtype, sm_count, st);
      case 4: return launch_kb<4, IN, false, true>(p, dtype, sm_count, st);
      case 8: return launch_kb<8, IN, false, true>(p, dtype, sm_count, st);
      default: break;
    }
  }
  switch (p.nint) {
    case 1: return launch_kb<1, IN>(p, dtype, sm_count, st);
    case 2: return launch_kb<2, IN>(p, dtype, sm_count, st);
    case 4: return launch_kb<4, IN>(p, dtype, sm_count, st);
    case 8: return launch_kb<8, IN>(p, dtype, sm_count, st);
    case 16: return launch_kb<16, IN>(p, dtype, sm_count, st);
    case 32: return launch_kb<32, IN>(p, dtype, sm_count, st);
    case 64: return launch_kb<64, IN>(p, dtype, sm_count, st);
    default:
      if (p.nint < BF_LO_NINT) return cudaErrorNotSupported;   // bf_umma_supported lets no such shape through
      return launch_kb<0, IN>(p, dtype, sm_count, st);
  }
}

}  // namespace

cudaError_t bf_launch_umma_kblock(const BfParams &p, int dtype, int sm_count, cudaStream_t st) {
  if (dtype == BF_CF16) return launch_kb_nint<BF_CF16>(p, dtype, sm_count, st);
  if (dtype == BF_CI4) return launch_kb_nint<BF_CI4>(p, dtype, sm_count, st);
  return launch_kb_nint<BF_CI8>(p, dtype, sm_count, st);
}
