// bf_umma.cu -- the fused tensor-core beamformer for small arrays (2*nant <= 64, complex int8 input):
// hot-path rows a2..a5 in ONE persistent kernel.
//
//   a2 ingest      int8 (re,im) voltages  --cp.async.bulk (TMA engine)-->  raw shared-memory ring
//                  --LDS.128 / PRMT / HSUB2-->  fp16, written back to shared memory in the
//                  128-byte-swizzled K-major layout tcgen05.mma reads
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
//   warps 0-15  epilogue: warp w owns TMEM lanes 32*(w&3).. and columns 64*(w>>2).. of every tile
//   warps 16..  convert (CONV_WARPS): raw int8 stage -> fp16 operand stage
//   next 2      MMA issue, one warp (one elected lane) per TMEM accumulator stage; TMEM allocation
//   last warp   one thread issuing the bulk copies (voltage tiles; coefficient tiles on channel change)
// Pipelines (all mbarrier based): raw stages full/empty (TMA <-> convert), operand stages full/empty
// (convert <-> MMA), coefficient buffers full/empty (TMA <-> MMA), TMEM accumulator stages full/empty
// (MMA <-> epilogue).
#include <type_traits>

#include "bf_tmap.h"
#include "bf_umma_common.cuh"

namespace {

using namespace bfk;

constexpr int MAX_INPUT_PIECES = TILE_T * 4;  // 16-byte input pieces per tile at nant = 32

template <bool SPREAD, int CONV_WARPS> constexpr int k64_threads_v = SPREAD ? 1024 : (EPI_WARPS + CONV_WARPS + 3) * 32;

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

// NINT_T: integration length if it is a power of two <= 64; 0 = a larger multiple of 64 (each epilogue
// warp adds the partial sum of its 64 columns atomically into a zeroed output).
// SPREAD: with <= 64 beams only the first TMEM lane quadrants hold real rows, and a quadrant can only be
// read by warps w with w % 4 == quadrant -- which all sit on SM sub-partition `quadrant`.  For <= 16
// beams the whole epilogue therefore lands on sub-partition 0; SPREAD launches 32 warps and puts the
// convert / MMA / TMA warps on sub-partitions 1-3 only, so that sub-partition 0 does nothing else.
// LO: two-term coefficients (bf_internal.h, BF_LO_NINT): every coefficient buffer holds GROUP "hi" tiles followed by
// GROUP "lo" tiles and a voltage tile is contracted against both (8 MMAs per accumulator tile instead of 4).
template <int NINT_T, int GROUP, int NSTAGE, int NRAW, int CONV_WARPS, bool SPREAD, int IN, bool BEAMS, bool LO>
__global__ void __launch_bounds__(k64_threads_v<SPREAD, CONV_WARPS>, 1)
bf_umma_k64_kernel(const BfParams p, const long long total_items, const int nG, const int nTt, const int nks) {
  extern __shared__ uint8_t smem_raw[];
  constexpr int CONV_THREADS = CONV_WARPS * 32;
  static_assert(CONV_WARPS == 8, "role table below assumes 8 convert warps");
  static_assert(GROUP > 1 || NSTAGE == 2, "GROUP == 1: each MMA warp must see every completion of the operand stages it waits on");

  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  constexpr int APB = (LO ? 2 : 1) * GROUP;                       // coefficient tiles per buffer
  const uint32_t sA = smem_base;                                  // 2 buffers x APB coefficient tiles
  const uint32_t sB = sA + 2 * APB * A_TILE_BYTES;                // NSTAGE fp16 operand stages
  const uint32_t sR = sB + NSTAGE * B_STAGE_BYTES;                // NRAW raw int8 stages
  const uint32_t sBar = sR + NRAW * RAW_STAGE_BYTES;              // barriers
  const uint32_t bar_b_full = sBar, bar_b_empty = sBar + 8 * NSTAGE;
  const uint32_t bar_r_full = sBar + 16 * NSTAGE, bar_r_empty = bar_r_full + 8 * NRAW;
  const uint32_t bar_a_full = bar_r_full + 16 * NRAW, bar_a_empty = bar_a_full + 16;
  const uint32_t bar_t_full = bar_a_full + 32, bar_t_empty = bar_t_full + 16;
  const uint32_t s_tmem = bar_t_full + 32;

  // warp index through a shuffle so that the compiler knows it is warp-uniform (role code then
  // runs on the uniform datapath: descriptors in uniform registers, no per-lane waterfall loops)
  const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0), lane = threadIdx.x & 31;
  // role table: cw = convert-warp index (0..7) or -1, mw = MMA-warp index (0/1) or -1
  int cw = -1, mw = -1, ew = -1;     // ew = epilogue-warp index (0..15) or -1
  bool is_tma = false;
  if (!SPREAD) {
    // The warp scheduler favours the higher warp index among eligible warps, and the epilogue warps are the chain
    // everything else waits for: convert warps sit at the bottom (0-7), the epilogue above them (8-23; 8 % 4 == 0, so
    // warp & 3 is still the TMEM lane quadrant), the MMA and TMA warps on top (24-26).
    if (warp < 8) cw = warp;
    else if (warp < 8 + EPI_WARPS) ew = warp - 8;
    else if (warp < 8 + EPI_WARPS + 2) mw = warp - (8 + EPI_WARPS);
    else if (warp == 8 + EPI_WARPS + 2) is_tma = true;
  } else if (warp < EPI_WARPS) {
    ew = warp;
  } else if (warp >= EPI_WARPS && (warp & 3) != 0) {  // 32 warps; nothing but epilogue on sub-partition 0
    const int r = (warp - EPI_WARPS) >> 2, q = warp & 3;   // r = 0..3, q = 1..3
    if (r < 3) { const int k = r * 3 + (q - 1); if (k < 8) cw = k; }   // 17,18,19,21,22,23,25,26
    else if (q < 3) mw = q - 1;                                        // 29, 30
    else is_tma = true;                                                // 31
  }

  // full rows (nant = 32): the convert warps work as two groups of four on alternate tiles (see the convert role)
  const bool split = p.nant == 32;
  if (threadIdx.x == 0) {
    const int nconv = split ? CONV_WARPS / 2 : CONV_WARPS;   // warps that convert one tile
    for (int s = 0; s < NSTAGE; ++s) { mbar_init(bar_b_full + 8 * s, nconv); mbar_init(bar_b_empty + 8 * s, 2); }
    for (int s = 0; s < NRAW; ++s) { mbar_init(bar_r_full + 8 * s, 1); mbar_init(bar_r_empty + 8 * s, nconv); }
    for (int s = 0; s < 2; ++s) {
      mbar_init(bar_a_full + 8 * s, 1); mbar_init(bar_a_empty + 8 * s, 2);
      mbar_init(bar_t_full + 8 * s, 1);          mbar_init(bar_t_empty + 8 * s, EPI_WARPS);
    }
    fence_barrier_init();
  }
  if (mw == 0) tmem_alloc(s_tmem, 512);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(s_tmem));
  tmem_base = __shfl_sync(0xffffffffu, tmem_base, 0);
  probe_mark(p.probe, 0);

  // this CTA's contiguous item range
  const long long it0 = total_items * blockIdx.x / gridDim.x;
  const long long it1 = total_items * (blockIdx.x + 1) / gridDim.x;
  const int n_items = (int)(it1 - it0);
  const int nMt = p.nMt;

  if (ew >= 0) {
    // =========================================================================== epilogue
    // 16 warps: warp w owns TMEM lanes 32*(w&3).. and columns 64*(w>>2).. of EVERY accumulator tile.
    // The TMEM stage is handed back to the MMA warp as soon as this warp's last tcgen05.ld has
    // landed in registers -- the squaring of that last chunk, the shuffle and the store run in the
    // shadow of the next tile's MMAs.  The kernel is bound by instruction issue around the tensor
    // pipe (profiles/), so everything that does not change from tile to tile is computed once per
    // (chan, beam group) run and the accumulator stage of a tile is a compile-time constant:
    // tile m of an item uses stage m & 1 (GROUP even), item i uses stage i & 1 (GROUP == 1).
    constexpr int BPW = NINT_T == 0 ? 1 : 64 / NINT_T;       // bins per warp and tile
    constexpr int BPT = NINT_T == 0 ? 0 : TILE_T / NINT_T;   // bins per tile
    const int quad = ew & 3, slot = ew >> 2;
    const bool lane0 = lane == 0;
    uint32_t t_lane = tmem_base + ((uint32_t)(quad * 32) << 16) + slot * 64;
    uint32_t b_full = bar_t_full;
    asm volatile("" : "+r"(t_lane), "+r"(b_full));           // keep in registers, do not rematerialise
    const int bl = quad * 16 + (lane & 15);                  // this lane's beam inside an M-tile
    const int nbeam = p.nbeam, nbin = p.nbin;
    const size_t mstride = (size_t)BF_TILE_BEAMS * nbin;     // output distance between M-tiles
    const bool vec_ok = (nbin % 4 == 0) && ((reinterpret_cast<uintptr_t>(p.pow) & 15) == 0);
    const bool ragged = (p.nsamp % TILE_T) != 0;             // the last time tile of a channel is partial
    const bool bvec_ok = BEAMS && (p.nsamp % 4 == 0) && ((reinterpret_cast<uintptr_t>(p.beams) & 15) == 0);
    Item it = decode_item(it0, nG, nTt);
    uint32_t par0 = 0, par1 = 0;                             // parity of the next completion of t_full[0/1]
    int i = 0;
    constexpr bool DEFER = !BEAMS;
    EpiPend<NINT_T> pend;
    epi_pend_init<NINT_T>(pend);
    while (i < n_items) {
      // ---- one run: the items of one (chan, beam group) inside my range; time tiles it.tt ..
      const int run = min(n_items - i, nTt - it.tt);
      const int gm = min(GROUP, nMt - it.g * GROUP);
      const int beam0 = it.g * GROUP * BF_TILE_BEAMS + bl;
      uint32_t rows = 0, wr = 0;                             // bit m: quadrant holds real rows / this lane stores
#pragma unroll
      for (int m = 0; m < GROUP; ++m) {
        const int beam = beam0 + m * BF_TILE_BEAMS;
        if (m < gm && beam - (lane & 15) < nbeam) rows |= 1u << m;
        if (m < gm && lane < 16 && beam < nbeam) wr |= 1u << m;
      }
      float *ptr = p.pow + ((size_t)it.c * nbeam + beam0) * nbin + (NINT_T == 0 ? 0 : it.tt * BPT + slot * BPW);
      // voltage-beam mode (row f4): this lane's beam at the first column of this warp in tile it.tt
      __half2 *bptr = reinterpret_cast<__half2 *>(p.beams) + ((size_t)it.c * nbeam + beam0) * p.nsamp + it.tt * TILE_T + slot * 64;
      uint32_t bok = 0;                                      // bit m: this lane's beam of M-tile m exists
#pragma unroll
      for (int m = 0; m < GROUP; ++m)
        if (m < gm && beam0 + m * BF_TILE_BEAMS < nbeam) bok |= 1u << m;
      int tt = it.tt;
      int k = 0;
      if constexpr (DEFER && NINT_T != 0 && EpiPend<NINT_T>::DEFER) {
        // ---- lean loop: the interior of a run (every quadrant holds real rows, every bin of the tile exists).  The
        // kernel's time follows the instructions the SM sub-partitions issue (profiles/), and the general loop below
        // spends more of them on predicates, pointer arithmetic and re-convergence than on squares; here a tile is
        // wait -> tcgen05.ld x2 -> 32 FFMA2 -> add tree, with everything else hoisted to the run.
        const bool all_rows = rows == (1u << GROUP) - 1;       // implies gm == GROUP
        const int n_lean = all_rows ? ((ragged && it.tt + run == nTt) ? run - 1 : run) : 0;
        bool wrm[GROUP];
#pragma unroll
        for (int m = 0; m < GROUP; ++m) wrm[m] = (wr >> m) & 1;
        const bool vec = vec_ok;
        if (n_lean > 0) epi_pend_flush<NINT_T>(pend);           // a tail left by the general loop: the lean flush below assumes whole tiles
        // one tile on accumulator stage ACC (a compile-time constant, so its barriers and TMEM columns are immediates)
        auto lean_tile = [&](auto acc_c, int m) {
          constexpr int ACC = decltype(acc_c)::value;
          uint32_t &par = ACC ? par1 : par0;
          // (sleeping between polls was measured at 64 beams: 0.188 vs 0.172 ms -- the wake-up latency is on the chain)
          mbar_wait_tight(b_full + 8 * ACC, par);
          par ^= 1;
          tc_fence_after();
          epilogue_tile_defer<NINT_T, true>(t_lane + ACC * TILE_T, ptr + m * mstride, wrm[m], 1 << 30, vec, b_full + 16 + 8 * ACC, lane0,
                                            pend);
        };
        if constexpr (GROUP == 1) {   // items alternate between the two stages: walk them in (even, odd) pairs
          if ((i & 1) && k < n_lean) { lean_tile(std::integral_constant<int, 1>{}, 0); ++k; ++i; ptr += BPT; }
          for (; k + 1 < n_lean; k += 2, i += 2) {
            lean_tile(std::integral_constant<int, 0>{}, 0); ptr += BPT;
            lean_tile(std::integral_constant<int, 1>{}, 0); ptr += BPT;
          }
          if (k < n_lean) { lean_tile(std::integral_constant<int, 0>{}, 0); ++k; ++i; ptr += BPT; }
        } else {
          for (; k < n_lean; ++k, ++i, ptr += BPT) {
#pragma unroll
            for (int m = 0; m < GROUP; ++m) {
              if (m & 1) lean_tile(std::integral_constant<int, 1>{}, m);
              else lean_tile(std::integral_constant<int, 0>{}, m);
            }
          }
        }
        tt += n_lean;
      }
      for (; k < run; ++k, ++i, ++tt, ptr += BPT, bptr += TILE_T) {
        int nvalid = 1 << 30;
        float *out = ptr;
        if (BEAMS) {
          nvalid = p.nsamp - (tt * TILE_T + slot * 64);
        } else if (NINT_T == 0) {
          const int t_first = tt * TILE_T + slot * 64;       // first time sample of this warp's columns
          out = ptr + t_first / p.nint;
          nvalid = t_first < p.nsamp ? 1 : 0;
        } else if (ragged && tt == nTt - 1) {
          nvalid = nbin - (tt * BPT + slot * BPW);
        }
        auto one = [&](auto acc_c, int m) {
          constexpr int ACC = decltype(acc_c)::value;
          uint32_t &par = ACC ? par1 : par0;
          mbar_wait_tight(b_full + 8 * ACC, par);
          par ^= 1;
          tc_fence_after();
          if (!((rows >> m) & 1)) {                          // warp-uniform: only padding rows in this quadrant
            epilogue_skip(b_full + 16 + 8 * ACC, lane0);
            return;
          }
          if constexpr (!BEAMS && NINT_T == 0) {
            if (p.nint % 64 != 0) {   // any other bin length >= 16: running sums per lane, flushed where a bin ends
              epilogue_tile_anynint(t_lane + ACC * TILE_T, ptr + m * mstride, (wr >> m) & 1, tt * TILE_T + slot * 64, p.nint, nbin,
                                    b_full + 16 + 8 * ACC, lane0);
              return;
            }
          }
          if constexpr (BEAMS)
            epilogue_beams_tile(t_lane + ACC * TILE_T, bptr + (size_t)m * BF_TILE_BEAMS * p.nsamp, (bok >> m) & 1, nvalid,
                                bvec_ok, p.beam_scale, lane >= 16, b_full + 16 + 8 * ACC, lane0);
          else if constexpr (DEFER)
            epilogue_tile_defer<NINT_T>(t_lane + ACC * TILE_T, out + m * mstride, (wr >> m) & 1, nvalid, NINT_T != 0 && vec_ok,
                                        b_full + 16 + 8 * ACC, lane0, pend);
          else
            epilogue_tile<NINT_T>(t_lane + ACC * TILE_T, out + m * mstride, (wr >> m) & 1, nvalid, NINT_T != 0 && vec_ok,
                                  b_full + 16 + 8 * ACC, lane0);
        };
        if constexpr (GROUP == 1) {
          if (i & 1) one(std::integral_constant<int, 1>{}, 0);
          else one(std::integral_constant<int, 0>{}, 0);
        } else {
#pragma unroll
          for (int m = 0; m < GROUP; ++m)
            if (m < gm) {
              if (m & 1) one(std::integral_constant<int, 1>{}, m);
              else one(std::integral_constant<int, 0>{}, m);
            }
        }
      }
      it.tt = 0;
      if (++it.g == nG) { it.g = 0; ++it.c; }
    }
    if constexpr (DEFER) epi_pend_flush<NINT_T>(pend);     // the tail of this CTA's last tile
  } else if (cw >= 0) {
    // =========================================================================== convert
    // 16-byte input pieces per thread per tile: int8 rows are 2*nant bytes, 4-bit rows nant bytes
    constexpr int PIECES = (IN == BF_CI4 ? MAX_INPUT_PIECES / 2 : MAX_INPUT_PIECES) / CONV_THREADS;
    constexpr int CPP = IN == BF_CI4 ? 4 : 2;    // 16-byte fp16 output chunks per input piece
    const int ctid = cw * 32 + lane;
    const int npr = IN == BF_CI4 ? p.nant / 16 : p.nant / 8;   // pieces per time sample
    const int npieces = TILE_T * npr;
    // zero the operand stages once: K' columns beyond 2*nant must read as 0, never as stale NaN patterns
    for (int o = ctid * 16; o < NSTAGE * B_STAGE_BYTES; o += CONV_THREADS * 16) st_shared_v4(sB + o, 0, 0, 0, 0);
    asm volatile("bar.sync 1, %0;" ::"n"(CONV_THREADS) : "memory");

    // a thread converts the same pieces of every tile: row t, 16-byte piece q of that row.  Raw rows
    // are compact (2*nant bytes), so piece pc sits at byte 16*pc of the raw stage.
    uint32_t p_dst[PIECES];  // byte offset of the first output chunk inside a stage (second chunk: ^ 16)
#pragma unroll
    for (int k = 0; k < PIECES; ++k) {
      const int pc = ctid + k * CONV_THREADS;
      const int t = pc / npr, q = pc - t * npr;
      p_dst[k] = pc < npieces ? (uint32_t)((t >> 3) * 1024 + (t & 7) * 128 + (((CPP * q) ^ (t & 7)) << 4)) : 0xffffffffu;
    }
    int rs = 0, st = 0;              // raw slot / operand stage of the current item
    uint32_t rpar = 0, bpar = 1;     // parities to wait for on r_full[rs] / b_empty[st]
    if (split) {
      // ---- full rows (nant = 32), two groups of four warps on alternate tiles.  A tile's conversion is a chain of
      // dependent latencies (barrier, LDS, barrier, STS, proxy fence, arrive) that one warp walks once per tile; with
      // all eight warps on the same tile that chain, not the ring depth, set the rate.  Two tiles are now in
      // conversion at any time.  Thread gtid of a group owns pieces gtid + 128 k: row (gtid + 128 k) / NPR, so piece
      // k sits KSTEP bytes after piece 0 in the operand stage and 16 * GT bytes after it in the raw slot: all
      // shared-memory accesses are [register + immediate].
      constexpr int NPR = IN == BF_CI4 ? 2 : 4;                          // 16-byte pieces per time sample
      constexpr int GT = CONV_THREADS / 2, GP = TILE_T * NPR / GT;       // threads per group, pieces per thread
      constexpr uint32_t KSTEP = (GT / NPR / 8) * 1024;
      const int grp = cw >> 2, gtid = ctid & (GT - 1);
      const int t0 = gtid / NPR, q0 = gtid % NPR;
      const uint32_t raw0 = sR + 16 * gtid;
      const uint32_t dst0 = sB + (uint32_t)((t0 >> 3) * 1024 + (t0 & 7) * 128 + (((CPP * q0) ^ (t0 & 7)) << 4));
      for (int i = grp; i < n_items; i += 2) {
        const int rs = i % NRAW, st = i % NSTAGE;
        const uint32_t raw = raw0 + rs * RAW_STAGE_BYTES, dst = dst0 + st * B_STAGE_BYTES;
        mbar_wait(bar_r_full + 8 * rs, (uint32_t)((i / NRAW) & 1));
        constexpr int RP = GP, r0 = 0;
        uint4 x[GP];
#pragma unroll
        for (int k = 0; k < GP; ++k) x[k] = ld_shared_v4(raw + k * (16 * GT));
        mbar_wait(bar_b_empty + 8 * st, (uint32_t)(((i / NSTAGE) & 1) ^ 1));
        {
          if (IN == BF_CI4) {
            const uint32_t d1 = dst ^ 16u, d2 = dst ^ 32u, d3 = dst ^ 48u;
#pragma unroll
            for (int k = 0; k < RP; ++k) {
              uint32_t h[4];
              cvt_i4x8_f16x8(x[k].x, h); st_shared_v4(dst + (r0 + k) * KSTEP, h[0], h[1], h[2], h[3]);
              cvt_i4x8_f16x8(x[k].y, h); st_shared_v4(d1 + (r0 + k) * KSTEP, h[0], h[1], h[2], h[3]);
              cvt_i4x8_f16x8(x[k].z, h); st_shared_v4(d2 + (r0 + k) * KSTEP, h[0], h[1], h[2], h[3]);
              cvt_i4x8_f16x8(x[k].w, h); st_shared_v4(d3 + (r0 + k) * KSTEP, h[0], h[1], h[2], h[3]);
            }
          } else {
            const uint32_t d1 = dst ^ 16u;
#pragma unroll
            for (int k = 0; k < RP; ++k) {
              uint32_t h[8];
              cvt_i8x4_f16x4(x[k].x, h[0], h[1]);
              cvt_i8x4_f16x4(x[k].y, h[2], h[3]);
              cvt_i8x4_f16x4(x[k].z, h[4], h[5]);
              cvt_i8x4_f16x4(x[k].w, h[6], h[7]);
              st_shared_v4(dst + (r0 + k) * KSTEP, h[0], h[1], h[2], h[3]);
              st_shared_v4(d1 + (r0 + k) * KSTEP, h[4], h[5], h[6], h[7]);
            }
          }
        }
        fence_proxy_async_smem();
        __syncwarp();
        if (lane == 0) {
          mbar_arrive(bar_r_empty + 8 * rs);  // raw bytes are converted: slot may be refilled
          mbar_arrive(bar_b_full + 8 * st);
        }
      }
    } else {
      // ---- short rows (nant < 32): generic piece table
      for (int i = 0; i < n_items; ++i) {
        mbar_wait(bar_r_full + 8 * rs, rpar);
        uint4 x[PIECES];
        convert_load<PIECES, CONV_THREADS>(sR + rs * RAW_STAGE_BYTES, ctid, p_dst, x);
        mbar_wait(bar_b_empty + 8 * st, bpar);
        if (IN == BF_CI4) convert_store_ci4<PIECES>(sB + st * B_STAGE_BYTES, p_dst, x);
        else convert_store<PIECES>(sB + st * B_STAGE_BYTES, p_dst, x);
        fence_proxy_async_smem();
        __syncwarp();
        if (lane == 0) {
          mbar_arrive(bar_r_empty + 8 * rs);  // raw bytes are in registers / converted: slot may be refilled
          mbar_arrive(bar_b_full + 8 * st);
        }
        if (++rs == NRAW) { rs = 0; rpar ^= 1; }
        if (++st == NSTAGE) { st = 0; bpar ^= 1; }
      }
    }
  } else if (mw >= 0) {
    // =========================================================================== MMA issue (2 warps)
    // tcgen05.mma issue is (nearly) blocking: measured, the issuing thread gets control back only
    // ~160 clk before its 4 MMAs (512 clk) finish, so any bookkeeping + barrier wait longer than that
    // between two tiles idles the tensor pipe.  Hence one issuing warp PER ACCUMULATOR STAGE: while
    // warp 0 is blocked issuing into stage 0, warp 1 does its waits for stage 1 and queues behind it.
    // The whole warp walks the loop (all values warp-uniform); one elected lane issues.
    const int id = mw;  // = the accumulator stage this warp feeds
    // stage of a tile (the epilogue uses the same compile-time rule): GROUP even -> tile m of an item
    // goes to stage m & 1; GROUP == 1 -> item i goes to stage i & 1
    constexpr uint32_t idesc = make_idesc_f16(BF_TILE_ROWS, TILE_T);
    constexpr uint32_t dhi = sdesc_k_sw128_hi();
    const uint32_t a_lo0 = sdesc_k_sw128_lo(sA), b_lo0 = sdesc_k_sw128_lo(sB);   // descriptor low words: address >> 4
    const uint32_t d = tmem_base + id * TILE_T;
    const uint32_t t_full = bar_t_full + 8 * id, t_empty = bar_t_empty + 8 * id;
    Item it = decode_item(it0, nG, nTt);
    int ag = 0, ab = 0;
    int st = 0;                 // operand stage and the parity its "full" barrier completes next
    uint32_t st_par = 0;
    uint32_t te_par = 1;        // parity of t_empty[id] to wait for (first use passes on the fresh barrier)
    int gm = min(GROUP, nMt - it.g * GROUP);
    for (int i = 0; i < n_items; ++i) {
      if (i == 0 || it.tt == 0) {  // (chan, beam group) changes exactly when the time tile wraps
        if (ag > 0 && elect_one()) tc_commit(bar_a_empty + 8 * ab);  // my MMAs so far have left the old buffer
        ab = ag & 1;
        gm = min(GROUP, nMt - it.g * GROUP);
        mbar_wait(bar_a_full + 8 * ab, (ag >> 1) & 1);
        ++ag;
      }
      const bool mine = GROUP == 1 ? ((i & 1) == id) : (id < gm);
      // A warp with no tile in this item (the second warp when the last beam group holds ONE M-tile) still takes part in
      // the hand-shake of the item's operand stage: it waits for "full" and gives its own arrival to "empty".  A parity wait
      // cannot tell completion n from n + 2, so the warp must neither run ahead of a stage it does not look at (it walked
      // past a run of such items and then multiplied a STALE stage at its next own item: wrong powers in the second M-tile
      // of one time tile, one launch in a few) nor fall two completions behind it (if the other warp arrived twice on its
      // behalf, nothing would hold the ring back for a late warp, and it would wait for ever).  Found by
      // tests/test_gpu_combos.py::test_fifty_runs_are_bit_equal and tests/test_zy_jitter.py.
      // (GROUP == 1: the warps alternate items on two stages; each owns every completion of its own stage.)
      if (GROUP > 1 && !mine) {
        mbar_wait(bar_b_full + 8 * st, st_par);
        if (elect_one()) mbar_arrive(bar_b_empty + 8 * st);   // nothing of mine reads the stage: a plain arrival
      }
      if (mine) {
        const uint32_t b_full = bar_b_full + 8 * st, b_empty = bar_b_empty + 8 * st;
        mbar_wait(b_full, st_par);
        const uint32_t b_lo = b_lo0 + st * (B_STAGE_BYTES >> 4);
        for (int m = (GROUP == 1 ? 0 : id); m < gm; m += 2) {
          mbar_wait(t_empty, te_par);
          te_par ^= 1;
          tc_fence_after();
          const uint32_t a_lo = a_lo0 + (ab * APB + m) * (A_TILE_BYTES >> 4);
          const bool last = m + 2 >= gm;
          if (elect_one()) {
#pragma unroll
            for (int k = 0; k < 4; ++k)  // advance 16 fp16 = 32 bytes along K inside the swizzle atom
              if (k < nks) mma_f16_ss_lo(d, a_lo + 2 * k, b_lo + 2 * k, dhi, idesc, k > 0);
            if constexpr (LO) {          // the residual term of the coefficients against the same voltages
#pragma unroll
              for (int k = 0; k < 4; ++k)
                if (k < nks) mma_f16_ss_lo(d, a_lo + GROUP * (A_TILE_BYTES >> 4) + 2 * k, b_lo + 2 * k, dhi, idesc, 1);
            }
            tc_commit(t_full);
            if (last) {
              tc_commit(b_empty);
              if (GROUP == 1) tc_commit(b_empty);  // the stage is mine alone: both arrivals
            }
          }
        }
      }
      if (++st == NSTAGE) { st = 0; st_par ^= 1; }
      next_item(it, nG, nTt);
    }
  } else if (is_tma && lane == 0) {
    // =========================================================================== bulk-copy producer (one thread)
    const size_t row_bytes = IN == BF_CI4 ? (size_t)p.nant : (size_t)2 * p.nant;
    const char *volt = reinterpret_cast<const char *>(p.volt);
    int ag = 0, prev_c = -1, prev_g = -1;
    Item it = decode_item(it0, nG, nTt);
    for (int i = 0; i < n_items; ++i, next_item(it, nG, nTt)) {
      if (it.c != prev_c || it.g != prev_g) {
        // new (channel, beam group): its coefficient tiles (already the swizzled smem image) -> other A buffer
        prev_c = it.c; prev_g = it.g;
        const int ab = ag & 1;
        mbar_wait(bar_a_empty + 8 * ab, ((ag >> 1) & 1) ^ 1);
        const int gm = min(GROUP, nMt - it.g * GROUP);
        const char *wsrc = reinterpret_cast<const char *>(p.wop) + ((size_t)it.c * nMt + (size_t)it.g * GROUP) * A_TILE_BYTES;
        mbar_arrive_expect_tx(bar_a_full + 8 * ab, (LO ? 2 : 1) * gm * A_TILE_BYTES);
        bulk_g2s(sA + ab * APB * A_TILE_BYTES, wsrc, gm * A_TILE_BYTES, bar_a_full + 8 * ab);
        if constexpr (LO) {
          const char *lsrc = reinterpret_cast<const char *>(p.wop_lo) + ((size_t)it.c * nMt + (size_t)it.g * GROUP) * A_TILE_BYTES;
          bulk_g2s(sA + (ab * APB + GROUP) * A_TILE_BYTES, lsrc, gm * A_TILE_BYTES, bar_a_full + 8 * ab);
        }
        ++ag;
      }
      const int rs = i % NRAW;
      mbar_wait(bar_r_empty + 8 * rs, ((i / NRAW) & 1) ^ 1);
      const int t_base = it.tt * TILE_T;
      const int rows = min(TILE_T, p.nsamp - t_base);  // tail tile: the stale rest of the stage is finite
      const uint32_t bytes = (uint32_t)(rows * row_bytes);  // int8 and only feeds bins >= nbin, never stored
      mbar_arrive_expect_tx(bar_r_full + 8 * rs, bytes);
      bulk_g2s(sR + rs * RAW_STAGE_BYTES, volt + ((size_t)it.c * p.nsamp + t_base) * row_bytes, bytes, bar_r_full + 8 * rs);
    }
  }

  tc_fence_before();
  __syncthreads();
  if (mw == 0) tmem_dealloc(tmem_base, 512);
  probe_mark(p.probe, 1);
}

template <int NINT_T, int GROUP, int NSTAGE, int NRAW, int CONV_WARPS, bool SPREAD, int IN, bool BEAMS = false, bool LO = false>
cudaError_t launch_k64(const BfParams &p, int sm_count, cudaStream_t st) {
  const int nG = (p.nMt + GROUP - 1) / GROUP;
  const int nTt = (p.nsamp + TILE_T - 1) / TILE_T;
  const long long total = (long long)p.nchan_run * nG * nTt;
  const int nks = (2 * p.nant + 15) / 16;
  const size_t smem = 1024 + 2 * (LO ? 2 : 1) * GROUP * A_TILE_BYTES + NSTAGE * B_STAGE_BYTES + NRAW * RAW_STAGE_BYTES + 256;
  auto kern = bf_umma_k64_kernel<NINT_T, GROUP, NSTAGE, NRAW, CONV_WARPS, SPREAD, IN, BEAMS, LO>;
  static thread_local int attr_dev = -1;   // once per instantiation and device
  cudaError_t e = bf_set_smem_once(kern, smem, &attr_dev);
  if (e != cudaSuccess) return e;
  if (NINT_T == 0 && !BEAMS) {
    e = cudaMemsetAsync(p.pow, 0, (size_t)p.nchan_run * p.nbeam * p.nbin * sizeof(float), st);
    if (e != cudaSuccess) return e;
  }
  const int grid = (int)(total < sm_count ? total : sm_count);
  kern<<<grid, k64_threads_v<SPREAD, CONV_WARPS>, smem, st>>>(p, total, nG, nTt, nks);
  return cudaGetLastError();
}

template <int NINT_T, int IN>
cudaError_t launch_k64_nint(const BfParams &p, int sm_count, cudaStream_t st) {
  if constexpr (NINT_T != 0 && NINT_T < BF_LO_NINT) {
    // short bins: two-term coefficients (the output stream, 4 bytes per beam and bin, hides the second set of MMAs)
    if (p.wop_lo != nullptr) {
      if (p.nMt == 1) return launch_k64<NINT_T, 1, 2, 4, 8, false, IN, false, true>(p, sm_count, st);
      return launch_k64<NINT_T, 2, 2, 2, 8, false, IN, false, true>(p, sm_count, st);
    }
  }
  // <= 64 beams: HBM-bound.  A raw slot is held for the whole HBM latency plus the conversion (~3 us
  // measured), so the bytes in flight per SM decide the bandwidth: 8 raw slots of 16 KiB.
  // <= 32 beams: rows only in lane quadrants 0-1, the epilogue gets those sub-partitions to itself (SPREAD).  Not for the
  // 4-bit format: its unpack is three instructions per antenna and needs all four sub-partitions (measured on the
  // sweep at 16 beams: 0.220 ms SPREAD, 0.195 ms plain)
  if (p.nbeam <= 32 && IN != BF_CI4) return launch_k64<NINT_T, 1, 2, 8, 8, true, IN>(p, sm_count, st);
  if (p.nMt == 1) return launch_k64<NINT_T, 1, 2, 8, 8, false, IN>(p, sm_count, st);
  if (p.nMt <= 2) return launch_k64<NINT_T, 2, 3, 4, 8, false, IN>(p, sm_count, st);
  return launch_k64<NINT_T, 4, 2, 2, 8, false, IN>(p, sm_count, st);                  // many beams: MMA-bound, big A group
}

}  // namespace

// bins the fp16 kernels integrate: 2^k <= 64 in registers / by shuffles (compile-time), multiples of 64 as one atomic add per
// warp and tile, and ANY other length >= BF_LO_NINT through epilogue_tile_anynint (atomic adds where a bin ends).  Below
// BF_LO_NINT only the powers of two exist: those kernels also contract the residual coefficient plane.
static bool nint_ok(int I) { return (I <= 64 && (I & (I - 1)) == 0) || I >= BF_LO_NINT; }

// which tensor-core kernel takes this shape: 1 = coefficients-resident (2*nant <= 64), 2 = K-blocked
static int umma_variant(int dtype, int nant) {
  if (dtype == BF_CI8 && nant % 8 == 0 && nant <= 32) return 1;
  if (dtype == BF_CI4 && nant % 16 == 0 && nant <= 32) return 1;  // bulk copies need rows of 16 bytes
  if (dtype == BF_CI8 && nant % 8 == 0) return 2;   // TMA rows must be multiples of 16 bytes
  if (dtype == BF_CF16 && nant % 4 == 0) return 2;
  if (dtype == BF_CI4 && nant % 16 == 0) return 2;  // K-blocks of 32 antennas = 32 bytes per sample
  return 0;
}

bool bf_umma_shape_supported(const bf_ctx *c, const char **why) {
  if (!umma_variant(c->dtype, c->nant)) { *why = "needs nant % 8 == 0 (int8), % 4 == 0 (fp16) or % 16 == 0 (4-bit)"; return false; }
  return true;
}

bool bf_umma_supported(const bf_ctx *c, const char **why) {
  if (!bf_umma_shape_supported(c, why)) return false;
  // 33-64 beams on 32 antennas: the bin-per-lane kernel integrates any even nint >= 16 (bf_bl_shape)
  if (!nint_ok(c->nint) && !bf_bl_shape(c->dtype, BF_MODE_POWER, c->nant, c->nbeam, c->nint, c->nbin)) {
    *why = "needs nint a power of two or >= 16";
    return false;
  }
  return true;
}

// voltage-beam mode: the output (4 bytes per beam-sample) dominates the traffic; nint plays no role
template <int IN>
static cudaError_t launch_k64_beams(const BfParams &p, int sm_count, cudaStream_t st) {
  if (p.nMt == 1) return launch_k64<64, 1, 2, 8, 8, false, IN, true>(p, sm_count, st);
  if (p.nMt <= 2) return launch_k64<64, 2, 3, 4, 8, false, IN, true>(p, sm_count, st);
  return launch_k64<64, 4, 2, 2, 8, false, IN, true>(p, sm_count, st);
}

template <int IN>
static cudaError_t launch_k64_in(const BfParams &p, int sm_count, cudaStream_t st) {
  if (p.mode == BF_MODE_BEAMS) return launch_k64_beams<IN>(p, sm_count, st);
  switch (p.nint) {
    case 1: return launch_k64_nint<1, IN>(p, sm_count, st);
    case 2: return launch_k64_nint<2, IN>(p, sm_count, st);
    case 4: return launch_k64_nint<4, IN>(p, sm_count, st);
    case 8: return launch_k64_nint<8, IN>(p, sm_count, st);
    case 16: return launch_k64_nint<16, IN>(p, sm_count, st);
    case 32: return launch_k64_nint<32, IN>(p, sm_count, st);
    case 64: return launch_k64_nint<64, IN>(p, sm_count, st);
    default:
      if (p.nint < BF_LO_NINT) return cudaErrorNotSupported;   // bf_umma_supported lets no such shape through
      return launch_k64_nint<0, IN>(p, sm_count, st);          // any other length: atomic partial sums into zeroed powers
  }
}

cudaError_t bf_launch_umma(const BfParams &p, int dtype, int sm_count, cudaStream_t st) {
  const int v = umma_variant(dtype, p.nant);
  if (v == 2) return bf_launch_umma_kblock(p, dtype, sm_count, st);
  if (v != 1) return cudaErrorNotSupported;
  // 33-64 beams on 32 antennas, bins of an even number >= 16 of samples: the bin-per-lane kernel with the voltages in
  // tensor memory (bf_umma_bl.cu; sweep at 64 / 48 / 40 beams 0.168 / 0.151 / 0.146 -> 0.145 / 0.137 / 0.132 ms)
  if (bf_umma_bl_takes(p, dtype)) return bf_launch_umma_bl(p, dtype, sm_count, st);
  return dtype == BF_CI4 ? launch_k64_in<BF_CI4>(p, sm_count, st) : launch_k64_in<BF_CI8>(p, sm_count, st);
}
