// bf_umma_i8b.cu -- the int8-operand few-beam kernel with ONE OUTPUT BIN PER TMEM LANE (hot-path rows a2..a5,
// <= 32 beams, 32 antennas, complex int8 or 4+4-bit input, even nint).
//
// bf_umma_i8.cu puts TIME on the M axis of tcgen05.mma kind::i8 (so that TMEM holds only real beams) and then has
// to integrate ACROSS the lanes of a warp: a transposing butterfly of shuffles, selects and adds that costs as much
// as the detection itself (profiles/r02_roles.md, sweep-B32: 2723 epilogue instructions per 256 samples, of which
// FSEL + SHFL + FADD are 450 and the rest is six instructions per beam and sample).  Here the TMA engine does the
// transposition on the way in: the voltages are viewed as the tensor
//      { 128 bytes = two samples of 32 antennas,  1,  nbin,  nint / 2 rows per bin,  nchan }
// and a tile is the box {128, 1, 128, 1, 1}: row g of 128 CONSECUTIVE BINS.  Row r of the A operand (= TMEM lane r)
// therefore belongs to bin 128 sp + r in every one of the G = nint / 2 tiles of a super-tile, and the integration
// P[c][b][j] = sum_t |y|^2 is a plain running sum in the registers of the thread that owns the
// lane: no shuffle, no select, and the stores of a warp are 32 consecutive bins of one beam (128 bytes).
//   a3 contraction  as in bf_umma_i8.cu (WIDE form): four MMAs per tile slice the 128-byte rows along K, even
//                   sample -> accumulator E, odd sample -> accumulator O; two-limb 15-bit weights (A21)
//   a4 detection    re = 128 hi + lo (IMAD), I2F, then ONE packed FFMA2 squares (re, im) into a float2 running sum:
//                   five instructions per beam and sample
//   a5 integration  in registers over the G tiles, (x + y) * scale^2, one coalesced fp32 store per beam
// 4+4-bit input (row f1): the raw byte masked to its high nibble IS the int8 number 16 re, shifted
// left by four and masked it is 16 im; two PRMT interleave them -- five ALU instructions per four antennas turn a raw
// row of 128 bytes (four samples) into two int8 operand rows, which the same MMAs and the same epilogue consume
// (scale / 16).  Up to 16 beams the operand rows are written to TENSOR MEMORY (tcgen05.st) and the MMAs take their A
// operand from there; 17-32 beams keep shared-memory operand stages (no TMEM columns left).
//
// Warp roles (one persistent CTA per SM over a contiguous range of (channel, super-tile)): 4 * NSETS epilogue warps
// (sets of one warp per TMEM lane quadrant: column sets split the 8-beam chunks of a tile, tile sets take alternate
// tiles -- see b_csets / b_tsets), then one MMA-issuing warp (+ TMEM allocation), two TMA producer warps (tiles of even
// / odd index) and, for 4-bit input, four unpack warps.
#include <cuda.h>

#include "bf_internal.h"
#include "bf_tmap.h"
#include "ptx.cuh"

namespace {

constexpr int B_ROW_BYTES = 128;                       // one operand row: two samples x 32 antennas x (re, im)
constexpr int B_STAGE_BYTES = 128 * B_ROW_BYTES;       // 16 KiB: 128 bins x two samples
constexpr int B_W_ROW_BYTES = 64;                      // coefficient rows (bf_internal.h: int8 two-limb operand)
#ifndef B_WAIT_NS
#define B_WAIT_NS 400
#endif
constexpr int B_UNPACK_WARPS = 4;
// epilogue sets of four warps (one per TMEM lane quadrant): CS column sets split the 8-beam chunks of a tile, TS tile
// sets take alternate tiles of a super-tile (their partial sums meet in shared memory at its end).  A warp's work on
// a tile is one chain -- barrier, tcgen05.ld, 5 instructions per beam and sample -- of 300-400 clk whatever the beam
// count; with a single chunk (<= 8 beams) two tile sets keep up with 4-bit input (at 9-16 beams two column sets
// alone measured faster than 2 x 2 sets: fewer warps polling).
__host__ __device__ constexpr int b_csets(int ncol) { return ncol / 32 >= 4 ? 4 : (ncol / 32 >= 2 ? 2 : 1); }
__host__ __device__ constexpr int b_tsets(int ncol) { return ncol / 32 >= 2 ? 1 : 2; }
__host__ __device__ constexpr int b_nsets(int ncol) { return b_csets(ncol) * b_tsets(ncol); }

__host__ __device__ constexpr int b_ilog2(int x) { return x <= 1 ? 0 : 1 + b_ilog2(x >> 1); }

// unpack groups (4-bit input): groups of four warps on alternate raw tiles.  ONE: a second group (and likewise a second
// MMA-issuing warp) was measured and changes nothing (sweep-ci4, 8 beams: 0.0638 / 0.0646 / 0.0667 ms)
__host__ __device__ constexpr int b_ugroups(int ncol) { return 1; }
template <int NCOL, int IN> constexpr int i8b_threads_v = (4 * b_nsets(NCOL) + 3 + (IN == BF_CI4 ? B_UNPACK_WARPS * b_ugroups(NCOL) : 0)) * 32;

// NCOL: accumulator columns = 4 * beam capacity (32 / 64 / 128 -> 8 / 16 / 32 beams).  NST: operand stages (int8:
// filled by TMA; 4-bit: filled by the unpack warps from NRAW raw stages).
template <int NCOL, int NST, int NRAW, int IN>
__global__ void __launch_bounds__(i8b_threads_v<NCOL, IN>, 1)
bf_umma_i8b_kernel(const BfParams p, const __grid_constant__ CUtensorMap tmap, const long long total_super,
                   const int n_super_chan, const int G) {
  extern __shared__ uint8_t smem_raw[];
  constexpr bool CI4 = IN == BF_CI4;
  constexpr int W_BYTES = NCOL * B_W_ROW_BYTES;
  // ATM: 4-bit input up to 16 beams -- the unpacked int8 rows go to TENSOR MEMORY as the MMA's A operand (tcgen05.st,
  // 32 columns per operand tile) instead of shared memory: through shared memory every raw tile costs 96 KiB of
  // traffic (TMA write 16, LDS 16, STS 32, operand read 32) against the 128 B/clk an SM has, which capped the 4-bit
  // path at 0.55 of its HBM roofline whatever the beam count
  constexpr bool ATM = CI4 && NCOL <= 64;
  constexpr int NA = 4, A_COL0 = 384;                       // ATM: A-operand stages of 32 columns at 384 ..
  constexpr int NACC = ATM ? A_COL0 / (2 * NCOL) > 4 ? 4 : A_COL0 / (2 * NCOL) : 512 / (2 * NCOL);   // accumulator PAIRS (even, odd sample) in TMEM
  constexpr int NCH = NCOL / 32;                            // 8-beam column chunks
  constexpr int NSETS = b_nsets(NCOL), CS = b_csets(NCOL), TS = b_tsets(NCOL);
  static_assert(TS == 1 || NACC % TS == 0, "an accumulator slot must always belong to the same tile set");
  constexpr int B_MMA_WARP = 4 * NSETS, B_TMA_WARP = B_MMA_WARP + 1, B_UNPACK_WARP = B_MMA_WARP + 3;
  constexpr int CPS = NCH / CS;                             // chunks per column set
  constexpr int BPS = 128;                                  // bins per super-tile: one per TMEM lane
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t sW = smem_base;                            // 2 coefficient buffers
  const uint32_t sA = sW + 2 * W_BYTES;                     // NST operand stages (W_BYTES is a multiple of 1024)
  const uint32_t sR = sA + NST * B_STAGE_BYTES;             // NRAW raw stages (4-bit input)
  const uint32_t sX = sR + NRAW * B_STAGE_BYTES;            // tile-set exchange: [2][4 quadrants][CS][8 CPS][32 lanes] floats
  constexpr int X_BYTES = TS > 1 ? 2 * 4 * CS * 8 * CPS * 32 * 4 : 0;
  const uint32_t sBar = sX + X_BYTES;
  constexpr int NAB = NST > 4 ? NST : 4;                    // operand-stage barriers (smem stages or the four TMEM stages)
  const uint32_t bar_a_full = sBar, bar_a_empty = bar_a_full + 8 * NAB;
  const uint32_t bar_r_full = bar_a_empty + 8 * NAB, bar_r_empty = bar_r_full + 8 * (NRAW + 1);
  const uint32_t bar_w_full = bar_r_empty + 8 * (NRAW + 1), bar_w_empty = bar_w_full + 16;
  const uint32_t bar_t_full = bar_w_empty + 16, bar_t_empty = bar_t_full + 8 * NACC;
  const uint32_t s_tmem = bar_t_empty + 8 * NACC;

  const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0), lane = threadIdx.x & 31;

  if (threadIdx.x == 0) {
    // operand stage "full": one TMA transaction (int8) or the unpack warps (4-bit); "empty": the MMA's commit
    for (int s = 0; s < (ATM ? NA : NST); ++s) { mbar_init(bar_a_full + 8 * s, CI4 ? B_UNPACK_WARPS : 1); mbar_init(bar_a_empty + 8 * s, 1); }
    for (int s = 0; s < NRAW; ++s) { mbar_init(bar_r_full + 8 * s, 1); mbar_init(bar_r_empty + 8 * s, B_UNPACK_WARPS); }   // one group per stage
    for (int s = 0; s < 2; ++s) { mbar_init(bar_w_full + 8 * s, 1); mbar_init(bar_w_empty + 8 * s, 1); }
    for (int s = 0; s < NACC; ++s) { mbar_init(bar_t_full + 8 * s, 1); mbar_init(bar_t_empty + 8 * s, 4 * CS); }
    fence_barrier_init();
  }
  if (warp == B_MMA_WARP) tmem_alloc(s_tmem, 512);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  uint32_t tmem_base;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(s_tmem));
  tmem_base = __shfl_sync(0xffffffffu, tmem_base, 0);
  probe_mark(p.probe, 0);

  // this CTA's contiguous range of super-tiles (super-tile = 128 bins of one channel = G tiles; 4-bit input: G
  // raw tiles of four samples per bin, each unpacked into two operand tiles)
  const long long s0 = total_super * blockIdx.x / gridDim.x;
  const long long s1 = total_super * (blockIdx.x + 1) / gridDim.x;
  const int n_super = (int)(s1 - s0);
  const int c0 = (int)(s0 / n_super_chan), sp0 = (int)(s0 % n_super_chan);
  const int GT = CI4 ? 2 * G : G;                           // operand tiles per super-tile

  if (warp < 4 * NSETS) {
    // =========================================================================== epilogue
    const int quad = warp & 3, set = (warp >> 2) % CS, tset = (warp >> 2) / CS;
    const bool lane0 = lane == 0;
    // The kernel is bound by the instructions its sub-partitions issue (profiles/r02_ncu_full_summary.md: issue slots
    // 74-76 % busy at 16-32 beams), so the visit to an accumulator pair is kept lean: barrier and TMEM base addresses
    // live in registers, and everything that does not change inside a super-tile is hoisted out of its tile loop.
    uint32_t t_lane = tmem_base + ((uint32_t)(quad * 32) << 16) + set * (CPS * 32);
    uint32_t bt_full = bar_t_full;
    asm volatile("" : "+r"(t_lane), "+r"(bt_full));          // keep in registers, do not rematerialise
    const uint32_t xch = sX + (uint32_t)(((quad * CS + set) * 8 * CPS) * 32 + lane) * 4;   // + buffer, + 128 per value
    const int nbeam = p.nbeam, nbin = p.nbin;
    int c = c0, sp = sp0;
    int a = 0;                                              // accumulator pair of the next operand tile, parity of its "full"
    uint32_t apar = 0;
    for (int s = 0; s < n_super; ++s) {
      const int bin = BPS * sp + 32 * quad + lane;
      const bool live = BPS * sp + 32 * quad < nbin;  // warp-uniform: this quadrant holds real bins
      // requested now, used after the G tiles: a load at the END of the super-tile would stall every warp for a
      // DRAM round trip per super-tile
      const float sc = (float)p.i8scale[c] * (CI4 ? 0.0625f : 1.0f);         // 4-bit operands carry 16 x
      float2 acc[CPS][8];
#pragma unroll
      for (int k = 0; k < CPS; ++k)
#pragma unroll
        for (int i = 0; i < 8; ++i) acc[k][i] = make_float2(0.f, 0.f);
      for (int g = 0; g < GT; ++g) {
        const int a_ = a;
        const uint32_t apar_ = apar;
        if (++a == NACC) { a = 0; apar ^= 1; }
        // (by the parity of the accumulator slot = of the CTA's tile counter, NOT of g: a barrier must be seen in every
        // phase by the set that waits on it -- a parity wait cannot tell phase n from n + 2 -- and with an odd number of
        // tiles per super-tile g would hand a slot to the other set every other super-tile)
        if (TS > 1 && (a_ & (TS - 1)) != tset) continue;    // the other tile set's
        const uint32_t bf_a = bt_full + 8 * a_;             // "full" of this accumulator pair; its "empty" is NACC barriers on
        mbar_wait_hinted(bf_a, apar_, B_WAIT_NS);
        tc_fence_after();
        if (!live) {                                        // bins past the end of the channel (zero-filled rows)
          __syncwarp();
          if (lane0) mbar_arrive(bf_a + 8 * NACC);
          continue;
        }
        const uint32_t t_acc = t_lane + a_ * (2 * NCOL);
#pragma unroll
        for (int k = 0; k < CPS; ++k) {
          uint32_t v[32], u[32];
          BF_TMEM_LD_32x32b_X32(t_acc + 32 * k, v);          // even samples
          BF_TMEM_LD_32x32b_X32(t_acc + NCOL + 32 * k, u);   // odd samples
          tc_wait_ld();
          if (k == CPS - 1) {  // all of this warp's columns are in registers: hand the accumulator pair back
            tc_fence_before();
            __syncwarp();
            if (lane0) mbar_arrive(bf_a + 8 * NACC);
          }
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            const int re = ((int)v[4 * i] << 7) + (int)v[4 * i + 2];         // 128 hi + lo, exact
            const int im = ((int)v[4 * i + 1] << 7) + (int)v[4 * i + 3];
            const int ro = ((int)u[4 * i] << 7) + (int)u[4 * i + 2];
            const int io = ((int)u[4 * i + 1] << 7) + (int)u[4 * i + 3];
            const float2 e = make_float2((float)re, (float)im), o = make_float2((float)ro, (float)io);
            acc[k][i] = ffma2(e, e, acc[k][i]);
            acc[k][i] = ffma2(o, o, acc[k][i]);
          }
        }
      }
      if constexpr (TS > 1) {
        // tile set 1 hands its partial sums to tile set 0 of the same (quadrant, column set): double-buffered by
        // super-tile parity, one named barrier per pair of warps
        const uint32_t xb = xch + (uint32_t)(s & 1) * (X_BYTES / 2);
        if (tset == 1 && live) {
#pragma unroll
          for (int k = 0; k < CPS; ++k)
#pragma unroll
            for (int i = 0; i < 8; ++i)
              asm volatile("st.shared.f32 [%0], %1;" ::"r"(xb + (k * 8 + i) * 128), "f"(acc[k][i].x + acc[k][i].y) : "memory");
        }
        asm volatile("bar.sync %0, 64;" ::"r"(1 + quad * CS + set) : "memory");
        if (tset == 0 && live) {
#pragma unroll
          for (int k = 0; k < CPS; ++k)
#pragma unroll
            for (int i = 0; i < 8; ++i) {
              float o;
              asm volatile("ld.shared.f32 %0, [%1];" : "=f"(o) : "r"(xb + (k * 8 + i) * 128) : "memory");
              acc[k][i].x += o;
            }
        }
      }
      if (live && tset == 0) {
        const float sc2 = sc * sc;
        float *out = p.pow + (size_t)c * nbeam * nbin + bin;
        const bool writer = bin < nbin;
#pragma unroll
        for (int k = 0; k < CPS; ++k)
#pragma unroll
          for (int i = 0; i < 8; ++i) {
            const float tot = acc[k][i].x + acc[k][i].y;
            const int beam = 8 * (set * CPS + k) + i;
            if (writer && beam < nbeam) out[(size_t)beam * nbin] = tot * sc2;
          }
      }
      if (++sp == n_super_chan) { sp = 0; ++c; }
    }
  } else if (warp == B_MMA_WARP) {
    // =========================================================================== MMA issue
    constexpr uint32_t idesc = make_idesc_i8(128, NCOL);
    int c = c0, sp = sp0, prev_c = -1, wi = 0, wb = 0;
    int st = 0, a = 0;
    uint32_t st_par = 0, apar = 1;       // parities of a_full[st] / t_empty[a] to wait for
    constexpr int NSTG = ATM ? NA : NST;
    for (int s = 0; s < n_super; ++s) {
      if (c != prev_c) {
        if (wi > 0 && elect_one()) tc_commit(bar_w_empty + 8 * wb);   // my MMAs so far have left the old buffer
        prev_c = c;
        wb = wi & 1;
        mbar_wait(bar_w_full + 8 * wb, (uint32_t)((wi >> 1) & 1));
        ++wi;
      }
      const uint64_t bdesc = make_sdesc_k_sw64(sW + wb * W_BYTES);
      for (int g = 0; g < GT; ++g) {
        mbar_wait(bar_a_full + 8 * st, st_par);
        mbar_wait(bar_t_empty + 8 * a, apar);
        tc_fence_after();
        if (elect_one()) {
          const uint32_t d = tmem_base + a * 2 * NCOL;
          if constexpr (ATM) {           // A operand in tensor memory: 8 columns per 32 bytes of the row
            const uint32_t at = tmem_base + A_COL0 + st * 32;
            mma_i8_ts(d, at, bdesc, idesc, 0);
            mma_i8_ts(d, at + 8, bdesc + 2, idesc, 1);
            mma_i8_ts(d + NCOL, at + 16, bdesc, idesc, 0);
            mma_i8_ts(d + NCOL, at + 24, bdesc + 2, idesc, 1);
          } else {
            const uint64_t adesc = make_sdesc_k_sw128(sA + st * B_STAGE_BYTES);
            mma_i8_ss(d, adesc, bdesc, idesc, 0);                  // even sample: row bytes 0..31
            mma_i8_ss(d, adesc + 2, bdesc + 2, idesc, 1);          //              row bytes 32..63
            mma_i8_ss(d + NCOL, adesc + 4, bdesc, idesc, 0);       // odd sample:  row bytes 64..95
            mma_i8_ss(d + NCOL, adesc + 6, bdesc + 2, idesc, 1);   //              row bytes 96..127
          }
          tc_commit(bar_t_full + 8 * a);
          tc_commit(bar_a_empty + 8 * st);
        }
        __syncwarp();
        if (++st == NSTG) { st = 0; st_par ^= 1; }
        if (++a == NACC) { a = 0; apar ^= 1; }
      }
      if (++sp == n_super_chan) { sp = 0; ++c; }
    }
  } else if (warp == B_TMA_WARP || warp == B_TMA_WARP + 1) {
    // =========================================================================== TMA producers (two warps)
    // lane 0 of producer j issues the tiles of parity j; producer 0 also brings in the coefficients.  int8: the
    // tiles are the operand stages themselves; 4-bit: raw stages for the unpack warps.
    const int pj = warp - B_TMA_WARP;
    constexpr int NRING = CI4 ? NRAW : NST;
    static_assert(NRING % 2 == 0, "stages are dealt to the producers by parity");
    const uint32_t ring = CI4 ? sR : sA, full = CI4 ? bar_r_full : bar_a_full, empty = CI4 ? bar_r_empty : bar_a_empty;
    if (lane == 0) tma_prefetch_desc(&tmap);
    int c = c0, sp = sp0, prev_c = -1, wi = 0;
    int ti = 0, st = pj;
    uint32_t st_par = 1;                 // parity of empty[st] to wait for (passes on the fresh barrier)
    // (A tile takes 128 bytes out of every bin, so the G tiles of a super-tile cover one contiguous region only
    // together, over the super-tile's whole duration: from DRAM the strided copies run at 5.9 instead of 6.3 TB/s,
    // while from a resident L2 they are FASTER than contiguous ones.  Prefetching the next super-tile's region into
    // the L2 -- cp.async.bulk.prefetch.L2 or prefetch.global.L2 from this warp -- was measured and is 2-5 % slower.)
    for (int s = 0; s < n_super; ++s) {
      if (c != prev_c) {
        prev_c = c;
        if (pj == 0 && lane == 0) {
          const int wb = wi & 1;
          mbar_wait(bar_w_empty + 8 * wb, (uint32_t)(((wi >> 1) & 1) ^ 1));
          mbar_arrive_expect_tx(bar_w_full + 8 * wb, W_BYTES);
          bulk_g2s(sW + wb * W_BYTES, reinterpret_cast<const char *>(p.wop8) + (size_t)c * W_BYTES, W_BYTES, bar_w_full + 8 * wb);
        }
        ++wi;
      }
      for (int g = 0; g < G; ++g, ++ti) {
        if ((ti & 1) != pj) continue;
        if (lane == 0) {
          mbar_wait(empty + 8 * st, st_par);
          mbar_arrive_expect_tx(full + 8 * st, B_STAGE_BYTES);
          tma_load_5d(ring + st * B_STAGE_BYTES, &tmap, 0, 0, BPS * sp, g, c, full + 8 * st);   // row g of bins BPS sp ..
        }
        __syncwarp();
        if ((st += 2) >= NRING) { st -= NRING; st_par ^= 1; }
      }
      if (++sp == n_super_chan) { sp = 0; ++c; }
    }
  } else if (ATM && warp >= B_UNPACK_WARP) {
    // =========================================================================== unpack into TENSOR MEMORY (4-bit input, <= 16 beams)
    // Thread (quadrant, lane) owns raw row r = 32 quadrant + lane (the four unpack warps cover the four quadrants):
    // 128 bytes = FOUR samples of 32 antennas.  Samples 0, 1 become row r of operand tile 2 i, samples 2, 3 of tile
    // 2 i + 1: 32 TMEM columns each, written with one tcgen05.st.32x32b.x32 -- the int8 operands never touch shared
    // memory.  Per raw word (four antennas): mask = 16 re, shift + mask = 16 im, two PRMT interleave (re, im).
    constexpr int UG = b_ugroups(NCOL);   // groups of four warps on alternate raw tiles: a tile's unpack is one chain
    static_assert(NRAW % UG == 0 && NA % (2 * UG) == 0, "stages are dealt to the unpack groups");
    const int quad = warp & 3, grp = (warp - B_UNPACK_WARP) >> 2;
    const int r = 32 * quad + lane;
    const uint32_t t_row = tmem_base + ((uint32_t)(quad * 32) << 16) + A_COL0;
    const uint32_t row_off = (uint32_t)r * 128u, sw = (uint32_t)(r & 7);
    int rs = grp, as = 2 * grp;           // group j: raw tiles j, j + UG, .. -> raw stage i % NRAW, operand stages 2 i % NA, + 1
    uint32_t rpar = 0, apar = 1;
    const int n_raw = n_super * G;
    for (int i = grp; i < n_raw; i += UG) {
      mbar_wait(bar_r_full + 8 * rs, rpar);
      const uint32_t src = sR + rs * B_STAGE_BYTES + row_off;
      uint4 x[8];
#pragma unroll
      for (int j = 0; j < 8; ++j)       // the raw stage is 128-byte swizzled by TMA
        asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(x[j].x), "=r"(x[j].y), "=r"(x[j].z), "=r"(x[j].w)
                     : "r"(src + (((uint32_t)j ^ sw) << 4)));
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        uint32_t o[32];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const uint32_t w[4] = {x[4 * h + j].x, x[4 * h + j].y, x[4 * h + j].z, x[4 * h + j].w};
#pragma unroll
          for (int m = 0; m < 4; ++m) {
            const uint32_t hi = w[m] & 0xF0F0F0F0u;             // 16 re of four antennas
            const uint32_t lo = (w[m] << 4) & 0xF0F0F0F0u;      // 16 im
            o[8 * j + 2 * m] = __byte_perm(hi, lo, 0x5140);     // (re0, im0, re1, im1)
            o[8 * j + 2 * m + 1] = __byte_perm(hi, lo, 0x7362); // (re2, im2, re3, im3)
          }
        }
        if (h == 1) {  // the whole raw row has been consumed: the stage may be refilled
          __syncwarp();
          if (lane == 0) mbar_arrive(bar_r_empty + 8 * rs);
        }
        mbar_wait(bar_a_empty + 8 * (as + h), apar);
        tc_fence_after();
        BF_TMEM_ST_32x32b_X32(t_row + (as + h) * 32, o);
      }
      tc_wait_st();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) {
        mbar_arrive(bar_a_full + 8 * as);
        mbar_arrive(bar_a_full + 8 * (as + 1));
      }
      if ((rs += UG) >= NRAW) { rs -= NRAW; rpar ^= 1; }
      if ((as += 2 * UG) >= NA) { as -= NA; apar ^= 1; }
    }
  } else if (CI4 && warp >= B_UNPACK_WARP) {
    // =========================================================================== unpack (4-bit input, UG groups of 4 warps)
    // A raw row is 128 bytes = FOUR samples of 32 antennas (high nibble re, low nibble im).  Masked
    // to the high nibbles a byte is the int8 number 16 re, shifted left by four it is 16 im; PRMT interleaves the
    // two into (re, im) byte pairs.  Samples 0, 1 of every row go to operand tile 2r, samples 2, 3 to tile 2r+1.
    // Thread t of a group's 128 handles the 16-byte piece t & 7 of rows (t >> 3) + 16 k: piece q holds the antennas
    // 16 (q & 1) .. of sample q >> 1, i.e. 32 bytes of operand row at byte 64 (q >> 1 & 1) + 32 (q & 1) of tile q >> 2.
    constexpr int UG = b_ugroups(NCOL);
    static_assert(NRAW % UG == 0, "raw stages are dealt to the unpack groups");
    const int grp = (warp - B_UNPACK_WARP) >> 2;
    const int ut = ((warp - B_UNPACK_WARP) & 3) * 32 + lane;
    const int q = ut & 7, r0 = ut >> 3;
    const uint32_t src0 = (uint32_t)(r0 * 128 + ((q ^ (r0 & 7)) << 4));              // raw stage is 128-byte swizzled by TMA
    const uint32_t ch0 = (uint32_t)(4 * ((q >> 1) & 1) + 2 * (q & 1));               // first 16-byte chunk of the output
    const uint32_t dst0 = (uint32_t)(r0 * 128 + ((ch0 ^ (r0 & 7)) << 4));            // second chunk: ^ 16
    const uint32_t tsel = (uint32_t)(q >> 2);
    int rs = grp, st = 2 * grp;            // group j: raw tiles j, j + UG, .. -> raw stage i % NRAW, operand stages 2 i % NST, + 1
    uint32_t rpar = 0, spar = 1;
    const int n_raw = n_super * G;
    for (int i = grp; i < n_raw; i += UG) {
      mbar_wait(bar_r_full + 8 * rs, rpar);
      uint4 x[8];
#pragma unroll
      for (int k = 0; k < 8; ++k)   // rows r0 + 16 k: the swizzle term (row & 7) is the same for all of them
        asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(x[k].x), "=r"(x[k].y), "=r"(x[k].z), "=r"(x[k].w)
                     : "r"(sR + rs * B_STAGE_BYTES + src0 + k * 2048));
      // both operand tiles of this raw tile must be free
      const int st1 = st + 1 == NST ? 0 : st + 1;
      const uint32_t spar1 = st + 1 == NST ? spar ^ 1 : spar;
      mbar_wait(bar_a_empty + 8 * st, spar);
      mbar_wait(bar_a_empty + 8 * st1, spar1);
      const uint32_t dst = sA + (tsel ? st1 : st) * B_STAGE_BYTES + dst0;
#pragma unroll
      for (int k = 0; k < 8; ++k) {
        const uint32_t w[4] = {x[k].x, x[k].y, x[k].z, x[k].w};
        uint32_t o[8];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          const uint32_t hi = w[j] & 0xF0F0F0F0u;             // 16 re of four antennas
          const uint32_t lo = (w[j] << 4) & 0xF0F0F0F0u;      // 16 im
          o[2 * j] = __byte_perm(hi, lo, 0x5140);             // (re0, im0, re1, im1)
          o[2 * j + 1] = __byte_perm(hi, lo, 0x7362);         // (re2, im2, re3, im3)
        }
        asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"(dst + k * 2048), "r"(o[0]), "r"(o[1]), "r"(o[2]), "r"(o[3]) : "memory");
        asm volatile("st.shared.v4.b32 [%0], {%1,%2,%3,%4};" ::"r"((dst ^ 16u) + k * 2048), "r"(o[4]), "r"(o[5]), "r"(o[6]), "r"(o[7]) : "memory");
      }
      fence_proxy_async_smem();
      __syncwarp();
      if (lane == 0) {
        mbar_arrive(bar_r_empty + 8 * rs);
        mbar_arrive(bar_a_full + 8 * st);
        mbar_arrive(bar_a_full + 8 * st1);
      }
      if ((rs += UG) >= NRAW) { rs -= NRAW; rpar ^= 1; }
      if ((st += 2 * UG) >= NST) { st -= NST; spar ^= 1; }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == B_MMA_WARP) tmem_dealloc(tmem_base, 512);
  probe_mark(p.probe, 1);
}

// 4-D view of one launch's voltages: {128 bytes, rows per bin, nbin, nchan}; box {128, 1, 128, 1}, 128-byte swizzle.
// A row is two int8 samples (rows per bin = nint / 2) or four 4-bit samples (nint / 4); bins past nbin are zero-filled.
template <int IN>
cudaError_t make_tmap_bins(CUtensorMap *tm, const BfParams &p, int nint) {
  PFN_encodeTiled enc = bf_get_encode();
  if (!enc) return cudaErrorNotSupported;
  const int spr = IN == BF_CI4 ? 4 : 2;                                 // samples per 128-byte row
  const cuuint64_t chan_bytes = (cuuint64_t)p.nsamp * (128 / spr);
  // {byte in row, 1, bin, row in bin, channel}: a tile = row g of 128 consecutive bins
  cuuint64_t dims[5] = {128, 1, (cuuint64_t)p.nbin, (cuuint64_t)(nint / spr), (cuuint64_t)p.nchan_run};
  cuuint64_t strides[4] = {128, (cuuint64_t)nint * (128 / spr), 128, chan_bytes};
  cuuint32_t box[5] = {128, 1, 128, 1, 1};
  cuuint32_t estr[5] = {1, 1, 1, 1, 1};
  CUresult r = enc(tm, CU_TENSOR_MAP_DATA_TYPE_UINT8, 5, const_cast<void *>(p.volt), dims, strides, box, estr,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

template <int NCOL, int IN>
cudaError_t launch_i8b(const BfParams &p, int sm_count, cudaStream_t st) {
  constexpr bool CI4 = IN == BF_CI4, ATM = CI4 && NCOL <= 64;   // ATM: operands in tensor memory, no shared-memory operand stages
  constexpr int NST = ATM ? 0 : (CI4 ? 6 : 12), NRAW = ATM ? 12 : (CI4 ? 6 : 0);
  CUtensorMap tm;
  cudaError_t e = bf_cached_tmap(&tm, p, CI4 ? 21 : 11, p.nint, make_tmap_bins<IN>);
  if (e != cudaSuccess) return e;
  const int G = p.nint / (CI4 ? 4 : 2);           // raw rows per bin
  const int n_super_chan = (p.nbin + 127) / 128;
  const long long total = (long long)p.nchan_run * n_super_chan;
  constexpr int X_BYTES = b_tsets(NCOL) > 1 ? 2 * 4 * 8 * (NCOL / 32) * 32 * 4 : 0;   // tile-set exchange buffers
  const size_t smem = 1024 + 2 * NCOL * B_W_ROW_BYTES + (size_t)(NST + NRAW) * B_STAGE_BYTES + X_BYTES + 1024;
  auto kern = bf_umma_i8b_kernel<NCOL, NST, NRAW, IN>;
  static thread_local int attr_dev = -1;   // once per instantiation and device
  if ((e = bf_set_smem_once(kern, smem, &attr_dev)) != cudaSuccess) return e;
  const int grid = (int)(total < sm_count ? total : sm_count);
  kern<<<grid, i8b_threads_v<NCOL, IN>, smem, st>>>(p, tm, total, n_super_chan, G);
  return cudaGetLastError();
}

// (Tiles with two / four lanes per bin -- chunks of 256 / 512 contiguous bytes, one / two shuffle-adds per beam at the end
// of a super-tile -- were measured on the sweep and are slower at every beam count, 32 beams: 0.117 / 0.156 / 0.237 ms for
// 1 / 2 / 4 lanes per bin; DESIGN.md 5.3d.  Only one lane per bin is built.)

}  // namespace

// Shapes this kernel takes (the caller has checked int8 / 4-bit input, nant % 8 == 0, <= 32 beams): 32 antennas,
// nint a multiple of the samples per 128-byte row, and enough bins that the 128 lanes of a super-tile are not
// mostly padding (a channel's last super-tile is partial: at most a fifth wasted).
bool bf_umma_i8b_takes(const BfParams &p, int dtype) {
  if (p.mode != BF_MODE_POWER || p.nant != 32) return false;
  if (p.nint % (dtype == BF_CI4 ? 4 : 2) != 0) return false;
  if ((long long)p.nint * 64 >= (1ll << 32)) return false;
  return p.nbin % 128 == 0 || p.nbin >= 512;
}

cudaError_t bf_launch_umma_i8b(const BfParams &p, int dtype, int sm_count, cudaStream_t st) {
  if (dtype == BF_CI4) {
    if (p.nbeam <= 8) return launch_i8b<32, BF_CI4>(p, sm_count, st);
    if (p.nbeam <= 16) return launch_i8b<64, BF_CI4>(p, sm_count, st);
    return launch_i8b<128, BF_CI4>(p, sm_count, st);
  }
  if (p.nbeam <= 8) return launch_i8b<32, BF_CI8>(p, sm_count, st);
  if (p.nbeam <= 16) return launch_i8b<64, BF_CI8>(p, sm_count, st);
  return launch_i8b<128, BF_CI8>(p, sm_count, st);
}
