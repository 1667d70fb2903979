// bf_simt.cu -- generic CUDA-core beamformer (any nant / nbeam / nint, both dtypes).
//
// Structure is the paper's Algorithm 1 with beams and time swapped to suit the
// fused power + integration epilogue: a block owns one channel, 128 beams (one per thread) and a
// bin-aligned time range; antennas are processed in groups, the group's coefficients are loaded
// cooperatively into shared memory ("Cooperatively load coefficients subset and store in coeffs",
// PAPER.md:79), and every thread keeps register accumulators ("local beam accumulators",
// PAPER.md:73) -- here one complex accumulator per time sample of the pass.  |y|^2 and the sum over
// nint happen in registers, so complex beams never reach HBM.
// This is the fall-back for shapes the tensor-core kernel does not take, and the cross-check for it.
#include "bf_internal.h"

#define SIMT_TT 16   // time samples per pass (complex accumulators per thread)
#define SIMT_NC 16   // antennas per shared-memory group
#define SIMT_BEAMS 128

template <int DTYPE>
__device__ __forceinline__ float2 load_volt(const void *volt, size_t idx) {
  if (DTYPE == BF_CI8) {
    char2 v = reinterpret_cast<const char2 *>(volt)[idx];
    return make_float2((float)v.x, (float)v.y);
  } else if (DTYPE == BF_CI4) {  // 4+4-bit two's complement, high nibble real
    const int b = reinterpret_cast<const unsigned char *>(volt)[idx];
    return make_float2((float)(((b >> 4) ^ 8) - 8), (float)(((b & 15) ^ 8) - 8));
  } else {
    __half2 v = reinterpret_cast<const __half2 *>(volt)[idx];
    return __half22float2(v);
  }
}

template <int DTYPE, bool BEAMS>
__global__ void __launch_bounds__(SIMT_BEAMS) bf_simt_kernel(BfParams p, int samples_per_block) {
  __shared__ float2 Ws[SIMT_NC][SIMT_BEAMS + 1];
  __shared__ float2 Xs[SIMT_TT][SIMT_NC];
  const int tid = threadIdx.x;
  const int c = blockIdx.z;
  const int b0 = blockIdx.y * SIMT_BEAMS;
  const int b = b0 + tid;
  const int t_begin = blockIdx.x * samples_per_block;
  const int t_end = min(p.nsamp, t_begin + samples_per_block);
  const size_t wop_chan = (size_t)p.nMt * p.nKb * BF_TILE_ROWS * BF_KBLOCK;
  const __half *wc = p.wop + (size_t)c * wop_chan;
  const __half *wl = p.wop_lo ? p.wop_lo + (size_t)c * wop_chan : nullptr;   // second coefficient term (BF_LO_NINT)
  float binacc = 0.f;
  for (int t0 = t_begin; t0 < t_end; t0 += SIMT_TT) {
    float2 acc[SIMT_TT];
#pragma unroll
    for (int t = 0; t < SIMT_TT; ++t) acc[t] = make_float2(0.f, 0.f);
    for (int n0 = 0; n0 < p.nant; n0 += SIMT_NC) {
      __syncthreads();
      for (int i = tid; i < SIMT_TT * SIMT_NC; i += SIMT_BEAMS) {
        int t = i / SIMT_NC, n = i % SIMT_NC;
        float2 x = make_float2(0.f, 0.f);
        if (t0 + t < t_end && n0 + n < p.nant)
          x = load_volt<DTYPE>(p.volt, ((size_t)c * p.nsamp + (t0 + t)) * p.nant + (n0 + n));
        Xs[t][n] = x;
      }
      for (int i = tid; i < SIMT_NC * SIMT_BEAMS; i += SIMT_BEAMS) {
        int bl = i / SIMT_NC, n = i % SIMT_NC;
        int bb = b0 + bl, nn = n0 + n;
        float2 w = make_float2(0.f, 0.f);
        if (bb < p.nbeam && nn < p.nant) {
          int mt = bb / BF_TILE_BEAMS, bt = bb % BF_TILE_BEAMS;
          int kb = (2 * nn) / BF_KBLOCK, kk = (2 * nn) % BF_KBLOCK;
          size_t base = ((size_t)mt * p.nKb + kb) * (BF_TILE_ROWS * BF_KBLOCK);
          w.x = __half2float(wc[base + bf_tile_off(bf_beam_row(bt, 0), kk)]);
          w.y = __half2float(wc[base + bf_tile_off(bf_beam_row(bt, 1), kk)]);
          if (wl) {
            w.x += __half2float(wl[base + bf_tile_off(bf_beam_row(bt, 0), kk)]);
            w.y += __half2float(wl[base + bf_tile_off(bf_beam_row(bt, 1), kk)]);
          }
        }
        Ws[n][bl] = w;
      }
      __syncthreads();
#pragma unroll 4
      for (int n = 0; n < SIMT_NC; ++n) {
        float2 w = Ws[n][tid];
#pragma unroll
        for (int t = 0; t < SIMT_TT; ++t) {
          float2 x = Xs[t][n];
          acc[t].x = fmaf(w.x, x.x, acc[t].x);
          acc[t].x = fmaf(-w.y, x.y, acc[t].x);
          acc[t].y = fmaf(w.x, x.y, acc[t].y);
          acc[t].y = fmaf(w.y, x.x, acc[t].y);
        }
      }
    }
#pragma unroll
    for (int t = 0; t < SIMT_TT; ++t) {
      int tt = t0 + t;
      if (BEAMS) {  // voltage-beam mode (row f4): y itself as fp16 (re, im)
        if (tt < t_end && b < p.nbeam)
          reinterpret_cast<__half2 *>(p.beams)[((size_t)c * p.nbeam + b) * p.nsamp + tt] =
              __floats2half2_rn(acc[t].x * p.beam_scale, acc[t].y * p.beam_scale);
      } else if (tt < t_end) {
        binacc = fmaf(acc[t].x, acc[t].x, binacc);
        binacc = fmaf(acc[t].y, acc[t].y, binacc);
        if ((tt + 1) % p.nint == 0) {
          if (b < p.nbeam) p.pow[((size_t)c * p.nbeam + b) * p.nbin + tt / p.nint] = binacc;
          binacc = 0.f;
        }
      }
    }
  }
}

cudaError_t bf_launch_simt(const BfParams &p, int dtype, cudaStream_t st) {
  // bin-aligned time range per block, about 512 samples
  int bins_per_block = p.nint >= 512 ? 1 : 512 / p.nint;
  int samples_per_block = bins_per_block * p.nint;
  dim3 grid((p.nsamp + samples_per_block - 1) / samples_per_block, (p.nbeam + SIMT_BEAMS - 1) / SIMT_BEAMS,
            p.nchan_run);
  if (grid.z > 65535 || grid.y > 65535) return cudaErrorInvalidConfiguration;
  if (p.mode == BF_MODE_BEAMS) {
    if (dtype == BF_CI8)      bf_simt_kernel<BF_CI8, true><<<grid, SIMT_BEAMS, 0, st>>>(p, samples_per_block);
    else if (dtype == BF_CI4) bf_simt_kernel<BF_CI4, true><<<grid, SIMT_BEAMS, 0, st>>>(p, samples_per_block);
    else                      bf_simt_kernel<BF_CF16, true><<<grid, SIMT_BEAMS, 0, st>>>(p, samples_per_block);
  } else if (dtype == BF_CI8) bf_simt_kernel<BF_CI8, false><<<grid, SIMT_BEAMS, 0, st>>>(p, samples_per_block);
  else if (dtype == BF_CI4)   bf_simt_kernel<BF_CI4, false><<<grid, SIMT_BEAMS, 0, st>>>(p, samples_per_block);
  else                        bf_simt_kernel<BF_CF16, false><<<grid, SIMT_BEAMS, 0, st>>>(p, samples_per_block);
  return cudaGetLastError();
}
