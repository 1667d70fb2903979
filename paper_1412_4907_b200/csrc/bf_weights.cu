// bf_weights.cu -- phase-weight generator (hot-path row a1).
//
// W[c][b][n] = exp(-i 2 pi f_c/c0 (r_n . s_b)): the steering factor e^{-i k0.r_n} of Eq. 1
// (PAPER.md:23-28).  The paper computes the coefficients on the CPU between pipeline iterations
// (PAPER.md:220); here one kernel writes them straight into the tensor-core operand layout
// (bf_internal.h).  The phase in turns is formed and range-reduced in fp64 -- at 408 MHz over a
// 310 m array it is ~200 turns, so an fp32 phase would already cost 6e-5 of the 1e-3 budget --
// then sincospi, then one rounding to fp16.
#include "bf_internal.h"

#define BF_C0 299792458.0

// W'[c][b][n] = g[c][n] e^{-i 2 pi f_c/c0 (r_n . s_b)} in fp64
__device__ __forceinline__ void steering_weight(const double *__restrict__ ant, const double *__restrict__ freq,
                                                const double *__restrict__ dir, const double *__restrict__ gain,
                                                int nant, int c, int b, int n, double &wre, double &wim) {
  double dot = ant[3 * n] * dir[3 * b] + ant[3 * n + 1] * dir[3 * b + 1] + ant[3 * n + 2] * dir[3 * b + 2];
  double turns = freq[c] * dot / BF_C0;
  turns -= rint(turns);  // |turns| <= 1/2: exact subtraction, no accuracy lost to the big phase
  double s, co;
  sincospi(2.0 * turns, &s, &co);
  wre = co; wim = -s;  // e^{-i phi}
  if (gain) {  // W' = g W: antenna mask / gain calibration folded into the coefficients
    const double gre = gain[2 * ((size_t)c * nant + n)], gim = gain[2 * ((size_t)c * nant + n) + 1];
    const double tre = gre * wre - gim * wim, tim = gre * wim + gim * wre;
    wre = tre; wim = tim;
  }
}

__global__ void bf_weights_kernel(const double *__restrict__ ant, const double *__restrict__ freq,
                                  const double *__restrict__ dir, const double *__restrict__ gain,
                                  __half *__restrict__ wop, __half *__restrict__ wop_lo, int nant,
                                  int nchan, int nbeam, int nMt, int nKb) {
  // one thread per (chan, mt, row, n-slot) where n-slot covers the padded K' / 2
  const int npad = nKb * (BF_KBLOCK / 2);
  long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  long long total = (long long)nchan * nMt * BF_TILE_ROWS * npad;
  if (idx >= total) return;
  int n = (int)(idx % npad);
  long long t = idx / npad;
  int r = (int)(t % BF_TILE_ROWS);
  t /= BF_TILE_ROWS;
  int mt = (int)(t % nMt);
  int c = (int)(t / nMt);
  int b = bf_row_beam(mt, r);
  int part = bf_row_part(r);
  double a0 = 0.0, a1 = 0.0;
  if (b < nbeam && n < nant) {
    double wre, wim;
    steering_weight(ant, freq, dir, gain, nant, c, b, n, wre, wim);
    if (part == 0) { a0 = wre; a1 = -wim; }
    else           { a0 = wim; a1 = wre; }
  }
  int kb = (2 * n) / BF_KBLOCK, kk = (2 * n) % BF_KBLOCK;
  size_t o = (((size_t)c * nMt + mt) * nKb + kb) * (BF_TILE_ROWS * BF_KBLOCK) + bf_tile_off(r, kk);
  const __half2 hi = __floats2half2_rn((float)a0, (float)a1);
  *reinterpret_cast<__half2 *>(wop + o) = hi;
  if (wop_lo)  // the rounding residual as a second fp16 term (bf_internal.h, BF_LO_NINT)
    *reinterpret_cast<__half2 *>(wop_lo + o) =
        __floats2half2_rn((float)(a0 - (double)__low2float(hi)), (float)(a1 - (double)__high2float(hi)));
}

// the same weights as two int8 limbs in the bf_umma_i8.cu operand layout (bf_internal.h); one thread per
// (chan, row, antenna slot 0..31)
__global__ void bf_weights_i8_kernel(const double *__restrict__ ant, const double *__restrict__ freq,
                                     const double *__restrict__ dir, const double *__restrict__ gain,
                                     const double *__restrict__ scale, signed char *__restrict__ wop8, int nant,
                                     int nchan, int nbeam, int ncol) {
  long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  long long total = (long long)nchan * ncol * 32;
  if (idx >= total) return;
  const int n = (int)(idx & 31);
  const int row = (int)((idx >> 5) % ncol);
  const int c = (int)((idx >> 5) / ncol);
  const int b = 8 * (row >> 5) + ((row & 31) >> 2), j = row & 3;   // j: 0 re-hi, 1 im-hi, 2 re-lo, 3 im-lo
  int l0 = 0, l1 = 0;
  if (b < nbeam && n < nant) {
    double wre, wim;
    steering_weight(ant, freq, dir, gain, nant, c, b, n, wre, wim);
    const double a0 = (j & 1) ? wim : wre, a1 = (j & 1) ? wre : -wim;   // coefficients of x_re, x_im
    const int q0 = (int)rint(a0 / scale[c]), q1 = (int)rint(a1 / scale[c]);
    const int h0 = (q0 + 64) >> 7, h1 = (q1 + 64) >> 7;                 // floor((q + 64) / 128)
    l0 = (j & 2) ? q0 - 128 * h0 : h0;
    l1 = (j & 2) ? q1 - 128 * h1 : h1;
  }
  const int k = 2 * n;                                                  // byte position inside the 64-byte row
  const size_t o = ((size_t)c * ncol + row) * 64 + ((((k >> 4) ^ ((row >> 1) & 3)) << 4) | (k & 15));
  *reinterpret_cast<char2 *>(wop8 + o) = make_char2((signed char)l0, (signed char)l1);
}

cudaError_t bf_launch_weights(const bf_ctx *c, cudaStream_t st) {
  long long total = (long long)c->nchan * c->nMt * BF_TILE_ROWS * c->nKb * (BF_KBLOCK / 2);
  int threads = 256;
  long long blocks = (total + threads - 1) / threads;
  bf_weights_kernel<<<(unsigned)blocks, threads, 0, st>>>(c->d_ant, c->d_freq, c->d_dir,
                                                          c->have_gains ? c->d_gain : nullptr, c->d_wop, c->d_wop_lo, c->nant,
                                                          c->nchan, c->nbeam, c->nMt, c->nKb);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess || !c->d_wop8) return e;
  const int ncol = bf_i8_ncol(c->nbeam);
  total = (long long)c->nchan * ncol * 32;
  blocks = (total + threads - 1) / threads;
  bf_weights_i8_kernel<<<(unsigned)blocks, threads, 0, st>>>(c->d_ant, c->d_freq, c->d_dir,
                                                             c->have_gains ? c->d_gain : nullptr, c->d_i8scale,
                                                             c->d_wop8, c->nant, c->nchan, c->nbeam, ncol);
  return cudaGetLastError();
}

// operand layout -> logical fp32 [chan][beam][ant][2] (for bf_get_weights)
__global__ void bf_decode_weights_kernel(const __half *__restrict__ wop, const __half *__restrict__ wop_lo,
                                         float *__restrict__ out, int nant,
                                         int nchan, int nbeam, int nMt, int nKb) {
  long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  long long total = (long long)nchan * nbeam * nant;
  if (idx >= total) return;
  int n = (int)(idx % nant);
  long long t = idx / nant;
  int b = (int)(t % nbeam);
  int c = (int)(t / nbeam);
  int mt = b / BF_TILE_BEAMS, bl = b % BF_TILE_BEAMS;
  int kb = (2 * n) / BF_KBLOCK, kk = (2 * n) % BF_KBLOCK;
  size_t base = (((size_t)c * nMt + mt) * nKb + kb) * (BF_TILE_ROWS * BF_KBLOCK);
  float wre = __half2float(wop[base + bf_tile_off(bf_beam_row(bl, 0), kk)]);
  float wim = __half2float(wop[base + bf_tile_off(bf_beam_row(bl, 1), kk)]);
  if (wop_lo) {
    wre += __half2float(wop_lo[base + bf_tile_off(bf_beam_row(bl, 0), kk)]);
    wim += __half2float(wop_lo[base + bf_tile_off(bf_beam_row(bl, 1), kk)]);
  }
  out[2 * idx] = wre;
  out[2 * idx + 1] = wim;
}

// int8 two-limb operand -> logical fp32 [chan][beam][ant][2]
__global__ void bf_decode_weights_i8_kernel(const signed char *__restrict__ wop8, const double *__restrict__ scale,
                                            float *__restrict__ out, int nant, int nchan, int nbeam, int ncol) {
  long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  long long total = (long long)nchan * nbeam * nant;
  if (idx >= total) return;
  int n = (int)(idx % nant);
  long long t = idx / nant;
  int b = (int)(t % nbeam);
  int c = (int)(t / nbeam);
  const int row0 = 32 * (b >> 3) + 4 * (b & 7), k = 2 * n;
  auto at = [&](int row) { return (int)wop8[((size_t)c * ncol + row) * 64 + ((((k >> 4) ^ ((row >> 1) & 3)) << 4) | (k & 15))]; };
  // coefficient of x_re in the re row is W_re, in the im row W_im
  out[2 * idx] = (float)((128 * at(row0) + at(row0 + 2)) * scale[c]);
  out[2 * idx + 1] = (float)((128 * at(row0 + 1) + at(row0 + 3)) * scale[c]);
}

cudaError_t bf_launch_decode_weights(const bf_ctx *c, float *d_out, bool int8_operand, cudaStream_t st) {
  long long total = (long long)c->nchan * c->nbeam * c->nant;
  int threads = 256;
  long long blocks = (total + threads - 1) / threads;
  if (int8_operand && c->d_wop8) {
    // the int8 kernel is the one bf_run launches: report ITS operand
    bf_decode_weights_i8_kernel<<<(unsigned)blocks, threads, 0, st>>>(c->d_wop8, c->d_i8scale, d_out, c->nant, c->nchan,
                                                                      c->nbeam, bf_i8_ncol(c->nbeam));
    return cudaGetLastError();
  }
  bf_decode_weights_kernel<<<(unsigned)blocks, threads, 0, st>>>(c->d_wop, c->d_wop_lo, d_out, c->nant, c->nchan, c->nbeam,
                                                                 c->nMt, c->nKb);
  return cudaGetLastError();
}
