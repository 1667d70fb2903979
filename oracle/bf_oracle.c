/*
 * bf_oracle.c -- the ORACLE: a plain, slow, fp64 CPU coherent beamformer.
 *
 * TEST INFRASTRUCTURE ONLY.  Nothing on the product path may import, link or call this
 * file; only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs use it.  It shares no code, header, table or constant with the CUDA path under
 * paper_1412_4907_b200/csrc/.
 *
 * What it computes (arXiv 1412.4907; line numbers are /root/reference/PAPER.md):
 *
 *   W[c][b][n] = exp(-i 2 pi f_c/c0 (r_n . s_b))          steering factor e^{-i k0.r_n} of
 *                                                         Eq. 1, k0 = 2 pi f_c/c0 s_b
 *   y[c][b][t] = sum_n W[c][b][n] x[c][t][n]              per-channel N_b x N_a matrix times the
 *                                                         antenna vector (Sec. 2.1); loop nest of
 *                                                         the "simple implementation", one (f,t,b) triplet
 *                                                         combining all antennas
 *   P[c][b][j] = sum_{t=jI}^{(j+1)I-1} |y[c][b][t]|^2     "absolute power computation" with
 *                                                         the data "reduced within the GPU itself"
 *
 * It is the definition written out: fp64 everywhere, antennas summed in plain n order,
 * time summed in plain t order, no blocking, no fusion, no normalisation (reading A6).
 * OpenMP splits the channel loop only (channels are independent).
 *
 * Pins (tests/test_oracle_pins.py; incoherent and voltage beams: tests/test_oracle_pins_modes.py): Eq. 1 closed forms for a linear and a grid array,
 * N^2 A^2 coherent gain, incoherent N level, a Parseval identity on a DFT beam grid, hand
 * cases with N=1 and N=2, algebraic invariants, and an independent numpy einsum.
 * Unpinned: value-level agreement with the paper itself -- it prints no beam powers
 * (Figs. 5-7 are images): "parity unpinned" against the paper's own numbers.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_C0 299792458.0 /* speed of light, m/s (exact SI value) */

enum { ORACLE_CI8 = 0, ORACLE_CF16 = 1, ORACLE_C128 = 2, ORACLE_CI4 = 3 };

int oracle_num_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/* Eq. 1 steering weights for ONE channel: w[b][n] = cos(2 pi u) - i sin(2 pi u),
 * u = f (r_n . s_b)/c0 in turns.  wr, wi: [nbeam][nant]. */
static void channel_weights(int nant, int nbeam, const double *ant_xyz, double freq_hz,
                            const double *beam_dir, double *wr, double *wi) {
  const double two_pi = 2.0 * 3.14159265358979323846;
  for (int b = 0; b < nbeam; ++b) {
    for (int n = 0; n < nant; ++n) {
      double dot = ant_xyz[3 * n + 0] * beam_dir[3 * b + 0] + ant_xyz[3 * n + 1] * beam_dir[3 * b + 1] +
                   ant_xyz[3 * n + 2] * beam_dir[3 * b + 2];
      double turns = freq_hz * dot / ORACLE_C0;
      wr[(size_t)b * nant + n] = cos(two_pi * turns);
      wi[(size_t)b * nant + n] = -sin(two_pi * turns);
    }
  }
}

/* W[c][b][n] as interleaved (re, im) doubles: out[((c*nbeam+b)*nant+n)*2 + {0,1}]. */
int oracle_weights(int nant, int nchan, int nbeam, const double *ant_xyz, const double *chan_freq_hz,
                   const double *beam_dir, double *out) {
  if (nant <= 0 || nchan <= 0 || nbeam <= 0) return -1;
  double *wr = (double *)malloc(sizeof(double) * nbeam * nant);
  double *wi = (double *)malloc(sizeof(double) * nbeam * nant);
  if (!wr || !wi) { free(wr); free(wi); return -5; }
  for (int c = 0; c < nchan; ++c) {
    channel_weights(nant, nbeam, ant_xyz, chan_freq_hz[c], beam_dir, wr, wi);
    for (size_t k = 0; k < (size_t)nbeam * nant; ++k) {
      out[((size_t)c * nbeam * nant + k) * 2 + 0] = wr[k];
      out[((size_t)c * nbeam * nant + k) * 2 + 1] = wi[k];
    }
  }
  free(wr); free(wi);
  return 0;
}

/* one complex voltage sample -> fp64, exactly */
static inline void load_sample(const void *volt, int dtype, size_t idx, double *xr, double *xi) {
  if (dtype == ORACLE_CI8) {
    const int8_t *p = (const int8_t *)volt;
    *xr = (double)p[2 * idx]; *xi = (double)p[2 * idx + 1];
  } else if (dtype == ORACLE_CF16) {
    const _Float16 *p = (const _Float16 *)volt;
    *xr = (double)p[2 * idx]; *xi = (double)p[2 * idx + 1];
  } else if (dtype == ORACLE_CI4) {
    /* the paper's F-engine format: "4-bit, two's complement, complex voltages ... each antenna value as
     * a single byte".  Nibble order is not stated: high nibble = real, low nibble =
     * imaginary (reading A20).  Written out with plain integer arithmetic. */
    const uint8_t b = ((const uint8_t *)volt)[idx];
    int re = b >> 4, im = b & 15;
    if (re >= 8) re -= 16;
    if (im >= 8) im -= 16;
    *xr = (double)re; *xi = (double)im;
  } else {
    const double *p = (const double *)volt;
    *xr = p[2 * idx]; *xi = p[2 * idx + 1];
  }
}

/*
 * The whole path.  voltages: [nchan][nsamp][nant] complex interleaved (re,im), element type `dtype`.
 * powers (out): [nchan][nbeam][nsamp/nint] fp64.  Channels c with c % chan_stride != 0 are skipped
 * (left untouched) so that a bounded sample of a big workload can be timed/checked; pass 1 for all.
 * Returns 0, or -1 on bad arguments (nsamp % nint != 0 is rejected: DESIGN.md reading A8).
 */
int oracle_beamform(int nant, int nchan, int nbeam, int nsamp, int nint, int dtype, const double *ant_xyz,
                    const double *chan_freq_hz, const double *beam_dir, const void *voltages,
                    double *powers, int chan_stride) {
  if (nant <= 0 || nchan <= 0 || nbeam <= 0 || nsamp <= 0 || nint <= 0) return -1;
  if (nsamp % nint != 0 || chan_stride <= 0) return -1;
  if (dtype != ORACLE_CI8 && dtype != ORACLE_CF16 && dtype != ORACLE_C128 && dtype != ORACLE_CI4) return -1;
  const int nbin = nsamp / nint;
  int err = 0;
#pragma omp parallel for schedule(dynamic, 1)
  for (int c = 0; c < nchan; ++c) {
    if (c % chan_stride != 0) continue;
    double *wr = (double *)malloc(sizeof(double) * nbeam * nant);
    double *wi = (double *)malloc(sizeof(double) * nbeam * nant);
    double *xr = (double *)malloc(sizeof(double) * nant);
    double *xi = (double *)malloc(sizeof(double) * nant);
    if (!wr || !wi || !xr || !xi) {
      err = -5; free(wr); free(wi); free(xr); free(xi);
      continue;
    }
    channel_weights(nant, nbeam, ant_xyz, chan_freq_hz[c], beam_dir, wr, wi);
    double *P = powers + (size_t)c * nbeam * nbin;
    for (size_t k = 0; k < (size_t)nbeam * nbin; ++k) P[k] = 0.0;
    for (int t = 0; t < nsamp; ++t) {
      const int j = t / nint;
      for (int n = 0; n < nant; ++n) load_sample(voltages, dtype, ((size_t)c * nsamp + t) * nant + n, &xr[n], &xi[n]);
      for (int b = 0; b < nbeam; ++b) {
        const double *wrb = wr + (size_t)b * nant, *wib = wi + (size_t)b * nant;
        double yr = 0.0, yi = 0.0;
        for (int n = 0; n < nant; ++n) { /* complex multiply-accumulate: 8 flop */
          yr += wrb[n] * xr[n] - wib[n] * xi[n];
          yi += wrb[n] * xi[n] + wib[n] * xr[n];
        }
        P[(size_t)b * nbin + j] += yr * yr + yi * yi;
      }
    }
    free(wr); free(wi); free(xr); free(xi);
  }
  return err;
}

/* Raw complex beams y[c][b][t] (interleaved fp64) for small cases; used only by the pins. */
int oracle_beams(int nant, int nchan, int nbeam, int nsamp, int dtype, const double *ant_xyz,
                 const double *chan_freq_hz, const double *beam_dir, const void *voltages, double *beams) {
  if (nant <= 0 || nchan <= 0 || nbeam <= 0 || nsamp <= 0) return -1;
  double *wr = (double *)malloc(sizeof(double) * nbeam * nant);
  double *wi = (double *)malloc(sizeof(double) * nbeam * nant);
  if (!wr || !wi) { free(wr); free(wi); return -5; }
  for (int c = 0; c < nchan; ++c) {
    channel_weights(nant, nbeam, ant_xyz, chan_freq_hz[c], beam_dir, wr, wi);
    for (int t = 0; t < nsamp; ++t)
      for (int b = 0; b < nbeam; ++b) {
        double yr = 0.0, yi = 0.0;
        for (int n = 0; n < nant; ++n) {
          double xr, xi;
          load_sample(voltages, dtype, ((size_t)c * nsamp + t) * nant + n, &xr, &xi);
          yr += wr[(size_t)b * nant + n] * xr - wi[(size_t)b * nant + n] * xi;
          yi += wr[(size_t)b * nant + n] * xi + wi[(size_t)b * nant + n] * xr;
        }
        size_t o = (((size_t)c * nbeam + b) * nsamp + t) * 2;
        beams[o] = yr; beams[o + 1] = yi;
      }
  }
  free(wr); free(wi);
  return 0;
}

/*
 * Incoherent beam: "Squaring and adding the signals of all the elements together is the process of
 * incoherent beamforming" -- the wide-field, low-sensitivity alternative the paper names
 * next to coherent beams.  No weights, no geometry:
 *     P_inc[c][j] = sum_{t=jI}^{(j+1)I-1} sum_n |x[c][t][n]|^2
 * out: [nchan][nsamp/nint] fp64.  Plain t, n order, fp64, no normalisation (reading A6).
 */
int oracle_incoherent(int nant, int nchan, int nsamp, int nint, int dtype, const void *voltages, double *out) {
  if (nant <= 0 || nchan <= 0 || nsamp <= 0 || nint <= 0 || nsamp % nint != 0) return -1;
  if (dtype != ORACLE_CI8 && dtype != ORACLE_CF16 && dtype != ORACLE_C128 && dtype != ORACLE_CI4) return -1;
  const int nbin = nsamp / nint;
  for (int c = 0; c < nchan; ++c)
    for (int j = 0; j < nbin; ++j) {
      double acc = 0.0;
      for (int t = j * nint; t < (j + 1) * nint; ++t)
        for (int n = 0; n < nant; ++n) {
          double xr, xi;
          load_sample(voltages, dtype, ((size_t)c * nsamp + t) * nant + n, &xr, &xi);
          acc += xr * xr + xi * xi;
        }
      out[(size_t)c * nbin + j] = acc;
    }
  return 0;
}
