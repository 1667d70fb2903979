// bf_internal.h -- shared declarations of the CUDA path (not part of the public ABI).
#pragma once
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <vector>

#include "../../include/bf.h"

// ---- weight operand layout -------------------------------------------
// The complex contraction y = W x is run as a REAL contraction over k' = 2n + {0,1} against the
// interleaved (re, im) voltages:
//   row "re" of beam b:  A[2n] =  W_re, A[2n+1] = -W_im   ->  sum_k' A x' = Re y
//   row "im" of beam b:  A[2n] =  W_im, A[2n+1] =  W_re   ->  sum_k' A x' = Im y
// Rows are grouped in M-tiles of 128 rows = 64 beams.  Inside a tile, row r = 32 q + l holds
// beam 64 mt + 16 q + (l & 15), part (l >> 4) (0 = re, 1 = im): a warp that owns TMEM lanes
// 32q..32q+31 finds re and im of one beam 16 lanes apart (one shuffle per OUTPUT bin, not per sample).
// K' is padded to a multiple of 64 (zeros).  Memory: fp16 [chan][mt][kb][128 rows][64 k'] -- every
// (chan, mt, kb) block is one contiguous 16 KiB K-major tile, stored as the exact shared-memory image
// tcgen05.mma wants (128-byte swizzle: the 16-byte chunk index of a row is XORed with row & 7), so one
// cp.async.bulk per tile brings it in with no fix-up.
// Two-term coefficients: one fp16 rounding of a coefficient (|error| <= 2^-12) is independent from sample to
// sample, so it averages out over a bin -- measured worst row 4.0e-4 of the bin mean at nint = 16, but 1.45e-3 at
// nint = 1, above BASELINE.json's 1e-3.  Below BF_LO_NINT the generator therefore also stores the rounding
// residual lo = fp16(a - fp16(a)) in a second operand plane of the same layout and every kernel contracts both
// (hi + lo carries 22 bits); the extra MMAs hide under the output traffic, which dominates at such short bins.
#define BF_LO_NINT 16
#define BF_TILE_ROWS 128
#define BF_TILE_BEAMS 64
#define BF_KBLOCK 64

__host__ __device__ inline int bf_row_beam(int mt, int r) { return mt * BF_TILE_BEAMS + ((r >> 5) << 4) + (r & 15); }
__host__ __device__ inline int bf_row_part(int r) { return (r >> 4) & 1; }
// element offset of (row r, column k) inside one 128 x 64 tile (128-byte swizzle)
__host__ __device__ inline int bf_tile_off(int r, int k) { return r * BF_KBLOCK + ((((k >> 3) ^ (r & 7)) << 3) | (k & 7)); }
// row of (beam-in-tile bl, part)
__host__ __device__ inline int bf_beam_row(int bl, int part) { return ((bl >> 4) << 5) + (part << 4) + (bl & 15); }

enum { BF_MODE_POWER = 0, BF_MODE_BEAMS = 1 };

struct BfParams {
  int nant, nbeam, nsamp, nint, nbin;
  int nMt, nKb;
  int nchan_run;        // channels processed by this launch
  const void *volt;     // device, first channel of this launch
  float *pow;           // device, first channel of this launch
  void *beams;          // voltage-beam mode (bf_run_beams): fp16 (re, im) [chan][beam][nsamp], first channel of this launch
  float beam_scale;     // voltage-beam mode: y is multiplied by this before rounding to fp16
  int mode;             // BF_MODE_POWER (|y|^2 integrated over nint -> pow) or BF_MODE_BEAMS (y -> beams)
  const __half *wop;    // device, weight operand of the first channel of this launch
  const __half *wop_lo; // second fp16 term of every coefficient (same layout), or NULL: see BF_LO_NINT
  const signed char *wop8;  // int8 two-limb weight operand of the first channel (bf_umma_i8.cu), or NULL
  const double *i8scale;    // per channel: y = (128 hi + lo) * i8scale[c]
  unsigned long long *probe;  // bf_set_clock_probe: 4 words written by CTA 0, or NULL
};

// ---- int8 two-limb weight operand (bf_umma_i8.cu; few beams, small arrays) ---------------------
// Each real coefficient a (the (re, -im) / (im, re) expansion above, gains folded in) is quantised to 15 bits,
// q = rint(a / scale_c), scale_c = gmax_c / 16256 (gmax_c = largest |gain| of the channel, 1 without gains), and
// split into two int8 limbs q = 128 hi + lo, hi = floor((q + 64) / 128) in [-127, 127], lo in [-64, 63].
// Rows (= accumulator columns): 32 per chunk of 8 beams, row 32 ch + 4 i + j holds beam 8 ch + i,
// j = 0 re-hi, 1 im-hi, 2 re-lo, 3 im-lo.  Memory: int8 [chan][ncol rows][64 bytes], each row's 16-byte chunk k
// stored at chunk k ^ ((row >> 1) & 3): the 64-byte-swizzled shared-memory image tcgen05.mma reads.
#define BF_I8_MAX_BEAMS 32
#define BF_I8_QSCALE 16256.0
__host__ __device__ inline int bf_i8_ncol(int nbeam) { return nbeam <= 8 ? 32 : nbeam <= 16 ? 64 : 128; }

// ---- shapes of the bin-per-lane fp16 kernel (bf_umma_bl.cu) -------------------------------------
// THE predicate: bf_umma_supported (does the fp16 family integrate this nint?), bf_launch_umma (which kernel) and
// bf_kernel_name (what to report) all call it.  Complex int8 or 4+4-bit input, 32 antennas, 33-64 beams (one coefficient
// tile), power mode, single-term coefficients (nint >= BF_LO_NINT), any EVEN nint (the running sum of a bin lives in the
// registers of the thread that owns its TMEM lane), and enough bins that the 256 lanes of an item are not mostly padding.
inline bool bf_bl_shape(int dtype, int mode, int nant, int nbeam, int nint, int nbin) {
  if ((dtype != BF_CI8 && dtype != BF_CI4) || mode != BF_MODE_POWER || nant != 32 || nbeam <= 32 || nbeam > BF_TILE_BEAMS) return false;
  if (nint < BF_LO_NINT || nint % 2 != 0 || (long long)nint * 64 >= (1ll << 32)) return false;
  return nbin % 256 == 0 || nbin >= 1024;
}

struct bf_ctx {
  int nant, nchan, nbeam, nsamp, nint, nbin;
  int dtype, kernel_forced;
  int nMt, nKb;
  void *ws;
  size_t ws_bytes;
  double *d_ant, *d_freq, *d_dir;
  double *d_gain;          // [nchan][nant][2] complex gains (always per channel on the device)
  bool have_gains;         // false = all ones (d_gain not read)
  std::vector<double> h_gain, h_i8scale;
  __half *d_wop;
  __half *d_wop_lo;        // residual plane (nint < BF_LO_NINT), else NULL
  __half *wop_lo_buf[2];
  signed char *d_wop8;     // int8 two-limb operand (NULL when the shape never takes the int8 kernel)
  double *d_i8scale;       // [nchan]
  bool have_geom;
  // tracking beams (row f3): up to two (geometry, weight operand) buffers; runs read `active`, an update
  // writes the other one on its own stream and the next run switches over behind an event
  int nwbuf, active, pending;      // pending: -1 none, else the buffer the next run switches to
  char *geom_buf[2];
  __half *wop_buf[2];
  signed char *wop8_buf[2];
  cudaEvent_t ev_upd, ev_use[2];
  bool have_wevents, used[2];
  std::vector<double> h_geom;
  long long launches;
  int sm_count;     // 0 = device not probed yet
  int device_ok;    // -1 unknown, 0 no, 1 yes
  cudaEvent_t ev_copied[2], ev_done[2], ev_kdone[2];   // H2D landed / D2H landed / kernel finished, per staging half
  cudaStream_t d2h_stream;                             // bf_run_host's read-back queue (created with the events)
  bool have_events;
  unsigned long long *d_probe;   // bf_set_clock_probe
  char err[512];
};

size_t bf_in_bytes_per_chan(const bf_ctx *c);
size_t bf_wop_bytes_per_chan(const bf_ctx *c);

// kernels (each returns a cudaError_t from the launch)
cudaError_t bf_launch_weights(const bf_ctx *c, cudaStream_t st);
cudaError_t bf_launch_decode_weights(const bf_ctx *c, float *d_out, bool int8_operand, cudaStream_t st);
int bf_prepare_weight_readback(bf_ctx *c, cudaStream_t st, bool *int8_operand);   // bf_api.cu, for bf_weights_noalloc.cu
cudaError_t bf_launch_simt(const BfParams &p, int dtype, cudaStream_t st);
bool bf_umma_supported(const bf_ctx *c, const char **why);
bool bf_umma_shape_supported(const bf_ctx *c, const char **why);  // ignoring nint (voltage-beam mode)
bool bf_umma_i8_supported(const bf_ctx *c, int mode);
cudaError_t bf_launch_umma_i8(const BfParams &p, int dtype, int sm_count, cudaStream_t st);
bool bf_umma_i8b_takes(const BfParams &p, int dtype);   // bf_umma_i8b.cu: one output bin per TMEM lane
cudaError_t bf_launch_umma_i8b(const BfParams &p, int dtype, int sm_count, cudaStream_t st);
bool bf_umma_bl_takes(const BfParams &p, int dtype);    // bf_umma_bl.cu: 33-64 beams, bin per lane, voltages as the A operand in TMEM
cudaError_t bf_launch_umma_bl(const BfParams &p, int dtype, int sm_count, cudaStream_t st);
cudaError_t bf_launch_incoherent(const bf_ctx *c, const void *volt, float *out, cudaStream_t st);
cudaError_t bf_launch_umma(const BfParams &p, int dtype, int sm_count, cudaStream_t st);
cudaError_t bf_launch_umma_kblock(const BfParams &p, int dtype, int sm_count, cudaStream_t st);
