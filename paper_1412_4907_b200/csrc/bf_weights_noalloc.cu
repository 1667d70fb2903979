// bf_weights_noalloc.cu -- bf_get_weights_noalloc: read the weights back without allocating device memory.
//
// Who needs this.  bf_get_weights is the one call of the library that allocates on the device: it cudaMalloc's a
// buffer for the decoded weights and cudaFree's it before returning.  Three kinds of caller cannot afford that:
//   * a running observation.  cudaFree (and often cudaMalloc) synchronises the whole device, so logging the
//     coefficients in use -- the paper recomputes them between iterations for tracking beams -- would
//     stall every stream that is beamforming at that moment, and a real-time backend drops data when that happens;
//   * a process whose device memory already belongs to a pool (a framework's caching allocator, a telescope
//     backend that sizes all its buffers at start-up): a raw cudaMalloc there fails, or takes memory the pool expects;
//   * a thread that runs while another thread of the process captures a stream in the default (global) capture mode:
//     cudaMalloc is forbidden for every thread until that capture ends, and calling it breaks the capture.
// For them the decoded weights land in a fixed array that is part of the library image instead.
//
// The scratch.  bf_noalloc_scratch below is a file-scope __device__ array of BF_NOALLOC_MAX_BYTES = 8 MiB -- enough for
// one channel of the largest BASELINE.json shape (1024 beams x 1024 antennas x 8 bytes).  Every GPU on which the
// process loads libbf.so carries these 8 MiB from the moment the library's module is loaded until the process exits,
// whether or not this entry point is ever called.  Requests above the limit are refused (BF_ENOMEM); a caller reads a
// big weight set a few channels at a time (chan0 / nchan_out).
//
// Host code must not hand `bf_noalloc_scratch` itself to a kernel: in host code that name is only the host-side shadow
// of the symbol, not a device address.  The device address is looked up once per device with cudaGetSymbolAddress,
// with that device current, by the first call made on that device (scratch_of_current_device), and kept in a table.
// That first call should therefore be made before any stream capture starts; later calls do no set-up.
//
// Sharing.  There is ONE array per GPU for all contexts, streams and threads, and it keeps whatever the last call left
// in it.  Nothing has to start at zero here: the decode kernel writes every element that the call then copies out, and
// nothing else is read.  The call waits for its own copy (cudaStreamSynchronize) before it returns, so calls made one
// after the other from one thread never overlap; calls made at the same time from several threads (on any contexts or
// streams of the same GPU) would overwrite each other's scratch, so the entry point serialises them with a lock for
// the whole call.
//
// No cudaMalloc, cudaFree, cudaMallocAsync or library routine that allocates is called on this path.
#include <stdio.h>

#include <mutex>

#include "bf_internal.h"

#define BF_NOALLOC_MAX_DEVICES 64   // BF_NOALLOC_MAX_BYTES: include/bf.h

static __device__ __align__(256) float bf_noalloc_scratch[BF_NOALLOC_MAX_BYTES / sizeof(float)];

static std::mutex g_noalloc_mu;                           // set-up table and the scratch itself
static float *g_scratch_addr[BF_NOALLOC_MAX_DEVICES];     // device address of the array on each GPU; NULL = not looked up yet

// device address of bf_noalloc_scratch on the CURRENT device (g_noalloc_mu held)
static cudaError_t scratch_of_current_device(float **out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= BF_NOALLOC_MAX_DEVICES) return cudaErrorInvalidDevice;
  if (!g_scratch_addr[dev]) {
    float *p = nullptr;
    e = cudaGetSymbolAddress((void **)&p, bf_noalloc_scratch);
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    g_scratch_addr[dev] = p;
  }
  *out = g_scratch_addr[dev];
  return cudaSuccess;
}

// Variant of bf_decode_weights_kernel (bf_weights.cu) for a channel range: fp16 operand image (+ residual plane) of
// channels [chan0, chan0 + nchan_out) -> fp32 (re, im) [nchan_out][nbeam][nant] in `out`.
__global__ void bf_decode_weights_range_kernel(const __half *__restrict__ wop, const __half *__restrict__ wop_lo,
                                               float *__restrict__ out, int nant, int chan0, int nchan_out, int nbeam,
                                               int nMt, int nKb) {
  const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (long long)nchan_out * nbeam * nant) return;
  const int n = (int)(idx % nant);
  const int b = (int)((idx / nant) % nbeam);
  const int c = chan0 + (int)(idx / nant / nbeam);
  const int k = 2 * n;   // the x_re column of antenna n: W_re in the beam's "re" row, W_im in its "im" row
  const size_t tile = (((size_t)c * nMt + b / BF_TILE_BEAMS) * nKb + k / BF_KBLOCK) * (BF_TILE_ROWS * BF_KBLOCK);
  const size_t o_re = tile + bf_tile_off(bf_beam_row(b % BF_TILE_BEAMS, 0), k % BF_KBLOCK);
  const size_t o_im = tile + bf_tile_off(bf_beam_row(b % BF_TILE_BEAMS, 1), k % BF_KBLOCK);
  float wre = __half2float(wop[o_re]), wim = __half2float(wop[o_im]);
  if (wop_lo) { wre += __half2float(wop_lo[o_re]); wim += __half2float(wop_lo[o_im]); }
  out[2 * idx] = wre;
  out[2 * idx + 1] = wim;
}

// The same for the int8 two-limb operand (bf_internal.h): W = (128 hi + lo) * scale[c].
__global__ void bf_decode_weights_i8_range_kernel(const signed char *__restrict__ wop8, const double *__restrict__ scale,
                                                  float *__restrict__ out, int nant, int chan0, int nchan_out, int nbeam,
                                                  int ncol) {
  const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (long long)nchan_out * nbeam * nant) return;
  const int n = (int)(idx % nant);
  const int b = (int)((idx / nant) % nbeam);
  const int c = chan0 + (int)(idx / nant / nbeam);
  const int row0 = 32 * (b >> 3) + 4 * (b & 7), k = 2 * n;   // rows: re-hi, im-hi, re-lo, im-lo
  int limb[4];
  for (int j = 0; j < 4; ++j) {
    const int row = row0 + j;
    limb[j] = wop8[((size_t)c * ncol + row) * 64 + ((((k >> 4) ^ ((row >> 1) & 3)) << 4) | (k & 15))];
  }
  out[2 * idx] = (float)((128 * limb[0] + limb[2]) * scale[c]);
  out[2 * idx + 1] = (float)((128 * limb[1] + limb[3]) * scale[c]);
}

static int noalloc_fail(bf_ctx *c, int code, const char *msg) {
  snprintf(c->err, sizeof(c->err), "bf_get_weights_noalloc: %s", msg);
  return code;
}

extern "C" int bf_get_weights_noalloc(bf_ctx *c, int chan0, int nchan_out, float *host_out, void *stream) {
  if (!c) return BF_EINVAL;
  if (!host_out) return noalloc_fail(c, BF_EINVAL, "output pointer is NULL");
  if (chan0 < 0 || nchan_out <= 0 || chan0 > c->nchan - nchan_out)
    return noalloc_fail(c, BF_EINVAL, "channel range [chan0, chan0 + nchan_out) is empty or outside the context's channels");
  if (!c->have_geom) return noalloc_fail(c, BF_ENOGEOM, "no geometry set");
  const size_t per_chan = (size_t)c->nbeam * c->nant * 2 * sizeof(float);
  const size_t bytes = per_chan * (size_t)nchan_out;
  if (bytes > BF_NOALLOC_MAX_BYTES) {
    char msg[256];
    if (per_chan > BF_NOALLOC_MAX_BYTES)
      snprintf(msg, sizeof(msg), "one channel of weights is %zu bytes, above the %u-byte static scratch "
               "(use bf_get_weights, which allocates)", per_chan, BF_NOALLOC_MAX_BYTES);
    else
      snprintf(msg, sizeof(msg), "%d channels of weights are %zu bytes, above the %u-byte static scratch: "
               "ask for at most %zu channels per call", nchan_out, bytes, BF_NOALLOC_MAX_BYTES,
               BF_NOALLOC_MAX_BYTES / per_chan);
    return noalloc_fail(c, BF_ENOMEM, msg);
  }
  cudaStream_t st = (cudaStream_t)stream;
  std::lock_guard<std::mutex> hold(g_noalloc_mu);   // one scratch per GPU: one call at a time
  float *d = nullptr;
  cudaError_t e = scratch_of_current_device(&d);
  if (e != cudaSuccess) {
    char msg[256];
    snprintf(msg, sizeof(msg), "cudaGetSymbolAddress(bf_noalloc_scratch): %s", cudaGetErrorString(e));
    return noalloc_fail(c, BF_ECUDA, msg);
  }
  bool int8_operand = false;
  int rc = bf_prepare_weight_readback(c, st, &int8_operand);
  if (rc != BF_OK) return rc;
  const long long total = (long long)nchan_out * c->nbeam * c->nant;
  const int threads = 256;
  const unsigned blocks = (unsigned)((total + threads - 1) / threads);
  if (int8_operand)
    bf_decode_weights_i8_range_kernel<<<blocks, threads, 0, st>>>(c->d_wop8, c->d_i8scale, d, c->nant, chan0, nchan_out,
                                                                  c->nbeam, bf_i8_ncol(c->nbeam));
  else
    bf_decode_weights_range_kernel<<<blocks, threads, 0, st>>>(c->d_wop, c->d_wop_lo, d, c->nant, chan0, nchan_out,
                                                               c->nbeam, c->nMt, c->nKb);
  e = cudaGetLastError();
  if (e == cudaSuccess) { c->launches += 1; e = cudaMemcpyAsync(host_out, d, bytes, cudaMemcpyDeviceToHost, st); }
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);   // the scratch is free again when the call returns
  if (e != cudaSuccess) return noalloc_fail(c, BF_ECUDA, cudaGetErrorString(e));
  return BF_OK;
}
