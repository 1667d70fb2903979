// bf_api.cu -- the C-ABI boundary (include/bf.h): context, validation, workspace, dispatch.
// Problem statement: PAPER.md:56-64; static weights per buffer: PAPER.md:64, 100; host<->device
// overlap with two streams: PAPER.md:140.
#include <math.h>
#include <stdarg.h>
#include <stdio.h>
#include <string.h>

#include <new>

#include "bf_internal.h"

#define BF_ALIGN 1024

static size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

static int fail(bf_ctx *c, int code, const char *fmt, ...) {
  if (c) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(c->err, sizeof(c->err), fmt, ap);
    va_end(ap);
  }
  return code;
}
static int cuda_fail(bf_ctx *c, cudaError_t e, const char *what) {
  return fail(c, BF_ECUDA, "%s: %s", what, cudaGetErrorString(e));
}

// every stream-ordering guarantee of the library (tracking beams, host / streaming overlap) rests on these two
static int wait_event(bf_ctx *c, cudaStream_t st, cudaEvent_t ev) {
  cudaError_t e = cudaStreamWaitEvent(st, ev, 0);
  return e == cudaSuccess ? BF_OK : cuda_fail(c, e, "cudaStreamWaitEvent");
}
static int record_event(bf_ctx *c, cudaEvent_t ev, cudaStream_t st) {
  cudaError_t e = cudaEventRecord(ev, st);
  return e == cudaSuccess ? BF_OK : cuda_fail(c, e, "cudaEventRecord");
}

size_t bf_in_bytes_per_chan(const bf_ctx *c) {
  return (size_t)c->nsamp * c->nant * (c->dtype == BF_CI8 ? 2 : c->dtype == BF_CI4 ? 1 : 4);
}
size_t bf_wop_bytes_per_chan(const bf_ctx *c) {
  return (size_t)c->nMt * c->nKb * BF_TILE_ROWS * BF_KBLOCK * sizeof(__half);
}
static size_t geom_bytes(const bf_ctx *c) {  // positions, frequencies, directions, gains, int8-operand scales
  return align_up(sizeof(double) * (3 * (size_t)c->nant + c->nchan + 3 * (size_t)c->nbeam +
                                    2 * (size_t)c->nchan * c->nant + c->nchan), BF_ALIGN);
}
// the int8 two-limb operand exists whenever the shape could take bf_umma_i8.cu (any nint)
static bool i8_shape(const bf_ctx *c) {
  if (c->nbeam > BF_I8_MAX_BEAMS) return false;
  if (c->dtype == BF_CI4) return c->nant == 32;       // 4+4-bit rows unpack to int8 operands in bf_umma_i8b.cu
  return c->dtype == BF_CI8 && c->nant % 8 == 0 && c->nant <= 32;
}
static size_t wop8_bytes(const bf_ctx *c) {
  return i8_shape(c) ? align_up((size_t)c->nchan * bf_i8_ncol(c->nbeam) * 64, BF_ALIGN) : 0;
}

#ifdef BF_JITTER
extern "C" const char *bf_version(void) { return "paper_1412_4907_b200 0.1 (sm_100a) [jitter build: test only]"; }
#else
extern "C" const char *bf_version(void) { return "paper_1412_4907_b200 0.1 (sm_100a)"; }
#endif

extern "C" bf_ctx *bf_create(int nant, int nchan, int nbeam, int nsamp, int nint) {
  if (nant <= 0 || nchan <= 0 || nbeam <= 0 || nsamp <= 0 || nint <= 0) return nullptr;
  if (nsamp % nint != 0) return nullptr;  // DESIGN.md reading A8
  if ((long long)nchan * nbeam > (1LL << 40)) return nullptr;
  bf_ctx *c = new (std::nothrow) bf_ctx();
  if (!c) return nullptr;
  c->nant = nant; c->nchan = nchan; c->nbeam = nbeam; c->nsamp = nsamp; c->nint = nint;
  c->nbin = nsamp / nint;
  c->dtype = BF_CI8;
  c->kernel_forced = BF_KERNEL_AUTO;
  c->nMt = (nbeam + BF_TILE_BEAMS - 1) / BF_TILE_BEAMS;
  c->nKb = (2 * nant + BF_KBLOCK - 1) / BF_KBLOCK;
  c->ws = nullptr; c->ws_bytes = 0;
  c->d_ant = c->d_freq = c->d_dir = nullptr; c->d_wop = nullptr;
  c->have_geom = false;
  c->d_gain = nullptr; c->have_gains = false;
  c->launches = 0;
  c->sm_count = 0; c->device_ok = -1;
  c->have_events = false;
  c->nwbuf = 1; c->active = 0; c->pending = -1;
  c->geom_buf[0] = c->geom_buf[1] = nullptr; c->wop_buf[0] = c->wop_buf[1] = nullptr;
  c->wop_lo_buf[0] = c->wop_lo_buf[1] = nullptr; c->d_wop_lo = nullptr;
  c->wop8_buf[0] = c->wop8_buf[1] = nullptr; c->d_wop8 = nullptr; c->d_i8scale = nullptr;
  c->have_wevents = false; c->used[0] = c->used[1] = false;
  c->d_probe = nullptr;
  c->err[0] = 0;
  return c;
}

extern "C" void bf_destroy(bf_ctx *c) {
  if (!c) return;
  if (c->have_events)
  {
    for (int i = 0; i < 2; ++i) { cudaEventDestroy(c->ev_copied[i]); cudaEventDestroy(c->ev_done[i]); cudaEventDestroy(c->ev_kdone[i]); }
    cudaStreamDestroy(c->d2h_stream);
  }
  if (c->have_wevents) { cudaEventDestroy(c->ev_upd); cudaEventDestroy(c->ev_use[0]); cudaEventDestroy(c->ev_use[1]); }
  delete c;
}

extern "C" const char *bf_last_error(const bf_ctx *c) { return c ? c->err : "null context"; }

extern "C" int bf_set_dtype(bf_ctx *c, int dtype) {
  if (!c) return BF_EINVAL;
  if (dtype != BF_CI8 && dtype != BF_CF16 && dtype != BF_CI4) return fail(c, BF_EINVAL, "unknown dtype %d", dtype);
  // the workspace layout (which weight operands exist) depends on the element type
  if (c->ws && dtype != c->dtype) return fail(c, BF_EINVAL, "bf_set_dtype must be called before bf_set_workspace");
  c->dtype = dtype;
  return BF_OK;
}

extern "C" int bf_set_clock_probe(bf_ctx *c, void *dev_u64x4) {
  if (!c) return BF_EINVAL;
  if (((uintptr_t)dev_u64x4) % 8) return fail(c, BF_EINVAL, "clock probe must be 8-byte aligned");
  c->d_probe = (unsigned long long *)dev_u64x4;
  return BF_OK;
}

extern "C" int bf_set_kernel(bf_ctx *c, int kernel) {
  if (!c) return BF_EINVAL;
  if (kernel != BF_KERNEL_AUTO && kernel != BF_KERNEL_SIMT && kernel != BF_KERNEL_UMMA &&
      kernel != BF_KERNEL_UMMA_F16 && kernel != BF_KERNEL_UMMA_I8)
    return fail(c, BF_EINVAL, "unknown kernel %d", kernel);
  c->kernel_forced = kernel;
  return BF_OK;
}

// the int8 kernel takes over below this many beams (measured crossover against the fp16 kernel)
#define BF_I8_AUTO_BEAMS 32

// which kernel bf_run launches: BF_KERNEL_SIMT, BF_KERNEL_UMMA_F16 or BF_KERNEL_UMMA_I8; 0 + *why if the
// forced kernel cannot run the shape
static int pick_kernel(const bf_ctx *c, int mode, const char **why) {
  int k = c->kernel_forced;
  *why = "";
  if (k == BF_KERNEL_SIMT) return BF_KERNEL_SIMT;
  const bool i8_ok = i8_shape(c) && bf_umma_i8_supported(c, mode) && (c->d_wop8 != nullptr || c->ws == nullptr);
  if (k == BF_KERNEL_UMMA_I8) {
    if (!i8_ok) *why = "int8-operand kernel needs int8 input with nant % 8 == 0 and <= 32 (4-bit: nant = 32, nint % 4 == 0), <= 32 beams, "
                       "nint 2^k <= 32, % 32 == 0, or even with nbin % 128 == 0 or >= 512";
    return i8_ok ? BF_KERNEL_UMMA_I8 : 0;
  }
  if (k != BF_KERNEL_UMMA_F16 && i8_ok && c->nbeam <= BF_I8_AUTO_BEAMS) return BF_KERNEL_UMMA_I8;
  const bool f16_ok = mode == BF_MODE_BEAMS ? bf_umma_shape_supported(c, why) : bf_umma_supported(c, why);
  if (f16_ok) return BF_KERNEL_UMMA_F16;
  if (i8_ok && k != BF_KERNEL_UMMA_F16) return BF_KERNEL_UMMA_I8;   // e.g. nint = 96: only the int8 kernel integrates it
  return k == BF_KERNEL_AUTO ? BF_KERNEL_SIMT : 0;
}

extern "C" int bf_selected_kernel(const bf_ctx *c) {
  if (!c) return BF_EINVAL;
  const char *why;
  const int k = pick_kernel(c, BF_MODE_POWER, &why);
  if (k == 0) return c->kernel_forced == BF_KERNEL_UMMA_I8 || c->kernel_forced == BF_KERNEL_UMMA_F16 ? BF_KERNEL_UMMA : c->kernel_forced;
  return k == BF_KERNEL_SIMT ? BF_KERNEL_SIMT : BF_KERNEL_UMMA;
}

extern "C" const char *bf_kernel_name(const bf_ctx *c) {
  if (!c) return "";
  const char *why;
  switch (pick_kernel(c, BF_MODE_POWER, &why)) {
    case BF_KERNEL_SIMT: return "simt";
    case BF_KERNEL_UMMA_I8: return "umma-i8";
    case BF_KERNEL_UMMA_F16: {
      if (!(2 * c->nant <= 64 && c->dtype != BF_CF16)) return "umma-f16-kblock";
      const bool binlane = bf_bl_shape(c->dtype, BF_MODE_POWER, c->nant, c->nbeam, c->nint, c->nbin);   // bf_umma_bl.cu
      return binlane ? "umma-f16-binlane" : "umma-f16-resident";
    }
    default: return "unsupported";
  }
}

extern "C" long long bf_launch_count(const bf_ctx *c) { return c ? c->launches : 0; }

static size_t wop_bytes(const bf_ctx *c) { return align_up((size_t)c->nchan * bf_wop_bytes_per_chan(c), BF_ALIGN); }
static size_t wop_lo_bytes(const bf_ctx *c) { return c->nint < BF_LO_NINT ? wop_bytes(c) : 0; }

extern "C" size_t bf_workspace_bytes(const bf_ctx *c) {
  if (!c) return 0;
  return (size_t)c->nwbuf * (geom_bytes(c) + wop_bytes(c) + wop8_bytes(c) + wop_lo_bytes(c));
}

extern "C" int bf_set_weight_buffers(bf_ctx *c, int n) {
  if (!c) return BF_EINVAL;
  if (n != 1 && n != 2) return fail(c, BF_EINVAL, "weight buffers must be 1 or 2");
  if (c->ws) return fail(c, BF_EINVAL, "bf_set_weight_buffers must be called before bf_set_workspace");
  c->nwbuf = n;
  return BF_OK;
}

// point the generator / the kernels at (geometry, weight operand) buffer i
static void select_buffer(bf_ctx *c, int i) {
  char *p = c->geom_buf[i];
  c->d_ant = (double *)p;
  c->d_freq = c->d_ant + 3 * (size_t)c->nant;
  c->d_dir = c->d_freq + c->nchan;
  c->d_gain = c->d_dir + 3 * (size_t)c->nbeam;
  c->d_i8scale = c->d_gain + 2 * (size_t)c->nchan * c->nant;
  c->d_wop = c->wop_buf[i];
  c->d_wop_lo = c->wop_lo_buf[i];
  c->d_wop8 = c->wop8_buf[i];
}

// no fallback: the device must be Blackwell (compute capability 10.x)
static int probe_device(bf_ctx *c) {
  if (c->device_ok == 1) return BF_OK;
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return cuda_fail(c, e, "cudaGetDevice");
  int major = 0, sms = 0;
  e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev);
  if (e != cudaSuccess) return cuda_fail(c, e, "cudaDeviceGetAttribute");
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  if (major != 10) {
    c->device_ok = 0;
    return fail(c, BF_EUNSUPPORTED, "device compute capability %d.x is not sm_100 (no fallback)", major);
  }
  c->sm_count = sms;
  c->device_ok = 1;
  return BF_OK;
}

extern "C" int bf_set_workspace(bf_ctx *c, void *dev_ptr, size_t bytes) {
  if (!c) return BF_EINVAL;
  if (!dev_ptr) return fail(c, BF_EINVAL, "workspace pointer is NULL");
  if (((uintptr_t)dev_ptr) % BF_ALIGN) return fail(c, BF_EINVAL, "workspace must be %d-byte aligned", BF_ALIGN);
  if (bytes < bf_workspace_bytes(c))
    return fail(c, BF_ENOMEM, "workspace too small: %zu < %zu", bytes, bf_workspace_bytes(c));
  c->ws = dev_ptr;
  c->ws_bytes = bytes;
  char *p = (char *)dev_ptr;
  for (int i = 0; i < c->nwbuf; ++i) {
    c->geom_buf[i] = p + (size_t)i * geom_bytes(c);
    c->wop_buf[i] = (__half *)(p + (size_t)c->nwbuf * geom_bytes(c) + (size_t)i * wop_bytes(c));
    c->wop_lo_buf[i] = wop_lo_bytes(c) ? (__half *)(p + (size_t)c->nwbuf * (geom_bytes(c) + wop_bytes(c) + wop8_bytes(c)) + (size_t)i * wop_lo_bytes(c))
                                       : nullptr;
    c->wop8_buf[i] = wop8_bytes(c) ? (signed char *)(p + (size_t)c->nwbuf * (geom_bytes(c) + wop_bytes(c)) + (size_t)i * wop8_bytes(c))
                                   : nullptr;
  }
  c->active = 0; c->pending = -1; c->used[0] = c->used[1] = false;
  select_buffer(c, 0);
  c->have_geom = false;
  return BF_OK;
}

// per-channel scale of the int8 two-limb operand: (largest |gain| of the channel) / 16256
static cudaError_t upload_i8scale(bf_ctx *c, cudaStream_t st) {
  if (!c->d_wop8) return cudaSuccess;
  c->h_i8scale.assign(c->nchan, 1.0 / BF_I8_QSCALE);
  if (c->have_gains)
    for (int ch = 0; ch < c->nchan; ++ch) {
      double g2 = 0.0;
      for (int n = 0; n < c->nant; ++n) {
        const double *g = c->h_gain.data() + 2 * ((size_t)ch * c->nant + n);
        const double a = g[0] * g[0] + g[1] * g[1];
        if (a > g2) g2 = a;
      }
      c->h_i8scale[ch] = (g2 > 0.0 ? sqrt(g2) : 1.0) / BF_I8_QSCALE;
    }
  return cudaMemcpyAsync(c->d_i8scale, c->h_i8scale.data(), c->nchan * sizeof(double), cudaMemcpyHostToDevice, st);
}

static int check_geometry(bf_ctx *c, const double *ant, const double *freq, const double *dir) {
  if (!ant || !freq || !dir) return fail(c, BF_EINVAL, "geometry pointer is NULL");
  for (int i = 0; i < 3 * c->nant; ++i)
    if (!isfinite(ant[i])) return fail(c, BF_EINVAL, "antenna position %d is not finite", i / 3);
  for (int i = 0; i < c->nchan; ++i)
    if (!isfinite(freq[i]) || freq[i] <= 0.0) return fail(c, BF_EINVAL, "channel frequency %d is not positive/finite", i);
  for (int b = 0; b < c->nbeam; ++b) {
    double n2 = dir[3 * b] * dir[3 * b] + dir[3 * b + 1] * dir[3 * b + 1] + dir[3 * b + 2] * dir[3 * b + 2];
    if (!isfinite(n2) || fabs(sqrt(n2) - 1.0) > 1e-6) return fail(c, BF_EINVAL, "beam direction %d is not a unit vector", b);
  }
  return BF_OK;
}

// copy the geometry (+ gains) into the currently selected buffer and generate its weights on `st`
static int upload_and_generate(bf_ctx *c, const double *ant, const double *freq, const double *dir, cudaStream_t st) {
  size_t na = 3 * (size_t)c->nant, nf = c->nchan, nd = 3 * (size_t)c->nbeam;
  c->h_geom.resize(na + nf + nd);
  memcpy(c->h_geom.data(), ant, na * sizeof(double));
  memcpy(c->h_geom.data() + na, freq, nf * sizeof(double));
  memcpy(c->h_geom.data() + na + nf, dir, nd * sizeof(double));
  cudaError_t e = cudaMemcpyAsync(c->d_ant, c->h_geom.data(), (na + nf + nd) * sizeof(double), cudaMemcpyHostToDevice, st);
  if (e != cudaSuccess) return cuda_fail(c, e, "geometry H2D copy");
  if (c->have_gains) {
    e = cudaMemcpyAsync(c->d_gain, c->h_gain.data(), c->h_gain.size() * sizeof(double), cudaMemcpyHostToDevice, st);
    if (e != cudaSuccess) return cuda_fail(c, e, "gain H2D copy");
  }
  if ((e = upload_i8scale(c, st)) != cudaSuccess) return cuda_fail(c, e, "int8 scale H2D copy");
  e = bf_launch_weights(c, st);
  if (e != cudaSuccess) return cuda_fail(c, e, "weight generator launch");
  c->launches += c->d_wop8 ? 2 : 1;
  return BF_OK;
}

extern "C" int bf_set_geometry(bf_ctx *c, const double *ant, const double *freq, const double *dir, void *stream) {
  if (!c) return BF_EINVAL;
  int rc = check_geometry(c, ant, freq, dir);
  if (rc != BF_OK) return rc;
  if (!c->ws) return fail(c, BF_ENOGEOM, "bf_set_workspace must be called before bf_set_geometry");
  if ((rc = probe_device(c)) != BF_OK) return rc;
  if (c->pending >= 0) {  // an update in flight is superseded: this call defines the weights of the next run
    if ((rc = wait_event(c, (cudaStream_t)stream, c->ev_upd)) != BF_OK) return rc;
    c->active = c->pending; c->pending = -1;
  }
  select_buffer(c, c->active);
  if ((rc = upload_and_generate(c, ant, freq, dir, (cudaStream_t)stream)) != BF_OK) return rc;
  c->have_geom = true;
  return BF_OK;
}

static int ensure_wevents(bf_ctx *c) {
  if (c->have_wevents) return BF_OK;
  cudaError_t e = cudaEventCreateWithFlags(&c->ev_upd, cudaEventDisableTiming);
  if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_use[0], cudaEventDisableTiming);
  if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_use[1], cudaEventDisableTiming);
  if (e != cudaSuccess) return cuda_fail(c, e, "cudaEventCreate");
  c->have_wevents = true;
  return BF_OK;
}

// Tracking beams (row f3): new pointings are generated into the buffer the kernels are
// NOT reading, on the caller's update stream, while bf_run keeps using the active one.
extern "C" int bf_update_geometry(bf_ctx *c, const double *ant, const double *freq, const double *dir, void *update_stream) {
  if (!c) return BF_EINVAL;
  if (c->nwbuf != 2) return fail(c, BF_EINVAL, "bf_update_geometry needs bf_set_weight_buffers(ctx, 2)");
  int rc = check_geometry(c, ant, freq, dir);
  if (rc != BF_OK) return rc;
  if (!c->have_geom) return fail(c, BF_ENOGEOM, "bf_set_geometry must be called once before bf_update_geometry");
  if ((rc = ensure_wevents(c)) != BF_OK) return rc;
  cudaStream_t us = (cudaStream_t)update_stream;
  const int target = 1 - c->active;  // a second update before any run overwrites the same (unused) buffer
  // runs that read `target` before the last switch may still be executing on the run stream
  if (c->used[target] && (rc = wait_event(c, us, c->ev_use[target])) != BF_OK) return rc;
  select_buffer(c, target);
  rc = upload_and_generate(c, ant, freq, dir, us);
  select_buffer(c, c->active);
  if (rc != BF_OK) return rc;
  if ((rc = record_event(c, c->ev_upd, us)) != BF_OK) return rc;
  c->pending = target;
  return BF_OK;
}

extern "C" int bf_set_antenna_gains(bf_ctx *c, const double *gains, int per_channel, void *stream) {
  if (!c) return BF_EINVAL;
  if (!gains) {
    c->have_gains = false;
    c->h_gain.clear();
  } else {
    const size_t n = 2 * (size_t)c->nant * (per_channel ? c->nchan : 1);
    for (size_t i = 0; i < n; ++i)
      if (!isfinite(gains[i])) return fail(c, BF_EINVAL, "antenna gain %zu is not finite", i / 2);
    c->h_gain.resize(2 * (size_t)c->nant * c->nchan);
    for (int ch = 0; ch < c->nchan; ++ch)
      memcpy(c->h_gain.data() + 2 * (size_t)ch * c->nant, gains + (per_channel ? 2 * (size_t)ch * c->nant : 0),
             2 * (size_t)c->nant * sizeof(double));
    c->have_gains = true;
  }
  if (!c->have_geom) {
    if (!c->ws) return fail(c, BF_ENOGEOM, "bf_set_workspace must be called before bf_set_antenna_gains");
    return BF_OK;  // takes effect at the next bf_set_geometry
  }
  cudaStream_t st = (cudaStream_t)stream;
  cudaError_t e = cudaSuccess;
  if (c->pending >= 0) {  // regenerate the weights the next run will use
    int rc = wait_event(c, st, c->ev_upd);
    if (rc != BF_OK) return rc;
    c->active = c->pending; c->pending = -1;
    select_buffer(c, c->active);
  }
  if (c->have_gains) e = cudaMemcpyAsync(c->d_gain, c->h_gain.data(), c->h_gain.size() * sizeof(double), cudaMemcpyHostToDevice, st);
  if (e == cudaSuccess) e = upload_i8scale(c, st);
  if (e == cudaSuccess) e = bf_launch_weights(c, st);
  if (e != cudaSuccess) return cuda_fail(c, e, "weight regeneration");
  c->launches += c->d_wop8 ? 2 : 1;
  return BF_OK;
}

extern "C" int bf_get_weights(bf_ctx *c, float *host_out, void *stream) {
  if (!c) return BF_EINVAL;
  if (!host_out) return fail(c, BF_EINVAL, "output pointer is NULL");
  if (!c->have_geom) return fail(c, BF_ENOGEOM, "no geometry set");
  cudaStream_t st = (cudaStream_t)stream;
  if (c->pending >= 0) {  // report the weights the next run will use
    int rc = wait_event(c, st, c->ev_upd);
    if (rc != BF_OK) return rc;
    c->active = c->pending; c->pending = -1;
    select_buffer(c, c->active);
  }
  size_t bytes = (size_t)c->nchan * c->nbeam * c->nant * 2 * sizeof(float);
  float *d = nullptr;  // verification helper: the one place the library allocates device memory itself
  cudaError_t e = cudaMalloc(&d, bytes);
  if (e != cudaSuccess) return cuda_fail(c, e, "cudaMalloc (bf_get_weights)");
  const char *why;
  e = bf_launch_decode_weights(c, d, pick_kernel(c, BF_MODE_POWER, &why) == BF_KERNEL_UMMA_I8, st);
  if (e == cudaSuccess) { c->launches += 1; e = cudaMemcpyAsync(host_out, d, bytes, cudaMemcpyDeviceToHost, st); }
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  cudaFree(d);
  if (e != cudaSuccess) return cuda_fail(c, e, "bf_get_weights");
  return BF_OK;
}

// For bf_weights_noalloc.cu (bf_get_weights_noalloc): the preparation bf_get_weights does before it decodes -- adopt a
// pending tracking update behind its event on `st`, and say which operand bf_run reads (the int8 two-limb one or the
// fp16 one).  The caller has already checked c and have_geom.
int bf_prepare_weight_readback(bf_ctx *c, cudaStream_t st, bool *int8_operand) {
  if (c->pending >= 0) {
    int rc = wait_event(c, st, c->ev_upd);
    if (rc != BF_OK) return rc;
    c->active = c->pending; c->pending = -1;
    select_buffer(c, c->active);
  }
  const char *why;
  *int8_operand = pick_kernel(c, BF_MODE_POWER, &why) == BF_KERNEL_UMMA_I8 && c->d_wop8 != nullptr;
  return BF_OK;
}

// launch the selected kernel over channels [chan0, chan0 + nchan_run); mode BF_MODE_POWER writes `out` as
// fp32 powers, BF_MODE_BEAMS as fp16 (re, im) voltage beams scaled by `scale`
static int launch_range(bf_ctx *c, const void *volt, void *out, int chan0, int nchan_run, cudaStream_t st,
                        int mode = BF_MODE_POWER, float scale = 1.f) {
  BfParams p;
  p.nant = c->nant; p.nbeam = c->nbeam; p.nsamp = c->nsamp; p.nint = c->nint; p.nbin = c->nbin;
  p.nMt = c->nMt; p.nKb = c->nKb;
  p.nchan_run = nchan_run;
  p.volt = volt;
  p.pow = mode == BF_MODE_POWER ? (float *)out : nullptr;
  p.beams = mode == BF_MODE_BEAMS ? out : nullptr;
  p.beam_scale = scale;
  p.mode = mode;
  p.wop = c->d_wop + (size_t)chan0 * (bf_wop_bytes_per_chan(c) / sizeof(__half));
  p.wop_lo = c->d_wop_lo ? c->d_wop_lo + (size_t)chan0 * (bf_wop_bytes_per_chan(c) / sizeof(__half)) : nullptr;
  p.wop8 = c->d_wop8 ? c->d_wop8 + (size_t)chan0 * bf_i8_ncol(c->nbeam) * 64 : nullptr;
  p.i8scale = c->d_i8scale + chan0;
  p.probe = c->d_probe;
  const char *why = "";
  const int k = pick_kernel(c, mode, &why);
  if (k == 0) return fail(c, BF_EUNSUPPORTED, "tensor-core kernel cannot run this shape: %s", why);
  cudaError_t e = k == BF_KERNEL_UMMA_I8    ? bf_launch_umma_i8(p, c->dtype, c->sm_count, st)
                  : k == BF_KERNEL_UMMA_F16 ? bf_launch_umma(p, c->dtype, c->sm_count, st)
                                            : bf_launch_simt(p, c->dtype, st);
  if (e != cudaSuccess) return cuda_fail(c, e, k == BF_KERNEL_SIMT ? "SIMT kernel launch" : "tensor-core kernel launch");
  c->launches += 1;
  return BF_OK;
}

static int check_run(bf_ctx *c, const void *volt, const void *pow) {
  if (!c) return BF_EINVAL;
  if (!volt || !pow) return fail(c, BF_EINVAL, "voltages / powers pointer is NULL");
  if (!c->have_geom) return fail(c, BF_ENOGEOM, "bf_set_geometry has not been called");
  return probe_device(c);
}

// tracking beams (row f3): switch to freshly generated weights once their generator has finished
static int begin_run(bf_ctx *c, cudaStream_t st) {
  if (c->pending >= 0) {
    int rc = wait_event(c, st, c->ev_upd);
    if (rc != BF_OK) return rc;
    c->active = c->pending;
    c->pending = -1;
    select_buffer(c, c->active);
  }
  return BF_OK;
}
// ... and remember when the last reader of the active buffer is done, for the next update of it
static int end_run(bf_ctx *c, cudaStream_t st) {
  if (c->nwbuf != 2) return BF_OK;
  int rc = ensure_wevents(c);
  if (rc == BF_OK) rc = record_event(c, c->ev_use[c->active], st);
  if (rc == BF_OK) c->used[c->active] = true;
  return rc;
}
// a failed launch must still leave the buffer bookkeeping consistent; the first error wins
static int finish_run(bf_ctx *c, cudaStream_t st, int rc) {
  char msg[sizeof(c->err)];
  memcpy(msg, c->err, sizeof(msg));
  const int rc2 = end_run(c, st);
  if (rc != BF_OK) { memcpy(c->err, msg, sizeof(msg)); return rc; }
  return rc2;
}

extern "C" int bf_run(bf_ctx *c, const void *voltages, float *powers, void *stream) {
  int rc = check_run(c, voltages, powers);
  if (rc != BF_OK) return rc;
  if (((uintptr_t)voltages) % 16) return fail(c, BF_EINVAL, "voltages must be 16-byte aligned");
  if (((uintptr_t)powers) % 4) return fail(c, BF_EINVAL, "powers must be 4-byte aligned");
  if ((rc = begin_run(c, (cudaStream_t)stream)) != BF_OK) return rc;
  rc = launch_range(c, voltages, powers, 0, c->nchan, (cudaStream_t)stream);
  return finish_run(c, (cudaStream_t)stream, rc);
}

extern "C" int bf_run_beams(bf_ctx *c, const void *voltages, void *beams, float scale, void *stream) {
  int rc = check_run(c, voltages, beams);
  if (rc != BF_OK) return rc;
  if (((uintptr_t)voltages) % 16) return fail(c, BF_EINVAL, "voltages must be 16-byte aligned");
  if (((uintptr_t)beams) % 4) return fail(c, BF_EINVAL, "beams must be 4-byte aligned");
  if (!isfinite(scale) || scale == 0.f) return fail(c, BF_EINVAL, "scale must be finite and non-zero");
  if ((rc = begin_run(c, (cudaStream_t)stream)) != BF_OK) return rc;
  rc = launch_range(c, voltages, beams, 0, c->nchan, (cudaStream_t)stream, BF_MODE_BEAMS, scale);
  return finish_run(c, (cudaStream_t)stream, rc);
}

extern "C" int bf_run_incoherent(bf_ctx *c, const void *voltages, float *powers, void *stream) {
  if (!c) return BF_EINVAL;
  if (!voltages || !powers) return fail(c, BF_EINVAL, "voltages / powers pointer is NULL");
  int rc = probe_device(c);  // needs neither geometry nor workspace: there are no weights
  if (rc != BF_OK) return rc;
  cudaError_t e = bf_launch_incoherent(c, voltages, powers, (cudaStream_t)stream);
  if (e != cudaSuccess) return cuda_fail(c, e, "incoherent-beam kernel launch");
  c->launches += 1;
  return BF_OK;
}

static int ensure_events(bf_ctx *c) {
  if (c->have_events) return BF_OK;
  for (int i = 0; i < 2; ++i) {
    cudaError_t e = cudaEventCreateWithFlags(&c->ev_copied[i], cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_done[i], cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_kdone[i], cudaEventDisableTiming);
    if (e != cudaSuccess) return cuda_fail(c, e, "cudaEventCreate");
  }
  // the read-back queue of bf_run_host (the one stream the library owns)
  cudaError_t e = cudaStreamCreateWithFlags(&c->d2h_stream, cudaStreamNonBlocking);
  if (e != cudaSuccess) return cuda_fail(c, e, "cudaStreamCreate");
  c->have_events = true;
  return BF_OK;
}

extern "C" size_t bf_staging_bytes(const bf_ctx *c, int chan_per_chunk) {
  if (!c || chan_per_chunk <= 0) return 0;
  if (chan_per_chunk > c->nchan) chan_per_chunk = c->nchan;
  size_t in = align_up((size_t)chan_per_chunk * bf_in_bytes_per_chan(c), BF_ALIGN);
  size_t out = align_up((size_t)chan_per_chunk * c->nbeam * c->nbin * sizeof(float), BF_ALIGN);
  return 2 * (in + out);
}

extern "C" int bf_run_host(bf_ctx *c, const void *host_volt, float *host_pow, void *staging, size_t staging_bytes,
                           int chan_per_chunk, void *compute_stream, void *copy_stream) {
  int rc = check_run(c, host_volt, host_pow);
  if (rc != BF_OK) return rc;
  if (chan_per_chunk <= 0) return fail(c, BF_EINVAL, "chan_per_chunk must be positive");
  if (chan_per_chunk > c->nchan) chan_per_chunk = c->nchan;
  if (!staging || ((uintptr_t)staging) % BF_ALIGN) return fail(c, BF_EINVAL, "staging must be a %d-byte aligned device pointer", BF_ALIGN);
  if (staging_bytes < bf_staging_bytes(c, chan_per_chunk)) return fail(c, BF_ENOMEM, "staging too small");
  if ((rc = ensure_events(c)) != BF_OK) return rc;
  cudaStream_t cs = (cudaStream_t)compute_stream, xs = (cudaStream_t)copy_stream, ds = c->d2h_stream;
  const size_t in_chan = bf_in_bytes_per_chan(c), out_chan = (size_t)c->nbeam * c->nbin * sizeof(float);
  const size_t in_buf = align_up((size_t)chan_per_chunk * in_chan, BF_ALIGN);
  const size_t out_buf = align_up((size_t)chan_per_chunk * out_chan, BF_ALIGN);
  char *in[2] = {(char *)staging, (char *)staging + in_buf};
  char *out[2] = {(char *)staging + 2 * in_buf, (char *)staging + 2 * in_buf + out_buf};
  cudaError_t e;
  int k = 0;
  if ((rc = begin_run(c, cs)) != BF_OK) return rc;
  // Three queues: H2D on the copy stream, kernels on the compute stream, D2H on the library's own stream, so
  // that kernel k+1 never waits for the read-back of chunk k (the step takes "the duration of the
  // slowest stage").  Input half b is free once kernel k-2 has run (ev_kdone), output half b once its D2H is done.
  for (int c0 = 0; c0 < c->nchan && rc == BF_OK; c0 += chan_per_chunk, ++k) {
    const int n = c->nchan - c0 < chan_per_chunk ? c->nchan - c0 : chan_per_chunk;
    const int b = k & 1;
    if (k >= 2 && (rc = wait_event(c, xs, c->ev_kdone[b])) != BF_OK) break;
    e = cudaMemcpyAsync(in[b], (const char *)host_volt + (size_t)c0 * in_chan, (size_t)n * in_chan, cudaMemcpyHostToDevice, xs);
    if (e != cudaSuccess) { rc = cuda_fail(c, e, "voltage H2D copy"); break; }
    if ((rc = record_event(c, c->ev_copied[b], xs)) != BF_OK) break;
    if ((rc = wait_event(c, cs, c->ev_copied[b])) != BF_OK) break;
    if (k >= 2 && (rc = wait_event(c, cs, c->ev_done[b])) != BF_OK) break;   // out[b] has been read back
    if ((rc = launch_range(c, in[b], (float *)out[b], c0, n, cs)) != BF_OK) break;
    if ((rc = record_event(c, c->ev_kdone[b], cs)) != BF_OK) break;
    if ((rc = wait_event(c, ds, c->ev_kdone[b])) != BF_OK) break;
    e = cudaMemcpyAsync((char *)host_pow + (size_t)c0 * out_chan, out[b], (size_t)n * out_chan, cudaMemcpyDeviceToHost, ds);
    if (e != cudaSuccess) { rc = cuda_fail(c, e, "power D2H copy"); break; }
    rc = record_event(c, c->ev_done[b], ds);
  }
  // whoever synchronises the two caller streams has the powers on the host, and the next call on this context
  // cannot overwrite staging that is still in flight
  for (int b = 0; b < (k > 1 ? 2 : 1) && rc == BF_OK && k > 0; ++b) {
    if ((rc = wait_event(c, cs, c->ev_done[b])) != BF_OK) break;
    rc = wait_event(c, xs, c->ev_done[b]);
  }
  // A failure part-way leaves read-backs of earlier chunks queued on the library's own stream: they still write host_pow
  // and read staging, and nothing the caller can synchronise covers them (its streams were not made to wait above).  Do not
  // hand the error back while that DMA is in flight -- the caller may free or reuse both buffers straight away.
  if (rc != BF_OK) (void)cudaStreamSynchronize(ds);
  return finish_run(c, cs, rc);
}

extern "C" int bf_run_streaming(bf_ctx *c, const void *const *host_blocks, int nblocks, float *powers, void *staging,
                                size_t staging_bytes, void *compute_stream, void *copy_stream) {
  int rc = check_run(c, host_blocks, powers);
  if (rc != BF_OK) return rc;
  if (nblocks <= 0) return fail(c, BF_EINVAL, "nblocks must be positive");
  for (int i = 0; i < nblocks; ++i)
    if (!host_blocks[i]) return fail(c, BF_EINVAL, "host block %d is NULL", i);
  const size_t in_bytes = (size_t)c->nchan * bf_in_bytes_per_chan(c);
  const size_t in_buf = align_up(in_bytes, BF_ALIGN);
  if (!staging || ((uintptr_t)staging) % BF_ALIGN) return fail(c, BF_EINVAL, "staging must be a %d-byte aligned device pointer", BF_ALIGN);
  if (staging_bytes < 2 * in_buf) return fail(c, BF_ENOMEM, "staging too small: need %zu", 2 * in_buf);
  if ((rc = ensure_events(c)) != BF_OK) return rc;
  cudaStream_t cs = (cudaStream_t)compute_stream, xs = (cudaStream_t)copy_stream;
  const size_t out_elems = (size_t)c->nchan * c->nbeam * c->nbin;
  char *in[2] = {(char *)staging, (char *)staging + in_buf};
  cudaError_t e;
  if ((rc = begin_run(c, cs)) != BF_OK) return rc;
  int i = 0;
  for (; i < nblocks && rc == BF_OK; ++i) {
    const int b = i & 1;
    if (i >= 2 && (rc = wait_event(c, xs, c->ev_kdone[b])) != BF_OK) break;
    e = cudaMemcpyAsync(in[b], host_blocks[i], in_bytes, cudaMemcpyHostToDevice, xs);
    if (e != cudaSuccess) { rc = cuda_fail(c, e, "block H2D copy"); break; }
    if ((rc = record_event(c, c->ev_copied[b], xs)) != BF_OK) break;
    if ((rc = wait_event(c, cs, c->ev_copied[b])) != BF_OK) break;
    if ((rc = launch_range(c, in[b], powers + (size_t)i * out_elems, 0, c->nchan, cs)) != BF_OK) break;
    rc = record_event(c, c->ev_kdone[b], cs);
  }
  for (int b = 0; b < (i > 1 ? 2 : 1) && rc == BF_OK && i > 0; ++b) rc = wait_event(c, xs, c->ev_kdone[b]);
  return finish_run(c, cs, rc);
}
