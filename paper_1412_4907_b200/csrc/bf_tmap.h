// bf_tmap.h -- host-side helpers shared by the kernels that use TMA tensor copies: the driver entry point for
// cuTensorMapEncodeTiled (resolved through the runtime, so the library links against libcudart only) and a small
// cache of encoded maps.  The maps depend only on (pointer, nant, nsamp, nchan, view): a streaming caller alternates
// between a few buffers, so the last few encodings are kept (host-side cost only; launch-bound shapes notice).
#pragma once
#include <cuda.h>

#include "bf_internal.h"

typedef CUresult (*PFN_encodeTiled)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                    const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

inline PFN_encodeTiled bf_get_encode() {
  static PFN_encodeTiled fn = nullptr;
  if (!fn) {
    void *ptr = nullptr;
    cudaDriverEntryPointQueryResult qres;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ptr, cudaEnableDefault, &qres) == cudaSuccess &&
        qres == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<PFN_encodeTiled>(ptr);
  }
  return fn;
}

// view: which tensor-map recipe (each kernel numbers its own), rows: box rows
struct BfTmapKey { const void *ptr; int nant, nsamp, nchan, view, rows; };
struct BfTmapSlot { BfTmapKey k; CUtensorMap tm; bool used; };

template <typename F>
inline cudaError_t bf_cached_tmap(CUtensorMap *tm, const BfParams &p, int view, int rows, F make) {
  static thread_local BfTmapSlot slots[16];
  static thread_local int next = 0;
  const BfTmapKey k = {p.volt, p.nant, p.nsamp, p.nchan_run, view, rows};
  for (BfTmapSlot &s : slots)
    if (s.used && s.k.ptr == k.ptr && s.k.nant == k.nant && s.k.nsamp == k.nsamp && s.k.nchan == k.nchan &&
        s.k.view == k.view && s.k.rows == k.rows) { *tm = s.tm; return cudaSuccess; }
  cudaError_t e = make(tm, p, rows);
  if (e != cudaSuccess) return e;
  BfTmapSlot &s = slots[next];
  next = (next + 1) % 16;
  s.k = k; s.tm = *tm; s.used = true;
  return cudaSuccess;
}

// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) once per kernel instantiation and device, not per launch
template <typename K>
inline cudaError_t bf_set_smem_once(K kern, size_t smem, int *done_dev) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (*done_dev == dev) return cudaSuccess;
  e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e == cudaSuccess) *done_dev = dev;
  return e;
}
