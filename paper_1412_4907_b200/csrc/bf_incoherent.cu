// bf_incoherent.cu -- incoherent beam.
//
// "Squaring and adding the signals of all the elements together is the process of incoherent
// beamforming"; the paper names it as the way to trade sensitivity for maximal field of
// view.  No weights and no geometry:
//     P_inc[c][j] = sum_{t in bin j} sum_n |x[c][t][n]|^2
// In the [chan][time][ant] layout a bin is ONE contiguous run of nint * nant samples, so this is a pure
// streaming reduction: every input byte is read once, 4 bytes are written per bin -- HBM-bound, nothing
// for the tensor cores to do.  One warp per bin (bins up to 16 KiB) or one block per bin (larger), 16-byte
// loads, int8 squares by DP4A (exact in integers, widened to 64 bits across the warp), fp16 in fp32.
#include "bf_internal.h"

namespace {

// sum of squares of the 16 int8 values in v (each dp4a <= 4 * 128^2, so a thread can take 2^14 pieces)
__device__ __forceinline__ unsigned sq_i8x16(uint4 v, unsigned acc) {
  acc = (unsigned)__dp4a((int)v.x, (int)v.x, (int)acc);
  acc = (unsigned)__dp4a((int)v.y, (int)v.y, (int)acc);
  acc = (unsigned)__dp4a((int)v.z, (int)v.z, (int)acc);
  acc = (unsigned)__dp4a((int)v.w, (int)v.w, (int)acc);
  return acc;
}
// 4+4-bit two's complement nibbles: split a word into its 4 high and 4 low nibbles u, form
// x = u ^ 8 (0..15) and the signed value x - 8 per byte as x + 0xF8 without carries between bytes: add the
// low 7 bits (x + 0x78 <= 0x87 stays inside the byte), then flip bit 7.  The bytes are then int8 values
// in -8..7 and DP4A squares them.
__device__ __forceinline__ unsigned sq_i4x8(unsigned w, unsigned acc) {
  const unsigned hi = ((w >> 4) & 0x0F0F0F0Fu) ^ 0x08080808u, lo = (w & 0x0F0F0F0Fu) ^ 0x08080808u;
  const unsigned h = (hi + 0x78787878u) ^ 0x80808080u;
  const unsigned l = (lo + 0x78787878u) ^ 0x80808080u;
  acc = (unsigned)__dp4a((int)h, (int)h, (int)acc);
  acc = (unsigned)__dp4a((int)l, (int)l, (int)acc);
  return acc;
}
__device__ __forceinline__ float sq_f16x8(uint4 v, float acc) {
  const unsigned w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    const float2 f = __half22float2(*reinterpret_cast<const __half2 *>(&w[k]));
    acc = fmaf(f.x, f.x, acc);
    acc = fmaf(f.y, f.y, acc);
  }
  return acc;
}

// BLOCK_PER_BIN = false: a warp owns a bin; true: the block's warps share one bin (combined through shared memory)
template <int DTYPE, bool BLOCK_PER_BIN>
__global__ void __launch_bounds__(256) bf_incoherent_kernel(const void *__restrict__ volt, float *__restrict__ out,
                                                            long long nbins, long long bin_bytes, int vec_ok) {
  __shared__ double part[8];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
  const long long stride = BLOCK_PER_BIN ? gridDim.x : (long long)gridDim.x * nwarp;
  for (long long bin = BLOCK_PER_BIN ? blockIdx.x : (long long)blockIdx.x * nwarp + warp; bin < nbins; bin += stride) {
    const unsigned char *src = reinterpret_cast<const unsigned char *>(volt) + bin * bin_bytes;
    const int t0 = BLOCK_PER_BIN ? threadIdx.x : lane, tstep = BLOCK_PER_BIN ? blockDim.x : 32;
    unsigned long long isum = 0;
    float fsum = 0.f;
    if (vec_ok) {
      const uint4 *s4 = reinterpret_cast<const uint4 *>(src);
      const long long np = bin_bytes >> 4;
      unsigned acc = 0;
      int cnt = 0;
      for (long long i = t0; i < np; i += tstep) {
        const uint4 v = __ldg(s4 + i);
        if (DTYPE == BF_CI8) acc = sq_i8x16(v, acc);
        else if (DTYPE == BF_CI4) { acc = sq_i4x8(v.x, acc); acc = sq_i4x8(v.y, acc); acc = sq_i4x8(v.z, acc); acc = sq_i4x8(v.w, acc); }
        else fsum = sq_f16x8(v, fsum);
        if (++cnt == 8192) { isum += acc; acc = 0; cnt = 0; }   // 8192 * 16 * 128^2 < 2^32
      }
      isum += acc;
    } else {  // unaligned bins (odd nint * nant): one element at a time
      if (DTYPE == BF_CF16) {
        const __half *h = reinterpret_cast<const __half *>(src);
        for (long long i = t0; i < (bin_bytes >> 1); i += tstep) { const float f = __half2float(h[i]); fsum = fmaf(f, f, fsum); }
      } else {
        for (long long i = t0; i < bin_bytes; i += tstep) {
          const int b = src[i];
          if (DTYPE == BF_CI8) { const int x = (signed char)b; isum += (unsigned)(x * x); }
          else { const int re = ((b >> 4) ^ 8) - 8, im = ((b & 15) ^ 8) - 8; isum += (unsigned)(re * re + im * im); }
        }
      }
    }
    double tot;
    if (DTYPE == BF_CF16) {
#pragma unroll
      for (int o = 16; o >= 1; o >>= 1) fsum += __shfl_xor_sync(0xffffffffu, fsum, o);
      tot = (double)fsum;
    } else {
#pragma unroll
      for (int o = 16; o >= 1; o >>= 1) isum += __shfl_xor_sync(0xffffffffu, isum, o);
      tot = (double)isum;  // exact below 2^53
    }
    if (!BLOCK_PER_BIN) {
      if (lane == 0) out[bin] = (float)tot;
    } else {
      __syncthreads();
      if (lane == 0) part[warp] = tot;
      __syncthreads();
      if (threadIdx.x == 0) {
        double s = 0.0;
        for (int w = 0; w < nwarp; ++w) s += part[w];
        out[bin] = (float)s;
      }
    }
  }
}

template <int DTYPE>
cudaError_t launch(const void *volt, float *out, long long nbins, long long bin_bytes, int sm_count, cudaStream_t st) {
  const int vec_ok = (bin_bytes % 16 == 0) && ((reinterpret_cast<uintptr_t>(volt) & 15) == 0);
  if (bin_bytes > 16384) {
    const long long g = nbins < (long long)sm_count * 8 ? nbins : (long long)sm_count * 8;
    bf_incoherent_kernel<DTYPE, true><<<(unsigned)g, 256, 0, st>>>(volt, out, nbins, bin_bytes, vec_ok);
  } else {
    const long long need = (nbins + 7) / 8;
    const long long g = need < (long long)sm_count * 8 ? need : (long long)sm_count * 8;
    bf_incoherent_kernel<DTYPE, false><<<(unsigned)g, 256, 0, st>>>(volt, out, nbins, bin_bytes, vec_ok);
  }
  return cudaGetLastError();
}

}  // namespace

cudaError_t bf_launch_incoherent(const bf_ctx *c, const void *volt, float *out, cudaStream_t st) {
  const long long nbins = (long long)c->nchan * c->nbin;
  const long long bin_bytes = (long long)c->nint * c->nant * (c->dtype == BF_CI8 ? 2 : c->dtype == BF_CI4 ? 1 : 4);
  const int sms = c->sm_count > 0 ? c->sm_count : 148;
  if (c->dtype == BF_CI8) return launch<BF_CI8>(volt, out, nbins, bin_bytes, sms, st);
  if (c->dtype == BF_CI4) return launch<BF_CI4>(volt, out, nbins, bin_bytes, sms, st);
  return launch<BF_CF16>(volt, out, nbins, bin_bytes, sms, st);
}
