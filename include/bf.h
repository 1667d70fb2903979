/*
 * bf.h -- C ABI of the B200-native coherent beamformer (arXiv 1412.4907 hot path).
 *
 * The operation (line numbers are /root/reference/PAPER.md):
 *
 *   W[c][b][n] = exp(-i 2 pi f_c/c0 (r_n . s_b))       steering factor e^{-i k0 . r_n} of Eq. 1
 *                                                      (PAPER.md:23-28), k0 = (2 pi f_c/c0) s_b; the paper
 *                                                      computes these coefficients on the host between
 *                                                      iterations -- here a GPU kernel
 *   y[c][b][t] = sum_n W[c][b][n] x[c][t][n]           per-channel N_b x N_a coefficient matrix times the
 *                                                      antenna vector (Sec. 2.1; Algorithm 1,
 *                                                      PAPER.md:66-98)
 *   P[c][b][j] = sum_{t=j*nint}^{(j+1)*nint-1} |y|^2   "absolute power computation" fused into the kernel
 *                                                      (PAPER.md:62), reduced on the GPU
 *
 * Weights are static between bf_set_geometry calls (the paper's assumption that "beam coefficients
 * do not need to change within small time frames").  No normalisation is applied.
 *
 * Conventions
 *   - plain C, no exceptions cross the ABI; every call returns a bf_status code (or NULL / 0);
 *     bf_last_error(ctx) gives a human-readable message for the last failure on that context.
 *   - "host" / "device" is stated for every pointer.  The caller owns every buffer it passes
 *     (voltages, powers, workspaces); the context owns only its host-side state.
 *   - bf_run only enqueues work on `stream` (a cudaStream_t passed as void*, NULL = default
 *     stream) and returns without synchronising.
 *   - one context per stream; a context is not thread-safe.
 *   - there is NO CPU fallback: without an sm_100 device the compute calls fail with
 *     BF_ECUDA / BF_EUNSUPPORTED.
 */
#ifndef BF_H_
#define BF_H_

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct bf_ctx bf_ctx; /* opaque */

enum bf_status {
  BF_OK = 0,
  BF_EINVAL = -1,       /* bad argument (NULL, non-positive size, nsamp % nint != 0, non-unit direction ...) */
  BF_ENOGEOM = -2,      /* bf_run before bf_set_geometry / bf_set_workspace */
  BF_ECUDA = -3,        /* a CUDA runtime call failed (message in bf_last_error) */
  BF_EUNSUPPORTED = -4, /* device is not sm_100, or a forced kernel cannot run this shape */
  BF_ENOMEM = -5        /* workspace too small / host allocation failed */
};

enum bf_dtype {
  BF_CI8 = 0, /* complex int8, interleaved (re, im): 2 bytes per antenna-sample (BASELINE.json configs) */
  BF_CF16 = 1, /* complex IEEE fp16, interleaved (re, im): 4 bytes per antenna-sample */
  BF_CI4 = 2   /* the paper's F-engine format: 4-bit + 4-bit two's complement in ONE byte per
                  antenna-sample, high nibble real, low nibble imaginary; layout [nchan][nsamp][nant] bytes */
};

enum bf_kernel {
  BF_KERNEL_AUTO = 0, /* pick the fastest kernel that supports the shape.  NOTE: shapes no tensor-core kernel takes -- nant
                         not a multiple of 8 (int8) / 4 (fp16) / 16 (4+4-bit), or an nint below 16 that is no power of two
                         (except on 32 antennas with <= 32 beams, where any EVEN nint integrates on tensor cores when
                         nsamp / nint is a multiple of 128 or >= 512) -- fall through to BF_KERNEL_SIMT without an error,
                         about 30x slower on the `tiny` shape; bf_kernel_name / bf_selected_kernel say which family will
                         run, and BF_KERNEL_UMMA turns the fall-through into BF_EUNSUPPORTED.  Every nint >= 16 that
                         divides nsamp runs on tensor cores */
  BF_KERNEL_SIMT = 1, /* generic fp32 CUDA-core kernel (any shape; Algorithm 1's structure) */
  BF_KERNEL_UMMA = 2, /* tcgen05/TMEM tensor-core kernels with the fused |.|^2 + integrate epilogue (the library
                         picks the variant) */
  BF_KERNEL_UMMA_F16 = 3, /* only the fp16-operand variants (int8 input converted in-kernel) */
  BF_KERNEL_UMMA_I8 = 4   /* only the int8-operand variants (kind::i8, two-limb weights; <= 32 beams, nant <= 32; int8 input, and
                             4+4-bit input on 32 antennas with nint % 4 == 0 and nsamp / nint a multiple of 128 or >= 512) */
};

/*
 * Create a context for nant antennas, nchan channels, nbeam beams, nsamp time samples per channel
 * per bf_run call and an integration length of nint samples (output has nsamp/nint time bins).
 * Pure host call (no CUDA).  Returns NULL if any size is <= 0 or nsamp % nint != 0.
 * The voltage element type defaults to BF_CI8.
 */
bf_ctx *bf_create(int nant, int nchan, int nbeam, int nsamp, int nint);

/* Free the context (host state only; caller-owned device memory is untouched).  NULL is allowed. */
void bf_destroy(bf_ctx *ctx);

/* Select the voltage element type (enum bf_dtype): complex int8 (BASELINE.json configs), complex fp16, or the paper's
 * F-engine wire format, "4-bit, two's complement ... real and imaginary components ... a single byte".
 * Call before bf_workspace_bytes / bf_set_workspace: the workspace layout depends on it, and a different type after
 * bf_set_workspace is refused with BF_EINVAL. */
int bf_set_dtype(bf_ctx *ctx, int dtype);

/* Force a kernel (enum bf_kernel); default BF_KERNEL_AUTO.  All kernels compute the same operation (Sec. 2.1,
 * PAPER.md:60-64); BF_KERNEL_SIMT keeps the structure of the paper's Algorithm 1.  BF_EUNSUPPORTED is reported by bf_run
 * if the forced kernel cannot run the context's shape. */
int bf_set_kernel(bf_ctx *ctx, int kernel);

/* Which kernel family bf_run will launch for this context: BF_KERNEL_SIMT (CUDA cores, Algorithm 1's structure,
 * PAPER.md:66-98) or BF_KERNEL_UMMA (tensor cores: the N_b x N_a matrix product of PAPER.md:62). */
int bf_selected_kernel(const bf_ctx *ctx);

/* Name of the kernel bf_run will launch: "simt", "umma-f16-resident", "umma-f16-binlane", "umma-f16-kblock", "umma-i8". */
const char *bf_kernel_name(const bf_ctx *ctx);

/* Number of kernels this context has launched so far (all streams), for accounting (the bench line's
 * gpu_launches). */
long long bf_launch_count(const bf_ctx *ctx);

/*
 * Device workspace: geometry copy + the weight operand(s) -- the beam coefficients of Eq. 1, kept on
 * the device because they "do not need to change within small time frames".  The caller allocates `bytes` >=
 * bf_workspace_bytes(ctx) of DEVICE memory, 1024-byte aligned, and keeps it alive while the
 * context is used.  Returns BF_EINVAL on NULL / misaligned pointer, BF_ENOMEM if too small.
 */
size_t bf_workspace_bytes(const bf_ctx *ctx);
int bf_set_workspace(bf_ctx *ctx, void *dev_ptr, size_t bytes);

/*
 * Set the array geometry and (re)generate the phase weights on the device (kernel on `stream`):
 *   ant_xyz_m    HOST fp64 [nant][3]   antenna positions r_n in metres
 *   chan_freq_hz HOST fp64 [nchan]     channel centre frequencies f_c in Hz
 *   beam_dir     HOST fp64 [nbeam][3]  unit vectors s_b in the same frame as ant_xyz_m
 * W = exp(-i 2 pi f_c/c0 (r_n . s_b)); the phase is computed and range-reduced in fp64, then rounded
 * to the tensor-core operand type (fp16).  The arrays are copied before the call returns.
 * BF_EINVAL: NULL, non-finite values, | |s_b| - 1 | > 1e-6, f_c <= 0.  BF_ENOGEOM: no workspace yet.
 */
int bf_set_geometry(bf_ctx *ctx, const double *ant_xyz_m, const double *chan_freq_hz,
                    const double *beam_dir, void *stream);

/*
 * Tracking beams.  The paper recomputes the coefficients between pipeline
 * iterations so that "beam pointings [can] change dynamically during pipeline execution, which is useful
 * for tracking observations" (stationary and tracking beams: PAPER.md:180).  With two
 * weight buffers the regeneration overlaps the beamforming of the current block:
 *   bf_set_weight_buffers(ctx, 2)   before bf_workspace_bytes / bf_set_workspace (the workspace doubles)
 *   bf_update_geometry(...)         same arguments and validation as bf_set_geometry, but the new weights are
 *                                   generated into the buffer the kernels are NOT reading, on `update_stream`
 *                                   (any stream; it may differ from the run stream).  Calls to bf_run* that
 *                                   were enqueued before keep the old weights; the NEXT bf_run* call waits (on
 *                                   the device, through an event) for the generator and switches over.  The
 *                                   library also orders a later update behind the last run that still reads
 *                                   the buffer it is about to overwrite, so no host synchronisation is needed.
 * BF_EINVAL without two buffers; BF_ENOGEOM before the first bf_set_geometry.
 */
int bf_set_weight_buffers(bf_ctx *ctx, int n);
int bf_update_geometry(bf_ctx *ctx, const double *ant_xyz_m, const double *chan_freq_hz,
                       const double *beam_dir, void *update_stream);

/*
 * Per-antenna complex gains folded into the weights: W'[c][b][n] = g[c][n] * W[c][b][n].  This is the
 * paper's sub-arraying "antenna mask in the kernel" (g = 0 drops an antenna) and the gain
 * calibration its X-engine provides -- free in the beamforming kernel because only the
 * coefficients change.
 *   gains  HOST fp64, (re, im) pairs: [nant][2] if per_channel == 0, else [nchan][nant][2];
 *          NULL resets all gains to 1.
 * If a geometry is already set the weights are regenerated on `stream`; otherwise the gains take effect
 * at the next bf_set_geometry.  BF_EINVAL: non-finite gain.  BF_ENOGEOM: no workspace yet.
 */
int bf_set_antenna_gains(bf_ctx *ctx, const double *gains, int per_channel, void *stream);

/*
 * Copy the generated weights back as fp32 (re, im) pairs, HOST [nchan][nbeam][nant][2] -- the values
 * the kernels actually use (after rounding to the operand type).  Synchronises `stream`.
 */
int bf_get_weights(bf_ctx *ctx, float *host_out, void *stream);

/*
 * bf_get_weights for callers that must not allocate device memory.  bf_get_weights cudaMalloc's (and cudaFree's) a
 * buffer for the decoded weights; that is out of the question (a) while an observation runs -- cudaFree synchronises
 * the whole device, so reading back the coefficients of a tracking update would stall every stream that
 * is beamforming, (b) in a process whose device memory is owned by a pool (a framework's caching allocator, a backend
 * that sizes everything at start-up), where a raw cudaMalloc fails or steals from the pool, and (c) on any thread while
 * another thread captures a stream in the default global mode, where cudaMalloc is forbidden.  This variant decodes
 * into a fixed array inside the library image instead and calls no cudaMalloc / cudaFree / allocating routine.
 *   chan0, nchan_out  the channels wanted, [chan0, chan0 + nchan_out) inside [0, nchan)
 *   host_out          HOST fp32 (re, im) pairs [nchan_out][nbeam][nant][2]; same values as bf_get_weights gives
 *                     for those channels
 * Limit: nchan_out * nbeam * nant * 8 bytes <= BF_NOALLOC_MAX_BYTES (8 MiB: one channel of 1024 beams x 1024
 * antennas); more is refused with BF_ENOMEM and a message that says how many channels fit -- read a large weight set
 * a few channels per call.  Cost: each GPU on which the process loads this library holds the 8 MiB until exit.
 * The first call on a device looks up the array's device address (no allocation); make that call before any stream
 * capture begins.  All contexts, streams and threads of a process share the one array per GPU: the call synchronises
 * `stream` before it returns and holds a process-wide lock meanwhile, because two such read-backs overlapping on the
 * GPU would overwrite each other's scratch.  Other errors as bf_get_weights (BF_EINVAL, BF_ENOGEOM, BF_ECUDA).
 */
#define BF_NOALLOC_MAX_BYTES (8u << 20)
int bf_get_weights_noalloc(bf_ctx *ctx, int chan0, int nchan_out, float *host_out, void *stream);

/*
 * The hot path.  voltages: DEVICE, [nchan][nsamp][nant][2] (re, im interleaved) of the context's
 * dtype ([nchan][nsamp][nant] bytes for BF_CI4), 16-byte aligned.  powers: DEVICE fp32 [nchan][nbeam][nsamp/nint], 4-byte
 * aligned (16-byte aligned powers with nsamp/nint a multiple of 4 get vector stores), fully overwritten.
 * Enqueues on `stream` and returns.  BF_ENOGEOM before bf_set_geometry; BF_EINVAL for a misaligned pointer.
 *
 * Reproducibility: the result of a call depends only on its inputs -- repeated calls give bit-equal powers (tested: 50
 * launches per kernel, also with randomly delayed barrier waits) -- with ONE exception: an nint that is no power of two
 * <= 64 on the fp16-operand kernels ("umma-f16-resident" / "umma-f16-kblock": multiples of 64 above 64, and any other
 * length >= 16) is integrated with fp32 atomic adds into powers zeroed by a cudaMemsetAsync the call enqueues first; the
 * order of those adds varies, so such results agree from run to run only to fp32 rounding of the partial sums (well
 * inside the 1e-3 bar).
 *
 * CUDA graphs: a bf_run on a context with ONE weight buffer enqueues only a kernel (plus that memset) and may be captured
 * into a graph once the SAME call has been made un-captured before (the first launch of a kernel variant sets function
 * attributes and encodes tensor maps on the host; the maps are then taken from a cache keyed by the buffer addresses).  The
 * captured launch refers to the voltages / powers / workspace addresses it was given.  With two weight buffers the call
 * also records events for bf_update_geometry and is not meant to be captured.
 */
int bf_run(bf_ctx *ctx, const void *voltages, float *powers, void *stream);

/*
 * Voltage-beam output: the raw complex beams y[c][b][t] = sum_n W x, with no
 * detection and no integration -- the S-engine's "electric-field ... beams ... output as 16-bit
 * complex-valued words" for downstream coherent processing.  Same contraction, same kernels,
 * a different epilogue.
 *   beams  DEVICE fp16 (re, im) pairs, [nchan][nbeam][nsamp][2], 4-byte aligned (16-byte aligned and
 *          nsamp % 4 == 0 for vector stores), fully overwritten with fp16(scale * y)
 *   scale  finite, non-zero; choose it so that scale * |y| stays below 65504 (|y| <= nant * max|x|)
 * nint is ignored.  BF_ENOGEOM before bf_set_geometry.
 */
int bf_run_beams(bf_ctx *ctx, const void *voltages, void *beams, float scale, void *stream);

/*
 * Incoherent beam: "squaring and adding the signals of all the elements together"
 * (PAPER.md:21), the wide-field alternative to coherent beams:
 *   powers[c][j] = sum_{t=j*nint}^{(j+1)*nint-1} sum_n |x[c][t][n]|^2     DEVICE fp32 [nchan][nsamp/nint]
 * Needs neither geometry nor workspace (there are no weights).  Integer inputs are summed exactly and
 * rounded once to fp32.
 */
int bf_run_incoherent(bf_ctx *ctx, const void *voltages, float *powers, void *stream);

/*
 * End-to-end variant with HOST buffers (the paper's PCIe concern: "this data overhead
 * can essentially be masked by using two CUDA streams ... however this would also require additional
 * global memory").  The nchan channels are cut into chunks of `chan_per_chunk` channels; chunk k+1 is
 * copied host->device on `copy_stream` while chunk k is beamformed on `compute_stream`, and each chunk's
 * powers are copied back device->host behind its kernel.
 *   host_voltages  HOST (pinned for overlap; pageable works but serialises), same layout as bf_run
 *   host_powers    HOST fp32 [nchan][nbeam][nsamp/nint]
 *   staging        DEVICE scratch of >= bf_staging_bytes(ctx, chan_per_chunk) bytes, 1024-byte aligned
 * Returns after enqueuing; synchronise both streams before reading host_powers.  If the call fails part-way (BF_ECUDA),
 * it first waits for the read-backs it had already queued, so host_powers and staging are not touched after it returns.
 */
size_t bf_staging_bytes(const bf_ctx *ctx, int chan_per_chunk);
int bf_run_host(bf_ctx *ctx, const void *host_voltages, float *host_powers, void *staging,
                size_t staging_bytes, int chan_per_chunk, void *compute_stream, void *copy_stream);

/*
 * Streaming mode: `nblocks` consecutive input blocks, each one bf_run input, in (pinned) HOST memory
 * at host_blocks[i]; powers: DEVICE fp32, nblocks outputs back to back.  Block i+1 is copied on
 * `copy_stream` into one of two staging buffers while block i runs on `compute_stream`
 * (PAPER.md:140).  staging: DEVICE scratch of >= 2 * (one bf_run input) bytes.
 */
int bf_run_streaming(bf_ctx *ctx, const void *const *host_blocks, int nblocks, float *powers,
                     void *staging, size_t staging_bytes, void *compute_stream, void *copy_stream);

/*
 * Measurement hook: when `dev_u64x4` is a non-NULL DEVICE pointer to four 64-bit words,
 * CTA 0 of every hot-path kernel the context launches afterwards writes
 *   { clock64 at start, globaltimer (ns) at start, clock64 at end, globaltimer (ns) at end }
 * so the caller can compute the SM clock the kernel really ran at, (c1 - c0) / (t1 - t0) GHz -- nvidia-smi's
 * sampled clock is too coarse for a millisecond kernel.  NULL switches it off (the default).  Two scalar
 * stores per launch; no effect on the result.  The four words must stay allocated until the probe is switched off (NULL)
 * or the context is destroyed and every launch made meanwhile has finished: the library keeps only the address.
 */
int bf_set_clock_probe(bf_ctx *ctx, void *dev_u64x4);

/* Message for the last error on this context ("" if none).  Valid until the next call on ctx.  (Error reporting of the
 * ABI itself; no passage of the paper.) */
const char *bf_last_error(const bf_ctx *ctx);

/* Library version string (names the target architecture, sm_100a). */
const char *bf_version(void);

#ifdef __cplusplus
}
#endif
#endif /* BF_H_ */
