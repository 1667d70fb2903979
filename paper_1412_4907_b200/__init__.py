"""paper_1412_4907_b200 -- thin Python binding over the C-ABI beamformer library (include/bf.h).

Argument marshalling only: every step of the hot path (weights, ingest, contraction, |.|^2,
integration) runs in the CUDA kernels under ``csrc/``.  PyTorch is used by callers for device
memory and streams; this module itself needs only ctypes.  There is no CPU fallback: if
``libbf.so`` has not been built (``python -m paper_1412_4907_b200.build``) loading fails loudly.

The functions carry the same names as the C entry points (bf_create, bf_set_geometry, bf_run ...).
``Beamformer`` is a small convenience wrapper that owns the context and a torch workspace.
"""
from __future__ import annotations

import ctypes
import os

_HERE = os.path.dirname(os.path.abspath(__file__))
# BF_LIBRARY: load another build of the same library instead (the tests point it at the jitter build, libbf_jitter.so)
LIB_PATH = os.environ.get("BF_LIBRARY") or os.path.join(_HERE, "libbf.so")

BF_OK, BF_EINVAL, BF_ENOGEOM, BF_ECUDA, BF_EUNSUPPORTED, BF_ENOMEM = 0, -1, -2, -3, -4, -5
BF_CI8, BF_CF16, BF_CI4 = 0, 1, 2
BF_KERNEL_AUTO, BF_KERNEL_SIMT, BF_KERNEL_UMMA, BF_KERNEL_UMMA_F16, BF_KERNEL_UMMA_I8 = 0, 1, 2, 3, 4

# every symbol include/bf.h declares: name -> (restype, argtypes)
_vp, _i, _sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_size_t
_dp = ctypes.POINTER(ctypes.c_double)
SYMBOLS = {
    "bf_create": (_vp, [_i, _i, _i, _i, _i]),
    "bf_destroy": (None, [_vp]),
    "bf_set_dtype": (_i, [_vp, _i]),
    "bf_set_kernel": (_i, [_vp, _i]),
    "bf_selected_kernel": (_i, [_vp]),
    "bf_kernel_name": (ctypes.c_char_p, [_vp]),
    "bf_launch_count": (ctypes.c_longlong, [_vp]),
    "bf_workspace_bytes": (_sz, [_vp]),
    "bf_set_workspace": (_i, [_vp, _vp, _sz]),
    "bf_set_geometry": (_i, [_vp, _dp, _dp, _dp, _vp]),
    "bf_set_antenna_gains": (_i, [_vp, _dp, _i, _vp]),
    "bf_get_weights": (_i, [_vp, _vp, _vp]),
    "bf_get_weights_noalloc": (_i, [_vp, _i, _i, _vp, _vp]),
    "bf_run": (_i, [_vp, _vp, _vp, _vp]),
    "bf_run_beams": (_i, [_vp, _vp, _vp, ctypes.c_float, _vp]),
    "bf_run_incoherent": (_i, [_vp, _vp, _vp, _vp]),
    "bf_set_weight_buffers": (_i, [_vp, _i]),
    "bf_update_geometry": (_i, [_vp, _dp, _dp, _dp, _vp]),
    "bf_staging_bytes": (_sz, [_vp, _i]),
    "bf_run_host": (_i, [_vp, _vp, _vp, _vp, _sz, _i, _vp, _vp]),
    "bf_run_streaming": (_i, [_vp, ctypes.POINTER(_vp), _i, _vp, _vp, _sz, _vp, _vp]),
    "bf_set_clock_probe": (_i, [_vp, _vp]),
    "bf_last_error": (ctypes.c_char_p, [_vp]),
    "bf_version": (ctypes.c_char_p, []),
}

_lib = None


class BfError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"bf error {code}: {msg}")
        self.code = code


def lib() -> ctypes.CDLL:
    """Load libbf.so (built in-tree).  Fails loudly if it is missing -- there is no fallback."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} not found: build it with `python -m paper_1412_4907_b200.build`")
        L = ctypes.CDLL(LIB_PATH)
        for name, (res, args) in SYMBOLS.items():
            fn = getattr(L, name)
            fn.restype = res
            fn.argtypes = args
        _lib = L
    return _lib


def _ptr(x):
    """Raw address of a torch tensor / numpy array / int / None."""
    if x is None:
        return None
    if isinstance(x, int):
        return x
    if hasattr(x, "data_ptr"):
        return x.data_ptr()
    if hasattr(x, "ctypes"):
        return x.ctypes.data
    raise TypeError(type(x))


def _stream(s):
    if s is None:
        return None
    return s.cuda_stream if hasattr(s, "cuda_stream") else int(s)


# ---- same-name wrappers (marshalling only) ---------------------------------------------------
def bf_create(nant, nchan, nbeam, nsamp, nint):
    return lib().bf_create(int(nant), int(nchan), int(nbeam), int(nsamp), int(nint))


def bf_destroy(ctx):
    lib().bf_destroy(ctx)


def bf_set_dtype(ctx, dtype):
    return lib().bf_set_dtype(ctx, int(dtype))


def bf_set_kernel(ctx, kernel):
    return lib().bf_set_kernel(ctx, int(kernel))


def bf_selected_kernel(ctx):
    return lib().bf_selected_kernel(ctx)


def bf_kernel_name(ctx):
    return lib().bf_kernel_name(ctx).decode()


def bf_launch_count(ctx):
    return int(lib().bf_launch_count(ctx))


def bf_workspace_bytes(ctx):
    return int(lib().bf_workspace_bytes(ctx))


def bf_set_workspace(ctx, dev_ptr, nbytes):
    return lib().bf_set_workspace(ctx, _ptr(dev_ptr), int(nbytes))


def bf_set_geometry(ctx, ant_xyz_m, chan_freq_hz, beam_dir, stream=None):
    import numpy as np

    def dp(a):
        if a is None:
            return None, None
        a = np.ascontiguousarray(a, dtype=np.float64)
        return a, a.ctypes.data_as(_dp)
    a, pa = dp(ant_xyz_m)
    f, pf = dp(chan_freq_hz)
    d, pd = dp(beam_dir)
    return lib().bf_set_geometry(ctx, pa, pf, pd, _stream(stream))


def bf_set_weight_buffers(ctx, n):
    return lib().bf_set_weight_buffers(ctx, int(n))


def bf_update_geometry(ctx, ant_xyz_m, chan_freq_hz, beam_dir, update_stream=None):
    import numpy as np

    a = np.ascontiguousarray(ant_xyz_m, dtype=np.float64)
    f = np.ascontiguousarray(chan_freq_hz, dtype=np.float64)
    d = np.ascontiguousarray(beam_dir, dtype=np.float64)
    return lib().bf_update_geometry(ctx, a.ctypes.data_as(_dp), f.ctypes.data_as(_dp), d.ctypes.data_as(_dp),
                                    _stream(update_stream))


def bf_set_antenna_gains(ctx, gains, per_channel=False, stream=None):
    """gains: complex array [nant] (or [nchan][nant] with per_channel), or None to reset to 1."""
    import numpy as np

    if gains is None:
        return lib().bf_set_antenna_gains(ctx, None, 0, _stream(stream))
    g = np.ascontiguousarray(np.asarray(gains, dtype=np.complex128))
    return lib().bf_set_antenna_gains(ctx, g.view(np.float64).ctypes.data_as(_dp), 1 if per_channel else 0, _stream(stream))


def bf_get_weights(ctx, host_out, stream=None):
    return lib().bf_get_weights(ctx, _ptr(host_out), _stream(stream))


BF_NOALLOC_MAX_BYTES = 8 << 20  # include/bf.h


def bf_get_weights_noalloc(ctx, chan0, nchan_out, host_out, stream=None):
    """bf_get_weights without cudaMalloc / cudaFree (for callers that must not allocate on the device: a running
    observation, a process whose memory belongs to a pool, a thread beside a global-mode stream capture).  At most
    BF_NOALLOC_MAX_BYTES of weights per call -- see include/bf.h."""
    return lib().bf_get_weights_noalloc(ctx, int(chan0), int(nchan_out), _ptr(host_out), _stream(stream))


def bf_run(ctx, voltages, powers, stream=None):
    return lib().bf_run(ctx, _ptr(voltages), _ptr(powers), _stream(stream))


def bf_run_beams(ctx, voltages, beams, scale=1.0, stream=None):
    return lib().bf_run_beams(ctx, _ptr(voltages), _ptr(beams), float(scale), _stream(stream))


def bf_run_incoherent(ctx, voltages, powers, stream=None):
    return lib().bf_run_incoherent(ctx, _ptr(voltages), _ptr(powers), _stream(stream))


def bf_staging_bytes(ctx, chan_per_chunk):
    return int(lib().bf_staging_bytes(ctx, int(chan_per_chunk)))


def bf_run_host(ctx, host_voltages, host_powers, staging, staging_bytes, chan_per_chunk, compute_stream=None,
                copy_stream=None):
    return lib().bf_run_host(ctx, _ptr(host_voltages), _ptr(host_powers), _ptr(staging), int(staging_bytes),
                             int(chan_per_chunk), _stream(compute_stream), _stream(copy_stream))


def bf_run_streaming(ctx, host_blocks, powers, staging, staging_bytes, compute_stream=None, copy_stream=None):
    n = len(host_blocks)
    arr = (_vp * n)(*[_ptr(b) for b in host_blocks])
    return lib().bf_run_streaming(ctx, arr, n, _ptr(powers), _ptr(staging), int(staging_bytes),
                                  _stream(compute_stream), _stream(copy_stream))


def bf_set_clock_probe(ctx, dev_u64x4):
    return lib().bf_set_clock_probe(ctx, _ptr(dev_u64x4))


def bf_last_error(ctx):
    s = lib().bf_last_error(ctx)
    return s.decode() if s else ""


def bf_version():
    return lib().bf_version().decode()


# ---- convenience wrapper ---------------------------------------------------------------------
class Beamformer:
    """Owns a bf_ctx plus its device workspace (a torch uint8 tensor)."""

    def __init__(self, nant, nchan, nbeam, nsamp, nint, dtype=BF_CI8, kernel=BF_KERNEL_AUTO, device="cuda:0",
                 weight_buffers=1):
        import torch

        self.shape = (nant, nchan, nbeam, nsamp, nint)
        self.ctx = bf_create(nant, nchan, nbeam, nsamp, nint)
        if not self.ctx:
            raise BfError(BF_EINVAL, "bf_create rejected the sizes (all > 0, nsamp % nint == 0)")
        self._check(bf_set_dtype(self.ctx, dtype))
        self._check(bf_set_kernel(self.ctx, kernel))
        self._check(bf_set_weight_buffers(self.ctx, weight_buffers))
        self.dtype = dtype
        self.device = torch.device(device)
        nbytes = bf_workspace_bytes(self.ctx)
        self.workspace = torch.empty(nbytes + 1024, dtype=torch.uint8, device=self.device)
        off = (-self.workspace.data_ptr()) % 1024
        self._check(bf_set_workspace(self.ctx, self.workspace.data_ptr() + off, nbytes))
        self._staging = None
        self._probe = None   # the tensor bf_set_clock_probe points at, kept alive while the library may write to it

    def _check(self, rc):
        if rc != BF_OK:
            raise BfError(rc, bf_last_error(self.ctx))

    @property
    def nbin(self):
        return self.shape[3] // self.shape[4]

    def set_geometry(self, ant_xyz_m, chan_freq_hz, beam_dir, stream=None):
        self._check(bf_set_geometry(self.ctx, ant_xyz_m, chan_freq_hz, beam_dir, stream))

    def update_geometry(self, ant_xyz_m, chan_freq_hz, beam_dir, update_stream=None):
        """Tracking beams: regenerate the weights into the inactive buffer on `update_stream`."""
        self._check(bf_update_geometry(self.ctx, ant_xyz_m, chan_freq_hz, beam_dir, update_stream))

    def set_antenna_gains(self, gains, per_channel=False, stream=None):
        self._check(bf_set_antenna_gains(self.ctx, gains, per_channel, stream))

    def weights(self):
        import numpy as np

        nant, nchan, nbeam = self.shape[:3]
        out = np.empty((nchan, nbeam, nant, 2), dtype=np.float32)
        self._check(bf_get_weights(self.ctx, out))
        return out[..., 0] + 1j * out[..., 1]

    def weights_noalloc(self):
        """weights() through bf_get_weights_noalloc: no device allocation, as many channels per call as fit."""
        import numpy as np

        nant, nchan, nbeam = self.shape[:3]
        out = np.empty((nchan, nbeam, nant, 2), dtype=np.float32)
        step = max(1, BF_NOALLOC_MAX_BYTES // (nbeam * nant * 8))
        for c0 in range(0, nchan, step):
            n = min(step, nchan - c0)
            self._check(bf_get_weights_noalloc(self.ctx, c0, n, out[c0:c0 + n]))
        return out[..., 0] + 1j * out[..., 1]

    def empty_powers(self):
        import torch

        nant, nchan, nbeam, nsamp, nint = self.shape
        return torch.empty((nchan, nbeam, nsamp // nint), dtype=torch.float32, device=self.device)

    def run(self, voltages, powers=None, stream=None):
        import torch

        if powers is None:
            powers = self.empty_powers()
        if stream is None:
            stream = torch.cuda.current_stream(self.device)
        self._check(bf_run(self.ctx, voltages, powers, stream))
        return powers

    def run_beams(self, voltages, beams=None, scale=1.0, stream=None):
        """Voltage beams y[c][b][t] as fp16 (re, im): tensor [nchan][nbeam][nsamp][2]."""
        import torch

        nant, nchan, nbeam, nsamp, nint = self.shape
        if beams is None:
            beams = torch.empty((nchan, nbeam, nsamp, 2), dtype=torch.float16, device=self.device)
        if stream is None:
            stream = torch.cuda.current_stream(self.device)
        self._check(bf_run_beams(self.ctx, voltages, beams, scale, stream))
        return beams

    def run_incoherent(self, voltages, powers=None, stream=None):
        """Incoherent beam sum_n |x_n|^2 integrated over nint: tensor [nchan][nsamp // nint] fp32."""
        import torch

        nant, nchan, nbeam, nsamp, nint = self.shape
        if powers is None:
            powers = torch.empty((nchan, nsamp // nint), dtype=torch.float32, device=self.device)
        if stream is None:
            stream = torch.cuda.current_stream(self.device)
        self._check(bf_run_incoherent(self.ctx, voltages, powers, stream))
        return powers

    def _get_staging(self, nbytes):
        import torch

        if self._staging is None or self._staging.numel() < nbytes + 1024:
            self._staging = torch.empty(nbytes + 1024, dtype=torch.uint8, device=self.device)
        off = (-self._staging.data_ptr()) % 1024
        return self._staging.data_ptr() + off

    def run_host(self, host_voltages, host_powers, chan_per_chunk, compute_stream, copy_stream):
        nbytes = bf_staging_bytes(self.ctx, chan_per_chunk)
        st = self._get_staging(nbytes)
        self._check(bf_run_host(self.ctx, host_voltages, host_powers, st, nbytes, chan_per_chunk, compute_stream,
                                copy_stream))

    def run_streaming(self, host_blocks, powers, compute_stream, copy_stream):
        nant, nchan, nbeam, nsamp, nint = self.shape
        in_bytes = nchan * nsamp * nant * {BF_CI8: 2, BF_CF16: 4, BF_CI4: 1}[self.dtype]
        nbytes = 2 * ((in_bytes + 1023) // 1024 * 1024)
        st = self._get_staging(nbytes)
        self._check(bf_run_streaming(self.ctx, host_blocks, powers, st, nbytes, compute_stream, copy_stream))

    def set_clock_probe(self, dev_u64x4):
        """dev_u64x4: torch int64 tensor of 4 elements on the device (or None): see bf_set_clock_probe.  The library keeps
        only the address and every later launch writes there, so this object holds on to the tensor until the probe is
        switched off or the context is closed."""
        if dev_u64x4 is not None:
            import torch

            if not (isinstance(dev_u64x4, torch.Tensor) and dev_u64x4.is_cuda and dev_u64x4.dtype == torch.int64
                    and dev_u64x4.numel() >= 4 and dev_u64x4.is_contiguous()):
                raise BfError(BF_EINVAL, "clock probe must be a contiguous int64 CUDA tensor of at least 4 elements")
        self._check(bf_set_clock_probe(self.ctx, dev_u64x4))
        self._probe = dev_u64x4

    @property
    def selected_kernel(self):
        return bf_selected_kernel(self.ctx)

    @property
    def kernel_name(self):
        return bf_kernel_name(self.ctx)

    @property
    def launches(self):
        return bf_launch_count(self.ctx)

    def close(self):
        if self.ctx:
            bf_destroy(self.ctx)
            self.ctx = None
        self._probe = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
