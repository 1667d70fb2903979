"""ORACLE -- test infrastructure only (see bf_oracle.c header).

A ctypes loader for the plain fp64 CPU beamformer in ``bf_oracle.c``.  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may
import this package.  It imports nothing from ``paper_1412_4907_b200`` and shares no code with it.

Operation: arXiv 1412.4907 Eq. 1 steering weights, per-channel
matrix-vector beamforming and absolute power integrated over ``nint``
samples.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "bf_oracle.c")
_LIB = os.path.join(_HERE, "libbf_oracle.so")

CI8, CF16, C128, CI4 = 0, 1, 2, 3
_lib = None


def build(force: bool = False) -> str:
    """Compile bf_oracle.c with gcc (-O2 -fopenmp). Building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11", "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB)
        dp = ctypes.POINTER(ctypes.c_double)
        lib.oracle_num_threads.restype = ctypes.c_int
        lib.oracle_weights.restype = ctypes.c_int
        lib.oracle_weights.argtypes = [ctypes.c_int] * 3 + [dp, dp, dp, dp]
        lib.oracle_beamform.restype = ctypes.c_int
        lib.oracle_beamform.argtypes = [ctypes.c_int] * 6 + [dp, dp, dp, ctypes.c_void_p, dp, ctypes.c_int]
        lib.oracle_beams.restype = ctypes.c_int
        lib.oracle_beams.argtypes = [ctypes.c_int] * 5 + [dp, dp, dp, ctypes.c_void_p, dp]
        lib.oracle_incoherent.restype = ctypes.c_int
        lib.oracle_incoherent.argtypes = [ctypes.c_int] * 5 + [ctypes.c_void_p, dp]
        _lib = lib
    return _lib


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _geom(ant_xyz, chan_freq_hz, beam_dir):
    r = np.ascontiguousarray(ant_xyz, dtype=np.float64).reshape(-1, 3)
    f = np.ascontiguousarray(chan_freq_hz, dtype=np.float64).reshape(-1)
    s = np.ascontiguousarray(beam_dir, dtype=np.float64).reshape(-1, 3)
    return r, f, s


def _volt(voltages, nchan, nant):
    """Accept int8 [C][T][N][2], float16 [C][T][N][2], complex128 [C][T][N], or uint8 [C][T][N]
    (4+4-bit packed complex, high nibble real: PAPER.md:102)."""
    v = np.ascontiguousarray(voltages)
    if v.dtype == np.uint8:
        dt = CI4
    elif v.dtype == np.int8:
        dt = CI8
    elif v.dtype == np.float16:
        dt = CF16
    elif v.dtype == np.complex128:
        dt = C128
    else:
        raise TypeError(f"unsupported voltage dtype {v.dtype}")
    if dt in (C128, CI4):
        if v.ndim != 3 or v.shape[0] != nchan or v.shape[2] != nant:
            raise ValueError(f"bad voltage shape {v.shape}")
    else:
        if v.ndim != 4 or v.shape[0] != nchan or v.shape[2] != nant or v.shape[3] != 2:
            raise ValueError(f"bad voltage shape {v.shape}")
    return v, dt, v.shape[1]


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def weights(ant_xyz, chan_freq_hz, beam_dir) -> np.ndarray:
    """W[c][b][n] complex128 (Eq. 1 steering factor)."""
    r, f, s = _geom(ant_xyz, chan_freq_hz, beam_dir)
    out = np.empty((f.size, s.shape[0], r.shape[0]), dtype=np.complex128)
    rc = _load().oracle_weights(r.shape[0], f.size, s.shape[0], _dp(r), _dp(f), _dp(s), _dp(out.view(np.float64)))
    if rc != 0:
        raise ValueError(f"oracle_weights failed rc={rc}")
    return out


def beamform(ant_xyz, chan_freq_hz, beam_dir, voltages, nint: int, chan_stride: int = 1) -> np.ndarray:
    """P[c][b][j] fp64: the whole hot path.  Channels with c % chan_stride != 0 are left as NaN."""
    r, f, s = _geom(ant_xyz, chan_freq_hz, beam_dir)
    v, dt, nsamp = _volt(voltages, f.size, r.shape[0])
    if nint <= 0 or nsamp % nint != 0:
        raise ValueError("nsamp must be a positive multiple of nint")
    out = np.full((f.size, s.shape[0], nsamp // nint), np.nan, dtype=np.float64)
    rc = _load().oracle_beamform(r.shape[0], f.size, s.shape[0], nsamp, nint, dt, _dp(r), _dp(f), _dp(s),
                                 v.ctypes.data_as(ctypes.c_void_p), _dp(out), chan_stride)
    if rc != 0:
        raise ValueError(f"oracle_beamform failed rc={rc}")
    return out


def beams(ant_xyz, chan_freq_hz, beam_dir, voltages) -> np.ndarray:
    """Raw complex beams y[c][b][t] complex128 (small cases only)."""
    r, f, s = _geom(ant_xyz, chan_freq_hz, beam_dir)
    v, dt, nsamp = _volt(voltages, f.size, r.shape[0])
    out = np.empty((f.size, s.shape[0], nsamp), dtype=np.complex128)
    rc = _load().oracle_beams(r.shape[0], f.size, s.shape[0], nsamp, dt, _dp(r), _dp(f), _dp(s),
                              v.ctypes.data_as(ctypes.c_void_p), _dp(out.view(np.float64)))
    if rc != 0:
        raise ValueError(f"oracle_beams failed rc={rc}")
    return out


def incoherent(voltages, nint: int) -> np.ndarray:
    """Incoherent beam P_inc[c][j] = sum over the bin and over antennas of |x|^2, fp64."""
    v = np.ascontiguousarray(voltages)
    nchan, nant = v.shape[0], v.shape[2]
    v, dt, nsamp = _volt(v, nchan, nant)
    if nint <= 0 or nsamp % nint != 0:
        raise ValueError("nsamp must be a positive multiple of nint")
    out = np.empty((nchan, nsamp // nint), dtype=np.float64)
    rc = _load().oracle_incoherent(nant, nchan, nsamp, nint, dt, v.ctypes.data_as(ctypes.c_void_p), _dp(out))
    if rc != 0:
        raise ValueError(f"oracle_incoherent failed rc={rc}")
    return out
