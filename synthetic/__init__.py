"""Seeded synthetic inputs for the beamformer: geometry arrays and voltage buffers.

This module serves BOTH the oracle and the CUDA path and therefore holds none of the
method's arithmetic (no steering weights, no beam sums, no powers).  It only builds inputs:
antenna positions, channel frequencies, beam directions and antenna voltages with the shapes
and statistics of the paper's BEST-2 workloads as restated by
BASELINE.json ``configs``.  An injected plane-wave source is part of the *signal model* of the
input (reading A1/A10 in DESIGN.md): x_n = A e^{i phi_t} e^{+i 2 pi f/c0 (r_n . s_src)}.

No dataset, recording or third-party item is reproduced here; everything is drawn from a
seeded generator.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional

import numpy as np

C0 = 299792458.0  # m/s


# ----------------------------------------------------------------------------- geometry
def ula(nant: int, spacing_m: float) -> np.ndarray:
    """Uniform linear array along x: r_n = (n d, 0, 0).  [nant][3] fp64."""
    r = np.zeros((nant, 3), dtype=np.float64)
    r[:, 0] = np.arange(nant) * spacing_m
    return r


def grid(nx: int, ny: int, dx_m: float, dy_m: float) -> np.ndarray:
    """Planar grid, index n = nx*j_y + i_x, r = (i_x dx, j_y dy, 0) (reading A5)."""
    r = np.zeros((nx * ny, 3), dtype=np.float64)
    iy, ix = np.divmod(np.arange(nx * ny), nx)
    r[:, 0] = ix * dx_m
    r[:, 1] = iy * dy_m
    return r


def chan_centres(f_lo_hz: float, bw_hz: float, nchan: int) -> np.ndarray:
    """Channel centre frequencies f_c = f_lo + (c + 1/2) BW/C (reading A4)."""
    return f_lo_hz + (np.arange(nchan) + 0.5) * (bw_hz / nchan)


def zenith_fan(nbeam: int, half_width_deg: float = 30.0) -> np.ndarray:
    """Beams evenly spaced over +-half_width from zenith in the x-z plane, endpoints
    included; a single beam points at zenith (reading A3).  [nbeam][3] unit vectors."""
    if nbeam == 1:
        th = np.zeros(1)
    else:
        th = np.deg2rad(-half_width_deg + 2.0 * half_width_deg * np.arange(nbeam) / (nbeam - 1))
    s = np.zeros((nbeam, 3), dtype=np.float64)
    s[:, 0] = np.sin(th)
    s[:, 2] = np.cos(th)
    return s


def lm_grid(nl: int, nm: int, l_half: float, m_half: float, endpoint: bool = True) -> np.ndarray:
    """Regular sky grid in direction cosines (l, m, sqrt(1-l^2-m^2)); beam b = nl*j_m + i_l."""
    def axis(n, h):
        if n == 1:
            return np.zeros(1)
        return np.linspace(-h, h, n, endpoint=True) if endpoint else (-h + 2.0 * h * np.arange(n) / n)
    l = axis(nl, l_half)
    m = axis(nm, m_half)
    L, M = np.meshgrid(l, m, indexing="xy")  # shape [nm][nl]
    L = L.reshape(-1)
    M = M.reshape(-1)
    s = np.stack([L, M, np.sqrt(1.0 - L * L - M * M)], axis=1)
    return np.ascontiguousarray(s, dtype=np.float64)


# ----------------------------------------------------------------------------- voltages
def _source_term(ant_xyz, freqs, src_dir, amp, phases):
    """Plane wave of constant modulus `amp` and per-(c,t) phase from direction src_dir:
    [C][T][N] complex128 (signal model of the INPUT, reading A1/A10)."""
    geo = (ant_xyz @ np.asarray(src_dir, dtype=np.float64))  # [N] metres of path
    ph_n = np.exp(2j * np.pi * np.outer(freqs, geo) / C0)  # [C][N]
    return amp * np.exp(1j * phases)[:, :, None] * ph_n[:, None, :]


def voltages_ci8(rng: np.random.Generator, nchan: int, nsamp: int, nant: int, sigma: float = 16.0,
                 sources=None, ant_xyz=None, freqs=None) -> np.ndarray:
    """Complex int8 voltages [C][T][N][2]: circular Gaussian, sigma per real component, plus
    optional plane-wave sources [(dir, amp), ...] added BEFORE quantisation; quantisation is
    clip(rint(.), -127, 127), round-half-even, -128 never occurs (reading A9)."""
    out = np.empty((nchan, nsamp, nant, 2), dtype=np.int8)
    for c in range(nchan):  # channel at a time keeps the temporaries small
        z = rng.standard_normal((nsamp, nant, 2), dtype=np.float32).astype(np.float64) * sigma
        if sources:
            for (sdir, amp) in sources:
                ph = rng.uniform(0.0, 2.0 * np.pi, size=(1, nsamp))
                s = _source_term(ant_xyz, freqs[c:c + 1], sdir, amp, ph)[0]
                z[..., 0] += s.real
                z[..., 1] += s.imag
        out[c] = np.clip(np.rint(z), -127, 127).astype(np.int8)
    return out


def pack_ci4(re, im) -> np.ndarray:
    """Two's-complement nibbles, high nibble real, low nibble imaginary (reading A20). re, im in [-8, 7]."""
    return (((np.asarray(re).astype(np.int16) & 15) << 4) | (np.asarray(im).astype(np.int16) & 15)).astype(np.uint8)


def voltages_ci4(rng: np.random.Generator, nchan: int, nsamp: int, nant: int, sigma: float = 2.0,
                 sources=None, ant_xyz=None, freqs=None) -> np.ndarray:
    """4+4-bit packed complex voltages [C][T][N] uint8 (the paper's F-engine format):
    Gaussian sigma per component + optional sources, clip(rint(.), -7, 7) (-8 never occurs)."""
    out = np.empty((nchan, nsamp, nant), dtype=np.uint8)
    for c in range(nchan):
        z = rng.standard_normal((nsamp, nant, 2), dtype=np.float32).astype(np.float64) * sigma
        if sources:
            for (sdir, amp) in sources:
                ph = rng.uniform(0.0, 2.0 * np.pi, size=(1, nsamp))
                s = _source_term(ant_xyz, freqs[c:c + 1], sdir, amp, ph)[0]
                z[..., 0] += s.real
                z[..., 1] += s.imag
        q = np.clip(np.rint(z), -7, 7).astype(np.int16)
        out[c] = pack_ci4(q[..., 0], q[..., 1])
    return out


def voltages_cf16(rng: np.random.Generator, nchan: int, nsamp: int, nant: int, sigma: float = 1.0,
                  sources=None, ant_xyz=None, freqs=None) -> np.ndarray:
    """Complex fp16 voltages [C][T][N][2] (Gaussian sigma per component + sources, rounded RN)."""
    out = np.empty((nchan, nsamp, nant, 2), dtype=np.float16)
    for c in range(nchan):
        z = rng.standard_normal((nsamp, nant, 2), dtype=np.float32).astype(np.float64) * sigma
        if sources:
            for (sdir, amp) in sources:
                ph = rng.uniform(0.0, 2.0 * np.pi, size=(1, nsamp))
                s = _source_term(ant_xyz, freqs[c:c + 1], sdir, amp, ph)[0]
                z[..., 0] += s.real
                z[..., 1] += s.imag
        out[c] = z.astype(np.float16)
    return out


# ----------------------------------------------------------------------------- configs
@dataclasses.dataclass
class Workload:
    name: str
    nant: int
    nchan: int
    nbeam: int
    nsamp: int
    nint: int
    dtype: str  # "ci8" | "cf16"
    seed: int
    ant_xyz: np.ndarray
    freqs: np.ndarray
    beam_dir: np.ndarray
    sigma: float
    sources: list  # [(unit vector, amplitude)]

    @property
    def nbin(self) -> int:
        return self.nsamp // self.nint

    @property
    def in_bytes(self) -> int:
        return self.nchan * self.nsamp * self.nant * {"ci8": 2, "cf16": 4, "ci4": 1}[self.dtype]

    @property
    def out_bytes(self) -> int:
        return self.nchan * self.nbeam * self.nbin * 4

    @property
    def cmac(self) -> int:
        return self.nchan * self.nbeam * self.nant * self.nsamp

    def make_voltages(self, nchan: Optional[int] = None, nsamp: Optional[int] = None, chan0: int = 0,
                      block: int = 0) -> np.ndarray:
        """Host (numpy) voltages; optionally only the first `nchan` channels starting at chan0 and
        `nsamp` samples -- each (seed, chan0, block) draws its own stream so sub-buffers are cheap."""
        nchan = self.nchan if nchan is None else nchan
        nsamp = self.nsamp if nsamp is None else nsamp
        rng = np.random.default_rng([self.seed, chan0, block])
        f = self.freqs[chan0:chan0 + nchan]
        fn = {"ci8": voltages_ci8, "cf16": voltages_cf16, "ci4": voltages_ci4}[self.dtype]
        return fn(rng, nchan, nsamp, self.nant, self.sigma, self.sources, self.ant_xyz, f)

    def sub(self, nchan: Optional[int] = None, nsamp: Optional[int] = None, nbeam: Optional[int] = None,
            chan_idx=None) -> "Workload":
        """A reduced copy (fewer channels / samples / beams) for oracle-sized checks."""
        w = dataclasses.replace(self)
        if chan_idx is not None:
            w.freqs = self.freqs[np.asarray(chan_idx)].copy()
            w.nchan = len(w.freqs)
        elif nchan is not None:
            w.freqs = self.freqs[:nchan].copy()
            w.nchan = nchan
        if nsamp is not None:
            assert nsamp % self.nint == 0
            w.nsamp = nsamp
        if nbeam is not None:
            w.beam_dir = self.beam_dir[:nbeam].copy()
            w.nbeam = nbeam
        return w


def _src_at_beam(beam_dir, seed, k=1):
    rng = np.random.default_rng([seed, 777])
    idx = rng.choice(beam_dir.shape[0], size=k, replace=False)
    return [int(i) for i in idx]


def make_workload(name: str, nbeam: Optional[int] = None) -> Workload:
    """The five BASELINE.json configs (recipes: DESIGN.md 'Synthetic inputs')."""
    if name == "tiny":
        N, C, B, T, I = 32, 64, 16, 1024, 16
        return Workload(name, N, C, B, T, I, "ci8", 0, ula(N, 10.0), chan_centres(408e6, 8e6, C),
                        zenith_fan(B, 30.0), 16.0, [])
    if name == "medium":
        N, C, B, T, I = 32, 1024, 128, 32768, 64
        r = grid(4, 8, 5.7, 10.0)
        s = lm_grid(16, 8, 0.06, 0.03)
        (ib,) = _src_at_beam(s, 1)
        return Workload(name, N, C, B, T, I, "ci8", 1, r, chan_centres(400e6, 16e6, C), s, 16.0, [(s[ib].copy(), 8.0)])
    if name == "medium-ci4":
        # the medium geometry with the paper's own 4+4-bit wire format
        w = make_workload("medium")
        return dataclasses.replace(w, name=name, dtype="ci4", sigma=2.0, sources=[(w.sources[0][0], 1.0)])
    if name == "sweep-ci4":
        # the beam-count sweep on the paper's 4+4-bit wire format (halves the input bytes, which moves the
        # bandwidth -> compute crossover to fewer beams)
        w = make_workload("sweep", nbeam=nbeam)
        return dataclasses.replace(w, name=w.name.replace("sweep", "sweep-ci4"), dtype="ci4", sigma=2.0)
    if name == "streaming-ci4":
        # the 1024-antenna aperture array fed 4+4-bit samples: half the PCIe bytes per antenna-sample
        w = make_workload("streaming")
        return dataclasses.replace(w, name=name, dtype="ci4", sigma=2.0)
    if name == "sweep":
        N, C, T, I = 32, 512, 16384, 16
        B = 64 if nbeam is None else nbeam
        return Workload(f"sweep-B{B}", N, C, B, T, I, "ci8", 2, ula(N, 10.0), chan_centres(404e6, 8e6, C),
                        zenith_fan(B, 30.0), 16.0, [])
    if name == "large-N":
        N, C, B, T, I = 256, 256, 256, 8192, 32
        r = grid(16, 16, 2.0, 2.0)
        s = lm_grid(16, 16, 0.5, 0.5)
        i0, i1 = _src_at_beam(s, 3, 2)
        return Workload(name, N, C, B, T, I, "cf16", 3, r, chan_centres(50e6, 300e6, C), s, 1.0,
                        [(s[i0].copy(), 0.5), (s[i1].copy(), 0.25)])
    if name == "streaming":
        N, C, B, T, I = 1024, 64, 1024, 4096, 64
        r = grid(32, 32, 1.5, 1.5)
        s = lm_grid(32, 32, 0.5, 0.5, endpoint=False)
        return Workload(name, N, C, B, T, I, "ci8", 4, r, chan_centres(100e6, 50e6, C), s, 16.0, [])
    raise KeyError(name)


SWEEP_BEAMS = (1, 4, 16, 64, 256, 1024)


# ----------------------------------------------------------------------------- device-side fill
def make_case(nant: int, nchan: int, nbeam: int, nsamp: int, nint: int, dtype: str, seed: int = 0) -> Workload:
    """A small seeded test case of arbitrary shape: scattered near-planar array, random beam directions within
    ~35 deg of zenith, noise plus one source at the centre of beam nbeam // 2 (the recipe of the parity tests)."""
    rng = np.random.default_rng([seed, nant, nchan, nbeam, nsamp])
    r = rng.uniform(-40, 40, size=(nant, 3)); r[:, 2] *= 0.05
    f = np.linspace(380e6, 420e6, nchan) if nchan > 1 else np.array([408e6])
    s = rng.normal(size=(nbeam, 3)); s[:, 2] = np.abs(s[:, 2]) + 1.5; s /= np.linalg.norm(s, axis=1, keepdims=True)
    sig, amp = {"ci8": (16.0, 4.0), "cf16": (1.0, 0.5), "ci4": (2.0, 1.0)}[dtype]
    return Workload("case", nant, nchan, nbeam, nsamp, nint, dtype, seed, r, f, s, sig, [(s[nbeam // 2].copy(), amp)])


def fill_voltages_torch(w: Workload, device, chunk_chan: int = 16):
    """Full-size voltages generated ON `device` with torch's seeded generator (reading A11):
    same statistics as make_voltages(); bytes are what they are -- parity checks copy the very
    same bytes to the oracle.  Returns a torch tensor [C][T][N][2] int8 or float16."""
    import torch

    g = torch.Generator(device=device)
    g.manual_seed(1000 + w.seed)
    dt = {"ci8": torch.int8, "cf16": torch.float16, "ci4": torch.uint8}[w.dtype]
    shape = (w.nchan, w.nsamp, w.nant) if w.dtype == "ci4" else (w.nchan, w.nsamp, w.nant, 2)
    out = torch.empty(shape, dtype=dt, device=device)
    r = torch.as_tensor(w.ant_xyz, device=device)
    for c0 in range(0, w.nchan, chunk_chan):
        c1 = min(w.nchan, c0 + chunk_chan)
        z = torch.randn((c1 - c0, w.nsamp, w.nant, 2), generator=g, device=device, dtype=torch.float32) * w.sigma
        for (sdir, amp) in w.sources:
            f = torch.as_tensor(w.freqs[c0:c1], device=device)
            geo = r @ torch.as_tensor(sdir, device=device)  # [N]
            ph_n = 2.0 * math.pi * torch.outer(f, geo) / C0  # [c][N] fp64
            ph_t = torch.rand((c1 - c0, w.nsamp), generator=g, device=device, dtype=torch.float64) * (2.0 * math.pi)
            ph = (ph_t[:, :, None] + ph_n[:, None, :])
            z[..., 0] += (amp * torch.cos(ph)).float()
            z[..., 1] += (amp * torch.sin(ph)).float()
        if w.dtype == "ci8":
            out[c0:c1] = torch.clamp(torch.round(z), -127, 127).to(torch.int8)
        elif w.dtype == "ci4":
            q = torch.clamp(torch.round(z), -7, 7).to(torch.int16)
            out[c0:c1] = (((q[..., 0] & 15) << 4) | (q[..., 1] & 15)).to(torch.uint8)
        else:
            out[c0:c1] = z.to(torch.float16)
    return out
