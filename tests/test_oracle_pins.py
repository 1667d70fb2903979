"""Pins for the oracle (oracle/bf_oracle.c): closed forms, invariants, hand cases.

None of these re-types the oracle's loop.  Source voltages for the closed forms are built
here, independently of synthetic/ and of the oracle, straight from the plane-wave model
x_n = A e^{+i 2 pi f/c0 (r_n . s_src)} (reading A1), and the expected values are the
textbook array-factor results that Eq. 1 of the paper reduces to.
"""
import math
import os

import numpy as np
import pytest

import oracle
import synthetic

C0 = 299792458.0


def plane_wave(r, f, s_src, amp, nsamp, phase_t=None):
    """[C][T][N] complex128 noise-free voltages of one source."""
    geo = r @ s_src
    x = amp * np.exp(2j * np.pi * np.outer(f, geo) / C0)[:, None, :]
    if phase_t is None:
        phase_t = np.zeros((len(f), nsamp))
    return np.ascontiguousarray(x * np.exp(1j * phase_t)[:, :, None])


def dirichlet_sq(n, psi):
    """|sum_{k<n} e^{i k psi}|^2 with the psi -> 0 limit n^2."""
    psi = np.asarray(psi, dtype=np.float64)
    num = np.sin(n * psi / 2.0) ** 2
    den = np.sin(psi / 2.0) ** 2
    with np.errstate(divide="ignore", invalid="ignore"):
        out = np.where(den < 1e-24, float(n * n), num / den)
    return out


# ---------------------------------------------------------------- weights (Eq. 1 steering factor)
def test_weight_quarter_turn_is_minus_i():
    # f d / c0 = 1/4 turn along the look direction  ->  W = e^{-i pi/2} = -i  (sign convention A1)
    f = 100e6
    d = C0 / f / 4.0
    W = oracle.weights([[0, 0, 0], [d, 0, 0], [2 * d, 0, 0]], [f], [[1.0, 0, 0], [0, 0, 1.0]])
    np.testing.assert_allclose(W[0, 0], [1.0, -1j, -1.0], atol=1e-12)
    np.testing.assert_allclose(W[0, 1], [1.0, 1.0, 1.0], atol=1e-15)  # zenith beam of a planar array


def test_weight_z_term_hand_values():
    """The z component of r . s (every other closed-form pin is planar).  One antenna a quarter
    wavelength ABOVE the reference: the zenith beam sees a quarter turn (W = -i), a horizon beam none; a beam
    30 deg from zenith sees cos(30 deg)/4 turn from height alone."""
    f = 150e6
    lam = C0 / f
    r = [[0, 0, 0], [0, 0, lam / 4], [0, 0, -lam / 2]]
    th = np.deg2rad(30.0)
    s = [[0, 0, 1.0], [1.0, 0, 0], [math.sin(th), 0, math.cos(th)]]
    W = oracle.weights(r, [f], s)
    np.testing.assert_allclose(W[0, 0], [1.0, -1j, -1.0], atol=1e-12)          # zenith: -i at +lam/4, e^{+i pi} at -lam/2
    np.testing.assert_allclose(W[0, 1], [1.0, 1.0, 1.0], atol=1e-12)           # horizon beam: height is invisible
    np.testing.assert_allclose(W[0, 2], [1.0, np.exp(-2j * np.pi * math.cos(th) / 4), np.exp(+2j * np.pi * math.cos(th) / 2)],
                               atol=1e-12)


def test_tilted_plane_grid_array_factor():
    """Closed form with z != 0: a uniform line of N antennas climbing a slope (spacing d along x, rise h per step).
    r_n . (s_b - s_src) = n (d (l_b - l_s) + h (n_b - n_s)), so the pattern is the Dirichlet kernel in
    psi = 2 pi f/c0 (d dl + h dn) -- drop the z term (or swap it with y) and psi, hence every power, changes."""
    N, f, d, h, A, I = 12, 200e6, 0.9, 0.35, 1.5, 4
    r = np.stack([np.arange(N) * d, np.zeros(N), np.arange(N) * h], axis=1)
    def unit(l):
        return np.array([l, 0.0, math.sqrt(1.0 - l * l)])
    src = unit(0.2)
    beams = np.stack([unit(l) for l in np.linspace(-0.6, 0.6, 25)])
    x = plane_wave(r, np.array([f]), src, A, I)
    P = oracle.beamform(r, [f], beams, x, I)
    dl = beams[:, 0] - src[0]
    dn = beams[:, 2] - src[2]
    psi = 2.0 * np.pi * f / C0 * (d * dl + h * dn)
    np.testing.assert_allclose(P[0, :, 0], I * A * A * dirichlet_sq(N, psi), rtol=1e-9, atol=1e-9)
    # and the slope matters: the planar formula (h = 0) is off by far more than the tolerance
    psi0 = 2.0 * np.pi * f / C0 * (d * dl)
    assert np.abs(I * A * A * dirichlet_sq(N, psi0) - P[0, :, 0]).max() > 1.0


def test_weights_unit_modulus_and_conjugate_symmetry():
    rng = np.random.default_rng(5)
    r = rng.normal(size=(7, 3)) * 20
    s = rng.normal(size=(5, 3)); s /= np.linalg.norm(s, axis=1, keepdims=True)
    f = np.array([50e6, 408e6])
    W = oracle.weights(r, f, s)
    np.testing.assert_allclose(np.abs(W), 1.0, atol=1e-13)
    np.testing.assert_allclose(oracle.weights(r, f, -s), W.conj(), atol=1e-13)
    # independent evaluation with numpy
    ref = np.exp(-2j * np.pi * f[:, None, None] * (s @ r.T)[None] / C0)
    np.testing.assert_allclose(W, ref, atol=1e-9)  # un-reduced numpy phase of ~1e3 rad: 1e-9 is its own error


# ---------------------------------------------------------------- P1: ULA closed form
def test_p1_ula_array_factor():
    N, d, A = 32, 10.0, 3.0
    f = np.array([408e6, 412.5e6])
    r = synthetic.ula(N, d)
    th0 = math.radians(7.3)
    s_src = np.array([math.sin(th0), 0.0, math.cos(th0)])
    th = np.radians(np.linspace(-30, 30, 41))
    beams = np.stack([np.sin(th), np.zeros_like(th), np.cos(th)], axis=1)
    x = plane_wave(r, f, s_src, A, 4)
    P = oracle.beamform(r, f, beams, x, nint=1)  # |y|^2 per sample
    for c in range(2):
        psi = 2 * np.pi * f[c] * d * (math.sin(th0) - np.sin(th)) / C0
        want = A * A * dirichlet_sq(N, psi)
        np.testing.assert_allclose(P[c, :, 0], want, rtol=0, atol=1e-7 * N * N * A * A)
        np.testing.assert_allclose(P[c, :, 3], want, rtol=0, atol=1e-7 * N * N * A * A)
    # the pattern is not flat: the pin would fail on a dropped phase term
    assert P.max() / np.median(P) > 10


# ---------------------------------------------------------------- P2: grid closed form
def test_p2_grid_array_factor_and_index_order():
    nx, ny, dx, dy, A = 4, 8, 5.7, 10.0, 2.0
    r = synthetic.grid(nx, ny, dx, dy)
    f = np.array([401e6, 415e6])
    l0, m0 = 0.013, -0.021
    s_src = np.array([l0, m0, math.sqrt(1 - l0 * l0 - m0 * m0)])
    beams = synthetic.lm_grid(9, 7, 0.06, 0.03)
    x = plane_wave(r, f, s_src, A, 2)
    P = oracle.beamform(r, f, beams, x, nint=2)
    for c in range(2):
        px = 2 * np.pi * f[c] * dx * (l0 - beams[:, 0]) / C0
        py = 2 * np.pi * f[c] * dy * (m0 - beams[:, 1]) / C0
        want = 2 * A * A * dirichlet_sq(nx, px) * dirichlet_sq(ny, py)
        np.testing.assert_allclose(P[c, :, 0], want, rtol=0, atol=1e-7 * 2 * (nx * ny * A) ** 2)


# ---------------------------------------------------------------- P3: coherent gain
@pytest.mark.parametrize("N,A,I", [(32, 3.0, 16), (8, 1.5, 4)])
def test_p3_coherent_gain_I_N2_A2(N, A, I):
    r = synthetic.grid(4, N // 4, 5.7, 10.0)
    f = np.array([408e6, 409e6, 416e6])
    beams = synthetic.lm_grid(3, 3, 0.05, 0.02)
    rng = np.random.default_rng(0)
    T = 4 * I
    for b in (0, 4, 8):
        x = plane_wave(r, f, beams[b], A, T, rng.uniform(0, 2 * np.pi, (3, T)))
        P = oracle.beamform(r, f, beams, x, nint=I)
        np.testing.assert_allclose(P[:, b, :], I * N * N * A * A, rtol=1e-11)  # e.g. 16*32^2*3^2 = 147456
        other = np.delete(P, b, axis=1)
        assert other.max() < I * N * N * A * A * 0.999  # off-source beams are strictly lower


def test_p3_golden_value():
    # tests/golden/coherent_gain.txt: closed-form I*N^2*A^2 values (not oracle output)
    path = os.path.join(os.path.dirname(__file__), "golden", "coherent_gain.txt")
    rows = [ln.split() for ln in open(path) if ln.strip() and not ln.startswith("#")]
    for N, A, I, want in rows:
        N, A, I, want = int(N), float(A), int(I), float(want)
        r = synthetic.ula(N, 10.0)
        f = np.array([408e6])
        th = math.radians(11.0)
        s = np.array([[math.sin(th), 0, math.cos(th)]])
        x = plane_wave(r, f, s[0], A, I)
        P = oracle.beamform(r, f, s, x, nint=I)
        assert P.shape == (1, 1, 1)
        np.testing.assert_allclose(P[0, 0, 0], want, rtol=1e-11)


# ---------------------------------------------------------------- P4: incoherent level
def test_p4_incoherent_noise_level():
    # unit-modulus weights on i.i.d. noise: E|y|^2 = N * E|x|^2 (prop. to N, not N^2)  (reading A19)
    w = synthetic.make_workload("tiny").sub(nchan=8)
    v = w.make_voltages()
    P = oracle.beamform(w.ant_xyz, w.freqs, w.beam_dir, v, w.nint)
    ex2 = (v.astype(np.float64) ** 2).sum(axis=-1).mean()  # measured E|x|^2 (= 2(sigma^2+1/12) up to clamping)
    assert abs(ex2 / (2 * (16.0 ** 2 + 1 / 12)) - 1) < 0.01
    want = w.nint * w.nant * ex2
    nsamp_total = P.size * w.nint
    assert abs(P.mean() / want - 1) < 4.0 / math.sqrt(nsamp_total)
    assert P.mean() < 0.1 * w.nint * w.nant ** 2 * ex2  # far below the coherent N^2 level


# ---------------------------------------------------------------- P5: Parseval on the DFT grid
def test_p5_parseval_dft_beams_exact_integer():
    N, d, f0 = 32, 10.0, 408e6
    r = synthetic.ula(N, d)
    f = np.array([f0])
    sin_b = np.arange(-N // 2, N // 2) * C0 / (N * f0 * d)
    beams = np.stack([sin_b, np.zeros(N), np.sqrt(1 - sin_b ** 2)], axis=1)
    rng = np.random.default_rng(11)
    v = np.clip(np.rint(rng.normal(size=(1, 64, N, 2)) * 16), -127, 127).astype(np.int8)
    I = 16
    P = oracle.beamform(r, f, beams, v, nint=I)
    lhs = P.sum(axis=1)[0]  # sum over beams, per bin
    e = (v.astype(np.int64) ** 2).sum(axis=(2, 3))[0].reshape(-1, I).sum(axis=1)  # exact integers
    np.testing.assert_allclose(lhs, N * e, rtol=1e-12)


# ---------------------------------------------------------------- P6: independent library contraction
@pytest.mark.parametrize("dtype", ["ci8", "cf16"])
def test_p6_numpy_einsum(dtype):
    rng = np.random.default_rng(3)
    N, C, B, T, I = 12, 3, 7, 40, 8
    r = rng.normal(size=(N, 3)) * 15
    f = np.array([120e6, 300e6, 410e6])
    s = rng.normal(size=(B, 3)); s[:, 2] = np.abs(s[:, 2]) + 1; s /= np.linalg.norm(s, axis=1, keepdims=True)
    if dtype == "ci8":
        v = rng.integers(-127, 128, size=(C, T, N, 2)).astype(np.int8)
    else:
        v = rng.normal(size=(C, T, N, 2)).astype(np.float16)
    x = v[..., 0].astype(np.float64) + 1j * v[..., 1].astype(np.float64)
    turns = f[:, None, None] * (s @ r.T)[None] / C0
    turns -= np.rint(turns)
    W = np.exp(-2j * np.pi * turns)
    y = np.einsum("cbn,ctn->cbt", W, x)
    want = (np.abs(y) ** 2).reshape(C, B, T // I, I).sum(-1)
    P = oracle.beamform(r, f, s, v, nint=I)
    np.testing.assert_allclose(P, want, rtol=1e-11)
    np.testing.assert_allclose(oracle.beams(r, f, s, v), y, rtol=0, atol=1e-9 * np.abs(y).max())
    # same numbers handed over as complex128
    np.testing.assert_allclose(oracle.beamform(r, f, s, np.ascontiguousarray(x), nint=I), P, rtol=1e-14)


# ---------------------------------------------------------------- P7: hand-checkable brute force
def test_p7_single_antenna_any_geometry():
    rng = np.random.default_rng(2)
    v = rng.integers(-127, 128, size=(2, 12, 1, 2)).astype(np.int8)
    s = synthetic.zenith_fan(5)
    P = oracle.beamform([[3.0, -4.0, 1.0]], [100e6, 200e6], s, v, nint=4)
    e = (v.astype(np.float64) ** 2).sum(axis=(2, 3)).reshape(2, 3, 4).sum(-1)
    for b in range(5):
        np.testing.assert_allclose(P[:, b, :], e, rtol=1e-13)


def test_p7_two_antennas_half_and_quarter_turn():
    f = 150e6
    x = np.array([[[2 + 1j, -1 + 3j], [0.5 - 2j, 4 + 0j]]])  # [1][T=2][N=2]
    s = np.array([[1.0, 0, 0]])
    # half turn: W = (1, -1)  ->  y = x0 - x1
    d = C0 / f / 2
    P = oracle.beamform([[0, 0, 0], [d, 0, 0]], [f], s, x, nint=1)
    np.testing.assert_allclose(P[0, 0], np.abs(x[0, :, 0] - x[0, :, 1]) ** 2, rtol=1e-12)
    # quarter turn: W = (1, -i)  ->  y = x0 - i x1
    d = C0 / f / 4
    P = oracle.beamform([[0, 0, 0], [d, 0, 0]], [f], s, x, nint=2)
    np.testing.assert_allclose(P[0, 0, 0], (np.abs(x[0, :, 0] - 1j * x[0, :, 1]) ** 2).sum(), rtol=1e-12)


# ---------------------------------------------------------------- P8: algebraic invariants
def test_p8_invariants():
    w = synthetic.make_workload("tiny").sub(nchan=4, nsamp=128)
    v = w.make_voltages()
    r, f, s, I = w.ant_xyz, w.freqs, w.beam_dir, w.nint
    P = oracle.beamform(r, f, s, v, I)
    assert P.shape == (4, 16, 8) and np.isfinite(P).all()
    # x -> 2x  =>  P -> 4P   (v small enough not to clip: use the complex128 entry)
    x = v[..., 0].astype(np.float64) + 1j * v[..., 1]
    np.testing.assert_allclose(oracle.beamform(r, f, s, 2 * x, I), 4 * P, rtol=1e-13)
    # permuting antennas together with their positions changes nothing
    perm = np.random.default_rng(0).permutation(w.nant)
    np.testing.assert_allclose(oracle.beamform(r[perm], f, s, np.ascontiguousarray(v[:, :, perm]), I), P, rtol=1e-12)
    # translating the array is a global phase
    np.testing.assert_allclose(oracle.beamform(r + np.array([13.0, -7.0, 2.5]), f, s, v, I), P, rtol=1e-9)
    # P_{2I}[j] = P_I[2j] + P_I[2j+1]
    np.testing.assert_allclose(oracle.beamform(r, f, s, v, 2 * I), P[:, :, 0::2] + P[:, :, 1::2], rtol=1e-13)
    # beams and channels are independent
    np.testing.assert_array_equal(oracle.beamform(r, f, s[3:7], v, I), P[:, 3:7])
    np.testing.assert_array_equal(oracle.beamform(r, f[2:3], s, v[2:3], I), P[2:3])
    # chan_stride sampling leaves skipped channels untouched (NaN) and the rest identical
    Ps = oracle.beamform(r, f, s, v, I, chan_stride=2)
    np.testing.assert_array_equal(Ps[0::2], P[0::2])
    assert np.isnan(Ps[1::2]).all()
    # a swapped re/im or conjugated input does change the answer (guards the pin's power)
    assert not np.allclose(oracle.beamform(r, f, s, np.ascontiguousarray(x.conj()), I), P, rtol=1e-3)


def test_fp16_and_int8_inputs_agree_on_common_values():
    rng = np.random.default_rng(9)
    v8 = rng.integers(-100, 101, size=(2, 16, 8, 2)).astype(np.int8)
    v16 = v8.astype(np.float16)  # exact
    r = synthetic.grid(4, 2, 2.0, 2.0)
    s = synthetic.lm_grid(3, 2, 0.4, 0.3)
    f = [70e6, 333e6]
    np.testing.assert_array_equal(oracle.beamform(r, f, s, v8, 4), oracle.beamform(r, f, s, v16, 4))


def test_ci4_decode_by_hand_and_against_int8():
    """4+4-bit two's complement, one byte per antenna, high nibble real (reading A20)."""
    # 0x7F = (+7, -1), 0x80 = (-8, 0), 0x19 = (+1, -7), 0xF0 = (-1, 0)
    v = np.array([[[0x7F], [0x80], [0x19], [0xF0]]], dtype=np.uint8)  # [C=1][T=4][N=1]
    P = oracle.beamform([[0, 0, 0]], [100e6], [[0, 0, 1.0]], v, nint=1)
    np.testing.assert_allclose(P[0, 0], [49 + 1, 64 + 0, 1 + 49, 1 + 0], rtol=1e-14)
    rng = np.random.default_rng(4)
    re = rng.integers(-8, 8, size=(2, 32, 8)); im = rng.integers(-8, 8, size=(2, 32, 8))
    v4 = synthetic.pack_ci4(re, im)
    v8 = np.stack([re, im], axis=-1).astype(np.int8)
    r = synthetic.grid(4, 2, 2.0, 2.0); s = synthetic.lm_grid(3, 2, 0.4, 0.3); f = [70e6, 333e6]
    np.testing.assert_array_equal(oracle.beamform(r, f, s, v4, 8), oracle.beamform(r, f, s, v8, 8))


def test_rejects_bad_nint():
    w = synthetic.make_workload("tiny").sub(nchan=1, nsamp=32)
    with pytest.raises(ValueError):
        oracle.beamform(w.ant_xyz, w.freqs, w.beam_dir, w.make_voltages(), 5)


def test_golden_tiny_regression():
    """tests/golden/tiny_oracle_sample.txt is written by tests/golden/make_golden.py (oracle only)."""
    path = os.path.join(os.path.dirname(__file__), "golden", "tiny_oracle_sample.txt")
    w = synthetic.make_workload("tiny")
    v = w.make_voltages()
    P = oracle.beamform(w.ant_xyz, w.freqs, w.beam_dir, v, w.nint)
    for ln in open(path):
        if ln.startswith("#") or not ln.strip():
            continue
        c, b, j, val = ln.split()
        np.testing.assert_allclose(P[int(c), int(b), int(j)], float(val), rtol=1e-12)
