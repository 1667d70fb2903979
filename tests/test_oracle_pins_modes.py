"""Pins for the oracle's two extra outputs:

* ``oracle.beams``      -- raw complex beams y[c][b][t] ("electric-field beams ... 16-bit complex-valued
                           words")
* ``oracle.incoherent`` -- incoherent beam sum_n |x_n|^2

Expected values come from what the mathematics fixes (Eq. 1 closed forms, hand cases, exact integer
sums, a Parseval identity that ties the incoherent beam to the already pinned coherent powers), never
from re-typing the oracle's loops.
"""
import numpy as np
import pytest

import oracle
import synthetic

C0 = 299792458.0


# ---------------------------------------------------------------- voltage beams
def test_beams_ula_geometric_series_complex_value():
    """Noise-free source at theta0, beam at theta: y = A sum_n e^{i n psi} = A (1 - e^{iN psi})/(1 - e^{i psi}),
    psi = 2 pi f d (sin theta0 - sin theta)/c0 -- Eq. 1 with A_n = 1; pins phase AND sign."""
    N, d, f, A = 16, 7.0, 233e6, 2.5
    r = synthetic.ula(N, d)
    th0 = np.deg2rad(11.0)
    ths = np.deg2rad(np.array([-20.0, 3.0, 11.0, 25.0]))
    s = np.stack([np.sin(ths), np.zeros(4), np.cos(ths)], axis=1)
    x = (A * np.exp(2j * np.pi * f * (np.arange(N) * d) * np.sin(th0) / C0))[None, None, :]
    x = np.ascontiguousarray(np.repeat(x, 3, axis=1))  # [1][T=3][N]
    y = oracle.beams(r, [f], s, x)
    psi = 2 * np.pi * f * d * (np.sin(th0) - np.sin(ths)) / C0
    with np.errstate(divide="ignore", invalid="ignore"):
        ref = np.where(np.abs(psi) < 1e-12, N + 0j, (1 - np.exp(1j * N * psi)) / (1 - np.exp(1j * psi))) * A
    for t in range(3):
        np.testing.assert_allclose(y[0, :, t], ref, atol=1e-9)
    assert abs(y[0, 2, 0] - N * A) < 1e-9  # steered beam: all antennas in phase, real and positive


def test_beams_two_antennas_by_hand():
    f = 150e6
    x = np.array([[[2 + 1j, -1 + 3j], [0.5 - 2j, 4 + 0j]]])  # [1][T=2][N=2]
    s = np.array([[1.0, 0, 0]])
    d = C0 / f / 4  # quarter turn: W = (1, -i)
    y = oracle.beams([[0, 0, 0], [d, 0, 0]], [f], s, x)
    np.testing.assert_allclose(y[0, 0], x[0, :, 0] - 1j * x[0, :, 1], atol=1e-12)
    # (2+1j) - 1j(-1+3j) = 5+2j ; (0.5-2j) - 1j*4 = 0.5-6j
    np.testing.assert_allclose(y[0, 0], [5 + 2j, 0.5 - 6j], atol=1e-12)


def test_beams_square_to_the_pinned_powers():
    """|y|^2 summed over nint reproduces oracle.beamform (itself pinned by test_oracle_pins.py)."""
    w = synthetic.make_workload("tiny").sub(nchan=2, nsamp=64)
    v = w.make_voltages()
    y = oracle.beams(w.ant_xyz, w.freqs, w.beam_dir, v)
    P = oracle.beamform(w.ant_xyz, w.freqs, w.beam_dir, v, 16)
    np.testing.assert_allclose((np.abs(y) ** 2).reshape(2, w.nbeam, 4, 16).sum(-1), P, rtol=1e-12)


def test_beams_linear_in_the_voltages():
    rng = np.random.default_rng(8)
    r = synthetic.grid(4, 2, 3.0, 5.0); s = synthetic.lm_grid(3, 2, 0.3, 0.2); f = [120e6]
    a = rng.normal(size=(1, 5, 8)) + 1j * rng.normal(size=(1, 5, 8))
    b = rng.normal(size=(1, 5, 8)) + 1j * rng.normal(size=(1, 5, 8))
    ya, yb = oracle.beams(r, f, s, a), oracle.beams(r, f, s, b)
    np.testing.assert_allclose(oracle.beams(r, f, s, a + (2 - 3j) * b), ya + (2 - 3j) * yb, atol=1e-11)


# ---------------------------------------------------------------- incoherent beam
def test_incoherent_hand_values():
    # x = 3+4i on every antenna: |x|^2 = 25  ->  P = 25 N I
    v = np.zeros((2, 8, 5, 2), dtype=np.int8); v[..., 0] = 3; v[..., 1] = 4
    np.testing.assert_array_equal(oracle.incoherent(v, 4), np.full((2, 2), 25.0 * 5 * 4))
    # one non-zero sample lands in exactly one bin of one channel
    v = np.zeros((2, 8, 5, 2), dtype=np.int8); v[1, 6, 3] = (-7, 2)
    exp = np.zeros((2, 4)); exp[1, 3] = 53.0
    np.testing.assert_array_equal(oracle.incoherent(v, 2), exp)


@pytest.mark.parametrize("kind", ["ci8", "cf16", "ci4"])
def test_incoherent_exact_sum_of_squares(kind):
    rng = np.random.default_rng(21)
    C, T, N, I = 3, 48, 12, 8
    if kind == "ci8":
        v = rng.integers(-127, 128, size=(C, T, N, 2)).astype(np.int8)
        e = (v.astype(np.int64) ** 2).sum(axis=(2, 3))
    elif kind == "cf16":
        v = rng.integers(-40, 41, size=(C, T, N, 2)).astype(np.float16)  # small integers: exact in fp16
        e = (v.astype(np.int64) ** 2).sum(axis=(2, 3))
    else:
        re = rng.integers(-8, 8, size=(C, T, N)); im = rng.integers(-8, 8, size=(C, T, N))
        v = synthetic.pack_ci4(re, im)
        e = (re.astype(np.int64) ** 2 + im.astype(np.int64) ** 2).sum(axis=2)
    np.testing.assert_array_equal(oracle.incoherent(v, I), e.reshape(C, T // I, I).sum(-1).astype(np.float64))


def test_incoherent_equals_single_antenna_coherent_power():
    """N = 1: any unit-modulus weight gives |W x|^2 = |x|^2, so coherent = incoherent (pinned P7 case)."""
    rng = np.random.default_rng(2)
    v = rng.integers(-127, 128, size=(2, 12, 1, 2)).astype(np.int8)
    P = oracle.beamform([[3.0, -4.0, 1.0]], [100e6, 200e6], synthetic.zenith_fan(3), v, nint=4)
    inc = oracle.incoherent(v, 4)
    for b in range(3):
        np.testing.assert_allclose(P[:, b, :], inc, rtol=1e-13)


def test_incoherent_parseval_against_coherent_dft_beams():
    """ULA with the N DFT beams: W is sqrt(N) x unitary, so sum_b P_coh[c][b][j] = N P_inc[c][j]."""
    N, d, f0 = 16, 10.0, 408e6
    r = synthetic.ula(N, d)
    sin_b = np.arange(-N // 2, N // 2) * C0 / (N * f0 * d)
    beams = np.stack([sin_b, np.zeros(N), np.sqrt(1 - sin_b ** 2)], axis=1)
    rng = np.random.default_rng(12)
    v = np.clip(np.rint(rng.normal(size=(1, 64, N, 2)) * 16), -127, 127).astype(np.int8)
    P = oracle.beamform(r, [f0], beams, v, nint=8)
    np.testing.assert_allclose(P.sum(axis=1), N * oracle.incoherent(v, 8), rtol=1e-12)


def test_incoherent_noise_level_and_rejects_bad_nint():
    # i.i.d. N(0, 16^2) rounded: E|x|^2 = 2 (sigma^2 + 1/12) per antenna-sample
    w = synthetic.make_workload("tiny").sub(nchan=4)
    v = w.make_voltages()
    inc = oracle.incoherent(v, w.nint)
    per = inc.mean() / (w.nint * w.nant)
    assert abs(per / (2 * (256 + 1 / 12)) - 1) < 0.01
    with pytest.raises(ValueError):
        oracle.incoherent(v, 5)
