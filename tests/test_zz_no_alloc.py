"""bf_get_weights_noalloc against bf_get_weights (GPU).

bf_get_weights cudaMalloc's a buffer for the decoded weights and cudaFree's it again.  Some users of the library
cannot do that: a backend in the middle of an observation (cudaFree synchronises the whole device and would stall the
streams that are beamforming), a process whose device memory is owned by a pool, a thread running beside a stream
capture in global mode (cudaMalloc is forbidden then).  bf_get_weights_noalloc gives them the same numbers out of a
fixed 8 MiB array inside libbf.so.  That array is shared by every context of the process and keeps the last call's
contents, so the checks below always make two calls in a row and alternate between contexts of different size: a stale
or misplaced element would show up as a difference from bf_get_weights, which must be bit-equal (same arithmetic).

This file is named to be collected last: `pytest -x` stops at the first failure, and a failure here must not hide
the parity tests.  It passes alone in a fresh process and after the rest of the suite.
"""
import numpy as np
import pytest

import synthetic

pytestmark = pytest.mark.gpu

DT = {"ci8": 0, "cf16": 1, "ci4": 2}

# (nant, nchan, nbeam, nsamp, nint, dtype): which operand bf_get_weights decodes, and how it fits the 8 MiB
CASES = [
    (32, 64, 16, 1024, 16, "ci8"),    # int8 two-limb operand (the kernel `tiny` runs); 256 KiB, one call
    (32, 8, 130, 256, 4, "ci8"),      # fp16 operand with the residual plane (nint < 16), three M-tiles; 260 KiB
    (256, 20, 256, 512, 32, "cf16"),  # fp16 K-blocked operand; 512 KiB per channel: 10 MiB = two calls of 16 + 4 channels
]


@pytest.fixture(scope="module")
def bf():
    from paper_1412_4907_b200 import build
    build.build()
    import paper_1412_4907_b200 as bf
    bf.lib()
    return bf


def make(bf, shape):
    nant, nchan, nbeam, nsamp, nint, dtype = shape
    w = synthetic.make_case(nant, nchan, nbeam, nsamp, nint, dtype, seed=5)
    B = bf.Beamformer(nant, nchan, nbeam, nsamp, nint, dtype=DT[dtype], device="cuda:0")
    B.set_geometry(w.ant_xyz, w.freqs, w.beam_dir)
    return w, B


def test_noalloc_equals_get_weights_two_calls_in_a_row(bf):
    made = [make(bf, s) for s in CASES]
    ref = [B.weights() for _, B in made]          # the allocating path
    assert all(np.isfinite(r).all() and np.abs(r).max() > 0.5 for r in ref)
    # twice each, then interleaved: a smaller request follows a larger one and the other way round, so every call finds
    # the array full of another context's weights
    for i in (0, 0, 1, 1, 2, 2, 0, 2, 1, 0):
        got = made[i][1].weights_noalloc()
        assert got.shape == ref[i].shape
        assert np.array_equal(got, ref[i]), f"case {CASES[i]}: differs from bf_get_weights"
    for _, B in made:
        B.close()


def test_noalloc_channel_pieces_and_limit(bf):
    shape = CASES[2]
    nant, nchan, nbeam = shape[:3]
    w, B = make(bf, shape)
    ref = np.empty((nchan, nbeam, nant, 2), dtype=np.float32)
    assert bf.bf_get_weights(B.ctx, ref) == bf.BF_OK
    # the whole set is 10 MiB: refused, and the message says how many channels fit
    out = np.full_like(ref, np.nan)
    assert bf.bf_get_weights_noalloc(B.ctx, 0, nchan, out) == bf.BF_ENOMEM
    msg = bf.bf_last_error(B.ctx)
    assert "at most 16 channels" in msg and str(bf.BF_NOALLOC_MAX_BYTES) in msg, msg
    assert np.isnan(out).all()                    # a refused call writes nothing
    # exactly the limit is accepted; pieces of uneven size, out of order, land where they belong
    assert 16 * nbeam * nant * 8 == bf.BF_NOALLOC_MAX_BYTES
    for c0, n in ((16, 4), (0, 16), (7, 1), (19, 1)):
        piece = np.full((n, nbeam, nant, 2), np.nan, dtype=np.float32)
        assert bf.bf_get_weights_noalloc(B.ctx, c0, n, piece) == bf.BF_OK, bf.bf_last_error(B.ctx)
        assert np.array_equal(piece, ref[c0:c0 + n]), (c0, n)
    # argument errors
    for c0, n in ((-1, 1), (0, 0), (nchan, 1), (nchan - 1, 2), (2 ** 31 - 1, 2)):
        assert bf.bf_get_weights_noalloc(B.ctx, c0, n, out) == bf.BF_EINVAL, (c0, n)
    assert bf.bf_get_weights_noalloc(B.ctx, 0, 1, None) == bf.BF_EINVAL
    ctx = bf.bf_create(32, 4, 16, 256, 16)        # no geometry yet
    assert bf.bf_get_weights_noalloc(ctx, 0, 1, out) == bf.BF_ENOGEOM
    bf.bf_destroy(ctx)
    B.close()


def test_noalloc_sees_a_tracking_update(bf):
    """Two weight buffers: after bf_update_geometry the read-back reports the weights the next run will use, like
    bf_get_weights does -- the case a running observation wants to log without a cudaFree in its way."""
    nant, nchan, nbeam, nsamp, nint = 32, 6, 48, 4096, 16
    w = synthetic.make_case(nant, nchan, nbeam, nsamp, nint, "ci8", seed=9)
    B = bf.Beamformer(nant, nchan, nbeam, nsamp, nint, device="cuda:0", weight_buffers=2)
    B.set_geometry(w.ant_xyz, w.freqs, w.beam_dir)
    first = B.weights_noalloc()
    moved = w.beam_dir[::-1].copy()               # new pointings
    B.update_geometry(w.ant_xyz, w.freqs, moved)
    a = B.weights_noalloc()                       # adopts the pending buffer
    b = B.weights_noalloc()
    ref = B.weights()
    assert np.array_equal(a, ref) and np.array_equal(b, ref)
    assert np.array_equal(ref, first[:, ::-1])    # same directions in reverse order: the same weights, reordered
    assert not np.array_equal(ref, first)
    B.close()
