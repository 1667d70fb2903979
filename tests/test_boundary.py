"""CPU-side checks of the C-ABI boundary: the library loads, exports every symbol include/bf.h
declares, and validates its arguments.  No compute calls (no GPU here)."""
import ctypes
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def bf():
    from paper_1412_4907_b200 import build
    build.build()
    import paper_1412_4907_b200 as bf
    bf.lib()
    return bf


def test_header_symbols_all_exported(bf):
    hdr = open(os.path.join(ROOT, "include", "bf.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(bf_[a-z_]+)\s*\(", hdr))
    assert declared, "no declarations found"
    assert declared == set(bf.SYMBOLS), (declared ^ set(bf.SYMBOLS))
    L = ctypes.CDLL(bf.LIB_PATH)
    for name in declared:
        assert hasattr(L, name), name
    assert "sm_100a" in bf.bf_version()


def test_create_validation(bf):
    assert bf.bf_create(32, 64, 16, 1024, 16)
    for bad in [(0, 1, 1, 16, 16), (1, 0, 1, 16, 16), (1, 1, 0, 16, 16), (1, 1, 1, 0, 16), (1, 1, 1, 16, 0),
                (-3, 1, 1, 16, 16), (32, 64, 16, 1000, 16)]:  # last: nsamp % nint != 0 (reading A8)
        assert not bf.bf_create(*bad), bad
    ctx = bf.bf_create(5, 3, 1, 7, 7)  # odd sizes and a single beam are legal
    assert ctx
    bf.bf_destroy(ctx)
    bf.bf_destroy(None)


def test_argument_errors_without_gpu(bf):
    ctx = bf.bf_create(32, 4, 16, 256, 16)
    assert bf.bf_set_dtype(ctx, 7) == bf.BF_EINVAL
    assert "dtype" in bf.bf_last_error(ctx)
    assert bf.bf_set_dtype(ctx, bf.BF_CF16) == bf.BF_OK
    assert bf.bf_set_dtype(ctx, bf.BF_CI8) == bf.BF_OK
    assert bf.bf_set_kernel(ctx, 9) == bf.BF_EINVAL
    assert bf.bf_workspace_bytes(ctx) > 4 * 16 * 32 * 4
    assert bf.bf_workspace_bytes(ctx) % 1024 == 0
    assert bf.bf_set_workspace(ctx, None, 1 << 20) == bf.BF_EINVAL
    assert bf.bf_set_workspace(ctx, 0x1000 + 8, 1 << 30) == bf.BF_EINVAL  # misaligned
    assert bf.bf_set_workspace(ctx, 0x10000, 16) == bf.BF_ENOMEM
    # run before geometry
    assert bf.bf_run(ctx, 0x10000, 0x20000) == bf.BF_ENOGEOM
    assert bf.bf_run(ctx, None, 0x20000) == bf.BF_EINVAL
    # geometry validation happens before any device access
    r = np.zeros((32, 3)); f = np.full(4, 408e6); s = np.tile([0.0, 0.0, 1.0], (16, 1))
    assert bf.bf_set_geometry(ctx, r, f, s) == bf.BF_ENOGEOM  # no workspace yet
    assert bf.bf_set_geometry(ctx, None, f, s) == bf.BF_EINVAL
    s_bad = s.copy(); s_bad[3] = [0.0, 0.0, 1.1]
    assert bf.bf_set_geometry(ctx, r, f, s_bad) == bf.BF_EINVAL
    assert "unit vector" in bf.bf_last_error(ctx)
    f_bad = f.copy(); f_bad[1] = np.nan
    assert bf.bf_set_geometry(ctx, r, f_bad, s) == bf.BF_EINVAL
    r_bad = r.copy(); r_bad[0, 0] = np.inf
    assert bf.bf_set_geometry(ctx, r_bad, f, s) == bf.BF_EINVAL
    assert bf.bf_set_antenna_gains(ctx, np.ones(32, dtype=complex)) == bf.BF_ENOGEOM  # no workspace yet
    gbad = np.ones(32, dtype=complex); gbad[5] = np.nan
    assert bf.bf_set_antenna_gains(ctx, gbad) == bf.BF_EINVAL
    assert bf.bf_staging_bytes(ctx, 2) >= 2 * (2 * 256 * 32 * 2 + 2 * 16 * 16 * 4)
    assert bf.bf_launch_count(ctx) == 0
    bf.bf_destroy(ctx)


def test_no_device_means_error_not_fallback(bf):
    """On a box without a GPU the compute entry points must fail loudly (BF_ECUDA/BF_EUNSUPPORTED)."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    ctx = bf.bf_create(8, 2, 4, 64, 16)
    assert bf.bf_set_workspace(ctx, 0x7f0000000000, bf.bf_workspace_bytes(ctx)) == bf.BF_OK  # pointer only recorded
    r = np.zeros((8, 3)); f = np.full(2, 100e6); s = np.tile([0.0, 0.0, 1.0], (4, 1))
    rc = bf.bf_set_geometry(ctx, r, f, s)
    assert rc in (bf.BF_ECUDA, bf.BF_EUNSUPPORTED), rc
    assert bf.bf_last_error(ctx)
    bf.bf_destroy(ctx)


def test_kernel_selection_is_static_function_of_shape(bf):
    ctx = bf.bf_create(5, 3, 1, 7, 7)  # odd nant: only the generic kernel takes it
    assert bf.bf_selected_kernel(ctx) == bf.BF_KERNEL_SIMT
    bf.bf_set_kernel(ctx, bf.BF_KERNEL_UMMA)
    assert bf.bf_selected_kernel(ctx) == bf.BF_KERNEL_UMMA  # forced; bf_run would report BF_EUNSUPPORTED
    bf.bf_destroy(ctx)


def test_mode_entry_points_validate_without_gpu(bf):
    """Rows f3/f4: voltage beams, incoherent beam, double-buffered weights -- argument checks only."""
    ctx = bf.bf_create(32, 4, 16, 256, 16)
    one = bf.bf_workspace_bytes(ctx)
    assert bf.bf_set_weight_buffers(ctx, 3) == bf.BF_EINVAL
    assert bf.bf_set_weight_buffers(ctx, 2) == bf.BF_OK
    assert bf.bf_workspace_bytes(ctx) == 2 * one          # a second (geometry, weight operand) buffer
    assert bf.bf_set_weight_buffers(ctx, 1) == bf.BF_OK
    r = np.zeros((32, 3)); f = np.full(4, 408e6); s = np.tile([0.0, 0.0, 1.0], (16, 1))
    assert bf.bf_update_geometry(ctx, r, f, s) == bf.BF_EINVAL     # needs two buffers
    assert "bf_set_weight_buffers" in bf.bf_last_error(ctx)
    assert bf.bf_run_beams(ctx, 0x10000, 0x20000, 1.0) == bf.BF_ENOGEOM
    assert bf.bf_run_beams(ctx, None, 0x20000, 1.0) == bf.BF_EINVAL
    assert bf.bf_run_incoherent(ctx, None, 0x20000) == bf.BF_EINVAL
    assert bf.bf_run_incoherent(ctx, 0x10000, None) == bf.BF_EINVAL
    assert bf.bf_set_workspace(ctx, 0x10000, 1 << 30) == bf.BF_OK
    assert bf.bf_set_weight_buffers(ctx, 2) == bf.BF_EINVAL        # too late: the workspace is laid out
    bf.bf_destroy(ctx)


def test_dtype_is_fixed_once_the_workspace_is_set(bf):
    """The workspace layout depends on the element type (which weight operands exist): bf_set_dtype after
    bf_set_workspace must be refused, not silently leave a kernel without its operand."""
    ctx = bf.bf_create(32, 4, 16, 256, 16)
    assert bf.bf_set_dtype(ctx, bf.BF_CF16) == bf.BF_OK
    n = bf.bf_workspace_bytes(ctx)
    assert bf.bf_set_workspace(ctx, 0x10000, n) == bf.BF_OK          # pointer is only recorded (no CUDA call)
    assert bf.bf_set_dtype(ctx, bf.BF_CF16) == bf.BF_OK              # same type: fine
    assert bf.bf_set_dtype(ctx, bf.BF_CI8) == bf.BF_EINVAL
    assert "before bf_set_workspace" in bf.bf_last_error(ctx)
    bf.bf_destroy(ctx)


def test_workspace_grows_with_the_second_coefficient_term(bf):
    """nint < 16 carries a second fp16 term per coefficient (bf_internal.h BF_LO_NINT): the workspace says so."""
    a = bf.bf_create(64, 4, 40, 256, 16)
    b = bf.bf_create(64, 4, 40, 256, 8)
    assert bf.bf_workspace_bytes(b) > bf.bf_workspace_bytes(a) * 1.8
    bf.bf_destroy(a); bf.bf_destroy(b)


def test_clock_probe_argument(bf):
    ctx = bf.bf_create(32, 4, 16, 256, 16)
    assert bf.bf_set_clock_probe(ctx, None) == bf.BF_OK
    assert bf.bf_set_clock_probe(ctx, 0x1004) == bf.BF_EINVAL        # 8-byte alignment
    assert bf.bf_set_clock_probe(ctx, 0x1008) == bf.BF_OK
    bf.bf_destroy(ctx)
