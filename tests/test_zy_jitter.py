"""The parity and repeatability lists once more on the JITTER build of the library (GPU).

libbf_jitter.so is libbf.so compiled with -DBF_JITTER=1: a pseudo-random sleep of 0-2 us in front of one mbarrier wait
in four (csrc/ptx.cuh), different in every warp, CTA and launch.  The warp-specialised kernels (TMA producer, convert
warps, MMA warps, epilogue sets) then meet their barriers with leads and in orders the undisturbed kernels never show.
Results must not move: every tensor-core parity case stays within the 1e-3 bar of the oracle and the 50-run cases stay
bit-equal.  This stands in for compute-sanitizer's race checks, which are closed on this pool;
the idle-MMA-warp race fixed in bf_umma.cu / bf_umma_kblock.cu is the kind of fault it is there to catch.

The lists run in a child pytest with BF_LIBRARY pointing at the jitter build, so this process keeps the product library.
"""
import ctypes
import os
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def jitter_lib():
    from paper_1412_4907_b200 import build
    path = build.build(jitter=True)     # in-tree, rebuilt only when a source is newer
    L = ctypes.CDLL(path)
    L.bf_version.restype = ctypes.c_char_p
    assert b"jitter" in L.bf_version(), L.bf_version()
    return path


def run_child(jitter_lib, args):
    env = dict(os.environ, BF_LIBRARY=jitter_lib)
    r = subprocess.run([sys.executable, "-m", "pytest", "-q", "-x", "-m", "gpu", "-p", "no:cacheprovider"] + args,
                       cwd=ROOT, env=env, capture_output=True, text=True, timeout=1500)
    tail = r.stdout[-2500:] + r.stderr[-1500:]
    assert r.returncode == 0, tail
    assert " passed" in r.stdout and "failed" not in r.stdout, tail
    return r.stdout


def test_combinations_and_fifty_runs_under_jitter(jitter_lib):
    out = run_child(jitter_lib, ["tests/test_gpu_combos.py"])
    print(out.strip().splitlines()[-1])


def test_tensor_core_parity_lists_under_jitter(jitter_lib):
    # every shape list that launches a tensor-core kernel; the CUDA-core kernel has no barriers to shake
    out = run_child(jitter_lib, ["tests/test_gpu_parity.py", "-k",
                                 "(small_shapes and not simt) or i8_kernel or bin_per_lane or extreme or full_size"])
    print(out.strip().splitlines()[-1])


def test_side_modes_under_jitter(jitter_lib):
    out = run_child(jitter_lib, ["tests/test_gpu_modes.py", "-k", "voltage_beams or tracking or gains_chunks"])
    print(out.strip().splitlines()[-1])
