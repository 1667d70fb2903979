"""GPU parity of the "next" rows: voltage beams and the incoherent beam (f4) and
double-buffered weight updates for tracking beams (f3), each through the C ABI against the oracle.

Tolerances:
* voltage beams: per (channel, beam) row  max_t |y_gpu/scale - y_ref| <= 4e-3 * rms_t |y_ref|.
  Two error sources, both per sample: the fp16 weight operand (rms 2e-4 of |y|, worst sample of a few
  thousand ~8e-4) and ONE rounding of each output component to fp16 (2^-11 = 4.9e-4 of that component,
  components reach ~4 rms).  The sum stays below 3e-3 rms; 4e-3 is the bar.
* incoherent beam: integer inputs are summed exactly and rounded once to fp32 (rel 2^-24 = 6e-8): bar 2e-7;
  fp16 inputs are summed in fp32 (rel ~ sqrt(n) 2^-24): bar 1e-5.
* tracking: the power bar of test_gpu_parity.py (1e-3 per row), for every block with ITS geometry.
"""
import os

import numpy as np
import pytest

import oracle
import synthetic

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def bf():
    import paper_1412_4907_b200 as bf
    bf.lib()
    return bf


def bf_dtype(bf, w):
    return {"ci8": bf.BF_CI8, "cf16": bf.BF_CF16, "ci4": bf.BF_CI4}[w.dtype]


# ------------------------------------------------------------------ f4: voltage beams
BEAM_CASES = [
    # nant nchan nbeam nsamp dtype
    (32, 2, 16, 512, "ci8"),
    (32, 2, 3, 1000, "ci8"),     # ragged time tail, padding rows in the quadrant
    (32, 1, 65, 260, "ci8"),     # second M tile, tail tile of 4 samples
    (32, 1, 130, 256, "ci8"),    # three M tiles (beam groups of 4)
    (32, 2, 8, 250, "ci8"),      # nsamp % 4 != 0: scalar stores
    (16, 2, 9, 300, "ci8"),
    (64, 2, 33, 512, "ci8"),     # K-blocked kernel, int8
    (64, 2, 16, 256, "cf16"),    # K-blocked kernel, fp16
    (5, 2, 3, 77, "ci8"),        # generic kernel only
    (32, 2, 16, 256, "ci4"),
    (32, 3, 1, 2050, "ci8"),     # int8 kernel: one beam, several tiles, ragged tail of one sample pair
    (32, 2, 32, 768, "ci8"),     # int8 kernel: 128 accumulator columns
    (64, 2, 16, 256, "ci4"),     # 4+4-bit input on the K-blocked kernel in voltage-beam mode
    (1024, 1, 70, 256, "ci4"),   # ... with 32 K-blocks and a second, partial M-tile
]


@pytest.mark.parametrize("nant,nchan,nbeam,nsamp,dtype", BEAM_CASES)
@pytest.mark.parametrize("kernel", ["simt", "auto", "f16"])
def test_voltage_beams_match_oracle(bf, nant, nchan, nbeam, nsamp, dtype, kernel):
    import torch
    w = synthetic.make_case(nant, nchan, nbeam, nsamp, 1, dtype)
    v = w.make_voltages()
    ref = oracle.beams(w.ant_xyz, w.freqs, w.beam_dir, v)  # [C][B][T] complex128
    scale = 0.25 if dtype != "cf16" else 2.0
    k = {"simt": bf.BF_KERNEL_SIMT, "auto": bf.BF_KERNEL_AUTO, "f16": bf.BF_KERNEL_UMMA_F16}[kernel]
    if kernel == "f16" and (nant % 8 != 0 or (dtype == "ci4" and nant % 16 != 0)):
        pytest.skip("no fp16 tensor-core variant for this shape")
    B = bf.Beamformer(w.nant, w.nchan, w.nbeam, w.nsamp, 1, dtype=bf_dtype(bf, w), kernel=k)
    B.set_geometry(w.ant_xyz, w.freqs, w.beam_dir)
    y = torch.full((w.nchan, w.nbeam, w.nsamp, 2), float("nan"), dtype=torch.float16, device="cuda")
    B.run_beams(torch.from_numpy(v).cuda(), y, scale=scale)
    torch.cuda.synchronize()
    out = y.cpu().numpy().astype(np.float64)
    B.close()
    assert np.isfinite(out).all()
    yg = (out[..., 0] + 1j * out[..., 1]) / scale
    err = np.abs(yg - ref).max(axis=-1)
    rms = np.sqrt((np.abs(ref) ** 2).mean(axis=-1))
    worst = (err / rms).max()
    assert worst <= 4e-3, f"worst row error {worst:.3e}"


def test_voltage_beams_square_to_the_powers(bf):
    """|y|^2 summed over nint (from the fp16 beams) agrees with bf_run's fused powers on the same input."""
    import torch
    w = synthetic.make_workload("tiny").sub(nchan=4)
    v = torch.from_numpy(w.make_voltages()).cuda()
    B = bf.Beamformer(w.nant, w.nchan, w.nbeam, w.nsamp, w.nint)
    B.set_geometry(w.ant_xyz, w.freqs, w.beam_dir)
    P = B.run(v).cpu().numpy().astype(np.float64)
    y = B.run_beams(v, scale=0.5).cpu().numpy().astype(np.float64) / 0.5
    B.close()
    P2 = (y ** 2).sum(-1).reshape(w.nchan, w.nbeam, -1, w.nint).sum(-1)
    assert (np.abs(P2 - P).max(axis=-1) / P.mean(axis=-1)).max() < 2e-3


# ------------------------------------------------------------------ f4: incoherent beam
INC_CASES = [
    # nant nchan nsamp nint dtype
    (32, 3, 1024, 16, "ci8"),
    (32, 2, 4096, 64, "ci8"),
    (8, 2, 128, 1, "ci8"),        # one sample per bin, 16-byte bins
    (5, 2, 77, 7, "ci8"),         # unaligned bins
    (256, 2, 512, 64, "ci8"),     # 32 KiB bins: one block per bin
    (32, 2, 256, 16, "ci4"),
    (3, 2, 50, 5, "ci4"),
    (16, 2, 256, 32, "cf16"),
    (256, 1, 256, 128, "cf16"),
]


@pytest.mark.parametrize("nant,nchan,nsamp,nint,dtype", INC_CASES)
def test_incoherent_beam_matches_oracle(bf, nant, nchan, nsamp, nint, dtype):
    import torch
    w = synthetic.make_case(nant, nchan, 1, nsamp, nint, dtype)
    v = w.make_voltages()
    ref = oracle.incoherent(v, nint)
    B = bf.Beamformer(nant, nchan, 1, nsamp, nint, dtype=bf_dtype(bf, w))
    P = torch.full((nchan, nsamp // nint), float("nan"), dtype=torch.float32, device="cuda")
    B.run_incoherent(torch.from_numpy(v).cuda(), P)   # no geometry needed
    torch.cuda.synchronize()
    out = P.cpu().numpy().astype(np.float64)
    B.close()
    tol = 1e-5 if dtype == "cf16" else 2e-7
    assert np.isfinite(out).all()
    assert (np.abs(out - ref) / ref).max() <= tol


def test_incoherent_full_size_sampled(bf):
    """medium-sized buffer in the launch configuration bench.py --mode incoherent times; sampled bins vs the oracle."""
    import torch
    w = synthetic.make_workload("medium").sub(nchan=64)
    v = synthetic.fill_voltages_torch(w, torch.device("cuda"))
    B = bf.Beamformer(w.nant, w.nchan, w.nbeam, w.nsamp, w.nint)
    P = B.run_incoherent(v).cpu().numpy().astype(np.float64)
    B.close()
    for c in (0, 31, 63):
        ref = oracle.incoherent(v[c:c + 1].cpu().numpy(), w.nint)[0]
        assert (np.abs(P[c] - ref) / ref).max() <= 2e-7


# ------------------------------------------------------------------ f3: tracking beams (double-buffered weights)
def test_tracking_updates_switch_weights_between_runs(bf):
    import torch
    w = synthetic.make_workload("tiny").sub(nchan=8)
    v = w.make_voltages()
    vd = torch.from_numpy(v).cuda()
    # three pointings: the beam fan drifts by a fraction of a beam width per block
    dirs = []
    for k in range(3):
        th = np.deg2rad(np.linspace(-30, 30, w.nbeam) + 0.7 * k)
        dirs.append(np.stack([np.sin(th), np.zeros_like(th), np.cos(th)], axis=1))
    refs = [oracle.beamform(w.ant_xyz, w.freqs, d, v, w.nint) for d in dirs]
    B = bf.Beamformer(w.nant, w.nchan, w.nbeam, w.nsamp, w.nint, weight_buffers=2)
    run_s, upd_s = torch.cuda.Stream(), torch.cuda.Stream()
    B.set_geometry(w.ant_xyz, w.freqs, dirs[0], stream=run_s)
    outs = []
    # no host synchronisation anywhere in the loop: ordering is the library's job
    for rep in range(4):
        for k in range(3):
            P = B.run(vd, stream=run_s)
            outs.append((k, P))
            B.update_geometry(w.ant_xyz, w.freqs, dirs[(k + 1) % 3], update_stream=upd_s)
    torch.cuda.synchronize()
    for k, P in outs:
        out = P.cpu().numpy().astype(np.float64)
        worst = (np.abs(out - refs[k]).max(axis=-1) / refs[k].mean(axis=-1)).max()
        assert worst <= 1e-3, (k, worst)
    # the pointings really differ (the test would pass trivially otherwise)
    assert (np.abs(refs[1] - refs[0]).max(axis=-1) / refs[0].mean(axis=-1)).max() > 0.05
    # weights reported after an update are the new ones
    B.update_geometry(w.ant_xyz, w.freqs, dirs[2], update_stream=upd_s)
    Wg = B.weights()
    Wo = oracle.weights(w.ant_xyz, w.freqs, dirs[2])
    assert np.abs(Wg - Wo).max() < 2.0 ** -10
    B.close()


def test_update_geometry_needs_two_buffers(bf):
    w = synthetic.make_workload("tiny").sub(nchan=2)
    B = bf.Beamformer(w.nant, w.nchan, w.nbeam, w.nsamp, w.nint)
    B.set_geometry(w.ant_xyz, w.freqs, w.beam_dir)
    with pytest.raises(bf.BfError) as e:
        B.update_geometry(w.ant_xyz, w.freqs, w.beam_dir)
    assert e.value.code == bf.BF_EINVAL
    B.close()


# ------------------------------------------------------------------ boundary: a failing stream-ordering call is reported
def test_stream_ordering_failures_surface_as_bf_ecuda():
    """every cudaStreamWaitEvent / cudaEventRecord of the library is checked.  The compute stream
    handed to bf_run_host is put into graph-capture mode first: waiting there on the "copy landed" event, which is
    recorded on the (non-capturing) copy stream, is illegal, so the library's cudaStreamWaitEvent fails and the call must
    come back with BF_ECUDA.  (A destroyed stream handle is not a usable injection: the runtime accepted it.)  Run in a
    subprocess: the broken capture must not leak into the other tests."""
    import subprocess
    import sys
    code = r'''
import ctypes, sys, numpy as np, torch
sys.path.insert(0, ".")
import synthetic, paper_1412_4907_b200 as bf
w = synthetic.make_workload("tiny").sub(nchan=4, nsamp=256)
B = bf.Beamformer(w.nant, w.nchan, w.nbeam, w.nsamp, w.nint)
B.set_geometry(w.ant_xyz, w.freqs, w.beam_dir)
hv = torch.from_numpy(w.make_voltages()).pin_memory()
hp = torch.empty((w.nchan, w.nbeam, w.nbin), dtype=torch.float32).pin_memory()
try:
    rt = ctypes.CDLL("libcudart.so.12")
except OSError:
    rt = ctypes.CDLL("/usr/local/cuda/lib64/libcudart.so.12")
cs, xs = torch.cuda.Stream(), torch.cuda.Stream()
B.run_host(hv, hp, 2, cs, xs)                      # the same call is fine on ordinary streams
cs.synchronize(); xs.synchronize()
assert rt.cudaStreamBeginCapture(ctypes.c_void_p(cs.cuda_stream), 0) == 0
try:
    B.run_host(hv, hp, 2, cs, xs)
    print("RESULT no-error")
except bf.BfError as e:
    print("RESULT", e.code, str(e)[:120])
'''
    r = subprocess.run([sys.executable, "-c", code], capture_output=True, text=True, timeout=300,
                       cwd=os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("RESULT")]
    assert lines, (r.returncode, r.stdout[-500:], r.stderr[-1500:])
    assert lines[0].split()[1] == "-3", lines[0]          # BF_ECUDA


@pytest.mark.parametrize("dtype,nbeam", [("ci8", 24), ("ci4", 12), ("ci4", 28)])
def test_bin_per_lane_kernel_with_gains_chunks_and_tracking(bf, dtype, nbeam):
    """The bin-per-lane int8-operand kernel (bf_umma_i8b.cu: 17-32 beams on int8 input, <= 32 beams on 4+4-bit input, its
    <= 16-beam form with the operands in tensor memory) behind the rest of the API: per-channel antenna gains folded into
    its two-limb weights, bf_run_host's channel chunks (other base pointers and channel counts: fresh tensor maps), and a
    tracking update that switches its weight buffer.  256 bins per channel, so the automatic choice is this kernel."""
    import torch
    N, C, T, I = 32, 6, 4096, 16
    w = synthetic.make_case(N, C, nbeam, T, I, dtype, seed=21)
    v = w.make_voltages()
    if dtype == "ci8":
        x = v[..., 0].astype(np.float64) + 1j * v[..., 1]
    else:  # high nibble re, low nibble im, two's complement (A20)
        re = (v >> 4).astype(np.int16); im = (v & 0xF).astype(np.int16)
        x = np.where(re > 7, re - 16, re).astype(np.float64) + 1j * np.where(im > 7, im - 16, im)
    rng = np.random.default_rng(5)
    g = rng.uniform(0.5, 1.5, (C, N)) * np.exp(2j * np.pi * rng.random((C, N)))
    dirs = [w.beam_dir, np.roll(w.beam_dir, 3, axis=0)]
    refs = [oracle.beamform(w.ant_xyz, w.freqs, d, np.ascontiguousarray(x * g[:, None, :]), I) for d in dirs]
    B = bf.Beamformer(N, C, nbeam, T, I, dtype=bf_dtype(bf, w), weight_buffers=2)
    assert B.kernel_name == "umma-i8"
    B.set_antenna_gains(g, per_channel=True)
    B.set_geometry(w.ant_xyz, w.freqs, dirs[0])
    vd = torch.from_numpy(v).cuda()
    direct = B.run(vd).cpu().numpy()
    err = (np.abs(direct - refs[0]).max(axis=-1) / refs[0].mean(axis=-1)).max()
    assert err <= 1e-3, err
    cs, xs = torch.cuda.Stream(), torch.cuda.Stream()
    pinned = torch.from_numpy(v).pin_memory()
    for cpc in (4, 1):   # 6 channels in chunks of 4 + 2, then one by one
        hp = torch.empty((C, nbeam, T // I), dtype=torch.float32).pin_memory()
        hp.fill_(float("nan"))
        B.run_host(pinned, hp, cpc, cs, xs)
        cs.synchronize(); xs.synchronize()
        np.testing.assert_array_equal(hp.numpy(), direct)
    upd = torch.cuda.Stream()
    B.update_geometry(w.ant_xyz, w.freqs, dirs[1], update_stream=upd)
    out1 = B.run(vd).cpu().numpy()
    err = (np.abs(out1 - refs[1]).max(axis=-1) / refs[1].mean(axis=-1)).max()
    assert err <= 1e-3, err
    assert (np.abs(refs[1] - refs[0]).max(axis=-1) / refs[0].mean(axis=-1)).max() > 0.05
    B.close()
