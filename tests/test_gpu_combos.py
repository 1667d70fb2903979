"""GPU parity of combinations the per-kernel lists do not reach, and repeatability of every tensor-core kernel.

Each case names the code path it is there for:
* the coefficients-resident kernel with a LAST beam group of one M-tile (gm == 1: the second MMA warp idles and its
  "operand free" commit is issued by the first) -- 260 / 520 beams on 32 antennas, groups of four tiles;
* two-term coefficients (nint < 16) with more than one beam group, the last one a single tile -- 192 beams at nint 4 / 8;
* two-term coefficients together with two weight buffers (the residual plane of buffer 1) -- tracking at nint 4;
* bf_run_host's channel chunks on the bin-per-lane fp16 kernel (fresh 5-D tensor maps per chunk base pointer);
* every tensor-core kernel 50 times on one input, bit-equal each time, half of the runs with a device-to-device copy
  hammering HBM / L2 on a second stream: compute-sanitizer is closed on this pool, so the mbarrier protocols of the
  warp-specialised kernels are shaken by repetition under changed timing instead.  (nint = 64 k on the fp16 kernels
  accumulates with fp32 atomics and is not bit-reproducible; it is left out, see include/bf.h.)
"""
import numpy as np
import pytest

import oracle
import synthetic

pytestmark = pytest.mark.gpu

TOL = 1e-3
DT = {"ci8": 0, "cf16": 1, "ci4": 2}


@pytest.fixture(scope="module")
def bf():
    import paper_1412_4907_b200 as bf
    bf.lib()
    return bf


def worst_row(out, ref):
    out = np.asarray(out, dtype=np.float64)
    assert out.shape == ref.shape and np.isfinite(out).all()
    return (np.abs(out - ref).max(axis=-1) / ref.mean(axis=-1)).max()


GROUP_CASES = [
    # nant nchan nbeam nsamp nint dtype kernel
    (32, 2, 260, 512, 16, "ci8", "umma-f16-resident"),   # 5 M-tiles = one group of 4 + a group of ONE
    (32, 1, 321, 512, 32, "ci8", "umma-f16-resident"),   # 6 M-tiles = 4 + 2, the last tile holds one beam
    (32, 1, 520, 256, 64, "ci4", "umma-f16-resident"),   # 9 M-tiles = 4 + 4 + 1 on 4+4-bit input
    (32, 3, 192, 512, 4, "ci8", "umma-f16-resident"),    # two-term coefficients, groups of two tiles: 2 + 1
    (32, 2, 192, 768, 8, "ci8", "umma-f16-resident"),
    (32, 2, 129, 512, 2, "ci4", "umma-f16-resident"),    # two-term, 3 tiles, the last with a single beam, 4-bit unpack
]


@pytest.mark.parametrize("case", GROUP_CASES, ids=lambda s: "N%d-C%d-B%d-T%d-I%d-%s" % s[:6])
def test_beam_groups_with_a_single_tile(bf, case):
    import torch
    N, C, B, T, I, dtype, name = case
    w = synthetic.make_case(N, C, B, T, I, dtype, seed=11)
    v = w.make_voltages()
    ref = oracle.beamform(w.ant_xyz, w.freqs, w.beam_dir, v, I)
    Bf = bf.Beamformer(N, C, B, T, I, dtype=DT[dtype])
    assert Bf.kernel_name == name
    Bf.set_geometry(w.ant_xyz, w.freqs, w.beam_dir)
    P = Bf.empty_powers().fill_(float("nan"))
    Bf.run(torch.from_numpy(v).cuda(), P)
    torch.cuda.synchronize()
    assert worst_row(P.cpu().numpy(), ref) <= TOL
    Bf.close()


def test_tracking_with_two_term_coefficients(bf):
    """nint = 4: every weight buffer has a residual plane; the update writes buffer 1's, the next run reads it."""
    import torch
    N, C, B, T, I = 32, 4, 70, 512, 4
    w = synthetic.make_case(N, C, B, T, I, "ci8", seed=13)
    v = w.make_voltages()
    vd = torch.from_numpy(v).cuda()
    dirs = [w.beam_dir, np.roll(w.beam_dir, 5, axis=0), w.beam_dir[::-1].copy()]
    refs = [oracle.beamform(w.ant_xyz, w.freqs, d, v, I) for d in dirs]
    Bf = bf.Beamformer(N, C, B, T, I, weight_buffers=2)
    assert Bf.kernel_name == "umma-f16-resident"
    run_s, upd_s = torch.cuda.Stream(), torch.cuda.Stream()
    Bf.set_geometry(w.ant_xyz, w.freqs, dirs[0], stream=run_s)
    outs = []
    for rep in range(3):
        for k in range(3):
            outs.append((k, Bf.run(vd, stream=run_s)))
            Bf.update_geometry(w.ant_xyz, w.freqs, dirs[(k + 1) % 3], update_stream=upd_s)
    torch.cuda.synchronize()
    for k, P in outs:
        assert worst_row(P.cpu().numpy(), refs[k]) <= TOL, k
    assert worst_row(refs[1], refs[0]) > 0.05   # the pointings really differ
    # what bf_get_weights reports is hi + lo of the buffer the next run uses: 22 bits
    Wg, Wo = Bf.weights(), oracle.weights(w.ant_xyz, w.freqs, dirs[0])
    assert np.abs(Wg - Wo).max() <= 2.0 ** -21
    Bf.close()


@pytest.mark.parametrize("dtype", ["ci8", "ci4"])
def test_run_host_chunks_on_the_bin_per_lane_fp16_kernel(bf, dtype):
    import torch
    N, C, B, T, I = 32, 7, 48, 4096, 16
    w = synthetic.make_case(N, C, B, T, I, dtype, seed=17)
    v = w.make_voltages()
    ref = oracle.beamform(w.ant_xyz, w.freqs, w.beam_dir, v, I)
    Bf = bf.Beamformer(N, C, B, T, I, dtype=DT[dtype])
    assert Bf.kernel_name == "umma-f16-binlane"
    Bf.set_geometry(w.ant_xyz, w.freqs, w.beam_dir)
    hv = torch.from_numpy(v).pin_memory()
    cs, xs = torch.cuda.Stream(), torch.cuda.Stream()
    for cpc in (2, 3, 7):          # 2 + 2 + 2 + 1, 3 + 3 + 1, one chunk
        hp = torch.full((C, B, T // I), float("nan"), dtype=torch.float32).pin_memory()
        Bf.run_host(hv, hp, cpc, cs, xs)
        cs.synchronize(); xs.synchronize()
        assert worst_row(hp.numpy(), ref) <= TOL, cpc
    direct = Bf.run(torch.from_numpy(v).cuda())
    torch.cuda.synchronize()
    assert np.array_equal(direct.cpu().numpy(), hp.numpy())   # chunks change nothing: bit-equal to bf_run
    Bf.close()


REPEAT_CASES = [
    # nant nchan nbeam nsamp nint dtype forced-kernel expected-name
    (32, 40, 16, 4096, 16, "ci8", "auto", "umma-i8"),            # time-on-M, two samples per row (bf_umma_i8.cu, wide)
    (16, 40, 9, 3000, 4, "ci8", "auto", "umma-i8"),              # time-on-M, narrow rows, ragged tail
    (32, 40, 24, 4096, 16, "ci8", "auto", "umma-i8"),            # bin per lane, int8 operands in shared memory
    (32, 40, 5, 3072, 6, "ci8", "auto", "umma-i8"),              # bin per lane, two tile sets, three tiles per super-tile
    (32, 40, 12, 4096, 16, "ci4", "auto", "umma-i8"),            # bin per lane, unpacked operands in tensor memory
    (32, 40, 28, 4096, 16, "ci4", "auto", "umma-i8"),            # bin per lane, 4-bit through shared memory
    (32, 40, 64, 8192, 16, "ci8", "auto", "umma-f16-binlane"),   # fp16 bin per lane, voltages as the A operand in TMEM
    (32, 40, 48, 5632, 22, "ci4", "auto", "umma-f16-binlane"),   # ... 4-bit input, eleven raw rows per bin
    (32, 40, 128, 2048, 64, "ci8", "auto", "umma-f16-resident"),  # the headline kernel (medium's per-channel shape)
    (32, 40, 130, 1024, 4, "ci4", "auto", "umma-f16-resident"),  # two-term coefficients, 4-bit unpack, groups 2 + 1
    (32, 40, 16, 4096, 16, "ci8", "f16", "umma-f16-resident"),   # the SPREAD variant (<= 32 beams forced to fp16)
    (32, 40, 260, 1024, 16, "ci8", "auto", "umma-f16-resident"),  # groups of four tiles + a group of ONE: the second MMA warp idles
    (32, 40, 192, 1024, 8, "ci8", "auto", "umma-f16-resident"),  # the same with two-term coefficients (groups 2 + 1)
    (1024, 40, 130, 1024, 32, "ci8", "auto", "umma-f16-kblock"),  # K-blocked, groups 2 + 1 with 32 K-blocks per item
    (256, 30, 192, 1024, 32, "cf16", "auto", "umma-f16-kblock"),  # K-blocked fp16 input, groups 2 + 1, 8 K-blocks
    (256, 6, 256, 1024, 32, "cf16", "auto", "umma-f16-kblock"),  # K-blocked (large-N's per-channel shape)
    (64, 9, 256, 992, 32, "ci8", "auto", "umma-f16-kblock"),     # K-blocked, int8 conversion, ragged tail
    (1024, 2, 128, 512, 32, "ci4", "auto", "umma-f16-kblock"),   # K-blocked, 4-bit, 32 K-blocks
]


@pytest.mark.parametrize("case", REPEAT_CASES, ids=lambda s: "N%d-C%d-B%d-T%d-I%d-%s-%s" % s[:7])
def test_fifty_runs_are_bit_equal(bf, case):
    import torch
    N, C, B, T, I, dtype, forced, name = case
    w = synthetic.make_case(N, C, B, T, I, dtype, seed=23)
    dev = torch.device("cuda")
    v = synthetic.fill_voltages_torch(w, dev, chunk_chan=8)
    Bf = bf.Beamformer(N, C, B, T, I, dtype=DT[dtype], kernel={"auto": bf.BF_KERNEL_AUTO, "f16": bf.BF_KERNEL_UMMA_F16}[forced])
    assert Bf.kernel_name == name
    Bf.set_geometry(w.ant_xyz, w.freqs, w.beam_dir)
    run_s, noise_s = torch.cuda.Stream(), torch.cuda.Stream()   # non-blocking streams: order everything explicitly
    noise_a = torch.empty(64 << 20, dtype=torch.uint8, device=dev)
    noise_b = torch.empty_like(noise_a)
    outs = [Bf.empty_powers() for _ in range(4)]
    first = Bf.empty_powers()
    torch.cuda.synchronize()
    with torch.cuda.stream(run_s):
        first.fill_(float("nan"))
        Bf.run(v, first, stream=run_s)
    run_s.synchronize()
    assert torch.isfinite(first).all() and float(first.mean()) > 0
    # one channel against the oracle: what is repeated is also right
    c = C // 2
    ref = oracle.beamform(w.ant_xyz, w.freqs[c:c + 1], w.beam_dir, v[c:c + 1].cpu().numpy(), I)
    assert worst_row(first[c:c + 1].cpu().numpy(), ref) <= TOL
    bad = 0
    for it in range(50):
        P = outs[it % 4]
        if it % 2:   # other traffic on the memory system while the kernel runs
            with torch.cuda.stream(noise_s):
                for _ in range(3):
                    noise_b.copy_(noise_a, non_blocking=True)
        with torch.cuda.stream(run_s):
            P.fill_(float("nan"))
            Bf.run(v, P, stream=run_s)
        run_s.synchronize()
        bad += int(not torch.equal(P, first))
    torch.cuda.synchronize()
    assert bad == 0, f"{bad} of 50 runs differ from the first"
    Bf.close()


GRAPH_CASES = [
    # nant nchan nbeam nsamp nint dtype kernel
    (32, 64, 16, 1024, 16, "ci8", "umma-i8"),              # BASELINE.json's `tiny`
    (32, 24, 24, 4096, 16, "ci8", "umma-i8"),              # bin per lane (5-D tensor map from the cache)
    (32, 24, 64, 8192, 16, "ci4", "umma-f16-binlane"),
    (32, 24, 128, 2048, 64, "ci8", "umma-f16-resident"),
    (256, 4, 256, 1024, 32, "cf16", "umma-f16-kblock"),
    (64, 4, 70, 1024, 128, "ci8", "umma-f16-kblock"),      # nint = 128: the memset + atomics path is two graph nodes
]


@pytest.mark.parametrize("case", GRAPH_CASES, ids=lambda s: "N%d-C%d-B%d-T%d-I%d-%s" % s[:6])
def test_bf_run_in_a_cuda_graph(bf, case):
    """include/bf.h: bf_run with one weight buffer may be captured once the same call has run un-captured.  Capture three
    calls on two alternating inputs, replay the graph 100 times, and compare with the direct calls."""
    import torch
    N, C, B, T, I, dtype, name = case
    dev = torch.device("cuda")
    w = synthetic.make_case(N, C, B, T, I, dtype, seed=29)
    va = synthetic.fill_voltages_torch(w, dev, chunk_chan=8)
    vb = torch.roll(va, 1, dims=1).contiguous()
    Bf = bf.Beamformer(N, C, B, T, I, dtype=DT[dtype])
    assert Bf.kernel_name == name
    Bf.set_geometry(w.ant_xyz, w.freqs, w.beam_dir)
    Pa, Pb = Bf.run(va), Bf.run(vb)          # un-captured first: attributes set, tensor maps cached
    torch.cuda.synchronize()
    ref = oracle.beamform(w.ant_xyz, w.freqs[:1], w.beam_dir, va[:1].cpu().numpy(), I)
    assert worst_row(Pa[:1].cpu().numpy(), ref) <= TOL
    atomic = name != "umma-i8" and I > 64
    Ga, Gb, Ga2 = (Bf.empty_powers() for _ in range(3))
    s = torch.cuda.Stream()
    g = torch.cuda.CUDAGraph()
    n0 = Bf.launches
    with torch.cuda.graph(g, stream=s):
        cur = torch.cuda.current_stream()
        Bf.run(va, Ga, stream=cur)
        Bf.run(vb, Gb, stream=cur)
        Bf.run(va, Ga2, stream=cur)
    assert Bf.launches - n0 == 3
    for rep in range(100):
        if rep in (0, 57):
            for G_ in (Ga, Gb, Ga2):
                G_.fill_(float("nan"))
            torch.cuda.synchronize()
        g.replay()
    torch.cuda.synchronize()
    for got, want in ((Ga, Pa), (Gb, Pb), (Ga2, Pa)):
        if atomic:   # fp32 atomics: equal to rounding of the partial sums
            assert worst_row(got.cpu().numpy(), want.cpu().numpy().astype(np.float64)) <= 1e-5
        else:
            assert torch.equal(got, want)
    Bf.close()


def test_bf_run_rejects_misaligned_pointers(bf):
    import torch
    w = synthetic.make_case(32, 2, 16, 256, 16, "ci8", seed=31)
    Bf = bf.Beamformer(32, 2, 16, 256, 16)
    Bf.set_geometry(w.ant_xyz, w.freqs, w.beam_dir)
    v = torch.zeros(2 * 256 * 32 * 2 + 64, dtype=torch.int8, device="cuda")
    P = torch.zeros(2 * 16 * 16 * 4 + 64, dtype=torch.uint8, device="cuda")
    assert bf.bf_run(Bf.ctx, v.data_ptr(), P.data_ptr()) == bf.BF_OK
    assert bf.bf_run(Bf.ctx, v.data_ptr(), P.data_ptr() + 4) == bf.BF_OK        # 4-byte aligned powers are fine
    assert bf.bf_run(Bf.ctx, v.data_ptr(), P.data_ptr() + 2) == bf.BF_EINVAL
    assert "powers" in bf.bf_last_error(Bf.ctx)
    assert bf.bf_run(Bf.ctx, v.data_ptr() + 8, P.data_ptr()) == bf.BF_EINVAL
    assert "voltages" in bf.bf_last_error(Bf.ctx)
    torch.cuda.synchronize()
    Bf.close()
