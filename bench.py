#!/usr/bin/env python
"""bench.py -- headline benchmark of the B200 coherent beamformer (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config medium] [--impl ours|reference]

One "step" is one pass of the whole hot path (ingest -> contraction -> |.|^2 -> integrate) over one
synthetic `medium` buffer (BASELINE.json configs[1]: 32 antennas, 1024 channels, 128 beams, 32768
samples, complex int8, nint 64).  Prints ONE JSON line (rank 0).  Metric: beamforming TFLOP/s at
8 flop per complex MAC.  N > 1 runs one replica per GPU on its own buffer (channels
are independent, so the path shards with no exchange; "weak" scaling) and reports the aggregate.

--impl reference times the fp64 CPU oracle (oracle/) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "beamforming TFLOP/s (8 flop/complex MAC)"
UNIT = "TFLOP/s"


def load_peaks():
    """Measured roofline denominators (driver-written), else the profiling guide's fallback."""
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            d = json.load(open(path))
            return {"hbm_gbs": float(d["hbm_gbs"]), "tensor_tflops": float(d.get("bf16_tflops_sustained", d["bf16_tflops"])),
                    "tensor_tflops_burst": float(d["bf16_tflops"]), "source": "measured"}
        except Exception:
            pass
    return {"hbm_gbs": 6650.0, "tensor_tflops": 1400.0, "tensor_tflops_burst": 1590.0, "source": "fallback"}


def workload_for(name):
    import synthetic
    if name.startswith("sweep-"):
        return synthetic.make_workload("sweep", nbeam=int(name.split("-")[1]))
    return synthetic.make_workload(name)


def algorithmic_bytes(w):
    """per channel read the voltages once, the weights once, write the powers."""
    return w.in_bytes + w.nchan * w.nbeam * w.nant * 4 + w.out_bytes


def rank_seed(base_seed: int, rank: int) -> int:
    """Every replica beamforms its own buffer (weak scaling, no exchange between ranks)."""
    return base_seed + 100 * rank


def aggregate(total_ms_local: float, units_local: float, dist_mod=None, device=None):
    """(max over ranks of the timed region, sum over ranks of the units processed).  With one
    process this is the identity; with several it is two all-reduces (MAX, SUM) on `device`."""
    if dist_mod is None:
        return total_ms_local, units_local
    import torch
    t = torch.tensor([total_ms_local], dtype=torch.float64, device=device)
    u = torch.tensor([units_local], dtype=torch.float64, device=device)
    dist_mod.all_reduce(t, op=dist_mod.ReduceOp.MAX)
    dist_mod.all_reduce(u, op=dist_mod.ReduceOp.SUM)
    return float(t.item()), float(u.item())


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.proc = None
        self.index = index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "20"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        time.sleep(0.05)
        self.proc.terminate()
        try:
            text, _ = self.proc.communicate(timeout=5)
        except Exception:
            self.proc.kill()
            text = ""
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in text.splitlines():
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for nm, val in zip(names, f[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(nm)
        if sm:
            out.update(sm_mhz=statistics.median(sm), sm_max_mhz=max(mx), samples=len(sm))
        out["reasons"] = sorted(reasons)
        return out


def time_oracle_sample(w, v_host_fn, target_s=15.0, max_chan=1 << 30):
    """The oracle as it stands on the host cores, on whole channels of the workload; returns
    (TFLOP/s, cores, description).  v_host_fn(chan_list) -> numpy voltages of those channels."""
    import numpy as np
    import oracle
    cores = oracle.num_threads()
    # calibrate on `cores` channels (one per thread), then size the sample for ~target_s
    n0 = min(w.nchan, cores)
    chans = list(range(n0))
    ws = w.sub(chan_idx=chans)
    v = v_host_fn(chans)
    t0 = time.perf_counter()
    oracle.beamform(ws.ant_xyz, ws.freqs, ws.beam_dir, v, ws.nint)
    dt0 = time.perf_counter() - t0
    per_chan = dt0 / n0
    n = int(max(n0, min(max_chan, w.nchan, target_s / max(per_chan, 1e-9))))
    n = max(cores, n // cores * cores) if n >= cores else n
    n = min(n, w.nchan)
    if n > n0:
        chans = list(range(n))
        ws = w.sub(chan_idx=chans)
        v = v_host_fn(chans)
        t0 = time.perf_counter()
        oracle.beamform(ws.ant_xyz, ws.freqs, ws.beam_dir, v, ws.nint)
        dt = time.perf_counter() - t0
    else:
        n, dt = n0, dt0
    flop = 8.0 * n * w.nbeam * w.nant * w.nsamp
    return flop / dt / 1e12, cores, f"{n} of {w.nchan} channels x all {w.nbeam} beams x all {w.nsamp} samples, {dt:.2f} s", dt, n


def run_reference(args):
    """--impl reference: the fp64 oracle on the host cores, each step a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import numpy as np
    import oracle
    w = workload_for(args.config)
    cores = oracle.num_threads()
    nchan = min(w.nchan, cores)  # one channel per thread per step keeps K+W steps within minutes
    chans = list(range(nchan))
    ws = w.sub(chan_idx=chans)
    v = w.make_voltages(nchan=nchan)
    steps = max(1, args.steps)
    for _ in range(max(0, args.warmup)):
        oracle.beamform(ws.ant_xyz, ws.freqs, ws.beam_dir, v, ws.nint)
    t0 = time.perf_counter()
    for _ in range(steps):
        oracle.beamform(ws.ant_xyz, ws.freqs, ws.beam_dir, v, ws.nint)
    dt = (time.perf_counter() - t0) / steps
    flop = 8.0 * nchan * w.nbeam * w.nant * w.nsamp
    val = flop / dt / 1e12
    sample = f"{nchan} of {w.nchan} channels x all {w.nbeam} beams x all {w.nsamp} samples per step"
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
        "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "nant": w.nant, "nchan": w.nchan, "nbeam": w.nbeam, "nsamp": w.nsamp,
                   "nint": w.nint, "input": w.dtype, "sample": sample},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="medium")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--kernel", default="auto", choices=["auto", "simt", "umma", "f16", "i8"])
    ap.add_argument("--mode", default="power", choices=["power", "beams", "incoherent"],
                    help="power = the headline path (bf_run); beams / incoherent = SURVEY 8(f) row f4 side modes")
    ap.add_argument("--nbeam", type=int, default=0, help="override the workload's beam count (beams mode: default 8)")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: weak = one full replica per rank (default); strong = ONE workload, channels sharded over the ranks")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--chan-per-chunk", type=int, default=0, help="e2e: channels per H2D chunk (0 = nchan/8)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import numpy as np
    import torch
    import synthetic
    import paper_1412_4907_b200 as bf

    bf.lib()  # fail loudly if the CUDA library is missing: there is no fallback
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dist = world > 1
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if dist:
        import torch.distributed as td
        td.init_process_group("nccl", device_id=dev)

    W = max(3, args.warmup)
    K = max(1, args.steps)
    if args.config.startswith("sweep") and args.nbeam:
        # the sweep's beam rule (A3) for any beam count, named sweep-B<n>
        args.config, args.nbeam = f"sweep-{args.nbeam}", 0
    w = workload_for(args.config)
    if args.mode == "beams" or args.nbeam:
        # the S-engine ships "8 beams from the generated 128-beam grid ... as 16-bit complex-valued words"
        w = w.sub(nbeam=args.nbeam or 8)
    if args.mode != "power":
        args.no_e2e = True
        args.no_cpu_baseline = True
    if args.scaling == "strong" and world > 1:
        from paper_1412_4907_b200 import shard
        c0, c1 = shard.channel_range(w.nchan, world, rank)   # channels are independent: no exchange
        w = w.sub(chan_idx=list(range(c0, c1)))
    else:
        w.seed = rank_seed(w.seed, rank)
    peaks = load_peaks()
    kern = {"auto": bf.BF_KERNEL_AUTO, "simt": bf.BF_KERNEL_SIMT, "umma": bf.BF_KERNEL_UMMA,
            "f16": bf.BF_KERNEL_UMMA_F16, "i8": bf.BF_KERNEL_UMMA_I8}[args.kernel]
    dt = {"ci8": bf.BF_CI8, "cf16": bf.BF_CF16, "ci4": bf.BF_CI4}[w.dtype]

    B = bf.Beamformer(w.nant, w.nchan, w.nbeam, w.nsamp, w.nint, dtype=dt, kernel=kern, device=dev)
    B.set_geometry(w.ant_xyz, w.freqs, w.beam_dir)
    v = synthetic.fill_voltages_torch(w, dev)
    P = B.empty_powers()
    stream = torch.cuda.current_stream(dev)
    run_step = lambda: B.run(v, P, stream)
    if args.mode == "beams":
        Y = torch.empty((w.nchan, w.nbeam, w.nsamp, 2), dtype=torch.float16, device=dev)
        run_step = lambda: B.run_beams(v, Y, 0.25, stream)
    elif args.mode == "incoherent":
        Pi = torch.empty((w.nchan, w.nbin), dtype=torch.float32, device=dev)
        run_step = lambda: B.run_incoherent(v, Pi, stream)

    def barrier():
        if dist:
            td.barrier()
        torch.cuda.synchronize(dev)

    # ---------------------------------------------------------------- device-resident timing
    for _ in range(W):
        run_step()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(K + 1)]
    l0 = B.launches
    barrier()
    ev[0].record(stream)
    for k in range(K):
        run_step()
        ev[k + 1].record(stream)
    barrier()
    launches = B.launches - l0
    clocks = sampler.stop() if rank == 0 else None
    total_ms = ev[0].elapsed_time(ev[K])
    per_launch_ms = [ev[k].elapsed_time(ev[k + 1]) for k in range(K)]
    flop_step = 8.0 * w.cmac if args.mode != "incoherent" else 4.0 * w.nchan * w.nsamp * w.nant  # |x|^2 + add
    total_ms_max, flop_all = aggregate(total_ms, flop_step * K, td if dist else None, dev)
    value = flop_all / (total_ms_max * 1e-3) / 1e12
    ms_per_step = total_ms_max / K
    avg_kernel_ms = statistics.mean(per_launch_ms)

    # roofline of the dominant (only) kernel: a dense contraction -> tensor bound; HBM-bound when
    # the algorithmic bytes at measured bandwidth take longer than the flops at measured tensor peak
    abytes = algorithmic_bytes(w)
    if args.mode == "beams":
        abytes = w.in_bytes + w.nchan * w.nbeam * w.nant * 4 + w.nchan * w.nbeam * w.nsamp * 4  # fp16 complex out
    elif args.mode == "incoherent":
        abytes = w.in_bytes + w.nchan * w.nbin * 4
    t_hbm = abytes / (peaks["hbm_gbs"] * 1e9)
    # which measured GEMM figure is the tensor roofline: the BURST one for a kernel timed alone in a short region at
    # full clocks, the SUSTAINED one once the timed region is long or the power cap was seen during it (the
    # cuBLAS loop behind the sustained figure runs power-capped at ~1.3 GHz; this kernel settles at ~1.4 GHz)
    capped = bool(clocks) and "sw_power_cap" in (clocks.get("reasons") or [])
    sustained = capped or total_ms >= 1000.0
    tpeak = peaks["tensor_tflops"] if sustained else peaks["tensor_tflops_burst"]
    tkind = ("sustained (power cap seen or timed region >= 1 s)" if sustained
             else f"burst (timed region {total_ms:.0f} ms at full clocks, no power cap seen)")
    t_tensor = flop_step / (tpeak * 1e12)
    traffic = None
    tpath = os.path.join(ROOT, "profiles", "traffic.json")
    if os.path.exists(tpath) and args.mode == "power":
        try:
            traffic = json.load(open(tpath)).get(w.name)
        except Exception:
            traffic = None
    if t_tensor >= t_hbm:
        ach = flop_step / (avg_kernel_ms * 1e-3) / 1e12
        roof = {"bound": "tensor", "achieved": ach, "peak": tpeak, "unit": "TFLOP/s",
                "frac": ach / tpeak, "traffic": traffic, "peak_kind": peaks["source"] + " bf16/fp16 dense GEMM, " + tkind,
                "frac_of_burst": ach / peaks["tensor_tflops_burst"], "frac_of_sustained": ach / peaks["tensor_tflops"],
                "kernel_ms": avg_kernel_ms}
    else:
        ach = abytes / (avg_kernel_ms * 1e-3) / 1e9
        roof = {"bound": "hbm", "achieved": ach, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                "frac": ach / peaks["hbm_gbs"], "traffic": traffic, "peak_kind": peaks["source"] + " copy bandwidth",
                "kernel_ms": avg_kernel_ms}

    # ---------------------------------------------------------------- end to end through the C ABI with HOST buffers
    e2e = None
    if not args.no_e2e:
        hv = torch.empty(v.shape, dtype=v.dtype, pin_memory=True)
        hv.copy_(v)
        hp = torch.empty(P.shape, dtype=torch.float32, pin_memory=True)
        cpc = args.chan_per_chunk or max(1, w.nchan // 8)
        cs, xs = torch.cuda.Stream(dev), torch.cuda.Stream(dev)
        del v
        torch.cuda.empty_cache()
        Ke = min(K, 10)
        if w.name == "streaming":
            # BASELINE.json config 5: continuous blocks from pinned host memory, H2D on a side stream
            # overlapped with compute (bf_run_streaming, double-buffered staging); 2 distinct blocks cycled
            hv2 = torch.empty(hv.shape, dtype=hv.dtype, pin_memory=True)
            hv2.copy_(torch.roll(hv, 1, dims=1))
            nblk = 8
            blocks = [hv if (i % 2 == 0) else hv2 for i in range(nblk)]
            Pb = torch.empty((nblk,) + tuple(P.shape), dtype=torch.float32, device=dev)
            run_e2e = lambda: B.run_streaming(blocks, Pb, cs, xs)
            steps_per_call, api = nblk, "bf_run_streaming (8 pinned host blocks per call, 2 streams, powers stay on device)"
            d2h = 0
        else:
            run_e2e = lambda: B.run_host(hv, hp, cpc, cs, xs)
            steps_per_call, api = 1, "bf_run_host (pinned host in/out, 2 streams)"
            d2h = int(w.out_bytes)
        for _ in range(2):
            run_e2e()
        cs.synchronize(); xs.synchronize()
        barrier()
        e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
        e0.record(cs)
        for _ in range(Ke):
            run_e2e()
        cs.wait_stream(xs)
        e1.record(cs)
        cs.synchronize(); xs.synchronize()
        barrier()
        Ke *= steps_per_call
        e2e_ms = e0.elapsed_time(e1)
        e2e_ms, e2e_flop = aggregate(e2e_ms, flop_step * Ke, td if dist else None, dev)
        e2e = {"value": e2e_flop / (e2e_ms * 1e-3) / 1e12, "unit": UNIT,
               "h2d_bytes_per_step": int(w.in_bytes), "d2h_bytes_per_step": d2h, "steps": Ke,
               "ms_per_step": e2e_ms / Ke, "h2d_gbs": w.in_bytes / (e2e_ms / Ke * 1e-3) / 1e9,
               "ant_samples_per_s": world * w.nchan * w.nsamp * w.nant * Ke / (e2e_ms * 1e-3),
               "chan_per_chunk": cpc, "api": api}
        sample_src = hv
    else:
        sample_src = v

    # ---------------------------------------------------------------- oracle on the host cores (rank 0, N=1)
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        def v_host(chans):
            return sample_src[chans].cpu().numpy() if sample_src.is_cuda else sample_src[chans].numpy()
        val, cores, desc, _, _ = time_oracle_sample(w, v_host)
        cpu = {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc}

    if rank == 0:
        line = {
            "metric": METRIC if args.mode == "power" else METRIC + " [side mode: %s]" % args.mode, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": args.scaling if world > 1 else "weak", "vs_baseline": None,
            "dtype": "i8->i32 (dp4a)" if args.mode == "incoherent" else {"umma-i8": "i8xi8->i32", "simt": "f32"}.get(B.kernel_name, "f16xf16->f32"),
            "data": "synthetic",
            "config": {"workload": w.name if args.mode == "power" else w.name + ":" + args.mode, "nant": w.nant, "nchan": w.nchan, "nbeam": w.nbeam, "nsamp": w.nsamp,
                       "nint": w.nint, "input": w.dtype, "l2": "input buffer (%.0f MB) >> L2 (126 MB), no flush needed" % (w.in_bytes / 1e6),
                       "kernel": B.kernel_name, "parallelism": (f"channel shards x{world}" if args.scaling == "strong" and world > 1 else f"replicas x{world}")},
            "ant_samples_per_s": world * w.nchan * w.nsamp * w.nant * K / (total_ms_max * 1e-3),
            "roofline": roof, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks,
            "context": {"paper_k20_tflops": 1.3, "note": "paper's number is a Tesla K20 with 4-bit input (PAPER.md:15): context, not a baseline for this config"},
        }
        print(json.dumps(line))
    B.close()
    if dist:
        td.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
