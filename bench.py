#!/usr/bin/env python
"""bench.py -- headline benchmark of the B200 coherent beamformer (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config medium] [--impl ours|reference]

One "step" is one pass of the whole hot path (ingest -> contraction -> |.|^2 -> integrate) over one
synthetic `medium` buffer (BASELINE.json configs[1]: 32 antennas, 1024 channels, 128 beams, 32768
samples, complex int8, nint 64).  Prints ONE JSON line (rank 0).  Metric: beamforming TFLOP/s at
8 flop per complex MAC.

The default run (N = 1, --config medium) also times every other BASELINE.json configuration (tiny, the six
beam-count sweep points, large-N, streaming) with the same procedure and reports them under "configs", and
compares the GPU powers of ALL channels of the headline buffer with the oracle ("max_err").

--gpus N > 1 without a torchrun environment starts N ranks itself (torch.distributed.run, one per GPU);
each rank beamforms its own replica (channels are independent, so the path shards with no exchange; "weak"
scaling), or with --scaling strong a contiguous range of ONE workload's channels; NCCL is used only for the
barrier and the two timing all-reduces.

--impl reference times the fp64 CPU oracle (oracle/) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import socket
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "beamforming TFLOP/s (8 flop/complex MAC)"
UNIT = "TFLOP/s"
L2_BYTES = 126e6
ALL_CONFIGS = ["tiny", "sweep-1", "sweep-4", "sweep-16", "sweep-64", "sweep-256", "sweep-1024", "large-N", "streaming"]
EXTRA_CONFIGS = ["sweep-32"]   # not a BASELINE.json point: the top of the int8-operand kernel's range
F1_CONFIGS = ["medium-ci4", "sweep-ci4-1", "sweep-ci4-16", "sweep-ci4-64", "streaming-ci4"]   # the paper's 4+4-bit input


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
    if name.startswith("sweep-ci4-"):
        return synthetic.make_workload("sweep-ci4", nbeam=int(name.split("-")[2]))
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


# ------------------------------------------------------------------------------------------ multi-rank launcher
def free_port() -> int:
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def launcher_command(ngpus: int, argv, port=None):
    """The torchrun command `bench.py --gpus N` re-executes itself under when no rank environment is set."""
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={ngpus}",
            "--master-addr", "127.0.0.1", "--master-port", str(port or free_port()), os.path.abspath(__file__)] + list(argv)


def maybe_spawn(args, argv):
    """--gpus N > 1 and no WORLD_SIZE: start the N ranks here and pass their output through."""
    if args.gpus <= 1 or "WORLD_SIZE" in os.environ:
        return None
    return subprocess.call(launcher_command(args.gpus, argv))


def launcher_selftest(args) -> int:
    """CPU check of the multi-rank plumbing (tests/test_multirank_cpu.py): every rank joins a gloo group,
    'processes' (rank + 1) units in (rank + 1) ms, and rank 0 prints the aggregate -- the code path of the real
    bench (environment, barrier, MAX / SUM all-reduces, one JSON line) without a GPU."""
    import torch.distributed as td
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    if world > 1:
        td.init_process_group("gloo")
        td.barrier()
    ms, units = aggregate(float(rank + 1), float(rank + 1), td if world > 1 else None, "cpu")
    if rank == 0:
        print(json.dumps({"selftest": "launcher", "n_gpus": world, "requested_gpus": args.gpus, "max_ms": ms, "units": units,
                          "value": units / ms}))
    if world > 1:
        td.destroy_process_group()
    return 0


# ------------------------------------------------------------------------------------------ clocks
class ClockSampler:
    """SM clock, power and throttle reasons sampled DURING the timed region: NVML in a thread of this
    process (one sample every ~1 ms), nvidia-smi as the fallback."""
    REASONS = {"hw_slowdown": 0x8, "hw_thermal_slowdown": 0x40, "sw_thermal_slowdown": 0x20, "sw_power_cap": 0x4}

    def __init__(self, index=0, period_s=0.001):
        self.index, self.period = index, period_s
        self.samples, self.reasons, self.power = [], set(), []
        self.max_mhz = None
        self._stop = threading.Event()
        self._thread = None
        self._smi = None
        self.source = None

    def _loop(self, nv, h):
        while not self._stop.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM))
                self.power.append(nv.nvmlDeviceGetPowerUsage(h) / 1000.0)
                mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                for nm, bit in self.REASONS.items():
                    if mask & bit:
                        self.reasons.add(nm)
            except Exception:
                pass
            time.sleep(self.period)

    def start(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            idx = self.index
            vis = os.environ.get("CUDA_VISIBLE_DEVICES")
            if vis:
                try:
                    idx = int(vis.split(",")[self.index])
                except Exception:
                    pass
            h = nv.nvmlDeviceGetHandleByIndex(idx)
            self.max_mhz = float(nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM))
            self._thread = threading.Thread(target=self._loop, args=(nv, h), daemon=True)
            self._thread.start()
            self.source = "nvml"
            return
        except Exception:
            self._thread = None
        try:
            q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
                 "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
            self._smi = subprocess.Popen(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader,nounits", "-i", str(self.index),
                                          "-lms", "20"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.source = "nvidia-smi"
        except Exception:
            self._smi = None

    def stop(self):
        out = {"sm_mhz": None, "sm_min_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "samples": 0, "power_w_max": None,
               "source": self.source}
        if self._thread is not None:
            self._stop.set()
            self._thread.join(timeout=2)
        elif self._smi is not None:
            time.sleep(0.05)
            self._smi.terminate()
            try:
                text, _ = self._smi.communicate(timeout=5)
            except Exception:
                self._smi.kill()
                text = ""
            names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
            for ln in text.splitlines():
                f = [x.strip() for x in ln.split(",")]
                if len(f) < 7:
                    continue
                try:
                    self.samples.append(float(f[0]))
                    self.max_mhz = float(f[1])
                    self.power.append(float(f[2]))
                except ValueError:
                    continue
                for nm, val in zip(names, f[3:7]):
                    if val.lower().startswith("active"):
                        self.reasons.add(nm)
            out["sm_max_mhz"] = self.max_mhz
        if self.samples:
            out.update(sm_mhz=statistics.median(self.samples), sm_min_mhz=min(self.samples), samples=len(self.samples))
        if self.power:
            out["power_w_max"] = max(self.power)
        out["reasons"] = sorted(self.reasons)
        return out


# ------------------------------------------------------------------------------------------ oracle legs
def time_oracle_sample(w, v_host_fn, target_s=15.0, max_chan=1 << 30):
    """The oracle as it stands on the host cores, on whole channels of the workload; returns
    (TFLOP/s, cores, description, seconds, channels, powers of those channels).  v_host_fn(chan_list) -> numpy voltages."""
    import oracle
    cores = oracle.num_threads()
    # calibrate on `cores` channels (one per thread), then size the sample for ~target_s
    n0 = min(w.nchan, cores)
    chans = list(range(n0))
    ws = w.sub(chan_idx=chans)
    v = v_host_fn(chans)
    t0 = time.perf_counter()
    ref = oracle.beamform(ws.ant_xyz, ws.freqs, ws.beam_dir, v, ws.nint)
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
        ref = oracle.beamform(ws.ant_xyz, ws.freqs, ws.beam_dir, v, ws.nint)
        dt = time.perf_counter() - t0
    else:
        n, dt = n0, dt0
    flop = 8.0 * n * w.nbeam * w.nant * w.nsamp
    return flop / dt / 1e12, cores, f"{n} of {w.nchan} channels x all {w.nbeam} beams x all {w.nsamp} samples, {dt:.2f} s", dt, n, ref


def row_error(P_gpu, P_ref):
    """north_star's bar: worst over (chan, beam) rows of max_j |P_gpu - P_ref| / mean_j P_ref."""
    import numpy as np
    P_gpu = np.asarray(P_gpu, dtype=np.float64)
    err = np.abs(P_gpu - P_ref).max(axis=-1)
    return float((err / np.maximum(P_ref.mean(axis=-1), 1e-300)).max())


def run_reference(args):
    """--impl reference: the fp64 oracle on the host cores, each step a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
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


# ------------------------------------------------------------------------------------------ one configuration on the device
class Timed:
    """One workload resident on the device, timed with CUDA events on the launching stream."""

    def __init__(self, bf, synthetic, torch, w, dev, kernel, mode="power"):
        self.bf, self.torch, self.w, self.dev, self.mode = bf, torch, w, dev, mode
        dt = {"ci8": bf.BF_CI8, "cf16": bf.BF_CF16, "ci4": bf.BF_CI4}[w.dtype]
        self.B = bf.Beamformer(w.nant, w.nchan, w.nbeam, w.nsamp, w.nint, dtype=dt, kernel=kernel, device=dev)
        self.B.set_geometry(w.ant_xyz, w.freqs, w.beam_dir)
        v = synthetic.fill_voltages_torch(w, dev)
        # inputs smaller than twice the L2 are rotated through enough copies that no launch finds its input cached
        self.ncopy = 1 if w.in_bytes >= 2 * L2_BYTES else int(math.ceil(2 * L2_BYTES / w.in_bytes)) + 1
        self.v = [v] + [v.clone() for _ in range(self.ncopy - 1)]
        self.l2 = ("input buffer (%.0f MB) > 2 x L2 (126 MB): no flush needed" % (w.in_bytes / 1e6) if self.ncopy == 1 else
                   "input (%.1f MB) fits L2: %d copies rotated (%.0f MB > 2 x L2) so every launch reads HBM" %
                   (w.in_bytes / 1e6, self.ncopy, self.ncopy * w.in_bytes / 1e6))
        self.P = self.B.empty_powers()
        self.stream = torch.cuda.current_stream(dev)
        self.probe = torch.zeros(4, dtype=torch.int64, device=dev)
        self.B.set_clock_probe(self.probe)
        self.k = 0
        if mode == "beams":
            self.Y = torch.empty((w.nchan, w.nbeam, w.nsamp, 2), dtype=torch.float16, device=dev)
        elif mode == "incoherent":
            self.Pi = torch.empty((w.nchan, w.nbin), dtype=torch.float32, device=dev)

    def step(self):
        v = self.v[self.k % self.ncopy]
        self.k += 1
        if self.mode == "beams":
            self.B.run_beams(v, self.Y, 0.25, self.stream)
        elif self.mode == "incoherent":
            self.B.run_incoherent(v, self.Pi, self.stream)
        else:
            self.B.run(v, self.P, self.stream)

    def graph_replay_ms(self, replays=20):
        """The short-launch regime (hard part 8): n consecutive bf_run calls, each on another copy of the
        input, captured into ONE CUDA graph and replayed; returns ms per call.  Against the plain back-to-back figure
        this separates what the kernel costs from what launching it costs."""
        torch = self.torch
        n = max(self.ncopy, 16)
        g, s = torch.cuda.CUDAGraph(), torch.cuda.Stream(self.dev)
        torch.cuda.synchronize(self.dev)
        with torch.cuda.graph(g, stream=s):
            cur = torch.cuda.current_stream(self.dev)
            for k in range(n):
                self.B.run(self.v[k % self.ncopy], self.P, cur)
        for _ in range(3):
            g.replay()
        torch.cuda.synchronize(self.dev)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(replays):
            g.replay()
        e1.record()
        torch.cuda.synchronize(self.dev)
        return e0.elapsed_time(e1) / (replays * n), n

    def flop_step(self):
        w = self.w
        return 8.0 * w.cmac if self.mode != "incoherent" else 4.0 * w.nchan * w.nsamp * w.nant  # |x|^2 + add

    def abytes(self):
        w = self.w
        if self.mode == "beams":
            return w.in_bytes + w.nchan * w.nbeam * w.nant * 4 + w.nchan * w.nbeam * w.nsamp * 4  # fp16 complex out
        if self.mode == "incoherent":
            return w.in_bytes + w.nchan * w.nbin * 4
        return algorithmic_bytes(w)

    def measure(self, K, W, barrier, sample_clocks=True, rank=0):
        torch = self.torch
        for _ in range(W):
            self.step()
        barrier()
        sampler = ClockSampler(self.dev.index or 0)
        if sample_clocks and rank == 0:
            sampler.start()
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(K + 1)]
        l0 = self.B.launches
        barrier()
        ev[0].record(self.stream)
        for k in range(K):
            self.step()
            ev[k + 1].record(self.stream)
        barrier()
        launches = self.B.launches - l0
        clocks = sampler.stop() if (sample_clocks and rank == 0) else None
        total_ms = ev[0].elapsed_time(ev[K])
        per = [ev[k].elapsed_time(ev[k + 1]) for k in range(K)]
        pr = [int(x) for x in self.probe.cpu().tolist()]
        if clocks is not None and pr[3] > pr[1]:
            # the SM clock the LAST timed launch really ran at, from the kernel's own counters (bf_set_clock_probe)
            clocks["kernel_sm_mhz"] = (pr[2] - pr[0]) / (pr[3] - pr[1]) * 1e3
            clocks["kernel_cta0_ms"] = (pr[3] - pr[1]) * 1e-6
        return total_ms, per, launches, clocks

    def roofline(self, kernel_ms, total_ms, clocks, peaks, traffic):
        """Roofline of the dominant (only) kernel: a dense contraction -> tensor bound; HBM-bound when the
        algorithmic bytes at measured bandwidth take longer than the flops at the measured tensor peak."""
        flop, ab = self.flop_step(), self.abytes()
        t_hbm = ab / (peaks["hbm_gbs"] * 1e9)
        # ONE tensor peak for `frac` in every row: the measured BURST GEMM figure (MEASURED_PEAKS.json).  The sustained figure
        # is printed beside it as frac_of_sustained.  (Choosing the peak from NVML's throttle reasons mixed two denominators in
        # one table and published fractions above 1: NVML does not see the clock a millisecond kernel really ran at -- the
        # kernel's own probe, clocks.kernel_sm_mhz, does.)
        tpeak = peaks["tensor_tflops_burst"]
        tkind = f"burst (one peak for every row; timed region {total_ms:.0f} ms)"
        t_tensor = flop / (peaks["tensor_tflops_burst"] * 1e12)
        if t_tensor >= t_hbm:
            ach = flop / (kernel_ms * 1e-3) / 1e12
            return {"bound": "tensor", "achieved": ach, "peak": tpeak, "unit": "TFLOP/s", "frac": ach / tpeak, "traffic": traffic,
                    "traffic_source": TRAFFIC_SOURCE if traffic is not None else None, "frac_above_peak": bool(ach > tpeak),
                    "peak_kind": peaks["source"] + " bf16/fp16 dense GEMM, " + tkind,
                    "frac_of_burst": ach / peaks["tensor_tflops_burst"], "frac_of_sustained": ach / peaks["tensor_tflops"],
                    "kernel_ms": kernel_ms, "algorithmic_flop": flop, "algorithmic_bytes": ab}
        ach = ab / (kernel_ms * 1e-3) / 1e9
        return {"bound": "hbm", "achieved": ach, "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": ach / peaks["hbm_gbs"],
                "traffic": traffic, "traffic_source": TRAFFIC_SOURCE if traffic is not None else None,
                "frac_above_peak": bool(ach > peaks["hbm_gbs"]),
                "peak_kind": peaks["source"] + " copy bandwidth", "kernel_ms": kernel_ms,
                "algorithmic_flop": flop, "algorithmic_bytes": ab}

    def close(self):
        self.B.close()
        self.v = None


# `traffic` is NOT measured in the bench run: it is the dram__bytes_read.sum + dram__bytes_write.sum of one committed
# `ncu --set full` capture of the same kernel and workload
TRAFFIC_SOURCE = "profiles/traffic.json (ncu --set full capture, per launch; not measured in this run)"


def streaming_e2e_row(bf, synthetic, torch, dev, barrier, kernel_ms):
    """BASELINE.json config 5's own end-to-end leg: "continuous blocks ... from pinned host memory with H2D copies overlapped
    on a side stream ... reports end-to-end sustained samples/s vs input data rate".  8 pinned host blocks per
    bf_run_streaming call (two distinct ones cycled), double-buffered staging, powers stay on the device; what the input
    link delivers (H2D GB/s) is the input data rate D = C*T*A*W of PAPER.md:176 that the GPU can be fed with."""
    w = workload_for("streaming")
    T = Timed(bf, synthetic, torch, w, dev, bf.BF_KERNEL_AUTO)
    v = T.v[0]
    hv = torch.empty(v.shape, dtype=v.dtype, pin_memory=True)
    hv.copy_(v)
    hv2 = torch.empty(v.shape, dtype=v.dtype, pin_memory=True)
    hv2.copy_(torch.roll(v, 1, dims=1))
    nblk, calls = 8, 3
    blocks = [hv if (i % 2 == 0) else hv2 for i in range(nblk)]
    Pb = torch.empty((nblk,) + tuple(T.P.shape), dtype=torch.float32, device=dev)
    cs, xs = torch.cuda.Stream(dev), torch.cuda.Stream(dev)
    T.B.run_streaming(blocks, Pb, cs, xs)
    cs.synchronize(); xs.synchronize()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(cs)
    for _ in range(calls):
        T.B.run_streaming(blocks, Pb, cs, xs)
    cs.wait_stream(xs)
    e1.record(cs)
    cs.synchronize(); xs.synchronize()
    ms = e0.elapsed_time(e1) / (calls * nblk)
    row = {"ms": ms, "bound": "pcie", "frac": None, "unit": "GB/s", "achieved": w.in_bytes / (ms * 1e-3) / 1e9,
           "h2d_gbs": w.in_bytes / (ms * 1e-3) / 1e9, "ant_samples_per_s": w.nchan * w.nsamp * w.nant / (ms * 1e-3),
           "tflops": T.flop_step() / (ms * 1e-3) / 1e12, "kernel_ms_per_block": kernel_ms,
           "kernel_share_of_block_time": kernel_ms / ms, "steps": calls * nblk, "traffic": None, "kernel": T.B.kernel_name,
           "api": "bf_run_streaming (8 pinned host blocks per call, 2 streams, double-buffered staging, powers stay on device)",
           "note": "frac is null: the bound is the host link, for which MEASURED_PEAKS.json has no figure; the kernel needs "
                   "kernel_share_of_block_time of each block's transfer time"}
    T.close()
    return row


def load_traffic(name):
    tpath = os.path.join(ROOT, "profiles", "traffic.json")
    try:
        return json.load(open(tpath)).get(name)
    except Exception:
        return None


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
    ap.add_argument("--no-configs", action="store_true", help="skip the table of the other BASELINE.json configurations")
    ap.add_argument("--chan-per-chunk", type=int, default=0, help="e2e: channels per H2D chunk (0 = nchan/8)")
    ap.add_argument("--selftest-launcher", action="store_true", help="CPU check of the --gpus N launcher (no GPU work)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    rc = maybe_spawn(args, sys.argv[1:])
    if rc is not None:
        return rc
    if args.selftest_launcher:
        return launcher_selftest(args)

    import numpy as np  # noqa: F401
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
    if local >= torch.cuda.device_count():
        raise SystemExit(f"rank {rank}: local rank {local} has no GPU ({torch.cuda.device_count()} visible)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    td = None
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

    def barrier():
        if dist:
            td.barrier()
        torch.cuda.synchronize(dev)

    # ---------------------------------------------------------------- device-resident timing (headline)
    T = Timed(bf, synthetic, torch, w, dev, kern, args.mode)
    B = T.B
    total_ms, per_launch_ms, launches, clocks = T.measure(K, W, barrier, rank=rank)
    flop_step = T.flop_step()
    total_ms_max, flop_all = aggregate(total_ms, flop_step * K, td, dev)
    value = flop_all / (total_ms_max * 1e-3) / 1e12
    ms_per_step = total_ms_max / K
    avg_kernel_ms = statistics.mean(per_launch_ms)
    roof = T.roofline(avg_kernel_ms, total_ms, clocks, peaks, load_traffic(w.name) if args.mode == "power" else None)
    kernel_name, l2_note = B.kernel_name, T.l2
    v, P = T.v[0], T.P

    # ---------------------------------------------------------------- end to end through the C ABI with HOST buffers
    e2e = None
    if not args.no_e2e:
        hv = torch.empty(v.shape, dtype=v.dtype, pin_memory=True)
        hv.copy_(v)
        hp = torch.empty(P.shape, dtype=torch.float32, pin_memory=True)
        cpc = args.chan_per_chunk or max(1, w.nchan // 8)
        cs, xs = torch.cuda.Stream(dev), torch.cuda.Stream(dev)
        P_dev = P.clone()   # the device-resident result, kept for the whole-buffer parity figure below
        T.v = None
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
        e2e_ms, e2e_flop = aggregate(e2e_ms, flop_step * Ke, td, dev)
        e2e = {"value": e2e_flop / (e2e_ms * 1e-3) / 1e12, "unit": UNIT,
               "h2d_bytes_per_step": int(w.in_bytes), "d2h_bytes_per_step": d2h, "steps": Ke,
               "ms_per_step": e2e_ms / Ke, "h2d_gbs": w.in_bytes / (e2e_ms / Ke * 1e-3) / 1e9,
               "ant_samples_per_s": world * w.nchan * w.nsamp * w.nant * Ke / (e2e_ms * 1e-3),
               "chan_per_chunk": cpc, "api": api}
        sample_src = hv
    else:
        sample_src = v
        P_dev = P

    # ---------------------------------------------------------------- oracle on the host cores (rank 0, N=1)
    cpu, max_err = None, None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        def v_host(chans):
            return sample_src[chans].cpu().numpy() if sample_src.is_cuda else sample_src[chans].numpy()
        val, cores, desc, _, nref, ref = time_oracle_sample(w, v_host)
        cpu = {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc}
        # whole-buffer parity of the very launch configuration that was timed: every channel the oracle computed
        # (outside the timed region) against the device-resident powers
        max_err = {"value": row_error(P_dev[:nref].cpu().numpy(), ref), "bar": 1e-3, "channels": nref, "of": w.nchan,
                   "definition": "max over (chan, beam) rows of max_j |P_gpu - P_ref| / mean_j P_ref"}
        del ref
    T.close()
    v = None
    del T, P, P_dev, sample_src, v
    torch.cuda.empty_cache()

    # ---------------------------------------------------------------- the other BASELINE.json configurations
    configs = None
    if rank == 0 and world == 1 and args.config == "medium" and args.mode == "power" and not args.no_configs and not args.nbeam:
        configs = {"medium": {"ms": avg_kernel_ms, "bound": roof["bound"], "frac": roof["frac"],
                              "frac_of_burst": roof.get("frac_of_burst"), "frac_of_sustained": roof.get("frac_of_sustained"),
                              "achieved": roof["achieved"], "unit": roof["unit"], "traffic": roof["traffic"], "kernel": kernel_name,
                              "tflops": flop_step / (avg_kernel_ms * 1e-3) / 1e12, "steps": K, "clocks": clocks, "l2": l2_note}}
        # The HBM-bound rows are timed first: they are clock-sensitive (issue-bound at 1.9 GHz), and once the tensor-bound
        # configurations have run back to back the power governor keeps the SM clock near 1.5 GHz for a while (measured:
        # sweep-32 0.109 ms at 1.87 GHz, 0.133 ms at 1.48 GHz right after `streaming`).  Every row carries its own `clocks`.
        table = ALL_CONFIGS + EXTRA_CONFIGS + F1_CONFIGS
        few = [n for n in table if n == "tiny" or (n.startswith("sweep-") and int(n.split("-")[-1]) <= 32)]
        table = few + [n for n in table if n not in few]
        for name in table:
            wc = workload_for(name)
            Tc = Timed(bf, synthetic, torch, wc, dev, bf.BF_KERNEL_AUTO)
            Kc = 200 if name == "tiny" else 30
            tot, per, _, clk = Tc.measure(Kc, 5, barrier)
            ms = statistics.mean(per)
            r = Tc.roofline(ms, tot, clk, peaks, load_traffic(wc.name))
            configs[wc.name] = {
                "ms": ms, "bound": r["bound"], "frac": r["frac"], "frac_of_burst": r.get("frac_of_burst"),
                "frac_of_sustained": r.get("frac_of_sustained"), "achieved": r["achieved"], "unit": r["unit"],
                "traffic": r["traffic"], "kernel": Tc.B.kernel_name, "tflops": Tc.flop_step() / (ms * 1e-3) / 1e12,
                "steps": Kc, "clocks": clk, "l2": Tc.l2}
            if name == "tiny":
                # the same launches out of a CUDA graph: per-call time without the host's launch cost
                gms, gn = Tc.graph_replay_ms()
                rg = Tc.roofline(gms, gms * gn * 20, clk, peaks, None)
                configs["tiny:graph"] = dict(configs[wc.name], ms=gms, frac=rg["frac"], achieved=rg["achieved"], traffic=None,
                                             tflops=Tc.flop_step() / (gms * 1e-3) / 1e12, steps=gn * 20,
                                             note="%d bf_run calls captured in one CUDA graph, 20 replays" % gn)
            Tc.close()
            del Tc
            torch.cuda.empty_cache()
        if "streaming" in configs:
            try:
                configs["streaming:e2e"] = streaming_e2e_row(bf, synthetic, torch, dev, barrier, configs["streaming"]["ms"])
            except Exception as exc:  # a leg that cannot run (no pinned memory left) must not cost the whole line
                configs["streaming:e2e"] = {"error": repr(exc)[:200]}
            torch.cuda.empty_cache()
        # side modes on medium's input: voltage beams (the S-engine ships 8 of the beams as 16-bit
        # complex words; 32 and 128 show the output-bound regime) and the incoherent beam
        for label, mode, nb in (("medium:beams-8", "beams", 8), ("medium:beams-32", "beams", 32), ("medium:beams-128", "beams", 128),
                                ("medium:incoherent", "incoherent", 0)):
            wc = workload_for("medium")
            if nb:
                wc = wc.sub(nbeam=nb)
            Tc = Timed(bf, synthetic, torch, wc, dev, bf.BF_KERNEL_AUTO, mode)
            tot, per, _, clk = Tc.measure(20, 3, barrier)
            ms = statistics.mean(per)
            r = Tc.roofline(ms, tot, clk, peaks, None)
            configs[label] = {"ms": ms, "bound": r["bound"], "frac": r["frac"], "frac_of_burst": r.get("frac_of_burst"),
                              "frac_of_sustained": r.get("frac_of_sustained"), "achieved": r["achieved"], "unit": r["unit"],
                              "traffic": None, "kernel": Tc.B.kernel_name if mode == "beams" else "incoherent-dp4a",
                              "tflops": Tc.flop_step() / (ms * 1e-3) / 1e12, "steps": 20, "clocks": clk, "l2": Tc.l2}
            Tc.close()
            del Tc
            torch.cuda.empty_cache()

    if rank == 0:
        line = {
            "metric": METRIC if args.mode == "power" else METRIC + " [side mode: %s]" % args.mode, "value": value, "unit": UNIT,
            "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": args.scaling if world > 1 else "weak", "vs_baseline": None,
            "dtype": "i8->i32 (dp4a)" if args.mode == "incoherent" else {"umma-i8": "i8xi8->i32", "simt": "f32"}.get(kernel_name, "f16xf16->f32"),
            "data": "synthetic",
            "config": {"workload": w.name if args.mode == "power" else w.name + ":" + args.mode, "nant": w.nant, "nchan": w.nchan,
                       "nbeam": w.nbeam, "nsamp": w.nsamp, "nint": w.nint, "input": w.dtype, "l2": l2_note, "kernel": kernel_name,
                       "parallelism": (f"channel shards x{world}" if args.scaling == "strong" and world > 1 else f"replicas x{world}")},
            "ant_samples_per_s": world * w.nchan * w.nsamp * w.nant * K / (total_ms_max * 1e-3),
            "roofline": roof, "cpu_baseline": cpu, "max_err": max_err, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks,
            "configs": configs,
            "context": {"paper_k20_tflops": 1.3, "note": "paper's number is a Tesla K20 with 4-bit input (PAPER.md:15): context, not a baseline for this config"},
        }
        if configs:
            # compact copy of the table as the LAST key, so that it survives a reader that keeps only the tail of the line:
            # name -> [ms per launch, frac of roofline (tensor rows: burst GEMM peak; hbm rows: copy bandwidth), "t" | "h",
            # SM MHz from the kernel's own clock probe]
            line["summary"] = {n: [round(c["ms"], 5), None if c["frac"] is None else round(c["frac"], 4), c["bound"][0],
                                   round((c.get("clocks") or {}).get("kernel_sm_mhz") or 0)]
                               for n, c in configs.items() if "ms" in c}
        print(json.dumps(line))
    if dist:
        td.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
