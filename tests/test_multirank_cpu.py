"""N > 1 host logic on CPU: two gloo ranks.  The path shards with NO data-path collective (channels
and replicas are independent); what the ranks share is the barrier + max-over-ranks timing
and the sum of the units they processed (bench.py aggregate), and each rank draws its own buffer."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    import oracle
    import synthetic
    # each rank: its own seeded buffer, its own (oracle-computed) slab -- no exchange of data
    w = synthetic.make_workload("tiny").sub(nchan=2, nsamp=64)
    w.seed = bench.rank_seed(w.seed, rank)
    v = w.make_voltages()
    P = oracle.beamform(w.ant_xyz, w.freqs, w.beam_dir, v, w.nint)
    local_ms = 10.0 + 5.0 * rank          # pretend timings: rank 1 is the slow one
    units = float(w.cmac) * 8
    dist.barrier()
    t_max, u_sum = bench.aggregate(local_ms, units, dist, torch.device("cpu"))
    # channel sharding of ONE workload (strong scaling): rank r holds channels [c0, c1) and the gather
    # rebuilds the cube every rank would have computed alone
    from paper_1412_4907_b200 import shard
    wf = synthetic.make_workload("tiny").sub(nchan=5, nsamp=64)      # 5 channels over 2 ranks: 3 + 2
    c0, c1 = shard.channel_range(wf.nchan, world, rank)
    ws = wf.sub(chan_idx=list(range(c0, c1)))
    Ps = oracle.beamform(ws.ant_xyz, ws.freqs, ws.beam_dir, wf.make_voltages()[c0:c1], ws.nint)
    full = shard.gather_powers(torch.from_numpy(Ps), wf.nchan, dist).numpy()
    ref = oracle.beamform(wf.ant_xyz, wf.freqs, wf.beam_dir, wf.make_voltages(), wf.nint)
    out[rank] = (t_max, u_sum, float(P.sum()), int(v.astype(np.int64).sum()), (c0, c1), bool(np.array_equal(full, ref)))
    dist.destroy_process_group()


def test_two_ranks_aggregate_and_shard():
    world = 2
    mgr = mp.Manager()
    out = mgr.dict()
    mp.spawn(_worker, args=(world, _free_port(), out), nprocs=world, join=True)
    assert set(out.keys()) == {0, 1}
    (t0, u0, p0, s0, r0, ok0), (t1, u1, p1, s1, r1, ok1) = out[0], out[1]
    assert r0 == (0, 3) and r1 == (3, 5) and ok0 and ok1   # channel shards tile the cube, gather is exact
    assert t0 == t1 == 15.0                       # max over ranks
    assert u0 == u1 and u0 == 2 * 8 * 2 * 16 * 32 * 64  # sum over ranks of 8*C*B*N*T
    assert s0 != s1 and p0 != p1                  # the replicas really beamformed different buffers


def test_channel_range_properties():
    from paper_1412_4907_b200 import shard
    for nchan in (0, 1, 5, 64, 1023):
        for world in (1, 2, 3, 8):
            r = [shard.channel_range(nchan, world, k) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == nchan
            assert all(r[k][1] == r[k + 1][0] for k in range(world - 1))
            sizes = [b - a for a, b in r]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard.channel_range(4, 2, 2)
    t = torch.arange(24.0).reshape(2, 3, 4)
    assert shard.gather_powers(t, 2) is t


def test_single_process_aggregate_is_identity():
    import bench
    assert bench.aggregate(3.5, 7.0) == (3.5, 7.0)
    assert bench.rank_seed(1, 0) == 1 and bench.rank_seed(1, 3) == 301


def test_bench_gpus_flag_starts_the_ranks_itself():
    """`python bench.py --gpus 2` with no torchrun environment must start two ranks:
    the launcher path is driven end to end with gloo ranks that do no GPU work (--selftest-launcher)."""
    import json
    import subprocess
    env = {k: v for k, v in os.environ.items() if k not in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--gpus", "2", "--selftest-launcher"],
                       capture_output=True, text=True, timeout=300, env=env)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [json.loads(ln) for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1                          # rank 0 alone prints
    d = lines[0]
    assert d["n_gpus"] == 2 and d["requested_gpus"] == 2
    assert d["max_ms"] == 2.0 and d["units"] == 3.0  # max over ranks of (rank + 1) ms, sum of (rank + 1) units


def test_launcher_command_shape():
    import bench
    cmd = bench.launcher_command(4, ["--gpus", "4", "--steps", "2"], port=29999)
    assert cmd[1:3] == ["-m", "torch.distributed.run"] and "--nproc-per-node=4" in cmd
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1" and cmd[cmd.index("--master-port") + 1] == "29999"
    assert cmd[-4:] == ["--gpus", "4", "--steps", "2"] and cmd[-5].endswith("bench.py")
