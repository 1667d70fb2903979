"""Channel sharding across ranks: host-side helpers only.

Frequency channels are independent -- each has its own weights and its own output slab -- so the hot path
shards over channels with NO data-path collective (the paper instead replicates the input on every GPU and
splits beams).  A rank beamforms channels [c0, c1) with the single-GPU library; the optional
``gather_powers`` hands the whole power cube to every rank (one consumer downstream) with one all_gather over
torch.distributed (NCCL over NVLink on GPUs, gloo on CPU).  No arithmetic of the method lives here.
"""
from __future__ import annotations


def channel_range(nchan: int, world: int, rank: int):
    """Contiguous, balanced slice [c0, c1) of the channels for `rank` of `world` (sizes differ by at most one)."""
    if nchan < 0 or world <= 0 or not (0 <= rank < world):
        raise ValueError("bad (nchan, world, rank)")
    base, extra = divmod(nchan, world)
    c0 = rank * base + min(rank, extra)
    return c0, c0 + base + (1 if rank < extra else 0)


def gather_powers(local, nchan: int, dist_mod=None):
    """All ranks contribute their [c1 - c0][nbeam][nbin] slab and receive the full [nchan][nbeam][nbin] cube.
    With one process (dist_mod None or world 1) this is the identity."""
    import torch

    if dist_mod is None or dist_mod.get_world_size() == 1:
        if local.shape[0] != nchan:
            raise ValueError("a single rank must hold every channel")
        return local
    world, rank = dist_mod.get_world_size(), dist_mod.get_rank()
    sizes = [channel_range(nchan, world, r) for r in range(world)]
    c0, c1 = sizes[rank]
    if local.shape[0] != c1 - c0:
        raise ValueError(f"rank {rank} must hold channels [{c0}, {c1})")
    most = max(b - a for a, b in sizes)
    pad = torch.zeros((most,) + tuple(local.shape[1:]), dtype=local.dtype, device=local.device)
    pad[: c1 - c0] = local
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist_mod.all_gather(parts, pad)
    return torch.cat([parts[r][: b - a] for r, (a, b) in enumerate(sizes)], dim=0)
