"""Multi-GPU host logic: the path shards with NO data-path collective.

Time sharding: rank r owns output samples [o0, o1) of every DM trial and needs input samples
[o0, o1 + max_shift) of every channel (a max_shift halo; no add is repeated).  DM sharding: rank
r owns a contiguous slice of dm_list and needs the whole input.  Only timing and reporting use
a collective (max / sum over ranks).  No method arithmetic lives here.
"""
from __future__ import annotations

from dataclasses import dataclass


@dataclass(frozen=True)
class TimeShard:
    rank: int
    out_start: int   # first output sample this rank produces
    out_stop: int    # one past the last
    in_start: int    # first input sample it needs
    in_stop: int     # one past the last: out_stop + max_shift

    @property
    def out_len(self) -> int:
        return self.out_stop - self.out_start

    @property
    def nsamps(self) -> int:
        return self.in_stop - self.in_start


def time_shards(nsamps: int, max_shift: int, world: int) -> list[TimeShard]:
    """Split out_len = nsamps - max_shift output samples into `world` contiguous shards whose
    lengths differ by at most one.  Ranks beyond out_len get empty shards."""
    if world <= 0:
        raise ValueError("world must be positive")
    out_len = nsamps - max_shift
    if out_len <= 0:
        raise ValueError("max_shift must be smaller than nsamps")
    base, rem = divmod(out_len, world)
    shards, o0 = [], 0
    for r in range(world):
        n = base + (1 if r < rem else 0)
        o1 = o0 + n
        shards.append(TimeShard(r, o0, o1, o0, (o1 + max_shift) if n else o0))
        o0 = o1
    return shards


def dm_shards(ndm: int, world: int) -> list[tuple[int, int]]:
    """Contiguous [start, stop) slices of the DM list, lengths differing by at most one."""
    if world <= 0:
        raise ValueError("world must be positive")
    base, rem = divmod(ndm, world)
    out, d0 = [], 0
    for r in range(world):
        n = base + (1 if r < rem else 0)
        out.append((d0, d0 + n))
        d0 += n
    return out


def job_throughput(units_this_rank: float, ms_this_rank: float, dist=None, device=None):
    """Whole-job units/s = sum over ranks of units / max over ranks of time (bench.py contract).
    `dist` is torch.distributed (already initialised) or None for a single process."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return units_this_rank / (ms_this_rank * 1e-3), ms_this_rank
    import torch
    t = torch.tensor([ms_this_rank], dtype=torch.float64, device=device)
    u = torch.tensor([units_this_rank], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(u.item()) / (float(t.item()) * 1e-3), float(t.item())
