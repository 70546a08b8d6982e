"""theta-sharding over ranks: host logic only, no arithmetic of the method.

log L(theta) of one hyper-parameter point needs nothing from any other point, so N GPUs split a batch of
theta and replicate the catalogue; there is no collective on the data path.  The only communication is
the gather of the `[n_theta]` results and the max-over-ranks of a device time, both through
`torch.distributed` (NCCL on GPUs; the CPU tests use gloo).
"""
from __future__ import annotations

from typing import Optional, Tuple

import torch
import torch.distributed as dist


def theta_range(n_theta: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous, balanced [lo, hi) of the theta batch owned by `rank` (sizes differ by at most one)."""
    if world < 1 or not (0 <= rank < world) or n_theta < 0:
        raise ValueError("bad rank/world/n_theta")
    base, extra = divmod(n_theta, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def gather_theta_results(local: torch.Tensor, n_theta: int, group: Optional[dist.ProcessGroup] = None) -> torch.Tensor:
    """All ranks receive the full `[n_theta, ...]` result, assembled in theta order from every rank's
    `theta_range` slice.  Ragged slices are padded to the largest one for the all_gather."""
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    lo, hi = theta_range(n_theta, rank, world)
    if local.shape[0] != hi - lo:
        raise ValueError("rank %d holds %d results, expected %d" % (rank, local.shape[0], hi - lo))
    width = -(-n_theta // world)
    pad = torch.zeros((width,) + tuple(local.shape[1:]), dtype=local.dtype, device=local.device)
    pad[: hi - lo] = local
    parts = [torch.empty_like(pad) for _ in range(world)]
    dist.all_gather(parts, pad, group=group)
    out = []
    for r in range(world):
        a, b = theta_range(n_theta, r, world)
        out.append(parts[r][: b - a])
    return torch.cat(out, 0)


def max_over_ranks(value: float, device, group: Optional[dist.ProcessGroup] = None) -> float:
    """Max of a per-rank scalar (a device-side duration): multi-GPU times are the slowest rank's."""
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())
