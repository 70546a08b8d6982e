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


# ---- event / injection sharding: for catalogues that outgrow one GPU or very small theta batches --
# Each rank owns a contiguous block of events (balanced by samples) and a contiguous block of the found injections,
# evaluates every theta on them with the ordinary calls (gwc_event_loglik, gwc_selection_logxi with the GLOBAL
# n_draw), and the ranks exchange two small arrays: an all-reduce of sum_i log L_i  [n_theta]  and an all-gather of
# (log xi_r, N_eff,r)  [world][n_theta][2], combined in rank order so that every rank gets the same bits.
def event_range(ev_sample_off: torch.Tensor, rank: int, world: int) -> Tuple[int, int]:
    """[lo, hi) of the events owned by `rank`: contiguous blocks cut where the cumulative sample count crosses
    k * n_samples / world (every event belongs to exactly one rank; a rank may own none)."""
    if world < 1 or not (0 <= rank < world):
        raise ValueError("bad rank/world")
    off = ev_sample_off.detach().cpu().to(torch.int64)
    n_events = off.numel() - 1
    total = int(off[-1] - off[0])
    if n_events <= 0:
        return 0, 0
    mid = (off[:-1] + off[1:]).to(torch.float64) * 0.5 - float(off[0])     # event centres in sample units
    owner = torch.clamp((mid * world / max(total, 1)).floor().to(torch.int64), 0, world - 1) if total > 0 else \
        torch.div(torch.arange(n_events) * world, n_events, rounding_mode="floor")
    lo = int((owner < rank).sum())
    return lo, lo + int((owner == rank).sum())


def combine_event_sharded(sum_logL_local: torch.Tensor, logxi_local: torch.Tensor, neff_inj_local: torch.Tensor,
                          n_events_total: int, group: Optional[dist.ProcessGroup] = None):
    """log L(theta) = sum over ALL events of log L_i - n_events_total * log xi from per-rank pieces.
    sum_logL_local [n_theta]: sum of log L_i over this rank's events (0 for a rank without events).
    logxi_local, neff_inj_local [n_theta]: selection term over this rank's injections, computed with the global
    n_draw, so that xi = sum_r xi_r; N_eff = (sum_r S1_r)^2 / sum_r S2_r with S1_r = xi_r, S2_r = xi_r^2 / N_eff,r.
    Returns (total, logxi, neff_inj), identical on every rank (fixed rank order)."""
    world = dist.get_world_size(group)
    s = sum_logL_local.clone()
    parts = [torch.empty_like(s) for _ in range(world)]
    dist.all_gather(parts, s, group=group)                   # gathered, then summed in rank order: same bits everywhere
    sum_logL = torch.stack(parts, 0).sum(0) if world > 1 else s
    pair = torch.stack([logxi_local, neff_inj_local], -1).contiguous()
    pairs = [torch.empty_like(pair) for _ in range(world)]
    dist.all_gather(pairs, pair, group=group)
    lx = torch.stack([p[..., 0] for p in pairs], 0)          # [world][n_theta]
    ne = torch.stack([p[..., 1] for p in pairs], 0)
    m = lx.max(0).values
    m_safe = torch.where(torch.isfinite(m), m, torch.zeros_like(m))
    s1 = torch.exp(lx - m_safe)                              # xi_r relative to e^m  (0 for -inf)
    s2 = torch.where(ne > 0, s1 * s1 / ne.clamp_min(1e-300), torch.zeros_like(s1))
    S1, S2 = s1.sum(0), s2.sum(0)
    logxi = torch.where(S1 > 0, m_safe + torch.log(S1.clamp_min(1e-300)), torch.full_like(m, float("-inf")))
    neff = torch.where(S2 > 0, S1 * S1 / S2.clamp_min(1e-300), torch.zeros_like(S1))
    total = sum_logL - float(n_events_total) * logxi
    total = torch.where(torch.isneginf(sum_logL) | torch.isneginf(logxi), torch.full_like(total, float("-inf")), total)
    nan = torch.isnan(sum_logL) | torch.isnan(lx).any(0)
    total = torch.where(nan, torch.full_like(total, float("nan")), total)
    return total, logxi, neff
