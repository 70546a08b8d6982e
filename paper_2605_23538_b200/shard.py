"""Sharding over ranks: host logic only -- index ranges and `torch.distributed` exchanges.  The
arithmetic of the method stays behind the C ABI: the cross-rank combine of an event / injection-sharded evaluation is
`gwc_combine_sharded` (device tensors) or `gwc_combine_sharded_host` (host tensors) of libgwc.so.

theta-sharding: log L(theta) of one hyper-parameter point needs nothing from any other point, so N GPUs split a batch
of theta and replicate the catalogue; there is no collective on the data path, only the gather of the `[n_theta]`
results and the max-over-ranks of a device time (NCCL on GPUs; the CPU tests use gloo).
Event / injection sharding: for the sampler's one-theta-per-call pattern and for catalogues that outgrow one GPU; one
all-gather of 3 x n_theta doubles per rank, then the combine.
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
# n_draw), and the ranks exchange one small array: an all-gather of (sum_i log L_i, log xi_r, N_eff,r)
# [world][3][n_theta], combined in rank order by gwc_combine_sharded so that every rank gets the same bits.
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


def event_shard(ev: dict, lo: int, hi: int) -> dict:
    """The sub-catalogue of events [lo, hi): sample arrays sliced, offsets rebased to 0; sample_row keeps the GLOBAL
    rows of the line-of-sight table, which every rank holds in full.  Indexing only."""
    off = ev["ev_sample_off"]
    a, b = int(off[lo]), int(off[hi])
    sub = {"ev_sample_off": (off[lo:hi + 1] - off[lo]).contiguous()}
    for k in ("dL", "m1z", "m2z", "sample_row", "log_pe_prior"):
        v = ev.get(k)
        sub[k] = None if v is None else v[a:b].contiguous()
    return sub


def injection_shard(inj: dict, rank: int, world: int) -> dict:
    """Rank `rank`'s contiguous block of the found injections (balanced like theta_range), with the GLOBAL n_draw, so
    that the xi of the whole set is the sum of the ranks' xi_r."""
    a, b = theta_range(inj["dL"].numel() if hasattr(inj["dL"], "numel") else len(inj["dL"]), rank, world)
    sub = {k: inj[k][a:b] for k in ("dL", "m1z", "m2z", "log_pdraw")}
    sub = {k: (v.contiguous() if hasattr(v, "contiguous") else v) for k, v in sub.items()}
    sub["n_draw"] = inj["n_draw"]
    return sub


def combine_event_sharded(sum_logL_local: torch.Tensor, logxi_local: torch.Tensor, neff_inj_local: torch.Tensor,
                          n_events_total: int, group: Optional[dist.ProcessGroup] = None, ctx=None):
    """log L(theta) = sum over ALL events of log L_i - n_events_total * log xi from per-rank pieces.
    sum_logL_local [n_theta]: sum of log L_i over this rank's events (0 for a rank without events).
    logxi_local, neff_inj_local [n_theta]: selection term over this rank's injections, computed with the global
    n_draw.  The pieces of all ranks are gathered (one all-gather of [3][n_theta]) and combined in rank order by
    libgwc.so: on the device through `ctx` (a gwc.Context) when the tensors are CUDA tensors, else by the host form.
    Returns (total, logxi, neff_inj), identical on every rank."""
    world = dist.get_world_size(group)
    trio = torch.stack([sum_logL_local, logxi_local, neff_inj_local], 0).to(torch.float64).contiguous()
    parts = [torch.empty_like(trio) for _ in range(world)]
    dist.all_gather(parts, trio, group=group)
    return combine_parts(parts, n_events_total, ctx)


def combine_parts(parts, n_events_total: int, ctx=None):
    """The combine step alone: `parts` is the rank-ordered list of [3][n_theta] tensors (sum log L_i, log xi_r,
    N_eff,r)."""
    from . import gwc
    allp = torch.stack(list(parts), 0)                       # [world][3][n_theta]
    pieces = [allp[:, k].contiguous() for k in range(3)]
    if allp.is_cuda:
        if ctx is None:
            raise ValueError("CUDA tensors need the gwc.Context to combine on")
        return ctx.gwc_combine_sharded(pieces[0], pieces[1], pieces[2], n_events_total)
    return gwc.Context.gwc_combine_sharded_host(pieces[0], pieces[1], pieces[2], n_events_total)
