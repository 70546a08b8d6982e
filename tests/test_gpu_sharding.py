"""Event / injection sharding through libgwc.so (the split a one-theta-per-call sampler needs,
PAPER.md:129, :166).  One B200 plays R ranks one after the other: every rank's block of events (global LOS rows) goes
through gwc_event_loglik, its block of injections through gwc_selection_logxi with the global n_draw, the pieces are
combined by gwc_combine_sharded -- and the result is compared with the unsharded GPU result and with the oracle."""
from __future__ import annotations

import numpy as np
import pytest
import torch

import oracle
from paper_2605_23538_b200 import shard, synth
from util import RTOL_F64, assert_close_log, to_dev, workload

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


@pytest.fixture(scope="module")
def ctx():
    from paper_2605_23538_b200 import gwc
    c = gwc.Context(0)
    yield c
    c.close()


def _np(t):
    return t.detach().cpu().numpy()


def _sharded(ctx, W, world):
    """What R ranks would compute, in rank order, on one device.  Returns the combined (total, logxi, neff_inj), the
    per-rank event ranges and the per-rank log L_i blocks."""
    zmax = W.spec.z_max
    th, los = W.theta.to(DEV), W.los.to(DEV)
    allsky = ctx.gwc_los_allsky(los, zmax)
    ev, inj = to_dev(W.ev, DEV), to_dev(W.inj, DEV)
    n_events = W.ev["ev_sample_off"].numel() - 1
    zeros = torch.zeros(th.shape[0], dtype=torch.float64, device=DEV)
    parts, ranges, blocks = [], [], []
    for r in range(world):
        lo, hi = shard.event_range(W.ev["ev_sample_off"], r, world)
        ranges.append((lo, hi))
        ctx.gwc_build_cosmo(th, zmax)                       # a rank builds its own tables
        if hi > lo:
            logL, _, _ = ctx.gwc_event_loglik(th, shard.event_shard(ev, lo, hi), los, zmax)
            s = ctx.gwc_combine_total(logL, zeros)          # sum_i log L_i - n * 0
            blocks.append(logL.clone())
        else:
            s = zeros.clone()
            blocks.append(None)
        lx, ne = ctx.gwc_selection_logxi(th, shard.injection_shard(inj, r, world), allsky, los.shape[1], zmax)
        parts.append(torch.stack([s, lx, ne], 0))
    out = shard.combine_parts(parts, n_events, ctx)
    ctx.gwc_check()
    return out, ranges, blocks, parts


def _unsharded(ctx, W):
    zmax = W.spec.z_max
    th, los = W.theta.to(DEV), W.los.to(DEV)
    allsky = ctx.gwc_los_allsky(los, zmax)
    ev, inj = to_dev(W.ev, DEV), to_dev(W.inj, DEV)
    total = ctx.gwc_total_loglik(th, ev, inj, los, zmax, allsky)
    ctx.gwc_build_cosmo(th, zmax)
    logL, _, _ = ctx.gwc_event_loglik(th, ev, los, zmax)
    lx, ne = ctx.gwc_selection_logxi(th, inj, allsky, los.shape[1], zmax)
    ctx.gwc_check()
    return total, logL, lx, ne


CASES = {
    "tiny": lambda: workload("tiny"),
    "ragged_o4_mini": lambda: workload("o4", n_theta=21, n_events=11, los_rows=500, n_inj=40_000, samples=(200, 6000),
                                       pixels=(8, 300)),
    "one_theta_production": lambda: workload("production", n_theta=1, n_events=40, los_rows=3000, n_inj=100_000),
    "two_events_three_ranks": lambda: workload("production", n_theta=3, n_events=2, los_rows=300, n_inj=20_000),
}


@pytest.mark.parametrize("world", [2, 3])
@pytest.mark.parametrize("case", sorted(CASES))
def test_event_and_injection_sharding_through_the_library(ctx, case, world):
    W = CASES[case]()
    n_events = W.ev["ev_sample_off"].numel() - 1
    (total, logxi, neff), ranges, blocks, parts = _sharded(ctx, W, world)
    u_total, u_logL, u_lx, u_ne = _unsharded(ctx, W)
    # the ranges partition the events; with fewer events than ranks somebody owns none
    assert ranges[0][0] == 0 and ranges[-1][1] == n_events
    assert all(ranges[r][1] == ranges[r + 1][0] for r in range(world - 1))
    if case == "two_events_three_ranks" and world == 3:
        assert any(hi == lo for lo, hi in ranges)
    # every event's log L_i on its rank against the unsharded call: the same terms, but where the event falls in the
    # work groups of the catalogue decides how its samples are cut into blocks, i.e. the order of the sum -- equal up
    # to that rounding (observed: bit-equal in most cases, 1 ulp otherwise), -inf where the other is -inf
    for (lo, hi), blk in zip(ranges, blocks):
        if blk is not None:
            assert_close_log(_np(blk), _np(u_logL[:, lo:hi]), 1e-14, "log L_i of events [%d, %d) on their rank" % (lo, hi))
    # sum_r S_r of the combine = the rank-ordered sum of the per-rank sums, bit for bit (total + n log xi undoes A6)
    S = torch.stack([p[0] for p in parts], 0)
    acc = torch.zeros_like(S[0])
    for r in range(world):
        acc = acc + S[r]
    fin = torch.isfinite(acc) & torch.isfinite(logxi)
    assert torch.equal((acc - float(n_events) * logxi)[fin], total[fin]) or \
        torch.allclose((acc - float(n_events) * logxi)[fin], total[fin], rtol=1e-15, atol=0.0)   # (an fma in the kernel)
    # against the unsharded GPU result
    assert_close_log(_np(logxi), _np(u_lx), 1e-12, "log xi, %d ranks vs one" % world)
    np.testing.assert_allclose(_np(neff), _np(u_ne), rtol=1e-10)
    assert_close_log(_np(total), _np(u_total), 1e-12, "log L(theta), %d ranks vs one" % world)
    # against the oracle, which knows nothing of ranks
    ev_np, inj_np, los_np = synth.to_numpy(W.ev), synth.to_numpy(W.inj), _np(W.los)
    o_total = oracle.total_loglik(_np(W.theta), ev_np, inj_np, los_np, W.spec.z_max)
    o_lx, o_ne = oracle.selection_logxi(_np(W.theta), inj_np, oracle.los_allsky(los_np, W.spec.z_max), W.spec.z_max)
    assert_close_log(_np(total), o_total, RTOL_F64, "log L(theta), %d ranks vs the oracle" % world)
    assert_close_log(_np(logxi), o_lx, RTOL_F64, "log xi, %d ranks vs the oracle" % world)
    np.testing.assert_allclose(_np(neff), o_ne, rtol=1e-7)
    # the host form of the combine (ranks that gathered through host memory) agrees with the device form
    h_total, h_lx, h_ne = shard.combine_parts([p.cpu() for p in parts], n_events)
    assert_close_log(_np(total), _np(h_total), 1e-14, "host combine vs device combine")
    assert_close_log(_np(logxi), _np(h_lx), 1e-14, "host combine vs device combine (log xi)")
