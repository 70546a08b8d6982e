"""GPU tests of the paths around the hot loop that round 1 left untested:
other node counts of the cosmology table, a LOS table that ends below the cosmology table, a user PE prior of wide
spread (the range rule of gwc.h), two contexts on two streams of one device, theta changed in place after the build,
the catalogue cache across host calls, the flag word of the packing, the n_z limit of the selection term."""
from __future__ import annotations

import threading

import numpy as np
import pytest
import torch

import oracle
from paper_2605_23538_b200 import synth
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


def _mini():
    """Ragged O4-like mini catalogue with a box-6 theta batch (every theta its own Om)."""
    W = workload("production", n_theta=23, n_events=9, los_rows=400, n_inj=20_000, samples=(300, 3000),
                 pixels=(16, 200))
    return W


@pytest.mark.parametrize("n_nodes", [257, 2049, 4097])
@pytest.mark.parametrize("table_prec", [0, 1])
def test_hot_path_other_node_counts(ctx, n_nodes, table_prec):
    """The whole hot path with M != 1025: the theta tile T, the table pitch and the shared-memory layout all change
    with M (M = 2049 -> T = 5, M = 4097 -> T = 2 for f64 nodes)."""
    W = _mini()
    zmax = W.spec.z_max
    th, ev, inj, los = W.theta.to(DEV), to_dev(W.ev, DEV), to_dev(W.inj, DEV), W.los.to(DEV)
    allsky = ctx.gwc_los_allsky(los, zmax)
    ctx.gwc_build_cosmo(th, zmax, n_nodes, table_prec)
    logL, neff, nlive = ctx.gwc_event_loglik(th, ev, los, zmax)
    logxi, neffi = ctx.gwc_selection_logxi(th, inj, allsky, los.shape[1], zmax)
    total = ctx.gwc_total_loglik(th, ev, inj, los, zmax, allsky, n_nodes, table_prec)
    gLp, _, gKp, gPp = ctx.gwc_event_loglik_pixcut(th, ev, los, zmax, 2.0)
    ctx.gwc_check()
    kw = dict(n_nodes=n_nodes, table_prec=table_prec)
    ev_np, inj_np, los_np, th_np = synth.to_numpy(W.ev), synth.to_numpy(W.inj), _np(W.los), _np(W.theta)
    oL, oN, oK = oracle.event_loglik(th_np, ev_np, los_np, zmax, **kw)
    oX, oXn = oracle.selection_logxi(th_np, inj_np, oracle.los_allsky(los_np, zmax), zmax, **kw)
    assert np.array_equal(_np(nlive), oK)
    assert_close_log(_np(logL), oL, RTOL_F64, "log L_i, M=%d" % n_nodes)
    assert_close_log(_np(logxi), oX, RTOL_F64, "log xi, M=%d" % n_nodes)
    assert_close_log(_np(total), oracle.total_from_parts(oL, oX), RTOL_F64, "log L(theta), M=%d" % n_nodes)
    fin = np.isfinite(oL)
    np.testing.assert_allclose(_np(neff)[fin], oN[fin], rtol=1e-7)
    oLp, _, oKp, oPp = oracle.event_loglik_pixcut(th_np, ev_np, los_np, zmax, 2.0, **kw)
    assert np.array_equal(_np(gPp), oPp) and np.array_equal(_np(gKp), oKp)
    assert_close_log(_np(gLp), oLp, RTOL_F64, "pixcut log L_i, M=%d" % n_nodes)


def test_los_zmax_below_cosmo_zmax(ctx):
    """gwc.h allows los->z_max <= the z_max of the build: samples with z >= los z_max are dead although the
    cosmology table still covers them (R11)."""
    W = workload("tiny")
    los_zmax = W.spec.z_max            # 1.5
    cosmo_zmax = 2.25
    th, ev, inj, los = W.theta.to(DEV), to_dev(W.ev, DEV), to_dev(W.inj, DEV), W.los.to(DEV)
    # push a good part of the samples beyond the LOS table but inside the cosmology table
    ev["dL"] = (ev["dL"] * 2.2).contiguous()
    ev_np = synth.to_numpy(W.ev)
    ev_np["dL"] = ev_np["dL"] * 2.2
    allsky = ctx.gwc_los_allsky(los, los_zmax)
    ctx.gwc_build_cosmo(th, cosmo_zmax, 1025, 0)
    logL, neff, nlive = ctx.gwc_event_loglik(th, ev, los, los_zmax)
    logxi, _ = ctx.gwc_selection_logxi(th, inj, allsky, los.shape[1], los_zmax)
    ctx.gwc_check()
    oL, oN, oK = oracle.event_loglik(_np(W.theta), ev_np, _np(W.los), los_zmax, z_max=cosmo_zmax)
    oX, _ = oracle.selection_logxi(_np(W.theta), synth.to_numpy(W.inj), oracle.los_allsky(_np(W.los), los_zmax),
                                   los_zmax, z_max=cosmo_zmax)
    oK_same_zmax = oracle.event_loglik(_np(W.theta), ev_np, _np(W.los), los_zmax)[2]
    assert (oK < W.ev["dL"].numel() // 4).any() and (oK > 0).any()
    assert np.array_equal(_np(nlive), oK)
    assert_close_log(_np(logL), oL, RTOL_F64, "log L_i, LOS z_max < cosmology z_max")
    assert_close_log(_np(logxi), oX, RTOL_F64, "log xi, LOS z_max < cosmology z_max")
    assert np.array_equal(oK, oK_same_zmax)     # same dead set as a table that ends where the LOS table ends
    from paper_2605_23538_b200 import gwc
    ctx.gwc_build_cosmo(th, 1.0, 1025, 0)       # a build that ends below the LOS table is refused
    with pytest.raises(gwc.GwcError) as e:
        ctx.gwc_event_loglik(th, ev, los, los_zmax)
    assert e.value.status == gwc.ERR_NOT_BUILT


def test_wide_log_pe_prior_range_rule(ctx):
    """R23 / gwc.h "Range": the sums are relative to max_k(-l_pi - ln m1z) over the VALID samples, whatever theta makes
    of them.  (a) The sample that sets the reference is dead for every theta and the live ones lie 250 nats below:
    still 1e-9.  (b) They lie 1000 nats below: the outputs of that event are NaN and gwc_check says GWC_ERR_RANGE --
    nothing is clamped silently.  The oracle's two-pass log-sum-exp handles both."""
    from paper_2605_23538_b200 import gwc
    W = workload("tiny")
    zmax = W.spec.z_max
    th, inj, los = W.theta.to(DEV), to_dev(W.inj, DEV), W.los.to(DEV)
    off = W.ev["ev_sample_off"]
    a, b = int(off[1]), int(off[2])
    for drop, expect_range in ((250.0, False), (1000.0, True)):
        ev_cpu = {k: (v.clone() if isinstance(v, torch.Tensor) else v) for k, v in W.ev.items()}
        lp = 2.0 * torch.log(ev_cpu["dL"])
        lp[a:b] += drop                    # event 1: every sample's prior raised ...
        lp[a] -= drop                      # ... except one, which sets the reference ...
        ev_cpu["m1z"][a] = 1e5             # ... and is dead for every theta (m1 > mmax), though valid
        ev_cpu["m2z"][a] = 9e4
        ev_cpu["log_pe_prior"] = lp.contiguous()
        ev = to_dev(ev_cpu, DEV)
        ctx.gwc_build_cosmo(th, zmax, 1025, 0)
        logL, neff, nlive = ctx.gwc_event_loglik(th, ev, los, zmax)
        gLp, _, gKp, gPp = ctx.gwc_event_loglik_pixcut(th, ev, los, zmax, 0.0)
        oL, oN, oK = oracle.event_loglik(_np(W.theta), synth.to_numpy(ev_cpu), _np(W.los), zmax)
        assert (oK[:, 1] > 0).all() and np.isfinite(oL[:, 1]).all()
        assert np.array_equal(_np(nlive), oK)
        if not expect_range:
            ctx.gwc_check()
            assert_close_log(_np(logL), oL, RTOL_F64, "log L_i, prior spread %g" % drop)
            np.testing.assert_allclose(_np(neff), oN, rtol=1e-7)
            assert_close_log(_np(gLp), oL, RTOL_F64, "pixcut(0) log L_i, prior spread %g" % drop)
        else:
            with pytest.raises(gwc.GwcError) as e:
                ctx.gwc_check()
            assert e.value.status == gwc.ERR_RANGE
            ctx.gwc_check()                                        # cleared
            g = _np(logL)
            assert np.isnan(g[:, 1]).all() and np.isnan(_np(neff)[:, 1]).all()
            keep = [0, 2, 3]
            assert_close_log(g[:, keep], oL[:, keep], RTOL_F64, "the other events")
    # the same rule for the selection term: one 8192-block of injections far below its reference
    inj_cpu = {k: (v.clone() if isinstance(v, torch.Tensor) else v) for k, v in W.inj.items()}
    lp = inj_cpu["log_pdraw"].clone()
    lp[:] += 1000.0
    lp[0] -= 1000.0
    inj_cpu["m1z"][0] = 1e5
    inj_cpu["m2z"][0] = 9e4
    inj_cpu["log_pdraw"] = lp
    allsky = ctx.gwc_los_allsky(los, zmax)
    ctx.gwc_build_cosmo(th, zmax, 1025, 0)
    logxi, _ = ctx.gwc_selection_logxi(th, to_dev(inj_cpu, DEV), allsky, los.shape[1], zmax)
    with pytest.raises(gwc.GwcError) as e:
        ctx.gwc_check()
    assert e.value.status == gwc.ERR_RANGE and torch.isnan(logxi).all()


def test_selection_block_out_of_range_but_negligible(ctx):
    """gwc.h "Range", selection term: a block of 8192 injections whose live weights all lie far below the block's own
    reference makes log xi NaN only if it could matter.  Block 1 of three: its first injection sets the reference
    and is dead for every theta (m1 > mmax); the others carry a draw density e^+600 larger, i.e. weights e^-600 of
    the other blocks'.  (a) The block's upper bound lies hundreds of nats under the other blocks: log xi and N_eff
    match the oracle (which sums everything exactly), GWC_OK.  (b) The same block with ordinary draw densities and
    only the reference sample 1000 nats up: it carries a third of xi, so NaN + GWC_ERR_RANGE as before."""
    from paper_2605_23538_b200 import gwc
    W = workload("production", n_theta=12, n_events=2, los_rows=300, n_inj=3 * 8192)
    zmax = W.spec.z_max
    th, los = W.theta.to(DEV), W.los.to(DEV)
    allsky = ctx.gwc_los_allsky(los, zmax)
    sky_np = oracle.los_allsky(_np(W.los), zmax)
    a, b = 8192, 2 * 8192
    for negligible in (True, False):
        inj_cpu = {k: (v.clone() if isinstance(v, torch.Tensor) else v) for k, v in W.inj.items()}
        lp = inj_cpu["log_pdraw"].clone()
        if negligible:
            lp[a + 1:b] += 600.0            # weights e^-600 of the other blocks'
            lp[a] -= 100.0                  # the dead reference sample: 700 nats above the block's live weights
        else:
            lp[a] -= 1000.0
        inj_cpu["m1z"][a] = 1e5
        inj_cpu["m2z"][a] = 9e4
        inj_cpu["log_pdraw"] = lp.contiguous()
        ctx.gwc_build_cosmo(th, zmax, 1025, 0)
        gX, gN = ctx.gwc_selection_logxi(th, to_dev(inj_cpu, DEV), allsky, los.shape[1], zmax)
        if negligible:
            ctx.gwc_check()
            oX, oN = oracle.selection_logxi(_np(W.theta), synth.to_numpy(inj_cpu), sky_np, zmax)
            assert np.isfinite(oX).all()
            assert_close_log(_np(gX), oX, RTOL_F64, "log xi with a negligible out-of-range block")
            np.testing.assert_allclose(_np(gN), oN, rtol=1e-7)
        else:
            with pytest.raises(gwc.GwcError) as e:
                ctx.gwc_check()
            assert e.value.status == gwc.ERR_RANGE and torch.isnan(gX).all() and torch.isnan(gN).all()
            ctx.gwc_check()


def test_two_contexts_two_streams(ctx):
    """Two contexts on two streams of one device, driven from two host threads at once (the per-theta
    constants of all contexts share the device's constant bank).  Results must equal the serial ones bit for bit."""
    from paper_2605_23538_b200 import gwc
    Wa = workload("o4", n_theta=700, n_events=40, los_rows=2000, n_inj=60_000)
    Wb = workload("production", n_theta=700, n_events=30, los_rows=2000, n_inj=50_000, seed=5)
    sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
    ca, cb = gwc.Context(0, stream=sa), gwc.Context(0, stream=sb)
    try:
        def prep(W):
            return (W.theta.to(DEV), to_dev(W.ev, DEV), to_dev(W.inj, DEV), W.los.to(DEV))
        A, B = prep(Wa), prep(Wb)
        torch.cuda.synchronize()
        ska, skb = ctx.gwc_los_allsky(A[3], Wa.spec.z_max), ctx.gwc_los_allsky(B[3], Wb.spec.z_max)
        ra = ctx.gwc_total_loglik(A[0], A[1], A[2], A[3], Wa.spec.z_max, ska).clone()
        rb = ctx.gwc_total_loglik(B[0], B[1], B[2], B[3], Wb.spec.z_max, skb).clone()
        torch.cuda.synchronize()
        assert torch.isfinite(ra).any() and torch.isfinite(rb).any()
        out = {"a": [], "b": []}

        def run(c, stream, X, W, sky, key):
            with torch.cuda.stream(stream):
                for _ in range(6):
                    out[key].append(c.gwc_total_loglik(X[0], X[1], X[2], X[3], W.spec.z_max, sky))
            stream.synchronize()

        ta = threading.Thread(target=run, args=(ca, sa, A, Wa, ska, "a"))
        tb = threading.Thread(target=run, args=(cb, sb, B, Wb, skb, "b"))
        ta.start(); tb.start(); ta.join(); tb.join()
        torch.cuda.synchronize()
        ca.gwc_check(); cb.gwc_check()
        for r in out["a"]:
            assert torch.equal(torch.nan_to_num(r, nan=1.0), torch.nan_to_num(ra, nan=1.0))
        for r in out["b"]:
            assert torch.equal(torch.nan_to_num(r, nan=1.0), torch.nan_to_num(rb, nan=1.0))
        # and interleaved from one thread, no synchronisation in between
        rs = []
        for _ in range(4):
            rs.append((ca.gwc_total_loglik(A[0], A[1], A[2], A[3], Wa.spec.z_max, ska),
                       cb.gwc_total_loglik(B[0], B[1], B[2], B[3], Wb.spec.z_max, skb)))
        torch.cuda.synchronize()
        for x, y in rs:
            assert torch.equal(torch.nan_to_num(x, nan=1.0), torch.nan_to_num(ra, nan=1.0))
            assert torch.equal(torch.nan_to_num(y, nan=1.0), torch.nan_to_num(rb, nan=1.0))
    finally:
        ca.close(); cb.close()


def test_theta_changed_in_place_after_build(ctx):
    """pointer identity is not enough.  A theta row updated in place after gwc_build_cosmo must not give
    the old point's results silently: its outputs are NaN and gwc_check says GWC_ERR_NOT_BUILT; the untouched rows
    keep their values; the KDE path (which reads the population parameters) behaves the same."""
    from paper_2605_23538_b200 import gwc
    W = workload("tiny")
    zmax = W.spec.z_max
    th, ev, inj, los = W.theta.to(DEV).clone(), to_dev(W.ev, DEV), to_dev(W.inj, DEV), W.los.to(DEV)
    allsky = ctx.gwc_los_allsky(los, zmax)
    ctx.gwc_build_cosmo(th, zmax, 1025, 0)
    ref, _, _ = ctx.gwc_event_loglik(th, ev, los, zmax)
    refx, _ = ctx.gwc_selection_logxi(th, inj, allsky, los.shape[1], zmax)
    refk, _, _ = ctx.gwc_event_loglik_kde(th, ev, los, zmax, 64, 0.0)
    ctx.gwc_check()
    th[3, 0] += 5.0           # H0 of point 3
    th[7, 6] += 1.0           # mu of point 7 (no table depends on it: only the constants do)
    for call in ("event", "pixcut", "kde", "selection"):
        if call == "event":
            got = ctx.gwc_event_loglik(th, ev, los, zmax)[0]
            want = ref
        elif call == "pixcut":
            got = ctx.gwc_event_loglik_pixcut(th, ev, los, zmax, 0.0)[0]
            want = ref
        elif call == "kde":
            got = ctx.gwc_event_loglik_kde(th, ev, los, zmax, 64, 0.0)[0]
            want = refk
        else:
            got = ctx.gwc_selection_logxi(th, inj, allsky, los.shape[1], zmax)[0][:, None]
            want = refx[:, None]
        with pytest.raises(gwc.GwcError) as e:
            ctx.gwc_check()
        assert e.value.status == gwc.ERR_NOT_BUILT, call
        assert torch.isnan(got[3]).all() and torch.isnan(got[7]).all(), call
        keep = [i for i in range(th.shape[0]) if i not in (3, 7)]
        if call == "pixcut":
            np.testing.assert_allclose(_np(got[keep]), _np(want[keep]), rtol=1e-13)
        else:
            assert torch.equal(got[keep], want[keep]), call
    # a rebuild makes the new values legal
    ctx.gwc_build_cosmo(th, zmax, 1025, 0)
    new, _, _ = ctx.gwc_event_loglik(th, ev, los, zmax)
    ctx.gwc_check()
    o = oracle.event_loglik(_np(th), synth.to_numpy(W.ev), _np(W.los), zmax)[0]
    assert_close_log(_np(new), o, RTOL_F64, "after the rebuild")
    assert not torch.equal(new[3], ref[3])


def test_host_calls_with_cache_on_and_two_catalogues(ctx):
    """gwc_total_loglik_host uploads into the same internal mirrors every call; with the catalogue cache
    on a second catalogue of the same shape must not reuse the first one's preparation."""
    W = workload("tiny")
    zmax = W.spec.z_max
    ev2 = dict(W.ev, dL=(W.ev["dL"] * 1.07).contiguous(), m1z=(W.ev["m1z"] * 0.97).contiguous())
    inj2 = dict(W.inj, dL=(W.inj["dL"] * 0.95).contiguous())
    o1 = oracle.total_loglik(_np(W.theta), synth.to_numpy(W.ev), synth.to_numpy(W.inj), _np(W.los), zmax)
    o2 = oracle.total_loglik(_np(W.theta), synth.to_numpy(ev2), synth.to_numpy(inj2), _np(W.los), zmax)
    ctx.gwc_cache_catalogue(True)
    try:
        a, _, _ = ctx.gwc_total_loglik_host(W.theta, W.ev, W.inj, W.los, zmax)
        a = a.clone()
        b, _, _ = ctx.gwc_total_loglik_host(W.theta, ev2, inj2, W.los, zmax)
        b = b.clone()
        c, _, _ = ctx.gwc_total_loglik_host(W.theta, W.ev, W.inj, W.los, zmax)
    finally:
        ctx.gwc_cache_catalogue(False)
    assert_close_log(a.numpy(), o1, RTOL_F64, "first catalogue")
    assert_close_log(b.numpy(), o2, RTOL_F64, "second catalogue, same shapes")
    assert np.array_equal(a.numpy(), c.numpy(), equal_nan=True)
    assert not np.array_equal(a.numpy(), b.numpy())


def test_pack_has_its_own_flag(ctx):
    """a theta-domain flag left by gwc_build_cosmo is neither reported nor consumed by gwc_pack_events /
    gwc_cap_pixels; a bad event id is reported by the packing itself and leaves nothing behind."""
    from paper_2605_23538_b200 import gwc
    th = torch.tensor([synth.THETA0, synth.THETA0], dtype=torch.float64)
    th[1, 0] = -1.0
    ctx.gwc_build_cosmo(th.to(DEV), 1.5, 257, 0)          # raises the sticky domain flag
    g = torch.Generator().manual_seed(3)
    eid = torch.randint(0, 5, (1000,), generator=g, dtype=torch.int32)
    row = torch.randint(0, 40, (1000,), generator=g, dtype=torch.int32)
    p = ctx.gwc_pack_events(eid.to(DEV), row.to(DEV), 5)  # valid input: must succeed
    o = oracle.pack_events(eid.numpy(), row.numpy(), 5)
    assert np.array_equal(_np(p["perm"]), o["perm"])
    ctx.gwc_cap_pixels(p, 3, 1)
    with pytest.raises(gwc.GwcError) as e:                # the domain flag is still there for gwc_check
        ctx.gwc_check()
    assert e.value.status == gwc.ERR_DOMAIN
    bad = eid.clone()
    bad[17] = 9
    with pytest.raises(gwc.GwcError) as e:
        ctx.gwc_pack_events(bad.to(DEV), row.to(DEV), 5)
    assert e.value.status == gwc.ERR_DOMAIN
    ctx.gwc_check()                                        # nothing left behind
    ctx.gwc_pack_events(eid.to(DEV), row.to(DEV), 5)       # and the next valid call is fine


def test_nz_limit_checked_before_any_work(ctx):
    from paper_2605_23538_b200 import gwc
    W = workload("tiny")
    th, ev, inj = W.theta.to(DEV), to_dev(W.ev, DEV), to_dev(W.inj, DEV)
    nz = 4097
    los = torch.rand(8, nz, dtype=torch.float64, device=DEV) + 0.5
    allsky = ctx.gwc_los_allsky(los, 1.5)
    n0 = ctx.gwc_launch_count()
    with pytest.raises(gwc.GwcError) as e:
        ctx.gwc_total_loglik(th, ev, inj, los, 1.5, allsky)
    assert e.value.status == gwc.ERR_SHAPE and ctx.gwc_launch_count() == n0
    # the event term alone takes it (the LOS rows stay in global memory)
    ctx.gwc_build_cosmo(th, 1.5, 1025, 0)
    logL, _, nlive = ctx.gwc_event_loglik(th, ev, los, 1.5)
    ctx.gwc_check()
    oL, _, oK = oracle.event_loglik(_np(W.theta), synth.to_numpy(W.ev), _np(los), 1.5)
    assert np.array_equal(_np(nlive), oK)
    assert_close_log(_np(logL), oL, RTOL_F64, "log L_i, n_z = 4097")


def _structured_events(pattern, rows0=5):
    """One event per entry of `pattern`; an entry is the list of its pixel sizes (runs of equal sample_row)."""
    g = torch.Generator().manual_seed(17)
    dl, m1, m2, row, off = [], [], [], [], [0]
    for e, sizes in enumerate(pattern):
        n = int(sum(sizes))
        dl.append(900.0 * torch.exp(0.25 * torch.randn(n, generator=g, dtype=torch.float64)))
        a = 42.0 * (1 + 0.07 * torch.randn(n, generator=g, dtype=torch.float64))
        b = 31.0 * (1 + 0.07 * torch.randn(n, generator=g, dtype=torch.float64))
        m1.append(torch.maximum(a, b))
        m2.append(torch.minimum(a, b))
        row.append(torch.repeat_interleave(torch.arange(len(sizes)) + rows0 + e, torch.tensor(sizes, dtype=torch.int64)))
        off.append(off[-1] + n)
    cat = lambda xs, dt: (torch.cat(xs).to(dt) if xs else torch.zeros(0, dtype=dt))
    return {"ev_sample_off": torch.tensor(off, dtype=torch.int64), "dL": cat(dl, torch.float64), "m1z": cat(m1, torch.float64),
            "m2z": cat(m2, torch.float64), "sample_row": cat(row, torch.int32), "log_pe_prior": None}


def test_pixcut_and_kde_on_structured_pixel_patterns(ctx):
    """The pixel-aligned padded copy (pixel-cut mode) and the chunk table (KDE) on run patterns chosen to hit their
    corners: only odd runs (every pixel padded), only single samples, one pixel longer than several 64-sample blocks
    and than a KDE chunk, runs that end exactly on block boundaries, an empty event in the middle, a one-sample
    event, pixels of 63 / 64 / 65 / 127 / 129 samples."""
    import oracle
    from paper_2605_23538_b200 import synth
    from util import RTOL_F64, assert_close_log
    W = workload("o4", n_theta=6, n_events=2, los_rows=400, n_inj=100)
    pattern = [[1, 3, 5, 7, 9, 11, 13], [1] * 40, [2600, 3, 1], [64, 64, 128, 2], [], [1], [63, 64, 65, 127, 129, 1, 2],
               [2] * 33 + [1], [1100, 1100, 7]]
    ev = _structured_events(pattern)
    zmax = W.spec.z_max
    th, evd, lo = W.theta.to(DEV), to_dev(ev, DEV), W.los.to(DEV)
    ev_np = {k: (v.numpy() if isinstance(v, torch.Tensor) else v) for k, v in ev.items()}
    ctx.gwc_build_cosmo(th, zmax)
    for thr in (0.0, 2.0, 5.0):
        gL, gN, gK, gP = ctx.gwc_event_loglik_pixcut(th, evd, lo, zmax, thr)
        ctx.gwc_check()
        oL, oN, oK, oP = oracle.event_loglik_pixcut(W.theta.numpy(), ev_np, W.los.numpy(), zmax, thr)
        assert np.array_equal(gP.cpu().numpy(), oP) and np.array_equal(gK.cpu().numpy(), oK), thr
        assert_close_log(gL.cpu().numpy(), oL, RTOL_F64, "pixel cut, structured patterns, threshold %g" % thr)
    for bw in ("scott", "silverman"):
        kL, kP, kU = ctx.gwc_event_loglik_kde(th, evd, lo, zmax, 256, 2.0, bw)
        ctx.gwc_check()
        rL, rP, rU = oracle.event_loglik_kde(W.theta.numpy(), ev_np, W.los.numpy(), zmax, n_grid=256, neff_min=2.0,
                                             bandwidth=bw, want_nused=True)
        assert np.array_equal(kP.cpu().numpy(), rP) and np.array_equal(kU.cpu().numpy(), rU), bw
        assert_close_log(kL.cpu().numpy(), rL, RTOL_F64, "KDE, structured patterns, %s" % bw)
    assert np.isneginf(gL.cpu().numpy()[:, 4]).all() and np.isneginf(kL.cpu().numpy()[:, 4]).all()   # the empty event


def test_pixcut_with_cache_on_between_plain_and_cut_calls(ctx):
    """gwc_cache_catalogue keeps the prepared samples AND their padded copy: plain, cut, plain, cut on one catalogue,
    then another catalogue in other arrays: every result equals the uncached one bit for bit."""
    Wa = workload("o4", n_theta=8, n_events=6, los_rows=400, n_inj=500)
    Wb = workload("o4", n_theta=8, n_events=5, los_rows=400, n_inj=500, seed=3)
    zmax = Wa.spec.z_max
    ref = {}
    for name, W in (("a", Wa), ("b", Wb)):
        th, ev, lo = W.theta.to(DEV), to_dev(W.ev, DEV), W.los.to(DEV)
        ctx.gwc_build_cosmo(th, zmax)
        ref[name] = (th, ev, lo, ctx.gwc_event_loglik(th, ev, lo, zmax)[0].clone(),
                     [x.clone() for x in ctx.gwc_event_loglik_pixcut(th, ev, lo, zmax, 2.0)])
    ctx.gwc_cache_catalogue(True)
    try:
        for name in ("a", "a", "b", "a"):
            th, ev, lo, plain, cut = ref[name]
            ctx.gwc_build_cosmo(th, zmax)
            for _ in range(2):
                assert torch.equal(ctx.gwc_event_loglik(th, ev, lo, zmax)[0].view(torch.int64), plain.view(torch.int64))
                got = ctx.gwc_event_loglik_pixcut(th, ev, lo, zmax, 2.0)
                assert all(torch.equal(g.view(torch.int64), c.view(torch.int64)) for g, c in zip(got, cut))
        ctx.gwc_check()
    finally:
        ctx.gwc_cache_catalogue(False)


def test_single_omega_batches_share_one_table(ctx):
    """A batch of 48 theta with one Omega_m stages one z(u) table per tile (16 theta per tile); the same batch with the
    Omega_m of its last point changed must not.  Both against the oracle, events, injections and the pixel cut."""
    import oracle
    from util import RTOL_F64, assert_close_log
    W = workload("o4", n_theta=48, n_events=6, los_rows=400, n_inj=3000)
    zmax = W.spec.z_max
    assert bool((W.theta[:, 1] == W.theta[0, 1]).all())
    ev, inj, lo = to_dev(W.ev, DEV), to_dev(W.inj, DEV), W.los.to(DEV)
    allsky = ctx.gwc_los_allsky(lo, zmax)
    ev_np, inj_np = synth.to_numpy(W.ev), synth.to_numpy(W.inj)
    for change in (False, True):
        th = W.theta.clone()
        if change:
            th[47, 1] = 0.27
        thd = th.to(DEV)
        total = ctx.gwc_total_loglik(thd, ev, inj, lo, zmax, allsky)
        ctx.gwc_build_cosmo(thd, zmax)
        gL, gN, gK, gP = ctx.gwc_event_loglik_pixcut(thd, ev, lo, zmax, 2.0)
        ctx.gwc_check()
        o = oracle.total_loglik(th.numpy(), ev_np, inj_np, W.los.numpy(), zmax)
        assert_close_log(total.cpu().numpy(), o, RTOL_F64, "log L(theta), single Omega_m %s" % (not change))
        oL, oN, oK, oP = oracle.event_loglik_pixcut(th.numpy(), ev_np, W.los.numpy(), zmax, 2.0)
        assert np.array_equal(gP.cpu().numpy(), oP) and np.array_equal(gK.cpu().numpy(), oK)
        assert_close_log(gL.cpu().numpy(), oL, RTOL_F64, "pixel cut, single Omega_m %s" % (not change))


def test_omega_hint(ctx):
    """gwc_set_omega_hint: what the caller knows about Omega_m replaces the device question (and its stream
    synchronisation) of gwc_build_cosmo.  "varies" and "single" on a single-Omega_m batch (48 points and 7 points)
    both match the oracle; "single" on a batch that breaks the promise is reported by gwc_check as
    GWC_ERR_INVALID_ARG; back on "detect" the same batch is right again."""
    import oracle
    from paper_2605_23538_b200 import gwc
    from util import RTOL_F64, assert_close_log
    W = workload("o4", n_theta=48, n_events=6, los_rows=400, n_inj=3000)
    zmax = W.spec.z_max
    ev, inj, lo = to_dev(W.ev, DEV), to_dev(W.inj, DEV), W.los.to(DEV)
    allsky = ctx.gwc_los_allsky(lo, zmax)
    ev_np, inj_np, los_np = synth.to_numpy(W.ev), synth.to_numpy(W.inj), W.los.numpy()
    o = oracle.total_loglik(W.theta.numpy(), ev_np, inj_np, los_np, zmax)
    try:
        for hint in ("varies", "single"):
            ctx.gwc_set_omega_hint(hint)
            for n in (48, 7):
                thd = W.theta[:n].contiguous().to(DEV)
                total = ctx.gwc_total_loglik(thd, ev, inj, lo, zmax, allsky)
                ctx.gwc_check()
                assert_close_log(total.cpu().numpy(), o[:n], RTOL_F64, "log L(theta), hint %s, %d points" % (hint, n))
        th = W.theta.clone()
        th[47, 1] = 0.27                                    # the promise of one Omega_m is broken
        thd = th.to(DEV)
        ctx.gwc_total_loglik(thd, ev, inj, lo, zmax, allsky)
        with pytest.raises(gwc.GwcError) as e:
            ctx.gwc_check()
        assert e.value.status == gwc.ERR_INVALID_ARG and "GWC_OMEGA_SINGLE" in str(e.value)
        ctx.gwc_check()
        ctx.gwc_set_omega_hint("detect")
        total = ctx.gwc_total_loglik(thd, ev, inj, lo, zmax, allsky)
        ctx.gwc_check()
        assert_close_log(total.cpu().numpy(), oracle.total_loglik(th.numpy(), ev_np, inj_np, los_np, zmax), RTOL_F64,
                         "log L(theta), detect, two Omega_m")
    finally:
        ctx.gwc_set_omega_hint("detect")


def test_single_omega_batch_with_points_outside_the_domain(ctx):
    """48 theta with one Omega_m, rows 0 and 16 outside the domain (sigma < 0; Omega_m itself valid and equal): they are
    the first points of their 16-point tiles, whose all-zero z(u) table must not be staged for the valid points beside
    them.  Only those two rows are NaN; every other row matches the oracle: events, pixel cut, injections, total."""
    import oracle
    from paper_2605_23538_b200 import gwc
    from util import RTOL_F64, assert_close_log
    W = workload("o4", n_theta=48, n_events=6, los_rows=400, n_inj=3000)
    zmax = W.spec.z_max
    assert bool((W.theta[:, 1] == W.theta[0, 1]).all())
    th = W.theta.clone()
    bad = [0, 16]
    th[bad, 7] = -1.0
    good = [t for t in range(48) if t not in bad]
    ev, inj, lo = to_dev(W.ev, DEV), to_dev(W.inj, DEV), W.los.to(DEV)
    allsky = ctx.gwc_los_allsky(lo, zmax)
    ev_np, inj_np = synth.to_numpy(W.ev), synth.to_numpy(W.inj)
    thd = th.to(DEV)
    total = ctx.gwc_total_loglik(thd, ev, inj, lo, zmax, allsky).cpu().numpy()
    ctx.gwc_build_cosmo(thd, zmax)
    gL, _, gK = ctx.gwc_event_loglik(thd, ev, lo, zmax)
    pL, _, pK, pP = ctx.gwc_event_loglik_pixcut(thd, ev, lo, zmax, 2.0)
    gX, _ = ctx.gwc_selection_logxi(thd, inj, allsky, lo.shape[1], zmax)
    with pytest.raises(gwc.GwcError) as e:
        ctx.gwc_check()
    assert e.value.status == gwc.ERR_DOMAIN
    ctx.gwc_check()
    gL, pL, gX = gL.cpu().numpy(), pL.cpu().numpy(), gX.cpu().numpy()
    assert np.isnan(total[bad]).all() and np.isnan(gL[bad]).all() and np.isnan(pL[bad]).all() and np.isnan(gX[bad]).all()
    tg = th[good].numpy()     # the oracle sees the valid rows only
    los_np = W.los.numpy()
    assert_close_log(total[good], oracle.total_loglik(tg, ev_np, inj_np, los_np, zmax), RTOL_F64, "log L(theta) beside invalid rows")
    oL, _, oK = oracle.event_loglik(tg, ev_np, los_np, zmax)
    assert_close_log(gL[good], oL, RTOL_F64, "log L_i beside invalid rows")
    assert np.array_equal(gK.cpu().numpy()[good], oK)
    qL, _, qK, qP = oracle.event_loglik_pixcut(tg, ev_np, los_np, zmax, 2.0)
    assert_close_log(pL[good], qL, RTOL_F64, "pixel cut beside invalid rows")
    assert np.array_equal(pK.cpu().numpy()[good], qK) and np.array_equal(pP.cpu().numpy()[good], qP)
    oX, _ = oracle.selection_logxi(tg, inj_np, oracle.los_allsky(los_np, zmax), zmax)
    assert_close_log(gX[good], oX, RTOL_F64, "log xi beside invalid rows")


def test_selection_with_injections_sorted_inside_the_library(ctx):
    """Calls of 2e8 (theta x injection) terms and up run the selection term on a copy of the injections in order of
    d_L (pack.cu).  Against the oracle (which sums in the caller's order) at the FP64 bar; with the catalogue cache on,
    a second injection set of the same shape in other arrays must not meet the first one's sorted copy; invalid
    injections (NaN, negative d_L) stay dead wherever the sort puts them."""
    import oracle
    from util import RTOL_F64, assert_close_log
    W = workload("production", n_theta=1024, n_events=2, los_rows=300, n_inj=200_000)
    zmax = W.spec.z_max
    th, lo = W.theta.to(DEV), W.los.to(DEV)
    allsky = ctx.gwc_los_allsky(lo, zmax)
    sky_np = oracle.los_allsky(W.los.numpy(), zmax)
    inj_a = {k: (v.clone() if isinstance(v, torch.Tensor) else v) for k, v in W.inj.items()}
    inj_a["dL"][5], inj_a["dL"][77], inj_a["m1z"][123] = float("nan"), -3.0, float("inf")
    inj_b = {k: (v.flip(0).contiguous() * (1.02 if k == "dL" else 1.0) if isinstance(v, torch.Tensor) else v)
             for k, v in W.inj.items()}
    ctx.gwc_build_cosmo(th, zmax)
    ctx.gwc_cache_catalogue(True)
    try:
        for inj in (inj_a, inj_b, inj_a):
            d = to_dev(inj, DEV)
            for _ in range(2):
                gX, gN = ctx.gwc_selection_logxi(th, d, allsky, lo.shape[1], zmax)
            ctx.gwc_check()
            oX, oN = oracle.selection_logxi(W.theta.numpy(), synth.to_numpy(inj), sky_np, zmax)
            assert_close_log(gX.cpu().numpy(), oX, RTOL_F64, "log xi on sorted injections")
            np.testing.assert_allclose(gN.cpu().numpy(), oN, rtol=1e-7)
    finally:
        ctx.gwc_cache_catalogue(False)


def test_two_contexts_pixcut_and_kde_concurrently(ctx):
    """Two contexts on two streams from two host threads, one running the pixel-cut event term (constant bank, padded
    copy), the other the KDE numerator (chunk table, scratch): the bits of the serial results."""
    from paper_2605_23538_b200 import gwc
    Wa = workload("o4", n_theta=400, n_events=30, los_rows=2000, n_inj=1000)
    Wb = workload("production", n_theta=12, n_events=20, los_rows=2000, n_inj=1000, seed=5)
    sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
    ca, cb = gwc.Context(0, stream=sa), gwc.Context(0, stream=sb)
    try:
        A = (Wa.theta.to(DEV), to_dev(Wa.ev, DEV), Wa.los.to(DEV))
        B = (Wb.theta.to(DEV), to_dev(Wb.ev, DEV), Wb.los.to(DEV))
        torch.cuda.synchronize()
        ctx.gwc_build_cosmo(A[0], Wa.spec.z_max)
        ra = [x.clone() for x in ctx.gwc_event_loglik_pixcut(A[0], A[1], A[2], Wa.spec.z_max, 2.0)]
        ctx.gwc_build_cosmo(B[0], Wb.spec.z_max)
        rb = [x.clone() for x in ctx.gwc_event_loglik_kde(B[0], B[1], B[2], Wb.spec.z_max, 256, 2.0)]
        torch.cuda.synchronize()
        out = {"a": [], "b": []}

        def run_a():
            with torch.cuda.stream(sa):
                for _ in range(5):
                    ca.gwc_build_cosmo(A[0], Wa.spec.z_max)
                    out["a"].append(ca.gwc_event_loglik_pixcut(A[0], A[1], A[2], Wa.spec.z_max, 2.0))
            sa.synchronize()

        def run_b():
            with torch.cuda.stream(sb):
                for _ in range(5):
                    cb.gwc_build_cosmo(B[0], Wb.spec.z_max)
                    out["b"].append(cb.gwc_event_loglik_kde(B[0], B[1], B[2], Wb.spec.z_max, 256, 2.0))
            sb.synchronize()

        ta, tb = threading.Thread(target=run_a), threading.Thread(target=run_b)
        ta.start(); tb.start(); ta.join(); tb.join()
        torch.cuda.synchronize()
        ca.gwc_check(); cb.gwc_check()
        eq = lambda x, y: torch.equal(torch.nan_to_num(x.double(), nan=1.0, neginf=-1e300), torch.nan_to_num(y.double(), nan=1.0, neginf=-1e300))
        for r in out["a"]:
            assert all(eq(x, y) for x, y in zip(r, ra))
        for r in out["b"]:
            assert all(eq(x, y) for x, y in zip(r, rb))
    finally:
        ca.close(); cb.close()


def test_two_contexts_share_the_constant_bank_across_streams(ctx):
    """Both contexts run the fused re-weighting kernel, which reads the per-theta constants from the device's ONE
    constant bank: two streams, two host threads, different theta batches of different sizes (700 and 400 points: three
    and two launches of at most 340 points each, so the bank is rewritten inside every call and between the contexts'
    launches).  A copy into the bank that overtook a kernel still reading it would change that kernel's results: every
    repetition must give the bits of the serial run.  One context does the event term, the other alternates the
    selection term and the event term."""
    from paper_2605_23538_b200 import gwc
    Wa = workload("production", n_theta=700, n_events=12, los_rows=1000, n_inj=30_000, seed=3)
    Wb = workload("production", n_theta=400, n_events=8, los_rows=1000, n_inj=40_000, seed=4)
    sa, sb = torch.cuda.Stream(), torch.cuda.Stream()
    ca, cb = gwc.Context(0, stream=sa), gwc.Context(0, stream=sb)
    try:
        A = (Wa.theta.to(DEV), to_dev(Wa.ev, DEV), Wa.los.to(DEV), to_dev(Wa.inj, DEV))
        B = (Wb.theta.to(DEV), to_dev(Wb.ev, DEV), Wb.los.to(DEV), to_dev(Wb.inj, DEV))
        za, zb = Wa.spec.z_max, Wb.spec.z_max
        sky_b = ctx.gwc_los_allsky(B[2], zb)
        nzb = B[2].shape[1]
        ctx.gwc_build_cosmo(A[0], za)
        ra = [x.clone() for x in ctx.gwc_event_loglik(A[0], A[1], A[2], za)]
        ctx.gwc_build_cosmo(B[0], zb)
        rb_x = [x.clone() for x in ctx.gwc_selection_logxi(B[0], B[3], sky_b, nzb, zb)]
        rb_e = [x.clone() for x in ctx.gwc_event_loglik(B[0], B[1], B[2], zb)]
        ctx.gwc_check()
        torch.cuda.synchronize()
        out = {"a": [], "bx": [], "be": []}
        go = threading.Barrier(2)

        def run_a():
            go.wait()
            with torch.cuda.stream(sa):
                for _ in range(6):
                    ca.gwc_build_cosmo(A[0], za)
                    out["a"].append(ca.gwc_event_loglik(A[0], A[1], A[2], za))
            sa.synchronize()

        def run_b():
            go.wait()
            with torch.cuda.stream(sb):
                for _ in range(6):
                    cb.gwc_build_cosmo(B[0], zb)
                    out["bx"].append(cb.gwc_selection_logxi(B[0], B[3], sky_b, nzb, zb))
                    out["be"].append(cb.gwc_event_loglik(B[0], B[1], B[2], zb))
            sb.synchronize()

        ta, tb = threading.Thread(target=run_a), threading.Thread(target=run_b)
        ta.start(); tb.start(); ta.join(); tb.join()
        torch.cuda.synchronize()
        ca.gwc_check(); cb.gwc_check()
        eq = lambda x, y: torch.equal(torch.nan_to_num(x.double(), nan=1.0, neginf=-1e300), torch.nan_to_num(y.double(), nan=1.0, neginf=-1e300))
        assert len(out["a"]) == 6 and len(out["bx"]) == 6 and len(out["be"]) == 6
        for r in out["a"]:
            assert all(eq(x, y) for x, y in zip(r, ra))
        for r in out["bx"]:
            assert all(eq(x, y) for x, y in zip(r, rb_x))
        for r in out["be"]:
            assert all(eq(x, y) for x, y in zip(r, rb_e))
    finally:
        ca.close(); cb.close()
