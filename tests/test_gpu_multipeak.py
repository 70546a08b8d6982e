"""GPU parity of the MULTIPEAK mass model with delta_m smoothing (NEXT row 3a; App. A, Table III
:263-274; R33-R36): the fused kernel (events, injections, pixel cut) and the KDE numerator against the
oracle, through the C ABI, at north_star's FP64 bar (1e-9 relative, integers bit-exact)."""
from __future__ import annotations

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
    c.gwc_set_mass_model("multipeak")
    yield c
    c.close()


def _np(t):
    return t.detach().cpu().numpy()


def _mp_workload(config, n_theta, **kw):
    """The config's catalogue with the masses of every second event and injection scaled down by `light` (the SNR cut
    of the generator keeps heavy binaries only: 30-45 Msun), so that half of the samples fall into the smoothing
    window [mmin, mmin + delta_m] and onto the low peak."""
    light = kw.pop("light", 0.2)
    W = workload(config, n_theta=n_theta, **kw)
    off = W.ev["ev_sample_off"]
    eid = torch.repeat_interleave(torch.arange(off.numel() - 1), off[1:] - off[:-1])
    f = torch.where(eid % 2 == 1, light, 1.0).to(torch.float64)
    W.ev["m1z"] = W.ev["m1z"] * f
    W.ev["m2z"] = W.ev["m2z"] * f
    g = torch.where(torch.arange(W.inj["m1z"].numel()) % 2 == 1, light, 1.0).to(torch.float64)
    W.inj["m1z"] = W.inj["m1z"] * g
    W.inj["m2z"] = W.inj["m2z"] * g
    th = synth.make_theta_multipeak(W.spec, synth.DEFAULT_SEED, "cpu", n_theta)
    return W, th


def _check_all(ctx, W, th, prec=0, los=None, n_nodes=1025):
    los = W.los if los is None else los
    zmax = W.spec.z_max
    thd, ev, inj, lo = th.to(DEV), to_dev(W.ev, DEV), to_dev(W.inj, DEV), los.to(DEV)
    allsky = ctx.gwc_los_allsky(lo, zmax)
    ctx.gwc_build_cosmo(thd, zmax, n_nodes, prec)
    gL, gN, gK = ctx.gwc_event_loglik(thd, ev, lo, zmax)
    gX, gNx = ctx.gwc_selection_logxi(thd, inj, allsky, lo.shape[1], zmax)
    gT = ctx.gwc_total_loglik(thd, ev, inj, lo, zmax, allsky, n_nodes, prec)
    ctx.gwc_check()
    with oracle.mass_model("multipeak"):
        oL, oN, oK = oracle.event_loglik(_np(th), synth.to_numpy(W.ev), _np(los), zmax, table_prec=prec, n_nodes=n_nodes)
        oX, oNx = oracle.selection_logxi(_np(th), synth.to_numpy(W.inj), oracle.los_allsky(_np(los), zmax), zmax,
                                         table_prec=prec, n_nodes=n_nodes)
    oT = oracle.total_from_parts(oL, oX)
    bad = np.argwhere(_np(gK) != oK)
    assert bad.size == 0, "nlive differs at %s" % bad[:8].tolist()
    e1 = assert_close_log(_np(gL), oL, RTOL_F64, "log L_i (MULTIPEAK)")
    e2 = assert_close_log(_np(gX), oX, RTOL_F64, "log xi (MULTIPEAK)")
    assert_close_log(_np(gT), oT, RTOL_F64, "log L(theta) (MULTIPEAK)")
    fin = np.isfinite(oL)
    np.testing.assert_allclose(_np(gN)[fin], oN[fin], rtol=1e-7)
    np.testing.assert_allclose(_np(gNx), oNx, rtol=1e-7)
    return e1, e2, oK


def test_multipeak_tiny(ctx):
    W, th = _mp_workload("tiny", 16)
    e1, e2, oK = _check_all(ctx, W, th)
    assert (oK > 0).mean() > 0.7
    print("MULTIPEAK tiny: max rel err log L_i %.2e, log xi %.2e" % (e1, e2))


def test_multipeak_window_is_exercised():
    """The synthetic masses reach into the smoothing window [mmin, mmin + delta_m]: the table path and S(m2) matter."""
    W, th = _mp_workload("tiny", 16)
    t3 = np.asarray(synth.THETA_TABLE3_MULTIPEAK)
    z = 0.3
    m1 = W.ev["m1z"].numpy() / (1 + z)
    m2 = W.ev["m2z"].numpy() / (1 + z)
    top = t3[4] + t3[12]
    assert (m1 < top).mean() > 0.2 and (m2 < top).mean() > 0.3 and (m2 > t3[4]).mean() > 0.9


@pytest.mark.parametrize("prec", [0, 1])
def test_multipeak_ragged(ctx, prec):
    """Ragged catalogue, a box-6 theta batch with every MULTIPEAK parameter varied, both table storages; several
    theta tiles and launches of the constant bank are not needed at this size, the tile loop is (T < n_theta)."""
    W, th = _mp_workload("production", 24, n_events=7, los_rows=300, n_inj=20000, samples=(300, 2600), pixels=(4, 150))
    los = W.los.to(torch.float32) if prec == 1 else W.los
    _check_all(ctx, W, th, prec=prec, los=los)


def test_multipeak_edge_parameters(ctx):
    """delta_m = 0 (no smoothing: the step at mmin), lambda_low = 0 / 1, lambda_g = 0 / 1, beta + 1 < 0, a window that
    swallows most of the mass range, and a theta outside the domain (NaN + GWC_ERR_DOMAIN)."""
    from paper_2605_23538_b200 import gwc
    W, th = _mp_workload("tiny", 10)
    th[1, 12] = 0.0
    th[2, 15] = 0.0
    th[3, 15] = 1.0
    th[4, 8] = 0.0
    th[5, 8] = 1.0
    th[6, 3] = -2.5
    th[7, 12] = 30.0
    th[8, 12] = 0.0
    th[8, 3] = -1.7
    _check_all(ctx, W, th)
    th[9, 12] = 90.0          # mmin + delta_m >= mmax
    zmax = W.spec.z_max
    thd, ev, lo = th.to(DEV), to_dev(W.ev, DEV), W.los.to(DEV)
    ctx.gwc_build_cosmo(thd, zmax)
    gL, _, _ = ctx.gwc_event_loglik(thd, ev, lo, zmax)
    with pytest.raises(gwc.GwcError) as e:
        ctx.gwc_check()
    assert e.value.status == gwc.ERR_DOMAIN
    g = _np(gL)
    assert np.isnan(g[9]).all() and np.isfinite(g[:9]).all()


def test_multipeak_reduces_to_plpeak_on_the_gpu(ctx):
    """delta_m = 0 and lambda_low = 0: bit-for-bit the same support decisions as the power-law+peak context and the
    same log L_i to rounding (two code paths of the same kernel)."""
    from paper_2605_23538_b200 import gwc
    W = workload("tiny")
    th12 = W.theta.clone()
    th16 = torch.cat([th12, torch.tensor([[0.0, 9.7, 0.7, 0.0]], dtype=torch.float64).repeat(th12.shape[0], 1)], dim=1)
    zmax = W.spec.z_max
    ev, lo = to_dev(W.ev, DEV), W.los.to(DEV)
    t16 = th16.to(DEV)
    ctx.gwc_build_cosmo(t16, zmax)
    gL, gN, gK = ctx.gwc_event_loglik(t16, ev, lo, zmax)
    ctx.gwc_check()
    c0 = gwc.Context(0)
    t12 = th12.to(DEV)
    c0.gwc_build_cosmo(t12, zmax)
    hL, hN, hK = c0.gwc_event_loglik(t12, ev, lo, zmax)
    c0.gwc_check()
    c0.close()
    assert torch.equal(gK, hK)
    assert_close_log(_np(gL), _np(hL), 1e-12, "MULTIPEAK(delta_m = 0, one peak) vs power law + peak")


def test_multipeak_pixcut(ctx):
    W, th = _mp_workload("production", 12, n_events=5, los_rows=300, n_inj=1000, samples=(500, 2600), pixels=(8, 120))
    zmax = W.spec.z_max
    thd, ev, lo = th.to(DEV), to_dev(W.ev, DEV), W.los.to(DEV)
    ctx.gwc_build_cosmo(thd, zmax)
    gL, gN, gK, gP = ctx.gwc_event_loglik_pixcut(thd, ev, lo, zmax, 2.0)
    ctx.gwc_check()
    with oracle.mass_model("multipeak"):
        oL, oN, oK, oP = oracle.event_loglik_pixcut(_np(th), synth.to_numpy(W.ev), _np(W.los), zmax, 2.0)
    assert np.array_equal(_np(gP), oP) and np.array_equal(_np(gK), oK)
    assert_close_log(_np(gL), oL, RTOL_F64, "pixel-cut log L_i (MULTIPEAK)")


def test_multipeak_kde(ctx):
    W, th = _mp_workload("tiny", 6)
    zmax = W.spec.z_max
    thd, ev, lo = th.to(DEV), to_dev(W.ev, DEV), W.los.to(DEV)
    ctx.gwc_build_cosmo(thd, zmax)
    for bw in ("scott", "silverman", "biweight_scott"):
        gL, gP, gU = ctx.gwc_event_loglik_kde(thd, ev, lo, zmax, 128, 2.0, bw)
        ctx.gwc_check()
        with oracle.mass_model("multipeak"):
            oL, oP, oU = oracle.event_loglik_kde(_np(th), synth.to_numpy(W.ev), _np(W.los), zmax, n_grid=128,
                                                 neff_min=2.0, bandwidth=bw, want_nused=True)
        assert np.array_equal(_np(gP), oP) and np.array_equal(_np(gU), oU), bw
        assert_close_log(_np(gL), oL, RTOL_F64, "KDE log L_i (MULTIPEAK, %s)" % bw)


def test_multipeak_host_call_and_model_switch(ctx):
    """gwc_total_loglik_host with 16-column rows; switching the model drops the tables (GWC_ERR_NOT_BUILT)."""
    from paper_2605_23538_b200 import gwc
    W, th = _mp_workload("tiny", 5)
    zmax = W.spec.z_max
    a, _, _ = ctx.gwc_total_loglik_host(th, W.ev, W.inj, W.los, zmax)
    with oracle.mass_model("multipeak"):
        o = oracle.total_loglik(_np(th), synth.to_numpy(W.ev), synth.to_numpy(W.inj), _np(W.los), zmax)
    assert_close_log(a.numpy(), o, RTOL_F64, "host call (MULTIPEAK)")
    thd, ev, lo = th.to(DEV), to_dev(W.ev, DEV), W.los.to(DEV)
    ctx.gwc_build_cosmo(thd, zmax)
    ctx.gwc_set_mass_model("plpeak")
    with pytest.raises(ValueError):          # the binding checks the row width against the selected model
        ctx.gwc_event_loglik(thd, ev, lo, zmax)
    with pytest.raises(ValueError):
        ctx.gwc_build_cosmo(thd, zmax)
    ctx.gwc_set_mass_model("multipeak")
    with pytest.raises(gwc.GwcError) as e:   # the tables built before the switch are gone
        ctx.gwc_event_loglik(thd, ev, lo, zmax)
    assert e.value.status == gwc.ERR_NOT_BUILT
    ctx.gwc_build_cosmo(thd, zmax)
    ctx.gwc_event_loglik(thd, ev, lo, zmax)
    ctx.gwc_check()
    assert ctx.gwc_theta_len("multipeak") == 16 and ctx.gwc_theta_len("plpeak") == 12
