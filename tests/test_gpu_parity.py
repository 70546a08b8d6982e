"""GPU parity tests: the CUDA path (through the C ABI binding) against the CPU oracle, element by element,
on the same seeded inputs.  Tolerances are north_star's: bit-exact integers, relative 1e-9 on log L_i and
log xi for the FP64 path, absolute 1e-4 on log L(theta) for the FP32-table path."""
from __future__ import annotations

import numpy as np
import pytest
import torch

import oracle
from paper_2605_23538_b200 import synth
from util import ATOL_F32, RTOL_F64, assert_close_log, to_dev, workload

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    from paper_2605_23538_b200 import gwc
    c = gwc.Context(0)
    yield c
    c.close()


DEV = "cuda:0"


def _np(t):
    return t.detach().cpu().numpy()


def _oracle_all(W, theta, los=None, table_prec=0, n_nodes=1025):
    los = W.los if los is None else los
    ev, inj = synth.to_numpy(W.ev), synth.to_numpy(W.inj)
    lt = _np(los)
    logL, neff, nlive = oracle.event_loglik(_np(theta), ev, lt, W.spec.z_max, table_prec=table_prec, n_nodes=n_nodes)
    allsky = oracle.los_allsky(lt, W.spec.z_max)
    logxi, neffi = oracle.selection_logxi(_np(theta), inj, allsky, W.spec.z_max, table_prec=table_prec,
                                          n_nodes=n_nodes)
    total = oracle.total_from_parts(logL, logxi)
    return dict(logL=logL, neff=neff, nlive=nlive, allsky=allsky, logxi=logxi, neff_inj=neffi, total=total)


def _gpu_all(ctx, W, theta, los=None, table_prec=0, n_nodes=1025):
    los = (W.los if los is None else los).to(DEV)
    th = theta.to(DEV)
    ev, inj = to_dev(W.ev, DEV), to_dev(W.inj, DEV)
    zmax = W.spec.z_max
    allsky = ctx.gwc_los_allsky(los, zmax)
    ctx.gwc_build_cosmo(th, zmax, n_nodes, table_prec)
    logL, neff, nlive = ctx.gwc_event_loglik(th, ev, los, zmax)
    logxi, neffi = ctx.gwc_selection_logxi(th, inj, allsky, los.shape[1], zmax)
    total = ctx.gwc_combine_total(logL, logxi)
    total2 = ctx.gwc_total_loglik(th, ev, inj, los, zmax, allsky, n_nodes, table_prec)
    torch.cuda.synchronize()
    return dict(logL=_np(logL), neff=_np(neff), nlive=_np(nlive), allsky=_np(allsky), logxi=_np(logxi),
                neff_inj=_np(neffi), total=_np(total), total2=_np(total2))


def _compare(g, o, rtol=RTOL_F64, check_nlive=True):
    np.testing.assert_allclose(g["allsky"], o["allsky"], rtol=1e-13, atol=0)
    if check_nlive:
        bad = np.argwhere(g["nlive"] != o["nlive"])
        assert bad.size == 0, "nlive differs at %s" % bad[:8].tolist()
    assert_close_log(g["logL"], o["logL"], rtol, "log L_i")
    assert_close_log(g["logxi"], o["logxi"], rtol, "log xi")
    fin = np.isfinite(o["logL"])
    np.testing.assert_allclose(g["neff"][fin], o["neff"][fin], rtol=1e-7)
    np.testing.assert_allclose(g["neff_inj"], o["neff_inj"], rtol=1e-7)
    # log L(theta): sum of E terms each within rtol
    assert_close_log(g["total"], o["total"], rtol, "log L(theta)")
    assert np.array_equal(g["total"], g["total2"], equal_nan=True), "gwc_total_loglik != composed calls"


# ---------------------------------------------------------------------------------------------
def test_math_functions(ctx):
    """exp/log/rcp/rsqrt of math64.cuh against torch's fp64 functions.  exp and log are built to ~2e-13 (cubic /
    quartic on a 256- / 128-entry table: DESIGN.md section 6), 5000x inside north_star's 1e-9; rcp and rsqrt are
    correctly rounded to an ulp or two."""
    g = torch.Generator(device="cpu").manual_seed(1)
    x = (torch.rand(1 << 16, generator=g, dtype=torch.float64) * 1400.0 - 700.0).to(DEV)
    for which in (0, 4):
        y = ctx.gwc_math_selftest(which, x)
        rel = ((y - torch.exp(x)) / torch.exp(x)).abs().max().item()
        assert rel < 3e-13, rel
    y = ctx.gwc_math_selftest(0, torch.tensor([-1e4, -float("inf"), -700.0], dtype=torch.float64, device=DEV))
    assert torch.all(torch.isfinite(y)) and y.max().item() < 1e-300
    xp = torch.exp((torch.rand(1 << 16, generator=g, dtype=torch.float64) * 40.0 - 20.0)).to(DEV)
    xs = torch.cat([xp, 1.0 + torch.rand(1 << 16, generator=g, dtype=torch.float64).to(DEV) * 3.0])
    y = ctx.gwc_math_selftest(1, xs)
    assert (y - torch.log(xs)).abs().max().item() < 3e-13
    y = ctx.gwc_math_selftest(2, xs)
    assert ((y * xs) - 1.0).abs().max().item() < 5e-16
    y = ctx.gwc_math_selftest(3, xs)
    assert ((y * y * xs) - 1.0).abs().max().item() < 1e-15


@pytest.mark.parametrize("n_nodes", [1025, 257, 2])
def test_cosmo_table_nodes(ctx, n_nodes):
    """A1: table nodes against the oracle's exact inverse (<= 1e-13) and its node slopes."""
    oms = [0.05, 0.1, 0.3, 0.315, 0.5, 1.0]
    th = torch.tensor([synth.THETA0] * len(oms), dtype=torch.float64)
    th[:, 1] = torch.tensor(oms, dtype=torch.float64)
    thd = th.to(DEV)
    for zmax in (1.5, 2.0):
        ctx.gwc_build_cosmo(thd, zmax, n_nodes, 0)
        z, dz, umax = ctx.gwc_export_cosmo(len(oms), n_nodes)
        ctx.gwc_check()
        for i, om in enumerate(oms):
            zt, dt, um = oracle.build_table(om, zmax, n_nodes)
            assert abs(umax[i].item() - um) <= 2e-15 * um
            np.testing.assert_allclose(_np(z[i]), zt, rtol=0, atol=1e-13)
            np.testing.assert_allclose(_np(dz[i]), dt, rtol=1e-12, atol=0)
            assert z[i, 0].item() == 0.0 and z[i, -1].item() == zmax


def test_cosmo_closed_forms(ctx):
    """A1 against the closed forms: Om = 1 => u = 2(1+z)(1 - (1+z)^-1/2); nodes must invert it."""
    th = torch.tensor([synth.THETA0], dtype=torch.float64)
    th[0, 1] = 1.0
    ctx.gwc_build_cosmo(th.to(DEV), 2.0, 1025, 0)
    z, _, umax = ctx.gwc_export_cosmo(1, 1025)
    z = _np(z[0])
    u = np.arange(1025) * (umax.item() / 1024)
    np.testing.assert_allclose(2 * (1 + z) * (1 - (1 + z) ** -0.5), u, rtol=0, atol=3e-13)


def test_tiny_parity(ctx):
    W = workload("tiny")
    o = _oracle_all(W, W.theta)
    g = _gpu_all(ctx, W, W.theta)
    ctx.gwc_check()
    _compare(g, o)


def test_ragged_o4_like_parity(ctx):
    """O4-scale layout cut down so the oracle runs in seconds: ragged S_i and P_i, several chunks and a tail."""
    W = workload("o4", n_theta=24, n_events=12, los_rows=600, n_inj=30_000, samples=(300, 4096), pixels=(16, 300))
    o = _oracle_all(W, W.theta)
    g = _gpu_all(ctx, W, W.theta)
    ctx.gwc_check()
    _compare(g, o)


def test_box6_theta_parity_f32_los(ctx):
    """Production-like: every theta has its own Om (table per theta), FP32 LOS table, FP64 cosmology table."""
    W = workload("production", n_theta=20, n_events=10, los_rows=500, n_inj=20_000, samples=(700, 1500),
                 pixels=(16, 200))
    assert W.los.dtype == torch.float32
    o = _oracle_all(W, W.theta)
    g = _gpu_all(ctx, W, W.theta)
    ctx.gwc_check()
    _compare(g, o)


def test_f32_table_variant(ctx):
    """FP32 storage of the cosmology table and the LOS table, arithmetic in FP64 (R22):
    within 1e-9 of the oracle run with the same rounded tables (nlive bit-exact), within 1e-4 of the FP64 result."""
    W = workload("stress", n_theta=16, n_events=10, los_rows=400, n_inj=20_000, big_samples=4096, big_pixels=300,
                 big_frac=0.2)
    los32 = W.los.to(torch.float32)
    o32 = _oracle_all(W, W.theta, los=los32, table_prec=1)
    g32 = _gpu_all(ctx, W, W.theta, los=los32, table_prec=1)
    _compare(g32, o32)      # same rounded tables on both sides: the FP64 bar, nlive bit-exact
    o64 = _oracle_all(W, W.theta)
    fin = np.isfinite(o64["total"]) & np.isfinite(g32["total"])
    assert fin.any()
    assert np.abs(g32["total"][fin] - o64["total"][fin]).max() <= ATOL_F32


def test_edge_cases(ctx):
    """Empty events, dead samples, invalid rows, lambda = 0, an invalid theta, user-supplied PE prior."""
    W = workload("tiny")
    ev = {k: (v.clone() if isinstance(v, torch.Tensor) else v) for k, v in W.ev.items()}
    n = ev["dL"].numel()
    # event 1 becomes empty: move its samples into event 0
    off = ev["ev_sample_off"].clone()
    off[1] = off[2]
    ev["ev_sample_off"] = off
    ev["dL"][3] = float("nan")
    ev["dL"][5] = -1.0
    ev["m1z"][7] = float("inf")
    ev["m2z"][9] = ev["m1z"][9] * 1.5       # m2z > m1z: dead
    ev["sample_row"][11] = 10_000           # out-of-range row: dead, no out-of-bounds read
    ev["sample_row"][12] = -3
    ev["dL"][n - 256:] = 1e9                # last event entirely beyond the table: log L_i = -inf
    ev["log_pe_prior"] = (2.0 * torch.log(W.ev["dL"]) + 1234.5).contiguous()   # arbitrary constant offset
    theta = W.theta.clone()
    theta[2, 8] = 0.0                       # lambda = 0: no Gaussian term
    theta[3, 8] = 1.0                       # lambda = 1: no power-law term
    theta[5, 0] = -70.0                     # invalid H0: NaN outputs, sticky flag
    W.ev = ev
    o = _oracle_all(W, theta)
    g = _gpu_all(ctx, W, theta)
    from paper_2605_23538_b200 import gwc
    with pytest.raises(gwc.GwcError) as e:
        ctx.gwc_check()
    assert e.value.status == gwc.ERR_DOMAIN
    ctx.gwc_check()  # flag cleared
    assert np.isnan(g["logL"][5]).all() and np.isnan(g["total"][5])
    assert np.isneginf(g["logL"][:5, 3]).all() and np.isneginf(g["logL"][:5, 1]).all()
    _compare(g, o)


def test_not_built_and_bad_args(ctx):
    from paper_2605_23538_b200 import gwc
    W = workload("tiny")
    th = W.theta.to(DEV)
    ev, los = to_dev(W.ev, DEV), W.los.to(DEV)
    ctx.gwc_build_cosmo(th, 1.5, 1025, 0)
    other = th.clone()
    with pytest.raises(gwc.GwcError) as e:
        ctx.gwc_event_loglik(other, ev, los, 1.5)
    assert e.value.status == gwc.ERR_NOT_BUILT
    with pytest.raises(gwc.GwcError) as e:
        ctx.gwc_build_cosmo(th, 1.5, 1, 0)
    assert e.value.status == gwc.ERR_SHAPE
    with pytest.raises(gwc.GwcError) as e:
        ctx.gwc_build_cosmo(th, -1.0, 1025, 0)
    assert e.value.status == gwc.ERR_INVALID_ARG


def test_pack_events_bit_exact(ctx):
    """A0: permutation, offsets, distinct rows and run starts equal the oracle's, bit for bit."""
    g = torch.Generator().manual_seed(7)
    n, ne = 50_000, 37
    eid = torch.randint(0, ne, (n,), generator=g, dtype=torch.int32)
    eid[eid == 5] = 6                      # an empty event in the middle
    eid[eid == ne - 1] = 0                 # and at the end
    row = torch.randint(0, 300, (n,), generator=g, dtype=torch.int32)
    o = oracle.pack_events(eid.numpy(), row.numpy(), ne)
    p = ctx.gwc_pack_events(eid.to(DEV), row.to(DEV), ne)
    assert p["n_pixrefs"] == o["n_pixrefs"]
    for k in ("perm", "ev_sample_off", "ev_pix_off", "ev_pix_rows", "pix_sample_off"):
        assert np.array_equal(_np(p[k]), o[k]), k
    p0 = ctx.gwc_pack_events(eid[:0].to(DEV), row[:0].to(DEV), 3)
    assert p0["n_pixrefs"] == 0 and _np(p0["ev_sample_off"]).tolist() == [0, 0, 0, 0]


def test_host_api_matches_device_api(ctx):
    W = workload("tiny")
    g = _gpu_all(ctx, W, W.theta)
    out, up, down = ctx.gwc_total_loglik_host(W.theta, W.ev, W.inj, W.los, W.spec.z_max)
    assert np.array_equal(out.numpy(), g["total"], equal_nan=True)
    assert down == 8 * W.theta.shape[0] and up > W.los.numel() * 8


def test_determinism(ctx):
    W = workload("o4", n_theta=40, n_events=30, los_rows=600, n_inj=50_000, samples=(300, 3000), pixels=(16, 300))
    a = _gpu_all(ctx, W, W.theta)
    b = _gpu_all(ctx, W, W.theta)
    for k in ("logL", "neff", "logxi", "total"):
        assert np.array_equal(a[k], b[k], equal_nan=True), k


# ---- NEXT row 2: the per-pixel N_eff cut of Eq. 8 (R25) -------------------------------
def _pixcut_both(ctx, W, theta, thr, los=None):
    los = W.los if los is None else los
    zmax = W.spec.z_max
    th = theta.to(DEV)
    ctx.gwc_build_cosmo(th, zmax, 1025, 0)
    g = ctx.gwc_event_loglik_pixcut(th, to_dev(W.ev, DEV), los.to(DEV), zmax, thr)
    ctx.gwc_check()
    o = oracle.event_loglik_pixcut(_np(theta), synth.to_numpy(W.ev), _np(los), zmax, thr)
    return [_np(x) for x in g], o


def _pixcut_compare(g, o, what):
    gL, gN, gK, gP = g
    oL, oN, oK, oP = o
    bad = np.argwhere(gP != oP)
    assert bad.size == 0, "%s: npass differs at %s" % (what, bad[:8].tolist())
    bad = np.argwhere(gK != oK)
    assert bad.size == 0, "%s: nlive differs at %s" % (what, bad[:8].tolist())
    assert_close_log(gL, oL, RTOL_F64, what + " log L_i")
    fin = np.isfinite(oL)
    np.testing.assert_allclose(gN[fin], oN[fin], rtol=1e-7)


@pytest.mark.parametrize("thr", [0.0, 2.0, 5.0])
def test_pixcut_tiny(ctx, thr):
    W = workload("tiny")
    g, o = _pixcut_both(ctx, W, W.theta, thr)
    _pixcut_compare(g, o, "tiny thr=%g" % thr)
    if thr == 0.0:      # threshold 0 = the uncut path, bit for bit the same sums
        th = W.theta.to(DEV)
        ctx.gwc_build_cosmo(th, W.spec.z_max, 1025, 0)
        logL, neff, nlive = ctx.gwc_event_loglik(th, to_dev(W.ev, DEV), W.los.to(DEV), W.spec.z_max)
        np.testing.assert_allclose(g[0], _np(logL), rtol=1e-13, atol=0)
        assert np.array_equal(g[2], _np(nlive))


@pytest.mark.parametrize("thr", [2.0, 3.5])
def test_pixcut_ragged_catalogue(ctx, thr):
    """O4-like catalogue: ragged events, pixels of 1 to hundreds of samples, pixels that span blocks and warps."""
    W = workload("o4", n_theta=24, n_events=12, los_rows=600, n_inj=1000)
    g, o = _pixcut_both(ctx, W, W.theta, thr)
    _pixcut_compare(g, o, "o4-like thr=%g" % thr)
    assert (o[3] > 0).any() and (o[3] < o[3].max()).any()
    # the cut bites: some events lose pixels relative to threshold 0
    o0 = oracle.event_loglik_pixcut(_np(W.theta), synth.to_numpy(W.ev), _np(W.los), W.spec.z_max, 0.0)
    assert (o[3] < o0[3]).any()


def test_pixcut_long_and_short_pixels(ctx):
    """Stress layout: events of 32768 samples over thousands of pixels next to events of 512 over 16; plus a
    hand-made event whose single pixel spans many blocks and one with every sample its own pixel."""
    W = workload("stress", n_theta=8, n_events=8, los_rows=300, n_inj=1000, big_samples=6000, big_pixels=250,
                 big_frac=0.25)
    off = W.ev["ev_sample_off"]
    row = W.ev["sample_row"].clone()
    a, b = int(off[0]), int(off[1])
    row[a:b] = 7                                   # event 0: one pixel over the whole event
    a, b = int(off[1]), int(off[2])
    row[a:b] = (torch.arange(b - a) // 2 % 290).to(row.dtype)   # event 1: every pixel has two samples
    a, b = int(off[2]), int(off[3])
    row[a:b] = (torch.arange(b - a) % 290).to(row.dtype)        # event 2: every sample its own pixel
    W.ev["sample_row"] = row
    for thr in (2.0, 1.0):
        g, o = _pixcut_both(ctx, W, W.theta, thr)
        _pixcut_compare(g, o, "stress-like thr=%g" % thr)


def test_pixcut_determinism_and_args(ctx):
    from paper_2605_23538_b200 import gwc
    W = workload("o4", n_theta=8, n_events=6, los_rows=200, n_inj=500)
    th = W.theta.to(DEV)
    ev, los = to_dev(W.ev, DEV), W.los.to(DEV)
    ctx.gwc_build_cosmo(th, W.spec.z_max, 1025, 0)
    a = ctx.gwc_event_loglik_pixcut(th, ev, los, W.spec.z_max, 2.0)
    b = ctx.gwc_event_loglik_pixcut(th, ev, los, W.spec.z_max, 2.0)
    for x, y in zip(a, b):
        assert torch.equal(x, y)
    with pytest.raises(gwc.GwcError):
        ctx.gwc_event_loglik_pixcut(th, ev, los, W.spec.z_max, -1.0)
    with pytest.raises(gwc.GwcError):
        ctx.gwc_event_loglik_pixcut(th, ev, los, W.spec.z_max, float("nan"))


def test_pixcut_edge_cases_and_32bit_tables(ctx):
    """Pixel cut with empty events, dead / invalid samples (which still delimit pixels by their raw row value),
    a user PE prior, f32 LOS rows and the 32-bit cosmology table."""
    W = workload("o4", n_theta=12, n_events=6, los_rows=120, n_inj=500)
    ev = {k: (v.clone() if isinstance(v, torch.Tensor) else v) for k, v in W.ev.items()}
    off = ev["ev_sample_off"].clone()
    off[2] = off[3]                               # event 2 becomes empty, its samples join event 1
    ev["ev_sample_off"] = off
    ev["dL"][5] = float("nan")
    ev["dL"][17] = -2.0
    ev["sample_row"][40:44] = 10_000              # invalid rows: dead, but a pixel of their own
    ev["sample_row"][60] = -7
    ev["m2z"][80] = ev["m1z"][80] * 2.0
    g = torch.Generator().manual_seed(3)
    ev["log_pe_prior"] = 2.0 * torch.log(ev["dL"].abs().clamp_min(1.0)) + 0.3 * torch.rand(ev["dL"].numel(), generator=g,
                                                                                         dtype=torch.float64)
    zmax = W.spec.z_max
    th = W.theta.to(DEV)
    for los, prec in ((W.los, 0), (W.los.to(torch.float32), 0), (W.los.to(torch.float32), 1)):
        ctx.gwc_build_cosmo(th, zmax, 1025, prec)
        gq = [_np(x) for x in ctx.gwc_event_loglik_pixcut(th, to_dev(ev, DEV), los.to(DEV), zmax, 2.0)]
        ctx.gwc_check()
        o = oracle.event_loglik_pixcut(_np(W.theta), synth.to_numpy(ev), _np(los), zmax, 2.0, table_prec=prec)
        if prec == 0:
            _pixcut_compare(gq, o, "edge cases (%s LOS)" % los.dtype)
        else:   # 32-bit nodes: the oracle on the same rounded tables, same bar
            _pixcut_compare(gq, o, "edge cases (32-bit tables)")
    assert np.all(np.isneginf(gq[0][:, 2])) and np.all(gq[3][:, 2] == 0)


# ---- NEXT row 1: the paper's KDE numerator (Eq. 5-7, D1; R26-R30) -------------------------------------
def _kde_both(ctx, W, theta, ev=None, los=None, n_grid=256, neff_min=0.0, prec=0, bandwidth="scott"):
    ev = W.ev if ev is None else ev
    los = W.los if los is None else los
    zmax = W.spec.z_max
    th = theta.to(DEV)
    ctx.gwc_build_cosmo(th, zmax, 1025, prec)
    gL, gP, gU = ctx.gwc_event_loglik_kde(th, to_dev(ev, DEV), los.to(DEV), zmax, n_grid, neff_min, bandwidth)
    ctx.gwc_check()
    oL, oP, oU = oracle.event_loglik_kde(_np(theta), synth.to_numpy(ev), _np(los), zmax, n_grid=n_grid,
                                         neff_min=neff_min, table_prec=prec, want_nused=True, bandwidth=bandwidth)
    assert np.array_equal(_np(gU), oU), "nused differs"
    return (_np(gL), _np(gP)), (oL, oP)


def _kde_compare(g, o, what, rtol=RTOL_F64):
    bad = np.argwhere(g[1] != o[1])
    assert bad.size == 0, "%s: npass differs at %s" % (what, bad[:8].tolist())
    return assert_close_log(g[0], o[0], rtol, what + " log L_i (KDE)")


@pytest.mark.parametrize("n_grid,neff_min", [(256, 0.0), (256, 2.0), (100, 0.0), (33, 3.0)])
def test_kde_tiny(ctx, n_grid, neff_min):
    W = workload("tiny")
    g, o = _kde_both(ctx, W, W.theta, n_grid=n_grid, neff_min=neff_min)
    worst = _kde_compare(g, o, "tiny G=%d nmin=%g" % (n_grid, neff_min))
    assert np.isfinite(o[0]).any() and (o[1] > 0).any()
    print("KDE tiny G=%d: max rel err %.2e" % (n_grid, worst))


def test_kde_ragged_catalogue(ctx):
    """O4-like: ragged events, pixels of 1 sample (no bandwidth) to hundreds, f32 and f64 LOS rows."""
    W = workload("o4", n_theta=16, n_events=10, los_rows=500, n_inj=500)
    for los in (W.los, W.los.to(torch.float32)):
        g, o = _kde_both(ctx, W, W.theta, los=los, neff_min=2.0)
        _kde_compare(g, o, "o4-like %s" % los.dtype)
    assert (o[1] > 1).any()


def test_kde_edge_cases(ctx):
    from paper_2605_23538_b200 import gwc
    W = workload("o4", n_theta=10, n_events=6, los_rows=120, n_inj=500)
    ev = {k: (v.clone() if isinstance(v, torch.Tensor) else v) for k, v in W.ev.items()}
    off = ev["ev_sample_off"].clone()
    off[2] = off[3]                               # an empty event
    ev["ev_sample_off"] = off
    ev["dL"][5] = float("nan")
    ev["dL"][17] = -2.0
    ev["sample_row"][40:44] = 10_000              # invalid rows: a pixel of dead samples
    ev["m2z"][80] = ev["m1z"][80] * 2.0
    a, b = int(off[4]), int(off[5])
    ev["dL"][a:b] = 1e9                           # an event entirely beyond the table
    ev["dL"][int(off[0]) + 100:int(off[0]) + 103] = ev["dL"][int(off[0]) + 100]   # (nearly) repeated samples
    theta = W.theta.clone()
    theta[3, 8] = 0.0                             # lambda = 0
    theta[4, 7] = -1.0                            # invalid sigma: NaN row + GWC_ERR_DOMAIN
    zmax = W.spec.z_max
    th = theta.to(DEV)
    ctx.gwc_build_cosmo(th, zmax, 1025, 0)
    gL, gP, _ = ctx.gwc_event_loglik_kde(th, to_dev(ev, DEV), W.los.to(DEV), zmax, 256, 0.0)
    with pytest.raises(gwc.GwcError):
        ctx.gwc_check()
    oL, oP = oracle.event_loglik_kde(_np(theta), synth.to_numpy(ev), _np(W.los), zmax)
    _kde_compare((_np(gL), _np(gP)), (oL, oP), "edge cases")
    assert np.all(np.isnan(oL[4])) and np.all(np.isneginf(oL[[0, 1, 2, 3, 5]][:, 2])) and np.all(np.isneginf(oL[0, 4]))
    for bad in (1, 257):
        with pytest.raises(gwc.GwcError):
            ctx.gwc_event_loglik_kde(th, to_dev(ev, DEV), W.los.to(DEV), zmax, bad, 0.0)
    # determinism
    ctx.gwc_build_cosmo(th, zmax, 1025, 0)
    g2 = ctx.gwc_event_loglik_kde(th, to_dev(ev, DEV), W.los.to(DEV), zmax, 256, 0.0)
    try:
        ctx.gwc_check()
    except gwc.GwcError:
        pass
    assert torch.equal(torch.nan_to_num(g2[0], nan=7.0), torch.nan_to_num(gL, nan=7.0)) and torch.equal(g2[1], gP)


# ---- NEXT row 3b: the per-pixel sample cap (R31) -----------------------------------
def test_cap_pixels_bit_exact(ctx):
    """The kept permutation and both offset arrays equal the oracle's, bit for bit, for crowded and sparse pixels,
    several caps and seeds, an empty event and an empty catalogue; the capped catalogue then goes through the hot
    path like any other."""
    from paper_2605_23538_b200 import gwc
    g = torch.Generator().manual_seed(11)
    n, ne = 200_000, 23
    eid = torch.randint(0, ne, (n,), generator=g, dtype=torch.int32)
    eid[eid == 4] = 5                                                       # an empty event
    geo = torch.empty(n).geometric_(0.02, generator=g).to(torch.int32) - 1  # a few crowded pixels, a long tail
    row = torch.clamp(geo, max=900)
    o = oracle.pack_events(eid.numpy(), row.numpy(), ne)
    p = ctx.gwc_pack_events(eid.to(DEV), row.to(DEV), ne)
    sizes = np.diff(o["pix_sample_off"])
    assert sizes.max() > 300 and (sizes == 1).any()
    for cap, seed in ((1, 0), (16, 20260915), (250, 7), (10 ** 9, 3), (16, 2 ** 63 + 5)):
        gp, ge, gx = ctx.gwc_cap_pixels(p, cap, seed)
        op, oe, ox = oracle.cap_pixels(o["perm"], o["ev_sample_off"], o["pix_sample_off"], cap, seed)
        assert np.array_equal(_np(gp), op), (cap, seed)
        assert np.array_equal(_np(ge), oe) and np.array_equal(_np(gx), ox)
    assert np.array_equal(_np(p["perm"]), o["perm"])                        # the packed input was left untouched
    p0 = ctx.gwc_pack_events(eid[:0].to(DEV), row[:0].to(DEV), 3)
    k0, e0, x0 = ctx.gwc_cap_pixels(p0, 5, 1)
    assert k0.numel() == 0 and _np(e0).tolist() == [0, 0, 0, 0]
    with pytest.raises(gwc.GwcError):
        ctx.gwc_cap_pixels(p, 0, 1)
    # a capped catalogue through the hot path: pack + cap the tiny workload's samples, compare with the oracle
    W = workload("tiny")
    off = W.ev["ev_sample_off"]
    ev_id = torch.repeat_interleave(torch.arange(off.numel() - 1, dtype=torch.int32), off[1:] - off[:-1])
    pk = ctx.gwc_pack_events(ev_id.to(DEV), W.ev["sample_row"].to(DEV), off.numel() - 1)
    keep, eso, _ = ctx.gwc_cap_pixels(pk, 20, 5)
    kc = keep.cpu()
    evc = dict(ev_sample_off=eso.cpu(), dL=W.ev["dL"][kc], m1z=W.ev["m1z"][kc], m2z=W.ev["m2z"][kc],
               sample_row=W.ev["sample_row"][kc], log_pe_prior=None)
    assert kc.numel() < W.ev["dL"].numel()
    th = W.theta.to(DEV)
    ctx.gwc_build_cosmo(th, W.spec.z_max, 1025, 0)
    logL, _, nlive = ctx.gwc_event_loglik(th, to_dev(evc, DEV), W.los.to(DEV), W.spec.z_max)
    oL, _, oK = oracle.event_loglik(_np(W.theta), synth.to_numpy(evc), _np(W.los), W.spec.z_max)
    assert np.array_equal(_np(nlive), oK)
    assert_close_log(_np(logL), oL, RTOL_F64, "capped catalogue log L_i")


def test_theta_batch_across_constant_bank_launches(ctx):
    """The fused kernel takes its per-theta constants from the constant bank, 340 points per launch: a batch of 345
    (one full launch + a 5-point one, tiles of 10 cut at 340) must match the oracle point by point."""
    W = workload("tiny", n_theta=345)
    o = _oracle_all(W, W.theta)
    g = _gpu_all(ctx, W, W.theta)
    ctx.gwc_check()
    _compare(g, o)
    # the same points evaluated in another grouping give the same bits (no dependence on the launch split)
    th = W.theta.to(DEV)
    ev, los = to_dev(W.ev, DEV), W.los.to(DEV)
    sub = th[337:345].contiguous()
    ctx.gwc_build_cosmo(sub, W.spec.z_max, 1025, 0)
    logL_sub, _, _ = ctx.gwc_event_loglik(sub, ev, los, W.spec.z_max)
    assert np.array_equal(_np(logL_sub), g["logL"][337:345], equal_nan=True)


def test_kde_32bit_tables(ctx):
    """KDE numerator with f32 LOS rows and the 32-bit cosmology table (R22): against the oracle on the same rounded
    tables (1e-9, pixel counts bit-exact), and within 1e-4 per event of the FP64 result."""
    W = workload("o4", n_theta=8, n_events=6, los_rows=200, n_inj=500)
    los32 = W.los.to(torch.float32)
    g32, o32 = _kde_both(ctx, W, W.theta, los=los32, neff_min=2.0, prec=1)
    assert np.array_equal(g32[1], o32[1])
    assert_close_log(g32[0], o32[0], RTOL_F64, "KDE log L_i, 32-bit tables")
    g64, _ = _kde_both(ctx, W, W.theta, neff_min=2.0, prec=0)
    both = (g32[1] == g64[1]) & np.isfinite(g64[0]) & np.isfinite(g32[0])
    assert both.mean() > 0.9
    assert np.abs(g32[0][both] - g64[0][both]).max() <= ATOL_F32


def test_total_loglik_kde_composition(ctx):
    """gwc_total_loglik_kde = KDE event term + selection term + A6, against the oracle's pieces."""
    W = workload("tiny")
    zmax = W.spec.z_max
    th, ev, inj, los = W.theta.to(DEV), to_dev(W.ev, DEV), to_dev(W.inj, DEV), W.los.to(DEV)
    allsky = ctx.gwc_los_allsky(los, zmax)
    tot = _np(ctx.gwc_total_loglik_kde(th, ev, inj, los, zmax, allsky, 256, 2.0))
    ctx.gwc_check()
    oL, _ = oracle.event_loglik_kde(_np(W.theta), synth.to_numpy(W.ev), _np(W.los), zmax, n_grid=256, neff_min=2.0)
    oX, _ = oracle.selection_logxi(_np(W.theta), synth.to_numpy(W.inj), oracle.los_allsky(_np(W.los), zmax), zmax)
    assert_close_log(tot, oracle.total_from_parts(oL, oX), RTOL_F64, "log L(theta), KDE numerator")
    # composed calls give the same bits
    ctx.gwc_build_cosmo(th, zmax, 1025, 0)
    gL, _, _ = ctx.gwc_event_loglik_kde(th, ev, los, zmax, 256, 2.0)
    gX, _ = ctx.gwc_selection_logxi(th, inj, allsky, los.shape[1], zmax)
    assert np.array_equal(_np(ctx.gwc_combine_total(gL, gX)), tot, equal_nan=True)


def test_kde_silverman_bandwidth(ctx):
    """Eq. D2 on the GPU: the interquartile range by exact selection (bisection on the bit pattern of the live
    redshifts) against the oracle's sort, on pixels of 2 samples to hundreds; and it differs from Scott's rule."""
    from paper_2605_23538_b200 import gwc
    W = workload("o4", n_theta=12, n_events=8, los_rows=400, n_inj=500)
    g, o = _kde_both(ctx, W, W.theta, neff_min=0.0, bandwidth="silverman")
    _kde_compare(g, o, "silverman")
    gs, _ = _kde_both(ctx, W, W.theta, neff_min=0.0, bandwidth="scott")
    fin = np.isfinite(g[0]) & np.isfinite(gs[0])
    assert fin.any() and np.abs(g[0][fin] - gs[0][fin]).max() > 1e-3
    Wt = workload("tiny")
    g, o = _kde_both(ctx, Wt, Wt.theta, neff_min=2.0, bandwidth="silverman")
    _kde_compare(g, o, "silverman tiny")
    th = Wt.theta.to(DEV)
    ctx.gwc_build_cosmo(th, Wt.spec.z_max, 1025, 0)
    with pytest.raises(KeyError):
        ctx.gwc_event_loglik_kde(th, to_dev(Wt.ev, DEV), Wt.los.to(DEV), Wt.spec.z_max, 256, 0.0, "epanechnikov")


@pytest.mark.parametrize("rule", ["biweight", "biweight_scott"])
def test_kde_biweight_bandwidth(ctx, rule):
    """Eq. D3-D4 on the GPU (R37): median and MAD by exact selection on the live redshifts and on their
    absolute deviations, then the two sums; rule "biweight" takes h = D3 as printed (narrow kernels: the direct
    path of the KDE pass), "biweight_scott" puts sqrt(D3) into Scott's rule.  Pixels of 2 samples to hundreds,
    duplicated redshifts (MAD = 0: no bandwidth) included."""
    W = workload("o4", n_theta=12, n_events=8, los_rows=400, n_inj=500)
    ev = dict(W.ev)
    dl = ev["dL"].clone()
    dl[40:52] = dl[40]            # a run of identical samples inside one event
    ev["dL"] = dl
    ev["m1z"] = ev["m1z"].clone()
    ev["m1z"][40:52] = ev["m1z"][40]
    ev["m2z"] = ev["m2z"].clone()
    ev["m2z"][40:52] = ev["m2z"][40]
    for nmin in (0.0, 2.0):
        g, o = _kde_both(ctx, W, W.theta, ev=ev, neff_min=nmin, bandwidth=rule)
        _kde_compare(g, o, "%s nmin=%g" % (rule, nmin))
        assert (o[1] > 0).any()
    gs, _ = _kde_both(ctx, W, W.theta, ev=ev, neff_min=0.0, bandwidth="scott")
    fin = np.isfinite(g[0]) & np.isfinite(gs[0])
    assert fin.any() and np.abs(g[0][fin] - gs[0][fin]).max() > 1e-3
    Wt = workload("tiny")
    g, o = _kde_both(ctx, Wt, Wt.theta, neff_min=2.0, bandwidth=rule)
    _kde_compare(g, o, rule + " tiny")


def test_catalogue_cache_and_small_batches(ctx):
    """Latency mode: with the catalogue cache on, repeated small-batch calls (1, 2, 3, 5 theta: odd counts take the
    tail-only kernel variant) give the bits of the uncached calls; changing an array and presenting another pointer
    recomputes; turning the cache off forgets."""
    W = workload("tiny", n_theta=9)
    zmax = W.spec.z_max
    ev, inj, los = to_dev(W.ev, DEV), to_dev(W.inj, DEV), W.los.to(DEV)
    allsky = ctx.gwc_los_allsky(los, zmax)
    o = _oracle_all(W, W.theta)
    ref = {}
    for nt in (1, 2, 3, 5, 9):
        th = W.theta[:nt].to(DEV)
        ref[nt] = _np(ctx.gwc_total_loglik(th, ev, inj, los, zmax, allsky))
        assert_close_log(ref[nt], o["total"][:nt], RTOL_F64, "log L(theta), %d theta" % nt)
    ctx.gwc_cache_catalogue(True)
    try:
        n0 = ctx.gwc_launch_count()
        ctx.gwc_total_loglik(W.theta[:1].to(DEV), ev, inj, los, zmax, allsky)
        first = ctx.gwc_launch_count() - n0
        for nt in (1, 2, 3, 5, 9, 1):
            th = W.theta[:nt].to(DEV)
            n0 = ctx.gwc_launch_count()
            got = _np(ctx.gwc_total_loglik(th, ev, inj, los, zmax, allsky))
            assert np.array_equal(got, ref[nt], equal_nan=True)
            if nt == 1:
                assert ctx.gwc_launch_count() - n0 == first - 2       # the two preparation kernels are skipped
        # another array (new pointer, new contents): recomputed
        ev2 = dict(ev, dL=(ev["dL"] * 1.01))
        th = W.theta[:3].to(DEV)
        got2 = _np(ctx.gwc_total_loglik(th, ev2, inj, los, zmax, allsky))
        ev2_cpu = dict(W.ev, dL=W.ev["dL"] * 1.01)
        o2 = oracle.total_loglik(_np(W.theta[:3]), synth.to_numpy(ev2_cpu), synth.to_numpy(W.inj), _np(W.los), zmax)
        assert_close_log(got2, o2, RTOL_F64, "after a new d_L array")
    finally:
        ctx.gwc_cache_catalogue(False)
    got = _np(ctx.gwc_total_loglik(W.theta[:5].to(DEV), ev, inj, los, zmax, allsky))
    assert np.array_equal(got, ref[5], equal_nan=True)


def test_total_loglik_pixcut(ctx):
    """gwc_total_loglik_pixcut = the composed calls, bit for bit, and the oracle's pieces at the FP64 bar; threshold 0
    agrees with gwc_total_loglik to rounding."""
    W = workload("o4", n_theta=14, n_events=7, los_rows=400, n_inj=5000)
    zmax = W.spec.z_max
    th, ev, inj, los = W.theta.to(DEV), to_dev(W.ev, DEV), to_dev(W.inj, DEV), W.los.to(DEV)
    allsky = ctx.gwc_los_allsky(los, zmax)
    tot = ctx.gwc_total_loglik_pixcut(th, ev, inj, los, zmax, allsky, 2.0)
    ctx.gwc_build_cosmo(th, zmax)
    gL = ctx.gwc_event_loglik_pixcut(th, ev, los, zmax, 2.0)[0]
    gX, _ = ctx.gwc_selection_logxi(th, inj, allsky, los.shape[1], zmax)
    assert np.array_equal(_np(ctx.gwc_combine_total(gL, gX)), _np(tot), equal_nan=True)
    ctx.gwc_check()
    oL = oracle.event_loglik_pixcut(_np(W.theta), synth.to_numpy(W.ev), _np(W.los), zmax, 2.0)[0]
    oX, _ = oracle.selection_logxi(_np(W.theta), synth.to_numpy(W.inj), oracle.los_allsky(_np(W.los), zmax), zmax)
    assert_close_log(_np(tot), oracle.total_from_parts(oL, oX), RTOL_F64, "log L(theta) with the pixel cut")
    t0 = ctx.gwc_total_loglik_pixcut(th, ev, inj, los, zmax, allsky, 0.0)
    t1 = ctx.gwc_total_loglik(th, ev, inj, los, zmax, allsky)
    assert_close_log(_np(t0), _np(t1), 1e-13, "threshold 0 against the uncut total")
