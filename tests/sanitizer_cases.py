"""Small-case driver for every kernel variant of the library ("Race detection"): the tiny config
and ragged mini-catalogues, each result checked against the oracle.  compute-sanitizer is closed on the GPU pool this
repo is measured on (its refusal is kept in profiles/r02_sanitizer.md), so the evidence asked of
memcheck / racecheck / initcheck is gathered the other way: the library built with -DGWC_CHECKED (device-side bounds
checks on every table / row / sample / accumulator index, the invariants of the barrier-free segment hand-off -- a sum
buffer must be clear when a warp starts adding to it, the arrival count must be NWARPS and segments must be combined in
order -- and scratch memory poisoned with 0xff on allocation; a violation raises GWC_ERR_CUDA through gwc_check) runs
these cases,

    GWC_NVCC_FLAGS=-DGWC_CHECKED python -m paper_2605_23538_b200.build --force && python tests/sanitizer_cases.py

Not collected by pytest (no test_ prefix).  Cases: events (plain kernel, barrier-free segment hand-off), teams (short
segments share the CTA), odd (tail-only last step), pix (per-pixel N_eff cut), inj (selection term), t32 (32-bit
tables, f32 LOS rows), kde (every bandwidth rule), pack (A0 + cap + all-sky), host (gwc_total_loglik_host), mp (the
MULTIPEAK variants of the fused kernel and of the KDE kernel), repeat (the plain and the TEAMS kernel 20 times over:
bit-identical results, the check a race would fail).
"""
from __future__ import annotations

import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

import oracle  # noqa: E402
from paper_2605_23538_b200 import gwc, synth  # noqa: E402
from util import RTOL_F64, assert_close_log, to_dev, workload  # noqa: E402

DEV = "cuda:0"


def _np(t):
    return t.detach().cpu().numpy()


def _ragged(n_theta, long_events):
    """Ragged mini-catalogue: a box-6 theta batch (every theta its own Om); long events (>= 2048 samples on average:
    the plain kernel) or short ones (the TEAMS kernel)."""
    if long_events:
        return workload("production", n_theta=n_theta, n_events=3, los_rows=300, n_inj=9000, samples=(2100, 3300),
                        pixels=(16, 200))
    return workload("production", n_theta=n_theta, n_events=9, los_rows=300, n_inj=9000, samples=(40, 1500),
                    pixels=(4, 100))


def _events(ctx, W, prec=0, los=None, what=""):
    los = W.los if los is None else los
    zmax = W.spec.z_max
    th, ev, lo = W.theta.to(DEV), to_dev(W.ev, DEV), los.to(DEV)
    ctx.gwc_build_cosmo(th, zmax, 1025, prec)
    logL, neff, nlive = ctx.gwc_event_loglik(th, ev, lo, zmax)
    ctx.gwc_check()
    oL, oN, oK = oracle.event_loglik(_np(W.theta), synth.to_numpy(W.ev), _np(los), zmax, table_prec=prec)
    assert np.array_equal(_np(nlive), oK), what
    assert_close_log(_np(logL), oL, RTOL_F64, what)


def case_events(ctx):
    _events(ctx, _ragged(12, True), what="events, plain kernel")


def case_teams(ctx):
    _events(ctx, workload("tiny"), what="events, tiny (teams)")
    _events(ctx, _ragged(12, False), what="events, short ragged (teams)")


def case_odd(ctx):
    _events(ctx, _ragged(3, True), what="events, 3 theta (odd)")
    W = _ragged(1, False)
    _events(ctx, W, what="events, 1 theta (odd)")
    zmax = W.spec.z_max
    th, inj, lo = W.theta.to(DEV), to_dev(W.inj, DEV), W.los.to(DEV)
    allsky = ctx.gwc_los_allsky(lo, zmax)
    ctx.gwc_build_cosmo(th, zmax, 1025, 0)
    logxi, _ = ctx.gwc_selection_logxi(th, inj, allsky, lo.shape[1], zmax)
    ctx.gwc_check()
    oX, _ = oracle.selection_logxi(_np(W.theta), synth.to_numpy(W.inj), oracle.los_allsky(_np(W.los), zmax), zmax)
    assert_close_log(_np(logxi), oX, RTOL_F64, "log xi, 1 theta (odd)")


def case_pix(ctx):
    for W in (workload("tiny"), _ragged(12, True), _ragged(5, False)):
        zmax = W.spec.z_max
        th, ev, lo = W.theta.to(DEV), to_dev(W.ev, DEV), W.los.to(DEV)
        ctx.gwc_build_cosmo(th, zmax, 1025, 0)
        gL, gN, gK, gP = ctx.gwc_event_loglik_pixcut(th, ev, lo, zmax, 2.0)
        ctx.gwc_check()
        oL, oN, oK, oP = oracle.event_loglik_pixcut(_np(W.theta), synth.to_numpy(W.ev), _np(W.los), zmax, 2.0)
        assert np.array_equal(_np(gP), oP) and np.array_equal(_np(gK), oK)
        assert_close_log(_np(gL), oL, RTOL_F64, "pixcut")


def case_inj(ctx):
    for W in (workload("tiny"), _ragged(12, True)):
        zmax = W.spec.z_max
        th, inj, lo = W.theta.to(DEV), to_dev(W.inj, DEV), W.los.to(DEV)
        allsky = ctx.gwc_los_allsky(lo, zmax)
        ctx.gwc_build_cosmo(th, zmax, 1025, 0)
        logxi, _ = ctx.gwc_selection_logxi(th, inj, allsky, lo.shape[1], zmax)
        total = ctx.gwc_total_loglik(th, to_dev(W.ev, DEV), inj, lo, zmax, allsky)
        ctx.gwc_check()
        oX, _ = oracle.selection_logxi(_np(W.theta), synth.to_numpy(W.inj), oracle.los_allsky(_np(W.los), zmax), zmax)
        assert_close_log(_np(logxi), oX, RTOL_F64, "log xi")
        oT = oracle.total_loglik(_np(W.theta), synth.to_numpy(W.ev), synth.to_numpy(W.inj), _np(W.los), zmax)
        assert_close_log(_np(total), oT, RTOL_F64, "log L(theta)")


def case_t32(ctx):
    W = _ragged(12, True)
    _events(ctx, W, prec=1, los=W.los.to(torch.float32), what="events, 32-bit tables")


def case_kde(ctx):
    W = workload("tiny", n_theta=4)
    zmax = W.spec.z_max
    th, ev, lo = W.theta.to(DEV), to_dev(W.ev, DEV), W.los.to(DEV)
    ctx.gwc_build_cosmo(th, zmax, 1025, 0)
    for bw in gwc.BW_RULES:
        gL, gP, gU = ctx.gwc_event_loglik_kde(th, ev, lo, zmax, 64, 2.0, bw)
        ctx.gwc_check()
        oL, oP, oU = oracle.event_loglik_kde(_np(W.theta), synth.to_numpy(W.ev), _np(W.los), zmax, n_grid=64,
                                             neff_min=2.0, bandwidth=bw, want_nused=True)
        assert np.array_equal(_np(gP), oP) and np.array_equal(_np(gU), oU), bw
        assert_close_log(_np(gL), oL, RTOL_F64, "KDE %s" % bw)


def case_pack(ctx):
    g = torch.Generator().manual_seed(3)
    eid = torch.randint(0, 7, (5000,), generator=g, dtype=torch.int32)
    row = torch.randint(0, 60, (5000,), generator=g, dtype=torch.int32)
    p = ctx.gwc_pack_events(eid.to(DEV), row.to(DEV), 7)
    o = oracle.pack_events(eid.numpy(), row.numpy(), 7)
    for k in ("perm", "ev_sample_off", "ev_pix_off"):
        assert np.array_equal(_np(p[k]), o[k]), k
    ctx.gwc_cap_pixels(p, 5, 1)
    W = workload("tiny")
    a = ctx.gwc_los_allsky(W.los.to(DEV), W.spec.z_max)
    np.testing.assert_allclose(_np(a), oracle.los_allsky(_np(W.los), W.spec.z_max), rtol=1e-13)


def case_host(ctx):
    W = workload("tiny")
    zmax = W.spec.z_max
    a, _, _ = ctx.gwc_total_loglik_host(W.theta, W.ev, W.inj, W.los, zmax)
    o = oracle.total_loglik(_np(W.theta), synth.to_numpy(W.ev), synth.to_numpy(W.inj), _np(W.los), zmax)
    assert_close_log(a.numpy(), o, RTOL_F64, "host call")


def case_mp(ctx):
    ctx.gwc_set_mass_model("multipeak")
    try:
        W = _ragged(9, True)
        th = synth.make_theta_multipeak(W.spec, synth.DEFAULT_SEED, "cpu", 9)
        ev = dict(W.ev)
        ev["m1z"], ev["m2z"] = ev["m1z"] * 0.2, ev["m2z"] * 0.2   # into the smoothing window
        zmax = W.spec.z_max
        thd, evd, lo = th.to(DEV), to_dev(ev, DEV), W.los.to(DEV)
        ctx.gwc_build_cosmo(thd, zmax, 1025, 0)
        gL, _, gK = ctx.gwc_event_loglik(thd, evd, lo, zmax)
        qL, _, qK, qP = ctx.gwc_event_loglik_pixcut(thd, evd, lo, zmax, 2.0)
        kL, kP, kU = ctx.gwc_event_loglik_kde(thd, evd, lo, zmax, 64, 2.0, "scott")
        ctx.gwc_check()
        with oracle.mass_model("multipeak"):
            oL, _, oK = oracle.event_loglik(_np(th), synth.to_numpy(ev), _np(W.los), zmax)
            pL, _, pK, pP = oracle.event_loglik_pixcut(_np(th), synth.to_numpy(ev), _np(W.los), zmax, 2.0)
            rL, rP = oracle.event_loglik_kde(_np(th), synth.to_numpy(ev), _np(W.los), zmax, n_grid=64, neff_min=2.0)
        assert np.array_equal(_np(gK), oK) and np.array_equal(_np(qP), pP) and np.array_equal(_np(kP), rP)
        assert_close_log(_np(gL), oL, RTOL_F64, "MULTIPEAK events")
        assert_close_log(_np(qL), pL, RTOL_F64, "MULTIPEAK pixcut")
        assert_close_log(_np(kL), rL, RTOL_F64, "MULTIPEAK KDE")
    finally:
        ctx.gwc_set_mass_model("plpeak")


def case_repeat(ctx):
    for W in (_ragged(12, True), _ragged(12, False)):
        zmax = W.spec.z_max
        th, ev, lo = W.theta.to(DEV), to_dev(W.ev, DEV), W.los.to(DEV)
        ctx.gwc_build_cosmo(th, zmax, 1025, 0)
        first = None
        for _ in range(20):
            logL, neff, nlive = ctx.gwc_event_loglik(th, ev, lo, zmax)
            ctx.gwc_check()
            got = (logL.clone(), neff.clone(), nlive.clone())
            if first is None:
                first = got
            assert all(torch.equal(a.view(torch.int64), b.view(torch.int64)) for a, b in zip(first, got))


CASES = {"events": case_events, "teams": case_teams, "odd": case_odd, "pix": case_pix, "inj": case_inj,
         "t32": case_t32, "kde": case_kde, "pack": case_pack, "host": case_host, "mp": case_mp, "repeat": case_repeat}


def main(argv):
    names = argv or list(CASES)
    ctx = gwc.Context(0)
    for n in names:
        CASES[n](ctx)
        torch.cuda.synchronize()
        print("case %-7s ok (parity with the oracle)" % n, flush=True)
    print("sanitizer_cases: %d case(s) done, %d kernel launches" % (len(names), ctx.gwc_launch_count()), flush=True)
    ctx.close()


if __name__ == "__main__":
    main(sys.argv[1:])
