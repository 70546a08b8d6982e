"""Pins for the CPU oracle (no GPU).  Each test fixes the oracle to something other than itself:
closed forms, scipy quadrature, brute force, invariances the mathematics demands.
Citations: PAPER.md line numbers; readings R# are in DESIGN.md section 3."""
import math
import os

import numpy as np
import pytest
from scipy import integrate, special

import oracle as O

C = 299792.458
GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _gold():
    rows = []
    for line in open(os.path.join(GOLD, "survey_checks.txt")):
        line = line.split("--")[0].strip()
        if line and not line.startswith("#"):
            p = line.split()
            rows.append((p[0], [float(x) for x in p[1:]]))
    return rows


# ---------------------------------------------------------------- cosmology, Eq. 1
@pytest.mark.parametrize("z", [1e-4, 0.01, 0.3, 1.0, 2.0, 7.5])
def test_dL_closed_form_matter_only(z):
    # Om = 1: d_L = 2c(1+z)(1-(1+z)^-1/2)/H0   (north_star closed form)
    ref = 2 * C * (1 + z) * (1 - (1 + z) ** -0.5) / 70.0
    assert O.dL(z, 70.0, 1.0) == pytest.approx(ref, rel=2e-15)


@pytest.mark.parametrize("z", [1e-4, 0.01, 0.3, 1.0, 2.0, 7.5])
def test_dL_closed_form_lambda_only(z):
    # Om = 0 (Omega_Lambda = 1): d_L = c z (1+z)/H0
    assert O.dL(z, 55.0, 0.0) == pytest.approx(C * z * (1 + z) / 55.0, rel=2e-15)


@pytest.mark.parametrize("H0,Om,z", [(70, 0.3, 0.1), (70, 0.3, 1.0), (70, 0.3, 2.0), (67.4, 0.315, 1.0),
                                     (20, 0.1, 1.5), (140, 0.5, 1.5), (200, 0.25, 0.02)])
def test_dL_against_scipy_quad(H0, Om, z):
    val, _ = integrate.quad(lambda x: 1.0 / math.sqrt(Om * (1 + x) ** 3 + 1 - Om), 0, z, epsabs=0, epsrel=1e-13)
    assert O.dL(z, H0, Om) == pytest.approx((1 + z) * C / H0 * val, rel=1e-12)


def test_golden_survey_values(theta0):
    for kind, a in _gold():
        if kind == "dL":
            assert O.dL(a[0], a[1], a[2]) == pytest.approx(a[3], rel=1e-12)
        elif kind == "u":
            assert O.u_of_z(a[0], a[1]) == pytest.approx(a[2], rel=1e-12)
        elif kind == "ddLdz":
            z, H0, Om = a[:3]
            h = 1e-5
            fd = (O.dL(z + h, H0, Om) - O.dL(z - h, H0, Om)) / (2 * h)
            assert fd == pytest.approx(a[3], rel=1e-8)
        elif kind == "lnp":
            m1, m2 = a[0], a[1]
            assert math.log(O.p1(m1, theta0) * O.p2(m2, m1, theta0)) == pytest.approx(a[2], abs=2e-12)
        elif kind == "npl":
            assert O.norm_pl(theta0) == pytest.approx(a[0], rel=1e-11)
        elif kind == "ng":
            assert O.norm_g(theta0) == pytest.approx(a[0], rel=1e-11)
        elif kind == "psi":
            th = theta0.copy()
            th[9:12] = a[1:4]
            assert O.psi(a[0], th) == pytest.approx(a[4], rel=1e-12)


@pytest.mark.parametrize("Om", [0.05, 0.3, 0.5, 1.0])
def test_z_of_dL_round_trip_exact(Om):
    for z in [1e-6, 0.003, 0.2, 0.9, 1.7, 4.0]:
        for H0 in (20.0, 70.0, 200.0):
            assert O.z_of_dL(O.dL(z, H0, Om), H0, Om) == pytest.approx(z, rel=1e-12, abs=1e-15)


@pytest.mark.parametrize("Om,bound", [(0.3, 5e-11), (0.1, 2e-10), (0.5, 5e-11)])
def test_hermite_table_nodes_and_error(Om, bound):
    # reading R9: nodes are exact inverses; cubic Hermite error bounds measured in SURVEY 8c item 9
    zt, dt, um = O.build_table(Om, 2.0, 1025)
    assert zt[0] == 0.0 and zt[-1] == 2.0
    assert np.all(np.diff(zt) > 0) and np.all(dt > 0)
    du = um / 1024
    for m in (1, 7, 300, 777, 1023):
        assert O.u_of_z(zt[m], Om) == pytest.approx(m * du, rel=1e-13)
        assert O.z_table(m * du, zt, dt, um) == pytest.approx(zt[m], abs=4e-15)  # exact at nodes
        # slope: dz/du by central difference of the exact inverse
        h = 1e-6
        fd = (O.z_of_u(m * du + h, Om) - O.z_of_u(m * du - h, Om)) / (2 * h)
        assert dt[m] / du == pytest.approx(fd, rel=1e-8)
    rng = np.random.default_rng(1)
    err = max(abs(O.z_table(u, zt, dt, um) - O.z_of_u(u, Om)) for u in rng.uniform(0, um, 1500))
    assert err < bound
    assert O.z_table(um, zt, dt, um) is None and O.z_table(1.5 * um, zt, dt, um) is None  # u >= umax dead (R11)


# ---------------------------------------------------------------- population (readings R2-R4)
@pytest.mark.parametrize("th_mod", [{}, {2: 1.5, 6: 25.0, 7: 2.0, 8: 0.1}, {2: 5.0, 6: 45.0, 7: 8.0, 8: 0.0},
                                    {4: 4.6, 5: 86.3, 2: 2.9, 6: 30.7, 7: 6.3, 8: 0.4}])
def test_p1_normalised(theta0, th_mod):
    th = theta0.copy()
    for k, v in th_mod.items():
        th[k] = v
    val, _ = integrate.quad(lambda m: O.p1(m, th), th[4], th[5], points=[th[6]], epsabs=0, epsrel=1e-12, limit=400)
    assert val == pytest.approx(1.0, abs=1e-10)
    assert O.p1(th[4], th) == 0.0 and O.p1(th[5], th) > 0.0 and O.p1(th[5] * (1 + 1e-15) + 1e-9, th) == 0.0  # R15


@pytest.mark.parametrize("beta", [1.1, 0.0, -0.5, 4.0, -1.0])
def test_p2_normalised(theta0, beta):
    th = theta0.copy()
    th[3] = beta
    for m1 in (5.5, 30.0, 100.0):
        val, _ = integrate.quad(lambda m: O.p2(m, m1, th), th[4], m1, epsabs=0, epsrel=1e-12)
        assert val == pytest.approx(1.0, abs=1e-10)
    assert O.p2(th[4], 30.0, th) > 0 and O.p2(30.0, 30.0, th) > 0 and O.p2(30.0001, 30.0, th) == 0.0  # R15


def test_p1_lambda0_pure_power_law(theta0):
    th = theta0.copy()
    th[8] = 0.0
    a, lo, hi = th[2], th[4], th[5]
    for m in (5.1, 20.0, 99.0):
        ref = (1 - a) / (hi ** (1 - a) - lo ** (1 - a)) * m ** (-a)
        assert O.p1(m, th) == pytest.approx(ref, rel=1e-14)


def test_p1_peak_term(theta0):
    # lambda = 1: pure truncated Gaussian, compare against scipy's erf-normalised density
    th = theta0.copy()
    th[8] = 1.0
    mu, s, lo, hi = th[6], th[7], th[4], th[5]
    Z = 0.5 * (special.erf((hi - mu) / (s * math.sqrt(2))) - special.erf((lo - mu) / (s * math.sqrt(2))))
    for m in (20.0, 35.0, 50.0):
        ref = math.exp(-0.5 * ((m - mu) / s) ** 2) / (s * math.sqrt(2 * math.pi)) / Z
        assert O.p1(m, th) == pytest.approx(ref, rel=1e-13)


def test_rate(theta0):
    assert O.psi(0.0, theta0) == pytest.approx(1.0, rel=1e-15)
    # low-z slope gamma, high-z slope -kappa (Madau-Dickinson)
    g, k, zp = theta0[9:12]
    assert math.log(O.psi(1e-3, theta0)) / math.log1p(1e-3) == pytest.approx(g, abs=2e-2)
    z1, z2 = 400.0, 800.0
    slope = (math.log(O.psi(z2, theta0)) - math.log(O.psi(z1, theta0))) / (math.log1p(z2) - math.log1p(z1))
    assert slope == pytest.approx(-k, abs=1e-3)


def test_theta_domain(theta0):
    assert O.theta_valid(theta0)
    for idx, bad in [(0, 0.0), (0, -1.0), (1, 0.0), (1, 1.2), (7, 0.0), (4, 100.0), (4, -1.0), (8, -0.1), (8, 1.1),
                     (2, float("nan"))]:
        th = theta0.copy()
        th[idx] = bad
        assert not O.theta_valid(th)


# ---------------------------------------------------------------- LOS interpolation (reading R10)
def test_los_lerp():
    rng = np.random.default_rng(3)
    nz, zmax = 64, 1.5
    zb = np.linspace(0, zmax, nz)
    tab = np.stack([2.0 + 3.0 * zb, rng.uniform(0.1, 1, nz)])
    for b in (0, 1, 17, 62):
        assert O.los_lerp(tab, zmax, 1, zb[b]) == pytest.approx(tab[1, b], rel=1e-13)
    for z in rng.uniform(0, zmax, 50):
        assert O.los_lerp(tab, zmax, 0, z) == pytest.approx(2.0 + 3.0 * z, rel=1e-14)       # exact for linear
        assert O.los_lerp(tab, zmax, 1, z) == pytest.approx(np.interp(z, zb, tab[1]), rel=1e-12)
    t32 = tab.astype(np.float32)
    for z in rng.uniform(0, zmax, 50):
        assert O.los_lerp(t32, zmax, 1, z) == pytest.approx(O.los_lerp(tab, zmax, 1, z), rel=2.0 ** -23)
    a = O.los_allsky(tab, zmax)
    np.testing.assert_allclose(a, tab.mean(0), rtol=1e-15)


# ---------------------------------------------------------------- LSE / N_eff (Eq. 8)
def test_lse_properties():
    rng = np.random.default_rng(5)
    lw = rng.normal(-30, 3, 257)
    l, n = O.lse(lw)
    w = np.exp(lw)
    assert l == pytest.approx(math.log(w.sum()), rel=1e-14)
    assert n == pytest.approx(w.sum() ** 2 / (w ** 2).sum(), rel=1e-13)
    l2, n2 = O.lse(rng.permutation(lw))
    assert l2 == pytest.approx(l, rel=1e-15) and n2 == pytest.approx(n, rel=1e-13)
    l3, n3 = O.lse(lw + 7.25)
    assert l3 == pytest.approx(l + 7.25, rel=1e-15) and n3 == pytest.approx(n, rel=1e-13)
    l4, n4 = O.lse(np.concatenate([lw, lw]))
    assert l4 == pytest.approx(l + math.log(2), rel=1e-15) and n4 == pytest.approx(2 * n, rel=1e-13)
    l5, n5 = O.lse(np.full(100, -3.0))
    assert l5 == pytest.approx(-3.0 + math.log(100)) and n5 == pytest.approx(100.0)
    l6, n6 = O.lse(np.array([0.0, -800.0, -900.0]))
    assert l6 == pytest.approx(0.0, abs=1e-300) and n6 == pytest.approx(1.0)
    l7, n7 = O.lse(np.full(4, -np.inf))
    assert l7 == -np.inf and n7 == 0.0
    l8, _ = O.lse(np.array([-np.inf, -2.0]))
    assert l8 == pytest.approx(-2.0)
    # far outside the range of a double in linear space
    l9, _ = O.lse(np.array([-5000.0, -5000.0]))
    assert l9 == pytest.approx(-5000.0 + math.log(2))


# ---------------------------------------------------------------- whole weight: invariances
def _toy_event(n=300, seed=11, zmax=1.5, nz=128, rows=4):
    rng = np.random.default_rng(seed)
    dl = 1500.0 * np.exp(0.25 * rng.standard_normal(n))
    m1z = 45.0 * (1 + 0.08 * rng.standard_normal(n))
    m2z = 33.0 * (1 + 0.08 * rng.standard_normal(n))
    m1z, m2z = np.maximum(m1z, m2z), np.minimum(m1z, m2z)
    row = np.sort(rng.integers(0, rows, n)).astype(np.int32)
    tab = rng.uniform(0.2, 2.0, (rows, nz))
    ev = dict(ev_sample_off=np.array([0, n // 3, n], dtype=np.int64), dL=dl, m1z=m1z, m2z=m2z, sample_row=row,
              log_pe_prior=None)
    return ev, tab, zmax


@pytest.mark.parametrize("mode", [O.TABLE, O.EXACT])
def test_H0_scaling_invariance(theta0, mode):
    # Om fixed: (H0 -> s H0, dL -> dL/s) leaves z unchanged, adds 3 ln s to every live log w under the dL^2 prior
    ev, tab, zmax = _toy_event()
    s = 1.37
    th2 = theta0.copy()
    th2[0] *= s
    ev2 = dict(ev, dL=ev["dL"] / s)
    L1, n1, k1 = O.event_loglik(theta0, ev, tab, zmax, mode=mode)
    L2, n2, k2 = O.event_loglik(th2, ev2, tab, zmax, mode=mode)
    np.testing.assert_allclose(L2, L1 + 3 * math.log(s), rtol=0, atol=2e-12)
    np.testing.assert_allclose(n2, n1, rtol=1e-11)
    assert np.array_equal(k1, k2)
    # with an explicit prior passed unchanged the shift is 1 ln s
    lpe = 2 * np.log(ev["dL"])
    L3, _, _ = O.event_loglik(th2, dict(ev2, log_pe_prior=lpe), tab, zmax, mode=mode)
    np.testing.assert_allclose(L3, L1 + 1 * math.log(s), rtol=0, atol=2e-12)


def test_padding_and_permutation_invariance(theta0):
    # "padded indices do not contribute anything": zero-weight samples change log L_i by -log((S+p)/S)
    ev, tab, zmax = _toy_event()
    L1, n1, k1 = O.event_loglik(theta0, ev, tab, zmax)
    n = ev["dL"].size
    pad = 57
    ev2 = dict(ev_sample_off=np.array([0, n // 3, n + pad], dtype=np.int64),
               dL=np.concatenate([ev["dL"], np.full(pad, 1e7)]),          # beyond the z table: dead (R11)
               m1z=np.concatenate([ev["m1z"], np.full(pad, 40.0)]), m2z=np.concatenate([ev["m2z"], np.full(pad, 30.0)]),
               sample_row=np.concatenate([ev["sample_row"], np.zeros(pad, np.int32)]), log_pe_prior=None)
    L2, n2, k2 = O.event_loglik(theta0, ev2, tab, zmax)
    S1 = n - n // 3
    assert L2[0, 0] == pytest.approx(L1[0, 0], abs=1e-13)
    assert L2[0, 1] == pytest.approx(L1[0, 1] - math.log((S1 + pad) / S1), abs=1e-12)
    assert n2[0, 1] == pytest.approx(n1[0, 1], rel=1e-12) and k2[0, 1] == k1[0, 1]
    # permutation of the samples inside an event
    rng = np.random.default_rng(0)
    p = np.concatenate([rng.permutation(n // 3), n // 3 + rng.permutation(S1)])
    ev3 = dict(ev, dL=ev["dL"][p], m1z=ev["m1z"][p], m2z=ev["m2z"][p], sample_row=ev["sample_row"][p])
    L3, n3, k3 = O.event_loglik(theta0, ev3, tab, zmax)
    np.testing.assert_allclose(L3, L1, rtol=0, atol=1e-12)
    assert np.array_equal(k3, k1)


def test_dead_samples_and_bad_theta(theta0):
    ev, tab, zmax = _toy_event()
    ev = dict(ev)
    n = ev["dL"].size
    a = n // 3
    # every way a sample can be dead: none may give NaN or touch memory out of range
    ev["dL"] = ev["dL"].copy(); ev["m1z"] = ev["m1z"].copy(); ev["m2z"] = ev["m2z"].copy()
    ev["sample_row"] = ev["sample_row"].copy()
    ev["dL"][0] = np.nan; ev["dL"][1] = -5.0; ev["m1z"][2] = np.inf; ev["m2z"][3] = 0.0
    ev["sample_row"][4] = -1; ev["sample_row"][5] = 99; ev["m1z"][6] = 1.0; ev["m1z"][7] = 1e4; ev["dL"][8] = 1e9
    L, ne, k = O.event_loglik(theta0, ev, tab, zmax)
    assert np.all(np.isfinite(L)) and k[0, 0] <= a - 9
    # all dead => -inf, N_eff 0, and the total is -inf, never NaN
    ev["m1z"][:a] = 1.0
    L, ne, k = O.event_loglik(theta0, ev, tab, zmax)
    assert L[0, 0] == -np.inf and ne[0, 0] == 0.0 and k[0, 0] == 0 and np.isfinite(L[0, 1])
    tot = O.total_from_parts(L, np.array([-3.0]))
    assert tot[0] == -np.inf
    bad = theta0.copy(); bad[7] = -1.0
    L, ne, k = O.event_loglik(np.stack([theta0, bad]), ev, tab, zmax)
    assert np.all(np.isnan(L[1])) and not np.any(np.isnan(L[0]))
    assert np.isnan(O.total_from_parts(L, np.array([-3.0, -3.0]))[1])


def test_table_vs_exact_mode(theta0):
    ev, tab, zmax = _toy_event(n=600)
    for H0 in (40.0, 70.0, 110.0):
        th = theta0.copy(); th[0] = H0
        Lt, _, kt = O.event_loglik(th, ev, tab, zmax, mode=O.TABLE)
        Le, _, ke = O.event_loglik(th, ev, tab, zmax, mode=O.EXACT)
        np.testing.assert_allclose(Lt, Le, rtol=0, atol=3e-10)     # Hermite M=1025 (<= 3e-11 measured)
        assert np.array_equal(kt, ke)


def test_total_composition():
    # Eq. 3: log L = sum_i log L_i - N_det log xi
    L = np.array([[-1.0, -2.0, -3.5], [0.5, 0.25, -0.125]])
    xi = np.array([-4.0, 2.0])
    np.testing.assert_allclose(O.total_from_parts(L, xi), [-6.5 + 12.0, 0.625 - 6.0], rtol=1e-15)


# ---------------------------------------------------------------- whole estimator: Monte-Carlo toy vs quadrature
def test_mc_estimator_converges_to_source_frame_quadrature(theta0):
    """north_star's 1-event toy.  Samples ~ g(dL) g1(m1z) g2(m2z) (posterior under the dL^2 prior).  The estimator
    (1/S) sum w must converge to I = int dz R(z) p_los(z) g_d(dL(z))/dL(z)^2 int dm1 p1 g1(m1(1+z)) int dm2 p2 g2(m2(1+z)),
    written in SOURCE-frame coordinates: it contains no Jacobian, so it checks J's form and direction (Eq. 7, R6)."""
    rng = np.random.default_rng(2024)
    S = 400_000
    mu_d, s_d = math.log(2000.0), 0.2
    dl = np.exp(mu_d + s_d * rng.standard_normal(S))
    m1z = 45.0 + 2.25 * rng.standard_normal(S)
    m2z = 36.0 + 1.8 * rng.standard_normal(S)
    zmax, nz = 1.5, 512
    zb = np.linspace(0, zmax, nz)
    row = 0.4 + 0.3 * np.sin(5 * zb) + 2.0 * np.exp(-0.5 * ((zb - 0.38) / 0.02) ** 2)   # a galaxy spike on a smooth floor
    tab = row[None, :].copy()
    ev = dict(ev_sample_off=np.array([0, S], dtype=np.int64), dL=dl, m1z=m1z, m2z=m2z,
              sample_row=np.zeros(S, np.int32), log_pe_prior=None)
    L, neff, nlive = O.event_loglik(theta0, ev, tab, zmax, mode=O.EXACT)
    mc = math.exp(L[0, 0])
    stderr_rel = math.sqrt(1.0 / neff[0, 0] - 1.0 / S)

    H0, Om = theta0[0], theta0[1]
    norm = lambda x, m, s: np.exp(-0.5 * ((x - m) / s) ** 2) / (s * math.sqrt(2 * math.pi))
    xg, wg = np.polynomial.legendre.leggauss(48)

    def gl(f, a, b):
        return 0.5 * (b - a) * sum(w * f(0.5 * (b - a) * x + 0.5 * (a + b)) for x, w in zip(xg, wg))

    def mass_int(z):
        x = 1 + z
        lo1, hi1 = max(theta0[4], (45 - 7 * 2.25) / x), min(theta0[5], (45 + 7 * 2.25) / x)

        def inner(m1):
            lo2, hi2 = max(theta0[4], (36 - 7 * 1.8) / x), min(m1, (36 + 7 * 1.8) / x)
            if hi2 <= lo2:
                return 0.0
            return O.p1(m1, theta0) * norm(m1 * x, 45.0, 2.25) * gl(lambda m2: O.p2(m2, m1, theta0) * norm(m2 * x, 36.0, 1.8), lo2, hi2)
        return gl(inner, lo1, hi1) if hi1 > lo1 else 0.0

    def zint(z):
        d = O.dL(z, H0, Om)
        gd = math.exp(-0.5 * ((math.log(d) - mu_d) / s_d) ** 2) / (d * s_d * math.sqrt(2 * math.pi))
        return O.psi(z, theta0) / (1 + z) * np.interp(z, zb, row) * gd / d ** 2 * mass_int(z)

    # d_L ~ 2000 Mpc e^{+-6*0.2} maps to z in about [0.12, 1.0]; split at the spike for accuracy
    I = sum(gl(zint, a, b) for a, b in [(0.10, 0.30), (0.30, 0.36), (0.36, 0.40), (0.40, 0.46), (0.46, 0.7), (0.7, 1.2)])
    zscore = (mc - I) / (I * stderr_rel)
    assert abs(zscore) < 4.0, (mc, I, stderr_rel)
    assert stderr_rel < 5e-3


# ---------------------------------------------------------------- selection closed form
def test_selection_constant_weights(theta0):
    """Injections drawn exactly from the model at theta_0 (density ∝ p_pop R pbar in source coordinates, transformed to
    detector coordinates) have equal weights Z0 => xi = Z0 n_found/n_draw, N_eff = n_found (Eq. 4)."""
    rng = np.random.default_rng(9)
    zmax, nz = 1.5, 256
    zb = np.linspace(0, zmax, nz)
    allsky = 0.3 + zb ** 2 * np.exp(-2 * zb)
    # z from pz ∝ psi/(1+z) * pbar on [0, zmax), tabulated inverse CDF on a fine grid
    zf = np.linspace(0, zmax * (1 - 1e-9), 20001)
    dens = np.array([O.psi(z, theta0) for z in zf]) / (1 + zf) * np.interp(zf, zb, allsky)
    cdf = np.concatenate([[0], np.cumsum(0.5 * (dens[1:] + dens[:-1]) * np.diff(zf))])
    Z0 = cdf[-1]
    n = 3000
    z = np.interp(rng.uniform(0, 1, n), cdf / Z0, zf)
    # masses: anything inside the support; the proposal density is the model's own, so it cancels
    m1 = rng.uniform(6, 90, n)
    m2 = theta0[4] + (m1 - theta0[4]) * rng.uniform(0, 1, n)
    H0, Om = theta0[0], theta0[1]
    dl = np.array([O.dL(zz, H0, Om) for zz in z])
    h = 1e-6
    ddl = np.array([(O.dL(zz + h, H0, Om) - O.dL(zz - h, H0, Om)) / (2 * h) for zz in z])   # Jacobian by finite difference
    pz = np.interp(z, zf, dens)   # un-normalised: weights come out equal to exactly 1
    lp = np.log(pz) + np.log([O.p1(a, theta0) * O.p2(b, a, theta0) for a, b in zip(m1, m2)]) - 2 * np.log1p(z) - np.log(ddl)
    inj = dict(dL=dl, m1z=m1 * (1 + z), m2z=m2 * (1 + z), log_pdraw=lp, n_draw=7.0 * n)
    logxi, neff = O.selection_logxi(theta0, inj, allsky, zmax, mode=O.EXACT)
    assert logxi[0] == pytest.approx(math.log(n / (7.0 * n)), abs=2e-6)     # finite-difference Jacobian + grid interp
    assert neff[0] == pytest.approx(n, rel=1e-8)


# ---------------------------------------------------------------- A0 packing (integer, bit-exact)
def test_pack_events_against_lexsort():
    rng = np.random.default_rng(4)
    n, ne = 5000, 13
    eid = rng.integers(0, ne, n).astype(np.int32)
    eid[eid == 7] = 6                              # an empty event
    row = rng.integers(0, 40, n).astype(np.int32)
    out = O.pack_events(eid, row, ne)
    perm = np.lexsort((np.arange(n), row, eid))     # stable by construction
    assert np.array_equal(out["perm"], perm)
    assert np.array_equal(out["ev_sample_off"], np.concatenate([[0], np.cumsum(np.bincount(eid, minlength=ne))]))
    pairs = np.unique(np.stack([eid, row], 1), axis=0)
    assert out["n_pixrefs"] == len(pairs)
    assert np.array_equal(out["ev_pix_rows"], pairs[:, 1])
    assert np.array_equal(out["ev_pix_off"], np.concatenate([[0], np.cumsum(np.bincount(pairs[:, 0], minlength=ne))]))
    se, sr = eid[perm], row[perm]
    starts = np.flatnonzero(np.concatenate([[True], (se[1:] != se[:-1]) | (sr[1:] != sr[:-1])]))
    assert np.array_equal(out["pix_sample_off"], np.concatenate([starts, [n]]))
    assert out["ev_sample_off"][7] == out["ev_sample_off"][8]


# ---- NEXT row 2: the per-pixel N_eff cut of Eq. 8 ----------------------------------------------
def _runs(row, a, b):
    """[start, end) of the maximal runs of equal row inside samples a..b."""
    out, r0 = [], a
    while r0 < b:
        r1 = r0 + 1
        while r1 < b and row[r1] == row[r0]:
            r1 += 1
        out.append((r0, r1))
        r0 = r1
    return out


def test_pixcut_threshold_zero_is_the_uncut_estimator(theta0):
    # every pixel with a live sample passes N_eff >= 0, so the cut path must reproduce the pinned uncut one
    ev, tab, zmax = _toy_event()
    th = np.stack([theta0, theta0 * np.array([1.4] + [1.0] * 11)])
    L0, n0, k0 = O.event_loglik(th, ev, tab, zmax)
    L1, n1, k1, p1 = O.event_loglik_pixcut(th, ev, tab, zmax, 0.0)
    np.testing.assert_allclose(L1, L0, rtol=0, atol=1e-13)
    np.testing.assert_allclose(n1, n0, rtol=1e-12)
    assert np.array_equal(k1, k0)
    # and an unreachable threshold leaves nothing
    L2, n2, k2, p2 = O.event_loglik_pixcut(th, ev, tab, zmax, 1e9)
    assert np.all(np.isneginf(L2)) and np.all(n2 == 0) and np.all(k2 == 0) and np.all(p2 == 0)


def test_pixcut_equals_recombination_of_single_pixel_events(theta0):
    # Eq. 8 by another route: make every pixel its own event, take its N_eff and log L from the (pinned) uncut
    # path, keep the pixels with N_eff >= threshold and recombine:  L_i = (1/S_i) sum_pass S_j L_j.
    ev, tab, zmax = _toy_event(n=400, seed=5, rows=9)
    th = np.stack([theta0, theta0 * np.array([0.8] + [1.0] * 11), theta0 * np.array([1.5] + [1.0] * 11)])
    off = ev["ev_sample_off"]
    row = ev["sample_row"]
    for thr in (1.5, 2.0, 4.0, 12.5):
        L, N, K, P = O.event_loglik_pixcut(th, ev, tab, zmax, thr)
        for i in range(off.size - 1):
            runs = _runs(row, off[i], off[i + 1])
            sub_off = np.array([0] + [r1 - off[i] for _, r1 in runs], dtype=np.int64)
            sl = slice(off[i], off[i + 1])
            sub = dict(ev_sample_off=sub_off, dL=ev["dL"][sl], m1z=ev["m1z"][sl], m2z=ev["m2z"][sl],
                       sample_row=row[sl], log_pe_prior=None)
            Lj, Nj, Kj = O.event_loglik(th, sub, tab, zmax)
            Sj = np.diff(sub_off).astype(float)
            for t in range(th.shape[0]):
                ok = np.isfinite(Lj[t]) & (Nj[t] >= thr * (1 + 1e-12))
                edge = np.isfinite(Lj[t]) & (np.abs(Nj[t] - thr) <= thr * 1e-12)
                assert not edge.any()                      # no pixel sits on the threshold in this toy
                assert P[t, i] == ok.sum() and K[t, i] == Kj[t][ok].sum()
                if ok.any():
                    want = np.log(np.sum(Sj[ok] * np.exp(Lj[t][ok] - Lj[t][ok].max()))) + Lj[t][ok].max() \
                        - np.log(off[i + 1] - off[i])
                    assert L[t, i] == pytest.approx(want, abs=1e-12)
                else:
                    assert np.isneginf(L[t, i])
    # the cut can only remove weight
    Lc = O.event_loglik_pixcut(th, ev, tab, zmax, 2.0)[0]
    Lu = O.event_loglik(th, ev, tab, zmax)[0]
    assert np.all(Lc <= Lu + 1e-13)


def test_pixcut_equal_weights_count_the_samples(theta0):
    # a pixel of n identical samples has N_eff = n exactly (the decision is taken as W^2 >= n_min Q):
    # pixels of 1, 2, 3 and 5 copies of one sample -> thresholds 2, 3, 3.5 keep {2,3,5}, {3,5}, {5}
    ev, tab, zmax = _toy_event(n=30, seed=2, rows=4)
    reps = [1, 2, 3, 5]
    n = sum(reps)
    one = lambda key: np.full(n, ev[key][0])
    e1 = dict(ev_sample_off=np.array([0, n], dtype=np.int64), dL=one("dL"), m1z=one("m1z"), m2z=one("m2z"),
              sample_row=np.repeat(np.arange(4, dtype=np.int32), reps), log_pe_prior=None)
    tab1 = np.tile(tab[:1], (4, 1))                         # the same LOS row everywhere: identical weights
    L0, _, k0 = O.event_loglik(theta0, e1, tab1, zmax)
    assert k0[0, 0] == n
    lw = L0[0, 0]                                          # = log w of the one sample (mean of n equal weights)
    for thr, kept in ((2.0, [2, 3, 5]), (3.0, [3, 5]), (3.5, [5]), (1.0, reps), (5.0, [5]), (5.0001, [])):
        L, N, K, P = O.event_loglik_pixcut(theta0, e1, tab1, zmax, thr)
        assert P[0, 0] == len(kept) and K[0, 0] == sum(kept)
        if kept:
            assert L[0, 0] == pytest.approx(lw + math.log(sum(kept) / n), abs=1e-13)
            assert N[0, 0] == pytest.approx(sum(kept), rel=1e-12)
        else:
            assert np.isneginf(L[0, 0]) and N[0, 0] == 0


def test_pixcut_invariant_under_pixel_order_and_dead_padding(theta0):
    ev, tab, zmax = _toy_event(n=240, seed=8, rows=6)
    off = ev["ev_sample_off"]
    base = O.event_loglik_pixcut(theta0, ev, tab, zmax, 2.0)
    # reverse the order of the pixels inside each event (samples inside a pixel keep their order)
    idx = []
    for i in range(off.size - 1):
        for r0, r1 in reversed(_runs(ev["sample_row"], off[i], off[i + 1])):
            idx.extend(range(r0, r1))
    idx = np.array(idx)
    ev2 = dict(ev, dL=ev["dL"][idx], m1z=ev["m1z"][idx], m2z=ev["m2z"][idx], sample_row=ev["sample_row"][idx])
    got = O.event_loglik_pixcut(theta0, ev2, tab, zmax, 2.0)
    np.testing.assert_allclose(got[0], base[0], rtol=0, atol=1e-12)
    assert np.array_equal(got[2], base[2]) and np.array_equal(got[3], base[3])
    # dead samples appended to the last pixel of the last event change S_i only
    pad = 11
    n = ev["dL"].size
    ev3 = dict(ev_sample_off=np.array([off[0], off[1], n + pad], dtype=np.int64),
               dL=np.concatenate([ev["dL"], np.full(pad, 1e7)]), m1z=np.concatenate([ev["m1z"], np.full(pad, 40.0)]),
               m2z=np.concatenate([ev["m2z"], np.full(pad, 30.0)]),
               sample_row=np.concatenate([ev["sample_row"], np.full(pad, ev["sample_row"][-1], np.int32)]),
               log_pe_prior=None)
    got3 = O.event_loglik_pixcut(theta0, ev3, tab, zmax, 2.0)
    S1 = n - off[1]
    assert got3[0][0, 1] == pytest.approx(base[0][0, 1] - math.log((S1 + pad) / S1), abs=1e-12)
    assert np.array_equal(got3[3], base[3]) and np.array_equal(got3[2], base[2])


# ---- NEXT row 1: the paper's KDE numerator (Eq. 5-7, D1; R26-R30) -------------------------------------
def _kde_event(n=300, seed=21, rows=4, dl0=2600.0, pix_min=2):
    """One-or-two-event toy whose every pixel has >= pix_min samples well inside the z grid."""
    rng = np.random.default_rng(seed)
    dl = dl0 * np.exp(0.12 * rng.standard_normal(n))
    m1z = 50.0 * (1 + 0.06 * rng.standard_normal(n))
    m2z = 38.0 * (1 + 0.06 * rng.standard_normal(n))
    m1z, m2z = np.maximum(m1z, m2z), np.minimum(m1z, m2z)
    half = n // 2
    row = np.concatenate([np.sort(rng.integers(0, rows, half)), np.sort(rng.integers(0, rows, n - half))]).astype(np.int32)
    return dict(ev_sample_off=np.array([0, half, n], dtype=np.int64), dL=dl, m1z=m1z, m2z=m2z, sample_row=row,
                log_pe_prior=None)


def _theta_unit_rate(theta0):
    th = theta0.copy()
    th[9], th[10] = 1.0, -1.0       # gamma = 1, kappa = -1: psi(z)/(1+z) = 1 identically (psi0 = 2, denominator 2)
    return th


def test_kde_unit_rate_is_one(theta0):
    th = _theta_unit_rate(theta0)
    for z in (0.0, 0.3, 1.2):
        assert O.lib().orc_psi(z, O._p(O._theta(th))) / (1 + z) == pytest.approx(1.0, abs=1e-15)


def test_kde_linear_prior_equals_direct_sum(theta0):
    # int N(z; z_k, h) (a + b z) dz = a + b z_k: with a LOS row linear in z and a unit rate the KDE numerator is the
    # direct Monte-Carlo sum, whatever the bandwidth (kernels resolved by the grid, h >= 2 dz, and inside it).
    ev = _kde_event()
    zmax, nz = 1.5, 64
    zb = np.linspace(0, zmax, nz)
    tab = np.stack([0.7 + 0.0 * zb, 0.2 + 1.3 * zb, 2.0 - 0.9 * zb, 0.05 + 0.4 * zb])
    th = _theta_unit_rate(theta0)
    Ld, _, kd = O.event_loglik(th, ev, tab, zmax)
    Lk, npk = O.event_loglik_kde(th, ev, tab, zmax, n_grid=256)
    assert np.all(kd > 0) and np.all(npk == 4)
    np.testing.assert_allclose(Lk, Ld, rtol=0, atol=2e-7)     # Gaussian tails beyond the grid: < 1e-7
    # the grid resolution does not matter while h >= 2 dz
    Lk2, _ = O.event_loglik_kde(th, ev, tab, zmax, n_grid=200)
    np.testing.assert_allclose(Lk2, Lk, rtol=0, atol=1e-9)


def _pixel_runs(ev):
    off, row = ev["ev_sample_off"], ev["sample_row"]
    return [[(r0, r1) for r0, r1 in _runs(row, off[i], off[i + 1])] for i in range(off.size - 1)]


def _scott(z, v):
    """Eq. D1 with the v-weighted standard deviation of the pixel's redshifts and n = its live samples."""
    mu = np.sum(v * z) / np.sum(v)
    sig = math.sqrt(np.sum(v * (z - mu) ** 2) / np.sum(v))
    return 1.06 * sig * z.size ** (-0.2)


def test_kde_bandwidth_through_quadratic_prior(theta0):
    # int N(z; z_k, h) z^2 dz = z_k^2 + h^2: a LOS row equal to z^2 exposes the bandwidth of every pixel.
    ev = _kde_event(n=260, seed=4, rows=5)
    zmax, nz = 1.5, 4096                                   # fine LOS nodes: the lerp of z^2 is exact to 3e-8
    zb = np.linspace(0, zmax, nz)
    tab = np.tile(zb ** 2, (5, 1))
    th = _theta_unit_rate(theta0)
    z, lv = O.kde_samples(th, ev, 5, zmax)
    assert np.all(np.isfinite(lv))
    Lk, _ = O.event_loglik_kde(th, ev, tab, zmax, n_grid=256)
    off = ev["ev_sample_off"]
    for i, runs in enumerate(_pixel_runs(ev)):
        tot, tot_h0 = 0.0, 0.0
        for r0, r1 in runs:
            v = np.exp(lv[r0:r1])
            h = _scott(z[r0:r1], v)
            assert h > 2 * zmax / 255
            tot += np.sum(v * (z[r0:r1] ** 2 + h * h))
            tot_h0 += np.sum(v * z[r0:r1] ** 2)
        want = math.log(tot / (off[i + 1] - off[i]))
        assert Lk[0, i] == pytest.approx(want, abs=2e-6)
        # the h^2 term is what is being pinned: without it the value is off by far more than the tolerance
        assert abs(math.log(tot_h0 / (off[i + 1] - off[i])) - want) > 1e-3


def test_kde_against_continuous_quadrature(theta0):
    # generic theta (the rate term varies over the grid), one pixel, smooth prior: the 256-node trapezoid of
    # f(z) p_los(z) R(z) against scipy's adaptive quadrature of the same continuous integrand
    ev = _kde_event(n=40, seed=9, rows=1)
    ev = dict(ev, ev_sample_off=np.array([0, 40], dtype=np.int64))
    zmax, nz = 1.5, 16
    zb = np.linspace(0, zmax, nz)
    tab = (0.3 + 2.0 * zb)[None, :]                        # linear: its lerp is the function itself
    th = theta0.copy()
    z, lv = O.kde_samples(th, ev, 1, zmax)
    v = np.exp(lv)
    h = _scott(z, v)
    th_arr = O._theta(th)
    R = lambda x: O.lib().orc_psi(float(x), O._p(th_arr)) / (1 + x)
    f = lambda x: np.sum(v * np.exp(-0.5 * ((x - z) / h) ** 2)) / (h * math.sqrt(2 * math.pi)) * (0.3 + 2.0 * x) * R(x)
    I, _ = integrate.quad(f, 0, zmax, points=[z.min(), z.mean(), z.max()], epsabs=0, epsrel=1e-11, limit=400)
    Lk, npk = O.event_loglik_kde(th, ev, tab, zmax, n_grid=256)
    assert npk[0, 0] == 1
    assert Lk[0, 0] == pytest.approx(math.log(I / 40), abs=1e-6)
    # and it is not the direct sum: the prior's curvature times h^2 shows
    Ld, _, _ = O.event_loglik(th, ev, tab, zmax)
    assert abs(Ld[0, 0] - Lk[0, 0]) > 1e-5


def test_kde_pixel_rules_and_invariances(theta0):
    ev = _kde_event(n=120, seed=12, rows=3)
    zmax, nz = 1.5, 64
    tab = np.random.default_rng(1).uniform(0.2, 2.0, (5, nz))
    base, npb = O.event_loglik_kde(theta0, ev, tab, zmax)
    # a pixel of one sample has no bandwidth: appended to an event it changes S_i only
    n = ev["dL"].size
    off = ev["ev_sample_off"]
    ev2 = dict(ev_sample_off=np.array([off[0], off[1], n + 1], dtype=np.int64), dL=np.append(ev["dL"], ev["dL"][-1]),
               m1z=np.append(ev["m1z"], ev["m1z"][-1]), m2z=np.append(ev["m2z"], ev["m2z"][-1]),
               sample_row=np.append(ev["sample_row"], np.int32(4)), log_pe_prior=None)
    got, npg = O.event_loglik_kde(theta0, ev2, tab, zmax)
    S1 = n - off[1]
    assert got[0, 1] == pytest.approx(base[0, 1] - math.log((S1 + 1) / S1), abs=1e-12) and npg[0, 1] == npb[0, 1]
    # two identical samples: sigma = 0, no bandwidth either
    ev3 = dict(ev2, ev_sample_off=np.array([off[0], off[1], n + 2], dtype=np.int64), dL=np.append(ev2["dL"], ev["dL"][-1]),
               m1z=np.append(ev2["m1z"], ev["m1z"][-1]), m2z=np.append(ev2["m2z"], ev["m2z"][-1]),
               sample_row=np.append(ev2["sample_row"], np.int32(4)))
    got3, np3 = O.event_loglik_kde(theta0, ev3, tab, zmax)
    assert got3[0, 1] == pytest.approx(base[0, 1] - math.log((S1 + 2) / S1), abs=1e-12) and np3[0, 1] == npb[0, 1]
    # the N_eff cut of Eq. 8 on the KDE weights: unreachable threshold leaves nothing, threshold 0 everything
    assert np.all(np.isneginf(O.event_loglik_kde(theta0, ev, tab, zmax, neff_min=1e9)[0]))
    # permutation of the samples inside each pixel
    rng = np.random.default_rng(3)
    idx = np.concatenate([r0 + rng.permutation(r1 - r0) for runs in _pixel_runs(ev) for r0, r1 in runs])
    evp = dict(ev, dL=ev["dL"][idx], m1z=ev["m1z"][idx], m2z=ev["m2z"][idx])
    gotp, _ = O.event_loglik_kde(theta0, evp, tab, zmax)
    np.testing.assert_allclose(gotp, base, rtol=0, atol=1e-12)
    # H0 scaling (Om fixed): z unchanged, every v_k gains 3 ln s, bandwidths unchanged
    s = 1.3
    th2 = theta0.copy(); th2[0] *= s
    gots, _ = O.event_loglik_kde(th2, dict(ev, dL=ev["dL"] / s), tab, zmax)
    np.testing.assert_allclose(gots, base + 3 * math.log(s), rtol=0, atol=1e-11)


# ---- NEXT row 3b: the per-pixel sample cap (R31) -----------------------------------
def _cap_catalogue(seed=0, n=6000, n_events=5, rows=12):
    rng = np.random.default_rng(seed)
    ev = rng.integers(0, n_events, n).astype(np.int32)
    row = np.minimum(rng.geometric(0.35, n) - 1, rows - 1).astype(np.int32)   # a few crowded pixels, a long tail
    return ev, row, O.pack_events(ev, row, n_events)


def test_cap_pixels_properties():
    ev, row, P = _cap_catalogue()
    sizes = np.diff(P["pix_sample_off"])
    assert sizes.max() > 200 and sizes.min() < 5
    for cap in (1, 7, 100, 10 ** 6):
        perm, evo, pxo = O.cap_pixels(P["perm"], P["ev_sample_off"], P["pix_sample_off"], cap, 1234)
        assert np.array_equal(np.diff(pxo), np.minimum(sizes, cap))          # every pixel keeps min(n, cap)
        assert perm.size == pxo[-1] == evo[-1] and evo[0] == 0
        # the kept samples are a subsequence of the packed order (order preserved, no duplicates)
        pos = {v: i for i, v in enumerate(P["perm"])}
        where = np.array([pos[v] for v in perm])
        assert np.all(np.diff(where) > 0)
        # and they stay inside their own pixel and event
        for j in range(sizes.size):
            a, b = P["pix_sample_off"][j], P["pix_sample_off"][j + 1]
            assert set(perm[pxo[j]:pxo[j + 1]]) <= set(P["perm"][a:b])
        assert np.array_equal(np.diff(evo), np.bincount(ev[perm], minlength=5))
        if cap >= sizes.max():
            assert np.array_equal(perm, P["perm"])
    # seeded: same seed same choice, another seed another choice
    a = O.cap_pixels(P["perm"], P["ev_sample_off"], P["pix_sample_off"], 7, 99)[0]
    b = O.cap_pixels(P["perm"], P["ev_sample_off"], P["pix_sample_off"], 7, 99)[0]
    c = O.cap_pixels(P["perm"], P["ev_sample_off"], P["pix_sample_off"], 7, 100)[0]
    assert np.array_equal(a, b) and not np.array_equal(a, c)
    # the choice depends on the original sample index only, not on where packing put the sample:
    # relabelling the events (another packed order) keeps the same original samples
    P2 = O.pack_events((4 - ev).astype(np.int32), row, 5)
    d = O.cap_pixels(P2["perm"], P2["ev_sample_off"], P2["pix_sample_off"], 7, 99)[0]
    assert set(a) == set(d)


def test_cap_pixels_is_uniform_without_replacement():
    # one pixel of 40 samples, cap 10, 4000 seeds: every sample is kept with probability 1/4 (binomial, 5 sigma)
    n, cap, trials = 40, 10, 4000
    perm = np.arange(n, dtype=np.int64)
    evo, pxo = np.array([0, n]), np.array([0, n])
    counts = np.zeros(n)
    for s in range(trials):
        kept = O.cap_pixels(perm, evo, pxo, cap, s)[0]
        assert kept.size == cap and np.unique(kept).size == cap
        counts[kept] += 1
    sigma = math.sqrt(trials * 0.25 * 0.75)
    assert np.abs(counts - trials * 0.25).max() < 5 * sigma


def test_cap_pixels_against_numpy_lexsort():
    # the same rule written with numpy: inside a crowded pixel keep the cap smallest (hash32, packed position)
    ev, row, P = _cap_catalogue(seed=3)
    seed, cap = 20260915, 25
    def h32(idx):
        M = (1 << 64) - 1
        z = (seed + (int(idx) + 1) * 0x9E3779B97F4A7C15) & M
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & M
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & M
        return (z ^ (z >> 31)) >> 32
    keep = np.zeros(P["perm"].size, bool)
    pso = P["pix_sample_off"]
    for j in range(pso.size - 1):
        a, b = pso[j], pso[j + 1]
        if b - a <= cap:
            keep[a:b] = True
        else:
            h = np.array([h32(v) for v in P["perm"][a:b]], dtype=np.uint64)
            order = np.lexsort((np.arange(a, b), h))
            keep[a + order[:cap]] = True
    got = O.cap_pixels(P["perm"], P["ev_sample_off"], pso, cap, seed)[0]
    assert np.array_equal(got, P["perm"][keep])


def test_kde_silverman_bandwidth_through_quadratic_prior(theta0):
    # Eq. D2: h = 0.9 min(sigma, IQR / 1.34) n^(-1/5); the z^2 prior exposes it as for Scott's rule.  numpy's
    # percentile (linear interpolation) is the independent IQR; both branches of the min occur in the toy.
    ev = _kde_event(n=260, seed=4, rows=5)
    rng = np.random.default_rng(5)
    far = rng.choice(260, 12, replace=False)              # outliers: sigma inflates, the IQR does not
    ev["dL"][far] *= 1.6
    zmax, nz = 1.5, 4096
    zb = np.linspace(0, zmax, nz)
    tab = np.tile(zb ** 2, (5, 1))
    th = _theta_unit_rate(theta0)
    z, lv = O.kde_samples(th, ev, 5, zmax)
    assert np.all(np.isfinite(lv))
    Lk, _ = O.event_loglik_kde(th, ev, tab, zmax, n_grid=256, bandwidth="silverman")
    Ls, _ = O.event_loglik_kde(th, ev, tab, zmax, n_grid=256, bandwidth="scott")
    off = ev["ev_sample_off"]
    used_iqr = used_sigma = 0
    for i, runs in enumerate(_pixel_runs(ev)):
        tot = 0.0
        for r0, r1 in runs:
            v, zz = np.exp(lv[r0:r1]), z[r0:r1]
            mu = np.sum(v * zz) / np.sum(v)
            sig = math.sqrt(np.sum(v * (zz - mu) ** 2) / np.sum(v))
            q1, q3 = np.percentile(zz, [25, 75])
            used_iqr += (q3 - q1) / 1.34 < sig
            used_sigma += (q3 - q1) / 1.34 >= sig
            h = 0.9 * min(sig, (q3 - q1) / 1.34) * zz.size ** (-0.2)
            tot += np.sum(v * (zz ** 2 + h * h))
        want = math.log(tot / (off[i + 1] - off[i]))
        assert Lk[0, i] == pytest.approx(want, abs=2e-6)
        assert abs(Ls[0, i] - Lk[0, i]) > 1e-4            # and it is not Scott's bandwidth
    assert used_iqr > 0 and used_sigma > 0


# ---------------------------------------------------------------- 32-bit table storage (R22)
@pytest.mark.parametrize("Om,zmax,M", [(0.3, 2.0, 1025), (0.1, 1.5, 257), (1.0, 2.0, 1025)])
def test_round_table_32_quantisation_bounds(Om, zmax, M):
    """orc_round_table_32 against what R22 fixes: nodes are the nearest multiple of q = z_max/(2^32-1) (so
    |z32 - z64| <= q/2, z32/q an integer in [0, 2^32-1]); slopes are the nearest binary32 in units of q (relative
    error <= 2^-24, the stored number exactly a float)."""
    zt, dt, um = O.build_table(Om, zmax, M)
    z32, d32 = O.round_table_32(zt, dt, zmax)
    q = zmax / 4294967295.0
    assert np.abs(z32 - zt).max() <= 0.5 * q * (1 + 1e-9)
    k = z32 / q
    assert np.abs(k - np.rint(k)).max() <= 1e-5 and k.min() >= 0 and k.max() <= 4294967295.0 + 1e-5
    assert z32[0] == 0.0 and abs(z32[-1] - zmax) <= 1e-15
    # independent restatement with numpy's own rounding
    np.testing.assert_array_equal(np.rint(zt / q), np.rint(k))
    assert np.abs(d32 / dt - 1.0).max() <= 2.0 ** -24 * (1 + 1e-9)
    assert np.abs(d32 / dt - 1.0).max() > 2.0 ** -30          # the slopes really were rounded
    f = d32 / q
    np.testing.assert_allclose(f.astype(np.float32).astype(np.float64), f, rtol=4e-16, atol=0)
    np.testing.assert_allclose((dt / q).astype(np.float32).astype(np.float64) * q, d32, rtol=4e-16, atol=0)


def test_round_table_32_bound_on_loglik(theta0):
    """table_prec = 1 against table_prec = 0 on the toy event: the node and slope roundings move z by at most
    dz = q/2 + 2^-24 max|d_m| 4/27 (Hermite basis functions), hence log L_i by at most dz * max |d ln w / dz|;
    the LOS term dominates that derivative and is bounded from the table itself."""
    ev, tab, zmax = _toy_event(n=600)
    M = 1025
    zt, dt, um = O.build_table(theta0[1], zmax, M)
    q = zmax / 4294967295.0
    dz = 0.5 * q + 2.0 ** -24 * np.abs(dt).max() * (4.0 / 27.0)
    step = zmax / (tab.shape[1] - 1)
    g_los = (np.abs(np.diff(tab, axis=1)) / np.minimum(tab[:, 1:], tab[:, :-1])).max() / step
    bound = dz * (g_los + 60.0)       # 60: generous bound on the population / rate / Jacobian terms' slopes in z
    for H0 in (50.0, 70.0, 100.0):
        th = theta0.copy(); th[0] = H0
        L0, n0, k0 = O.event_loglik(th, ev, tab, zmax, table_prec=0, n_nodes=M)
        L1, n1, k1 = O.event_loglik(th, ev, tab, zmax, table_prec=1, n_nodes=M)
        assert np.array_equal(k0, k1)
        d = np.abs(L1 - L0).max()
        assert 1e-14 < d <= bound, (d, bound)
        # the look-up itself, restated: Hermite on the rounded arrays
        z32, d32 = O.round_table_32(zt, dt, zmax)
        for u in (0.1 * um, 0.37 * um, 0.9 * um):
            a, b = O.z_table(u, zt, dt, um), O.z_table(u, z32, d32, um)
            assert abs(a - b) <= dz * (1 + 1e-9)


def test_norm_pl_alpha_one_branch(theta0):
    """alpha = 1: the log limit of the power-law normalisation, 1 / ln(mmax/mmin), by quadrature and by continuity."""
    th = theta0.copy(); th[2] = 1.0; th[8] = 0.0
    assert O.norm_pl(th) == pytest.approx(1.0 / math.log(th[5] / th[4]), rel=1e-15)
    val, err = integrate.quad(lambda m: O.p1(m, th), th[4], th[5], epsabs=0, epsrel=1e-12, limit=200)
    assert val == pytest.approx(1.0, abs=1e-10)
    assert O.p1(20.0, th) == pytest.approx(1.0 / (20.0 * math.log(th[5] / th[4])), rel=1e-14)
    for eps in (1e-6, -1e-6):
        th2 = th.copy(); th2[2] = 1.0 + eps
        assert O.norm_pl(th2) == pytest.approx(O.norm_pl(th), rel=1e-5)
        assert O.p1(20.0, th2) == pytest.approx(O.p1(20.0, th), rel=1e-5)


# ---------------------------------------------------------------- MULTIPEAK with low-mass smoothing (NEXT row 3a)
# App. A, Table III :263-274; the formula is not in the paper: readings R33-R36 of DESIGN.md.
def _th_mp(**mod):
    for line in open(os.path.join(GOLD, "table3_multipeak.txt")):
        if line.strip() and not line.startswith("#"):
            th = np.array([float(x) for x in line.split()])
    names = dict(H0=0, Om=1, alpha=2, beta=3, mmin=4, mmax=5, mu=6, sigma=7, lam=8, dm=12, mul=13, sigl=14, laml=15)
    for k, v in mod.items():
        th[names[k]] = v
    return th


def test_mp_smoothing_closed_forms():
    """S(m) = 1/(1 + exp(dm/m' + dm/(m' - dm))): 0 at mmin, 1 from mmin + dm on, 1/2 at the middle of the window,
    S(mmin + x) + S(mmin + dm - x) = 1 (the exponent is odd about the middle), increasing; below e^-250 it is 0 (R35)."""
    lo, dm = 4.6, 4.8
    assert O.mp_smooth(lo, lo, dm) == 0.0 and O.mp_smooth(lo - 1.0, lo, dm) == 0.0
    assert O.mp_smooth(lo + dm, lo, dm) == 1.0 and O.mp_smooth(50.0, lo, dm) == 1.0
    assert O.mp_smooth(lo + 0.5 * dm, lo, dm) == pytest.approx(0.5, abs=1e-15)
    xs = np.linspace(0.02, 0.98, 49) * dm
    s = np.array([O.mp_smooth(lo + x, lo, dm) for x in xs])
    assert np.all(np.diff(s) > 0)
    np.testing.assert_allclose(s + s[::-1], 1.0, rtol=0, atol=1e-13)
    np.testing.assert_allclose(s, special.expit(-(dm / xs + dm / (xs - dm))), rtol=1e-13)
    # the e^-250 rule: the exponent at m' = dm/251 is 251 - 1/(1 - 1/251) = 249.996, at dm/253 it is 251.996
    assert O.mp_smooth(lo + dm / 253.0, lo, dm) == 0.0
    assert 0.0 < O.mp_smooth(lo + dm / 251.0, lo, dm) < 1e-108
    # dm = 0: a step at mmin, the lower edge included (R15)
    assert O.mp_smooth(lo, lo, 0.0) == 1.0 and O.mp_smooth(lo - 1e-9, lo, 0.0) == 0.0


@pytest.mark.parametrize("mod", [{}, dict(dm=0.0), dict(laml=0.0), dict(laml=1.0), dict(lam=0.0), dict(lam=1.0, dm=9.0),
                                 dict(alpha=1.5, mul=7.0, sigl=2.0, dm=2.0, beta=-0.5)])
def test_mp_p1_normalised(mod):
    th = _th_mp(**mod)
    lo, hi, top = th[4], th[5], th[4] + th[12]
    with O.mass_model("multipeak"):
        val, _ = integrate.quad(lambda m: O.p1(m, th), lo, hi, points=sorted({lo + 0.5 * th[12], top, th[13], th[6]}),
                                epsabs=0, epsrel=1e-12, limit=800)
        assert O.p1(lo, th) == 0.0 and O.p1(hi, th) > 0.0 and O.p1(hi + 1e-9, th) == 0.0
    assert val == pytest.approx(1.0, abs=1e-10)


@pytest.mark.parametrize("beta", [1.0, 0.0, -0.5, 4.0, -1.0, -2.5])
def test_mp_p2_normalised(beta):
    th = _th_mp(beta=beta)
    lo, top = th[4], th[4] + th[12]
    with O.mass_model("multipeak"):
        for m1 in (5.3, 6.5, 7.0, 9.0, top, 12.0, 80.0):
            val, _ = integrate.quad(lambda m: O.p2(m, m1, th), lo, m1, points=sorted({min(m1, lo + 0.5 * th[12]), min(m1, top)}),
                                    epsabs=0, epsrel=1e-12, limit=400)
            assert val == pytest.approx(1.0, abs=2e-10), (beta, m1)
        assert O.p2(lo, 30.0, th) == 0.0 and O.p2(30.0, 30.0, th) > 0 and O.p2(30.0001, 30.0, th) == 0.0


def test_mp_C_against_scipy_quad():
    th = _th_mp()
    lo, dm, b = th[4], th[12], th[3]
    f = lambda m: m ** b * special.expit(-(dm / (m - lo) + dm / (m - lo - dm))) if m < lo + dm else m ** b
    with O.mass_model("multipeak"):
        for m1 in (5.2, 6.0, 7.0, 8.5, 9.4, 9.5, 20.0, 86.3):
            ref, _ = integrate.quad(f, lo, m1, points=sorted({min(m1, 7.0), min(m1, lo + dm)}), epsabs=0, epsrel=1e-13,
                                    limit=400)
            assert O.mp_C(m1, th) == pytest.approx(ref, rel=2e-11), m1


def test_mp_reduces_to_power_law_plus_peak(theta0):
    """delta_m = 0 with one peak switched off is the (pinned) power-law+peak model: lambda_low = 1 keeps the LOW peak,
    lambda_low = 0 the HIGH one; in between p(m1) is linear in lambda_low; p(m2|m1) is the plain conditional power law."""
    th = _th_mp(dm=0.0)
    ms = (4.6000001, 5.0, 9.7, 12.0, 30.7, 60.0, 86.3)

    def plpeak(mu, sig):
        t = theta0.copy()
        t[:12] = th[:12]
        t[6], t[7] = mu, sig
        return np.array([O.p1(m, t) for m in ms]), np.array([O.p2(0.7 * m + 0.3 * 4.6, m, t) for m in ms])

    def multipeak(laml):
        t = th.copy()
        t[15] = laml
        with O.mass_model("multipeak"):
            return np.array([O.p1(m, t) for m in ms]), np.array([O.p2(0.7 * m + 0.3 * 4.6, m, t) for m in ms])

    lo1, lo2 = plpeak(th[13], th[14])
    hi1, hi2 = plpeak(th[6], th[7])
    a1, a2 = multipeak(1.0)
    b1, b2 = multipeak(0.0)
    np.testing.assert_allclose(a1, lo1, rtol=1e-12)
    np.testing.assert_allclose(b1, hi1, rtol=1e-12)
    np.testing.assert_allclose(a2, lo2, rtol=1e-13)
    np.testing.assert_allclose(b2, hi2, rtol=1e-13)
    c1, _ = multipeak(0.8)
    np.testing.assert_allclose(c1, 0.8 * lo1 + 0.2 * hi1, rtol=1e-12)
    assert abs(lo1[2] / hi1[2] - 1) > 0.5      # the two peaks really differ at 9.7 Msun
    # the whole event term agrees too (same support rules at delta_m = 0)
    ev, tab, zmax = _toy_event()
    ev = dict(ev, m1z=ev["m1z"] * 0.45, m2z=ev["m2z"] * 0.35)
    t12 = theta0.copy()
    t12[:12] = th[:12]
    t12[6], t12[7] = th[13], th[14]
    L0, n0, k0 = O.event_loglik(t12, ev, tab, zmax)
    t16 = th.copy()
    t16[15] = 1.0
    with O.mass_model("multipeak"):
        L1, n1, k1 = O.event_loglik(t16, ev, tab, zmax)
    assert np.array_equal(k0, k1) and k0.min() > 0
    np.testing.assert_allclose(L1, L0, rtol=0, atol=1e-11)


def test_mp_smoothing_shapes_p1_and_p2():
    """With everything else equal, switching delta_m on multiplies p(m1) by S(m1) N1(0)/N1(dm) and p(m2|m1) by
    S(m2) C0(m1)/C(m1): ratios at two masses isolate S, which the closed forms above pin."""
    th, th0 = _th_mp(), _th_mp(dm=0.0)
    lo, dm = th[4], th[12]
    with O.mass_model("multipeak"):
        ma, mb = 6.2, 8.1
        r = (O.p1(ma, th) / O.p1(ma, th0)) / (O.p1(mb, th) / O.p1(mb, th0))
        assert r == pytest.approx(O.mp_smooth(ma, lo, dm) / O.mp_smooth(mb, lo, dm), rel=1e-13)
        r2 = (O.p2(ma, 20.0, th) / O.p2(ma, 20.0, th0)) / (O.p2(mb, 20.0, th) / O.p2(mb, 20.0, th0))
        assert r2 == pytest.approx(O.mp_smooth(ma, lo, dm) / O.mp_smooth(mb, lo, dm), rel=1e-13)
        assert O.p1(20.0, th) / O.p1(20.0, th0) == pytest.approx(1.0 / O.mp_N1(th), rel=1e-12)   # N1(dm = 0) = 1
        assert O.mp_N1(th0) == pytest.approx(1.0, abs=1e-12)


def test_mp_selection_constant_weights():
    """As test_selection_constant_weights, under MULTIPEAK and with masses inside and above the smoothing window:
    injections drawn from the model itself have equal weights (Eq. 4)."""
    th = _th_mp()
    rng = np.random.default_rng(10)
    zmax, nz = 1.5, 256
    zb = np.linspace(0, zmax, nz)
    allsky = 0.3 + zb ** 2 * np.exp(-2 * zb)
    n = 2000
    with O.mass_model("multipeak"):
        zf = np.linspace(0, zmax * (1 - 1e-9), 20001)
        dens = np.array([O.psi(z, th) for z in zf]) / (1 + zf) * np.interp(zf, zb, allsky)
        cdf = np.concatenate([[0], np.cumsum(0.5 * (dens[1:] + dens[:-1]) * np.diff(zf))])
        z = np.interp(rng.uniform(0, 1, n), cdf / cdf[-1], zf)
        m1 = rng.uniform(5.5, 40, n)
        m2 = 5.2 + (m1 - 5.2) * rng.uniform(0, 1, n)
        H0, Om = th[0], th[1]
        dl = np.array([O.dL(zz, H0, Om) for zz in z])
        h = 1e-6
        ddl = np.array([(O.dL(zz + h, H0, Om) - O.dL(zz - h, H0, Om)) / (2 * h) for zz in z])
        lp = np.log(np.interp(z, zf, dens)) + np.log([O.p1(a, th) * O.p2(b, a, th) for a, b in zip(m1, m2)]) \
            - 2 * np.log1p(z) - np.log(ddl)
        inj = dict(dL=dl, m1z=m1 * (1 + z), m2z=m2 * (1 + z), log_pdraw=lp, n_draw=7.0 * n)
        logxi, neff = O.selection_logxi(th, inj, allsky, zmax, mode=O.EXACT)
    assert logxi[0] == pytest.approx(math.log(1 / 7.0), abs=2e-6)
    assert neff[0] == pytest.approx(n, rel=1e-8)


def test_mp_theta_domain():
    with O.mass_model("multipeak"):
        assert O.theta_valid(_th_mp())
        for bad in (dict(dm=-0.1), dict(dm=90.0), dict(sigl=0.0), dict(laml=1.2), dict(laml=-0.1)):
            assert not O.theta_valid(_th_mp(**bad)), bad


# ---------------------------------------------------------------- biweight midvariance bandwidth (Eq. D3-D4)
def _biweight_numpy(x):
    """Eq. D3-D4 with numpy's median for Q and the MAD."""
    Q = np.median(x)
    mad = np.median(np.abs(x - Q))
    u = (x - Q) / (9 * mad)
    I = np.abs(u) < 1
    return x.size * np.sum(((x - Q) ** 2 * (1 - u ** 2) ** 4)[I]) / np.sum(((1 - u ** 2) * (1 - 5 * u ** 2))[I]) ** 2


def test_biweight_midvariance_properties():
    """What the statistic is known for (ref. [54]): on a large normal sample it equals the variance; a few
    gross outliers ("more than nine MADs from the centre": zero weight) leave it alone while they wreck the sample
    variance; it is shift-invariant and scales with the square; a sample with MAD = 0 has no scale."""
    rng = np.random.default_rng(3)
    x = 0.4 + 0.05 * rng.standard_normal(40000)
    z2 = O.biweight_midvariance(x)
    assert z2 == pytest.approx(0.05 ** 2, rel=0.02)
    assert z2 == pytest.approx(_biweight_numpy(x), rel=1e-12)
    xo = np.concatenate([x, 0.4 + 0.05 * 60 * np.ones(400)])          # 1 % of points at 60 sigma
    assert np.var(xo) > 30 * 0.05 ** 2
    assert O.biweight_midvariance(xo) == pytest.approx(z2, rel=0.03)
    assert O.biweight_midvariance(3.0 * x - 7.0) == pytest.approx(9.0 * z2, rel=1e-11)
    assert O.biweight_midvariance(rng.permutation(x)) == pytest.approx(z2, rel=1e-13)
    # small samples, even and odd counts: numpy's median conventions
    for n in (2, 3, 4, 7, 10):
        y = rng.standard_normal(n)
        assert O.biweight_midvariance(y) == pytest.approx(_biweight_numpy(y), rel=1e-12), n
    assert math.isnan(O.biweight_midvariance(np.array([1.0, 1.0, 1.0, 2.0])))    # MAD = 0
    # the indicator: a point beyond 9 MAD contributes nothing, wherever it is
    y = np.array([-1.0, -0.5, 0.0, 0.5, 1.0, 50.0])
    y2 = y.copy()
    y2[-1] = 500.0
    assert O.biweight_midvariance(y) == O.biweight_midvariance(y2)


@pytest.mark.parametrize("rule", ["biweight_scott", "biweight"])
def test_kde_biweight_bandwidth_through_quadratic_prior(theta0, rule):
    """The z^2 prior exposes h of every pixel (as for Scott and Silverman): rule 3 is 1.06 sqrt(D3) n^(-1/5), rule 2 is
    D3 itself, the formula as the paper prints it (reading R37).  The toy's redshifts spread widely so that even
    h = D3 (a variance) is resolved by the 256-node grid; outliers make D3 differ from the plain variance."""
    ev = _kde_event(n=260, seed=4, rows=5)
    rng = np.random.default_rng(6)
    if rule == "biweight":
        ev["dL"] = ev["dL"] * np.exp(0.3 * rng.standard_normal(260))
    far = rng.choice(260, 10, replace=False)
    ev["dL"][far] *= 1.8 if rule == "biweight" else 1.6
    zmax, nz = 3.0, 8192
    zb = np.linspace(0, zmax, nz)
    tab = np.tile(zb ** 2, (5, 1))
    th = _theta_unit_rate(theta0)
    z, lv = O.kde_samples(th, ev, 5, zmax)
    Lk, npass = O.event_loglik_kde(th, ev, tab, zmax, n_grid=1024, bandwidth=rule)
    Ls, _ = O.event_loglik_kde(th, ev, tab, zmax, n_grid=1024, bandwidth="scott")
    off = ev["ev_sample_off"]
    for i, runs in enumerate(_pixel_runs(ev)):
        tot = 0.0
        for r0, r1 in runs:
            live = np.isfinite(lv[r0:r1])
            v, zz = np.exp(lv[r0:r1][live]), z[r0:r1][live]
            z2 = _biweight_numpy(zz)
            h = z2 if rule == "biweight" else 1.06 * math.sqrt(z2) * zz.size ** (-0.2)
            assert h > 2 * zmax / 1023 and zz.min() - 5.5 * h > 0 and zz.max() + 5.5 * h < zmax, (h, zz.min())
            tot += np.sum(v * (zz ** 2 + h * h))
        assert npass[0, i] == len(runs)
        want = math.log(tot / (off[i + 1] - off[i]))
        assert Lk[0, i] == pytest.approx(want, abs=2e-6)
        assert abs(Ls[0, i] - Lk[0, i]) > 1e-4            # and it is not Scott's bandwidth


def test_kde_kernel_underflow_rule(theta0):
    """Reading R38: a Gaussian kernel value whose exponent is below -700 is zero.  A two-sample pixel that sits midway
    between two grid nodes with a bandwidth far below the grid step contributes (and is counted in npass) while the
    exponent at its nearest node is above -700, and neither contributes nor is counted once it is below; log L_i of
    the event does not notice either way (the other pixel carries it)."""
    th = _theta_unit_rate(theta0)
    H0, Om = th[0], th[1]
    zmax, G = 1.5, 64
    dz = zmax / (G - 1)
    zc = 20.5 * dz                                    # midway between nodes 20 and 21
    tab = np.ones((2, 256))
    res = {}
    for name, g2 in (("above", 640.0), ("below", 770.0)):
        h = 0.5 * dz / math.sqrt(2.0 * g2)            # exponent (d / h)^2 / 2 = g2 at the nearest nodes, d = dz / 2
        delta = h / (1.06 * 2 ** -0.2)                # Scott: h = 1.06 sd 2^(-1/5), sd = delta for two equal weights
        zs = np.array([zc - delta, zc + delta, 0.30, 0.34, 0.38, 0.42])
        dl = np.array([O.dL(z, H0, Om) for z in zs])
        ev = dict(ev_sample_off=np.array([0, 6], dtype=np.int64), dL=dl, m1z=np.full(6, 50.0), m2z=np.full(6, 38.0),
                  sample_row=np.array([0, 0, 1, 1, 1, 1], np.int32), log_pe_prior=np.zeros(6))
        res[name] = O.event_loglik_kde(th, ev, tab, zmax, n_grid=G, mode=O.EXACT, want_nused=True)
    (La, Pa, Ua), (Lb, Pb, Ub) = res["above"], res["below"]
    assert Pa[0, 0] == 2 and Ua[0, 0] == 6            # e^-640 at the nearest nodes: the pixel still counts
    assert Pb[0, 0] == 1 and Ub[0, 0] == 4            # e^-770: it does not
    assert La[0, 0] == pytest.approx(Lb[0, 0], abs=1e-12)
