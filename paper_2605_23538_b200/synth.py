"""Seeded synthetic workloads shaped like the paper's catalogues.

This module only *makes inputs*: GW events with ragged posterior samples and sky pixels, a
galaxy-catalogue line-of-sight table, a found-injection set and hyper-parameter batches, for the five
configurations of BASELINE.json.  It serves both the CUDA path and the CPU oracle and holds none of
the likelihood's arithmetic -- neither of them imports anything from here but arrays.  The draws need
a fiducial cosmology and population to be realistic; those few formulas are restated here in torch,
on a fine grid, independently of both implementations.

The paper's own data (O5 mock catalogue PAPER.md:245, GWTC-4.0 + GLADE+ + O4 injections :249) is
not public (:241); these generators stand in for it.  Everything is a pure function of
(config, seed): a counter-based splitmix64 stream keyed by (seed, stream id, index) gives the same
uniforms on CPU and CUDA.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace
from typing import Dict, Optional, Tuple

import torch

C_KMS = 299792.458
NPAR = 12
# fiducial truth theta_0: H0, Om, alpha, beta, mmin, mmax, mu, sigma, lambda, gamma, kappa, zp
THETA0 = (70.0, 0.3, 3.4, 1.1, 5.0, 100.0, 35.0, 4.0, 0.04, 2.7, 2.9, 1.9)
DEFAULT_SEED = 20260915

_M64 = (1 << 64) - 1


def _s64(x: int) -> int:
    x &= _M64
    return x - (1 << 64) if x >= (1 << 63) else x


_GAMMA = _s64(0x9E3779B97F4A7C15)
_K1 = _s64(0xBF58476D1CE4E5B9)
_K2 = _s64(0x94D049BB133111EB)
_KS = _s64(0xD6E8FEB86659FD93)


def _lsr(x: torch.Tensor, s: int) -> torch.Tensor:
    return (x >> s) & ((1 << (64 - s)) - 1)


def _bits(seed: int, stream: int, n: int, device, start: int = 0) -> torch.Tensor:
    """splitmix64 of counter (seed, stream, start+i); int64 arithmetic wraps like uint64."""
    base = _s64((seed * 0x632BE59BD9B4E019 + stream * 0xD1342543DE82EF95) & _M64)
    x = torch.arange(start, start + n, dtype=torch.int64, device=device) * _GAMMA + base
    x = (x ^ _lsr(x, 30)) * _K1
    x = (x ^ _lsr(x, 27)) * _K2
    x = x ^ _lsr(x, 31)
    # second round decorrelates neighbouring streams
    x = (x + _KS)
    x = (x ^ _lsr(x, 30)) * _K1
    x = (x ^ _lsr(x, 27)) * _K2
    return x ^ _lsr(x, 31)


def uniform(seed: int, stream: int, n: int, device, start: int = 0) -> torch.Tensor:
    """float64 uniforms in (0,1)."""
    b = _lsr(_bits(seed, stream, n, device, start), 11)
    return (b.to(torch.float64) + 0.5) * (2.0 ** -53)


def normal(seed: int, stream: int, n: int, device, start: int = 0) -> torch.Tensor:
    u = uniform(seed, stream, n, device, start)
    return math.sqrt(2.0) * torch.erfinv(2.0 * u - 1.0)


def _interp(x: torch.Tensor, xp: torch.Tensor, fp: torch.Tensor) -> torch.Tensor:
    """np.interp for monotone xp."""
    i = torch.searchsorted(xp, x.contiguous(), right=True).clamp(1, xp.numel() - 1)
    x0, x1 = xp[i - 1], xp[i]
    t = ((x - x0) / (x1 - x0)).clamp(0.0, 1.0)
    return fp[i - 1] + t * (fp[i] - fp[i - 1])


def _cumtrapz(y: torch.Tensor, dx: float) -> torch.Tensor:
    c = torch.cumsum(0.5 * (y[1:] + y[:-1]) * dx, 0)
    return torch.cat([torch.zeros(1, dtype=y.dtype, device=y.device), c])


class _Fiducial:
    """Fiducial cosmology/population on a fine grid (generator-side only)."""

    def __init__(self, z_max: float, device, th=THETA0, n=40001):
        self.th = th
        self.device = device
        H0, Om = th[0], th[1]
        self.zg = torch.linspace(0.0, z_max, n, dtype=torch.float64, device=device)
        dz = z_max / (n - 1)
        self.Eg = torch.sqrt(Om * (1 + self.zg) ** 3 + (1 - Om))
        # cumulative trapezoid with the Euler-Maclaurin end correction -h^2/12 (f'(z) - f'(0)), f = 1/E
        fp = -1.5 * Om * (1 + self.zg) ** 2 / self.Eg ** 3
        self.Dg = _cumtrapz(1.0 / self.Eg, dz) - dz * dz / 12.0 * (fp - fp[0])
        self.dLg = (1 + self.zg) * (C_KMS / H0) * self.Dg
        self.dz = dz
        self.z_max = z_max

    def E(self, z):
        return torch.sqrt(self.th[1] * (1 + z) ** 3 + (1 - self.th[1]))

    def D(self, z):
        return _interp(z, self.zg, self.Dg)

    def dL(self, z):
        return (1 + z) * (C_KMS / self.th[0]) * self.D(z)

    def ddL_dz(self, z):
        return (C_KMS / self.th[0]) * (self.D(z) + (1 + z) / self.E(z))

    def psi(self, z):
        g, k, zp = self.th[9], self.th[10], self.th[11]
        return (1 + (1 + zp) ** (-(g + k))) * (1 + z) ** g / (1 + ((1 + z) / (1 + zp)) ** (g + k))

    # population at theta_0
    def norm_pl(self):
        a, lo, hi = self.th[2], self.th[4], self.th[5]
        return (1 - a) / (hi ** (1 - a) - lo ** (1 - a))

    def norm_g(self):
        lo, hi, mu, s = self.th[4], self.th[5], self.th[6], self.th[7]
        return 1.0 / (0.5 * (math.erf((hi - mu) / (s * math.sqrt(2))) - math.erf((lo - mu) / (s * math.sqrt(2)))))

    def log_p_m1m2(self, m1, m2):
        a, b, lo, hi, mu, s, lam = self.th[2], self.th[3], self.th[4], self.th[5], self.th[6], self.th[7], self.th[8]
        p1 = (1 - lam) * self.norm_pl() * m1 ** (-a) + lam * self.norm_g() * torch.exp(-0.5 * ((m1 - mu) / s) ** 2) / (
            s * math.sqrt(2 * math.pi))
        p2 = (b + 1) * m2 ** b / (m1 ** (b + 1) - lo ** (b + 1))
        return torch.log(p1) + torch.log(p2)

    def draw_masses(self, u_mix, u_m1, u_m2):
        a, b, lo, hi, mu, s, lam = self.th[2], self.th[3], self.th[4], self.th[5], self.th[6], self.th[7], self.th[8]
        # power-law branch, inverse CDF
        m_pl = (lo ** (1 - a) + u_m1 * (hi ** (1 - a) - lo ** (1 - a))) ** (1.0 / (1 - a))
        # truncated Gaussian branch, inverse CDF
        Fa = 0.5 * (1 + math.erf((lo - mu) / (s * math.sqrt(2))))
        Fb = 0.5 * (1 + math.erf((hi - mu) / (s * math.sqrt(2))))
        m_g = mu + s * math.sqrt(2.0) * torch.erfinv(2 * (Fa + u_m1 * (Fb - Fa)) - 1)
        m1 = torch.where(u_mix < lam, m_g, m_pl).clamp(lo * (1 + 1e-12), hi)
        m2 = (lo ** (b + 1) + u_m2 * (m1 ** (b + 1) - lo ** (b + 1))) ** (1.0 / (b + 1))
        m2 = torch.minimum(m2.clamp_min(lo), m1)
        return m1, m2


@dataclass(frozen=True)
class Spec:
    """One workload configuration (BASELINE.json `configs`, sizes per SURVEY.md section 8d)."""
    name: str
    n_theta: int
    n_events: int
    samples: Tuple[int, int]            # per-event S_i log-uniform in [lo, hi]
    pixels: Tuple[int, int]             # per-event P_i log-uniform in [lo, hi]
    los_rows: int
    n_z: int
    z_max: float
    z_c: float                          # completeness sigmoid centre
    n_inj: int
    r0: float                           # SNR proxy horizon scale, Mpc
    ev_z: Tuple[float, float]           # true-redshift range of events
    z_law: str                          # "z2" or "md"
    theta_box: Dict[str, Tuple[float, float]] = field(default_factory=dict)
    los_dtype: str = "f64"              # dtype of the primary LOS table ("f64" | "f32")
    big_frac: float = 0.0               # stress: fraction of events with big_samples/big_pixels
    big_samples: int = 0
    big_pixels: int = 0
    n_gal: int = 50


_BOX6 = {"H0": (20.0, 140.0), "Om": (0.1, 0.5), "alpha": (1.5, 5.0), "mu": (25.0, 45.0), "sigma": (2.0, 8.0),
         "lambda": (0.0, 0.1)}

CONFIGS: Dict[str, Spec] = {
    "tiny": Spec("tiny", 16, 4, (256, 256), (8, 8), 8, 512, 1.5, 0.3, 10_000, 100.0, (0.05, 0.5), "z2",
                 {"H0": (40.0, 120.0)}, "f64"),
    "o4": Spec("o4", 256, 200, (1024, 4096), (16, 512), 20_000, 1000, 2.0, 0.5, 100_000, 150.0, (0.05, 1.0), "z2",
               {"H0": (40.0, 120.0), "alpha": (1.5, 5.0), "mu": (25.0, 45.0)}, "f64"),
    "production": Spec("production", 1024, 1000, (4096, 4096), (16, 2048), 100_000, 1000, 2.0, 0.5, 1_000_000, 330.0,
                       (0.05, 1.5), "md", dict(_BOX6), "f32"),
    "o5": Spec("o5", 4096, 5000, (5000, 5000), (16, 4096), 200_000, 1000, 2.0, 0.5, 5_000_000, 330.0, (0.05, 1.5),
               "md", dict(_BOX6), "f32"),
    "stress": Spec("stress", 1024, 1000, (512, 512), (16, 16), 100_000, 1000, 2.0, 0.5, 1_000_000, 330.0, (0.05, 1.5),
                   "md", {**_BOX6, "H0": (20.0, 200.0)}, "f64", big_frac=0.02, big_samples=32768, big_pixels=8192),
}

_PAR_INDEX = {"H0": 0, "Om": 1, "alpha": 2, "beta": 3, "mmin": 4, "mmax": 5, "mu": 6, "sigma": 7, "lambda": 8,
              "gamma": 9, "kappa": 10, "zp": 11}


def scaled(spec: Spec, **kw) -> Spec:
    """A smaller (or otherwise altered) copy of a configuration, for tests."""
    return replace(spec, **kw)


@dataclass
class Workload:
    spec: Spec
    seed: int
    theta: torch.Tensor                 # [n_theta, 12] f64
    ev: Dict[str, Optional[torch.Tensor]]   # ev_sample_off i64, dL/m1z/m2z f64, sample_row i32, log_pe_prior None
    ev_pixels: torch.Tensor             # [n_events] i64 number of pixels requested per event
    inj: Dict[str, object]              # dL, m1z, m2z, log_pdraw f64; n_draw float
    los: torch.Tensor                   # [rows, n_z] primary table (spec.los_dtype)
    los_f64: Optional[torch.Tensor]     # f64 copy when the primary is f32 and it was kept
    truth: Dict[str, torch.Tensor]      # z, m1, m2 of the events (diagnostics only)

    @property
    def n_samples(self) -> int:
        return int(self.ev["dL"].numel())

    def los_f32(self) -> torch.Tensor:
        return self.los if self.los.dtype == torch.float32 else self.los.to(torch.float32)


# ---------------------------------------------------------------------------------------------
def make_theta(spec: Spec, seed: int, device, n_theta: Optional[int] = None, stream: int = 900) -> torch.Tensor:
    n = spec.n_theta if n_theta is None else n_theta
    th = torch.tensor(THETA0, dtype=torch.float64, device=device).repeat(n, 1)
    for j, (name, (lo, hi)) in enumerate(sorted(spec.theta_box.items())):
        u = uniform(seed, stream + j, n, device)
        th[:, _PAR_INDEX[name]] = lo + (hi - lo) * u
    return th


# Table III of the paper as a MULTIPEAK theta row (include/gwc.h: the 12 power-law+peak columns with
# the HIGH peak in mu / sigma and lambda_g in lambda, then delta_m, mu_g,low, sigma_g,low, lambda_g,low)
THETA_TABLE3_MULTIPEAK = (67.4, 0.315, 2.9, 1.0, 4.6, 86.3, 30.7, 6.3, 0.4, 3.3, 2.9, 2.5, 4.8, 9.7, 0.7, 0.8)
_MP_BOX = {12: (0.5, 8.0), 13: (7.0, 12.0), 14: (0.4, 2.5), 15: (0.0, 1.0)}   # delta_m, mu_low, sigma_low, lambda_low


def make_theta_multipeak(spec: Spec, seed: int, device, n_theta: Optional[int] = None, stream: int = 950,
                         mmin: float = 4.6) -> torch.Tensor:
    """A MULTIPEAK theta batch: the config's box on the first 12 columns (make_theta), Table III's values for what the
    box leaves fixed (mmin lowered to `mmin` so that the synthetic catalogues, drawn from a population that starts at
    5 Msun, put samples inside the smoothing window), the four extra columns uniform in _MP_BOX.  Row 0 is Table III."""
    n = spec.n_theta if n_theta is None else n_theta
    th = torch.tensor(THETA_TABLE3_MULTIPEAK, dtype=torch.float64, device=device).repeat(n, 1)
    box = make_theta(spec, seed, device, n)
    for name in spec.theta_box:
        j = _PAR_INDEX[name]
        th[:, j] = box[:, j]
    th[:, 4] = mmin
    for j, (lo, hi) in sorted(_MP_BOX.items()):
        th[:, j] = lo + (hi - lo) * uniform(seed, stream + j, n, device)
    th[0] = torch.tensor(THETA_TABLE3_MULTIPEAK, dtype=torch.float64, device=device)
    return th


def make_los(spec: Spec, seed: int, device, rows_chunk: int = 1024) -> torch.Tensor:
    """LOS table [rows][n_z] f64: Schechter-weighted Gaussian galaxies + uncatalogued volume term."""
    fid = _Fiducial(spec.z_max, device)
    zb = torch.linspace(0.0, spec.z_max, spec.n_z, dtype=torch.float64, device=device)
    dzb = spec.z_max / (spec.n_z - 1)
    pv = fid.D(zb) ** 2 / fid.E(zb)
    pv = pv / torch.trapezoid(pv, dx=dzb)
    comp = torch.sigmoid((spec.z_c - zb) / 0.05)
    cat = comp * pv
    A = torch.trapezoid(cat, dx=dzb)
    cdf = _cumtrapz(cat, dzb)
    cdf = cdf / cdf[-1]
    # Schechter luminosity weights x^aS e^-x on [0.05, 30], tabulated inverse CDF in log x
    lx = torch.linspace(math.log(0.05), math.log(30.0), 4001, dtype=torch.float64, device=device)
    pdf_l = torch.exp(lx * (-1.07 + 1.0) - torch.exp(lx))       # x^aS e^-x * x (dx = x dlogx)
    cdf_l = _cumtrapz(pdf_l, float(lx[1] - lx[0]))
    cdf_l = cdf_l / cdf_l[-1]
    G = spec.n_gal
    out = torch.empty((spec.los_rows, spec.n_z), dtype=torch.float64, device=device)
    unc = (1.0 - comp) * pv
    for r0 in range(0, spec.los_rows, rows_chunk):
        r1 = min(spec.los_rows, r0 + rows_chunk)
        n = (r1 - r0) * G
        zg = _interp(uniform(seed, 100, n, device, start=r0 * G), cdf, zb).view(-1, G, 1)
        xg = torch.exp(_interp(uniform(seed, 101, n, device, start=r0 * G), cdf_l, lx)).view(-1, G, 1)
        sg = 0.01 * (1.0 + zg)
        gauss = torch.exp(-0.5 * ((zb.view(1, 1, -1) - zg) / sg) ** 2) / (sg * math.sqrt(2 * math.pi))
        out[r0:r1] = A * (xg * gauss).sum(1) / xg.sum(1) + unc
    return out


def _z_sampler(spec_law: str, lo: float, hi: float, fid: _Fiducial):
    """Returns (draw(u)->z, logpdf(z)) for the redshift law on [lo, hi]."""
    if spec_law == "z2":
        a3, b3 = lo ** 3, hi ** 3

        def draw(u):
            return (a3 + u * (b3 - a3)) ** (1.0 / 3.0)

        def logpdf(z):
            return torch.log(3.0 * z * z / (b3 - a3))
        return draw, logpdf
    # "md": comoving-volume rate, Madau-Dickinson gamma=2.7
    zz = torch.linspace(lo, hi, 20001, dtype=torch.float64, device=fid.device)
    pdf = fid.D(zz) ** 2 / fid.E(zz) * fid.psi(zz) / (1 + zz)
    dzz = (hi - lo) / 20000
    cdf = _cumtrapz(pdf, dzz)
    norm = float(cdf[-1])
    cdf = cdf / cdf[-1]

    def draw(u):
        return _interp(u, cdf, zz)

    def logpdf(z):
        return torch.log(fid.D(z) ** 2 / fid.E(z) * fid.psi(z) / (1 + z) / norm)
    return draw, logpdf


def _theta_cdf_inv(device):
    """Inverse CDF of the Finn-Chernoff-like orientation factor P(T) = 5 T (4-T)^3 / 256 on [0,4]."""
    t = torch.linspace(0.0, 4.0, 8001, dtype=torch.float64, device=device)
    cdf = _cumtrapz(5.0 * t * (4.0 - t) ** 3 / 256.0, 4.0 / 8000)
    return t, cdf / cdf[-1]


def _candidates(spec: Spec, seed: int, stream0: int, start: int, n: int, fid: _Fiducial, zdraw, tgrid, tcdf):
    """n population draws (z, m1, m2) at theta_0 with the observed-SNR proxy rho."""
    dev = fid.device
    z = zdraw(uniform(seed, stream0 + 0, n, dev, start))
    m1, m2 = fid.draw_masses(uniform(seed, stream0 + 1, n, dev, start), uniform(seed, stream0 + 2, n, dev, start),
                             uniform(seed, stream0 + 3, n, dev, start))
    Th = _interp(uniform(seed, stream0 + 4, n, dev, start), tcdf, tgrid)
    dl = fid.dL(z)
    mc = (m1 * m2) ** 0.6 / (m1 + m2) ** 0.2
    rho = 8.0 * Th * (spec.r0 / dl) * (mc * (1 + z) / 1.2) ** (5.0 / 6.0) + normal(seed, stream0 + 5, n, dev, start)
    return z, m1, m2, dl, rho


def _found(spec: Spec, seed: int, stream0: int, n_want: int, fid: _Fiducial, zdraw, batch: int):
    """Draw until n_want candidates pass rho > 12; returns them and the number tried."""
    tgrid, tcdf = _theta_cdf_inv(fid.device)
    keep, got, start = [], 0, 0
    while got < n_want:
        z, m1, m2, dl, rho = _candidates(spec, seed, stream0, start, batch, fid, zdraw, tgrid, tcdf)
        idx = torch.nonzero(rho > 12.0).flatten()
        if got + idx.numel() >= n_want:
            idx = idx[: n_want - got]
            n_draw = start + int(idx[-1]) + 1
            keep.append((z[idx], m1[idx], m2[idx], dl[idx]))
            got = n_want
            break
        keep.append((z[idx], m1[idx], m2[idx], dl[idx]))
        got += idx.numel()
        start += batch
        if start > 4_000_000_000:
            raise RuntimeError("detection fraction too small for this configuration")
    z, m1, m2, dl = (torch.cat([k[i] for k in keep]) for i in range(4))
    return z, m1, m2, dl, n_draw


def _log_uniform_int(u: torch.Tensor, lo: int, hi: int) -> torch.Tensor:
    if lo == hi:
        return torch.full_like(u, lo, dtype=torch.int64)
    v = torch.exp(math.log(lo) + u * (math.log(hi) - math.log(lo)))
    return v.round().to(torch.int64).clamp(lo, hi)


def make_events(spec: Spec, seed: int, device, batch: int = 1 << 20):
    fid = _Fiducial(spec.z_max, device)
    zdraw, _ = _z_sampler(spec.z_law, spec.ev_z[0], spec.ev_z[1], fid)
    z, m1, m2, dl, _ = _found(spec, seed, 200, spec.n_events, fid, zdraw, batch)
    E = spec.n_events
    S = _log_uniform_int(uniform(seed, 210, E, device), *spec.samples)
    P = _log_uniform_int(uniform(seed, 211, E, device), *spec.pixels)
    if spec.big_frac > 0.0:
        nbig = max(1, int(round(spec.big_frac * E)))
        # deterministic, spread through the catalogue
        big = torch.zeros(E, dtype=torch.bool, device=device)
        big[torch.linspace(0, E - 1, nbig, device=device).round().to(torch.int64)] = True
        S = torch.where(big, torch.full_like(S, spec.big_samples), S)
        P = torch.where(big, torch.full_like(P, spec.big_pixels), P)
    P = torch.minimum(P, torch.full_like(P, spec.los_rows))
    off = torch.zeros(E + 1, dtype=torch.int64, device=device)
    off[1:] = torch.cumsum(S, 0)
    n = int(off[-1])
    ev_of = torch.repeat_interleave(torch.arange(E, device=device), S)
    dLs = dl[ev_of] * torch.exp(0.2 * normal(seed, 220, n, device))
    m1z = (m1 * (1 + z))[ev_of] * (1.0 + 0.05 * normal(seed, 221, n, device))
    m2z = (m2 * (1 + z))[ev_of] * (1.0 + 0.05 * normal(seed, 222, n, device))
    hi_m = torch.maximum(m1z, m2z)
    lo_m = torch.minimum(m1z, m2z)
    m1z, m2z = hi_m, lo_m
    # sky pixels: P_i consecutive rows from a random start; rank drawn ~ exp(-r/(P/6)) (sky-area-like skew)
    start = (uniform(seed, 212, E, device) * spec.los_rows).to(torch.int64).clamp(0, spec.los_rows - 1)
    Pf = P.to(torch.float64)[ev_of]
    tau = Pf / 6.0
    u = uniform(seed, 223, n, device)
    rank = torch.floor(-tau * torch.log1p(-u * (1.0 - torch.exp(-Pf / tau)))).to(torch.int64)
    rank = torch.minimum(rank.clamp_min(0), P[ev_of] - 1)
    row = (start[ev_of] + rank) % spec.los_rows
    # stored sorted by (event, row); ties keep draw order
    key = ev_of * spec.los_rows + row
    order = torch.sort(key, stable=True).indices
    ev = {
        "ev_sample_off": off,
        "dL": dLs[order].contiguous(),
        "m1z": m1z[order].contiguous(),
        "m2z": m2z[order].contiguous(),
        "sample_row": row[order].to(torch.int32).contiguous(),
        "log_pe_prior": None,
    }
    return ev, P, {"z": z, "m1": m1, "m2": m2}


def make_injections(spec: Spec, seed: int, device, batch: int = 1 << 22):
    fid = _Fiducial(spec.z_max, device)
    lo = 1e-4
    zdraw, zlogpdf = _z_sampler(spec.z_law, lo, spec.z_max, fid)
    z, m1, m2, dl, n_draw = _found(spec, seed, 300, spec.n_inj, fid, zdraw, batch)
    # draw density transformed to (dL, m1z, m2z): divide by (1+z)^2 d(dL)/dz
    log_pdraw = zlogpdf(z) + fid.log_p_m1m2(m1, m2) - 2.0 * torch.log1p(z) - torch.log(fid.ddL_dz(z))
    return {"dL": dl.contiguous(), "m1z": (m1 * (1 + z)).contiguous(), "m2z": (m2 * (1 + z)).contiguous(),
            "log_pdraw": log_pdraw.contiguous(), "n_draw": float(n_draw)}


def make_workload(config, seed: int = DEFAULT_SEED, device="cpu", keep_f64_los: bool = True) -> Workload:
    spec = CONFIGS[config] if isinstance(config, str) else config
    device = torch.device(device)
    theta = make_theta(spec, seed, device)
    los64 = make_los(spec, seed, device)
    ev, P, truth = make_events(spec, seed, device)
    inj = make_injections(spec, seed, device)
    if spec.los_dtype == "f32":
        los = los64.to(torch.float32)
        if not keep_f64_los:
            los64 = None
    else:
        los = los64
    return Workload(spec, seed, theta, ev, P, inj, los, los64, truth)


def to_numpy(d: Dict[str, object]) -> Dict[str, object]:
    """Host numpy view of an event / injection dict (for the oracle)."""
    out = {}
    for k, v in d.items():
        out[k] = v.detach().cpu().numpy() if isinstance(v, torch.Tensor) else v
    return out
