"""CPU oracle for the dark-siren likelihood -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

ctypes wrapper around ``oracle/gwc_oracle.c`` (plain scalar C, see its header for the passages of
PAPER.md each function follows).  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs may import this package; the product package
``paper_2605_23538_b200`` never does.  Inputs and outputs are numpy arrays.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gwc_oracle.c")
_LIB = os.path.join(_HERE, "libgwc_oracle.so")

NPAR = 12
NPAR_MULTIPEAK = 16
TABLE, EXACT = 0, 1
MASS_MODELS = {"plpeak": 0, "multipeak": 1}


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (no FMA contraction, OpenMP parallel-for over theta)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
               "-D_GNU_SOURCE", "-o", _LIB, _SRC, "-lm"]
        subprocess.check_call(cmd)
    return _LIB


class _Los(C.Structure):
    _fields_ = [("n_rows", C.c_int64), ("n_z", C.c_int32), ("z_max", C.c_double), ("prec", C.c_int32),
                ("table", C.c_void_p)]


class _Events(C.Structure):
    _fields_ = [("n_events", C.c_int64), ("n_samples", C.c_int64), ("ev_sample_off", C.c_void_p),
                ("dL", C.c_void_p), ("m1z", C.c_void_p), ("m2z", C.c_void_p), ("log_pe_prior", C.c_void_p),
                ("sample_row", C.c_void_p)]


class _Inj(C.Structure):
    _fields_ = [("n_found", C.c_int64), ("n_draw", C.c_double), ("dL", C.c_void_p), ("m1z", C.c_void_p),
                ("m2z", C.c_void_p), ("log_pdraw", C.c_void_p)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        d, i32, i64, vp = C.c_double, C.c_int32, C.c_int64, C.c_void_p
        sig = {
            "orc_E": (d, [d, d]), "orc_D": (d, [d, d]), "orc_dL": (d, [d, d, d]), "orc_u_of_z": (d, [d, d]),
            "orc_z_of_u": (d, [d, d]), "orc_z_of_dL": (d, [d, d, d]),
            "orc_build_table": (None, [d, d, C.c_int, vp, vp, vp]),
            "orc_z_table": (C.c_int, [d, vp, vp, C.c_int, d, vp]),
            "orc_round_table_32": (None, [vp, C.c_int, d]),
            "orc_theta_valid": (C.c_int, [vp]), "orc_norm_pl": (d, [vp]), "orc_norm_g": (d, [vp]),
            "orc_p1": (d, [d, vp]), "orc_p2": (d, [d, d, vp]), "orc_psi": (d, [d, vp]),
            "orc_los_lerp": (d, [vp, i64, d]), "orc_los_allsky": (None, [vp, vp]),
            "orc_lse": (None, [vp, i64, vp, vp]),
            "orc_event_loglik": (C.c_int, [vp, i64, vp, vp, C.c_int, d, C.c_int, C.c_int, vp, vp, vp]),
            "orc_event_loglik_pixcut": (C.c_int, [vp, i64, vp, vp, C.c_int, d, C.c_int, C.c_int, d, vp, vp, vp, vp]),
            "orc_event_loglik_kde": (C.c_int, [vp, i64, vp, vp, C.c_int, d, C.c_int, C.c_int, C.c_int, d, C.c_int, vp, vp, vp]),
            "orc_kde_samples": (C.c_int, [vp, vp, i64, d, C.c_int, d, C.c_int, vp, vp]),
            "orc_selection_logxi": (C.c_int, [vp, i64, vp, vp, i32, d, C.c_int, d, C.c_int, C.c_int, vp, vp]),
            "orc_total_from_parts": (None, [vp, vp, i64, i64, vp]),
            "orc_pack_events": (i64, [i64, i64, vp, vp, vp, vp, vp, vp, vp]),
            "orc_cap_pixels": (i64, [i64, i64, i64, vp, vp, vp, i64, C.c_uint64, vp]),
            "orc_num_threads": (C.c_int, []), "orc_set_num_threads": (None, [C.c_int]),
            "orc_biweight_midvariance": (d, [vp, i64, vp]),
            "orc_set_mass_model": (None, [C.c_int]), "orc_npar": (C.c_int, []),
            "orc_mp_smooth": (d, [d, d, d]), "orc_mp_C": (d, [d, vp]), "orc_mp_N1": (d, [vp]),
        }
        for name, (res, args) in sig.items():
            f = getattr(L, name)
            f.restype, f.argtypes = res, args
        _lib = L
    return _lib


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _theta(theta):
    th = _f64(theta)
    if th.ndim == 1:
        th = th[None, :]
    assert th.shape[1] == lib().orc_npar()
    return th


class mass_model:
    """``with oracle.mass_model("multipeak"): ...`` -- theta rows have 16 columns inside the block (the 12 of the
    power-law+peak row, then delta_m, mu_g,low, sigma_g,low, lambda_g,low; R33-R36)."""

    def __init__(self, name):
        self.model = MASS_MODELS[name]

    def __enter__(self):
        lib().orc_set_mass_model(self.model)
        return self

    def __exit__(self, *exc):
        lib().orc_set_mass_model(0)
        return False


def mp_smooth(m, mmin, dm): return lib().orc_mp_smooth(m, mmin, dm)
def mp_C(m1, th): th = _f64(th); return lib().orc_mp_C(m1, _p(th))
def mp_N1(th): th = _f64(th); return lib().orc_mp_N1(_p(th))


# ---- scalar pieces (used by the pins) -------------------------------------------------------
def E(z, Om): return lib().orc_E(z, Om)
def D(z, Om): return lib().orc_D(z, Om)
def dL(z, H0, Om): return lib().orc_dL(z, H0, Om)
def u_of_z(z, Om): return lib().orc_u_of_z(z, Om)
def z_of_u(u, Om): return lib().orc_z_of_u(u, Om)
def z_of_dL(dl, H0, Om): return lib().orc_z_of_dL(dl, H0, Om)


def theta_valid(th): th = _f64(th); return bool(lib().orc_theta_valid(_p(th)))
def norm_pl(th): th = _f64(th); return lib().orc_norm_pl(_p(th))
def norm_g(th): th = _f64(th); return lib().orc_norm_g(_p(th))
def p1(m1, th): th = _f64(th); return lib().orc_p1(m1, _p(th))
def p2(m2, m1, th): th = _f64(th); return lib().orc_p2(m2, m1, _p(th))
def psi(z, th): th = _f64(th); return lib().orc_psi(z, _p(th))


def build_table(Om, z_max, M=1025):
    zt, dt, um = np.empty(M), np.empty(M), np.empty(1)
    lib().orc_build_table(Om, z_max, M, _p(zt), _p(dt), _p(um))
    return zt, dt, float(um[0])


def round_table_32(zt, dt, z_max):
    """The 32-bit storage of a cosmology table (R22): returns the values a look-up reads back."""
    M = len(zt)
    buf = np.concatenate([_f64(zt), _f64(dt)])
    lib().orc_round_table_32(_p(buf), M, float(z_max))
    return buf[:M].copy(), buf[M:].copy()


def z_table(u, zt, dt, umax):
    z = C.c_double(0.0)
    dead = lib().orc_z_table(u, _p(zt), _p(dt), len(zt), umax, C.addressof(z))
    return None if dead else z.value


def _los_struct(table, z_max):
    t = np.ascontiguousarray(table)
    assert t.ndim == 2 and t.dtype in (np.float64, np.float32)
    s = _Los(t.shape[0], t.shape[1], float(z_max), 0 if t.dtype == np.float64 else 1, t.ctypes.data)
    return s, t


def los_lerp(table, z_max, row, z):
    s, keep = _los_struct(table, z_max)
    return lib().orc_los_lerp(C.addressof(s), row, z)


def los_allsky(table, z_max):
    s, keep = _los_struct(table, z_max)
    out = np.empty(keep.shape[1])
    lib().orc_los_allsky(C.addressof(s), _p(out))
    return out


def lse(lw):
    lw = _f64(lw)
    a, b = C.c_double(0), C.c_double(0)
    lib().orc_lse(_p(lw), lw.size, C.addressof(a), C.addressof(b))
    return a.value, b.value


# ---- drivers -----------------------------------------------------------------------------
def event_loglik(theta, ev, los_table, los_z_max, *, mode=TABLE, z_max=None, n_nodes=1025, table_prec=0):
    """ev: dict with ev_sample_off (int64), dL, m1z, m2z (f64), sample_row (int32), log_pe_prior (f64|None).
    Returns logL, neff (f64 [n_theta, n_events]) and nlive (int64)."""
    th = _theta(theta)
    off = np.ascontiguousarray(ev["ev_sample_off"], dtype=np.int64)
    dl, m1, m2 = _f64(ev["dL"]), _f64(ev["m1z"]), _f64(ev["m2z"])
    row = np.ascontiguousarray(ev["sample_row"], dtype=np.int32)
    lpe = ev.get("log_pe_prior")
    lpe = None if lpe is None else _f64(lpe)
    ne = off.size - 1
    es = _Events(ne, dl.size, off.ctypes.data, dl.ctypes.data, m1.ctypes.data, m2.ctypes.data,
                 None if lpe is None else lpe.ctypes.data, row.ctypes.data)
    ls, keep = _los_struct(los_table, los_z_max)
    nt = th.shape[0]
    logL, neff, nlive = np.empty((nt, ne)), np.empty((nt, ne)), np.empty((nt, ne), dtype=np.int64)
    zm = float(los_z_max if z_max is None else z_max)
    rc = lib().orc_event_loglik(_p(th), nt, C.addressof(es), C.addressof(ls), mode, zm, n_nodes, table_prec,
                                _p(logL), _p(neff), _p(nlive))
    assert rc == 0
    return logL, neff, nlive


def event_loglik_pixcut(theta, ev, los_table, los_z_max, neff_min, *, mode=TABLE, z_max=None, n_nodes=1025,
                        table_prec=0):
    """Event term with the per-pixel N_eff cut of Eq. 8 (R25).  Same inputs as
    event_loglik plus the threshold; returns logL, neff (f64), nlive, npass (int64), all [n_theta, n_events]."""
    th = _theta(theta)
    off = np.ascontiguousarray(ev["ev_sample_off"], dtype=np.int64)
    dl, m1, m2 = _f64(ev["dL"]), _f64(ev["m1z"]), _f64(ev["m2z"])
    row = np.ascontiguousarray(ev["sample_row"], dtype=np.int32)
    lpe = ev.get("log_pe_prior")
    lpe = None if lpe is None else _f64(lpe)
    ne = off.size - 1
    es = _Events(ne, dl.size, off.ctypes.data, dl.ctypes.data, m1.ctypes.data, m2.ctypes.data,
                 None if lpe is None else lpe.ctypes.data, row.ctypes.data)
    ls, keep = _los_struct(los_table, los_z_max)
    nt = th.shape[0]
    logL, neff = np.empty((nt, ne)), np.empty((nt, ne))
    nlive, npass = np.empty((nt, ne), dtype=np.int64), np.empty((nt, ne), dtype=np.int64)
    zm = float(los_z_max if z_max is None else z_max)
    rc = lib().orc_event_loglik_pixcut(_p(th), nt, C.addressof(es), C.addressof(ls), mode, zm, n_nodes, table_prec,
                                       float(neff_min), _p(logL), _p(neff), _p(nlive), _p(npass))
    assert rc == 0
    return logL, neff, nlive, npass


BW_RULES = {"scott": 0, "silverman": 1, "biweight": 2, "biweight_scott": 3}


def biweight_midvariance(x):
    """Eq. D3-D4 of a sample; NaN when the MAD is zero."""
    x = _f64(x)
    work = np.empty(2 * max(x.size, 1))
    return lib().orc_biweight_midvariance(_p(x), x.size, _p(work))


def _events_struct(ev):
    off = np.ascontiguousarray(ev["ev_sample_off"], dtype=np.int64)
    dl, m1, m2 = _f64(ev["dL"]), _f64(ev["m1z"]), _f64(ev["m2z"])
    row = np.ascontiguousarray(ev["sample_row"], dtype=np.int32)
    lpe = ev.get("log_pe_prior")
    lpe = None if lpe is None else _f64(lpe)
    es = _Events(off.size - 1, dl.size, off.ctypes.data, dl.ctypes.data, m1.ctypes.data, m2.ctypes.data,
                 None if lpe is None else lpe.ctypes.data, row.ctypes.data)
    return es, (off, dl, m1, m2, row, lpe)


def event_loglik_kde(theta, ev, los_table, los_z_max, *, n_grid=256, neff_min=0.0, mode=TABLE, z_max=None,
                     n_nodes=1025, table_prec=0, want_nused=False, bandwidth="scott"):
    """Event term with the paper's KDE numerator (Eq. 5-7, D1; R26-R30).  Returns logL (f64) and npass
    (int64), both [n_theta, n_events]."""
    th = _theta(theta)
    es, keep_ev = _events_struct(ev)
    ls, keep = _los_struct(los_table, los_z_max)
    nt, ne = th.shape[0], es.n_events
    logL, npass = np.empty((nt, ne)), np.empty((nt, ne), dtype=np.int64)
    nused = np.empty((nt, ne), dtype=np.int64)
    zm = float(los_z_max if z_max is None else z_max)
    rc = lib().orc_event_loglik_kde(_p(th), nt, C.addressof(es), C.addressof(ls), mode, zm, n_nodes, table_prec,
                                    int(n_grid), float(neff_min), BW_RULES[bandwidth], _p(logL),
                                    _p(npass), _p(nused))
    assert rc == 0
    if want_nused:
        return logL, npass, nused
    return logL, npass


def kde_samples(theta1, ev, n_rows, los_z_max, *, mode=TABLE, z_max=None, n_nodes=1025):
    """Per-sample (z_k, log v_k) of ONE theta: the inputs of the KDE (v = Eq. 7's weight without the z prior)."""
    th = _theta(theta1)
    assert th.shape[0] == 1
    es, keep_ev = _events_struct(ev)
    n = es.n_samples
    z, lv = np.empty(n), np.empty(n)
    zm = float(los_z_max if z_max is None else z_max)
    rc = lib().orc_kde_samples(_p(th), C.addressof(es), int(n_rows), float(los_z_max), mode, zm, n_nodes, _p(z), _p(lv))
    assert rc == 0
    return z, lv


def selection_logxi(theta, inj, allsky, los_z_max, *, mode=TABLE, z_max=None, n_nodes=1025, table_prec=0):
    """inj: dict with dL, m1z, m2z, log_pdraw (f64) and n_draw.  Returns logxi, neff_inj [n_theta]."""
    th = _theta(theta)
    dl, m1, m2, lp = _f64(inj["dL"]), _f64(inj["m1z"]), _f64(inj["m2z"]), _f64(inj["log_pdraw"])
    a = _f64(allsky)
    s = _Inj(dl.size, float(inj["n_draw"]), dl.ctypes.data, m1.ctypes.data, m2.ctypes.data, lp.ctypes.data)
    nt = th.shape[0]
    logxi, neff = np.empty(nt), np.empty(nt)
    zm = float(los_z_max if z_max is None else z_max)
    rc = lib().orc_selection_logxi(_p(th), nt, C.addressof(s), _p(a), a.size, float(los_z_max), mode, zm, n_nodes,
                                   table_prec, _p(logxi), _p(neff))
    assert rc == 0
    return logxi, neff


def total_from_parts(logL, logxi):
    logL, logxi = _f64(logL), _f64(logxi)
    nt, ne = logL.shape
    out = np.empty(nt)
    lib().orc_total_from_parts(_p(logL), _p(logxi), nt, ne, _p(out))
    return out


def total_loglik(theta, ev, inj, los_table, los_z_max, allsky=None, **kw):
    if allsky is None:
        allsky = los_allsky(los_table, los_z_max)
    logL, _, _ = event_loglik(theta, ev, los_table, los_z_max, **kw)
    logxi, _ = selection_logxi(theta, inj, allsky, los_z_max, **kw)
    return total_from_parts(logL, logxi)


def pack_events(event_id, row, n_events):
    eid = np.ascontiguousarray(event_id, dtype=np.int32)
    rw = np.ascontiguousarray(row, dtype=np.int32)
    n = eid.size
    perm = np.empty(n, dtype=np.int64)
    eso = np.empty(n_events + 1, dtype=np.int64)
    epo = np.empty(n_events + 1, dtype=np.int64)
    epr = np.empty(max(n, 1), dtype=np.int32)
    pso = np.empty(n + 1, dtype=np.int64)
    npx = lib().orc_pack_events(n, n_events, _p(eid), _p(rw), _p(perm), _p(eso), _p(epo), _p(epr), _p(pso))
    assert npx >= 0
    return dict(perm=perm, ev_sample_off=eso, ev_pix_off=epo, ev_pix_rows=epr[:npx].copy(),
                pix_sample_off=pso[:npx + 1].copy(), n_pixrefs=int(npx))


def num_threads():
    return lib().orc_num_threads()


def set_num_threads(n):
    lib().orc_set_num_threads(int(n))


def cap_pixels(perm, ev_sample_off, pix_sample_off, cap, seed):
    """Per-pixel sample cap on a packed catalogue (R31).  Returns perm_kept,
    ev_sample_off', pix_sample_off' (new arrays)."""
    perm = np.ascontiguousarray(perm, dtype=np.int64)
    evo = np.array(ev_sample_off, dtype=np.int64, copy=True)
    pxo = np.array(pix_sample_off, dtype=np.int64, copy=True)
    out = np.empty(max(perm.size, 1), dtype=np.int64)
    nk = lib().orc_cap_pixels(perm.size, evo.size - 1, pxo.size - 1, _p(perm), _p(evo), _p(pxo), int(cap),
                              int(seed) & 0xFFFFFFFFFFFFFFFF, _p(out))
    assert nk >= 0
    return out[:nk].copy(), evo, pxo

