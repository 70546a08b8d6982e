"""Thin Python binding of the C ABI in include/gwc.h (argument marshalling only).

Every function here has the name of the C entry point it calls and does nothing but turn torch
tensors into device pointers; every step of the path runs in the CUDA kernels of libgwc.so.  There is
no CPU fallback: loading fails loudly when the library has not been built
(`python -m paper_2605_23538_b200.build`), and creating a context fails without a CUDA device.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Dict, Optional

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libgwc.so")

NPAR = 12
NPAR_MULTIPEAK = 16
MASS_MODELS = {"plpeak": 0, "multipeak": 1}
F64, F32 = 0, 1
OK, ERR_INVALID_ARG, ERR_SHAPE, ERR_DOMAIN, ERR_NOT_BUILT, ERR_NOMEM, ERR_CUDA, ERR_RANGE = range(8)
_STATUS = ["GWC_OK", "GWC_ERR_INVALID_ARG", "GWC_ERR_SHAPE", "GWC_ERR_DOMAIN", "GWC_ERR_NOT_BUILT", "GWC_ERR_NOMEM",
           "GWC_ERR_CUDA", "GWC_ERR_RANGE"]

EXPORTS = ["gwc_create", "gwc_destroy", "gwc_check", "gwc_last_error", "gwc_launch_count", "gwc_set_mass_model",
           "gwc_theta_len", "gwc_build_cosmo",
           "gwc_export_cosmo", "gwc_pack_events", "gwc_cap_pixels", "gwc_los_allsky", "gwc_event_loglik", "gwc_event_loglik_pixcut", "gwc_event_loglik_kde",
           "gwc_selection_logxi",
           "gwc_combine_total", "gwc_total_loglik", "gwc_total_loglik_pixcut", "gwc_total_loglik_kde", "gwc_total_loglik_host", "gwc_cache_catalogue", "gwc_set_timing", "gwc_get_timing",
           "gwc_probe_fp64", "gwc_math_selftest", "gwc_los_allsky_static", "gwc_los_allsky_static_error",
           "gwc_combine_sharded", "gwc_combine_sharded_host", "gwc_set_omega_hint"]
OMEGA_HINTS = {"detect": 0, "varies": 1, "single": 2}
ALLSKY_STATIC_ROWS_PER_PART = 512
ALLSKY_STATIC_MAX_DOUBLES = 1 << 19


BW_RULES = {"scott": 0, "silverman": 1, "biweight": 2, "biweight_scott": 3}


class GwcError(RuntimeError):
    def __init__(self, status: int, text: str):
        super().__init__("%s: %s" % (_STATUS[status] if 0 <= status < len(_STATUS) else status, text))
        self.status = status


class Events(C.Structure):
    _fields_ = [("n_events", C.c_int64), ("n_samples", C.c_int64), ("ev_sample_off", C.c_void_p),
                ("dL", C.c_void_p), ("m1z", C.c_void_p), ("m2z", C.c_void_p), ("log_pe_prior", C.c_void_p),
                ("sample_row", C.c_void_p), ("ev_pix_off", C.c_void_p), ("ev_pix_rows", C.c_void_p)]


class Los(C.Structure):
    _fields_ = [("n_rows", C.c_int64), ("n_z", C.c_int32), ("z_max", C.c_double), ("prec", C.c_int),
                ("table", C.c_void_p), ("allsky", C.c_void_p)]


class Injections(C.Structure):
    _fields_ = [("n_found", C.c_int64), ("n_draw", C.c_double), ("dL", C.c_void_p), ("m1z", C.c_void_p),
                ("m2z", C.c_void_p), ("log_pdraw", C.c_void_p)]


_lib = None


def load():
    """dlopen libgwc.so and declare the signatures of include/gwc.h."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError("libgwc.so is not built (run `python -m paper_2605_23538_b200.build`); "
                          "there is no CPU fallback for the CUDA path")
    L = C.CDLL(LIB_PATH)
    vp, i64, i32, dbl, ci = C.c_void_p, C.c_int64, C.c_int32, C.c_double, C.c_int
    sig = {
        "gwc_create": (ci, [C.POINTER(vp), ci, vp]),
        "gwc_destroy": (None, [vp]),
        "gwc_check": (ci, [vp]),
        "gwc_last_error": (C.c_char_p, [vp]),
        "gwc_launch_count": (i64, [vp]),
        "gwc_set_mass_model": (ci, [vp, ci]),
        "gwc_theta_len": (i32, [ci]),
        "gwc_set_omega_hint": (ci, [vp, ci]),
        "gwc_build_cosmo": (ci, [vp, vp, i64, dbl, i32, ci]),
        "gwc_export_cosmo": (ci, [vp, vp, vp, vp]),
        "gwc_pack_events": (ci, [vp, i64, i64, vp, vp, vp, vp, vp, vp, vp, C.POINTER(i64)]),
        "gwc_cap_pixels": (ci, [vp, i64, i64, i64, vp, vp, vp, i64, C.c_uint64, vp, C.POINTER(i64)]),
        "gwc_los_allsky": (ci, [vp, C.POINTER(Los), vp]),
        "gwc_event_loglik": (ci, [vp, vp, i64, C.POINTER(Events), C.POINTER(Los), vp, vp, vp]),
        "gwc_event_loglik_pixcut": (ci, [vp, vp, i64, C.POINTER(Events), C.POINTER(Los), dbl, vp, vp, vp, vp]),
        "gwc_event_loglik_kde": (ci, [vp, vp, i64, C.POINTER(Events), C.POINTER(Los), i32, dbl, i32, vp, vp, vp]),
        "gwc_selection_logxi": (ci, [vp, vp, i64, C.POINTER(Injections), C.POINTER(Los), vp, vp]),
        "gwc_combine_total": (ci, [vp, vp, vp, i64, i64, vp]),
        "gwc_total_loglik": (ci, [vp, vp, i64, C.POINTER(Events), C.POINTER(Injections), C.POINTER(Los), i32, ci, vp]),
        "gwc_total_loglik_pixcut": (ci, [vp, vp, i64, C.POINTER(Events), C.POINTER(Injections), C.POINTER(Los), i32, ci, dbl, vp]),
        "gwc_total_loglik_kde": (ci, [vp, vp, i64, C.POINTER(Events), C.POINTER(Injections), C.POINTER(Los), i32, ci, i32,
                                      dbl, i32, vp]),
        "gwc_total_loglik_host": (ci, [vp, vp, i64, C.POINTER(Events), C.POINTER(Injections), C.POINTER(Los), i32, ci,
                                       vp, C.POINTER(i64), C.POINTER(i64)]),
        "gwc_cache_catalogue": (ci, [vp, ci]),
        "gwc_set_timing": (ci, [vp, ci]),
        "gwc_get_timing": (ci, [vp, C.POINTER(i64), C.POINTER(dbl), C.POINTER(i64), C.POINTER(dbl)]),
        "gwc_probe_fp64": (ci, [vp, i64, C.POINTER(dbl), C.POINTER(dbl)]),
        "gwc_math_selftest": (ci, [vp, ci, i64, vp, vp]),
        "gwc_combine_sharded": (ci, [vp, i32, i64, i64, vp, vp, vp, vp, vp, vp]),
        "gwc_combine_sharded_host": (ci, [i32, i64, i64, vp, vp, vp, vp, vp, vp]),
        "gwc_los_allsky_static": (ci, [C.POINTER(Los), vp, vp]),
        "gwc_los_allsky_static_error": (C.c_char_p, []),
    }
    for name, (res, args) in sig.items():
        f = getattr(L, name)
        f.restype, f.argtypes = res, args
    _lib = L
    return L


def _ptr(t: Optional[torch.Tensor], dtype=None, cuda: bool = True):
    if t is None:
        return None
    if dtype is not None and t.dtype != dtype:
        raise TypeError("expected %s, got %s" % (dtype, t.dtype))
    if not t.is_contiguous():
        raise ValueError("tensor must be contiguous")
    if cuda and not t.is_cuda:
        raise ValueError("expected a CUDA tensor")
    if not cuda and t.is_cuda:
        raise ValueError("expected a host tensor")
    return t.data_ptr()


def _prec(t: torch.Tensor) -> int:
    if t.dtype == torch.float64:
        return F64
    if t.dtype == torch.float32:
        return F32
    raise TypeError("table must be float64 or float32")


def make_events(ev: Dict[str, Optional[torch.Tensor]], cuda: bool = True) -> Events:
    off = ev["ev_sample_off"]
    return Events(off.numel() - 1, ev["dL"].numel(), _ptr(off, torch.int64, cuda), _ptr(ev["dL"], torch.float64, cuda),
                  _ptr(ev["m1z"], torch.float64, cuda), _ptr(ev["m2z"], torch.float64, cuda),
                  _ptr(ev.get("log_pe_prior"), torch.float64, cuda), _ptr(ev["sample_row"], torch.int32, cuda),
                  _ptr(ev.get("ev_pix_off"), torch.int64, cuda), _ptr(ev.get("ev_pix_rows"), torch.int32, cuda))


def make_los(table: torch.Tensor, z_max: float, allsky: Optional[torch.Tensor] = None, cuda: bool = True) -> Los:
    if table.dim() != 2:
        raise ValueError("LOS table must be [n_rows, n_z]")
    return Los(table.shape[0], table.shape[1], float(z_max), _prec(table), _ptr(table, None, cuda),
               _ptr(allsky, torch.float64, cuda))


def make_injections(inj: Dict[str, object], cuda: bool = True) -> Injections:
    return Injections(inj["dL"].numel(), float(inj["n_draw"]), _ptr(inj["dL"], torch.float64, cuda),
                      _ptr(inj["m1z"], torch.float64, cuda), _ptr(inj["m2z"], torch.float64, cuda),
                      _ptr(inj["log_pdraw"], torch.float64, cuda))


class Context:
    """Owns a gwc_ctx bound to a CUDA device and a torch stream (None = torch's current stream at creation)."""

    def __init__(self, device: int = 0, stream: Optional[torch.cuda.Stream] = None):
        self._lib = load()
        if not torch.cuda.is_available():
            raise RuntimeError("gwc needs a CUDA device; there is no CPU fallback")
        self.device = torch.device("cuda", device)
        with torch.cuda.device(self.device):
            self.stream = stream if stream is not None else torch.cuda.current_stream()
        h = C.c_void_p()
        st = self._lib.gwc_create(C.byref(h), device, C.c_void_p(self.stream.cuda_stream))
        if st != OK:
            raise GwcError(st, self._lib.gwc_last_error(None).decode() or "gwc_create failed")
        self._h = h
        self._npar = NPAR   # row width of theta under the selected mass model (gwc_set_mass_model)

    def _theta(self, theta: torch.Tensor):
        """Device pointer of a theta batch after checking its row width against the selected mass model (the C entry
        points take no width: a [n, 12] array under MULTIPEAK would be read past its end)."""
        if theta.dim() != 2 or theta.shape[1] != self._npar:
            raise ValueError("theta must be [n_theta, %d] under the selected mass model, got %s"
                             % (self._npar, tuple(theta.shape)))
        return _ptr(theta, torch.float64)

    def close(self):
        if getattr(self, "_h", None):
            self._lib.gwc_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _ck(self, st: int):
        if st != OK:
            raise GwcError(st, self._lib.gwc_last_error(self._h).decode())

    # ---- one method per C entry point -------------------------------------------------------
    def gwc_check(self):
        self._ck(self._lib.gwc_check(self._h))

    def gwc_launch_count(self) -> int:
        return int(self._lib.gwc_launch_count(self._h))

    def gwc_set_mass_model(self, model: str):
        """"plpeak" (12-column theta rows) or "multipeak" (16 columns; include/gwc.h)."""
        self._ck(self._lib.gwc_set_mass_model(self._h, MASS_MODELS[model]))
        self._npar = int(self._lib.gwc_theta_len(MASS_MODELS[model]))

    def gwc_set_omega_hint(self, hint: str):
        """"detect" (default: gwc_build_cosmo asks the device and synchronises for batches of 40+ points), "varies"
        (never share a z(u) table, never synchronise) or "single" (the caller promises one Omega_m per batch and no
        invalid point; checked on the device, a broken promise -> GWC_ERR_INVALID_ARG from gwc_check)."""
        self._ck(self._lib.gwc_set_omega_hint(self._h, OMEGA_HINTS[hint]))

    def gwc_theta_len(self, model: str) -> int:
        return int(self._lib.gwc_theta_len(MASS_MODELS[model]))

    def gwc_build_cosmo(self, theta: torch.Tensor, z_max: float, n_nodes: int = 1025, table_prec: int = F64):
        self._ck(self._lib.gwc_build_cosmo(self._h, self._theta(theta), theta.shape[0], float(z_max), n_nodes,
                                           table_prec))

    def gwc_export_cosmo(self, n_theta: int, n_nodes: int):
        z = torch.empty((n_theta, n_nodes), dtype=torch.float64, device=self.device)
        dz = torch.empty_like(z)
        umax = torch.empty(n_theta, dtype=torch.float64, device=self.device)
        self._ck(self._lib.gwc_export_cosmo(self._h, z.data_ptr(), dz.data_ptr(), umax.data_ptr()))
        return z, dz, umax

    def gwc_pack_events(self, event_id: torch.Tensor, row: torch.Tensor, n_events: int):
        n = event_id.numel()
        dev = self.device
        perm = torch.empty(max(n, 1), dtype=torch.int64, device=dev)
        eso = torch.empty(n_events + 1, dtype=torch.int64, device=dev)
        epo = torch.empty(n_events + 1, dtype=torch.int64, device=dev)
        epr = torch.empty(max(n, 1), dtype=torch.int32, device=dev)
        pso = torch.empty(n + 1, dtype=torch.int64, device=dev)
        npx = C.c_int64(0)
        self._ck(self._lib.gwc_pack_events(self._h, n, n_events, _ptr(event_id, torch.int32), _ptr(row, torch.int32),
                                           perm.data_ptr(), eso.data_ptr(), epo.data_ptr(), epr.data_ptr(),
                                           pso.data_ptr(), C.byref(npx)))
        k = int(npx.value)
        return dict(perm=perm[:n], ev_sample_off=eso, ev_pix_off=epo, ev_pix_rows=epr[:k], pix_sample_off=pso[:k + 1],
                    n_pixrefs=k)

    def gwc_cap_pixels(self, packed: dict, cap: int, seed: int):
        """Per-pixel sample cap on the output of gwc_pack_events: returns perm_kept,
        ev_sample_off', pix_sample_off' (new tensors; `packed` is left untouched)."""
        perm = packed["perm"].contiguous()
        eso, pso = packed["ev_sample_off"].clone(), packed["pix_sample_off"].clone()
        n = perm.numel()
        out = torch.empty(max(n, 1), dtype=torch.int64, device=self.device)
        nk = C.c_int64(0)
        self._ck(self._lib.gwc_cap_pixels(self._h, n, eso.numel() - 1, pso.numel() - 1, perm.data_ptr(), eso.data_ptr(),
                                          pso.data_ptr(), int(cap), int(seed) & 0xFFFFFFFFFFFFFFFF, out.data_ptr(),
                                          C.byref(nk)))
        return out[:int(nk.value)], eso, pso

    def gwc_los_allsky(self, table: torch.Tensor, z_max: float) -> torch.Tensor:
        out = torch.empty(table.shape[1], dtype=torch.float64, device=self.device)
        los = make_los(table, z_max)
        self._ck(self._lib.gwc_los_allsky(self._h, C.byref(los), out.data_ptr()))
        return out

    @staticmethod
    def gwc_los_allsky_static(table: torch.Tensor, z_max: float, out: torch.Tensor) -> torch.Tensor:
        """gwc_los_allsky without any device allocation, for programs whose memory pool owns the whole GPU or whose
        other streams must not be stalled by cudaMalloc (include/gwc.h).  Needs no Context: the caller brings `out`
        ([n_z] float64 on the table's device) and the partial sums go to a fixed 4 MiB array inside libgwc.so, which
        limits the table to ceil(n_rows / 512) * n_z <= 2**19 (GwcError GWC_ERR_SHAPE beyond).  Runs on torch's
        current stream of the table's device; the first call on a device does a one-time set-up, so make it at
        start-up.  Calls that overlap on one GPU race on the shared array."""
        lib = load()
        if out.dim() != 1 or out.shape[0] != table.shape[1] or out.device != table.device:
            raise ValueError("out must be [n_z] on the table's device")
        los = make_los(table, z_max)
        with torch.cuda.device(table.device):
            st = lib.gwc_los_allsky_static(C.byref(los), _ptr(out, torch.float64),
                                           C.c_void_p(torch.cuda.current_stream().cuda_stream))
        if st != OK:
            raise GwcError(st, lib.gwc_los_allsky_static_error().decode())
        return out

    @staticmethod
    def gwc_los_allsky_static_error() -> str:
        return load().gwc_los_allsky_static_error().decode()

    def gwc_event_loglik(self, theta, ev, table, z_max, want_neff=True, want_nlive=True):
        nt, ne = theta.shape[0], ev["ev_sample_off"].numel() - 1
        logL = torch.empty((nt, ne), dtype=torch.float64, device=self.device)
        neff = torch.empty_like(logL) if want_neff else None
        nlive = torch.empty((nt, ne), dtype=torch.int64, device=self.device) if want_nlive else None
        es, los = make_events(ev), make_los(table, z_max)
        self._ck(self._lib.gwc_event_loglik(self._h, self._theta(theta), nt, C.byref(es), C.byref(los),
                                            logL.data_ptr(), _ptr(neff), _ptr(nlive)))
        return logL, neff, nlive

    def gwc_event_loglik_pixcut(self, theta, ev, table, z_max, neff_min):
        """Event term with the per-pixel N_eff cut of Eq. 8: returns logL, neff, nlive, npass."""
        nt, ne = theta.shape[0], ev["ev_sample_off"].numel() - 1
        logL = torch.empty((nt, ne), dtype=torch.float64, device=self.device)
        neff = torch.empty_like(logL)
        nlive = torch.empty((nt, ne), dtype=torch.int64, device=self.device)
        npass = torch.empty((nt, ne), dtype=torch.int64, device=self.device)
        es, los = make_events(ev), make_los(table, z_max)
        self._ck(self._lib.gwc_event_loglik_pixcut(self._h, self._theta(theta), nt, C.byref(es), C.byref(los),
                                                   float(neff_min), logL.data_ptr(), neff.data_ptr(),
                                                   nlive.data_ptr(), npass.data_ptr()))
        return logL, neff, nlive, npass

    def gwc_event_loglik_kde(self, theta, ev, table, z_max, n_grid=256, neff_min=0.0, bandwidth="scott"):
        """Event term with the paper's KDE numerator (Eq. 5-7, D1): returns logL, npass, nused."""
        nt, ne = theta.shape[0], ev["ev_sample_off"].numel() - 1
        logL = torch.empty((nt, ne), dtype=torch.float64, device=self.device)
        npass = torch.empty((nt, ne), dtype=torch.int64, device=self.device)
        nused = torch.empty((nt, ne), dtype=torch.int64, device=self.device)
        es, los = make_events(ev), make_los(table, z_max)
        self._ck(self._lib.gwc_event_loglik_kde(self._h, self._theta(theta), nt, C.byref(es), C.byref(los),
                                                int(n_grid), float(neff_min), BW_RULES[bandwidth], logL.data_ptr(),
                                                npass.data_ptr(), nused.data_ptr()))
        return logL, npass, nused

    def gwc_selection_logxi(self, theta, inj, allsky, n_z, z_max, want_neff=True):
        nt = theta.shape[0]
        logxi = torch.empty(nt, dtype=torch.float64, device=self.device)
        neff = torch.empty_like(logxi) if want_neff else None
        js = make_injections(inj)
        los = Los(1, n_z, float(z_max), F64, None, _ptr(allsky, torch.float64))
        self._ck(self._lib.gwc_selection_logxi(self._h, self._theta(theta), nt, C.byref(js), C.byref(los),
                                               logxi.data_ptr(), _ptr(neff)))
        return logxi, neff

    def gwc_combine_total(self, logL, logxi):
        nt, ne = logL.shape
        out = torch.empty(nt, dtype=torch.float64, device=self.device)
        self._ck(self._lib.gwc_combine_total(self._h, _ptr(logL, torch.float64), _ptr(logxi, torch.float64), nt, ne,
                                             out.data_ptr()))
        return out

    def gwc_combine_sharded(self, sum_logL_parts, logxi_parts, neff_inj_parts, n_events_total: int):
        """Pieces [n_parts, n_theta] of an event / injection-sharded evaluation (device tensors, rank order) ->
        (total, logxi, neff_inj), each [n_theta]."""
        R, nt = sum_logL_parts.shape
        if tuple(logxi_parts.shape) != (R, nt) or tuple(neff_inj_parts.shape) != (R, nt):
            raise ValueError("the three piece arrays must have the same [n_parts, n_theta] shape")
        out = [torch.empty(nt, dtype=torch.float64, device=self.device) for _ in range(3)]
        self._ck(self._lib.gwc_combine_sharded(self._h, R, nt, int(n_events_total), _ptr(sum_logL_parts, torch.float64),
                                               _ptr(logxi_parts, torch.float64), _ptr(neff_inj_parts, torch.float64),
                                               out[0].data_ptr(), out[1].data_ptr(), out[2].data_ptr()))
        return tuple(out)

    @staticmethod
    def gwc_combine_sharded_host(sum_logL_parts, logxi_parts, neff_inj_parts, n_events_total: int):
        """gwc_combine_sharded on HOST tensors; needs no context and no GPU."""
        R, nt = sum_logL_parts.shape
        if tuple(logxi_parts.shape) != (R, nt) or tuple(neff_inj_parts.shape) != (R, nt):
            raise ValueError("the three piece arrays must have the same [n_parts, n_theta] shape")
        out = [torch.empty(nt, dtype=torch.float64) for _ in range(3)]
        st = load().gwc_combine_sharded_host(R, nt, int(n_events_total), _ptr(sum_logL_parts, torch.float64, False),
                                             _ptr(logxi_parts, torch.float64, False),
                                             _ptr(neff_inj_parts, torch.float64, False), out[0].data_ptr(),
                                             out[1].data_ptr(), out[2].data_ptr())
        if st != OK:
            raise GwcError(st, "gwc_combine_sharded_host: bad arguments")
        return tuple(out)

    def gwc_total_loglik(self, theta, ev, inj, table, z_max, allsky, n_nodes=1025, table_prec=F64, out=None):
        nt = theta.shape[0]
        if out is None:
            out = torch.empty(nt, dtype=torch.float64, device=self.device)
        es, js, los = make_events(ev), make_injections(inj), make_los(table, z_max, allsky)
        self._ck(self._lib.gwc_total_loglik(self._h, self._theta(theta), nt, C.byref(es), C.byref(js),
                                            C.byref(los), n_nodes, table_prec, out.data_ptr()))
        return out

    def gwc_total_loglik_pixcut(self, theta, ev, inj, table, z_max, allsky, neff_min=2.0, n_nodes=1025, table_prec=F64):
        """gwc_total_loglik with the per-pixel N_eff cut of Eq. 8 on the event term."""
        nt = theta.shape[0]
        out = torch.empty(nt, dtype=torch.float64, device=self.device)
        es, js, los = make_events(ev), make_injections(inj), make_los(table, z_max, allsky)
        self._ck(self._lib.gwc_total_loglik_pixcut(self._h, self._theta(theta), nt, C.byref(es), C.byref(js),
                                                   C.byref(los), n_nodes, table_prec, float(neff_min), out.data_ptr()))
        return out

    def gwc_total_loglik_kde(self, theta, ev, inj, table, z_max, allsky, n_grid=256, neff_min=2.0, n_nodes=1025,
                             table_prec=F64, bandwidth="scott"):
        """The paper's likelihood in one call: KDE numerator + per-pixel N_eff cut + selection term."""
        nt = theta.shape[0]
        out = torch.empty(nt, dtype=torch.float64, device=self.device)
        es, js, los = make_events(ev), make_injections(inj), make_los(table, z_max, allsky)
        self._ck(self._lib.gwc_total_loglik_kde(self._h, self._theta(theta), nt, C.byref(es), C.byref(js),
                                                C.byref(los), n_nodes, table_prec, int(n_grid), float(neff_min),
                                                BW_RULES[bandwidth], out.data_ptr()))
        return out

    def gwc_total_loglik_host(self, theta, ev, inj, table, z_max, allsky=None, n_nodes=1025, table_prec=F64, out=None):
        """All tensors on the HOST (pinned memory makes the copies faster).  Returns (out, h2d_bytes, d2h_bytes)."""
        nt = theta.shape[0]
        if theta.dim() != 2 or theta.shape[1] != self._npar:
            raise ValueError("theta must be [n_theta, %d] under the selected mass model" % self._npar)
        if out is None:
            out = torch.empty(nt, dtype=torch.float64)
        es, js = make_events(ev, cuda=False), make_injections(inj, cuda=False)
        los = make_los(table, z_max, allsky, cuda=False)
        up, down = C.c_int64(0), C.c_int64(0)
        self._ck(self._lib.gwc_total_loglik_host(self._h, _ptr(theta, torch.float64, False), nt, C.byref(es),
                                                 C.byref(js), C.byref(los), n_nodes, table_prec,
                                                 _ptr(out, torch.float64, False), C.byref(up), C.byref(down)))
        return out, int(up.value), int(down.value)

    def gwc_cache_catalogue(self, on: bool):
        """Keep the theta-independent preparation between calls (the caller promises unchanged arrays)."""
        self._ck(self._lib.gwc_cache_catalogue(self._h, int(on)))

    def gwc_set_timing(self, on: bool):
        self._ck(self._lib.gwc_set_timing(self._h, int(on)))

    def gwc_get_timing(self):
        a, b = C.c_int64(0), C.c_int64(0)
        x, y = C.c_double(0), C.c_double(0)
        self._ck(self._lib.gwc_get_timing(self._h, C.byref(a), C.byref(x), C.byref(b), C.byref(y)))
        return dict(n_ev=int(a.value), ms_ev=x.value, n_inj=int(b.value), ms_inj=y.value)

    def gwc_probe_fp64(self, iters: int = 1 << 14):
        ms, n = C.c_double(0), C.c_double(0)
        self._ck(self._lib.gwc_probe_fp64(self._h, iters, C.byref(ms), C.byref(n)))
        return ms.value, n.value

    def gwc_math_selftest(self, which: int, x: torch.Tensor) -> torch.Tensor:
        out = torch.empty_like(x)
        self._ck(self._lib.gwc_math_selftest(self._h, which, x.numel(), _ptr(x, torch.float64), out.data_ptr()))
        return out
