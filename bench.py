#!/usr/bin/env python
"""bench.py -- throughput of the whole hot path (A1..A6, gwc_total_loglik) on synthetic catalogues.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload o5|production|o4|stress|tiny]
                    [--impl gwc|reference] [--theta-scale F]

A step = one pass of the whole hot path over one theta batch of the workload: cosmology tables, event
re-weighting, selection term, total.  `value` = (theta x sample) terms per second with inputs resident in
HBM (events + injections); `e2e` = the same through gwc_total_loglik_host with HOST buffers (uploads and
the download inside the timed region).  N > 1: one process per GPU (torchrun), the theta batch is sharded
by giving every rank its own full-size batch (weak scaling, replicated catalogue, no data-path collective).
`--impl reference` times the CPU oracle on a bounded sample of the same workload (rank 0 only).
Prints ONE JSON line.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np
import torch

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2605_23538_b200 import synth  # noqa: E402

METRIC = "(theta*event*sample) terms/s, whole hot path (events + injections)"
UNIT = "terms/s"
# FP64-pipe instructions per term of THIS formulation.  NECESSARY (what a live / a dead term needs: DESIGN.md section 7,
# counted from the SASS of the main loop) is what `roofline.frac` uses; EXECUTED is what the shipped event kernel runs
# per term, live or dead, MEASURED by ncu (sass__thread_inst_executed_true_per_opcode: DFMA + DADD + DMUL + DSETP over
# the terms of one 340-theta launch of the O5 catalogue; profiles/r02e_reweight_events_ncu_full.md).  Re-measure
# after any edit of the kernel: the profile names the command.
FP64_INSTR_LIVE = 104.0
FP64_INSTR_DEAD = 28.0
FP64_INSTR_EXECUTED = 108.26
FP64_COUNT_SOURCE = "necessary: static SASS count of the main loop (DESIGN.md 7); executed: ncu op counters, profiles/r02e_reweight_events_ncu_full.md"
# The counts above belong to ONE build of the fused kernel: profiles/fp64_counts.json records the SHA-256 of that
# build's SASS (the reweight_kernel functions of libgwc.so, `cuobjdump -sass`).  The bench line carries
# "count_stale": true when the library it ran hashes differently (the kernel was edited and the counts were not
# re-measured), null when cuobjdump is not there to tell.
FP64_COUNTS_FILE = os.path.join(os.path.dirname(os.path.abspath(__file__)), "profiles", "fp64_counts.json")


def reweight_sass_sha256(lib_path):
    """SHA-256 over the SASS instruction text of every reweight_kernel instantiation in `lib_path`, or None."""
    import hashlib
    import re
    import subprocess
    try:
        out = subprocess.run(["cuobjdump", "-sass", lib_path], capture_output=True, text=True, timeout=300).stdout
    except Exception:
        return None
    h, keep, n = hashlib.sha256(), False, 0
    for line in out.splitlines():
        if "Function :" in line:
            keep = "reweight_kernel" in line
            if keep:
                h.update(line.split("Function :")[1].strip().encode())
                n += 1
            continue
        if keep:
            m = re.match(r"\s*/\*[0-9a-f]{4,}\*/\s+(.*?);", line)      # address, instruction text (no encoding words)
            if m:
                h.update(m.group(1).encode())
    return h.hexdigest() if n else None


def _load_counts():
    """The tracked counts replace the constants above when the file is there (same numbers today: the file is what a
    re-measurement updates, together with the hash of the build it was made on)."""
    global FP64_INSTR_LIVE, FP64_INSTR_DEAD, FP64_INSTR_EXECUTED, FP64_COUNT_SOURCE
    import json as _json
    try:
        rec = _json.load(open(FP64_COUNTS_FILE))
        FP64_INSTR_LIVE = float(rec["fp64_instr_per_live_term_necessary"])
        FP64_INSTR_DEAD = float(rec["fp64_instr_per_dead_term_necessary"])
        FP64_INSTR_EXECUTED = float(rec["fp64_instr_executed_per_term"]["events_o5"])
        FP64_COUNT_SOURCE = rec.get("source", FP64_COUNT_SOURCE)
        return rec
    except Exception:
        return None


FP64_COUNTS = _load_counts()


def fp64_count_state(lib_path):
    import json as _json
    try:
        rec = _json.load(open(FP64_COUNTS_FILE))
    except Exception:
        return {"count_stale": None, "counts_file": None}
    sha = reweight_sass_sha256(lib_path)
    return {"count_stale": None if sha is None else sha != rec.get("reweight_sass_sha256"),
            "counts_file": "profiles/fp64_counts.json", "reweight_sass_sha256": sha}
# the KDE kernel: FP64 thread instructions per Gaussian evaluation, everything included (per-sample weights, per-pixel
# statistics, prior), measured the same way (profiles/r02f_kde_ncu_full.md)
KDE_FP64_INSTR_PER_EVAL = 4.81
# DRAM bytes of one 340-theta launch of the event kernel on the O5 catalogue (ncu dram__bytes_read.sum +
# dram__bytes_write.sum, same capture)
O5_DRAM_BYTES_PER_340_THETA = 7.247e9 + 0.068e9
# B200 FP64 issue peak derived from the unit counts: 148 SMs x 64 FP64 lanes x 1.965 GHz
FP64_PEAK_INSTR = 148 * 64 * 1.965e9


def _env_int(name, default):
    try:
        return int(os.environ.get(name, default))
    except ValueError:
        return default


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""

    FIELDS = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
              "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
              "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.gpu = gpu_index
        self.proc = None
        self.path = None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(prefix="gwc_clocks_", suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.gpu), "--query-gpu=" + self.FIELDS,
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        try:
            self.proc.terminate()
            self.proc.wait(timeout=5)
        except Exception:
            pass
        try:
            rows = [r.strip().split(", ") for r in open(self.path) if r.strip()]
            os.unlink(self.path)
        except Exception:
            return out
        sm, reasons, mx, pw = [], set(), None, []
        for r in rows:
            if len(r) < 9:
                continue
            try:
                sm.append(float(r[1]))
                mx = float(r[2])
                pw.append(float(r[3]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[5:9]):
                if v.strip().lower() == "active":
                    reasons.add(name)
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=mx, reasons=sorted(reasons), samples=len(sm),
                       power_w_max=max(pw) if pw else None)
        return out


def _bench_spec(name: str, theta_scale: float):
    spec = synth.CONFIGS[name]
    if theta_scale != 1.0:
        spec = synth.scaled(spec, n_theta=max(1, int(round(spec.n_theta * theta_scale))))
    return spec


def _hbm_peak():
    """Measured HBM copy bandwidth of this pool's B200s (driver-written MEASURED_PEAKS.json), else the profiling
    guide's fallback."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "MEASURED_PEAKS.json (hbm_gbs)"
    except Exception:
        return 6650.0, "of fallback (B200_PROFILING.md: 6.65 TB/s)"


def _pin(t):
    return t.pin_memory() if isinstance(t, torch.Tensor) else t


# ---------------------------------------------------------------------------------------------
def run_leg(args):
    """One leg alone (profiling runs: the command an ncu capture under profiles/ names): `events` = gwc_event_loglik,
    `pixcut` = gwc_event_loglik_pixcut at --pixcut, `kde` = gwc_event_loglik_kde on --kde-theta points, `inj` =
    gwc_selection_logxi.  W warm-up calls, K timed ones (kernel time by CUDA events on the library's stream)."""
    from paper_2605_23538_b200 import gwc
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the gwc path has no CPU fallback")
    dev = torch.device("cuda", 0)
    spec = _bench_spec(args.workload, args.theta_scale)
    W = synth.make_workload(spec, seed=args.seed, device=dev, keep_f64_los=False)
    mp = args.mass_model == "multipeak"
    theta = (synth.make_theta_multipeak if mp else synth.make_theta)(spec, args.seed, dev)
    ctx = gwc.Context(0)
    if mp:
        ctx.gwc_set_mass_model("multipeak")
    zmax = spec.z_max
    prec = gwc.F32 if args.table_prec == "f32" else gwc.F64
    if args.leg == "kde":
        theta = theta[:min(max(args.kde_theta, 1), theta.shape[0])].contiguous()
    allsky = ctx.gwc_los_allsky(W.los, zmax)
    ctx.gwc_build_cosmo(theta, zmax, args.n_nodes, prec)
    n_theta, n_samples = int(theta.shape[0]), W.n_samples
    units, extra = float(n_theta) * n_samples, {}

    def call():
        if args.leg == "events":
            return ctx.gwc_event_loglik(theta, W.ev, W.los, zmax, want_neff=False, want_nlive=True)[2]
        if args.leg == "pixcut":
            return ctx.gwc_event_loglik_pixcut(theta, W.ev, W.los, zmax, max(args.pixcut, 0.0))[3]
        if args.leg == "kde":
            return ctx.gwc_event_loglik_kde(theta, W.ev, W.los, zmax, 256, 2.0, args.kde_bandwidth)[2]
        return ctx.gwc_selection_logxi(theta, W.inj, allsky, W.los.shape[1], zmax)[0]

    for _ in range(max(args.warmup, 1)):
        r = call()
    torch.cuda.synchronize()
    ctx.gwc_set_timing(True)
    ctx.gwc_get_timing()
    for _ in range(args.steps):
        r = call()
    torch.cuda.synchronize()
    tm = ctx.gwc_get_timing()
    ctx.gwc_set_timing(False)
    ctx.gwc_check()
    key = "inj" if args.leg == "inj" else "ev"
    ms = tm["ms_" + key] / max(tm["n_" + key], 1)
    if args.leg == "inj":
        units = float(n_theta) * int(W.inj["dL"].numel())
    elif args.leg == "kde":
        extra["gaussian_evals_per_s"] = float(r.sum().item()) * 256.0 / (ms * 1e-3)
    elif args.leg == "events":
        extra["live_fraction"] = float(r.sum().item()) / units
    else:
        extra["mean_passing_pixels_per_event"] = float(r.double().mean())
    print(json.dumps(dict({"leg": args.leg, "workload": spec.name, "mass_model": args.mass_model, "n_theta": n_theta,
                           "kernel_ms": ms,
                           "terms_per_s": units / (ms * 1e-3)}, **extra)))
    ctx.close()


# ---------------------------------------------------------------------------------------------
def run_gwc(args):
    from paper_2605_23538_b200 import gwc
    rank, world, local = _env_int("RANK", 0), _env_int("WORLD_SIZE", 1), _env_int("LOCAL_RANK", 0)
    dist = world > 1
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the gwc path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if dist:
        import torch.distributed as td
        td.init_process_group("nccl", device_id=dev)
    spec = _bench_spec(args.workload, args.theta_scale)
    t_gen = time.time()
    W = synth.make_workload(spec, seed=args.seed, device=dev, keep_f64_los=False)
    # every rank owns a full-size theta batch of its own (weak scaling over theta)
    mp = args.mass_model == "multipeak"
    theta = (synth.make_theta_multipeak if mp else synth.make_theta)(spec, args.seed + 7919 * rank, dev)
    torch.cuda.synchronize()
    t_gen = time.time() - t_gen
    ctx = gwc.Context(local)
    if mp:
        # MULTIPEAK with delta_m smoothing (NEXT row 3a): 16-column theta rows; mmin = 4.6 keeps the catalogue's masses
        # (drawn from a population that starts at 5 Msun) inside the support
        ctx.gwc_set_mass_model("multipeak")
    zmax = spec.z_max
    prec = gwc.F32 if args.table_prec == "f32" else gwc.F64
    allsky = ctx.gwc_los_allsky(W.los, zmax)
    out = torch.empty(theta.shape[0], dtype=torch.float64, device=dev)
    n_samples, n_inj, n_theta = W.n_samples, int(W.inj["dL"].numel()), int(theta.shape[0])
    terms_ev, terms_inj = float(n_theta) * n_samples, float(n_theta) * n_inj
    terms = terms_ev + terms_inj

    def step():
        ctx.gwc_total_loglik(theta, W.ev, W.inj, W.los, zmax, allsky, args.n_nodes, prec, out=out)

    def barrier():
        torch.cuda.synchronize()
        if dist:
            td.barrier()
            torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    barrier()
    # live fraction (untimed): needed for the algorithmic instruction count
    ctx.gwc_build_cosmo(theta, zmax, args.n_nodes, prec)
    _, _, nlive = ctx.gwc_event_loglik(theta, W.ev, W.los, zmax, want_neff=False, want_nlive=True)
    live_frac_ev = float(nlive.sum().item()) / max(terms_ev, 1.0)
    del nlive
    barrier()
    ctx.gwc_set_timing(True)
    ctx.gwc_get_timing()
    launches0 = ctx.gwc_launch_count()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop() if rank == 0 else {}
    launches = ctx.gwc_launch_count() - launches0
    tm = ctx.gwc_get_timing()
    ctx.gwc_set_timing(False)
    ctx.gwc_check()
    if dist:
        t = torch.tensor([ms], dtype=torch.float64, device=dev)
        td.all_reduce(t, op=td.ReduceOp.MAX)
        ms = float(t.item())
    value = terms * world * args.steps / (ms * 1e-3)

    # ---- end to end through the host API (pinned host buffers, copies inside the timed region) ----
    h_theta = _pin(theta.cpu())
    h_ev = {k: _pin(v.cpu()) if isinstance(v, torch.Tensor) else v for k, v in W.ev.items()}
    h_inj = {k: _pin(v.cpu()) if isinstance(v, torch.Tensor) else v for k, v in W.inj.items()}
    h_los = _pin(W.los.cpu())
    h_out = _pin(torch.empty(n_theta, dtype=torch.float64))
    # (default: as many as the device-resident figure on the small configs, 2 on o5 where a step takes 1.2 s)
    e2e_cap = args.e2e_steps if args.e2e_steps > 0 else (2 if spec.name == "o5" else args.steps)
    e2e_steps = max(1, min(args.steps, e2e_cap))
    up = down = 0
    _, up, down = ctx.gwc_total_loglik_host(h_theta, h_ev, h_inj, h_los, zmax, None, args.n_nodes, prec, out=h_out)
    barrier()
    t0 = time.perf_counter()
    e0.record()
    for _ in range(e2e_steps):
        ctx.gwc_total_loglik_host(h_theta, h_ev, h_inj, h_los, zmax, None, args.n_nodes, prec, out=h_out)
    e1.record()
    barrier()
    ms_e2e = max(e0.elapsed_time(e1), (time.perf_counter() - t0) * 1e3 if not dist else 0.0)
    if dist:
        t = torch.tensor([ms_e2e], dtype=torch.float64, device=dev)
        td.all_reduce(t, op=td.ReduceOp.MAX)
        ms_e2e = float(t.item())
    e2e_value = terms * world * e2e_steps / (ms_e2e * 1e-3)
    same = bool(torch.equal(h_out, out.cpu()) or torch.allclose(h_out, out.cpu(), rtol=0, atol=0, equal_nan=True))

    if rank != 0:
        if dist:
            td.destroy_process_group()
        return
    # ---- roofline of the dominant kernel (event re-weighting), timed live with CUDA events on its stream ----
    ms_ev_kernel = tm["ms_ev"] / max(tm["n_ev"], 1)
    ms_inj_kernel = tm["ms_inj"] / max(tm["n_inj"], 1)
    # (MULTIPEAK: + 42 FP64 instructions per live term, static count of the added code, R36)
    instr_live = FP64_INSTR_LIVE + (42.0 if mp else 0.0)
    # executed FP64 instructions per term, ncu-measured on the workload they are quoted for (profiles/fp64_counts.json)
    ex = (FP64_COUNTS or {}).get("fp64_instr_executed_per_term", {})
    if mp:
        executed = ex.get("events_production_multipeak") if spec.name == "production" else None
    else:
        executed = FP64_INSTR_EXECUTED
    instr = terms_ev * (live_frac_ev * instr_live + (1.0 - live_frac_ev) * FP64_INSTR_DEAD)
    achieved = instr * 2.0 / (ms_ev_kernel * 1e-3) / 1e12          # FP64 issue slots x 2 flop
    peak_derived = FP64_PEAK_INSTR * 2.0 / 1e12
    # the denominator: the dependent-free DFMA probe of this very run (BASELINE.md section 3 asks for a measured FP64
    # figure; MEASURED_PEAKS.json has none), the best of three; the derived unit-count figure is reported beside it
    probe = [ctx.gwc_probe_fp64(1 << 13) for _ in range(3)]
    peak = max(n * 2.0 / (t * 1e-3) / 1e12 for t, n in probe)
    peak_instr = peak * 1e12 / 2.0
    # the injection instantiation (the step's second kernel): same formulation, same counts, its own live fraction
    # (counted by running the injections through the event entry point as 8192-sample pseudo-events on the all-sky row)
    ctx.gwc_build_cosmo(theta, zmax, args.n_nodes, prec)
    pseudo_off = torch.arange(0, n_inj + 8192, 8192, dtype=torch.int64, device=dev).clamp_(max=n_inj)
    pseudo = {"ev_sample_off": pseudo_off, "dL": W.inj["dL"], "m1z": W.inj["m1z"], "m2z": W.inj["m2z"],
              "log_pe_prior": W.inj["log_pdraw"], "sample_row": torch.zeros(n_inj, dtype=torch.int32, device=dev)}
    _, _, nlive_inj = ctx.gwc_event_loglik(theta, pseudo, allsky.view(1, -1).contiguous(), zmax, want_neff=False)
    live_frac_inj = float(nlive_inj.sum().item()) / max(terms_inj, 1.0)
    del nlive_inj
    instr_inj = terms_inj * (live_frac_inj * instr_live + (1.0 - live_frac_inj) * FP64_INSTR_DEAD)
    achieved_inj = instr_inj * 2.0 / (ms_inj_kernel * 1e-3) / 1e12
    roofline_inj = {"bound": "alu", "kernel": "reweight_kernel<injections>", "kernel_ms": ms_inj_kernel,
                    "kernel_share_of_step": ms_inj_kernel / (ms / args.steps), "achieved": achieved_inj, "peak": peak,
                    "unit": "TFLOP/s", "frac": achieved_inj / peak, "frac_vs_derived_peak": achieved_inj / peak_derived,
                    "live_fraction_injections": live_frac_inj,
                    "fp64_instr_executed_per_term": None if mp else ex.get("injections_o5"),
                    "frac_executed": None if mp or not ex.get("injections_o5") else
                    terms_inj * ex["injections_o5"] / (ms_inj_kernel * 1e-3) / peak_instr,
                    "note": "same necessary FP64 count per live / dead term as the event instantiation"}
    # DRAM bytes of the event kernel: an ncu figure (a capture, not this run), only for the workload it was taken on;
    # kernel_ms covers the ceil(n_theta / 340) launches of one step, so the traffic is scaled to them
    traffic = O5_DRAM_BYTES_PER_340_THETA * n_theta / 340.0 if spec.name == "o5" and args.table_prec == "f64" else None
    roofline = {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                "traffic": traffic, "traffic_source": "ncu dram__bytes_read.sum + dram__bytes_write.sum of one 340-theta "
                "launch, profiles/r02e_reweight_events_ncu_full.md, scaled to the step's launches (HBM does not bind)"
                if traffic else None, "kernel": "reweight_kernel<events>", "kernel_ms": ms_ev_kernel,
                "kernel_share_of_step": ms_ev_kernel / (ms / args.steps),
                "inj_kernel_ms": ms_inj_kernel,
                "fp64_instr_per_live_term": instr_live, "fp64_instr_per_dead_term": FP64_INSTR_DEAD,
                # the instructions the kernel executes per term (ncu-measured), against the same peak: the FP64 pipe's
                # utilisation as the run itself sees it
                "fp64_instr_executed_per_term": executed,
                "frac_executed": None if executed is None else terms_ev * executed / (ms_ev_kernel * 1e-3) / peak_instr,
                "frac_vs_derived_peak": achieved / peak_derived,
                "frac_executed_vs_derived_peak": None if executed is None else terms_ev * executed / (ms_ev_kernel * 1e-3)
                / FP64_PEAK_INSTR,
                "fp64_count_source": FP64_COUNT_SOURCE,
                # the same time against the budget BASELINE.md froze before any code (180 live / 30 dead): context only
                "frac_at_survey_budget_180_30": terms_ev * (live_frac_ev * 180.0 + (1.0 - live_frac_ev) * 30.0)
                / (ms_ev_kernel * 1e-3) / FP64_PEAK_INSTR,
                "live_fraction_events": live_frac_ev,
                "peak_source": "measured in this run: dependent-free DFMA probe on all SMs (gwc_probe_fp64, best of 3)",
                "peak_derived": peak_derived,
                "peak_derived_source": "148 SM x 64 FP64 lanes x 1.965 GHz x 2 (DESIGN.md section 7)",
                "peak_measured_dfma_probe": peak}
    roofline.update(fp64_count_state(gwc.LIB_PATH))
    # ---- NEXT row 2, reported beside the headline: the event term with the per-pixel N_eff cut (Eq. 8) ----
    pix = None
    if args.pixcut >= 0:
        ctx.gwc_build_cosmo(theta, zmax, args.n_nodes, prec)
        ctx.gwc_event_loglik_pixcut(theta, W.ev, W.los, zmax, args.pixcut)
        torch.cuda.synchronize()
        ctx.gwc_set_timing(True)
        ctx.gwc_get_timing()
        npass = None
        for _ in range(2):
            _, _, _, npass = ctx.gwc_event_loglik_pixcut(theta, W.ev, W.los, zmax, args.pixcut)
        torch.cuda.synchronize()
        tp = ctx.gwc_get_timing()
        ctx.gwc_set_timing(False)
        ms_pix = tp["ms_ev"] / max(tp["n_ev"], 1)
        pix = {"neff_min": args.pixcut, "event_kernel_ms": ms_pix, "event_terms_per_s": terms_ev / (ms_pix * 1e-3),
               "slowdown_vs_uncut": ms_pix / ms_ev_kernel, "mean_passing_pixels_per_event": float(npass.double().mean())}
        del npass
    # ---- NEXT row 1, reported beside the headline: the event term with the paper's KDE numerator (Eq. 5-7) on a
    # bounded slice of the theta batch (it needs 256 Gaussian evaluations per (theta, sample) instead of one term) ----
    kde = None
    if args.kde_theta > 0:
        th_k = theta[:min(args.kde_theta, n_theta)].contiguous()
        ctx.gwc_build_cosmo(th_k, zmax, args.n_nodes, prec)
        ctx.gwc_event_loglik_kde(th_k, W.ev, W.los, zmax, 256, 2.0)
        torch.cuda.synchronize()
        ctx.gwc_set_timing(True)
        ctx.gwc_get_timing()
        nused = None
        for _ in range(2):
            _, _, nused = ctx.gwc_event_loglik_kde(th_k, W.ev, W.los, zmax, 256, 2.0)
        torch.cuda.synchronize()
        tk = ctx.gwc_get_timing()
        ctx.gwc_set_timing(False)
        ms_kde = tk["ms_ev"] / max(tk["n_ev"], 1)
        evals = float(nused.sum().item()) * 256.0
        kde = {"n_theta": int(th_k.shape[0]), "n_grid": 256, "neff_min": 2.0, "kernel_ms": ms_kde,
               "event_terms_per_s": th_k.shape[0] * n_samples / (ms_kde * 1e-3),
               "gaussian_evals_per_s": evals / (ms_kde * 1e-3),
               "fp64_instr_per_eval": KDE_FP64_INSTR_PER_EVAL,
               "fp64_count_source": "ncu op counters over the Gaussian evaluations of the launch, profiles/r02f_kde_ncu_full.md",
               "roofline_frac_fp64": evals * KDE_FP64_INSTR_PER_EVAL / (ms_kde * 1e-3) / FP64_PEAK_INSTR,
               # (round 1 counted 10 instructions per evaluation for the kernel of that round: the same time on that scale)
               "roofline_frac_fp64_at_r01_count_10": evals * 10.0 / (ms_kde * 1e-3) / FP64_PEAK_INSTR}
        del nused
    # ---- NEXT row 4, reported beside the headline: one theta per call (the sampler's pattern), catalogue cache on ----
    lat = None
    if args.latency_calls > 0:
        th1 = theta[:1].contiguous()
        ctx.gwc_cache_catalogue(True)
        try:
            for _ in range(3):
                ctx.gwc_total_loglik(th1, W.ev, W.inj, W.los, zmax, allsky, args.n_nodes, prec)
            torch.cuda.synchronize()
            l0, l1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            t0 = time.perf_counter()
            l0.record()
            for _ in range(args.latency_calls):
                ctx.gwc_total_loglik(th1, W.ev, W.inj, W.los, zmax, allsky, args.n_nodes, prec)
            l1.record()
            torch.cuda.synchronize()
            wall = (time.perf_counter() - t0) / args.latency_calls * 1e3
            # what one call must stream (HBM-bound at one theta): the prepared samples (d_L, m1z, m2z, ln m1z, ln q, P: 48 B
            # + 4 B row per event sample) and the two LOS nodes of every event sample (2 x 4 B, f32 table)
            los_b = 2 * W.los.element_size()
            lat_bytes = n_samples * (52 + los_b) + n_inj * 48
            hbm, hbm_src = _hbm_peak()
            dev_ms = l0.elapsed_time(l1) / args.latency_calls
            lat = {"n_theta": 1, "calls": args.latency_calls, "device_ms_per_call": dev_ms,
                   "wall_ms_per_call": wall, "catalogue_cache": True,
                   "roofline": {"bound": "hbm", "bytes_per_call": lat_bytes, "achieved": lat_bytes / (dev_ms * 1e-3) / 1e9,
                                "peak": hbm, "unit": "GB/s", "frac": lat_bytes / (dev_ms * 1e-3) / 1e9 / hbm,
                                "peak_source": hbm_src}}
        finally:
            ctx.gwc_cache_catalogue(False)
    a0 = a0_report(ctx, W, spec, args.seed) if args.a0 else None
    cpu = (cpu_baseline(spec, args.seed, W=W, theta=theta, budget_s=args.cpu_seconds, mass_model=args.mass_model)
           if args.cpu_seconds > 0 else None)
    stress = stress_report(ctx, W, theta, zmax, allsky, args.n_nodes) if spec.name == "stress" else None
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": spec.name, "mass_model": args.mass_model, "n_theta": n_theta, "n_events": spec.n_events, "n_samples": n_samples,
                   "n_injections": n_inj, "los_rows": spec.los_rows, "n_z": spec.n_z, "los_dtype": spec.los_dtype,
                   "cosmo_table": "%s x %d nodes" % (args.table_prec, args.n_nodes), "seed": args.seed,
                   "parallelism": "theta-sharded x%d, catalogue replicated" % world,
                   "l2": "inputs larger than L2 (samples %.0f MB + LOS table %.0f MB per pass)"
                         % (n_samples * 28 / 1e6, W.los.numel() * W.los.element_size() / 1e6),
                   "generation_s": round(t_gen, 1)},
        "evals_per_s": n_theta * world * args.steps / (ms * 1e-3),
        "event_terms_per_s_kernel": terms_ev / (ms_ev_kernel * 1e-3),
        "inj_terms_per_s_kernel": terms_inj / (ms_inj_kernel * 1e-3) if ms_inj_kernel > 0 else None,
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": up, "d2h_bytes_per_step": down,
                "ms_per_step": ms_e2e / e2e_steps, "steps": e2e_steps, "matches_device_path": same},
        "gpu_launches": int(launches),
        "roofline": roofline,
        "roofline_inj": roofline_inj,
        "cpu_baseline": cpu,
    }
    if stress is not None:
        line["stress_report"] = stress
    if pix is not None:
        line["pixcut"] = pix
    if kde is not None:
        line["kde"] = kde
    if lat is not None:
        line["latency"] = lat
    if a0 is not None:
        line["a0_pack"] = a0
    print(json.dumps(line))
    if dist:
        td.destroy_process_group()


def a0_report(ctx, W, spec, seed):
    """A0 at full size (untimed region of the bench): gwc_pack_events + gwc_cap_pixels(2500) on the UNSORTED sample
    list of the workload (the synthetic samples come sorted; a seeded permutation unsorts them).  Checked at full size
    by what defines the answer (a permutation; keys ascending; equal keys in input order = the stable sort is unique);
    the bit-for-bit comparison with the oracle is tests/test_gpu_full_size.py::test_pack_full_size.  The paper re-fills its padded tensor on every likelihood
    call ("Fill Arrays": 5.38 ms per call at 2000 events on an H100); here it is one-time."""
    dev = W.ev["dL"].device
    off = W.ev["ev_sample_off"]
    n_ev = int(off.numel()) - 1
    n = int(off[-1])
    eid = torch.repeat_interleave(torch.arange(n_ev, dtype=torch.int32, device=dev), (off[1:] - off[:-1]))
    g = torch.Generator(device=dev).manual_seed(seed + 4242)
    shuf = torch.randperm(n, generator=g, device=dev)
    eid_u, row_u = eid[shuf].contiguous(), W.ev["sample_row"][shuf].contiguous()
    del eid, shuf
    ctx.gwc_pack_events(eid_u, row_u, n_ev)   # warm-up (scratch allocation)
    e0, e1, e2 = (torch.cuda.Event(enable_timing=True) for _ in range(3))
    torch.cuda.synchronize()
    e0.record()
    packed = ctx.gwc_pack_events(eid_u, row_u, n_ev)
    e1.record()
    kept, eso, pso = ctx.gwc_cap_pixels(packed, 2500, seed)
    e2.record()
    torch.cuda.synchronize()
    ms_pack, ms_cap = e0.elapsed_time(e1), e1.elapsed_time(e2)
    perm = packed["perm"]
    key = (eid_u[perm].to(torch.int64) << 32) | row_u[perm].to(torch.int64)
    ok_perm = bool(torch.equal(torch.sort(perm)[0], torch.arange(n, device=dev)))
    ok_sorted = bool((key[1:] >= key[:-1]).all())
    ok_stable = bool(((key[1:] != key[:-1]) | (perm[1:] > perm[:-1])).all())
    ok_off = bool(torch.equal(packed["ev_sample_off"], off))
    del key
    # bytes the packing must move at the least: the two 4-byte keys in, the 8-byte permutation out
    return {"n_samples": n, "n_events": n_ev, "n_pixrefs": int(packed["n_pixrefs"]), "pack_ms": ms_pack,
            "cap2500_ms": ms_cap, "samples_kept_cap2500": int(kept.numel()),
            "pack_samples_per_s": n / (ms_pack * 1e-3), "pack_GBps_algorithmic_16B_per_sample": n * 16 / (ms_pack * 1e-3) / 1e9,
            "full_size_checks": {"permutation": ok_perm, "keys_ascending": ok_sorted, "stable": ok_stable,
                                 "event_offsets": ok_off},
            "paper_fill_arrays_ms_per_call_H100_2000_events": 5.38}


def stress_report(ctx, W, theta, zmax, allsky, n_nodes):
    """Config 5: FP64 tables and FP32 tables (cosmology + LOS) side by side on the whole theta batch (untimed):
    max |delta log L(theta)|, the theta points where a sample flipped across a support edge, and N_eff per event."""
    from paper_2605_23538_b200 import gwc
    los64 = W.los if W.los.dtype == torch.float64 else W.los.to(torch.float64)
    los32 = los64.to(torch.float32)
    res = {}
    for name, los, prec in (("f64", los64, gwc.F64), ("f32", los32, gwc.F32)):
        ctx.gwc_build_cosmo(theta, zmax, n_nodes, prec)
        logL, neff, nlive = ctx.gwc_event_loglik(theta, W.ev, los, zmax)
        tot = ctx.gwc_total_loglik(theta, W.ev, W.inj, los, zmax, allsky, n_nodes, prec)
        res[name] = (logL, neff, nlive, tot)
    ctx.gwc_check()
    t64, t32 = res["f64"][3], res["f32"][3]
    both = torch.isfinite(t64) & torch.isfinite(t32)
    same = (res["f64"][2] == res["f32"][2]).all(dim=1)
    d = (t64 - t32).abs()
    neff = res["f64"][1]
    fin = torch.isfinite(res["f64"][0])
    q = torch.quantile(neff[fin][:: max(1, int(fin.sum()) // 1_000_000)], torch.tensor([0.0, 0.05, 0.5, 0.95, 1.0],
                                                                                      dtype=neff.dtype, device=neff.device))
    mx = lambda m: float(d[m].max().item()) if bool(m.any()) else None
    return {"n_theta_finite_both": int(both.sum()), "max_abs_dlogL_no_flip": mx(both & same),
            "n_theta_with_flip": int((~same).sum()), "max_abs_dlogL_with_flip": mx(both & ~same),
            "neff_per_event_quantiles_0_5_50_95_100": [float(x) for x in q],
            "frac_event_terms_minus_inf": float((~fin).float().mean().item())}


# ---------------------------------------------------------------------------------------------
def cpu_baseline(spec, seed, W=None, theta=None, budget_s=15.0, mass_model="plpeak"):
    """The oracle as it stands, on the host cores, on a bounded sample of the workload:
    the first theta points x the first events (all their samples) + the same theta x a slice of injections."""
    import oracle
    with oracle.mass_model(mass_model):
        return _cpu_baseline(oracle, spec, seed, W, theta, budget_s)


def _cpu_baseline(oracle, spec, seed, W, theta, budget_s):
    if W is None:
        small = synth.scaled(spec, n_events=min(spec.n_events, 64), n_inj=min(spec.n_inj, 50_000),
                             los_rows=min(spec.los_rows, 4096))
        W = synth.make_workload(small, seed=seed, device="cpu", keep_f64_los=False)
        theta = synth.make_theta(small, seed, "cpu")
    cores = oracle.num_threads()
    n_ev = min(int(W.ev["ev_sample_off"].numel()) - 1, 32)
    off = W.ev["ev_sample_off"][: n_ev + 1].cpu()
    ns = int(off[-1])
    rows = W.ev["sample_row"][:ns].cpu().to(torch.int64)
    r_lo, r_hi = int(rows.min()), int(rows.max()) + 1
    # only the touched block of LOS rows goes to the host (row ids shifted to match)
    los = W.los[r_lo:r_hi].cpu().numpy()
    ev = {"ev_sample_off": off.numpy(), "dL": W.ev["dL"][:ns].cpu().numpy(), "m1z": W.ev["m1z"][:ns].cpu().numpy(),
          "m2z": W.ev["m2z"][:ns].cpu().numpy(), "sample_row": (rows - r_lo).to(torch.int32).numpy(),
          "log_pe_prior": None}
    n_inj = min(int(W.inj["dL"].numel()), 4 * ns)
    inj = {k: (v[:n_inj].cpu().numpy() if isinstance(v, torch.Tensor) else v) for k, v in W.inj.items()}
    allsky = W.los.mean(0, dtype=torch.float64).cpu().numpy()   # plain torch, not the CUDA path
    th = theta.cpu().numpy()
    # calibrate on `cores` theta points, then size the timed run to the budget
    n0 = min(cores, th.shape[0])
    t0 = time.perf_counter()
    oracle.event_loglik(th[:n0], ev, los, spec.z_max)
    oracle.selection_logxi(th[:n0], inj, allsky, spec.z_max)
    t_cal = max(time.perf_counter() - t0, 1e-3)
    n_th = int(max(n0, min(th.shape[0], (budget_s / t_cal) * n0)))
    n_th = max(cores, (n_th // cores) * cores) if th.shape[0] >= cores else th.shape[0]
    n_th = min(n_th, th.shape[0])
    t0 = time.perf_counter()
    oracle.event_loglik(th[:n_th], ev, los, spec.z_max)
    oracle.selection_logxi(th[:n_th], inj, allsky, spec.z_max)
    dt = time.perf_counter() - t0
    terms = float(n_th) * (ns + n_inj)
    # the same oracle on ONE thread (terms/s/core), on as many theta points as ~2 s allow
    n1 = int(max(1, min(n0, round(2.0 / t_cal * n0 / max(cores, 1)))))
    oracle.set_num_threads(1)
    try:
        t0 = time.perf_counter()
        oracle.event_loglik(th[:n1], ev, los, spec.z_max)
        oracle.selection_logxi(th[:n1], inj, allsky, spec.z_max)
        dt1 = time.perf_counter() - t0
    finally:
        oracle.set_num_threads(cores)
    return {"value": terms / dt, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": "%d theta x (first %d events = %d samples + first %d injections), TABLE mode, %.1f s"
                      % (n_th, n_ev, ns, n_inj, dt),
            "seconds": dt, "value_one_core": float(n1) * (ns + n_inj) / dt1,
            "sample_one_core": "%d theta on 1 thread, %.1f s" % (n1, dt1)}


def run_reference(args):
    """--impl reference: the CPU oracle on a bounded sample, same metric/unit (rank 0 only)."""
    if _env_int("RANK", 0) != 0:
        return
    spec = _bench_spec(args.workload, args.theta_scale)
    small = synth.scaled(spec, n_events=min(spec.n_events, 32), n_inj=min(spec.n_inj, 100_000),
                         los_rows=min(spec.los_rows, 4096), n_theta=min(spec.n_theta, 256))
    W = synth.make_workload(small, seed=args.seed, device="cpu", keep_f64_los=False)
    theta = synth.make_theta(small, args.seed, "cpu")
    per_step = max(2.0, min(20.0, 120.0 / max(args.steps + args.warmup, 1)))
    res = None
    for _ in range(args.warmup):
        res = cpu_baseline(small, args.seed, W=W, theta=theta, budget_s=per_step)
    vals, secs = [], 0.0
    for _ in range(args.steps):
        res = cpu_baseline(small, args.seed, W=W, theta=theta, budget_s=per_step)
        vals.append(res["value"])
        secs += res["seconds"]
    value = float(np.mean(vals))
    res["value"] = value
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": _env_int("WORLD_SIZE", 1),
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": secs / max(args.steps, 1) * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": spec.name, "sample": res["sample"], "seed": args.seed},
            "cpu_baseline": res,
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="o5", choices=sorted(synth.CONFIGS))
    ap.add_argument("--impl", default="gwc", choices=["gwc", "reference"])
    ap.add_argument("--theta-scale", type=float, default=1.0, help="scale the theta batch (profiling runs only)")
    ap.add_argument("--table-prec", default="f64", choices=["f64", "f32"])
    ap.add_argument("--n-nodes", type=int, default=1025)
    ap.add_argument("--seed", type=int, default=synth.DEFAULT_SEED)
    ap.add_argument("--cpu-seconds", type=float, default=15.0, help="oracle timing budget (0 = skip)")
    ap.add_argument("--e2e-steps", type=int, default=0, help="0 = --steps, but 2 on o5")
    ap.add_argument("--latency-calls", type=int, default=50,
                    help="also time this many one-theta calls with the catalogue cache on (0: skip)")
    ap.add_argument("--kde-theta", type=int, default=16,
                    help="also time the KDE-numerator event term on this many theta points (0: skip)")
    ap.add_argument("--leg", default="all", choices=["all", "events", "pixcut", "kde", "inj"],
                    help="run one leg alone and print its kernel time (profiling runs)")
    ap.add_argument("--kde-bandwidth", default="scott")
    ap.add_argument("--mass-model", default="plpeak", choices=["plpeak", "multipeak"],
                    help="multipeak: the MULTIPEAK mass model with delta_m smoothing (16-column theta rows)")
    ap.add_argument("--no-a0", dest="a0", action="store_false",
                    help="skip the A0 line (gwc_pack_events + gwc_cap_pixels on the unsorted sample list)")
    ap.add_argument("--pixcut", type=float, default=2.0,
                    help="also time the event term with the per-pixel N_eff cut at this threshold (< 0: skip)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "gwc" and args.theta_scale == 1.0:
        args.warmup = 3
    if args.impl == "reference":
        run_reference(args)
    elif args.leg != "all":
        run_leg(args)
    else:
        run_gwc(args)


if __name__ == "__main__":
    main()
