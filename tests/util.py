"""Shared helpers of the parity tests: workloads on the host, oracle calls, comparison rules."""
from __future__ import annotations

import numpy as np
import torch

from paper_2605_23538_b200 import synth

# north_star tolerances
RTOL_F64 = 1e-9      # relative, log L_i and log xi, FP64 path
ATOL_F32 = 1e-4      # absolute, log L(theta), FP32-table path


def workload(config, seed=synth.DEFAULT_SEED, **kw):
    """Seeded workload generated on the CPU (so the oracle and the GPU see identical bits)."""
    spec = synth.CONFIGS[config] if isinstance(config, str) else config
    if kw:
        spec = synth.scaled(spec, **kw)
    return synth.make_workload(spec, seed=seed, device="cpu")


def to_dev(d, device):
    return {k: (v.to(device) if isinstance(v, torch.Tensor) else v) for k, v in d.items()}


def assert_close_log(gpu, ref, rtol, what):
    """Compare log-valued arrays: -inf must match -inf, NaN must match NaN, the rest within rtol (relative)."""
    gpu = np.asarray(gpu, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    assert gpu.shape == ref.shape, (what, gpu.shape, ref.shape)
    nan_g, nan_r = np.isnan(gpu), np.isnan(ref)
    assert np.array_equal(nan_g, nan_r), "%s: NaN pattern differs" % what
    inf_g, inf_r = np.isneginf(gpu), np.isneginf(ref)
    assert np.array_equal(inf_g, inf_r), "%s: -inf pattern differs (%d vs %d)" % (what, inf_g.sum(), inf_r.sum())
    fin = ~(nan_r | inf_r)
    if fin.any():
        err = np.abs(gpu[fin] - ref[fin]) / np.maximum(np.abs(ref[fin]), 1.0)
        worst = float(err.max())
        assert worst <= rtol, "%s: max relative error %.3e > %.1e" % (what, worst, rtol)
        return worst
    return 0.0
