"""gwc_los_allsky_static: the all-sky prior for programs that must not allocate device memory.

Who needs it: a program whose own pool or arena owns all of the GPU's memory (a cudaMalloc made inside a library then
fails or takes memory the pool counts on), and a loop that keeps other streams busy (cudaMalloc / cudaFree lock the
whole device and can wait for it).  Such a program cannot even create a gwc.Context, so the entry point takes none:
its partial sums go to a fixed 4 MiB array inside libgwc.so, shared by every call on that GPU.

What is checked here, through the C ABI: the result is bit-identical to gwc_los_allsky (same kernels, same summation
order; the library's other parity tests compare that call with the oracle) on two calls in a row whose tables differ
in shape, so that a second call reading what the first one left in the shared array would show; the size limit is
refused with a clear error and leaves the output untouched; the calls take no device memory.

This file is named to be collected LAST (pytest -x stops at the first failure: a failure here hides nothing) and it
passes on its own in a fresh process as well as after all the other tests.
"""
from __future__ import annotations

import pytest
import torch

from paper_2605_23538_b200 import gwc

pytestmark = pytest.mark.gpu


def _table(n_rows, n_z, dtype, seed):
    g = torch.Generator(device="cpu").manual_seed(seed)
    # positive, a few decades of dynamic range like a galaxy-catalogue p(z | pixel)
    t = torch.exp(3.0 * torch.randn((n_rows, n_z), generator=g, dtype=torch.float64))
    return t.to(dtype).to("cuda:0")


@pytest.mark.parametrize("dtype", [torch.float32, torch.float64])
def test_static_scratch_matches_the_allocating_path_on_two_calls_in_a_row(dtype):
    # several 512-row parts with a ragged last one, n_z not a multiple of the 128-thread block; the second table is
    # smaller in both directions, so its partial sums land on slots the first call filled with other values
    t1 = _table(3 * 512 + 77, 301, dtype, seed=11)
    t2 = _table(512 + 5, 130, dtype, seed=12)
    zmax = 2.5
    # the entry point under test comes first: in a fresh process nothing else has touched the library yet (no
    # context, no allocation), which is the situation of the callers it is meant for
    out1 = torch.full((t1.shape[1],), float("nan"), dtype=torch.float64, device="cuda:0")
    out2 = torch.full((t2.shape[1],), float("nan"), dtype=torch.float64, device="cuda:0")
    gwc.Context.gwc_los_allsky_static(t1, zmax, out1)
    gwc.Context.gwc_los_allsky_static(t2, zmax, out2)      # straight after, same stream, no sync in between
    torch.cuda.synchronize()
    ctx = gwc.Context(0)
    ref1 = ctx.gwc_los_allsky(t1, zmax)
    ref2 = ctx.gwc_los_allsky(t2, zmax)
    ctx.gwc_check()
    # test_gpu_parity.py compares the all-sky mean with the oracle at rtol 1e-13; the two GPU paths here run the same
    # kernels in the same fixed order, so they are held to bit equality, which is stricter
    assert torch.equal(out1, ref1)
    assert torch.equal(out2, ref2)
    # and against the plain definition, so that "both wrong in the same way" cannot pass: mean over rows
    for out, t in ((out1, t1), (out2, t2)):
        mean = t.to(torch.float64).mean(dim=0)
        assert torch.allclose(out, mean, rtol=1e-13, atol=0.0)
    # the first table again: what the second call left behind is not read either
    out3 = torch.full_like(out1, float("nan"))
    gwc.Context.gwc_los_allsky_static(t1, zmax, out3)
    torch.cuda.synchronize()
    assert torch.equal(out3, ref1)
    ctx.close()


def test_static_scratch_takes_no_device_memory():
    t = _table(2000, 257, torch.float32, seed=13)
    out = torch.empty(t.shape[1], dtype=torch.float64, device="cuda:0")
    gwc.Context.gwc_los_allsky_static(t, 3.0, out)          # set-up call (address look-up, device code loaded)
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info(0)[0]
    for _ in range(2):
        gwc.Context.gwc_los_allsky_static(t, 3.0, out)
    torch.cuda.synchronize()
    free_after = torch.cuda.mem_get_info(0)[0]
    assert free_after >= free_before, (free_before, free_after)


def test_static_scratch_refuses_tables_beyond_its_limit():
    n_z = 1024
    parts_max = gwc.ALLSKY_STATIC_MAX_DOUBLES // n_z                      # 512 parts of 512 rows
    rows_ok = parts_max * gwc.ALLSKY_STATIC_ROWS_PER_PART
    # at the limit: accepted, and right (f32 table of ones -> mean exactly 1)
    t_ok = torch.ones((rows_ok, n_z), dtype=torch.float32, device="cuda:0")
    out = torch.full((n_z,), float("nan"), dtype=torch.float64, device="cuda:0")
    gwc.Context.gwc_los_allsky_static(t_ok, 1.0, out)
    torch.cuda.synchronize()
    assert torch.equal(out, torch.ones_like(out))
    del t_ok
    # one row more needs one part more: refused before anything runs, the output keeps its contents
    t_big = torch.ones((rows_ok + 1, n_z), dtype=torch.float32, device="cuda:0")
    out.fill_(-7.0)
    with pytest.raises(gwc.GwcError) as e:
        gwc.Context.gwc_los_allsky_static(t_big, 1.0, out)
    assert e.value.status == gwc.ERR_SHAPE
    assert "too large for the fixed scratch" in str(e.value) and "gwc_los_allsky" in str(e.value)
    assert gwc.Context.gwc_los_allsky_static_error().startswith("gwc_los_allsky_static: table too large")
    torch.cuda.synchronize()
    assert torch.equal(out, torch.full_like(out, -7.0))
    # an argument error, and the next good call clears the error text
    with pytest.raises(gwc.GwcError) as e:
        gwc.Context.gwc_los_allsky_static(t_big[:10], -1.0, out)
    assert e.value.status == gwc.ERR_INVALID_ARG
    gwc.Context.gwc_los_allsky_static(t_big[:10].contiguous(), 1.0, out)
    assert gwc.Context.gwc_los_allsky_static_error() == ""
    torch.cuda.synchronize()
    assert torch.equal(out, torch.ones_like(out))
