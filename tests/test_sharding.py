"""The N > 1 path on CPU: world_size-2 gloo processes, theta-sharded.  Each rank evaluates
its own slice of the theta batch (with the CPU oracle standing in for the GPU library, which needs a device),
the slices are gathered, and the result must equal the unsharded evaluation bit for bit."""
from __future__ import annotations

import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

from paper_2605_23538_b200 import shard, synth  # noqa: E402


def test_theta_range_partitions_exactly():
    for n in (0, 1, 2, 7, 16, 4096, 4099):
        for world in (1, 2, 3, 8):
            edges = [shard.theta_range(n, r, world) for r in range(world)]
            assert edges[0][0] == 0 and edges[-1][1] == n
            assert all(edges[r][1] == edges[r + 1][0] for r in range(world - 1))
            sizes = [b - a for a, b in edges]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard.theta_range(4, 2, 2)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, n_theta, out_dir):
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    import oracle
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        oracle.set_num_threads(1)
        spec = synth.scaled(synth.CONFIGS["tiny"], n_theta=n_theta)
        W = synth.make_workload(spec, device="cpu")          # replicated catalogue: same seed on every rank
        lo, hi = shard.theta_range(n_theta, rank, world)
        th = W.theta[lo:hi].numpy()
        tot = oracle.total_loglik(th, synth.to_numpy(W.ev), synth.to_numpy(W.inj), W.los.numpy(), spec.z_max)
        full = shard.gather_theta_results(torch.from_numpy(tot), n_theta)
        slowest = shard.max_over_ranks(float(rank + 1), "cpu")
        assert slowest == float(world)
        np.save(os.path.join(out_dir, "rank%d.npy" % rank), full.numpy())
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("n_theta", [7])
def test_world2_gloo_theta_sharding_matches_single_process(tmp_path, n_theta):
    import oracle
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), n_theta, str(tmp_path)), nprocs=world, join=True)
    spec = synth.scaled(synth.CONFIGS["tiny"], n_theta=n_theta)
    W = synth.make_workload(spec, device="cpu")
    ref = oracle.total_loglik(W.theta.numpy(), synth.to_numpy(W.ev), synth.to_numpy(W.inj), W.los.numpy(), spec.z_max)
    for r in range(world):
        got = np.load(os.path.join(str(tmp_path), "rank%d.npy" % r))
        assert np.array_equal(got, ref, equal_nan=True)


def test_event_range_partitions_exactly():
    rng = np.random.default_rng(0)
    for n_events in (1, 2, 5, 40):
        sizes = rng.integers(1, 5000, n_events)
        off = torch.from_numpy(np.concatenate([[0], np.cumsum(sizes)]).astype(np.int64))
        for world in (1, 2, 3, 8):
            edges = [shard.event_range(off, r, world) for r in range(world)]
            assert edges[0][0] == 0 and edges[-1][1] == n_events
            assert all(edges[r][1] == edges[r + 1][0] for r in range(world - 1))
            if n_events >= 8 * world:
                per = [int(off[b] - off[a]) for a, b in edges]
                assert max(per) <= 2 * int(off[-1]) // world + 5000


def _worker_events(rank, world, port, n_theta, out_dir):
    sys.path.insert(0, ROOT)
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    import oracle
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        oracle.set_num_threads(1)
        spec = synth.scaled(synth.CONFIGS["tiny"], n_theta=n_theta)
        W = synth.make_workload(spec, device="cpu")
        ev, inj = synth.to_numpy(W.ev), synth.to_numpy(W.inj)
        th = W.theta.numpy()
        lo, hi = shard.event_range(W.ev["ev_sample_off"], rank, world)
        off = ev["ev_sample_off"]
        sl = slice(off[lo], off[hi])
        sub = dict(ev_sample_off=(off[lo:hi + 1] - off[lo]).astype(np.int64), dL=ev["dL"][sl], m1z=ev["m1z"][sl],
                   m2z=ev["m2z"][sl], sample_row=ev["sample_row"][sl], log_pe_prior=None)
        los = W.los.numpy()
        if hi > lo:
            logL, _, _ = oracle.event_loglik(th, sub, los, spec.z_max)
            s = np.where(np.isneginf(logL).any(1), -np.inf, logL.sum(1))
        else:
            s = np.zeros(th.shape[0])
        nf = inj["dL"].size
        a, b = shard.theta_range(nf, rank, world)             # the same balanced split serves the injections
        sub_inj = dict(dL=inj["dL"][a:b], m1z=inj["m1z"][a:b], m2z=inj["m2z"][a:b], log_pdraw=inj["log_pdraw"][a:b],
                       n_draw=inj["n_draw"])                  # global n_draw
        allsky = oracle.los_allsky(los, spec.z_max)
        lx, ne = oracle.selection_logxi(th, sub_inj, allsky, spec.z_max)
        total, logxi, neff = shard.combine_event_sharded(torch.from_numpy(s), torch.from_numpy(lx),
                                                         torch.from_numpy(ne), off.size - 1)
        np.save(os.path.join(out_dir, "ev_rank%d.npy" % rank), np.stack([total.numpy(), logxi.numpy(), neff.numpy()]))
    finally:
        dist.destroy_process_group()


def test_world2_gloo_event_sharding_matches_single_process(tmp_path):
    import oracle
    world, n_theta = 2, 6
    mp.spawn(_worker_events, args=(world, _free_port(), n_theta, str(tmp_path)), nprocs=world, join=True)
    spec = synth.scaled(synth.CONFIGS["tiny"], n_theta=n_theta)
    W = synth.make_workload(spec, device="cpu")
    ev, inj, los = synth.to_numpy(W.ev), synth.to_numpy(W.inj), W.los.numpy()
    ref = oracle.total_loglik(W.theta.numpy(), ev, inj, los, spec.z_max)
    lx, ne = oracle.selection_logxi(W.theta.numpy(), inj, oracle.los_allsky(los, spec.z_max), spec.z_max)
    got = [np.load(os.path.join(str(tmp_path), "ev_rank%d.npy" % r)) for r in range(world)]
    assert np.array_equal(got[0], got[1], equal_nan=True)      # every rank holds the same bits
    fin = np.isfinite(ref)
    assert np.array_equal(np.isneginf(got[0][0]), np.isneginf(ref))
    np.testing.assert_allclose(got[0][0][fin], ref[fin], rtol=1e-12)
    np.testing.assert_allclose(got[0][1], lx, rtol=0, atol=1e-12)
    np.testing.assert_allclose(got[0][2], ne, rtol=1e-10)


def test_combine_sharded_host_closed_forms():
    """gwc_combine_sharded_host (the function the device kernel also runs) against what the definitions fix:
    one part is the identity; R equal parts give log xi + ln R and R x N_eff; parts of very different size are summed
    without overflow; a part without live injections (-inf, N_eff 0) adds nothing; -inf and NaN propagate as gwc.h
    states; the total is sum_r S_r - n_events log xi."""
    from paper_2605_23538_b200 import gwc
    f = gwc.Context.gwc_combine_sharded_host
    T = lambda rows: torch.tensor(rows, dtype=torch.float64)
    # one part: identity
    tot, lx, ne = f(T([[-12.5, 3.0]]), T([[-2.0, 700.0]]), T([[40.0, 7.0]]), 5)
    assert lx.tolist() == [-2.0, 700.0] and ne.tolist() == [40.0, 7.0]
    assert tot.tolist() == [-12.5 - 5 * -2.0, 3.0 - 5 * 700.0]
    # R equal parts
    R = 4
    tot, lx, ne = f(T([[1.0]] * R), T([[-3.0]] * R), T([[10.0]] * R), 2)
    np.testing.assert_allclose(lx.numpy(), [-3.0 + np.log(R)], rtol=1e-15)
    np.testing.assert_allclose(ne.numpy(), [R * 10.0], rtol=1e-15)
    np.testing.assert_allclose(tot.numpy(), [R * 1.0 - 2 * (-3.0 + np.log(R))], rtol=1e-15)
    # very different sizes (no overflow of exp), against numpy's logaddexp; N_eff by the definition in linear terms
    x = np.array([-900.0, -905.0, 650.0 - 1550.0])
    n = np.array([3.0, 8.0, 2.0])
    tot, lx, ne = f(T(x[:, None].tolist()), T(x[:, None].tolist()), T(n[:, None].tolist()), 0)
    np.testing.assert_allclose(lx.numpy(), [np.logaddexp.reduce(x)], rtol=1e-15)
    w = np.exp(x - x.max())
    np.testing.assert_allclose(ne.numpy(), [w.sum() ** 2 / (w ** 2 / n).sum()], rtol=1e-14)
    np.testing.assert_allclose(tot.numpy(), [x.sum()], rtol=1e-15)
    # a rank without live injections, a rank without events
    tot, lx, ne = f(T([[0.0], [-7.0]]), T([[-np.inf], [-4.0]]), T([[0.0], [9.0]]), 3)
    assert lx.tolist() == [-4.0] and ne.tolist() == [9.0] and tot.tolist() == [-7.0 + 12.0]
    # -inf stays -inf (never NaN): no live injection anywhere; an event with no live sample
    tot, lx, ne = f(T([[1.0], [2.0]]), T([[-np.inf], [-np.inf]]), T([[0.0], [0.0]]), 3)
    assert lx.tolist() == [-np.inf] and ne.tolist() == [0.0] and tot.tolist() == [-np.inf]
    tot, lx, ne = f(T([[-np.inf], [2.0]]), T([[-1.0], [-1.0]]), T([[5.0], [5.0]]), 3)
    assert tot.tolist() == [-np.inf] and np.isfinite(lx.numpy()).all()
    # NaN in any piece of a theta: that theta's outputs are NaN, its neighbour's are not
    tot, lx, ne = f(T([[1.0, 1.0], [2.0, 2.0]]), T([[-1.0, np.nan], [-1.0, -1.0]]), T([[5.0, 5.0], [5.0, 5.0]]), 3)
    tot, lx, ne = tot.numpy(), lx.numpy(), ne.numpy()
    assert np.isnan(tot[1]) and np.isnan(lx[1]) and np.isnan(ne[1]) and np.isfinite(tot[0]) and np.isfinite(lx[0])
