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
