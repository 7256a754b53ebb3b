"""N > 1 path: shard by parameter point, all-gather the per-point results.

world_size-2 `gloo` processes on CPU.  The per-rank evaluator stands in for the rank's libphylino
context (a GPU is needed for that); what is tested here is the host logic of
paper_2502_15253_b200/sharding.py: slices, padding of uneven slices, order of the gathered rows,
and that the gathered batch equals the unsharded one bit for bit.
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2502_15253_b200 import sharding


def test_shard_points_partition():
    for P in (0, 1, 2, 3, 64, 603, 4096):
        for world in (1, 2, 3, 8):
            cuts = [sharding.shard_points(P, world, r) for r in range(world)]
            assert cuts[0][0] == 0 and cuts[-1][1] == P
            for (a, b), (c, d) in zip(cuts, cuts[1:]):
                assert b == c and a <= b and c <= d
            sizes = [b - a for a, b in cuts]
            assert max(sizes) - min(sizes) <= 1
            assert sizes == sorted(sizes, reverse=True)
            assert sizes == sharding.shard_sizes(P, world)
    with pytest.raises(ValueError):
        sharding.shard_points(4, 2, 2)


def test_single_process_passthrough():
    p = torch.arange(12, dtype=torch.float64).reshape(6, 2)
    out = sharding.sharded_eval(lambda q: q.sum(dim=1), p)
    assert torch.equal(out, p.sum(dim=1))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n_points, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import oracle
        import workloads
        wl = workloads.make_tiny(seed=4242, n_events=60, n_points=n_points, n_datasets=2)
        orc = oracle.Oracle(wl.model, wl.events)
        data = np.arange(orc.total_bins, dtype=np.float64) + 3.0
        params = torch.as_tensor(wl.params)
        seen = []

        def nll_of(p):                      # the rank's evaluator: one row per point of ITS slice
            seen.append(p.shape[0])
            if p.shape[0] == 0:
                return torch.empty(0, dtype=torch.float64)
            return torch.as_tensor(orc.nll(p.numpy(), data))

        def hist_of(p):
            if p.shape[0] == 0:
                return torch.empty((0, orc.total_bins), dtype=torch.float64)
            return torch.as_tensor(orc.spectra(p.numpy()))

        nll = sharding.sharded_eval(nll_of, params)
        hist = sharding.sharded_eval(hist_of, params)
        lo, hi = sharding.shard_points(n_points, world, rank)
        assert seen == [hi - lo]
        full_nll = orc.nll(wl.params, data)
        full_hist = orc.spectra(wl.params)
        assert nll.shape == (n_points,) and hist.shape == (n_points, orc.total_bins)
        assert np.array_equal(nll.numpy(), full_nll), "gathered NLL differs from the unsharded batch"
        assert np.array_equal(hist.numpy(), full_hist)
        with pytest.raises(ValueError):
            sharding.all_gather_points(torch.zeros(hi - lo + 1, dtype=torch.float64), n_points)
        np.save(os.path.join(out_dir, f"nll_{rank}.npy"), nll.numpy())
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("n_points", [5, 4, 1])
def test_world2_gloo_matches_unsharded(tmp_path, oracle_mod, n_points):
    """5 points -> slices of 3 + 2 (padding path), 4 -> 2 + 2, 1 -> 1 + 0 (empty slice)."""
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), n_points, str(tmp_path)), nprocs=world, join=True)
    a = np.load(tmp_path / "nll_0.npy")
    b = np.load(tmp_path / "nll_1.npy")
    assert np.array_equal(a, b) and a.shape == (n_points,)
