"""The N > 1 path on CPU: two processes over gloo (127.0.0.1).  The E_loc path shards by sample with no
data-path collective; what has to be right is the row partition, the mini-batch a rank
takes at a step, and the reduction of the per-rank statistics.  Per-rank E_loc values come from the fp64 oracle
(no GPU here); the combined statistics must equal the unsharded ones (Eq. 17 with collapsed
repeated samples, :196-202 batch split over GPUs)."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2208_05637_b200 import workloads as wl
from paper_2208_05637_b200.distributed import (all_reduce_gradient, all_reduce_stats, max_over_ranks, minibatch_of_step,
                                               shard_rows)
from oracle import eloc as oeloc
from oracle import grad as ograd


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _inputs():
    w = wl.WORKLOADS[1]
    h, g = wl.make_integrals(w.n_spatial, w.seed_integrals)
    x, z, c = wl.jw_pauli_terms(h, g)
    params = wl.make_made_params(w.n_qubits, w.hidden, w.seed_weights)
    samples, counts = wl.make_samples(w.n_spatial, w.n_alpha, w.n_beta, 37, w.max_count, w.seed_samples, w.unique)
    return w, wl.masks_to_codes(x, z, w.n_qubits), c, params, samples, counts


def _worker(rank, world, port, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w, codes, c, params, samples, counts = _inputs()
        lo, hi = shard_rows(len(samples), world, rank)
        e = oeloc.local_energy(codes, c, params, samples[lo:hi])
        stats = torch.from_numpy(oeloc.weighted_stats(e, counts[lo:hi], max_ratio=1.0 + rank))
        all_reduce_stats(stats)
        slowest = max_over_ranks(10.0 + rank)
        np.save(os.path.join(out_dir, f"rank{rank}.npy"), np.concatenate([stats.numpy(), [slowest, lo, hi]]))
        # gradient exchange: Eq. 7 on the shard with the GLOBAL baseline / normalisation, then a SUM
        tot, b = stats[0].item(), complex(stats[1].item(), stats[2].item()) / stats[0].item()
        cs = counts[lo:hi].astype(np.float64)
        g = ograd.flatten(ograd.dlogpsi_weighted(params, samples[lo:hi], cs * (e.real - b.real) / tot, cs * (e.imag - b.imag) / tot))
        g = torch.from_numpy(g)
        all_reduce_gradient(g)
        np.save(os.path.join(out_dir, f"grad{rank}.npy"), g.numpy())
    finally:
        dist.destroy_process_group()


def test_two_rank_statistics_equal_unsharded(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    w, codes, c, params, samples, counts = _inputs()
    ref = oeloc.weighted_stats(oeloc.local_energy(codes, c, params, samples), counts, max_ratio=2.0)
    got = [np.load(tmp_path / f"rank{r}.npy") for r in range(world)]
    for r in range(world):
        np.testing.assert_allclose(got[r][:4], ref[:4], rtol=1e-12, atol=1e-12)    # sums over the union of the shards
        assert got[r][4] == 2.0                                                      # max |ratio| over ranks
        assert got[r][5] == 11.0                                                     # timing rule: max over ranks
    assert (got[0][6], got[0][7], got[1][6], got[1][7]) == (0, 18, 18, 37)           # contiguous, disjoint, complete
    # the summed per-rank gradients equal Eq. 7 on the whole batch
    gref, _ = ograd.energy_gradient(params, samples, counts, oeloc.local_energy(codes, c, params, samples))
    for r in range(world):
        np.testing.assert_allclose(np.load(tmp_path / f"grad{r}.npy"), gref, rtol=1e-11, atol=1e-13)


def test_partitions_and_step_schedule():
    for n_rows in (0, 1, 37, 8192, 65536):
        for world in (1, 2, 3, 8):
            parts = [shard_rows(n_rows, world, r) for r in range(world)]
            assert parts[0][0] == 0 and parts[-1][1] == n_rows
            assert all(parts[r][1] == parts[r + 1][0] for r in range(world - 1))
            sizes = [hi - lo for lo, hi in parts]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard_rows(10, 2, 2)
    # one step of `world` ranks covers `world` distinct mini-batches; 8 / world steps cover the 8 of config 5 once
    for world in (1, 2, 4, 8):
        seen = [minibatch_of_step(k, r, world, 8) for k in range(8 // world) for r in range(world)]
        assert sorted(seen) == list(range(8))
    with pytest.raises(ValueError):
        all_reduce_stats(torch.zeros(4, dtype=torch.float64))
