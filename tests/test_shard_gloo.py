"""The N > 1 path on CPU: two gloo ranks each take their contiguous slice of one batch of
cells (no collective on the data path), and the timing reduction is a MAX all-reduce.
The per-slice results, computed here by the oracle standing in for the GPU, must tile the
single-process result exactly (cells are independent)."""
import os
import socket

import numpy as np
import pytest

import ckgen
import oracle
from paper_2008_08483_b200.shard import cell_slice, max_over_ranks, rank_cells

torch = pytest.importorskip("torch")


def test_cell_slices_partition_the_batch():
    for n in (0, 1, 7, 1024, 1 << 20, (1 << 20) + 3):
        for world in (1, 2, 3, 8):
            edges = [cell_slice(n, r, world) for r in range(world)]
            assert edges[0][0] == 0 and edges[-1][1] == n
            assert all(edges[r][1] == edges[r + 1][0] for r in range(world - 1))
            sizes = [hi - lo for lo, hi in edges]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        cell_slice(10, 2, 2)


def _rank_batch(cfg, n, rank, world, scaling):
    """The batch bench.py --gpus N gives a rank (same three lines as there)."""
    n_gen, lo, hi, off = rank_cells(n, rank, world, scaling)
    T, P, Y = ckgen.states(cfg, N=n_gen, seed_offset=off)
    return T[lo:hi], P[lo:hi], np.ascontiguousarray(Y[:, lo:hi])


def test_weak_batches_differ_and_strong_slices_tile_one_batch():
    cfg = ckgen.CONFIGS["tiny_1k"]
    n, world = 1001, 3
    weak = [_rank_batch(cfg, n, r, world, "weak") for r in range(world)]
    assert all(b[0].shape == (n,) and b[2].shape == (cfg.mech.S, n) for b in weak)
    for r in range(1, world):                       # rank-local seeded batches are different cells
        assert not np.array_equal(weak[0][0], weak[r][0]) and not np.array_equal(weak[0][2], weak[r][2])
    T, P, Y = ckgen.states(cfg, N=n)
    assert np.array_equal(weak[0][0], T)            # rank 0 of a weak run is the 1-GPU workload
    strong = [_rank_batch(cfg, n, r, world, "strong") for r in range(world)]
    assert np.array_equal(np.concatenate([b[0] for b in strong]), T)
    assert np.array_equal(np.concatenate([b[1] for b in strong]), P)
    assert np.array_equal(np.concatenate([b[2] for b in strong], axis=1), Y)
    assert sum(b[0].shape[0] for b in strong) == n
    with pytest.raises(ValueError):
        rank_cells(n, 0, world, "diagonal")


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n_total, out_dir):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        cfg = ckgen.CONFIGS["tiny_1k"]
        mech = ckgen.mechanism(cfg.mech)
        n_gen, lo, hi, off = rank_cells(n_total, rank, world, "strong")
        assert (lo, hi) == cell_slice(n_total, rank, world)
        T, P, Y = ckgen.states(cfg, N=n_gen, seed_offset=off)
        w, d, _ = oracle.source_terms(oracle.OracleMechanism(mech), T[lo:hi], P[lo:hi],
                                      np.ascontiguousarray(Y[:, lo:hi]), nthreads=1)
        np.savez(os.path.join(out_dir, "rank%d.npz" % rank), w=w, d=d, lo=lo, hi=hi)
        slowest = max_over_ranks(10.0 + rank, dist)          # rank 1 is "slower"
        assert slowest == 10.0 + world - 1
    finally:
        dist.destroy_process_group()


def test_two_ranks_tile_the_single_process_result(tmp_path):
    import torch.multiprocessing as mp
    n_total, world = 1001, 2
    mp.spawn(_worker, args=(world, _free_port(), n_total, str(tmp_path)), nprocs=world, join=True)
    cfg = ckgen.CONFIGS["tiny_1k"]
    mech = ckgen.mechanism(cfg.mech)
    T, P, Y = ckgen.states(cfg, N=n_total)
    w_ref, d_ref, _ = oracle.source_terms(oracle.OracleMechanism(mech), T, P, Y, nthreads=1)
    covered = 0
    for r in range(world):
        z = np.load(os.path.join(str(tmp_path), "rank%d.npz" % r))
        lo, hi = int(z["lo"]), int(z["hi"])
        assert np.array_equal(z["w"], w_ref[:, lo:hi]) and np.array_equal(z["d"], d_ref[lo:hi])
        covered += hi - lo
    assert covered == n_total
