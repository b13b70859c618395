"""Multi-rank host logic on CPU: world_size-2 gloo processes shard the target rows, each rank
computes its slice (with the oracle standing in for the per-rank CUDA call), the slices are
all-gathered with the product's ``sharding`` helpers and must equal the unsharded result.
What is under test is the partition and the ragged all-gather, not the arithmetic."""
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

from paper_1602_02170_b200 import sharding, workloads  # noqa: E402


def test_row_partition_covers_and_balances():
    for n in (0, 1, 2, 7, 2000, 15000, 172032, (1 << 20) + 3):
        for world in (1, 2, 3, 4, 8):
            part = sharding.row_partition(n, world)
            assert len(part) == world
            assert part[0][0] == 0 and sum(c for _, c in part) == n
            for r in range(1, world):
                assert part[r][0] == part[r - 1][0] + part[r - 1][1]
            counts = [c for _, c in part]
            assert max(counts) - min(counts) <= 1
            assert all(sharding.shard_rows(n, r, world) == part[r] for r in range(world))
    with pytest.raises(ValueError):
        sharding.shard_rows(10, 2, 2)
    with pytest.raises(ValueError):
        sharding.row_partition(10, 0)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def _worker(rank, world, port, n, k, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    os.environ["OMP_NUM_THREADS"] = "2"
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import oracle
        w = workloads.config1(seed=3, n=n, k=k)
        rb, rc = sharding.shard_rows(n, rank, world)
        rows = np.arange(rb, rb + rc, dtype=np.int64)
        local = oracle.matvec(oracle.WALL, w.pos, w.force, w.a, w.eta, rows=rows)      # [k, rc, 3]
        local_t = torch.from_numpy(np.ascontiguousarray(local))
        bufs = sharding.gather_buffers(n, k, world, local_t.dtype, local_t.device)
        full = sharding.gather_velocities(local_t, n, buffers=bufs)
        again = sharding.gather_velocities(local_t, n)                                  # fresh buffers
        assert torch.equal(full, again)
        # max-over-ranks reduction used by bench.py for the step time
        t = torch.tensor([float(rank + 1)], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        assert t.item() == float(world)
        np.save(os.path.join(out_dir, f"full_{rank}.npy"), full.numpy())
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("n,k", [(301, 2), (64, 1)])
def test_two_rank_gloo_row_sharding_matches_unsharded(tmp_path, n, k):
    import oracle
    world = 2
    port = _free_port()
    mp.spawn(_worker, args=(world, port, n, k, str(tmp_path)), nprocs=world, join=True)
    w = workloads.config1(seed=3, n=n, k=k)
    ref = oracle.matvec(oracle.WALL, w.pos, w.force, w.a, w.eta)
    for rank in range(world):
        got = np.load(tmp_path / f"full_{rank}.npy")
        assert got.shape == ref.shape == (k, n, 3)
        # rows are independent and the oracle sums each row in a fixed order: bit-identical
        assert np.array_equal(got, ref)


def _reduce_worker(rank, world, port, n, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    os.environ["OMP_NUM_THREADS"] = "2"
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import oracle
        w = workloads.config1(seed=5, n=n, k=1)
        # stand-in for rpy_wall_matvec_shard: a partial product for ALL rows (here: the contribution of
        # this rank's slice of the sources), full length on every rank
        lo, cnt = sharding.shard_rows(n, rank, world)
        lam = np.zeros_like(w.force); lam[:, lo:lo + cnt] = w.force[:, lo:lo + cnt]
        part = torch.from_numpy(oracle.matvec(oracle.WALL, w.pos, lam, w.a, w.eta))
        full = sharding.reduce_velocities(part)
        assert full is part
        np.save(os.path.join(out_dir, f"red_{rank}.npy"), full.numpy())
    finally:
        dist.destroy_process_group()


def test_two_rank_gloo_work_sharding_all_reduce(tmp_path):
    import oracle
    world, n = 2, 157
    mp.spawn(_reduce_worker, args=(world, _free_port(), n, str(tmp_path)), nprocs=world, join=True)
    w = workloads.config1(seed=5, n=n, k=1)
    ref = oracle.matvec(oracle.WALL, w.pos, w.force, w.a, w.eta)
    a, b = np.load(tmp_path / "red_0.npy"), np.load(tmp_path / "red_1.npy")
    assert np.array_equal(a, b)                       # every rank ends with the same u
    assert np.allclose(a, ref, rtol=1e-13, atol=1e-15)


def _hook_worker(rank, world, port, n, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    os.environ["OMP_NUM_THREADS"] = "2"
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import oracle
        w = workloads.config1(seed=6, n=n, k=1)
        reduce = sharding.solve_reduce_hook()              # what a sharded solve calls after each product
        lo, cnt = sharding.shard_rows(n, rank, world)
        outs = []
        for it in range(3):                                # three "iterations": a new lambda each time
            lam = np.roll(w.force, it, axis=1)
            mine = np.zeros_like(lam); mine[:, lo:lo + cnt] = lam[:, lo:lo + cnt]
            buf = np.ascontiguousarray(oracle.matvec(oracle.WALL, w.pos, mine, w.a, w.eta)).ravel()
            reduce(buf.ctypes.data, buf.size)              # raw address + count, as the C ABI hands them over
            outs.append(buf.copy())
        np.save(os.path.join(out_dir, f"hook_{rank}.npy"), np.stack(outs))
    finally:
        dist.destroy_process_group()


def test_two_rank_gloo_solve_reduce_hook(tmp_path):
    """The reduction hook of the sharded Krylov loop (rpy_rigid_solve_ext.reduce): a raw address and a count in,
    the sum over the ranks in place, the same on every rank; the oracle stands in for the per-rank CUDA product."""
    import oracle
    world, n = 2, 131
    mp.spawn(_hook_worker, args=(world, _free_port(), n, str(tmp_path)), nprocs=world, join=True)
    w = workloads.config1(seed=6, n=n, k=1)
    a, b = np.load(tmp_path / "hook_0.npy"), np.load(tmp_path / "hook_1.npy")
    assert np.array_equal(a, b)
    for it in range(3):
        ref = oracle.matvec(oracle.WALL, w.pos, np.roll(w.force, it, axis=1), w.a, w.eta).ravel()
        assert np.allclose(a[it], ref, rtol=1e-13, atol=1e-15)
