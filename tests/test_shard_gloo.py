"""N > 1 host logic on CPU: two gloo ranks shard a query range, evaluate their shares with the
oracle and the concatenation equals the single-rank result; the job time is the max over ranks."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2302_03343_b200 import shard, synth


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n, outdir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle
    oracle.build()
    spec = synth.grid_c0()
    x, q = synth.queries_inside(spec, n, seed=123, strict=True)
    lo, hi = shard.shard_range(n, rank, world)
    og = oracle.OracleGrid(spec.x_knots.numpy(), [t.numpy() for t in spec.q2_subgrids], spec.values.numpy(), spec.pids)
    part = og.xfxq2(spec.pids, x[lo:hi].numpy(), q[lo:hi].numpy())
    np.save(os.path.join(outdir, f"part{rank}.npy"), part)
    ranges = [None] * world
    dist.all_gather_object(ranges, (lo, hi))
    tmax = shard.max_over_ranks(dist, 1.0 + rank)
    if rank == 0:
        np.save(os.path.join(outdir, "meta.npy"), np.array([r for ab in ranges for r in ab] + [tmax]))
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_tile_the_queries(tmp_path, oracle_mod):
    n, world = 20_001, 2
    mp.spawn(_worker, args=(world, _free_port(), n, str(tmp_path)), nprocs=world, join=True)
    meta = np.load(tmp_path / "meta.npy")
    assert list(meta[:4]) == [0, 10_001, 10_001, n] and meta[4] == 2.0
    spec = synth.grid_c0()
    x, q = synth.queries_inside(spec, n, seed=123, strict=True)
    og = oracle_mod.OracleGrid(spec.x_knots.numpy(), [t.numpy() for t in spec.q2_subgrids], spec.values.numpy(), spec.pids)
    full = og.xfxq2(spec.pids, x.numpy(), q.numpy())
    got = np.concatenate([np.load(tmp_path / f"part{r}.npy") for r in range(world)])
    assert np.array_equal(full, got)


def test_shard_range_properties():
    for n in (0, 1, 7, 100, 1_000_003):
        for world in (1, 2, 3, 8):
            edges = [shard.shard_range(n, r, world) for r in range(world)]
            assert edges[0][0] == 0 and edges[-1][1] == n
            assert all(edges[r][1] == edges[r + 1][0] for r in range(world - 1))
            sizes = [b - a for a, b in edges]
            assert max(sizes) - min(sizes) <= 1


def test_table33_generator_shape():
    """NEXT-3 input recipe (Table 3.3): 2415 increasing x-points inside the C1 grid, member-major, one Q2"""
    import torch
    from paper_2302_03343_b200 import synth
    xg = synth.xgrid_table33()
    assert xg.numel() == synth.TABLE33_NX == 2415 and bool((xg[1:] > xg[:-1]).all())
    spec = synth.grid_c1()
    assert float(xg[0]) >= float(spec.x_knots[0]) and float(xg[-1]) < float(spec.x_knots[-1])
    assert float(spec.q2_subgrids[1][0]) < synth.TABLE33_Q2 < float(spec.q2_subgrids[1][-1])
    x, q2, mem = synth.queries_table33(3)
    assert x.numel() == q2.numel() == mem.numel() == 3 * 2415
    assert torch.equal(x[:2415], xg) and torch.equal(x[2415:4830], xg)
    assert torch.equal(mem, torch.arange(3, dtype=torch.int32).repeat_interleave(2415))
    assert bool((q2 == synth.TABLE33_Q2).all())


def _vegas_worker(rank, world, port, n, outdir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle
    oracle.build()
    nb = 16
    edges = np.tile(np.linspace(0.0, 1.0, nb + 1), (2, 1))
    u = np.random.default_rng(77).random((n, 2))
    lo, hi = shard.shard_range(n, rank, world)
    x, jac, bins = oracle.vegas_map(edges, u[lo:hi])
    f = np.exp(-((x - 0.3) ** 2).sum(axis=1) / 0.02)
    sums, hist = oracle.vegas_accumulate(nb, f, jac, bins)
    ts, th = torch.tensor(sums), torch.tensor(hist)
    shard.vegas_allreduce(dist, ts, th)
    new = oracle.vegas_refine(th.numpy(), edges)
    np.save(os.path.join(outdir, f"vegas{rank}.npy"), np.concatenate([ts.numpy(), th.numpy().ravel(), new.ravel()]))
    dist.barrier()
    dist.destroy_process_group()


def test_vegas_sums_allreduce_two_ranks(tmp_path, oracle_mod):
    """NEXT-1's only collective: two ranks sample halves of an iteration, all-reduce the sums and histograms, and both
    end with the single-rank estimate and the single-rank refined grid"""
    n, world, nb = 40_001, 2, 16
    mp.spawn(_vegas_worker, args=(world, _free_port(), n, str(tmp_path)), nprocs=world, join=True)
    a, b = np.load(tmp_path / "vegas0.npy"), np.load(tmp_path / "vegas1.npy")
    assert np.array_equal(a, b)
    edges = np.tile(np.linspace(0.0, 1.0, nb + 1), (2, 1))
    u = np.random.default_rng(77).random((n, 2))
    x, jac, bins = oracle_mod.vegas_map(edges, u)
    f = np.exp(-((x - 0.3) ** 2).sum(axis=1) / 0.02)
    sums, hist = oracle_mod.vegas_accumulate(nb, f, jac, bins)
    new = oracle_mod.vegas_refine(hist, edges)
    want = np.concatenate([sums, hist.ravel(), new.ravel()])
    assert np.max(np.abs(a - want) / (np.abs(want) + 1e-300)) < 1e-12
