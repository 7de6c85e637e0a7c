"""N > 1 host logic on CPU: world_size 2 over gloo (the path has no data-path collective)."""
import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1103_3373_b200 import shard, workloads as wl


def test_shard_range_partitions():
    for Ng in (0, 1, 5, 8192, 8191):
        for world in (1, 2, 3, 8):
            r = [shard.shard_range(Ng, k, world) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == Ng
            assert all(a[1] == b[0] for a, b in zip(r, r[1:]))
            sizes = [b - a for a, b in r]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard.shard_range(4, 2, 2)


def _worker(rank, world, port, Ng, q):
    from oracle import oracle as O
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    try:
        gamma = 5.0 / 3.0
        G = wl.amr_batch(Ng, g=2, gamma=gamma, seed=3, dtype="float64").numpy()
        lo, hi = shard.shard_range(Ng, rank, world)
        local = O.hydro_dt(G[lo:hi], gamma, 0) if hi > lo else 0.0
        t = torch.tensor(local, dtype=torch.float64)
        shard.global_max(t)
        # NaN on one rank must reach every rank as "bad"
        b = torch.tensor(float("nan") if rank == 1 else 1.0, dtype=torch.float64)
        shard.global_max(b)
        q.put((rank, lo, hi, float(t), float(b), O.hydro_dt(G, gamma, 0)))
    finally:
        dist.destroy_process_group()


def test_two_ranks_agree_on_dt():
    world, Ng = 2, 5
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + int(np.random.default_rng().integers(0, 2000))
    ps = [ctx.Process(target=_worker, args=(r, world, port, Ng, q)) for r in range(world)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [(r[1], r[2]) for r in res] == [(0, 3), (3, 5)]
    for r in res:
        assert r[3] == r[5]                  # sharded max == oracle's hydro_dt of the whole batch, exactly
        assert np.isnan(r[4])                # the bad-cell marker reached both ranks AS NaN (hydro_dt's contract), not +inf
