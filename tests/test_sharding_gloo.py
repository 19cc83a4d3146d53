"""N > 1 path on CPU: world_size 2 over gloo (the batch shards by system index, no
data-path collective).  Each rank generates and solves only its shard (with the oracle standing in for
the device kernels -- the host-side logic under test is the shard arithmetic, the per-rank input
generation keyed on the global system index, and the max-over-ranks timing reduction); the gathered
shards must equal the single-process solve of the whole batch bit for bit."""
import os
import socket

import numpy as np
import pytest

import inputs
import oracle
from paper_2107_05395_b200 import sharding

torch = pytest.importorskip("torch")


def test_shard_bounds_cover_exactly():
    for total in (0, 1, 7, 64, 65537):
        for world in (1, 2, 3, 8):
            spans = [sharding.shard_bounds(total, world, r) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == total
            assert all(a[1] == b[0] for a, b in zip(spans, spans[1:]))
            sizes = [b - a for a, b in spans]
            assert max(sizes) - min(sizes) <= 1
    assert sharding.weak_shard(65536, 3) == (196608, 262144)
    with pytest.raises(ValueError):
        sharding.shard_bounds(10, 2, 2)


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, n, total, out_dir):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        j0, j1 = sharding.shard_bounds(total, world, rank)
        ids = np.arange(j0, j1, dtype=np.uint64)
        rhs = inputs.uniform_rhs(n, len(ids), seed=3, systems=ids)     # local interleaved array, local batch
        f = oracle.penta_factor(*inputs.penta_lhs(n, 0.5))
        oracle.penta_solve_interleaved(f, rhs, nsteps=2)
        np.save(os.path.join(out_dir, f"shard{rank}.npy"), rhs)
        # timing reduction: job time is the max over ranks
        def all_max(x):
            t = torch.tensor([x], dtype=torch.float64)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            return float(t.item())
        ms = sharding.max_over_ranks_ms(10.0 + rank, world, all_max)
        assert ms == 10.0 + (world - 1)
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_two_rank_shards_equal_whole_batch(tmp_path):
    import torch.multiprocessing as mp
    oracle.build()
    n, total, world = 64, 1001, 2   # odd total: shards of 501 and 500
    mp.spawn(_worker, args=(world, _free_port(), n, total, str(tmp_path)), nprocs=world, join=True)
    whole = inputs.uniform_rhs(n, total, seed=3)
    oracle.penta_solve_interleaved(oracle.penta_factor(*inputs.penta_lhs(n, 0.5)), whole, nsteps=2)
    got = np.concatenate([np.load(tmp_path / f"shard{r}.npy") for r in range(world)], axis=1)
    assert got.shape == whole.shape
    assert np.array_equal(got, whole)
