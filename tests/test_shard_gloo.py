"""Multi-rank host logic on CPU (gloo, world size 2): walker sharding and the gather of the logL slices."""
import os
import socket

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2005_01827_b200 import shard


def test_shard_rows_partition_is_exact_and_balanced():
    for B in (0, 1, 2, 3, 7, 64, 1024, 1025):
        for world in (1, 2, 3, 8):
            ranges = [shard.shard_rows(B, world, r) for r in range(world)]
            assert ranges[0][0] == 0 and ranges[-1][1] == B
            assert all(ranges[i][1] == ranges[i + 1][0] for i in range(world - 1))
            sizes = [b - a for a, b in ranges]
            assert max(sizes) - min(sizes) <= 1 and sizes == sorted(sizes, reverse=True)
    with pytest.raises(ValueError):
        shard.shard_rows(4, 2, 2)


def _fake_loglike(rows):
    # a deterministic per-row function standing in for mbhl_loglike (host logic only is under test)
    return (rows * torch.arange(1, 12, dtype=torch.float64)).sum(dim=1) - 0.5 * rows[:, 0] ** 2


def _worker(rank, world, port, B, out_dir):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        g = torch.Generator().manual_seed(1234)
        params = torch.rand((B, 11), dtype=torch.float64, generator=g)       # identical on every rank
        calls = []

        def evaluate(rows):
            calls.append(int(rows.shape[0]))
            return _fake_loglike(rows)

        full = shard.sharded_loglike(evaluate, params)
        a, b = shard.shard_rows(B, world, rank)
        assert calls == [b - a]                                            # each rank evaluated only its rows
        np.save(os.path.join(out_dir, f"r{rank}.npy"), full.numpy())
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("B", [5, 64, 1])
def test_sharded_loglike_world_size_2_gloo(tmp_path, B):
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    mp.spawn(_worker, args=(2, port, B, str(tmp_path)), nprocs=2, join=True)
    g = torch.Generator().manual_seed(1234)
    params = torch.rand((B, 11), dtype=torch.float64, generator=g)
    ref = _fake_loglike(params).numpy()
    for r in range(2):
        got = np.load(tmp_path / f"r{r}.npy")
        assert np.array_equal(got, ref)                                     # bitwise: no arithmetic in the gather


def test_without_process_group_is_a_plain_call():
    p = torch.ones((3, 11), dtype=torch.float64)
    assert torch.equal(shard.sharded_loglike(_fake_loglike, p), _fake_loglike(p))
