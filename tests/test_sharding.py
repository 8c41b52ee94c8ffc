"""Host logic of the multi-GPU i-split, exercised with world_size = 2 on CPU (gloo)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_0902_4463_b200.sharding import gather_rows, i_range


def test_i_range_partitions_exactly():
    for n in (0, 1, 7, 1024, 1048576, 1000003):
        for world in (1, 2, 3, 4, 8):
            spans = [i_range(r, world, n) for r in range(world)]
            assert spans[0][0] == 0 and spans[-1][1] == n
            for a, b in zip(spans, spans[1:]):
                assert a[1] == b[0]
            sizes = [b - a for a, b in spans]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        i_range(2, 2, 10)


def _worker(rank, world, port, n, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        i0, i1 = i_range(rank, world, n)
        # stand-in for the per-rank force call: a deterministic function of the global row number
        rows = torch.arange(i0, i1, dtype=torch.float64)
        local = torch.stack([rows * 3 + 1, rows * rows, -rows], dim=1)
        full = gather_rows(local, n)
        t = torch.tensor([float(rank + 1)], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)            # the bench's max-over-ranks timing reduction
        if rank == 0:
            np.save(out, np.concatenate([full.numpy().ravel(), t.numpy()]))
    finally:
        dist.destroy_process_group()


def test_gather_rows_world2_gloo(tmp_path):
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    n, world = 1001, 2
    out = str(tmp_path / "full.npy")
    mp.spawn(_worker, args=(world, port, n, out), nprocs=world, join=True)
    got = np.load(out)
    rows = np.arange(n, dtype=np.float64)
    want = np.stack([rows * 3 + 1, rows * rows, -rows], axis=1).ravel()
    assert np.array_equal(got[:-1], want)
    assert got[-1] == 2.0
