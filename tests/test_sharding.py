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


# ---------------------------------------------------------------- j-split, host logic on CPU
class _OracleOps:
    """Stand-in for the library's device-side steps so that JSplit's sequencing and collectives can run
    on CPU: partial forces of the rank's j-slice from the oracle, and a numpy transcription of the key
    protocol include/g6.h states for g6x_jsplit_{pack,select,unpack}_dev."""
    NONE = np.iinfo(np.int64).max

    def __init__(self, orc, idx_j, xj, vj, mj):
        self.orc, self.idx_j, self.xj, self.vj, self.mj = orc, idx_j, xj, vj, mj

    def calc_dev(self, nj, ni, d_index, d_xi, d_vi, eps2, d_acc, d_jerk, d_pot, d_nn_index, d_nn_r2):
        r = self.orc.force(d_index.numpy(), d_xi.numpy().reshape(ni, 3), d_vi.numpy().reshape(ni, 3),
                           self.idx_j[:nj], self.xj[:nj], self.vj[:nj], self.mj[:nj], eps2)
        d_acc.copy_(torch.from_numpy(r["acc"].ravel())); d_jerk.copy_(torch.from_numpy(r["jerk"].ravel()))
        d_pot.copy_(torch.from_numpy(r["pot"])); d_nn_index.copy_(torch.from_numpy(r["nn_index"]))
        d_nn_r2.copy_(torch.from_numpy(r["nn_r2"].astype(np.float32).astype(np.float64)))

    def pack(self, ni, rank, d_nn_r2, d_nn_index, d_key):
        bits = d_nn_r2.numpy().astype(np.float32).view(np.uint32).astype(np.int64)
        key = np.where(d_nn_index.numpy() < 0, self.NONE, (bits << 32) | rank)
        d_key.copy_(torch.from_numpy(key))

    def select(self, ni, rank, d_key_min, d_nn_index, d_index_f64):
        k = d_key_min.numpy()
        mine = (k != self.NONE) & ((k & 0xffffffff) == rank)
        d_index_f64.copy_(torch.from_numpy(np.where(mine, d_nn_index.numpy().astype(np.float64), 0.0)))

    def unpack(self, ni, d_key_min, d_index_sum, d_nn_index, d_nn_r2):
        k = d_key_min.numpy()
        has = k != self.NONE
        d_nn_index.copy_(torch.from_numpy(np.where(has, d_index_sum.numpy().astype(np.int32), -1).astype(np.int32)))
        r2 = (k >> 32).astype(np.uint32).view(np.float32).astype(np.float64)
        d_nn_r2.copy_(torch.from_numpy(np.where(has, r2, np.inf)))

    def sync(self):
        pass


def _jsplit_worker(rank, world, port, n, ni, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    os.environ["OMP_NUM_THREADS"] = "2"
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from oracle import oracle as orc
        from paper_0902_4463_b200 import inputs
        from paper_0902_4463_b200.sharding import JSplit, j_range
        x, v, m, eps2 = inputs.config("C1", n=n)
        idx = (np.arange(n, dtype=np.int32) * 3 + 5).astype(np.int32)
        j0, j1 = j_range(rank, world, n)
        sel = inputs.active_subset(n, ni, 5)
        ops = _OracleOps(orc, idx[j0:j1], x[j0:j1], v[j0:j1], m[j0:j1])
        js = JSplit(ops, rank, world)
        t = lambda a, dt=torch.float64: torch.from_numpy(np.ascontiguousarray(a)).to(dt)
        acc, jerk, pot, nn, r2 = js.calc(j1 - j0, ni, t(idx[sel], torch.int32), t(x[sel]).reshape(-1), t(v[sel]).reshape(-1), eps2)
        np.savez(out + f".{rank}.npz", acc=acc.numpy(), jerk=jerk.numpy(), pot=pot.numpy(), nn=nn.numpy(), r2=r2.numpy())
    finally:
        dist.destroy_process_group()


def test_jsplit_world2_gloo(tmp_path, oracle):
    from paper_0902_4463_b200 import inputs
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    n, ni, world = 1500, 96, 2
    out = str(tmp_path / "js")
    mp.spawn(_jsplit_worker, args=(world, port, n, ni, out), nprocs=world, join=True)
    x, v, m, eps2 = inputs.config("C1", n=n)
    idx = (np.arange(n, dtype=np.int32) * 3 + 5).astype(np.int32)
    sel = inputs.active_subset(n, ni, 5)
    ref = oracle.force(idx[sel], x[sel], v[sel], idx, x, v, m, eps2)
    for rank in range(world):                        # complete and identical on every rank
        got = np.load(out + f".{rank}.npz")
        rel = lambda a, b: np.linalg.norm(a - b, axis=1) / np.linalg.norm(b, axis=1)
        assert rel(got["acc"], ref["acc"]).max() < 1e-12 and rel(got["jerk"], ref["jerk"]).max() < 1e-11
        assert np.allclose(got["pot"], ref["pot"], rtol=1e-13)
        assert np.array_equal(got["nn"], ref["nn_index"])
        assert np.allclose(got["r2"], ref["nn_r2"], rtol=1e-7)
