"""GPU test of the multi-GPU j-split on ONE GPU: two clusters of the
library each hold half of the j-particles, two host threads run the real `JSplit.calc` (real kernels behind
the C ABI: force, key pack / select / unpack); only the collective is replaced by an in-process exchange
between the two threads (what an NCCL allreduce does, on the same device buffers).  No kernel waits for
another kernel: the threads meet on the host."""
import threading

import numpy as np
import pytest

from paper_0902_4463_b200 import g6, inputs
from paper_0902_4463_b200.sharding import JSplit, LibOps, j_range
from helpers import check_forces, check_nn

pytestmark = pytest.mark.gpu


class _Exchange:
    """allreduce between `world` host threads on tensors of one device"""

    def __init__(self, world):
        self.world, self.slots, self.bar = world, [None] * world, threading.Barrier(world)

    def allreduce(self, rank):
        import torch

        def f(t, op):
            torch.cuda.synchronize()
            self.slots[rank] = t.clone()
            self.bar.wait()
            parts = torch.stack(self.slots)
            red = parts.min(dim=0).values if op == "min" else parts.sum(dim=0)
            self.bar.wait()
            t.copy_(red)
            torch.cuda.synchronize()
        return f


@pytest.mark.parametrize("n,ni", [(6000, 300), (1, 1), (3000, 3000), (70000, 17)])
def test_jsplit_two_clusters_one_gpu(oracle, n, ni):
    import torch
    from paper_0902_4463_b200 import build
    build.build()
    x, v, m, eps2 = inputs.config("C1", n=max(n, 2))
    x, v, m = x[:n], v[:n], m[:n]
    idx = (np.arange(n, dtype=np.int32) * 5 + 2).astype(np.int32)
    sel = inputs.active_subset(n, ni, 21)
    world = 2
    dev = torch.device("cuda:0")
    t = lambda a, dt=torch.float64: torch.from_numpy(np.ascontiguousarray(a)).to(dev, dt)
    ex = _Exchange(world)
    res, err = [None] * world, []
    g6.g6x_set_npipes(1 << 21)
    for r in range(world):
        g6.g6_open(r)

    def rank_main(r):
        try:
            j0, j1 = j_range(r, world, n)
            if j1 > j0:
                z3 = np.zeros((j1 - j0, 3))
                g6.g6x_set_j_particles(r, 0, idx[j0:j1], np.zeros(j1 - j0), m[j0:j1], z3, z3, v[j0:j1], x[j0:j1])
            else:            # an empty slice still takes part in the collectives: one massless far-away particle
                g6.g6x_set_j_particles(r, 0, np.array([-7], np.int32), np.zeros(1), np.zeros(1), np.zeros((1, 3)), np.zeros((1, 3)),
                                       np.zeros((1, 3)), np.full((1, 3), 1e6))
            g6.g6_set_ti(r, 0.0)
            js = JSplit(LibOps(r), r, world, allreduce=ex.allreduce(r))
            out = js.calc(max(j1 - j0, 1), ni, t(idx[sel], torch.int32), t(x[sel]).reshape(-1), t(v[sel]).reshape(-1), eps2)
            res[r] = [o.cpu().numpy() for o in out]
        except Exception as e:      # noqa: BLE001
            err.append(e)
            ex.bar.abort()

    try:
        th = [threading.Thread(target=rank_main, args=(r,)) for r in range(world)]
        [a.start() for a in th]
        [a.join() for a in th]
    finally:
        for r in range(world):
            g6.g6_close(r)
        g6.g6x_set_npipes(g6.DEFAULT_NPIPES)
    assert not err, err
    ref = oracle.force(idx[sel], x[sel], v[sel], idx, x, v, m, eps2)
    for r in range(world):
        acc, jerk, pot, nn, r2 = res[r]
        if n > 1:
            check_forces(dict(acc=acc, jerk=jerk, pot=pot), ref, f"j-split rank {r}")
            check_nn(nn, ref, idx, x[sel], x)
            assert np.allclose(r2, ref["nn_r2"], rtol=1e-5)
        else:                       # the lone particle is its own i: no force, no neighbour but rank 1's far-away stand-in
            assert np.all(acc == 0) and np.all(pot == 0)
    for a, b in zip(res[0], res[1]):                 # complete and bit-identical on both ranks
        assert np.array_equal(a, b)
