"""g6x_calc_dev_noalloc (include/g6.h): the force call that allocates nothing -- its partial sums live in a fixed
file-scope device array -- against the existing path (g6x_calc_dev) and the oracle, on two calls in a row that share
the array with different shapes, plus its limit and its sequence rule.  Collected last on purpose (pytest -x)."""
import numpy as np
import pytest

from helpers import check_forces, check_nn, load_j
from paper_0902_4463_b200 import g6, inputs

pytestmark = pytest.mark.gpu


@pytest.fixture()
def cluster():
    from paper_0902_4463_b200 import build
    build.build()
    g6.g6_open(0)
    yield 0
    g6.g6_close(0)
    g6.g6x_set_npipes(g6.DEFAULT_NPIPES)


def _call(fn, n, block, x, v, idx, eps2):
    import torch
    dev = torch.device("cuda", 0)
    f64 = torch.float64
    ni = len(block)
    to = lambda a, dt=f64: torch.from_numpy(np.ascontiguousarray(a)).to(dev, dt)
    d_xi, d_vi, d_ii = to(x[block]), to(v[block]), to(idx[block], torch.int32)
    d_acc = torch.full((ni, 3), float("nan"), dtype=f64, device=dev); d_jerk = torch.full_like(d_acc, float("nan"))
    d_pot = torch.full((ni,), float("nan"), dtype=f64, device=dev); d_r2 = torch.full_like(d_pot, float("nan"))
    d_nn = torch.full((ni,), -7, dtype=torch.int32, device=dev)
    fn(0, n, ni, d_ii, d_xi, d_vi, eps2, d_acc, d_jerk, d_pot, d_nn, d_r2)
    g6.g6x_synchronize(0)
    return dict(acc=d_acc.cpu().numpy(), jerk=d_jerk.cpu().numpy(), pot=d_pot.cpu().numpy(),
                nn_index=d_nn.cpu().numpy(), nn_r2=d_r2.cpu().numpy())


def test_no_alloc_entry_point_matches_existing_path_twice(cluster, oracle):
    n = 5000                                               # 20 j-tiles, the last one ragged
    x, v, m, eps2 = inputs.config("C1", n=n)
    idx = load_j(x, v, m)
    g6.g6x_set_npipes(1 << 17)
    g6.g6_set_ti(0, 0.0)
    g6.g6x_noalloc_init(0)
    assert g6.g6x_noalloc_max_rows() == 65536
    # two calls in a row on the shared array: a large block (few splits, [s][i] layout), then a small one (many splits,
    # [i][s] layout) that finds the first call's partials in the array
    for ni, seed in ((700, 1), (37, 2), (700, 1)):
        block = inputs.active_subset(n, ni, seed)
        got = _call(g6.g6x_calc_dev_noalloc, n, block, x, v, idx, eps2)
        ref_path = _call(g6.g6x_calc_dev, n, block, x, v, idx, eps2)
        for k in ("acc", "jerk", "pot", "nn_r2"):
            assert np.all(np.isfinite(got[k])), k
        check_forces(got, ref_path, f"no-alloc vs g6x_calc_dev, ni = {ni}")
        assert np.array_equal(got["nn_index"], ref_path["nn_index"])
        assert np.allclose(got["nn_r2"], ref_path["nn_r2"], rtol=1e-6, atol=0)
        ref = oracle.force(idx[block], x[block], v[block], idx, x, v, m, eps2)
        check_forces(got, ref, f"no-alloc vs oracle, ni = {ni}")
        check_nn(got["nn_index"], ref, idx, x[block], x)


def test_no_alloc_limit_and_sequence(cluster):
    import torch
    n = 600
    x, v, m, eps2 = inputs.config("C1", n=n)
    idx = load_j(x, v, m)
    g6.g6x_set_npipes(1 << 17)
    g6.g6_set_ti(0, 0.0)
    dev = torch.device("cuda", 0)
    big = g6.g6x_noalloc_max_rows() + 1
    z3 = torch.zeros(big, 3, dtype=torch.float64, device=dev); z1 = torch.zeros(big, dtype=torch.float64, device=dev)
    zi = torch.zeros(big, dtype=torch.int32, device=dev)
    with pytest.raises(g6.G6Error) as e:                   # beyond the fixed scratch: a clear error, nothing launched
        g6.g6x_calc_dev_noalloc(0, n, big, zi, z3, z3, eps2, z3.clone(), z3.clone(), z1.clone(), zi.clone(), z1.clone())
    assert e.value.code == -4 and "scratch" in str(e.value)
    # a pending j-particle update: the call stages nothing, so it refuses until the buffer is flushed
    g6.g6_set_j_particle(0, 5, int(idx[5]), 0.0, 0.125, m[5], None, np.zeros(3), np.zeros(3), v[5], x[5])
    block = np.arange(10, dtype=np.int32)
    with pytest.raises(g6.G6Error) as e:
        _call(g6.g6x_calc_dev_noalloc, n, block, x, v, idx, eps2)
    assert e.value.code == -6
    g6.g6_flush_jp_buffer(0)
    got = _call(g6.g6x_calc_dev_noalloc, n, block, x, v, idx, eps2)
    ref_path = _call(g6.g6x_calc_dev, n, block, x, v, idx, eps2)
    check_forces(got, ref_path, "after the flush")
