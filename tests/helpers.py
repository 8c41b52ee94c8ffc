"""Shared helpers of the GPU parity tests: load a particle set through the C ABI, compare with
the oracle under the tolerances BASELINE.json's north_star states."""
import numpy as np

from paper_0902_4463_b200 import g6

# north_star tolerances (GPU vs fp64 oracle, per particle)
TOL_ACC_MAX = 1e-5
TOL_ACC_MEDIAN = 1e-6
TOL_JERK_MAX = 1e-4
TOL_POT_MAX = 1e-6
TOL_NN_TIE = 1e-6      # nearest neighbour: exact except ties within this relative distance


def load_j(x, v, m, index=None, t=None, acc=None, jerk=None, clusterid=0, addr0=0):
    """bulk-load a particle set (physical acc/jerk, default 0; t default 0) and size npipes to it."""
    n = len(m)
    index = np.arange(n, dtype=np.int32) if index is None else index
    z3 = np.zeros((n, 3))
    g6.g6x_set_j_particles(clusterid, addr0, index, np.zeros(n) if t is None else t, m,
                           z3 if jerk is None else jerk, z3 if acc is None else acc, v, x)
    return index


def rel_err(got, want):
    """per-particle |got - want| / |want| for [n,3] vectors or [n] scalars"""
    got = np.asarray(got); want = np.asarray(want)
    if got.ndim == 1:
        return np.abs(got - want) / np.abs(want)
    return np.linalg.norm(got - want, axis=1) / np.linalg.norm(want, axis=1)


def check_nn(got_index, ref, index_j, xi, xj, tie=TOL_NN_TIE):
    """Nearest neighbours must be identical to the oracle's, except where the candidate the GPU
    picked is within `tie` relative distance of the oracle's minimum (FP32 cannot separate
    those): compare what is unique, check that the rest is valid."""
    diff = np.nonzero(got_index != ref["nn_index"])[0]
    addr_of = {int(ix): a for a, ix in enumerate(index_j)}
    for i in diff:
        assert got_index[i] >= 0, f"i={i}: GPU found no neighbour, oracle found {ref['nn_index'][i]}"
        a = addr_of[int(got_index[i])]
        d2 = float(np.sum((xj[a] - xi[i]) ** 2))
        dmin = float(ref["nn_r2"][i])
        assert abs(np.sqrt(d2) - np.sqrt(dmin)) <= tie * np.sqrt(dmin), \
            f"i={i}: GPU nn {got_index[i]} at r={np.sqrt(d2)!r}, oracle nn {ref['nn_index'][i]} at r={np.sqrt(dmin)!r}"
    return len(diff)


def check_forces(got, ref, what=""):
    ea = rel_err(got["acc"], ref["acc"]); ej = rel_err(got["jerk"], ref["jerk"]); ep = rel_err(got["pot"], ref["pot"])
    stats = dict(acc_max=ea.max(), acc_median=np.median(ea), jerk_max=ej.max(), jerk_median=np.median(ej),
                 pot_max=ep.max(), pot_median=np.median(ep))
    assert ea.max() <= TOL_ACC_MAX, (what, stats)
    assert np.median(ea) <= TOL_ACC_MEDIAN, (what, stats)
    assert ej.max() <= TOL_JERK_MAX, (what, stats)
    assert ep.max() <= TOL_POT_MAX, (what, stats)
    return stats


TOL_NB = 1e-6          # neighbour lists: membership exact except pairs with |r2 - h2| <= TOL_NB h2


def check_neighbours(got_count, got_list, orc_count, orc_list, index_j, xi, xj, h2, maxlen, tol=TOL_NB):
    """Neighbour lists of the CUDA path (callers' indices, -1 padded rows) against the oracle's
    (j addresses, NOT truncated: call the oracle with a maxlen above every count).  The sphere
    test r2 < h2 is taken in binary32 on the GPU and in fp64 by the oracle, so a pair whose fp64
    r2 is within `tol` (relative) of h2 may fall on either side; everything else must agree:
    compare what is unique, check that the rest is valid.  Lists must be in increasing j address
    and, on overflow, hold the neighbours with the smallest addresses.  Returns the number of
    borderline disagreements."""
    addr_of = {int(ix): a for a, ix in enumerate(index_j)}
    n_border = 0
    for i in range(len(got_count)):
        row = got_list[i]
        G = [addr_of[int(ix)] for ix in row[row >= 0]]
        assert all(a < b for a, b in zip(G, G[1:])), f"i={i}: list not in increasing j address: {G[:8]}..."
        assert len(G) == min(int(got_count[i]), maxlen), (i, len(G), int(got_count[i]), maxlen)
        assert int(orc_count[i]) <= orc_list.shape[1], "oracle list truncated: raise its maxlen"
        O = [int(a) for a in orc_list[i, : orc_count[i]]]

        def border(a):
            r2 = float(np.sum((xj[a] - xi[i]) ** 2))
            return abs(r2 - h2[i]) <= tol * h2[i]

        if got_count[i] <= maxlen and orc_count[i] <= maxlen:
            sym = set(G) ^ set(O)
        else:
            # overflow: stored entries are valid, and no neighbour below the last stored address is missing
            last = G[-1] if len(G) == maxlen else np.inf
            sym = (set(G) - set(O)) | {a for a in O if a < last and a not in set(G)}
            r2 = np.sum((xj - xi[i]) ** 2, axis=1)
            nb = int(np.sum(np.abs(r2 - h2[i]) <= tol * h2[i]))
            assert abs(int(got_count[i]) - int(orc_count[i])) <= nb, (i, int(got_count[i]), int(orc_count[i]), nb)
        for a in sym:
            assert border(a), f"i={i}: j address {a} in one list only and not borderline (h2={h2[i]!r})"
        n_border += len(sym)
    return n_border
