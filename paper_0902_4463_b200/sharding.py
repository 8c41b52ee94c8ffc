"""Multi-GPU sharding of the force path.  Two ways, one process per GPU:

i-split (option 2, `i_range` + `gather_rows`; what bench.py times under torchrun):

Every rank holds and predicts ALL j-particles and computes the forces on a contiguous slice of
the i-particles; results are only gathered, there is no data-path collective.  (The paper's own
multi-GPU scheme splits the j-particles instead and sums partial forces on the host,
PAPER.md:122; for a full sweep the i-split needs no reduction at all.)  Host logic only --
no arithmetic of the method lives here.

j-split (option 1, the paper's own scheme, section 2.4; `JSplit`): every rank holds N_j / Q of the
j-particles (increasing address ranges by rank) and computes partial forces on the SAME i-block; the
exchange step is two allreduces on device buffers -- MIN on 64-bit nearest-neighbour keys, then SUM on
[8][n_i] fp64 (acc, jerk, pot and the winner's neighbour index) -- NCCL over NVLink on GPUs.  The packing
of the keys and the selection of the winner run in the library's CUDA kernels (g6x_jsplit_*_dev); this
module only sequences calls and collectives.  The paper notes the scheme pays off only for large
N_j / Q (it loses below N ~ 64k on 4 GPUs): per force call it costs two small allreduces.
"""
from __future__ import annotations


def i_range(rank: int, world: int, n: int) -> tuple[int, int]:
    """[i0, i1) of `rank`: contiguous, sizes differ by at most one, all n covered exactly once."""
    if not (0 <= rank < world) or n < 0:
        raise ValueError((rank, world, n))
    q, r = divmod(n, world)
    i0 = rank * q + min(rank, r)
    return i0, i0 + q + (1 if rank < r else 0)


def gather_rows(local, n: int, group=None):
    """all-gather per-rank row blocks (torch tensors [ni_r, ...]) into the full [n, ...] tensor."""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size(group)
    sizes = [i_range(r, world, n)[1] - i_range(r, world, n)[0] for r in range(world)]
    pad = max(sizes)
    buf = torch.zeros((pad,) + tuple(local.shape[1:]), dtype=local.dtype, device=local.device)
    buf[: local.shape[0]] = local
    parts = [torch.empty_like(buf) for _ in range(world)]
    dist.all_gather(parts, buf, group=group)
    return torch.cat([p[:s] for p, s in zip(parts, sizes)], dim=0)


j_range = i_range       # the j-particles are split the same way: contiguous, increasing by rank


class JSplit:
    """One rank of a j-split force calculation.  `calc` is given the whole i-block on
    every rank and returns the complete forces on every rank.

    ops: an object with the four device-side steps
         calc_dev(nj, ni, d_index, d_xi, d_vi, eps2, d_acc, d_jerk, d_pot, d_nn_index, d_nn_r2)
         pack(ni, rank, d_nn_r2, d_nn_index, d_key), select(ni, rank, d_key_min, d_nn_index, d_index_f64),
         unpack(ni, d_key_min, d_index_sum, d_nn_index, d_nn_r2)
    -- `LibOps` binds them to libg6b200; tests may bind a stand-in to exercise the sequencing on CPU.
    allreduce(tensor, op): the collective ("min" / "sum"), default torch.distributed on `group`.
    """

    def __init__(self, ops, rank: int, world: int, group=None, allreduce=None):
        self.ops, self.rank, self.world, self.group = ops, rank, world, group
        self._allreduce = allreduce or self._dist_allreduce

    def _dist_allreduce(self, t, op):
        import torch.distributed as dist
        dist.all_reduce(t, op=dist.ReduceOp.MIN if op == "min" else dist.ReduceOp.SUM, group=self.group)

    def calc(self, nj_local, ni, d_index, d_xi, d_vi, eps2):
        """Returns (acc[ni,3], jerk[ni,3], pot[ni], nn_index[ni], nn_r2[ni]) complete on every rank.

        Stream-ordered: the device steps and the two collectives are enqueued back to back on ONE stream (`LibOps` puts
        the library on torch's current stream, on which torch.distributed orders its NCCL work), with no host
        synchronisation in between; the results are complete when that stream has drained (the caller synchronises
        when it reads them)."""
        import torch
        dev = d_xi.device
        f64 = torch.float64
        buf = torch.empty(8 * ni, dtype=f64, device=dev)             # acc | jerk | pot | winner's index: ONE sum-allreduce
        acc, jerk, pot, idxf = buf[: 3 * ni], buf[3 * ni: 6 * ni], buf[6 * ni: 7 * ni], buf[7 * ni:]
        nn = torch.empty(ni, dtype=torch.int32, device=dev)
        r2 = torch.empty(ni, dtype=f64, device=dev)
        key = torch.empty(ni, dtype=torch.int64, device=dev)
        self.ops.calc_dev(nj_local, ni, d_index, d_xi, d_vi, eps2, acc, jerk, pot, nn, r2)
        self.ops.pack(ni, self.rank, r2, nn, key)
        self._allreduce(key, "min")
        self.ops.select(ni, self.rank, key, nn, idxf)
        self._allreduce(buf, "sum")
        self.ops.unpack(ni, key, idxf, nn, r2)
        return acc.view(ni, 3), jerk.view(ni, 3), pot, nn, r2


class LibOps:
    """The device-side steps of `JSplit`, bound to libg6b200 (CUDA kernels behind the C ABI).

    The library normally works on a stream of its own; torch.distributed orders a collective after the work already
    enqueued on torch's CURRENT stream and makes that stream wait for the collective.  So that kernels and collectives
    are ordered without host synchronisation, the cluster is moved onto torch's current stream here (`g6x_set_stream`);
    `own_stream=True` keeps the library's stream and falls back to a host synchronisation around every collective."""

    def __init__(self, clusterid=0, own_stream=False):
        from . import g6
        self.g6, self.c, self.own_stream = g6, clusterid, own_stream
        if not own_stream:
            import torch
            # torch's default stream has handle 0, which g6x_set_stream reads as "the library's own": name it explicitly
            # (cudaStreamLegacy = 0x1)
            g6.g6x_set_stream(clusterid, torch.cuda.current_stream().cuda_stream or 1)

    def calc_dev(self, nj, ni, d_index, d_xi, d_vi, eps2, d_acc, d_jerk, d_pot, d_nn_index, d_nn_r2):
        self.g6.g6x_calc_dev(self.c, nj, ni, d_index, d_xi, d_vi, eps2, d_acc, d_jerk, d_pot, d_nn_index, d_nn_r2)

    def pack(self, ni, rank, d_nn_r2, d_nn_index, d_key):
        self.g6.g6x_jsplit_pack_dev(self.c, ni, rank, d_nn_r2, d_nn_index, d_key)
        self._fence()

    def select(self, ni, rank, d_key_min, d_nn_index, d_index_f64):
        self._fence()
        self.g6.g6x_jsplit_select_dev(self.c, ni, rank, d_key_min, d_nn_index, d_index_f64)
        self._fence()

    def unpack(self, ni, d_key_min, d_index_sum, d_nn_index, d_nn_r2):
        self._fence()
        self.g6.g6x_jsplit_unpack_dev(self.c, ni, d_key_min, d_index_sum, d_nn_index, d_nn_r2)

    def _fence(self):
        # only when the library keeps a stream of its own: both directions (library -> collective, collective -> library)
        if self.own_stream:
            import torch
            self.g6.g6x_synchronize(self.c)
            torch.cuda.current_stream().synchronize()

    def sync(self):
        self.g6.g6x_synchronize(self.c)
