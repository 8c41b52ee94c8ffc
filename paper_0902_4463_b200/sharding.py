"""Multi-GPU sharding of a force sweep over the i-particles (option 2).

Every rank holds and predicts ALL j-particles and computes the forces on a contiguous slice of
the i-particles; results are only gathered, there is no data-path collective.  (The paper's own
multi-GPU scheme splits the j-particles instead and sums partial forces on the host,
PAPER.md:122; for a full sweep the i-split needs no reduction at all.)  Host logic only --
no arithmetic of the method lives here.
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
