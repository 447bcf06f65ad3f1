"""Host-side logic for sharding the permutation loop over ranks (PAPER.md:219 farms the
permutations out as separate jobs).

Permutation p depends only on (seed, p), so a rank evaluates a contiguous window [p0, p0 + count) of the seed's
stream (`ET_OPT_PERM_OFFSET`) against the same observed sample.  No data-path collective is needed: combining the
shards is a concatenation of the `T_perm` windows and a sum of the integer counts, here done with one
`all_gather_object` (works over gloo on CPU and over NCCL).  Nothing in this module evaluates psi or T.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np


def shard_of(rank: int, world: int, nperm_total: int) -> tuple[int, int]:
    """Contiguous, balanced window (p0, count) of rank `rank`; the first `nperm_total % world` ranks get one more."""
    if world < 1 or not (0 <= rank < world) or nperm_total < 0:
        raise ValueError("bad shard request")
    q, r = divmod(nperm_total, world)
    p0 = rank * q + min(rank, r)
    return p0, q + (1 if rank < r else 0)


@dataclass
class Shard:
    """What one rank's et_permutation_test / et_podd_test call returns for its window."""
    p0: int
    T_obs: float
    T_perm: np.ndarray
    count_gt: int
    n_near: int


@dataclass
class Combined:
    T_obs: float
    T_perm: np.ndarray
    count_gt: int
    n_near: int
    nperm: int
    p_value: float


def combine(shards: list[Shard]) -> Combined:
    """Concatenates the windows in stream order and sums the counts.  Every rank evaluated the observed statistic with
    the same deterministic kernels on the same sample, so T_obs must agree bit for bit; windows must tile the range."""
    if not shards:
        raise ValueError("no shards")
    shards = sorted(shards, key=lambda s: s.p0)
    t0 = shards[0].T_obs
    nxt = shards[0].p0
    for s in shards:
        if np.float64(s.T_obs).tobytes() != np.float64(t0).tobytes():
            raise ValueError(f"ranks disagree on T_obs: {s.T_obs!r} vs {t0!r}")
        if s.p0 != nxt:
            raise ValueError(f"permutation windows do not tile the range: expected p0 = {nxt}, got {s.p0}")
        nxt += len(s.T_perm)
    T_perm = np.concatenate([np.asarray(s.T_perm, dtype=np.float64) for s in shards])
    count = int(sum(s.count_gt for s in shards))
    near = int(sum(s.n_near for s in shards))
    n = len(T_perm)
    return Combined(t0, T_perm, count, near, n, count / n if n else float("nan"))


def all_gather_combine(local: Shard, group=None) -> Combined:
    """Every rank contributes its shard and receives the combined result (torch.distributed must be initialised)."""
    import torch.distributed as dist

    world = dist.get_world_size(group)
    parts: list = [None] * world
    dist.all_gather_object(parts, local, group=group)
    return combine(parts)
