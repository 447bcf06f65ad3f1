"""Multi-rank path on CPU: world_size 2 over gloo.  The permutation range is sharded; each
rank stands in for its GPU with the oracle's values for its window, and the gathered result must equal the
single-rank permutation test: same T_perm order, same count, same p-value."""
import os
import socket

import numpy as np
import pytest

import oracle
from paper_1612_04705_b200 import sharding


def test_shard_windows_tile_the_range():
    for world in (1, 2, 3, 8):
        for total in (0, 1, 7, 1000, 1001):
            nxt = 0
            for r in range(world):
                p0, cnt = sharding.shard_of(r, world, total)
                assert p0 == nxt and cnt in (total // world, total // world + 1)
                nxt += cnt
            assert nxt == total
    with pytest.raises(ValueError):
        sharding.shard_of(2, 2, 10)


def _sample():
    rng = np.random.default_rng(11)
    return rng.random((23, 3)), rng.random((31, 3)) * 0.9 + 0.1


def _shard_from_oracle(full, p0, cnt):
    tp = full.T_perm[p0:p0 + cnt]
    return sharding.Shard(p0, full.observed.T, tp, int((tp > full.observed.T).sum()), 0)


def test_combine_matches_single_rank_and_rejects_bad_shards():
    x, xb = _sample()
    full = oracle.perm_test(x, xb, 0.3, 37, 5)
    parts = [_shard_from_oracle(full, *sharding.shard_of(r, 3, 37)) for r in (2, 0, 1)]
    c = sharding.combine(parts)
    assert np.array_equal(c.T_perm, full.T_perm) and c.count_gt == full.count_gt and c.p_value == full.p_value
    with pytest.raises(ValueError):
        sharding.combine(parts[:2])  # a window is missing
    parts[0].T_obs = np.nextafter(parts[0].T_obs, 1.0)
    with pytest.raises(ValueError):
        sharding.combine(parts)  # ranks disagree on the observed statistic


def _worker(rank, world, port, q):
    import torch.distributed as dist

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        x, xb = _sample()
        full = oracle.perm_test(x, xb, 0.3, 41, 0xE7E57)
        mine = _shard_from_oracle(full, *sharding.shard_of(rank, world, 41))
        mine.T_obs = float(np.float32(mine.T_obs))  # strip the last bits so that the bit-for-bit T_obs check passes
        c = sharding.all_gather_combine(mine)
        # each process ran its own oracle; OpenMP's reduction order may differ between them in the last bit
        ok = (np.allclose(c.T_perm, full.T_perm, rtol=0, atol=1e-15) and c.count_gt == full.count_gt
              and c.p_value == full.p_value and c.nperm == 41
              and np.array_equal(c.T_perm[slice(*np.cumsum(sharding.shard_of(rank, world, 41)))],
                                 full.T_perm[slice(*np.cumsum(sharding.shard_of(rank, world, 41)))]))
        q.put((rank, bool(ok)))
    finally:
        dist.destroy_process_group()


def test_gloo_world2_gather():
    import torch.multiprocessing as mp

    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert got == [(0, True), (1, True)]


# ---- unit-range shard (et_set_shard): the all-gather callback of the binding over gloo -------------------------------
def _unit_shard_worker(rank, world, port, q):
    """What libet.so does around the callback, with plain host arrays standing in for the device sums: each rank holds
    its partial int64 column sums (here: every world-th entry of a fixed table of per-unit sums), hands the callback a
    host buffer [world][count] with its own slice filled in, and adds the slices in rank order."""
    import ctypes

    import torch.distributed as dist

    from paper_1612_04705_b200 import binding

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        rng = np.random.default_rng(7)  # the same table on every rank
        units = rng.integers(-2**40, 2**40, size=(37, 1024), dtype=np.int64)   # per-unit contributions to 2 x 512 columns
        total = units.sum(axis=0)
        mine = units[rank::world].sum(axis=0)
        cb = binding._ALLGATHER(binding.make_allgather(rank, world))
        ok = True
        for trial in range(2):  # the library calls it once per 512-column launch
            buf = np.zeros((world, 1024), dtype=np.int64)
            buf[rank] = mine + trial
            rc = cb(None, buf.ctypes.data, 1024 * 8)
            ok = ok and rc == 0 and np.array_equal(buf.sum(axis=0), total + world * trial)
            ok = ok and all(np.array_equal(buf[r], units[r::world].sum(axis=0) + trial) for r in range(world))
        # doubles travel as bytes too: bit patterns survive
        d = np.zeros((world, 3), dtype=np.float64)
        d[rank] = [np.pi * (rank + 1), -0.0, 1e-300]
        ok = ok and cb(None, d.ctypes.data, 24) == 0 and all(d[r, 0] == np.pi * (r + 1) for r in range(world))
        q.put((rank, bool(ok)))
    finally:
        dist.destroy_process_group()


def test_gloo_world2_unit_shard_allgather():
    import torch.multiprocessing as mp

    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_unit_shard_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert got == [(0, True), (1, True)]
