"""Unit-range shard end to end with the binding's own all-gather (binding.make_allgather on torch.distributed): two
PROCESSES, one context each, gloo between them -- needs a B200 (-m gpu).  The box has one GPU, so both ranks use cuda:0;
no kernel of one rank waits for the other (the exchange is a host-side all-gather between launches), so this is not a
stand-in for two GPUs' timing, only for the data path: every rank must return the unsharded result bit for bit
(exact int64 column sums)."""
import os
import socket

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _worker(rank, world, port, q):
    import torch.distributed as dist

    from paper_1612_04705_b200 import binding
    from paper_1612_04705_b200 import datagen as dg

    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        c = dg.config(1, scale=0.2)
        s = dg.make_sample(c)
        c4 = dg.config(4, scale=0.02)
        s4 = dg.make_sample(c4)
        with binding.Context(0) as ref:                      # unsharded, in this process
            r0 = ref.permutation_test(s.x, s.xbar, 0.3, 600, c.perm_seed)
            t0 = ref.T(s.x, s.xbar, 0.3)
            p0 = ref.podd_test(s4.x, s4.mom_x, s4.xbar, s4.mom_xbar, c4.sigma, 300, c4.perm_seed)
        with binding.Context(0) as ctx:
            ctx.set_shard(rank, world)
            r1 = ctx.permutation_test(s.x, s.xbar, 0.3, 600, c.perm_seed)
            kern = ctx.stats().dominant_kernel
            t1 = ctx.T(s.x, s.xbar, 0.3)
            p1 = ctx.podd_test(s4.x, s4.mom_x, s4.xbar, s4.mom_xbar, c4.sigma, 300, c4.perm_seed)
        ok = (kern == "k_perm_tc" and np.array_equal(r0.T_perm, r1.T_perm) and r0.observed == r1.observed
              and (r0.count_gt, r0.n_near, r0.p_value) == (r1.count_gt, r1.n_near, r1.p_value)
              and np.array_equal(p0.p_odd.T_perm, p1.p_odd.T_perm) and p0.p_even == p1.p_even and p0.count == p1.count
              and abs(t0.T - t1.T) <= 1e-12 * t0.term_scale)   # fp64 partial sums of k_pairs_T: rank-order sum
        q.put((rank, bool(ok), float(r1.observed.T), int(r1.count_gt)))
    finally:
        dist.destroy_process_group()


def test_unit_shard_two_processes_over_gloo():
    import torch.multiprocessing as mp

    from paper_1612_04705_b200 import build

    build.build()   # once, here: the two ranks must not both decide to rebuild libet.so

    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=600) for _ in procs)
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    assert [g[:2] for g in got] == [(0, True), (1, True)], got
    assert got[0][2:] == got[1][2:]      # the ranks agree bit for bit
