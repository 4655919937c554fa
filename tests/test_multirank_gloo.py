"""World-size-2 CPU test (gloo) of the N>1 plumbing bench.py uses: no data-path collective,
independent observation per rank, time = max over ranks, work = sum over ranks."""
import os
import socket

import numpy as np
import torch.multiprocessing as mp


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close(); return p


def _worker(rank, world, port, q):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    from paper_2101_00941_b200 import dist_util, inputs as I
    import oracle
    assert dist_util.init("gloo")
    w = dist_util.rank_workload(I.scaled(I.workload(1), nsamp=4096, pulses=()), rank)
    x = I.fill(w)
    # each rank searches its own shard with no exchange: here through the oracle (CPU box)
    cands, geo = oracle.run(x, w, row_subset={0: [0, 5]})
    units = 2 * geo["nout"][0]
    dist_util.barrier()
    t = dist_util.max_over_ranks(1.0 + rank)                 # slowest rank decides
    total = dist_util.sum_over_ranks(units)
    q.put((rank, int(x[:64].sum()), t, total, units))
    dist_util.shutdown()


def test_two_ranks_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in ps:
        p.start()
    out = sorted(q.get(timeout=120) for _ in ps)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, s0, t0, tot0, u0), (r1, s1, t1, tot1, u1) = out
    assert s0 != s1                       # different observations (own noise seed)
    assert t0 == t1 == 2.0                # max over ranks
    assert tot0 == tot1 == u0 + u1        # whole-job units = sum over ranks


def test_single_process_helpers_are_noops():
    from paper_2101_00941_b200 import dist_util, inputs as I
    assert dist_util.max_over_ranks(3.5) == 3.5 and dist_util.sum_over_ranks(7) == 7
    w = I.workload(1)
    assert dist_util.rank_workload(w, 0) is w and dist_util.rank_workload(w, 3).noise_seed == w.noise_seed + 3000
