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


# ---- one observation sharded by time over the ranks -----------------------------------------
def _shard_setup(norm_block=2048):
    import math
    from paper_2101_00941_b200 import inputs as I
    import oracle
    w = I.scaled(I.workload(1), nsamp=30000, name="shardme",
                 pulses=(I.Pulse(dm=50.0, t0=7000, width=8, amp=3.0), I.Pulse(dm=90.0, t0=16380, width=16, amp=2.5),
                         I.Pulse(dm=20.0, t0=24500, width=4, amp=4.0)))
    w = I.scaled(w, norm_block=norm_block)
    x = I.fill(w)
    geo = oracle.geometry(w)
    bmax = max(r.bin for r in w.ranges)
    lcm = math.lcm(*[r.bin for r in w.ranges])
    tail = -(-(max(w.widths) - 1) * bmax // lcm) * lcm
    return w, x, geo, tail


def test_time_shards_partition_the_valid_span():
    from paper_2101_00941_b200 import dist_util
    for nsamp, maxshift, nb, tail, world in [(30000, 159, 2048, 31, 3), (1 << 20, 29664, 65536, 255, 8), (5000, 100, 4096, 31, 4)]:
        sh = dist_util.time_shards(nsamp, maxshift, nb, tail, world)
        assert len(sh) == world
        pos = 0
        for s in sh:
            if s.nsamp == 0:
                assert s.keep == 0
                continue
            assert s.t_first == pos and s.t_first % nb == 0 and s.t_first + s.nsamp <= nsamp
            assert s.nsamp >= s.keep + maxshift                      # every kept output sample has its DM sweep
            pos += s.keep
        assert pos == nsamp - maxshift                               # the kept spans tile [0, t_valid)


def _shard_worker(rank, world, port, q, norm_block=2048):
    os.environ.update(RANK=str(rank), WORLD_SIZE=str(world), LOCAL_RANK=str(rank),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    from paper_2101_00941_b200 import dist_util
    import oracle
    assert dist_util.init("gloo")
    w, x, geo, tail = _shard_setup(norm_block)
    shard = dist_util.time_shards(w.nsamp, geo["maxshift"], w.norm_block, tail, world)[rank]
    if shard.nsamp == 0:
        cands = np.empty(0, dtype=oracle.CAND_DTYPE)         # more ranks than normalisation blocks: nothing to search
    else:
        ws = dist_util.shard_workload(w, shard)
        # each rank searches only its own span -- here through the oracle (CPU box); on GPUs through aa_run
        cands, _ = oracle.run(np.ascontiguousarray(x[shard.t_first:shard.t_first + shard.nsamp]), ws)
    merged = dist_util.merge_shards(cands, shard)
    q.put((rank, None if merged is None else merged.tobytes()))
    dist_util.shutdown()


import pytest


@pytest.mark.parametrize("world,norm_block", [(2, 2048), (3, 16384)])     # 3 ranks for 2 blocks: the last shard is empty
def test_time_sharded_observation_equals_the_whole_gloo(world, norm_block):
    import oracle
    from paper_2101_00941_b200 import dist_util
    w, x, geo, tail = _shard_setup(norm_block)
    whole, _ = oracle.run(x, w)
    assert len(whole) > 100
    shards = dist_util.time_shards(w.nsamp, geo["maxshift"], w.norm_block, tail, world)
    assert (shards[-1].nsamp == 0) == (world == 3)
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_shard_worker, args=(r, world, port, q, norm_block)) for r in range(world)]
    for p in ps:
        p.start()
    out = dict(q.get(timeout=180) for _ in ps)
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert all(out[r] is None for r in range(1, world))
    assert out[0] == whole.tobytes()          # bit-identical candidate list, S/N included


def test_rank_placement_splits_the_cores_of_a_numa_node():
    """dist_util.rank_cpus: 8 ranks on a 2-node, 64-core host get 8 cores each, inside their GPU's node, disjoint
    among the ranks of a node; one rank alone keeps its whole node; unknown topology splits the allowed cores."""
    from paper_2101_00941_b200 import dist_util as D
    allowed = list(range(64))
    nodes = [list(range(0, 32)), list(range(32, 64))]
    got = [D.rank_cpus(r, 8, nodes[r // 4], allowed) for r in range(8)]
    assert all(len(g) == 8 and set(g) <= set(nodes[r // 4]) for r, g in enumerate(got))
    assert len(set(c for g in got for c in g)) == 64
    assert D.rank_cpus(0, 1, nodes[1], allowed) == nodes[1]
    two = [D.rank_cpus(r, 2, None, list(range(16))) for r in range(2)]
    assert sorted(two[0] + two[1]) == list(range(16))
    assert D._parse_cpulist("0-3,8,10-11\n") == [0, 1, 2, 3, 8, 10, 11]
    # best effort on whatever host runs the tests; never raises.  It narrows the process affinity and may set
    # OMP_NUM_THREADS: put both back so that no later test runs on fewer cores
    import os
    aff, omp = os.sched_getaffinity(0), os.environ.get("OMP_NUM_THREADS")
    try:
        info = D.place_rank(0, 1)
        assert "cpus" in info
    finally:
        os.sched_setaffinity(0, aff)
        if omp is None:
            os.environ.pop("OMP_NUM_THREADS", None)
        else:
            os.environ["OMP_NUM_THREADS"] = omp
    assert os.sched_getaffinity(0) == aff and os.environ.get("OMP_NUM_THREADS") == omp

