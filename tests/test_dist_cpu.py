"""World-size-2 CPU tests (gloo) of the multi-rank host logic: shard plan, barrier, and the
max-over-ranks / sum-over-ranks throughput aggregation bench.py uses.  No GPU, no collective on
the data path (the path shards with none)."""
import os
import socket
import sys

import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(world), LOCAL_WORLD_SIZE=str(world),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    from paper_2606_02916_b200 import dist as gdist
    r, lr, w = gdist.init("gloo")
    assert (r, lr, w) == (rank, rank, world)
    local_part, order = gdist.shard_plan(rank, world, 4, 10)
    gdist.barrier()
    # rank r "processes" 10 units in (1 + r) seconds
    value, tmax = gdist.aggregate_throughput(10.0, 1.0 + rank)
    # the ranks of one host split the pack-thread budget a single rank would take (read from LOCAL_WORLD_SIZE)
    threads = gdist.sum_over_ranks(float(gdist.host_threads_for_rank(hardware_threads=16)))
    assert threads == 6.0, threads                 # 0.4 x 16 = 6 threads on the host in total, 3 per rank
    q.put((rank, local_part, order, value, tmax, gdist.max_over_ranks(float(rank)), gdist.sum_over_ranks(1.0)))
    gdist.barrier()


def test_two_ranks_gloo_shard_and_aggregate():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    ps = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in ps:
        p.start()
    out = sorted(q.get(timeout=120) for _ in range(world))
    for p in ps:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, lp0, o0, v0, t0, m0, s0), (r1, lp1, o1, v1, t1, m1, s1) = out
    assert (lp0, lp1) == (0, 1)                      # rank r trains owner partition r mod P
    assert sorted(o0) == sorted(o1) == list(range(10))  # weak scaling: a full epoch each
    assert o0[0] == 0 and o1[0] == 5                 # rotated so ranks see different windows
    assert v0 == v1 == 20.0 / 2.0                    # units of all ranks / max time
    assert t0 == t1 == 2.0 and m0 == m1 == 1.0 and s0 == s1 == 2.0


def test_single_process_is_identity():
    sys.path.insert(0, ROOT)
    from paper_2606_02916_b200 import dist as gdist
    assert gdist.max_over_ranks(3.5) == 3.5 and gdist.sum_over_ranks(2.0) == 2.0
    assert gdist.aggregate_throughput(10.0, 2.0) == (5.0, 2.0)
    lp, order = gdist.shard_plan(0, 1, 4, 7)
    assert lp == 0 and order == list(range(7))


def test_pack_thread_split_between_ranks_of_one_host():
    sys.path.insert(0, ROOT)
    from paper_2606_02916_b200 import dist as gdist
    assert gdist.host_threads_for_rank(1, 16) == 0               # alone: the library's default
    assert gdist.host_threads_for_rank(2, 16) == 3 and gdist.host_threads_for_rank(4, 16) == 1
    assert gdist.host_threads_for_rank(8, 16) == 1               # never below one thread
    assert gdist.host_threads_for_rank(8, 192) == 2              # the budget is capped at 16 threads per host
    for n in (2, 4, 8):
        for hw in (8, 16, 64, 192):
            assert n * gdist.host_threads_for_rank(n, hw) <= max(n, min(16, max(2, (hw * 2 + 2) // 5)))
