"""N > 1 host logic on CPU: two gloo ranks shard the events, time a step and reduce max / sum."""
import os
import socket
import sys

import numpy as np
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, ws, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(RANK=str(rank), LOCAL_RANK=str(rank), WORLD_SIZE=str(ws), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    from paper_1705_02876_b200 import sharding
    from workloads import barrel_events as W
    r, lr, w = sharding.init("gloo")
    assert (r, w) == (rank, ws)
    ev = list(sharding.events_of_rank(3, rank))
    cfg = W.get_config(2)
    first = W.simulate_event(cfg, ev[0], n_tracks=8)
    sharding.barrier()
    t_max = sharding.max_over_ranks(10.0 + rank)
    n_sum = sharding.sum_over_ranks(float(len(ev) * 8))
    strong = list(sharding.split_events(7, rank, ws))
    q.put((rank, ev, float(first.par[3, 0]), t_max, n_sum, strong))
    sharding.shutdown()


def test_two_ranks_shard_events_without_overlap():
    ws, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, ws, port, q)) for r in range(ws)]
    for p in ps:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(ws))
    for p in ps:
        p.join(60)
        assert p.exitcode == 0
    (r0, ev0, x0, t0, n0, s0), (r1, ev1, x1, t1, n1, s1) = res
    assert ev0 == [0, 1, 2] and ev1 == [3, 4, 5]            # weak scaling: disjoint global event ids
    assert x0 != x1                                          # different events -> different tracks
    assert t0 == t1 == 11.0                                  # max over ranks
    assert n0 == n1 == 48.0                                  # whole-job unit count
    assert s0 + s1 == list(range(7)) and abs(len(s0) - len(s1)) <= 1


def test_single_process_defaults():
    from paper_1705_02876_b200 import sharding
    for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE"):
        os.environ.pop(k, None)
    assert sharding.world() == (0, 0, 1)
    assert sharding.max_over_ranks(3.5) == 3.5 and sharding.sum_over_ranks(2.0) == 2.0
    assert list(sharding.split_events(5, 0, 1)) == [0, 1, 2, 3, 4]
