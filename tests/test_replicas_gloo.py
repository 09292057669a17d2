"""N > 1 path of bench.py on CPU: two gloo ranks, replicas with their own seeds, MAX-over-ranks time
and SUM-over-ranks work (tier rule: the path does not shard, no data-path collective)."""
import os
import socket
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank),
                      WORLD_SIZE=str(world), LOCAL_RANK=str(rank))
    from paper_2511_15196_b200 import replicas
    dist.init_process_group("gloo", rank=rank, world_size=world)
    r, w, l = replicas.rank_info()
    assert (r, w, l) == (rank, world, rank)
    # rank 1 is the slow one and did more work
    t, u = replicas.reduce_stats({"run": 10.0 + 5.0 * rank, "e2e": 20.0 - rank},
                                 {"site_updates": 1000.0 * (rank + 1)})
    seeds = [replicas.replica_seed(s, rank) for s in range(3)]
    out.put((rank, t, u, seeds, replicas.throughput(u["site_updates"], t["run"])))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_reduction_and_seeds():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, t, u, seeds, thr in res:
        assert t == {"run": 15.0, "e2e": 20.0}           # MAX over ranks
        assert u == {"site_updates": 3000.0}             # SUM over ranks
        assert thr == pytest.approx(3000.0 / 15e-3)
    assert set(res[0][3]).isdisjoint(res[1][3])          # replicas draw different streams


def test_single_process_is_identity():
    sys.path.insert(0, ROOT)
    from paper_2511_15196_b200 import replicas
    t, u = replicas.reduce_stats({"run": 3.0}, {"site_updates": 7.0})
    assert t == {"run": 3.0} and u == {"site_updates": 7.0}
    assert replicas.replica_seed(5, 0) == 5 and replicas.replica_seed(5, 2) == 5 + 2 * 7919
