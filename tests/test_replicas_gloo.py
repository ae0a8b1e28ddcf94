"""N>1 path on CPU: world_size-2 gloo processes run the replicas host logic bench.py uses (seed per rank, max-time /
sum-units aggregation).  The path has no data-path collective (replicas only)."""
import os
import socket
import sys
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    sys.path.insert(0, str(ROOT))
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world),
                      LOCAL_RANK=str(rank))
    import torch.distributed as dist
    from paper_2005_14454_b200 import replicas

    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        r, lr, w = replicas.rank_world()
        seed = replicas.replica_seed(1, r)
        # rank r "measured" (10 + 5 r) ms for 1000 units
        ms, units = replicas.aggregate(10.0 + 5.0 * r, 1000.0, dist)
        q.put((r, lr, w, seed, ms, units, replicas.throughput(ms, units)))
    finally:
        dist.destroy_process_group()


def test_two_rank_replica_aggregation():
    import torch.multiprocessing as mp

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
    assert [x[0] for x in res] == [0, 1] and all(x[2] == 2 for x in res)
    assert res[0][3] != res[1][3]                       # distinct seeds
    for x in res:
        assert x[4] == 15.0 and x[5] == 2000.0          # max of times, sum of units, same on every rank
        assert x[6] == pytest.approx(2000.0 / 15e-3)


def test_single_process_and_validation():
    sys.path.insert(0, str(ROOT))
    from paper_2005_14454_b200 import replicas

    assert replicas.aggregate(3.0, 7.0, None) == (3.0, 7.0)
    assert replicas.replica_seed(0, 0) == 1 and replicas.replica_seed(1, 3) == 4
    with pytest.raises(ValueError):
        replicas.throughput(0.0, 1.0)
    with pytest.raises(ValueError):
        replicas.replica_seed(-1, 0)
