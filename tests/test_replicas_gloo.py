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


def test_bench_gpus_n_starts_n_ranks():
    """`python bench.py --gpus 2` started WITHOUT a torchrun environment must itself start 2 ranks (the way the driver
    runs it at N = 1 is the same command line).  The launcher self-test runs that path on CPU over gloo: same re-exec,
    same replicas.aggregate (max of the times, sum of the units), same JSON printing by rank 0 only."""
    import json
    import os
    import subprocess
    import sys
    from pathlib import Path

    root = Path(__file__).resolve().parent.parent
    env = {k: v for k, v in os.environ.items() if k not in ("RANK", "WORLD_SIZE", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT")}
    out = subprocess.run([sys.executable, str(root / "bench.py"), "--gpus", "2", "--steps", "3", "--selftest-launcher"],
                         capture_output=True, text=True, timeout=300, env=env, cwd=str(root))
    assert out.returncode == 0, out.stderr[-2000:]
    lines = [json.loads(ln) for ln in out.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, out.stdout                      # rank 0 alone prints
    rec = lines[0]
    assert rec["n_gpus"] == 2 and rec["ms"] == 20.0 and rec["units"] == 6000.0
    assert rec["value"] == 6000.0 / 20e-3 and rec["seed_of_last_rank"] == 2
    # a WORLD_SIZE that contradicts --gpus is refused instead of silently timing one GPU
    env2 = dict(env, WORLD_SIZE="1", RANK="0", LOCAL_RANK="0")
    bad = subprocess.run([sys.executable, str(root / "bench.py"), "--gpus", "2", "--selftest-launcher"],
                         capture_output=True, text=True, timeout=120, env=env2, cwd=str(root))
    assert bad.returncode != 0 and "WORLD_SIZE" in (bad.stderr + bad.stdout)
