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


def _slab_worker(rank, world, port, q):
    import os
    import torch
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        from paper_2005_14454_b200 import binding as ah
        nfield, plane = ah.AH_NHALO, 5
        # plane lists as SlabSimulation.halo_planes() returns them: send_lo, send_hi, recv_lo, recv_hi; the value of
        # an element names (rank, which boundary, field)
        planes = [[torch.full((plane,), 1000.0 * rank + 100.0 * side + a) for a in range(nfield)] for side in (1, 2)]
        planes += [[torch.full((plane,), -1.0) for _ in range(nfield)] for _ in range(2)]
        ops = []
        for a in range(nfield):
            for kind, which, peer in ah.halo_schedule(rank, world):
                ops.append(dist.P2POp(dist.isend if kind == "send" else dist.irecv, planes[which][a], peer))
        for r in dist.batch_isend_irecv(ops):
            r.wait()
        lo, hi = (rank - 1) % world, (rank + 1) % world
        ok = all(float(planes[2][a][0]) == 1000.0 * lo + 200.0 + a and      # ghost below = lower neighbour's LAST own plane
                 float(planes[3][a][0]) == 1000.0 * hi + 100.0 + a          # ghost above = upper neighbour's FIRST own plane
                 for a in range(nfield))
        # read-outs: counts and sums add, the last sum is a maximum
        counts, sums = [rank + 1] * ah.AH_NDIAG_INT, [0.5 * (rank + 1)] * ah.AH_NDIAG_FLT
        add = torch.tensor([float(c) for c in counts] + sums[:-1], dtype=torch.float64)
        mx = torch.tensor([sums[-1]], dtype=torch.float64)
        dist.all_reduce(add, op=dist.ReduceOp.SUM)
        dist.all_reduce(mx, op=dist.ReduceOp.MAX)
        tot = world * (world + 1) / 2
        ok = ok and add[:ah.AH_NDIAG_INT].tolist() == [tot] * ah.AH_NDIAG_INT and float(mx) == 0.5 * world
        q.put((rank, ok))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 3])
def test_slab_exchange_schedule_over_gloo(world):
    """Host logic of the z-slab exchange (binding.halo_schedule, the schedule DistributedSlab posts over NCCL): run
    with CPU tensors over gloo, every rank must end up with its neighbours' boundary planes in its ghost planes, for
    2 ranks (both neighbours are the same peer) and 3."""
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_slab_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
    assert res == [(r, True) for r in range(world)]


def test_slab_partition_and_schedule_host_logic():
    from paper_2005_14454_b200 import binding as ah
    for nz, n in ((25, 3), (1024, 8), (7, 7), (10, 1)):
        parts = [ah.slab_planes(nz, n, r) for r in range(n)]
        assert parts[0][0] == 0 and sum(p[1] for p in parts) == nz
        assert all(parts[r][0] + parts[r][1] == parts[r + 1][0] for r in range(n - 1))
        assert max(p[1] for p in parts) - min(p[1] for p in parts) <= 1
    with pytest.raises(ValueError):
        ah.slab_planes(4, 5, 0)
    assert ah.halo_schedule(0, 1) == [("send", 0, 0), ("recv", 3, 0), ("send", 1, 0), ("recv", 2, 0)]
    nf = ah.AH_NDIAG_FLT - 1
    assert ah.combine_partials([([1] * 5, [1.0] * nf + [3.0]), ([2] * 5, [0.5] * nf + [7.0])]) == ([3] * 5, [1.5] * nf + [7.0])
