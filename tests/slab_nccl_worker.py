"""Worker of tests/test_gpu_slabs.py::test_distributed_slab_two_ranks_over_nccl (one process per GPU, started by
torch.distributed.run): ONE lattice in world_size z slabs, boundary planes over NCCL point-to-point calls, against the
single lattice on rank 0, bit for bit.  Needs >= 2 GPUs: it has NOT been executed on this project's 1-GPU pool."""
import os
import sys
from pathlib import Path

import numpy as np
import torch
import torch.distributed as dist

sys.path.insert(0, str(Path(__file__).resolve().parent.parent))


def main():
    rank, local, world = int(os.environ["RANK"]), int(os.environ["LOCAL_RANK"]), int(os.environ["WORLD_SIZE"])
    torch.cuda.set_device(local)
    dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    from paper_2005_14454_b200 import binding as ah
    nx, ny, nz = 128, 9, 8 * world + 3            # unequal slabs
    P = ah.make_params(nx, ny, nz, p=1.0, s=1.0, tau_ref=3.0)
    ds = ah.DistributedSlab(P, dist, device=f"cuda:{local}")
    ds.slab.init_fields(2)
    recs = ds.step(6, 1.0, 0.1, diag_every=3)
    torch.cuda.synchronize()
    own = torch.from_numpy(np.ascontiguousarray(ds.slab.get_fields()[:, 1:-1])).cuda()      # (10, nz_own, ny, nx)
    sizes = [ah.slab_planes(nz, world, r)[1] for r in range(world)]
    parts = [torch.empty((10, n, ny, nx), dtype=own.dtype, device=own.device) for n in sizes]
    for r in range(world):                        # unequal shapes: one broadcast per slab
        if r == rank:
            parts[r].copy_(own)
        dist.broadcast(parts[r], src=r)
    ok = True
    if rank == 0:
        one = ah.Simulation(params=P, device=f"cuda:{local}")
        one.init_fields(2)
        want_recs = one.step_diag(6, 1.0, 0.1, 3)
        want = one.get_fields()
        got = torch.cat(parts, dim=1).cpu().numpy()
        ok = bool(np.array_equal(got, want))
        ok = ok and [a["n_wind"] for a in want_recs] == [b["n_wind"] for b in recs]
        ok = ok and all(abs(b["sum_L"] - a["sum_L"]) <= 1e-11 * abs(a["sum_L"]) for a, b in zip(want_recs, recs))
        one.close()
        print("SLAB_NCCL_OK" if ok else "SLAB_NCCL_MISMATCH", flush=True)
    ds.slab.close()
    dist.destroy_process_group()
    return 0 if ok else 1


if __name__ == "__main__":
    sys.exit(main())
