"""Worker of tests/test_gpu_multi.py, launched by `python -m torch.distributed.run`: one rank per
GPU over NCCL.  Every rank searches its contiguous shard of the templates on its own GPU (no
data-path collective), the 20-byte results are gathered once, and rank 0 checks them against the
unsharded search on its GPU and against the oracle.  Exit code 0 = all good."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def main() -> int:
    import paper_1805_05652_b200 as pkg
    from synth import Grid, tiny_workload

    rank, local, world = (int(os.environ[k]) for k in ("RANK", "LOCAL_RANK", "WORLD_SIZE"))
    torch.cuda.set_device(local)
    dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    try:
        grid = Grid(0, 1800, 23, 3600, 3600, 140)
        T = 2 * world + 3  # uneven shards
        wl = tiny_workload(801, 350, 0.1, grid, n_templates=T, phi_random=True)
        t = torch.from_numpy(wl.data.t).cuda()
        lo, cnt = pkg.template_shard(T, rank, world)
        for window in (pkg.EXP, pkg.RECT):
            if cnt:
                a = torch.from_numpy(wl.data.atoms[lo:lo + cnt]).cuda()
                raw = pkg.tfstat_search(a, t, window, grid).raw
            else:
                raw = torch.zeros((0, 5), dtype=torch.int32, device="cuda")
            got = pkg.gather_results(raw, T, dst=0)
            if rank == 0:
                full = pkg.tfstat_search(torch.from_numpy(wl.data.atoms).cuda(), t, window,
                                         grid).numpy()
                if window == pkg.RECT:
                    assert np.array_equal(got, full), "sharded != unsharded (rect)"
                else:  # two templates per CTA share a re-sum guard: last bits may differ
                    assert np.array_equal(got["n_valid"], full["n_valid"])
                    assert np.allclose(got["max2F"], full["max2F"], rtol=1e-4, atol=1e-4)
                    assert np.allclose(got["logB"], full["logB"], rtol=1e-4, atol=1e-4)
                import oracle
                from tests.parity import check_result

                for k in range(T):
                    ref = oracle.map2F(wl.data.atoms[k], wl.data.t, window, grid)
                    check_result(got[k], ref["twoF"], ref["flags"], grid.N_tau, f"w{window} tpl{k}")
        dist.barrier()
    finally:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
