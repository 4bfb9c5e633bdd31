"""The N > 1 path on CPU: templates sharded over world_size-2 `gloo` ranks, no data-path
collective, one gather of the 20-byte results.

On the CPU box there is no CUDA path, so each rank fills its shard's results with the ORACLE
(tests may call it); what is under test is the host logic of paper_1805_05652_b200/shard.py:
shard boundaries (uneven and empty shards), padding, template order after the gather.
"""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1805_05652_b200.binding import RESULT_DTYPE
from paper_1805_05652_b200.shard import gather_results, template_shard
from synth import Grid, TSFT, tiny_workload


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def test_template_shard_partitions_exactly():
    for T in (0, 1, 2, 5, 41, 4096, 4097):
        for world in (1, 2, 3, 8):
            spans = [template_shard(T, r, world) for r in range(world)]
            assert spans[0][0] == 0
            for (s0, c0), (s1, _) in zip(spans, spans[1:]):
                assert s1 == s0 + c0  # contiguous, in rank order
            assert sum(c for _, c in spans) == T
            counts = [c for _, c in spans]
            assert max(counts) - min(counts) <= 1
    with pytest.raises(ValueError):
        template_shard(4, 2, 2)


def _oracle_raw(wl, lo, cnt, window):
    import oracle

    out = np.zeros(cnt, dtype=RESULT_DTYPE)
    if cnt:
        res, _ = oracle.search(wl.data.atoms[lo:lo + cnt], wl.data.t, window, wl.grid)
        for i, r in enumerate(res):
            out[i] = (r.max2F, r.m, r.n, r.logB, r.n_valid)
    return torch.from_numpy(out.view(np.int32).reshape(cnt, 5).copy())


def _worker(rank, world, port, T, window, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        wl = tiny_workload(77, 60, 0.2, Grid(0, TSFT, 9, 2 * TSFT, TSFT, 11), n_templates=T,
                           phi_random=True)
        lo, cnt = template_shard(T, rank, world)
        local = _oracle_raw(wl, lo, cnt, window)
        everyone = gather_results(local, T)            # all_gather flavour
        only0 = gather_results(local, T, dst=0)        # gather-to-root flavour
        assert (only0 is None) == (rank != 0)
        if rank == 0:
            assert np.array_equal(everyone.view(np.int32), only0.view(np.int32))
        q.put((rank, everyone.view(np.int32).reshape(-1, 5).copy()))
        dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("T", [5, 1])  # uneven shards; one rank with an empty shard
def test_sharded_search_equals_unsharded_gloo_world2(T):
    window = 1  # exponential
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, T, window, q))
             for r in range(world)]
    for p in procs:
        p.start()
    got = dict(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    wl = tiny_workload(77, 60, 0.2, Grid(0, TSFT, 9, 2 * TSFT, TSFT, 11), n_templates=T,
                       phi_random=True)
    full = _oracle_raw(wl, 0, T, window).numpy()
    for r in range(world):
        assert np.array_equal(got[r], full), f"rank {r}: gathered results differ from unsharded"
