"""Template sharding over GPUs ("trivially further parallelise ...
splitting the (f, fdot) space over multiple GPUs").

Templates are independent, so the path shards with NO data-path collective: rank r searches the
contiguous template range `template_shard(T, r, world)` on its own GPU.  The only exchange is
the gather of the per-template results (20 bytes each), done once after the search.  This
module is host logic only (no arithmetic of the method) and works with any torch.distributed
backend (`nccl` on GPUs, `gloo` in the CPU tests).
"""
from __future__ import annotations

from typing import Optional, Tuple

import numpy as np
import torch

from .binding import RESULT_DTYPE


def template_shard(n_templates: int, rank: int, world: int) -> Tuple[int, int]:
    """(first template, count) of rank `rank`: contiguous, sizes differ by at most one, the
    first `n_templates % world` ranks take the extra template.  Ranks beyond the number of
    templates get an empty shard."""
    if n_templates < 0 or world < 1 or not (0 <= rank < world):
        raise ValueError("template_shard: need n_templates >= 0 and 0 <= rank < world")
    base, extra = divmod(n_templates, world)
    start = rank * base + min(rank, extra)
    return start, base + (1 if rank < extra else 0)


def gather_results(local_raw: torch.Tensor, n_templates: int, group=None,
                   dst: Optional[int] = None) -> Optional[np.ndarray]:
    """Collect the [count, 5] int32 images of tfstat_result from every rank into one
    RESULT_DTYPE array of length n_templates, in template order.

    `local_raw` is the `Results.raw` tensor of this rank's `tfstat_search` (any device).  With
    `dst=None` every rank gets the full array (all_gather); otherwise only rank `dst` does and
    the others return None.  Shards are padded to the largest shard for the collective and
    trimmed afterwards, so uneven and empty shards are fine."""
    import torch.distributed as dist

    world = dist.get_world_size(group)
    rank = dist.get_rank(group)
    start, count = template_shard(n_templates, rank, world)
    if local_raw.dim() != 2 or local_raw.shape[1] != 5 or local_raw.dtype != torch.int32:
        raise ValueError("gather_results: local_raw must be a [count, 5] int32 tensor")
    if local_raw.shape[0] != count:
        raise ValueError(f"gather_results: rank {rank} holds {local_raw.shape[0]} results, "
                         f"its shard has {count}")
    pad = max(template_shard(n_templates, r, world)[1] for r in range(world))
    buf = torch.zeros((max(pad, 1), 5), dtype=torch.int32, device=local_raw.device)
    buf[:count] = local_raw
    if dst is None:
        parts = [torch.empty_like(buf) for _ in range(world)]
        dist.all_gather(parts, buf, group=group)
    else:
        parts = [torch.empty_like(buf) for _ in range(world)] if rank == dst else None
        dist.gather(buf, parts, dst=dst, group=group)
        if rank != dst:
            return None
    out = np.empty(n_templates, dtype=RESULT_DTYPE)
    for r, p in enumerate(parts):
        s, c = template_shard(n_templates, r, world)
        if c:
            out[s:s + c] = p[:c].cpu().numpy().view(RESULT_DTYPE).reshape(-1)
    return out
