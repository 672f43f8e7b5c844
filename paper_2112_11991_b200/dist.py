"""Host-side plumbing for N > 1 ranks (one process per GPU).  The path shards over templates
(Alg. 1: every template is independent) and has no exchange step, so there is no
data-path collective: torch.distributed is used only to agree on timings and to concatenate the
per-rank candidate lists.  Works with backend "nccl" (cuda tensors) and "gloo" (cpu tensors)."""
from __future__ import annotations

import numpy as np
import torch
import torch.distributed as dist

from .workloads import shard_templates  # noqa: F401  (re-exported)


def world():
    if dist.is_available() and dist.is_initialized():
        return dist.get_rank(), dist.get_world_size()
    return 0, 1


def max_over_ranks(value: float, device="cpu") -> float:
    if world()[1] == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def gather_candidates(cands: np.ndarray, device="cpu") -> np.ndarray:
    """Concatenate every rank's candidate array (structured, 24-byte rows) on every rank, in
    rank order; shards are contiguous in template id, so the result stays sorted."""
    rank, n = world()
    if n == 1:
        return cands
    raw = torch.from_numpy(np.ascontiguousarray(cands).view(np.uint8).reshape(-1).copy()).to(device)
    sizes = [torch.zeros(1, dtype=torch.int64, device=device) for _ in range(n)]
    dist.all_gather(sizes, torch.tensor([raw.numel()], dtype=torch.int64, device=device))
    m = int(max(int(s.item()) for s in sizes))
    buf = torch.zeros(m, dtype=torch.uint8, device=device)
    buf[: raw.numel()] = raw
    bufs = [torch.zeros(m, dtype=torch.uint8, device=device) for _ in range(n)]
    dist.all_gather(bufs, buf)
    parts = [b[: int(s.item())].cpu().numpy().view(cands.dtype) for b, s in zip(bufs, sizes)]
    return np.concatenate(parts)
