"""World-size-2 CPU test (gloo) of the N>1 host logic: contiguous template shards, per-rank
template-id offsets, max-over-ranks timing and candidate concatenation.  The per-rank "search" is
the CPU oracle here (no GPU in this test); on the GPU box the same plumbing wraps the CUDA path."""
import os
import socket

import numpy as np
import pytest
import torch.multiprocessing as mp

CAND = np.dtype([("template_id", "<u4"), ("fold", "<u4"), ("bin", "<u4"), ("power", "<f4"), ("sigma", "<f4"),
                 ("pad", "<u4")])


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _to_array(cands):
    out = np.zeros(len(cands), dtype=CAND)
    for i, c in enumerate(cands):
        out[i] = (c[0], c[1], c[2], c[3], c[4], 0)
    return out


def _worker(rank, world, port, q):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from oracle import tb_oracle as orc
    from paper_2112_11991_b200 import dist as tbd, workloads
    wl = workloads.config1(n_templates=5)
    first, count = tbd.shard_templates(len(wl.templates), rank, world)
    mine = orc.search(wl.series, wl.tsamp, wl.templates[first:first + count], first_template_id=first,
                      sigma_threshold=4.5)
    merged = tbd.gather_candidates(_to_array(mine))
    slowest = tbd.max_over_ranks(10.0 + rank)
    if rank == 0:
        q.put((merged.tobytes(), slowest, first, count))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_sharded_search_equals_single_process():
    from oracle import tb_oracle as orc
    from paper_2112_11991_b200 import workloads
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    raw, slowest, first, count = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    wl = workloads.config1(n_templates=5)
    ref = _to_array(orc.search(wl.series, wl.tsamp, wl.templates, sigma_threshold=4.5))
    merged = np.frombuffer(raw, dtype=CAND)
    assert len(ref) > 0 and np.array_equal(merged, ref)
    assert slowest == 11.0 and (first, count) == (0, 3)
