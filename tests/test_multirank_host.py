"""World-size-2 gloo test (CPU) of the multi-GPU host logic: the curve partition and the max-over-ranks
timing.  The generator's per-curve results depend on the absolute curve number only, so the union of the ranks'
outputs must equal the single-rank output; checked here with the oracle standing in for the device library
(the oracle may be used by tests; the product path never imports it)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1909_06374_b200 import multirank, workloads


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, B_total, N, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle
    cfg = workloads.tiny(N=N, B=B_total)
    curve0, b_local = multirank.partition_curves(B_total, rank, world)
    rows = [oracle.erdf_sample_sorted(cfg["erdf"][0], cfg["grid_points"], N, cfg["seed"], curve0 + i, 1)[0]
            for i in range(b_local)]
    local = torch.from_numpy(np.stack(rows)) if rows else torch.empty((0, N), dtype=torch.float64)
    # gather variable-sized shards through a padded all_gather
    pad = torch.zeros((B_total, N), dtype=torch.float64)
    pad[:b_local] = local
    bufs = [torch.zeros_like(pad) for _ in range(world)]
    dist.all_gather(bufs, pad)
    counts = [multirank.partition_curves(B_total, r, world)[1] for r in range(world)]
    full = torch.cat([bufs[r][:counts[r]] for r in range(world)])
    tmax = multirank.max_over_ranks(10.0 + rank, dist=dist)
    if rank == 0:
        q.put((full.numpy(), tmax))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("B_total", [4, 5])
def test_partition_union_equals_single_rank(B_total):
    import oracle
    N, world = 256, 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, B_total, N, q)) for r in range(world)]
    for p in procs:
        p.start()
    full, tmax = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    cfg = workloads.tiny(N=N, B=B_total)
    ref = np.stack([oracle.erdf_sample_sorted(cfg["erdf"][0], cfg["grid_points"], N, cfg["seed"], b, 1)[0]
                    for b in range(B_total)])
    assert (full == ref).all()
    assert tmax == 11.0          # the slowest rank's time


def test_partition_covers_every_curve_once():
    for B_total in (1, 4, 7, 4096):
        for world in (1, 2, 3, 8):
            seen = []
            for r in range(world):
                c0, bl = multirank.partition_curves(B_total, r, world)
                seen += list(range(c0, c0 + bl))
            assert seen == list(range(B_total))
    assert multirank.weak_curve0(4, 3) == 12
    assert multirank.max_over_ranks(3.5) == 3.5
