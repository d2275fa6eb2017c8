"""world_size-2 CPU (gloo) cover of the N>1 path of bench.py: per-rank seeds, unit partition, barrier and
MAX-over-ranks timing, whole-job aggregation.  No GPU, no data-path collective (the path has none)."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2507_16697_b200 import multirank, workloads as wl


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        cfg = multirank.rank_config(wl.CONFIGS["C1"], rank)
        q = wl.make_tensor(cfg, "q")
        # every rank reports its first input values; rank 0 gathers to check that batches differ
        head = q.flatten()[:8].clone()
        gathered = [torch.zeros_like(head) for _ in range(world)]
        dist.all_gather(gathered, head)
        dist.barrier()
        ms = multirank.max_over_ranks(10.0 + 5.0 * rank, dist)          # slowest rank = 10 + 5*(world-1)
        units = list(multirank.shard_units(33, world, rank))
        counts = torch.tensor([len(units)], dtype=torch.int64)
        dist.all_reduce(counts)
        if rank == 0:
            out.put({"ms": ms, "total_units": int(counts.item()), "units0": units,
                     "distinct": not torch.equal(gathered[0], gathered[1]),
                     "value": multirank.aggregate_tflops(world, 1e12, ms)})
    finally:
        dist.destroy_process_group()


def test_two_ranks_gloo():
    world = 2
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    res = out.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res["ms"] == 15.0                       # MAX over ranks, not rank 0's own 10.0
    assert res["total_units"] == 33 and res["units0"] == list(range(17))
    assert res["distinct"]
    assert res["value"] == pytest.approx(2 * 1e12 / 15e-3 / 1e12)


def test_shard_units_partitions_exactly():
    for n in (1, 7, 16, 33, 128):
        for world in (1, 2, 3, 8):
            seen = []
            for r in range(world):
                seen += list(multirank.shard_units(n, world, r))
            assert seen == list(range(n))
            sizes = [len(multirank.shard_units(n, world, r)) for r in range(world)]
            assert max(sizes) - min(sizes) <= 1


def test_single_process_passthrough():
    assert multirank.max_over_ranks(3.5) == 3.5
    assert multirank.rank_config(wl.CONFIGS["C3"], 0).seed == wl.CONFIGS["C3"].seed
    assert multirank.rank_config(wl.CONFIGS["C3"], 3).seed == wl.CONFIGS["C3"].seed + 3000
