"""N>1 path on CPU: world-size-2 gloo processes partition the batch entries.

The path shards by batch entry only (no data-path collective): what has to be right on the host is
that ranks own disjoint entries with the documented seeds, that rank 0 reproduces the single-GPU
workload, and that the max-over-ranks timing reduction of bench.py works.  No GPU, no oracle compute.
"""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from workloads import make_config, shard_for_rank


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        w = shard_for_rank(make_config(3, n=(16, 16, 24), batch=4, steps=8), 3, rank, world)
        seeds = torch.tensor(w.seeds, dtype=torch.int64)
        gathered = [torch.zeros_like(seeds) for _ in range(world)]
        dist.all_gather(gathered, seeds)
        # digest of this rank's atom lists, gathered so rank 0 can check the ranks differ
        digest = torch.tensor([float(np.sum(a[:, :3])) for a in w.atoms], dtype=torch.float64)
        dg = [torch.zeros_like(digest) for _ in range(world)]
        dist.all_gather(dg, digest)
        # bench.py's timing reduction: max over ranks
        t = torch.tensor([10.0 + rank], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        # whole-job units = sum over ranks of per-rank units
        units = torch.tensor([float(w.cells) * w.batch * w.steps], dtype=torch.float64)
        dist.all_reduce(units, op=dist.ReduceOp.SUM)
        dist.barrier()
        if rank == 0:
            q.put(dict(seeds=[g.tolist() for g in gathered], digests=[d.tolist() for d in dg],
                       tmax=float(t.item()), units=float(units.item()), batch=w.batch, cells=w.cells, steps=w.steps))
    finally:
        dist.destroy_process_group()


def test_world_size_2_gloo_partition_of_batch_entries():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    out = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert out["seeds"] == [[3000, 3001, 3002, 3003], [3004, 3005, 3006, 3007]]      # disjoint, contiguous
    flat = [d for r in out["digests"] for d in r]
    assert len(set(round(x, 9) for x in flat)) == len(flat)                          # all entries differ
    assert out["tmax"] == 11.0
    assert out["units"] == world * out["cells"] * out["batch"] * out["steps"]


def test_rank0_reproduces_the_single_gpu_workload_and_ranks_follow_the_seed_rule():
    for idx in (0, 1, 2, 3, 4):
        kw = dict(n=(16, 16, 24), batch=3, steps=4)
        w = make_config(idx, **kw)
        w0 = shard_for_rank(w, idx, 0, 4)
        assert all(np.array_equal(a, b) for a, b in zip(w.atoms, w0.atoms))
        w2 = shard_for_rank(w, idx, 2, 4)
        assert w2.batch == w.batch and len(w2.atoms) == w.batch
        if idx == 3:
            assert w2.seeds == [3006, 3007, 3008]
            # a rank's entry equals the same global entry generated in one big batch
            big = make_config(3, n=(16, 16, 24), batch=9, steps=4)
            assert np.array_equal(w2.atoms[1], big.atoms[7])
        if idx in (0, 1):
            assert all(np.array_equal(a, b) for a, b in zip(w.atoms, w2.atoms))   # replicas only
