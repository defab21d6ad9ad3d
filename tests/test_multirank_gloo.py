"""N > 1 host logic on CPU: the path has no cross-GPU exchange ("replicas only"), so
the only multi-rank code is bench.py's timing reduction (max over ranks) and the aggregation of the replicas'
rates.  Two gloo ranks on 127.0.0.1 exercise exactly those functions, plus the per-rank input seeding."""
import os
import socket

import numpy as np
import torch
import torch.distributed as td
import torch.multiprocessing as mp


def _free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank: int, world: int, port: int, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    td.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import bench
        from workloads import gen, get_workload, scaled

        local_ms = 10.0 + 5.0 * rank                      # rank 1 is the slow one
        td.barrier()
        slowest = bench.max_over_ranks(local_ms)
        w = scaled(get_workload("tiny"), T=64)
        h = gen.hidden_all(w, rank, "cpu")                 # bench.py seeds each replica's hidden states with its rank
        h_again = gen.hidden_all(w, rank, "cpu")
        digest = torch.tensor([float(h.float().sum())], dtype=torch.float64)
        gathered = [torch.zeros_like(digest) for _ in range(world)]
        td.all_gather(gathered, digest)
        out.put((rank, slowest, bench.replica_value(w.T, world, slowest), bool(torch.equal(h, h_again)),
                 [float(g.item()) for g in gathered]))
    finally:
        td.destroy_process_group()


def test_replica_timing_and_aggregation_world2():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, out)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, slowest, value, reproducible, digests in res:
        assert slowest == 15.0                              # max over ranks, seen by every rank
        assert np.isclose(value, 2 * 64 / 15.0e-3)          # whole-job rate = units of all ranks / slowest rank's time
        assert reproducible                                 # same (workload, rank) -> same bytes
        assert digests[0] != digests[1]                     # replicas work on different inputs
    assert res[0][4] == res[1][4]
