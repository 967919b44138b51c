"""N > 1 path of bench.py on CPU: two gloo ranks compute their row assignments; within a step the ranks work on
disjoint rows and, over the steps, the replicas sweep the whole batch (replicas only: no data-path collective)."""
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench

    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    B, rows, steps = 729, 8, 50
    mine = torch.tensor(np.stack([bench.rows_for_step(B, rows, world, rank, i) for i in range(steps)]))
    gathered = [torch.zeros_like(mine) for _ in range(world)]
    dist.all_gather(gathered, mine)
    ms = torch.tensor([10.0 + rank], dtype=torch.float64)      # the timing reduction bench.py uses: max over ranks
    dist.all_reduce(ms, op=dist.ReduceOp.MAX)
    if rank == 0:
        out.put((torch.stack(gathered).numpy(), float(ms.item())))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_row_assignment():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    allrows, ms = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert ms == 11.0
    assert allrows.shape == (2, 50, 8)
    for i in range(50):
        assert len(set(allrows[0, i]) & set(allrows[1, i])) == 0            # disjoint within a step
    assert len(np.unique(allrows)) == 729                                    # the sweep is covered
