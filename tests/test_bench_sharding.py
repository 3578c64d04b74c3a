"""bench.py's N > 1 path on CPU (gloo, world size 2): ranks take disjoint blocks of the record and the step time is the
max over ranks (time shards, no data-path collective)."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def _worker(rank, world, port, out):
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    ids = bench.rank_block_ids(rank, n_blocks=5)
    t = torch.tensor([10.0 + 7.0 * rank, 3.0 - rank], dtype=torch.float64)
    t = bench.max_over_ranks(t, world)
    gathered = [None] * world
    dist.all_gather_object(gathered, ids)
    if rank == 0:
        out.put((gathered, t.tolist()))
    dist.destroy_process_group()


def test_two_ranks_take_disjoint_blocks_and_report_the_max_time():
    import bench
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() % 1000)
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    gathered, t = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert len(set(gathered[0]) & set(gathered[1])) == 0 and len(gathered[0]) == len(gathered[1]) == 5
    assert t == [17.0, 3.0]
    n_win, n_raw = bench.block_geometry(4096)
    assert n_win == 4096 * 16 and n_raw % 128 == 0
    # the last window of the last slide ends inside the whitened block
    m0 = bench.PSD_LEN - bench.STRIDE - bench.FILTER // 2
    assert m0 + (n_win - 1) * 128 + 8 * 2048 + 3072 + 1024 <= n_raw
