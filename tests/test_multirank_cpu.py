"""World-size-2 check (gloo, CPU) of the only multi-rank host logic there is: events are independent
(PAPER.md:L22, L233), so bench.py shards them by rank with no data-path collective and reduces the timing with
MAX over ranks.  The shards of two ranks must tile the single-rank draw exactly."""
import os
import socket
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, N, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    from types import SimpleNamespace
    args = SimpleNamespace(config=1)
    ev = bench.make_events(args, 6, N, rank)
    np.save(os.path.join(out_dir, f"mom{rank}.npy"), ev.mom)
    np.save(os.path.join(out_dir, f"col{rank}.npy"), ev.col)
    np.save(os.path.join(out_dir, f"hel{rank}.npy"), ev.hel)
    t = bench.max_over_ranks(10.0 + rank, world, torch.device("cpu"))
    assert t == 10.0 + world - 1
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_tile_the_workload(tmp_path):
    N, world = 257, 2
    mp.spawn(_worker, args=(world, _free_port(), N, str(tmp_path)), nprocs=world, join=True)
    from paper_2106_06507_b200 import workload as wl
    full = wl.config_events(1, N=world * N)
    for r in range(world):
        sl = slice(r * N, (r + 1) * N)
        assert np.array_equal(np.load(tmp_path / f"mom{r}.npy"), full.mom[sl])
        assert np.array_equal(np.load(tmp_path / f"col{r}.npy"), full.col[sl])
        assert np.array_equal(np.load(tmp_path / f"hel{r}.npy"), full.hel[sl])
