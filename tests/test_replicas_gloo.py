"""N > 1 path on CPU (gloo, world_size 2): the path does not shard ("replicas only"), so the
only collective in bench.py is the report: value = pairs processed by all ranks / max-over-ranks time."""
import os
import socket
import sys
from pathlib import Path

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = Path(__file__).resolve().parents[1]


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    sys.path.insert(0, str(ROOT))
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # rank r "processed" (r + 1) * 1000 pairs in (r + 1) * 2 ms
    pairs, ms = bench.aggregate(dist, torch, (rank + 1) * 1000.0, (rank + 1) * 2.0, torch.device("cpu"))
    dist.barrier()
    if rank == 0:
        Path(out).write_text(f"{pairs} {ms}")
    dist.destroy_process_group()


def test_replica_aggregation_world2(tmp_path):
    out = tmp_path / "agg.txt"
    mp.spawn(_worker, args=(2, _free_port(), str(out)), nprocs=2, join=True)
    pairs, ms = map(float, out.read_text().split())
    assert pairs == 3000.0      # sum over ranks
    assert ms == 4.0            # max over ranks


def test_single_process_passthrough():
    sys.path.insert(0, str(ROOT))
    import bench
    assert bench.aggregate(None, torch, 5.0, 7.0, torch.device("cpu")) == (5.0, 7.0)
