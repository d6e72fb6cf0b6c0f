"""N>1 path of bench.py on CPU (gloo, world_size 2): reactors are independent, so the multi-GPU run shards by
giving every rank its own batch and only reduces the TIMING (max over ranks) -- no collective on the data path."""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close()
    return p


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    from synth_inputs import make_config
    mech, y, p, _ = make_config("C2", n=512)
    ys, ps = bench.shard_states(y, p, rank)
    t = bench.max_over_ranks(10.0 + rank, dist)          # rank 1 is the slow one
    cols = torch.tensor(ys[:, :4].copy())
    gathered = [torch.zeros_like(cols) for _ in range(world)]
    dist.all_gather(gathered, cols)                       # test-only exchange, to compare the shards
    if rank == 0:
        torch.save(dict(t=t, g=[g.numpy() for g in gathered], y=y[:, :4].copy(), n=ys.shape[1],
                        ssum=float(np.sort(ys[0]).sum()), ysum=float(np.sort(y[0]).sum())), out)
    dist.destroy_process_group()


def test_weak_scaling_shards_and_max_timing(tmp_path):
    out = str(tmp_path / "r0.pt")
    mp.spawn(_worker, args=(2, _free_port(), out), nprocs=2, join=True)
    r = torch.load(out, weights_only=False)
    assert r["t"] == 11.0                                 # max over ranks, as the bench contract asks
    assert r["n"] == 512                                  # fixed work per rank (weak scaling)
    assert np.array_equal(r["g"][0], r["y"])              # rank 0 keeps the recipe order
    assert not np.array_equal(r["g"][1], r["y"])          # rank 1 holds a different column order ...
    assert abs(r["ssum"] - r["ysum"]) < 1e-9              # ... of the same states


def test_single_process_needs_no_process_group():
    import bench
    assert bench.max_over_ranks(3.5, None) == 3.5
