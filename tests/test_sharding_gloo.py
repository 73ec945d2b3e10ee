"""N > 1 path on CPU (world_size 2, gloo): the path shards by realization word with no
collective in the loop.  Each rank simulates its own words with the
oracle (first realization = rank * R_per_rank, the same rule bench.py uses for the CUDA
handles), the results are gathered, and the union must equal one process simulating all
words -- which is what makes per-rank CUDA handles with first_realization = shard offset a
correct multi-GPU run.  Also checks the max-over-ranks timing reduction bench.py uses.
"""
import os
import socket
import sys

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); p = s.getsockname()[1]; s.close(); return p


def _worker(rank, world, port, out_dir):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import bench
    from ea_inputs import temperature_ladder
    from oracle import Oracle
    L, nT, R_per_rank = 4, 6, 64
    betas = 1.0 / temperature_ladder(nT, 0.6, 2.0)
    r0 = bench.shard_first_realization(rank, R_per_rank)
    o = Oracle(L, nT, R_per_rank, betas, 11, r0=r0)
    o.sweep(25, 1)
    E = torch.from_numpy(o.energy().astype(np.int32))
    gathered = [torch.zeros_like(E) for _ in range(world)]
    dist.all_gather(gathered, E)
    t = bench.max_over_ranks(10.0 + rank, world, device="cpu")
    if rank == 0:
        np.save(os.path.join(out_dir, "E.npy"), torch.cat(gathered).numpy())
        np.save(os.path.join(out_dir, "t.npy"), np.array([t]))
    dist.destroy_process_group()


def test_two_rank_sharding_matches_single_process(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    sys.path.insert(0, ROOT)
    from ea_inputs import temperature_ladder
    from oracle import Oracle
    betas = 1.0 / temperature_ladder(6, 0.6, 2.0)
    full = Oracle(4, 6, 128, betas, 11)
    full.sweep(25, 1)
    assert (np.load(tmp_path / "E.npy") == full.energy()).all()
    assert np.load(tmp_path / "t.npy")[0] == 11.0       # max over ranks
