"""N>1 host logic on CPU: world_size 2 over gloo (127.0.0.1).  The path shards over systems with
no data-path collective: each rank draws ITS window of the seeded batch,
solves it alone (here with the oracle standing in for the device, the host logic is what is
tested) and the union of the shards must equal the single-process result bit for bit; the timing
reduction must be a MAX over ranks."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
import pent_inputs as pin
from paper_1807_07382_b200.sharding import max_over_ranks, shard_columns, whole_job_rate

N, M_TOTAL, SEED, SIGMA = 48, 101, 77, 2.5     # odd M: the shards are ragged


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank),
                      WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        col0, m = shard_columns(M_TOTAL, rank, world)
        f = pin.uniform_pm1(SEED, 0, N, m, col0, M_TOTAL)
        fac = oracle.factor(*pin.diagonals_I_plus_sigma_L2(N, SIGMA))   # replicated, no broadcast
        x = oracle.solve_batch(fac, f)
        np.save(os.path.join(out_dir, f"x{rank}.npy"), x)
        np.save(os.path.join(out_dir, f"f{rank}.npy"), f)
        dist.barrier()
        tmax = max_over_ranks(0.5 + rank)            # rank 1 is the slow one
        np.save(os.path.join(out_dir, f"t{rank}.npy"), np.array([tmax, col0, m]))
    finally:
        dist.destroy_process_group()


def test_shard_columns_partition():
    for M in (0, 1, 7, 64, 101):
        for world in (1, 2, 3, 8):
            blocks = [shard_columns(M, r, world) for r in range(world)]
            assert blocks[0][0] == 0
            for (c0, m0), (c1, _) in zip(blocks, blocks[1:]):
                assert c1 == c0 + m0
            assert blocks[-1][0] + blocks[-1][1] == M
            sizes = [m for _, m in blocks]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard_columns(4, 2, 2)


def test_world2_gloo_shards_equal_single_process(tmp_path):
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    f_full = pin.uniform_pm1(SEED, 0, N, M_TOTAL)
    x_full = oracle.solve_batch(oracle.factor(*pin.diagonals_I_plus_sigma_L2(N, SIGMA)), f_full)
    fs = [np.load(tmp_path / f"f{r}.npy") for r in range(world)]
    xs = [np.load(tmp_path / f"x{r}.npy") for r in range(world)]
    assert np.array_equal(np.concatenate(fs, axis=1), f_full)       # draws do not depend on the rank
    assert np.array_equal(np.concatenate(xs, axis=1), x_full)       # systems are independent
    ts = [np.load(tmp_path / f"t{r}.npy") for r in range(world)]
    assert ts[0][0] == ts[1][0] == 1.5                               # MAX over ranks, on every rank
    assert int(ts[0][2]) + int(ts[1][2]) == M_TOTAL and int(ts[1][1]) == int(ts[0][2])
    assert whole_job_rate(1000, world, 2.0) == 1000.0


def test_max_over_ranks_without_process_group():
    assert max_over_ranks(0.25) == 0.25
