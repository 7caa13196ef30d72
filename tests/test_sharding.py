"""Host-side multi-rank logic on CPU: gloo, world_size 2 (no GPU, no data-path
collective: only the final gather).  SURVEY.md section 8(e)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2404_07780_b200.sharding import gather_results, shard_galaxies


def test_shard_is_a_balanced_partition():
    rng = np.random.default_rng(0)
    sides = rng.choice([64, 96, 128, 192, 256], size=8289)
    px = sides.astype(np.int64) ** 2
    for world in (1, 2, 4, 8):
        shards = shard_galaxies(px, world)
        allidx = np.concatenate(shards)
        assert len(allidx) == len(px) and np.array_equal(np.sort(allidx), np.arange(len(px)))
        loads = np.array([px[s].sum() for s in shards])
        assert loads.max() - loads.min() <= 256 * 256          # within one largest galaxy
        assert all(np.all(np.diff(s) > 0) for s in shards)
    eq = shard_galaxies([128 * 128] * 10, 4)
    assert sorted(len(s) for s in eq) == [2, 2, 3, 3]


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n_total, P, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        px = (np.arange(n_total) % 3 + 1) * 1000
        mine = shard_galaxies(px, world)[rank]
        # stand-in for gm_fit on this rank's shard: a value that encodes the galaxy index
        params = torch.tensor(mine, dtype=torch.float32)[:, None] * 10 + torch.arange(P, dtype=torch.float32)
        chi2 = torch.tensor(mine, dtype=torch.float32) + 0.5
        full_p, full_c = gather_results(mine, params, chi2, n_total)
        if rank == 0:
            out.put((full_p.numpy(), full_c.numpy()))
        dist.barrier()
    finally:
        dist.destroy_process_group()


@pytest.mark.timeout(120)
def test_gather_world_size_2_gloo():
    world, n_total, P = 2, 11, 7
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n_total, P, q)) for r in range(world)]
    for p in procs:
        p.start()
    full_p, full_c = q.get(timeout=90)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    g = np.arange(n_total, dtype=np.float32)
    assert np.array_equal(full_c, g + 0.5)
    assert np.array_equal(full_p, g[:, None] * 10 + np.arange(P, dtype=np.float32))
