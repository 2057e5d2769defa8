"""Multi-process (gloo, world_size 2) test of the N > 1 path's host logic: contiguous pixel shards keyed by global
pixel id + the final gather reproduce the single-process inversion bit for bit (reading G0).

No GPU here, so the per-rank engine is the CPU oracle's GA (tests may use oracle/); the sharding layer under test,
paper_1208_0302_b200.sharding, is the one bench.py / a user drives `binding.ga_invert` with on the GPU box.
"""
import os
import socket
import sys

import numpy as np
import pytest

from paper_1208_0302_b200 import sharding as S

torch = pytest.importorskip("torch")


def test_pixel_shard_partitions():
    for n in (0, 1, 2, 7, 64, 65, 4194304, 3141529):
        for world in (1, 2, 3, 8):
            pos = 0
            for r in range(world):
                s, c = S.pixel_shard(n, r, world)
                assert s == pos and c >= 0
                pos += c
            assert pos == n
            counts = S.shard_counts(n, world)
            assert max(counts) - min(counts) <= 1
    with pytest.raises(ValueError):
        S.pixel_shard(10, 2, 2)
    with pytest.raises(ValueError):
        S.pixel_shard(-1, 0, 1)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, n_pixels, q):
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    for p in (root, os.path.join(root, "tests")):
        if p not in sys.path:
            sys.path.insert(0, p)
    import torch.distributed as dist
    from helpers import make_obs
    from oracle import api as orc
    from paper_1208_0302_b200 import workloads as W
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        c0 = W.config0()
        ga = W.ga_config(16, 6)
        mu = np.linspace(0.4, 1.0, n_pixels)
        truth, obs, ln = make_obs(c0, n_pixels, mu=mu, threads=1)

        def engine(obs_local, pixel_id_base=0, mu=None):
            r = orc.ga_invert(obs_local, c0["lam"], ln, ga, seed=W.SEED_GA, mu=mu, pixel_base=pixel_id_base, threads=1)
            return torch.from_numpy(r["params"]), torch.from_numpy(r["chi2"])

        start, count = S.pixel_shard(n_pixels, rank, world)
        p_loc, c_loc = S.invert_shard(engine, obs[start:start + count], start, mu=mu[start:start + count])
        p_all, c_all = S.gather_results(p_loc, c_loc, n_pixels)
        dist.barrier()
        if rank == 0:
            p_one, c_one = engine(obs, 0, mu=mu)
            wrong_p, _ = engine(obs[start + count:], 0, mu=mu[start + count:])       # rank 1's pixels keyed from 0
            q.put((torch.equal(p_all, p_one), torch.equal(c_all, c_one),
                   bool(torch.equal(wrong_p, p_one[start + count:])), tuple(p_all.shape)))
    finally:
        dist.destroy_process_group()


def test_two_rank_shards_reproduce_single_run():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    n_pixels, world = 7, 2                                    # ragged: shards of 4 and 3
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n_pixels, q)) for r in range(world)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(timeout=240)
    assert all(p.exitcode == 0 for p in procs), [p.exitcode for p in procs]
    same_p, same_c, wrong_same, shape = q.get(timeout=10)
    assert shape == (n_pixels, 9)
    assert same_p and same_c                                   # bit-identical to the single-process run
    assert not wrong_same                                      # and the global keying matters
