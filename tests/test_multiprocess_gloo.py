"""N > 1 host logic on CPU: two processes over gloo (the GPU path uses the same functions over NCCL).
Each rank runs the ORACLE on its shard of the disorders; the sharded job must draw the same instances and
the same uniforms as a single process (global disorder indexing), and the report reduction must give the
max of the times and the sum of the counts."""
import os
import sys

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _one_disorder(d, L, chi, beta, n_s, inst_seed, seed):
    from oracle import bmps, exact, metropolis, philox, sampler
    from tnmc_workloads import make_couplings
    Jr, Jd = make_couplings(L, 1, inst_seed, first_disorder=d)
    cache, _ = bmps.build_cache(Jr[0], Jd[0], beta, chi)
    u = np.empty((n_s, L, L))
    for r in range(L):
        for c in range(L):
            u[:, r, c] = philox.spin_uniforms(seed, d, np.arange(n_s), r * L + c)
    cfg, logq, _ = sampler.sample(cache, Jd[0], beta, u)
    E = exact.energy(cfg, Jr[0], Jd[0])
    um = philox.metropolis_uniforms(seed, d, np.arange(n_s))
    _, n_acc, *_ = metropolis.metropolis_scan(E, logq, beta, um)
    return int(n_acc), int(E.sum()), Jr[0]


def _worker(rank, world, port, out_dir):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2509_19006_b200 import shard
    n_dis = 2
    first = shard.first_disorder(rank, n_dis)
    acc, esum = 0, 0
    for d in range(first, first + n_dis):
        a, e, _ = _one_disorder(d, 4, 2, 1.0, 12, 77, 5)
        acc += a
        esum += e
    ms, total = shard.reduce_job(10.0 + rank, acc)
    _, etot = shard.reduce_job(0.0, esum)
    np.save(os.path.join(out_dir, f"r{rank}.npy"), np.array([first, ms, total, etot]))
    dist.destroy_process_group()


def test_two_rank_sharding_matches_single_process(tmp_path):
    world, port = 2, 29500 + (os.getpid() % 2000)
    mp.spawn(_worker, args=(world, port, str(tmp_path)), nprocs=world, join=True)
    res = [np.load(tmp_path / f"r{r}.npy") for r in range(world)]
    assert [int(r[0]) for r in res] == [0, 2]
    single = [_one_disorder(d, 4, 2, 1.0, 12, 77, 5) for d in range(4)]
    for r in res:
        assert r[1] == 11.0                                # max over ranks of the per-rank time
        assert r[2] == sum(s[0] for s in single)           # sum over ranks of the accepted counts
        assert r[3] == sum(s[1] for s in single)
    # the instances are functions of the global disorder index only
    from tnmc_workloads import make_couplings
    Jr_all, _ = make_couplings(4, 4, 77)
    for d in range(4):
        assert (Jr_all[d] == single[d][2]).all()


def test_reduce_job_without_process_group():
    sys.path.insert(0, ROOT)
    from paper_2509_19006_b200 import shard
    assert shard.reduce_job(3.5, 7) == (3.5, 7.0)
    assert shard.first_disorder(3, 100) == 300
