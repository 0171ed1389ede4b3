"""N > 1 host logic on CPU: world_size-2 gloo run of the by-source sharding.

One (N_LP, N_HP) workload is split over the ranks with multi.shard (round-robin by global source index); every rank
forms its raw accumulators S_LP, S_LPc, S_HP from its own sources, the ranks all-reduce them (multi.allreduce_sums)
and the result must be the single-process accumulators -- hence, after the division the library does
(tsm_combine_sums; written out here with numpy), the oracle's combiner on all sources.  Unequal (n_lp_r, n_hp_r) per
rank, a rank without any HP source, and N_HP = 0 are covered."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

CASES = [(9, 3), (9, 2), (5, 1), (4, 0), (3, 3)]      # (N_LP, N_HP): (5,2)+(4,1); (5,1)+(4,1); (3,1)+(2,0); ...
LEN = 7


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def per_source(n_lp, n_hp, seed):
    rng = np.random.default_rng(seed)
    lp = rng.normal(size=(n_lp, LEN)) + 1j * rng.normal(size=(n_lp, LEN))
    hp = rng.normal(size=(n_hp, LEN)) + 1j * rng.normal(size=(n_hp, LEN))
    return lp, hp


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_1401_6750_b200 import multi
    res = []
    for ci, (N_lp, N_hp) in enumerate(CASES):
        lp, hp = per_source(N_lp, N_hp, 100 + ci)          # every rank knows all arrays, uses only its own sources
        n_lp, n_hp, first, stride = multi.shard(N_lp, N_hp, rank, world)
        mine = [first + j * stride for j in range(n_lp)]
        sums = np.zeros((3, LEN), dtype=np.complex128)
        for j, r in enumerate(mine):
            sums[0] += lp[r]
            if j < n_hp:                                    # the first n_hp LOCAL sources are the rank's HP sources
                assert r < N_hp
                sums[1] += lp[r]
                sums[2] += hp[r]
        t = torch.from_numpy(sums.copy())
        multi.allreduce_sums(t)
        res.append((n_lp, n_hp, mine, t.numpy()))
    q.put((rank, res))
    dist.barrier()
    dist.destroy_process_group()


def test_sharded_sums_gloo(orc):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    world = 2
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = dict(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    for ci, (N_lp, N_hp) in enumerate(CASES):
        lp, hp = per_source(N_lp, N_hp, 100 + ci)
        got = [res[r][ci] for r in range(world)]
        # the shards cover every source exactly once, and every HP source is some rank's HP source
        assert sorted(sum((g[2] for g in got), [])) == list(range(N_lp))
        assert sum(g[0] for g in got) == N_lp and sum(g[1] for g in got) == N_hp
        assert max(g[1] for g in got) - min(g[1] for g in got) <= 1          # HP work is balanced
        S = np.stack([lp.sum(0), lp[:N_hp].sum(0), hp.sum(0)])
        for g in got:
            assert np.allclose(g[3], S, atol=1e-13)
            est = g[3][0] / N_lp + ((g[3][2] - g[3][1]) / N_hp if N_hp else 0)
            assert np.allclose(est, orc.tsm_combine(lp, hp), atol=1e-13)


def test_shard_edges():
    from paper_1401_6750_b200 import multi
    assert multi.shard(500, 20, 0, 8) == (63, 3, 0, 8)
    assert multi.shard(500, 20, 7, 8) == (62, 2, 7, 8)
    assert sum(multi.shard(500, 20, k, 8)[0] for k in range(8)) == 500
    assert sum(multi.shard(500, 20, k, 8)[1] for k in range(8)) == 20
    assert multi.shard(2, 1, 3, 4) == (0, 0, 3, 4)           # more ranks than sources
    assert multi.shard(7, 3, 0, 1) == (7, 3, 0, 1)
    with pytest.raises(ValueError):
        multi.shard(3, 4, 0, 2)
    with pytest.raises(ValueError):
        multi.shard(3, 1, 2, 2)
