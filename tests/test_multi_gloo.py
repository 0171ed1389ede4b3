"""N > 1 host logic on CPU: world_size-2 gloo run of the by-source combination."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_1401_6750_b200 import multi
    rng = np.random.default_rng(100 + rank)
    n_lp, n_hp = (6, 2) if rank == 0 else (3, 1)
    lp = rng.normal(size=(n_lp, 5)) + 1j * rng.normal(size=(n_lp, 5))
    hp = rng.normal(size=(n_hp, 5)) + 1j * rng.normal(size=(n_hp, 5))
    local = lp.mean(0) + (hp - lp[:n_hp]).mean(0)
    out = multi.combine_over_ranks(torch.from_numpy(local), n_lp, n_hp)
    ok_ratio = True
    try:
        multi.combine_over_ranks(torch.from_numpy(local), n_lp, n_hp + rank)
        ok_ratio = False
    except ValueError:
        pass
    q.put((rank, lp, hp, out.numpy(), ok_ratio, multi.rank_seed(5, rank)))
    dist.barrier()
    dist.destroy_process_group()


def test_combine_over_ranks_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted([q.get(timeout=120) for _ in procs], key=lambda t: t[0])
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    lp = np.concatenate([res[0][1], res[1][1]])
    hp_minus_lp = np.concatenate([res[0][2] - res[0][1][:2], res[1][2] - res[1][1][:1]])
    ref = lp.mean(0) + hp_minus_lp.mean(0)      # the single-process estimator over all 9 sources
    for r in res:
        assert np.allclose(r[3], ref, atol=1e-14)
        assert r[4]
    assert res[0][5] != res[1][5]
