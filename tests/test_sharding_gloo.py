"""N>1 path on CPU: world_size-2 gloo.  Each rank computes its q-shard's partial Sigma and K with the oracle
(q-range slices), the library's all-reduce helper sums them, and the result must equal the unsharded oracle.
This covers paper_2206_07660_b200.dist (shard planner + all-reduce plumbing) without a GPU."""
import os
import sys

import numpy as np
import pytest
import torch
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, ret):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    import gwgen
    import oracle
    from paper_2206_07660_b200.dist import shard_range, allreduce_sum_
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    p = gwgen.make_problem("T")
    cfg = p.cfg
    vb = oracle.VBlocks(cfg, p.V.numpy())
    P0t = oracle.polarization(cfg, vb, p.G)
    Wt = oracle.screened_interaction(cfg, p.T_wt, p.T_tw, P0t)
    q0, q1 = shard_range(cfg.nk, world, rank)
    Sg = np.zeros((cfg.ntau, cfg.nk, cfg.nao, cfg.nao), complex)
    K = np.zeros((cfg.nk, cfg.nao, cfg.nao), complex)
    for k in range(cfg.nk):
        K[k] = oracle.exchange_slice(cfg, vb, p.gamma, k, q0, q1)
        for t in range(cfg.ntau):
            Sg[t, k] = oracle.sigma_slice(cfg, vb, p.G[t], np.ascontiguousarray(Wt[t]), k, q0, q1)
    tS, tK = torch.from_numpy(Sg), torch.from_numpy(K)
    allreduce_sum_([tS, tK])
    if rank == 0:
        full_S = oracle.selfenergy(cfg, vb, p.G, Wt)
        full_K = oracle.exchange(cfg, vb, p.gamma)
        ret["eS"] = float(np.linalg.norm(tS.numpy() - full_S) / np.linalg.norm(full_S))
        ret["eK"] = float(np.linalg.norm(tK.numpy() - full_K) / np.linalg.norm(full_K))
    dist.destroy_process_group()


def test_shard_ranges_cover_all_q():
    from paper_2206_07660_b200.dist import shard_range
    for nk in (1, 6, 8, 64, 125):
        for world in (1, 2, 3, 4, 8):
            if world > nk:
                continue
            r = [shard_range(nk, world, i) for i in range(world)]
            assert r[0][0] == 0 and r[-1][1] == nk
            assert all(r[i][1] == r[i + 1][0] for i in range(world - 1))
            sizes = [b - a for a, b in r]
            assert max(sizes) - min(sizes) <= 1 and min(sizes) >= 1


@pytest.mark.timeout(300)
def test_two_rank_partial_sums_gloo():
    import oracle
    oracle.build()
    mgr = mp.Manager()
    ret = mgr.dict()
    port = 29500 + (os.getpid() % 1000)
    mp.spawn(_worker, args=(2, port, ret), nprocs=2, join=True)
    assert ret["eS"] < 1e-13 and ret["eK"] < 1e-13
