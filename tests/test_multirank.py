"""world_size-2 gloo test (CPU) of the N>1 host logic: z-sharding + one all-reduce of the per-cosmology sums
(DESIGN.md section 9).  The per-shard partial sums come from the oracle (no GPU here); what is under test is
paper_2212_01937_b200.sharding, which bench.py uses unchanged with the nccl backend."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2212_01937_b200 import sharding


def test_shard_bounds_partition():
    for n in (0, 1, 7, 1000, 1_000_003):
        for world in (1, 2, 3, 8):
            edges = [sharding.shard_bounds(n, world, r) for r in range(world)]
            assert edges[0][0] == 0 and edges[-1][1] == n
            assert all(edges[r][1] == edges[r + 1][0] for r in range(world - 1))
            sizes = [b - a for a, b in edges]
            assert max(sizes) - min(sizes) <= 1


def _worker(rank, world, port, n, S, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import oracle
    from paper_2212_01937_b200 import workloads as W
    w = W.config3_shard(n, world, rank, S=S)          # exactly what bench.py --gpus N gives rank `rank`
    MU = oracle.OBS.index("MU")
    gp = torch.zeros((4, S), dtype=torch.float64)
    for s in range(S):
        _, grad, _ = oracle.observables_batch(w.z, w.Om[s:s + 1], w.OL[s:s + 1], w.Or[s:s + 1], w.H0[s:s + 1], with_grad=True, threads=1)
        g = w.grad_out[0, s]
        for p in range(4):
            gp[p, s] = float((g * grad[:, MU, 1 + p].astype(np.float64)).sum())
    sharding.allreduce_sums(gp)
    if rank == 0:
        q.put(gp.numpy())
    dist.barrier()
    dist.destroy_process_group()


def test_gloo_two_ranks_match_single():
    import oracle
    from paper_2212_01937_b200 import workloads as W
    n, S = 301, 2
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, n, S, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    # the same job on ONE rank: the shards concatenated (W.config3_shard draws the global redshift array once and cuts it)
    shards = [W.config3_shard(n, 2, r, S=S) for r in range(2)]
    z = np.concatenate([w.z for w in shards]); g = np.concatenate([w.grad_out for w in shards], axis=2)
    one = W.config3_shard(2 * n, 1, 0, S=S)
    assert np.array_equal(z, one.z) and np.array_equal(shards[0].Om, one.Om) and (np.diff(z) >= 0).all()
    w = shards[0]
    MU = oracle.OBS.index("MU")
    for s in range(S):
        _, grad, _ = oracle.observables_batch(z, w.Om[s:s + 1], w.OL[s:s + 1], w.Or[s:s + 1], w.H0[s:s + 1], with_grad=True)
        for p in range(4):
            terms = g[0, s] * grad[:, MU, 1 + p].astype(np.float64)
            assert abs(got[p, s] - terms.sum()) <= 1e-12 * np.abs(terms).sum()
