"""World-size-2 gloo tests (CPU) of the multi-GPU host logic: ligand / chain sharding and the top-k merge."""
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
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2510_24186_b200 import shard
    g = torch.Generator().manual_seed(7)
    # ---- ligand sharding: 7 ligands, k = 2
    n_lig, k, stride = 7, 2, 9
    E = torch.randn(n_lig, k, 2, generator=g); P = torch.randn(n_lig, k, stride, generator=g)
    C = torch.randint(0, 50, (n_lig, k), generator=g, dtype=torch.int32)
    ids = shard.ligand_shard(n_lig, rank, world)
    e, p, c = shard.merge_ligand_shards(E[ids], P[ids], C[ids], n_lig)
    ok1 = torch.equal(e, E) and torch.equal(p, P) and torch.equal(c, C)
    # ---- chain sharding: 10 global chains, each rank holds its local top-3, merged to the global top-4
    n_ch, kk = 10, 4
    Eb = torch.tensor([[3., 1., 1., 5., -2., 7., 0., 1., 9., -2.]]).repeat(3, 1)      # ties on purpose
    Eb[1] = torch.randn(n_ch, generator=g); Eb[2] = torch.randn(n_ch, generator=g)
    base, n_local = shard.chain_shard(n_ch, rank, world)
    loc = Eb[:, base:base + n_local]
    order = torch.stack([torch.tensor(sorted(range(n_local), key=lambda i: (float(row[i]), i))[:3]) for row in loc])
    le = torch.stack([torch.gather(loc, 1, order), torch.gather(loc, 1, order) / 1.06], dim=-1)
    lp = order.float().unsqueeze(-1).repeat(1, 1, stride) + base
    me, mp_, mc = shard.merge_chain_shards(le, lp, order.to(torch.int32), base, kk)
    want = [sorted(range(n_ch), key=lambda i: (float(row[i]), i))[:kk] for row in Eb]
    ok2 = mc.tolist() == want and torch.equal(me[..., 0], torch.stack([Eb[r][want[r]] for r in range(3)]))
    ok2 = ok2 and torch.equal(mp_[..., 0], torch.tensor(want).float())
    # ---- uneven chain shards: 5 chains over 2 ranks = 3 + 2, local top-3 of a rank with 2 chains has only 2 candidates
    n_ch = 5
    Eu = torch.tensor([[4., -1., 2., -1., 0.5]])
    base, n_local = shard.chain_shard(n_ch, rank, world)
    loc = Eu[:, base:base + n_local]
    k_local = min(3, n_local)
    order = torch.stack([torch.tensor(sorted(range(n_local), key=lambda i: (float(row[i]), i))[:k_local]) for row in loc])
    le = torch.stack([torch.gather(loc, 1, order), torch.gather(loc, 1, order)], dim=-1)
    lp = order.float().unsqueeze(-1).repeat(1, 1, stride) + base
    me, mp_, mc = shard.merge_chain_shards(le, lp, order.to(torch.int32), base, 5)
    ok3 = mc.tolist() == [[1, 3, 4, 2, 0]] and me[0, :, 0].tolist() == [-1., -1., 0.5, 2., 4.]
    # more slots asked for than candidates exist: the tail is fillers (chain -1, +inf)
    me, mp_, mc = shard.merge_chain_shards(le[:, :1], lp[:, :1], order[:, :1].to(torch.int32), base, 3)
    ok3 = ok3 and mc.tolist() == [[1, 3, -1]] and torch.isinf(me[0, 2, 0]).item()
    try:
        shard.merge_chain_shards(le, lp, order.to(torch.int32), base, 2, cluster_rmsd=1.0)
        ok3 = False
    except ValueError:
        pass
    q.put((rank, bool(ok1), bool(ok2 and ok3)))
    dist.destroy_process_group()


def test_shard_and_merge_world2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = [q.get(timeout=120) for _ in procs]
    for p in procs:
        p.join(timeout=60)
    assert sorted(res) == [(0, True, True), (1, True, True)]


def test_shards_partition_the_work():
    from paper_2510_24186_b200 import shard
    for n, w in ((4096, 8), (7, 2), (1, 4), (65536, 8)):
        ids = sorted(i for r in range(w) for i in shard.ligand_shard(n, r, w))
        assert ids == list(range(n))
    for n, w in ((384, 8), (1024, 3), (5, 8)):
        blocks = [shard.chain_shard(n, r, w) for r in range(w)]
        covered = [c for b, m in blocks for c in range(b, b + m)]
        assert covered == list(range(n))
