"""Multi-GPU sharding of the docking job: one process per GPU, no collective inside the
step loop -- chains never communicate and ligands are independent.  Screens shard by
LIGAND, single docks by CHAIN (disjoint Philox chain ids via tridsk_dock_opts.chain_base, so results do not
depend on the GPU count).  The only exchange is the final top-k merge: one small all_gather.
Works on CPU tensors with gloo and CUDA tensors with nccl.
"""
from __future__ import annotations

import torch
import torch.distributed as dist


def ligand_shard(n_lig: int, rank: int, world: int):
    """Round-robin ligand ids of this rank (balanced when ligands are sorted or random in size)."""
    return list(range(rank, n_lig, world))


def chain_shard(n_chains: int, rank: int, world: int):
    """(chain_base, n_local) of this rank's contiguous block of global chain ids."""
    per = (n_chains + world - 1) // world
    base = min(rank * per, n_chains)
    return base, max(0, min(per, n_chains - base))


def merge_ligand_shards(energy, pose, chain, n_lig: int):
    """Inverse of ligand_shard: every rank gets [n_lig, k, ...] results for all ligands."""
    world, rank = dist.get_world_size(), dist.get_rank()
    per = (n_lig + world - 1) // world
    outs = []
    for t in (energy, pose, chain):
        pad = torch.zeros((per,) + tuple(t.shape[1:]), dtype=t.dtype, device=t.device)
        pad[: t.shape[0]] = t
        buf = [torch.empty_like(pad) for _ in range(world)]
        dist.all_gather(buf, pad)
        full = torch.zeros((n_lig,) + tuple(t.shape[1:]), dtype=t.dtype, device=t.device)
        for r in range(world):
            ids = ligand_shard(n_lig, r, world)
            full[ids] = buf[r][: len(ids)]
        outs.append(full)
    return tuple(outs)


def merge_chain_shards(energy, pose, chain, chain_base: int, k: int, cluster_rmsd: float = 0.0):
    """Global top-k per ligand from every rank's local top-k candidates: sort by (E_dock, global chain id) (O13).
    energy [n_lig, k_local, 2], pose [n_lig, k_local, stride], chain [n_lig, k_local] (local ids; -1 = an empty slot).
    k_local may differ between ranks (uneven chain shards: a rank with fewer chains than k returns fewer candidates):
    every rank's block is padded to the largest k_local with (+inf, zero pose, chain -1) before the all_gather, and the
    fillers sort last; if fewer than k real candidates exist overall the tail of the result is such fillers.
    Duplicate removal (tridsk_dock_opts.cluster_rmsd, O14) compares poses ACROSS chains, so per-shard filtered candidates
    cannot be merged by a sort: it is refused here -- shard such a job by ligand, or dock it on one GPU."""
    if cluster_rmsd > 0.0:
        raise ValueError("merge_chain_shards: duplicate-removing top-k (cluster_rmsd > 0) cannot be merged across chain "
                         "shards; shard by ligand or run the dock on one GPU")
    world = dist.get_world_size()
    k_loc = torch.tensor([energy.shape[1]], dtype=torch.int64, device=energy.device)
    ks = [torch.zeros_like(k_loc) for _ in range(world)]
    dist.all_gather(ks, k_loc)
    k_pad = int(max(int(v) for v in ks))
    valid = chain >= 0
    g_chain = torch.where(valid, chain.to(torch.int64) + int(chain_base), torch.full_like(chain, -1, dtype=torch.int64))
    e_in = energy.clone()
    e_in[~valid] = float("inf")

    def pad(t, fill):
        if t.shape[1] == k_pad:
            return t.contiguous()
        ext = torch.full((t.shape[0], k_pad - t.shape[1]) + tuple(t.shape[2:]), fill, dtype=t.dtype, device=t.device)
        return torch.cat([t, ext], dim=1).contiguous()

    parts = []
    for t, fill in ((e_in, float("inf")), (pose, 0.0), (g_chain, -1)):
        tp = pad(t, fill)
        buf = [torch.empty_like(tp) for _ in range(world)]
        dist.all_gather(buf, tp)
        parts.append(torch.cat(buf, dim=1))
    e, p, c = parts
    if e.shape[1] < k:                                                # fewer candidates than slots asked for
        short = k - e.shape[1]
        ext = lambda t, fill: torch.cat([t, torch.full((t.shape[0], short) + tuple(t.shape[2:]), fill, dtype=t.dtype, device=t.device)], dim=1)
        e, p, c = ext(e, float("inf")), ext(p, 0.0), ext(c, -1)
    # fillers (chain -1, +inf) must sort after every real candidate, also after a real +inf energy: key them by a huge id
    ckey = torch.where(c >= 0, c, torch.full_like(c, 2 ** 62))
    o1 = torch.argsort(ckey, dim=1, stable=True)                      # secondary key first
    e1 = torch.gather(e[..., 0], 1, o1)
    o2 = torch.argsort(e1, dim=1, stable=True)
    order = torch.gather(o1, 1, o2)[:, :k]
    take = lambda t: torch.gather(t, 1, order.reshape(order.shape + (1,) * (t.dim() - 2)).expand(order.shape + tuple(t.shape[2:])))
    return take(e), take(p), torch.gather(c, 1, order)
