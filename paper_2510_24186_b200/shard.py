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


def merge_chain_shards(energy, pose, chain, chain_base: int, k: int):
    """Global top-k per ligand from every rank's local top-k candidates: sort by (E_dock, global chain id) (O13).
    energy [n_lig, k_local, 2], pose [n_lig, k_local, stride], chain [n_lig, k_local] (local ids)."""
    world = dist.get_world_size()
    g_chain = chain.to(torch.int64) + int(chain_base)
    parts = []
    for t in (energy, pose, g_chain):
        buf = [torch.empty_like(t) for _ in range(world)]
        dist.all_gather(buf, t.contiguous())
        parts.append(torch.cat(buf, dim=1))
    e, p, c = parts
    o1 = torch.argsort(c, dim=1, stable=True)                         # secondary key first
    e1 = torch.gather(e[..., 0], 1, o1)
    o2 = torch.argsort(e1, dim=1, stable=True)
    order = torch.gather(o1, 1, o2)[:, :k]
    take = lambda t: torch.gather(t, 1, order.reshape(order.shape + (1,) * (t.dim() - 2)).expand(order.shape + tuple(t.shape[2:])))
    return take(e), take(p), torch.gather(c, 1, order)
