"""Multi-GPU sharding of a batch (host logic only).

Structures are independent (no edge joins two structures), so the path shards by
contiguous structure ranges with no data-path collective: every rank builds the CSR of its own
structures with the single-GPU library and only the per-rank atom / edge COUNTS are exchanged
(one all_gather of two integers) to place the local CSR in the global index space.
"""
from __future__ import annotations

import numpy as np


def shard_ranges(struct_ptr, world: int):
    """Contiguous structure ranges [(s0, s1)] * world, balanced by sum N_s^2 (the pair count that
    drives the kernels' work).  Every structure is in exactly one range."""
    struct_ptr = np.asarray(struct_ptr, np.int64)
    n = np.diff(struct_ptr)
    w = np.concatenate([[0], np.cumsum(n * n + 1)])          # +1: empty structures still cost a record
    total = int(w[-1])
    cuts = [0]
    for r in range(1, world):
        cuts.append(int(np.searchsorted(w, (total * r) // world, side="left")))
    cuts.append(len(n))
    cuts = np.maximum.accumulate(np.minimum(cuts, len(n)))
    return [(int(cuts[r]), int(cuts[r + 1])) for r in range(world)]


def shard_batch(pos, lattice, struct_ptr, rank: int, world: int):
    """Local (pos, lattice, struct_ptr rebased to 0, first global atom, first global structure)."""
    s0, s1 = shard_ranges(struct_ptr, world)[rank]
    struct_ptr = np.asarray(struct_ptr)
    a0, a1 = int(struct_ptr[s0]), int(struct_ptr[s1])
    return (np.ascontiguousarray(np.asarray(pos).reshape(-1, 3)[a0:a1]),
            np.ascontiguousarray(np.asarray(lattice).reshape(-1, 3, 3)[s0:s1]),
            (struct_ptr[s0:s1 + 1] - a0).astype(np.int32), a0, s0)


def stitch(local: dict, n_atoms_local: int, group=None):
    """Place a rank's CSR (row_ptr, src, dst of its own structures, local indices) in the global
    index space.  Exchanges (n_atoms, n_edges) of every rank with ONE all_gather; returns the dict
    with global row_ptr / src / dst plus atom_offset, edge_offset, n_edges_global."""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size(group)
    rank = dist.get_rank(group)
    mine = torch.tensor([int(n_atoms_local), int(local["n_edges"])], dtype=torch.int64)
    counts = [torch.zeros(2, dtype=torch.int64) for _ in range(world)]
    dist.all_gather(counts, mine, group=group)
    counts = torch.stack(counts).numpy()
    atom_off = int(counts[:rank, 0].sum())
    edge_off = int(counts[:rank, 1].sum())
    out = dict(local)
    out["row_ptr"] = np.asarray(local["row_ptr"], np.int64) + edge_off
    out["src"] = np.asarray(local["src"], np.int64) + atom_off
    out["dst"] = np.asarray(local["dst"], np.int64) + atom_off
    out.update(atom_offset=atom_off, edge_offset=edge_off, n_edges_global=int(counts[:, 1].sum()),
               n_atoms_global=int(counts[:, 0].sum()))
    return out
