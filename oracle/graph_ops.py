"""Oracle of the graph operations built on a finished edge list.  TEST INFRASTRUCTURE ONLY.

Plain numpy / Python, written from the paper's statements:
  * symmetric graph (section 3 "Symmetric graph"): the KNN graph is directed; the symmetric
    graph is the smallest symmetric multigraph that contains it: for every edge (i, j, tau) the edge
    (j, i, -tau) is added unless it is there, and every edge appears once;
  * triplets (Def. 3: Gamma_2; "Triplets generation"): the ordered pairs of
    distinct edges that share their source.
Shares no code with the CUDA package (its csrc/graph_ops.cuh).
"""
from __future__ import annotations

import numpy as np


def symmetrize(n_atoms: int, src, dst, tau, vec=None, dist=None) -> dict:
    """Edges as arrays (any order).  Returns the symmetric graph, CSR by source: inside a row first the
    row's own edges in their given order, then the added reverse edges sorted by (dst, tau)."""
    src = np.asarray(src, np.int64)
    dst = np.asarray(dst, np.int64)
    tau = np.asarray(tau, np.int64).reshape(-1, 3)
    e = src.shape[0]
    vec = np.zeros((e, 3)) if vec is None else np.asarray(vec, np.float64).reshape(-1, 3)
    dist = np.zeros(e) if dist is None else np.asarray(dist, np.float64)
    have = set()
    for q in range(e):
        key = (int(src[q]), int(dst[q]), int(tau[q, 0]), int(tau[q, 1]), int(tau[q, 2]))
        assert key not in have, "input edge list has a duplicate"
        have.add(key)
    rows = [[] for _ in range(n_atoms)]
    for q in range(e):
        rows[int(src[q])].append((int(dst[q]), tuple(int(t) for t in tau[q]), tuple(vec[q]), float(dist[q])))
    added = [[] for _ in range(n_atoms)]
    for q in range(e):
        i, j = int(src[q]), int(dst[q])
        rt = (-int(tau[q, 0]), -int(tau[q, 1]), -int(tau[q, 2]))
        if (j, i) + rt not in have:
            added[j].append((i, rt, tuple(-vec[q]), float(dist[q])))
    o_src, o_dst, o_tau, o_vec, o_dist, row_ptr = [], [], [], [], [], [0]
    for i in range(n_atoms):
        for (j, t, v, d) in rows[i] + sorted(added[i], key=lambda r: (r[0], r[1])):
            o_src.append(i); o_dst.append(j); o_tau.append(t); o_vec.append(v); o_dist.append(d)
        row_ptr.append(len(o_src))
    return dict(n_edges=len(o_src), row_ptr=np.asarray(row_ptr, np.int64), src=np.asarray(o_src, np.int64),
                dst=np.asarray(o_dst, np.int64), tau=np.asarray(o_tau, np.int64).reshape(-1, 3),
                vec=np.asarray(o_vec, np.float64).reshape(-1, 3), dist=np.asarray(o_dist, np.float64))


def triplets(row_ptr) -> dict:
    """Gamma_2 from a CSR row_ptr: for source i with edges e0 .. e0 + d - 1 the pairs (a, b), a != b,
    in the order (a, b).  Returns tri_ptr [n_atoms + 1], edge_a, edge_b."""
    row_ptr = np.asarray(row_ptr, np.int64)
    n = row_ptr.shape[0] - 1
    ea, eb, tri_ptr = [], [], [0]
    for i in range(n):
        e0, e1 = int(row_ptr[i]), int(row_ptr[i + 1])
        for a in range(e0, e1):
            for b in range(e0, e1):
                if a != b:
                    ea.append(a); eb.append(b)
        tri_ptr.append(len(ea))
    return dict(n_triplets=len(ea), tri_ptr=np.asarray(tri_ptr, np.int64), edge_a=np.asarray(ea, np.int64),
                edge_b=np.asarray(eb, np.int64))
