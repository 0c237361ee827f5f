"""Acceptance checks of a produced graph against the FP64 oracle.  TEST INFRASTRUCTURE ONLY.

Implements the acceptance rules of BASELINE.json north_star / SURVEY 8(c):
  * cutoff: the symmetric difference of the canonical (src, dst, tau) sets may only hold edges
    whose FP64 distance is within BAND = 1e-5 A of r_c; vec within 1e-5 A absolute.
  * KNN: k distinct entries per atom, none (i,i,0); wherever the produced row differs from the
    oracle row the two FP64 distances differ by <= BAND; every produced entry outside the oracle
    row has d <= d_k + BAND and every missing oracle entry has d >= d_k - BAND; vec within 1e-5.
Takes plain numpy arrays; imports nothing from the CUDA package.
"""
from __future__ import annotations

import numpy as np

from . import cutoff_graph, edge_distance, knn_graph

BAND = 1e-5       # Angstrom, north_star
VEC_TOL = 1e-5    # Angstrom absolute, north_star


def _keys(src, dst, tau):
    """Pack (src, dst, tau+128) into one int64 per edge: src 24 bits | dst 24 | 3 x 8 -> fits 63."""
    src = np.asarray(src, np.int64)
    dst = np.asarray(dst, np.int64)
    t = np.asarray(tau, np.int64).reshape(-1, 3) + 128
    assert src.size == 0 or (src.max() < (1 << 19) and dst.max() < (1 << 19)), "key packing range"
    assert t.size == 0 or (t.min() >= 0 and t.max() < 256)
    return (src << 43) | (dst << 24) | (t[:, 0] << 16) | (t[:, 1] << 8) | t[:, 2]


def check_csr(n_atoms, row_ptr, src, n_edges):
    row_ptr = np.asarray(row_ptr, np.int64)
    assert row_ptr.shape == (n_atoms + 1,), f"row_ptr shape {row_ptr.shape}"
    assert row_ptr[0] == 0 and row_ptr[-1] == n_edges, (row_ptr[0], row_ptr[-1], n_edges)
    assert np.all(np.diff(row_ptr) >= 0)
    expect_src = np.repeat(np.arange(n_atoms, dtype=np.int64), np.diff(row_ptr))
    assert np.array_equal(np.asarray(src, np.int64)[:n_edges], expect_src), "src does not follow row_ptr"


def check_cutoff(batch, r_c, got: dict, ref: dict | None = None) -> dict:
    """got: row_ptr, src, dst, offset [E,3], vec [E,3] (float32), optional dist, n_edges."""
    pos, lat, ptr = batch.pos, batch.lattice, batch.struct_ptr
    if ref is None:
        ref = cutoff_graph(pos, lat, ptr, r_c)
    rc = float(np.float32(r_c))
    e = int(got["n_edges"])
    src, dst = np.asarray(got["src"])[:e], np.asarray(got["dst"])[:e]
    tau = np.asarray(got["offset"]).reshape(-1, 3)[:e].astype(np.int32)
    vec = np.asarray(got["vec"]).reshape(-1, 3)[:e].astype(np.float64)
    check_csr(batch.n_atoms, got["row_ptr"], src, e)
    # dst in the same structure as src
    s_src = np.searchsorted(ptr, src, side="right") - 1
    s_dst = np.searchsorted(ptr, dst, side="right") - 1
    assert np.array_equal(s_src, s_dst), "edge joins two structures"
    assert not np.any((src == dst) & np.all(tau == 0, axis=1)), "(i,i,0) emitted"
    kg = _keys(src, dst, tau)
    ko = _keys(ref["src"], ref["dst"], ref["tau"])
    order = np.argsort(kg, kind="stable")
    kg_sorted = kg[order]
    assert np.all(np.diff(kg_sorted) != 0), "duplicate edges"
    only_g = np.setdiff1d(kg_sorted, ko, assume_unique=True)
    only_o = np.setdiff1d(ko, kg_sorted, assume_unique=True)
    # FP64 distances of every produced edge
    d64, v64 = edge_distance(pos, lat, ptr, src, dst, tau)
    if only_g.size:
        sel = np.isin(kg, only_g)
        assert np.all(np.abs(d64[sel] - rc) <= BAND), \
            f"{only_g.size} extra edges, worst |d-r_c| = {np.abs(d64[sel] - rc).max():.3e}"
    if only_o.size:
        sel = np.isin(ko, only_o)
        assert np.all(np.abs(ref["dist"][sel] - rc) <= BAND), \
            f"{only_o.size} missing edges, worst |d-r_c| = {np.abs(ref['dist'][sel] - rc).max():.3e}"
    vec_err = float(np.abs(vec - v64).max()) if e else 0.0
    assert vec_err <= VEC_TOL, f"vec error {vec_err:.3e}"
    dist_err = 0.0
    if got.get("dist") is not None:
        dist_err = float(np.abs(np.asarray(got["dist"])[:e].astype(np.float64) - d64).max()) if e else 0.0
        assert dist_err <= VEC_TOL, f"dist error {dist_err:.3e}"
    # common edges: oracle vec equals the recomputed one (ties the two oracle routes together)
    return dict(n_edges=e, n_ref=int(ref["n_edges"]), extra=int(only_g.size), missing=int(only_o.size),
                vec_err=vec_err, dist_err=dist_err)


def check_knn(batch, k, got: dict, ref: dict | None = None) -> dict:
    pos, lat, ptr = batch.pos, batch.lattice, batch.struct_ptr
    if ref is None:
        ref = knn_graph(pos, lat, ptr, k)
    n = batch.n_atoms
    e = int(got["n_edges"])
    assert e == k * n, (e, k, n)
    src, dst = np.asarray(got["src"])[:e], np.asarray(got["dst"])[:e]
    tau = np.asarray(got["offset"]).reshape(-1, 3)[:e].astype(np.int32)
    vec = np.asarray(got["vec"]).reshape(-1, 3)[:e].astype(np.float64)
    check_csr(n, got["row_ptr"], src, e)
    assert np.array_equal(np.asarray(got["row_ptr"], np.int64), k * np.arange(n + 1, dtype=np.int64))
    s_src = np.searchsorted(ptr, src, side="right") - 1
    s_dst = np.searchsorted(ptr, dst, side="right") - 1
    assert np.array_equal(s_src, s_dst), "edge joins two structures"
    assert not np.any((src == dst) & np.all(tau == 0, axis=1)), "(i,i,0) emitted"
    if e == 0:
        return dict(n_edges=0, exact_rows=0, mismatched_entries=0, vec_err=0.0)
    kg = _keys(src, dst, tau).reshape(n, k)
    ko = _keys(ref["src"], ref["dst"], ref["tau"]).reshape(n, k)
    assert np.all(np.diff(np.sort(kg, axis=1), axis=1) != 0), "duplicate neighbour in a row"
    d64, v64 = edge_distance(pos, lat, ptr, src, dst, tau)
    dg = d64.reshape(n, k)
    do = ref["dist"].reshape(n, k)
    dk = do[:, -1]
    # position-wise: different entry => distances inside the tie band
    diff = kg != ko
    if np.any(diff):
        worst = np.abs(dg - do)[diff].max()
        assert worst <= BAND, f"KNN order/selection mismatch outside the tie band: {worst:.3e}"
    # membership
    in_o = np.zeros_like(diff)
    in_g = np.zeros_like(diff)
    rows = np.nonzero(np.any(diff, axis=1))[0]
    for r in rows:
        in_o[r] = np.isin(kg[r], ko[r])
        in_g[r] = np.isin(ko[r], kg[r])
    if rows.size:
        extra = ~in_o[rows]
        miss = ~in_g[rows]
        assert np.all(dg[rows][extra] <= dk[rows][:, None].repeat(k, 1)[extra] + BAND)
        assert np.all(do[rows][miss] >= dk[rows][:, None].repeat(k, 1)[miss] - BAND)
    # produced order is non-decreasing in FP64 up to the band
    run_max = np.maximum.accumulate(dg, axis=1)
    assert np.all(dg >= run_max - BAND), "KNN row not sorted by distance"
    vec_err = float(np.abs(vec - v64).max())
    assert vec_err <= VEC_TOL, f"vec error {vec_err:.3e}"
    dist_err = 0.0
    if got.get("dist") is not None:
        dist_err = float(np.abs(np.asarray(got["dist"])[:e].astype(np.float64) - d64).max())
        assert dist_err <= VEC_TOL, f"dist error {dist_err:.3e}"
    return dict(n_edges=e, exact_rows=int(n - rows.size), mismatched_entries=int(diff.sum()),
                vec_err=vec_err, dist_err=dist_err)
