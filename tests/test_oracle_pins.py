"""Pins of the FP64 oracle against things that are NOT the oracle (CPU only).

The paper prints no worked example, so the pins are: textbook shell counts
(tests/golden/shells.txt), an integer sum-of-three-squares count, the fixed cases BASELINE.json
north_star lists, invariants of Def. 3, a [-12,12]^3 numpy brute force that
ignores every bound, and the nearest-image / open-boundary special cases written with numpy.
"""
import itertools
import os

import numpy as np
import pytest

import oracle
from workloads import crystals as C

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "shells.txt")


def _golden():
    table = {}
    with open(GOLDEN) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            name, d2, cnt = line.split()
            table.setdefault(name, []).append((float(d2), int(cnt)))
    return table


def _edge_set(g):
    return set(zip(g["src"].tolist(), g["dst"].tolist(), map(tuple, g["tau"].tolist())))


# ------------------------------------------------------------------ closed forms
@pytest.mark.parametrize("name", sorted(_golden().keys()))
@pytest.mark.parametrize("a", [1.0, 3.25])
def test_shell_counts(name, a):
    shells = _golden()[name]
    b = C.textbook(name, a)
    r = a * np.sqrt(shells[-1][0]) * 1.0005
    g = oracle.cutoff_graph(b.pos, b.lattice, b.struct_ptr, r)
    n = b.n_atoms
    want_d2 = np.array([d2 for d2, _ in shells])
    for i in range(n):
        d = g["dist"][g["row_ptr"][i]:g["row_ptr"][i + 1]]
        d2 = (d / a) ** 2
        nearest = np.abs(d2[:, None] - want_d2[None, :]).argmin(axis=1)
        # every neighbour sits on a listed shell (so no unlisted shell exists below the radius)
        assert np.abs(d2 - want_d2[nearest]).max() < 2e-6, (name, i)
        got = np.bincount(nearest, minlength=len(shells)).tolist()
        assert got == [c for _, c in shells], (name, i, got)


def test_sc_matches_sum_of_three_squares():
    # independent integer count r3(n), n <= 16
    r3 = {}
    for t in itertools.product(range(-4, 5), repeat=3):
        s = t[0] ** 2 + t[1] ** 2 + t[2] ** 2
        if 0 < s <= 16:
            r3[s] = r3.get(s, 0) + 1
    b = C.textbook("sc")
    g = oracle.cutoff_graph(b.pos, b.lattice, b.struct_ptr, 4.0005)
    got = {}
    for x in g["dist"]:
        got[int(round(x * x))] = got.get(int(round(x * x)), 0) + 1
    assert got == r3


@pytest.mark.parametrize("rc,count", [(1.01, 6), (1.42, 18), (1.74, 26), (2.01, 32)])
def test_sc_cumulative(rc, count):
    b = C.textbook("sc")
    assert oracle.cutoff_graph(b.pos, b.lattice, b.struct_ptr, rc)["n_edges"] == count


def test_strict_inequality_and_no_self_loop():
    b = C.textbook("sc")
    # d == r_c exactly is NOT an edge (Def. 3 strict '<'); (i,i,0) never appears
    assert oracle.cutoff_graph(b.pos, b.lattice, b.struct_ptr, 1.0)["n_edges"] == 0
    g = oracle.cutoff_graph(b.pos, b.lattice, b.struct_ptr, 1.5)
    assert not np.any(np.all(g["tau"] == 0, axis=1))
    assert np.all(g["src"] == 0) and np.all(g["dst"] == 0)   # self-images ARE edges


def test_fcc_bcc_first_shell_distances():
    b = C.textbook("fcc_conv", 4.0)
    g = oracle.cutoff_graph(b.pos, b.lattice, b.struct_ptr, 4.0 / np.sqrt(2) + 1e-3)
    assert np.all(np.diff(g["row_ptr"]) == 12)
    assert np.allclose(g["dist"], 4.0 / np.sqrt(2), atol=1e-6)
    b = C.textbook("bcc_conv", 3.0)
    g = oracle.cutoff_graph(b.pos, b.lattice, b.struct_ptr, 3.0 * np.sqrt(3) / 2 + 1e-3)
    assert np.all(np.diff(g["row_ptr"]) == 8)
    assert np.allclose(g["dist"], 3.0 * np.sqrt(3) / 2, atol=1e-6)


def test_knn_sc_order_pins_tiebreak():
    b = C.textbook("sc")
    first6 = [(-1, 0, 0), (0, -1, 0), (0, 0, -1), (0, 0, 1), (0, 1, 0), (1, 0, 0)]
    next6 = [(-1, -1, 0), (-1, 0, -1), (-1, 0, 1), (-1, 1, 0), (0, -1, -1), (0, -1, 1)]
    g = oracle.knn_graph(b.pos, b.lattice, b.struct_ptr, 6)
    assert list(map(tuple, g["tau"].tolist())) == first6
    g = oracle.knn_graph(b.pos, b.lattice, b.struct_ptr, 12)
    assert list(map(tuple, g["tau"].tolist())) == first6 + next6
    assert np.array_equal(g["row_ptr"], [0, 12])
    assert np.allclose(g["dist"][:6], 1.0) and np.allclose(g["dist"][6:], np.sqrt(2.0))


def test_knn_fcc_prim_is_first_shell():
    b = C.textbook("fcc_prim", 2.0)
    g = oracle.knn_graph(b.pos, b.lattice, b.struct_ptr, 12)
    assert np.allclose(g["dist"], 2.0 / np.sqrt(2.0), atol=1e-6)
    c = oracle.cutoff_graph(b.pos, b.lattice, b.struct_ptr, 2.0 / np.sqrt(2.0) + 1e-3)
    assert _edge_set(g) == _edge_set(c)


def test_knn_dst_tiebreak_two_atoms():
    # two atoms on a cubic cell, atom 1 at the body centre: from atom 0 the 8 nearest are images
    # of atom 1 at equal distance; order must be by tau lexicographic (dst equal).
    b = C.textbook("bcc_conv")
    g = oracle.knn_graph(b.pos, b.lattice, b.struct_ptr, 8)
    row0 = list(map(tuple, g["tau"][:8].tolist()))
    assert row0 == sorted(row0)
    assert np.all(g["dst"][:8] == 1) and np.all(g["dst"][8:] == 0)
    # k = 14: 8 body-centre images then 6 self images; dst ordering only matters inside ties
    g = oracle.knn_graph(b.pos, b.lattice, b.struct_ptr, 14)
    assert g["dst"][:14].tolist() == [1] * 8 + [0] * 6


# ------------------------------------------------------------------ definitions
def test_vec_and_dist_definition():
    b = C.small_batch(6, seed=3)
    g = oracle.cutoff_graph(b.pos, b.lattice, b.struct_ptr, 5.0)
    s_of = np.searchsorted(b.struct_ptr, g["src"], side="right") - 1
    p = b.pos.astype(np.float64)
    f = p[g["dst"]] + g["tau"] - p[g["src"]]
    v = np.einsum("ea,eac->ec", f, b.lattice.astype(np.float64)[s_of])   # row vector times lattice (R5)
    assert np.abs(v - g["vec"]).max() < 1e-12
    assert np.abs(np.linalg.norm(v, axis=1) - g["dist"]).max() < 1e-12
    assert np.all(g["dist"] < 5.0)
    # row_ptr / src / canonical order
    assert np.array_equal(np.repeat(np.arange(b.n_atoms), np.diff(g["row_ptr"])), g["src"])
    keys = list(zip(g["src"].tolist(), g["dst"].tolist(), map(tuple, g["tau"].tolist())))
    assert keys == sorted(keys)
    # edges never join two structures
    assert np.array_equal(s_of, np.searchsorted(b.struct_ptr, g["dst"], side="right") - 1)


def test_row_vectors_not_columns():
    # a cell whose transpose gives a different graph: pins R5 (rows are lattice vectors)
    lat = np.array([[[2.0, 0.0, 0.0], [1.5, 1.0, 0.0], [0.0, 0.0, 5.0]]], np.float32)
    pos = np.zeros((1, 3), np.float32)
    ptr = np.array([0, 1], np.int32)
    g = oracle.cutoff_graph(pos, lat, ptr, 1.6)
    # shortest lattice vectors: a2 - a1 = (-0.5, 1, 0) length 1.118, its negative; nothing else < 1.6
    assert sorted(map(tuple, g["tau"].tolist())) == [(-1, 1, 0), (1, -1, 0)]
    assert np.allclose(sorted(g["vec"][:, 0].tolist()), [-0.5, 0.5])


# ------------------------------------------------------------------ brute force without bounds
def _huge_box(pos, lat, rc, m=12):
    """Every image in [-m, m]^3, no search bound at all (numpy, float64)."""
    p = pos.astype(np.float64)
    A = lat.astype(np.float64)
    r = np.arange(-m, m + 1)
    tau = np.stack(np.meshgrid(r, r, r, indexing="ij"), -1).reshape(-1, 3)
    out = set()
    for i in range(p.shape[0]):
        for j in range(p.shape[0]):
            f = (p[j] - p[i])[None, :] + tau
            v = f @ A
            d = np.sqrt((v * v).sum(1))
            ok = d < rc
            for t in tau[ok]:
                if i == j and not t.any():
                    continue
                out.add((i, j, tuple(int(x) for x in t)))
    return out


@pytest.mark.parametrize("seed", range(6))
def test_bounded_box_equals_huge_box(seed):
    rng = np.random.default_rng(100 + seed)
    n = int(rng.integers(1, 5))
    while True:
        a, b_, c = rng.uniform(2.0, 5.0, 3)
        al, be, ga = rng.uniform(35.0, 145.0, 3)
        cell = C.cell_from_parameters(a, b_, c, al, be, ga)
        if cell is not None and C.gram_factor(al, be, ga) > 0.02:
            break
    # random rigid rotation: the oracle must not rely on the standard orientation
    q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    lat = (cell @ q).astype(np.float32)
    pos = rng.random((n, 3), dtype=np.float32)
    ptr = np.array([0, n], np.int32)
    rc = 4.0
    g = oracle.cutoff_graph(pos, lat[None], ptr, rc)
    # the [-12,12]^3 box must contain the cutoff sphere for the comparison to be meaningful
    hmin = abs(np.linalg.det(lat.astype(np.float64))) / max(
        np.linalg.norm(np.cross(lat[1].astype(np.float64), lat[2])),
        np.linalg.norm(np.cross(lat[2].astype(np.float64), lat[0])),
        np.linalg.norm(np.cross(lat[0].astype(np.float64), lat[1])))
    assert rc / hmin + 1 < 12
    assert _edge_set(g) == _huge_box(pos, lat, float(np.float32(rc)))


def test_search_bound_is_never_exceeded():
    # R14: with x in [0,1) no edge has |tau_a| > ceil(r_c / h_a); the oracle searches one cell
    # further and reports the largest |tau| it emitted.
    b = C.skewed_batch(24, seed=5)
    rc = 6.0
    for s in range(b.n_struct):
        sl = slice(b.struct_ptr[s], b.struct_ptr[s + 1])
        g = oracle.cutoff_graph(b.pos[sl], b.lattice[s:s + 1], np.array([0, sl.stop - sl.start], np.int32), rc)
        A = b.lattice[s].astype(np.float64)
        V = abs(np.linalg.det(A))
        h = [V / np.linalg.norm(np.cross(A[(a + 1) % 3], A[(a + 2) % 3])) for a in range(3)]
        bound = [int(np.ceil(rc / x)) for x in h]
        assert np.all(g["max_abs_tau"] <= bound), (g["max_abs_tau"], bound)


# ------------------------------------------------------------------ invariants
def test_edge_symmetry():
    b = C.small_batch(40, seed=1)
    g = oracle.cutoff_graph(b.pos, b.lattice, b.struct_ptr, 5.0)
    es = _edge_set(g)
    assert g["n_edges"] % 2 == 0
    for (i, j, t) in es:
        assert (j, i, (-t[0], -t[1], -t[2])) in es


def _exact_inputs(rng, n):
    """Inputs exactly representable in FP32 and closed under the integer maps used below."""
    while True:
        lat = rng.integers(-24, 25, size=(3, 3)).astype(np.float64) / 4.0
        if abs(np.linalg.det(lat)) > 8.0:
            break
    pos = rng.integers(0, 64, size=(n, 3)).astype(np.float64) / 64.0
    return lat, pos


def _vec_multiset(g):
    return sorted((int(s), int(d), tuple(np.round(v, 9))) for s, d, v in
                  zip(g["src"], g["dst"], g["vec"]))


@pytest.mark.parametrize("seed", range(4))
def test_translation_invariance(seed):
    rng = np.random.default_rng(seed)
    lat, pos = _exact_inputs(rng, 5)
    ptr = np.array([0, 5], np.int32)
    shift = rng.integers(0, 64, size=3) / 64.0
    pos2 = pos + shift
    wrap = np.floor(pos2)
    pos2 = pos2 - wrap
    g1 = oracle.cutoff_graph(pos, lat[None], ptr, 5.0)
    g2 = oracle.cutoff_graph(pos2, lat[None], ptr, 5.0)
    assert _vec_multiset(g1) == _vec_multiset(g2)
    # tau shifts by the wrap integers: tau' = tau + wrap[j] - wrap[i]
    e1 = _edge_set(g1)
    e2 = {(i, j, tuple(int(x) for x in (np.array(t) - wrap[j] + wrap[i]))) for (i, j, t) in _edge_set(g2)}
    assert e1 == e2


@pytest.mark.parametrize("seed", range(4))
def test_unimodular_basis_change(seed):
    rng = np.random.default_rng(10 + seed)
    lat, pos = _exact_inputs(rng, 4)
    ptr = np.array([0, 4], np.int32)
    # U = product of integer shears and a swap: det = +-1
    U = np.eye(3)
    for _ in range(3):
        a, b = rng.choice(3, 2, replace=False)
        E = np.eye(3)
        E[a, b] = rng.integers(-2, 3)
        U = E @ U
    P = np.eye(3)[[1, 0, 2]]
    U = P @ U
    assert abs(round(np.linalg.det(U))) == 1
    Uinv = np.round(np.linalg.inv(U))
    lat2 = U @ lat
    pos2 = pos @ Uinv
    pos2 = pos2 - np.floor(pos2)
    assert np.abs(pos2 @ lat2 - (pos @ lat) - np.round((pos2 @ lat2 - pos @ lat) @ np.linalg.inv(lat)) @ lat).max() < 1e-9
    g1 = oracle.cutoff_graph(pos, lat[None], ptr, 4.5)
    g2 = oracle.cutoff_graph(pos2, lat2[None], ptr, 4.5)
    assert g1["n_edges"] > 0
    assert _vec_multiset(g1) == _vec_multiset(g2)


def test_rotation_invariance_of_counts():
    b = C.small_batch(10, seed=9)
    rng = np.random.default_rng(0)
    q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    lat2 = (b.lattice.astype(np.float64) @ q).astype(np.float32)
    g1 = oracle.cutoff_graph(b.pos, b.lattice, b.struct_ptr, 5.0)
    g2 = oracle.cutoff_graph(b.pos, lat2, b.struct_ptr, 5.0)
    # FP32 rounding of the rotated cell can flip edges only within ~1e-6 of r_c
    near = np.sum(np.abs(g1["dist"] - 5.0) < 1e-5) + np.sum(np.abs(g2["dist"] - 5.0) < 1e-5)
    assert len(_edge_set(g1) ^ _edge_set(g2)) <= near


def test_knn_cutoff_consistency_and_prefix():
    b = C.small_batch(48, seed=2)
    k = 12
    g = oracle.knn_graph(b.pos, b.lattice, b.struct_ptr, k)
    g1 = oracle.knn_graph(b.pos, b.lattice, b.struct_ptr, k + 1)
    n = b.n_atoms
    assert g["n_edges"] == k * n
    assert np.array_equal(g["row_ptr"], k * np.arange(n + 1))
    d = g["dist"].reshape(n, k)
    assert np.all(np.diff(d, axis=1) >= 0)
    assert np.allclose(d[:, -1], g["kth_dist"])
    # KNN(k) is a prefix of KNN(k+1)
    for name in ("dst", "dist"):
        assert np.array_equal(g[name].reshape(n, k), g1[name].reshape(n, k + 1)[:, :k])
    assert np.array_equal(g["tau"].reshape(n, k, 3), g1["tau"].reshape(n, k + 1, 3)[:, :k])
    # every image strictly closer than the k-th neighbour is in the KNN row, and nothing closer
    # than the k-th distance is missing
    rmax = float(g["kth_dist"].max())
    c = oracle.cutoff_graph(b.pos, b.lattice, b.struct_ptr, rmax + 1e-3)
    ks = _edge_set(g)
    dk = g["kth_dist"]
    for s_, d_, t_, dist in zip(c["src"], c["dst"], map(tuple, c["tau"].tolist()), c["dist"]):
        if dist < dk[s_]:
            assert (int(s_), int(d_), t_) in ks
    cs = _edge_set(c)
    assert ks <= cs


def test_expected_count_matches_density():
    # mean edges per atom -> (4/3) pi r^3 N / V  (statistical sanity, SURVEY 8(c) invariant (v))
    b = C.small_batch(300, seed=4)
    rc = 6.0
    g = oracle.cutoff_graph(b.pos, b.lattice, b.struct_ptr, rc)
    n = np.diff(b.struct_ptr).astype(np.float64)
    vol = np.abs(np.linalg.det(b.lattice.astype(np.float64)))
    expect = np.sum(n * (4.0 / 3.0) * np.pi * rc ** 3 * n / vol)
    assert abs(g["n_edges"] - expect) / expect < 0.03


# ------------------------------------------------------------------ special cases = library routines
def test_nearest_image_special_case():
    # h_min > 2 r_c: the graph is the minimum-image neighbour list
    b = C.supercell_batch(1, seed=1)
    n = min(b.n_atoms, 300)
    pos, lat = b.pos[:n], b.lattice[0].astype(np.float64)
    rc = 8.0
    g = oracle.cutoff_graph(pos, b.lattice[:1], np.array([0, n], np.int32), rc)
    p = pos.astype(np.float64)
    df = p[None, :, :] - p[:, None, :]
    t = -np.rint(df)
    v = (df + t) @ lat
    d = np.linalg.norm(v, axis=2)
    ii, jj = np.nonzero((d < rc) & ~np.eye(n, dtype=bool))
    want = set(zip(ii.tolist(), jj.tolist(), map(tuple, t[ii, jj].astype(int).tolist())))
    assert _edge_set(g) == want


def test_open_boundary_limit():
    # a huge cell: no image matters, the graph is the all-pairs d < r_c test
    rng = np.random.default_rng(7)
    n = 30
    cart = rng.uniform(0.0, 8.0, size=(n, 3))
    lat = (np.eye(3) * 1000.0).astype(np.float32)
    pos = (cart / 1000.0).astype(np.float32)
    g = oracle.cutoff_graph(pos, lat[None], np.array([0, n], np.int32), 3.0)
    c = pos.astype(np.float64) * 1000.0
    d = np.linalg.norm(c[None] - c[:, None], axis=2)
    ii, jj = np.nonzero((d < 3.0) & ~np.eye(n, dtype=bool))
    assert set(zip(g["src"].tolist(), g["dst"].tolist())) == set(zip(ii.tolist(), jj.tolist()))
    assert np.all(g["tau"] == 0)


# ------------------------------------------------------------------ API edges
def test_positions_outside_unit_cell():
    b = C.small_batch(5, seed=8)
    g0 = oracle.cutoff_graph(b.pos, b.lattice, b.struct_ptr, 5.0)
    shift = np.array([3.0, -2.0, 1.0], np.float32)
    pos2 = b.pos.copy()
    pos2[::2] += shift           # exact in FP32 only approximately; compare with tolerance on counts
    g1 = oracle.cutoff_graph(pos2, b.lattice, b.struct_ptr, 5.0)
    # offsets are relative to the coordinates as given: tau' = tau - shift_j + shift_i
    sh = np.zeros_like(b.pos, dtype=np.int64)
    sh[::2] = shift.astype(np.int64)
    e1 = {(i, j, tuple(int(x) for x in (np.array(t) + sh[j] - sh[i]))) for (i, j, t) in _edge_set(g1)}
    e0 = _edge_set(g0)
    near = np.sum(np.abs(g0["dist"] - 5.0) < 1e-5) + np.sum(np.abs(g1["dist"] - 5.0) < 1e-5)
    assert len(e0 ^ e1) <= near


def test_empty_and_degenerate_inputs():
    g = oracle.cutoff_graph(np.zeros((0, 3), np.float32), np.zeros((0, 3, 3), np.float32),
                            np.array([0], np.int32), 5.0)
    assert g["n_edges"] == 0 and g["row_ptr"].tolist() == [0]
    # a structure with zero atoms in the middle of a batch
    a, c = C.textbook("sc"), C.textbook("bcc_conv")
    empty = C.Batch(pos=np.zeros((0, 3), np.float32), lattice=np.eye(3, dtype=np.float32)[None],
                    struct_ptr=np.array([0, 0], np.int32))
    b = C.concat([a, empty, c])
    g = oracle.cutoff_graph(b.pos, b.lattice, b.struct_ptr, 1.01)
    assert np.diff(g["row_ptr"]).tolist() == [6, 14, 14]
    g = oracle.knn_graph(b.pos, b.lattice, b.struct_ptr, 3)
    assert g["n_edges"] == 9
    with pytest.raises(ValueError):
        oracle.cutoff_graph(np.zeros((1, 3), np.float32), np.zeros((1, 3, 3), np.float32),
                            np.array([0, 1], np.int32), 5.0)


def test_checker_accepts_oracle_and_rejects_damage():
    from oracle import check
    b = C.small_batch(8, seed=0)
    ref = oracle.cutoff_graph(b.pos, b.lattice, b.struct_ptr, 5.0)
    got = dict(n_edges=ref["n_edges"], row_ptr=ref["row_ptr"], src=ref["src"], dst=ref["dst"],
               offset=ref["tau"].astype(np.int8), vec=ref["vec"].astype(np.float32), dist=ref["dist"].astype(np.float32))
    rep = check.check_cutoff(b, 5.0, got, ref)
    assert rep["extra"] == 0 and rep["missing"] == 0
    bad = dict(got)
    bad["offset"] = got["offset"].copy()
    bad["offset"][3, 0] += 1
    with pytest.raises(AssertionError):
        check.check_cutoff(b, 5.0, bad, ref)
    bad = dict(got)
    bad["vec"] = got["vec"].copy()
    bad["vec"][5, 1] += 1e-3
    with pytest.raises(AssertionError):
        check.check_cutoff(b, 5.0, bad, ref)
    kref = oracle.knn_graph(b.pos, b.lattice, b.struct_ptr, 12)
    kgot = dict(n_edges=kref["n_edges"], row_ptr=kref["row_ptr"], src=kref["src"], dst=kref["dst"],
                offset=kref["tau"].astype(np.int8), vec=kref["vec"].astype(np.float32))
    rep = check.check_knn(b, 12, kgot, kref)
    assert rep["mismatched_entries"] == 0
    bad = dict(kgot)
    bad["dst"] = kgot["dst"].copy()
    n0 = b.struct_ptr[1]
    if n0 > 1:
        bad["dst"][0] = (bad["dst"][0] + 1) % n0
        with pytest.raises(AssertionError):
            check.check_knn(b, 12, bad, kref)
    # swapping two entries of different distance must be rejected
    bad = {k_: (v.copy() if isinstance(v, np.ndarray) else v) for k_, v in kgot.items()}
    row = slice(0, 12)
    d = kref["dist"][row]
    j = int(np.argmax(np.diff(d) > 1e-3))
    for name in ("dst", "offset", "vec"):
        a_ = bad[name][j].copy()
        bad[name][j] = bad[name][j + 1]
        bad[name][j + 1] = a_
    with pytest.raises(AssertionError):
        check.check_knn(b, 12, bad, kref)


# ------------------------------------------------------------------ statistics the oracle reports
def _spacings_np(lat):
    A = lat.astype(np.float64)
    V = np.abs(np.linalg.det(A))
    return np.stack([V / np.linalg.norm(np.cross(A[:, (a + 1) % 3], A[:, (a + 2) % 3]), axis=1) for a in range(3)], axis=1)


def test_n_box_and_n_evaluated_are_what_they_say():
    # n_box = sum_s N_s^2 prod_a (2 ceil(r/h_a) + 1) (the search box of BASELINE.json's north_star);
    # n_evaluated = the oracle's own box, one cell wider per side, minus the skipped (i, i, 0)
    b = C.small_batch(20, seed=6)
    r = 4.25
    g = oracle.cutoff_graph(b.pos, b.lattice, b.struct_ptr, r)
    h = _spacings_np(b.lattice)
    n = np.diff(b.struct_ptr).astype(np.float64)
    assert g["n_box"] == float(np.sum(n * n * np.prod(2 * np.ceil(r / h) + 1, axis=1)))
    assert g["n_evaluated"] == int(np.sum(n * n * np.prod(2 * (np.ceil(r / h) + 1) + 1, axis=1) - n))


# ------------------------------------------------------------------ per-atom cutoffs
def test_radii_equal_to_a_constant_is_the_cutoff_graph():
    b = C.small_batch(10, seed=12)
    ref = oracle.cutoff_graph(b.pos, b.lattice, b.struct_ptr, 4.0)
    got = oracle.cutoff_graph_radii(b.pos, b.lattice, b.struct_ptr, np.full(b.n_atoms, 4.0, np.float32))
    for key in ("row_ptr", "src", "dst", "tau"):
        assert np.array_equal(ref[key], got[key]), key


def test_radii_rows_are_the_rows_of_the_constant_cutoff_graphs():
    # row i of the per-atom graph = row i of the constant-cutoff graph with r_c = c_i (Def. 3 is per source)
    b = C.small_batch(6, seed=13)
    rng = np.random.default_rng(5)
    radii = rng.choice(np.array([2.5, 3.5, 5.0], np.float32), size=b.n_atoms)
    got = oracle.cutoff_graph_radii(b.pos, b.lattice, b.struct_ptr, radii)
    for r in (2.5, 3.5, 5.0):
        ref = oracle.cutoff_graph(b.pos, b.lattice, b.struct_ptr, r)
        for i in np.nonzero(radii == np.float32(r))[0]:
            a = slice(ref["row_ptr"][i], ref["row_ptr"][i + 1])
            g = slice(got["row_ptr"][i], got["row_ptr"][i + 1])
            assert np.array_equal(ref["dst"][a], got["dst"][g]) and np.array_equal(ref["tau"][a], got["tau"][g])
    assert np.all(got["dist"] < radii[got["src"]].astype(np.float64))


def test_radii_break_edge_symmetry_sc_two_atoms():
    # two atoms 0.5 apart along x in a unit cube; c_0 = 0.6 reaches atom 1 (at 0.5, both ways), c_1 = 0.4 reaches nothing
    b = C.Batch(pos=np.array([[0, 0, 0], [0.5, 0, 0]], np.float32), lattice=np.eye(3, dtype=np.float32)[None],
                struct_ptr=np.array([0, 2], np.int32))
    g = oracle.cutoff_graph_radii(b.pos, b.lattice, b.struct_ptr, np.array([0.6, 0.4], np.float32))
    assert list(np.diff(g["row_ptr"])) == [2, 0]
    assert sorted(map(tuple, g["tau"].tolist())) == [(-1, 0, 0), (0, 0, 0)] and list(g["dst"]) == [1, 1]
