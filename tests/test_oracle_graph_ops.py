"""Pins of oracle/graph_ops.py (CPU): the symmetric graph and the triplets Gamma_2
 against things fixed by the definitions, not by the oracle's own code: hand-made
graphs, the closed-form counts of the simple cubic lattice, set algebra on Python tuples, and
itertools.permutations on a tiny graph."""
import itertools

import numpy as np

import oracle
from oracle import graph_ops as G
from workloads import crystals as C


def _edge_set(g):
    return {(int(s), int(d), *map(int, t)) for s, d, t in zip(g["src"], g["dst"], np.asarray(g["tau"]).reshape(-1, 3))}


def test_symmetrize_hand_example():
    # one directed edge 0 -> 1 in cell (1, 0, -2): the reverse 1 -> 0 in cell (-1, 0, 2) is added, vec negated
    g = G.symmetrize(2, [0], [1], [[1, 0, -2]], vec=[[0.5, -1.0, 2.0]], dist=[2.29])
    assert g["n_edges"] == 2 and list(g["row_ptr"]) == [0, 1, 2]
    assert _edge_set(g) == {(0, 1, 1, 0, -2), (1, 0, -1, 0, 2)}
    assert np.allclose(g["vec"][1], [-0.5, 1.0, -2.0]) and g["dist"][1] == 2.29


def test_symmetrize_keeps_a_symmetric_graph():
    # a periodic self image and its partner are each other's reverse: nothing to add
    g = G.symmetrize(1, [0, 0], [0, 0], [[1, 0, 0], [-1, 0, 0]])
    assert g["n_edges"] == 2


def test_symmetrize_sc_knn6_is_already_symmetric():
    # simple cubic, one atom, k = 6: the six nearest images come in +-tau pairs
    b = C.textbook("sc")
    k = oracle.knn_graph(b.pos, b.lattice, b.struct_ptr, 6)
    g = G.symmetrize(b.n_atoms, k["src"], k["dst"], k["tau"])
    assert g["n_edges"] == 6 and _edge_set(g) == _edge_set(k)


def test_symmetrize_cutoff_graph_is_a_fixed_point():
    # Def. 3 with a constant cutoff is symmetric ((i,j,tau) <-> (j,i,-tau) have the same length)
    b = C.small_batch(5, seed=4)
    c = oracle.cutoff_graph(b.pos, b.lattice, b.struct_ptr, 4.5)
    g = G.symmetrize(b.n_atoms, c["src"], c["dst"], c["tau"])
    assert g["n_edges"] == c["n_edges"] and _edge_set(g) == _edge_set(c)


def test_symmetrize_is_the_smallest_symmetric_superset():
    b = C.small_batch(12, seed=9)
    k = oracle.knn_graph(b.pos, b.lattice, b.struct_ptr, 5)
    g = G.symmetrize(b.n_atoms, k["src"], k["dst"], k["tau"], vec=k["vec"], dist=k["dist"])
    have = _edge_set(k)
    rev = {(d, s, -t0, -t1, -t2) for (s, d, t0, t1, t2) in have}
    out = _edge_set(g)
    assert out == have | rev and g["n_edges"] == len(have | rev)          # union, every edge once
    assert all((d, s, -a, -b_, -c) in out for (s, d, a, b_, c) in out)     # symmetric
    assert g["n_edges"] > k["n_edges"]                                    # KNN is not symmetric in general
    # CSR by source and vec of an added edge = - vec of its partner
    assert np.array_equal(g["src"], np.repeat(np.arange(b.n_atoms), np.diff(g["row_ptr"])))
    lookup = {(int(s), int(d), *map(int, t)): v for s, d, t, v in zip(g["src"], g["dst"], g["tau"], g["vec"])}
    for (s, d, a, b_, c), v in lookup.items():
        assert np.allclose(lookup[(d, s, -a, -b_, -c)], -np.asarray(v))


def test_triplets_tiny_graph_equals_permutations():
    row_ptr = np.array([0, 3, 3, 4, 6])        # degrees 3, 0, 1, 2
    t = G.triplets(row_ptr)
    expect = []
    for i in range(4):
        expect += list(itertools.permutations(range(row_ptr[i], row_ptr[i + 1]), 2))
    assert list(zip(t["edge_a"].tolist(), t["edge_b"].tolist())) == expect
    assert list(t["tri_ptr"]) == [0, 6, 6, 6, 8] and t["n_triplets"] == 8


def test_triplets_count_formula_and_sc():
    b = C.textbook("sc")
    k = oracle.knn_graph(b.pos, b.lattice, b.struct_ptr, 6)
    t = G.triplets(k["row_ptr"])
    assert t["n_triplets"] == 6 * 5                      # 30 ordered pairs of the six nearest neighbours
    b2 = C.small_batch(6, seed=2)
    c = oracle.cutoff_graph(b2.pos, b2.lattice, b2.struct_ptr, 4.0)
    t2 = G.triplets(c["row_ptr"])
    d = np.diff(c["row_ptr"])
    assert t2["n_triplets"] == int(np.sum(d * (d - 1)))
    # both edges of a triplet have the same source, and no pair repeats
    assert np.array_equal(c["src"][t2["edge_a"]], c["src"][t2["edge_b"]]) and np.all(t2["edge_a"] != t2["edge_b"])
    assert len(set(zip(t2["edge_a"].tolist(), t2["edge_b"].tolist()))) == t2["n_triplets"]
