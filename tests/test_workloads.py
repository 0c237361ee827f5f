"""The seeded input recipe (workloads/crystals.py): determinism, prefix property, the ranges of
BASELINE.json configs[0..4] and the minimum-distance rejection (checked through the oracle, which
the generator does not import)."""
import numpy as np

import oracle
from workloads import crystals as C


def _spacings(lat):
    A = lat.astype(np.float64)
    V = abs(np.linalg.det(A))
    return np.array([V / np.linalg.norm(np.cross(A[(a + 1) % 3], A[(a + 2) % 3])) for a in range(3)])


def test_deterministic_and_prefix():
    a = C.small_batch(12, seed=0)
    b = C.small_batch(12, seed=0)
    c = C.small_batch(5, seed=0)
    d = C.small_batch(12, seed=1)
    assert np.array_equal(a.pos, b.pos) and np.array_equal(a.lattice, b.lattice)
    assert np.array_equal(a.lattice[:5], c.lattice) and np.array_equal(a.pos[:c.n_atoms], c.pos)
    assert not np.array_equal(a.lattice, d.lattice)
    assert a.pos.dtype == np.float32 and a.lattice.dtype == np.float32 and a.struct_ptr.dtype == np.int32


def test_small_family_ranges():
    b = C.small_batch(200, seed=0)
    n = np.diff(b.struct_ptr)
    assert n.min() >= 1 and n.max() <= 20 and len(set(n.tolist())) > 10
    lengths = np.linalg.norm(b.lattice.astype(np.float64), axis=2)
    assert lengths.min() >= 3.0 - 1e-5 and lengths.max() <= 10.0 + 1e-5
    A = b.lattice.astype(np.float64)
    for (i, j) in ((1, 2), (0, 2), (0, 1)):
        cosang = np.einsum("sc,sc->s", A[:, i], A[:, j]) / (lengths[:, i] * lengths[:, j])
        ang = np.degrees(np.arccos(cosang))
        assert ang.min() >= 60.0 - 1e-3 and ang.max() <= 120.0 + 1e-3
    assert min(_spacings(l).min() for l in b.lattice) >= 1.0
    assert b.pos.min() >= 0.0 and b.pos.max() < 1.0
    # no periodic pair (self images included) closer than 1.0 A
    assert oracle.cutoff_graph(b.pos, b.lattice, b.struct_ptr, 1.0)["n_edges"] == 0
    # ... while plenty of pairs are closer than 2 A: the rejection is not vacuous
    assert oracle.cutoff_graph(b.pos, b.lattice, b.struct_ptr, 2.0)["n_edges"] > 0


def test_supercell_family():
    b = C.supercell_batch(2, seed=0)
    n = np.diff(b.struct_ptr)
    assert n.min() >= 500 and n.max() <= 2000
    vol = np.abs(np.linalg.det(b.lattice.astype(np.float64)))
    assert np.all(np.abs(n / vol - 0.08) < 1e-3)
    assert min(_spacings(l).min() for l in b.lattice) > 16.0     # > 2 r_c: nearest image regime
    assert oracle.cutoff_graph(b.pos, b.lattice, b.struct_ptr, 1.2)["n_edges"] == 0


def test_skewed_family_and_walk():
    b = C.skewed_batch(64, seed=0)
    n = np.diff(b.struct_ptr)
    assert n.min() >= 2 and n.max() <= 20
    assert min(_spacings(l).min() for l in b.lattice) >= 1.0
    steps = list(C.walk(b, 6, seed=0))
    again = list(C.walk(b, 6, seed=0))
    assert len(steps) == 6
    for s, t in zip(steps, again):
        assert np.array_equal(s.pos, t.pos) and np.array_equal(s.lattice, t.lattice)
        assert s.pos.min() >= 0.0 and s.pos.max() < 1.0
        assert min(_spacings(l).min() for l in s.lattice) >= 0.5
        assert np.array_equal(s.struct_ptr, b.struct_ptr)
    # cumulative walk: step t differs from step t-1 by about one step of noise
    d01 = np.abs(steps[1].lattice - steps[0].lattice).max()
    d05 = np.abs(steps[5].lattice - steps[0].lattice).max()
    assert 0 < d01 < 0.6 and d05 > d01 * 0.5
    rel = np.abs(steps[0].lattice.astype(np.float64) - b.lattice) .max() / np.abs(b.lattice).max()
    assert rel < 0.07


def test_config_table():
    assert C.config_batch(0).n_struct == 8
    assert C.config_batch(1, n_struct=16).n_struct == 16
    assert C.CONFIGS[2]["n_struct"] == 4096 and C.CONFIGS[2]["r_c"] == 6.0 and C.CONFIGS[2]["k"] == 12
    assert C.CONFIGS[4]["k"] == 24 and C.CONFIGS[4]["n_steps"] == 100


def test_paper_scale_family():
    b = C.paper_scale_batch(64, seed=1)
    n = np.diff(b.struct_ptr)
    assert n.min() >= 1 and n.max() <= 64 and n.max() > 20
    b2 = C.paper_scale_batch(32, seed=1)                      # smaller batches are prefixes
    assert np.array_equal(b2.pos, b.pos[:b2.n_atoms]) and np.array_equal(b2.lattice, b.lattice[:32])
    vol = np.abs(np.linalg.det(b.lattice.astype(np.float64)))
    assert 8.0 < np.median(vol / n) < 60.0                    # tens of cubic Angstrom per atom
