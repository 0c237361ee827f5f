"""GPU edge cases of the C ABI: empty and ragged batches, coordinates outside [0,1), dense cells
that overflow the shared-memory stash and the translation-table tile, capacity overflow, error
reporting, the two-phase count, and the host-buffer entry points."""
import numpy as np
import pytest

import oracle
from oracle import check
from workloads import crystals as C

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def mg():
    import paper_2307_05380_b200 as m
    return m


@pytest.fixture(scope="module")
def ctx(mg):
    c = mg.Context(0)
    yield c
    c.close()


def _run_cutoff(mg, ctx, b, r_c, capacity=None):
    pos, lat, ptr = mg.to_device(b)
    out = ctx.cutoff_graph(pos, lat, ptr, r_c, capacity=capacity, dist=True)
    return out.to_numpy(), ctx.mg_check()


def test_empty_batch(mg, ctx):
    b = C.Batch(pos=np.zeros((0, 3), np.float32), lattice=np.zeros((0, 3, 3), np.float32),
                struct_ptr=np.zeros(1, np.int32))
    got, status = _run_cutoff(mg, ctx, b, 5.0, capacity=0)
    assert status == 0 and got["n_edges"] == 0 and got["row_ptr"].tolist() == [0]
    pos, lat, ptr = mg.to_device(b)
    out = ctx.knn_graph(pos, lat, ptr, 4).to_numpy()
    assert out["n_edges"] == 0 and out["row_ptr"].tolist() == [0]


def test_batch_of_empty_structures_only(mg, ctx):
    b = C.Batch(pos=np.zeros((0, 3), np.float32), lattice=np.tile(np.eye(3, dtype=np.float32) * 5, (7, 1, 1)),
                struct_ptr=np.zeros(8, np.int32))
    got, status = _run_cutoff(mg, ctx, b, 5.0, capacity=0)
    assert status == 0 and got["n_edges"] == 0 and got["row_ptr"].tolist() == [0]
    pos, lat, ptr = mg.to_device(b)
    out = ctx.knn_graph(pos, lat, ptr, 4).to_numpy()
    assert ctx.mg_check() == 0 and out["n_edges"] == 0 and out["row_ptr"].tolist() == [0]


def test_empty_structures_inside_batch(mg, ctx):
    a = C.small_batch(5, seed=7)
    empty = C.Batch(pos=np.zeros((0, 3), np.float32), lattice=np.eye(3, dtype=np.float32)[None] * 4,
                    struct_ptr=np.zeros(2, np.int32))
    b = C.concat([empty, a, empty, empty, a, empty])
    got, status = _run_cutoff(mg, ctx, b, 5.0)
    assert status == 0
    rep = check.check_cutoff(b, 5.0, got)
    assert rep["extra"] == 0 and rep["missing"] == 0
    pos, lat, ptr = mg.to_device(b)
    got = ctx.knn_graph(pos, lat, ptr, 7, dist=True).to_numpy()
    assert ctx.mg_check() == 0
    check.check_knn(b, 7, got)


def test_positions_outside_unit_cell(mg, ctx):
    b = C.small_batch(24, seed=11)
    rng = np.random.default_rng(5)
    shift = rng.integers(-3, 4, size=b.pos.shape).astype(np.float32)
    b2 = C.Batch(pos=(b.pos + shift + np.float32(0.25)).astype(np.float32), lattice=b.lattice,
                 struct_ptr=b.struct_ptr)
    got, status = _run_cutoff(mg, ctx, b2, 4.5)
    assert status == 0
    rep = check.check_cutoff(b2, 4.5, got)
    assert rep["extra"] == 0 and rep["missing"] == 0 and rep["n_edges"] > 0
    pos, lat, ptr = mg.to_device(b2)
    gk = ctx.knn_graph(pos, lat, ptr, 9, dist=True).to_numpy()
    assert ctx.mg_check() == 0
    check.check_knn(b2, 9, gk)


def test_dense_cells_overflow_stash_and_table(mg, ctx):
    # 3-4 A cells with a 12 A cutoff: > 1024 cells per box (several table tiles) and thousands of
    # edges per row (rows do not fit their stash segment -> re-search path)
    items = []
    for s in range(6):
        rng = np.random.default_rng(100 + s)
        n = int(rng.integers(1, 21))
        cell = np.diag(rng.uniform(3.0, 4.0, 3)).astype(np.float32)
        cell[1, 0] = np.float32(rng.uniform(-1, 1))
        cell[2, 1] = np.float32(rng.uniform(-1, 1))
        items.append((cell, rng.random((n, 3), dtype=np.float32)))
    b = C._assemble(items)
    got, status = _run_cutoff(mg, ctx, b, 12.0)
    assert status == 0
    rep = check.check_cutoff(b, 12.0, got)
    assert rep["extra"] == 0 and rep["missing"] == 0
    assert np.diff(got["row_ptr"]).max() > 1000


def test_large_structure_with_tiled_table(mg, ctx):
    # 280 atoms (above the shared-memory staging limit) in a 5 A cell with a 15.5 A cutoff: the
    # per-pair sub-box has 7^3 = 343 cells (several table tiles) and a source row has > 256 pairs
    rng = np.random.default_rng(3)
    cell = (np.diag([5.0, 5.2, 5.4]) + rng.uniform(-0.3, 0.3, (3, 3))).astype(np.float32)
    b = C.Batch(pos=rng.random((280, 3), dtype=np.float32), lattice=cell[None],
                struct_ptr=np.array([0, 280], np.int32))
    got, status = _run_cutoff(mg, ctx, b, 15.5)
    assert status == 0
    rep = check.check_cutoff(b, 15.5, got)
    assert rep["extra"] == 0 and rep["missing"] == 0 and rep["n_edges"] > 5_000_000


def test_more_than_32_prep_blocks(mg, ctx):
    # above 4096 structures the search-bounds kernel scans its block sums itself (last block out);
    # below, the graph kernels scan the raw sums: this batch takes the first path
    part = C.small_batch(300, seed=17)
    b = C.concat([part] * 15)                       # 4500 structures
    got, status = _run_cutoff(mg, ctx, b, 4.0)
    assert status == 0
    rep = check.check_cutoff(b, 4.0, got)
    assert rep["extra"] == 0 and rep["missing"] == 0 and rep["n_edges"] > 100_000
    pos, lat, ptr = mg.to_device(b)
    gk = ctx.knn_graph(pos, lat, ptr, 8, dist=True).to_numpy()
    assert ctx.mg_check() == 0
    check.check_knn(b, 8, gk)


def test_mask_scratch_exhausted(mg, monkeypatch):
    # The count launch keeps the hit masks of a range in a fixed scratch (4096 words per warp); a
    # range with more blocks x words than that is evaluated again by the emit launch.  Real batches
    # reach this only above ~1e8 edges, so the test shrinks the scratch through the library's knob:
    # 0 words (everything evaluated twice), 8 and 40 (the switch happens in the middle of a range, for
    # tables of 1, 2 and up to 8 words per pair) — single-image structures included.
    small = C.small_batch(48, seed=5)
    big = C.config_batch(3, n_struct=1, seed=2)
    b = C.concat([small, big, small])
    want6 = None
    for words in ("0", "8", "40", "4096"):
        monkeypatch.setenv("MATGRAPH_MASK_WORDS", words)
        c = mg.Context(0)
        try:
            for r_c in (3.0, 6.0, 9.0):
                pos, lat, ptr = mg.to_device(b)
                got = c.cutoff_graph(pos, lat, ptr, r_c, dist=True).to_numpy()
                assert c.mg_check() == 0
                rep = check.check_cutoff(b, r_c, got)
                assert rep["extra"] == 0 and rep["missing"] == 0
                if r_c == 6.0:
                    key = (got["n_edges"], got["row_ptr"].tobytes())
                    want6 = want6 or key
                    assert key == want6
        finally:
            c.close()


def test_capacity_overflow_reports_required_count(mg, ctx):
    b = C.small_batch(16, seed=2)
    full, status = _run_cutoff(mg, ctx, b, 5.0)
    assert status == 0
    need = full["n_edges"]
    cap = need // 2
    got, status = _run_cutoff(mg, ctx, b, 5.0, capacity=cap)
    assert status == 6                       # MG_ERR_CAPACITY
    assert got["n_edges"] == need            # the required count is still reported
    assert np.array_equal(got["row_ptr"], full["row_ptr"])
    # edges below the capacity are complete rows' worth of valid data
    keep = full["src"] < 0
    keep[:cap] = True
    fk = np.stack([full["src"][:cap], full["dst"][:cap]], 1)
    gk = np.stack([got["src"], got["dst"]], 1)
    assert gk.shape[0] == cap
    # same multiset per row prefix is not guaranteed (row order is free): compare the src column
    assert np.array_equal(fk[:, 0], gk[:, 0])
    assert ctx.mg_check() == 0               # status word was cleared


def test_invalid_lattices_are_reported(mg, ctx):
    b = C.small_batch(6, seed=4)
    lat = b.lattice.copy()
    lat[2] = 0.0                              # singular
    bad = C.Batch(pos=b.pos, lattice=lat, struct_ptr=b.struct_ptr)
    got, status = _run_cutoff(mg, ctx, bad, 5.0)
    assert status == 3                        # MG_ERR_SINGULAR_LATTICE
    rows = np.diff(got["row_ptr"])
    s2 = slice(b.struct_ptr[2], b.struct_ptr[3])
    assert np.all(rows[s2] == 0)              # the invalid structure emits nothing
    good = np.ones(b.n_atoms, bool)
    good[s2] = False
    ref = oracle.cutoff_graph(b.pos, b.lattice, b.struct_ptr, 5.0)
    assert np.array_equal(rows[good], np.diff(ref["row_ptr"])[good])
    lat = b.lattice.copy()
    lat[1, 0, 0] = np.nan
    bad = C.Batch(pos=b.pos, lattice=lat, struct_ptr=b.struct_ptr)
    _, status = _run_cutoff(mg, ctx, bad, 5.0)
    assert status == 4                        # MG_ERR_NONFINITE


def test_offset_range_error(mg, ctx):
    # plane spacing 0.05 A with r_c = 8 would need |tau| = 160 > 127
    cell = np.diag([0.05, 5.0, 5.0]).astype(np.float32)
    b = C.Batch(pos=np.zeros((1, 3), np.float32), lattice=cell[None], struct_ptr=np.array([0, 1], np.int32))
    _, status = _run_cutoff(mg, ctx, b, 8.0, capacity=16)
    assert status == 5                        # MG_ERR_OFFSET_RANGE


def test_invalid_arguments(mg, ctx):
    b = C.small_batch(2, seed=0)
    pos, lat, ptr = mg.to_device(b)
    out = mg.Edges.allocate(b.n_atoms, 10, "cuda")
    with pytest.raises(mg.MatGraphError):
        ctx.mg_cutoff_graph(pos, lat, ptr, -1.0, out)
    with pytest.raises(mg.MatGraphError):
        ctx.mg_cutoff_graph(pos, lat, ptr, float("nan"), out)
    with pytest.raises(mg.MatGraphError):
        ctx.mg_knn_graph(pos, lat, ptr, 0, out)
    with pytest.raises(mg.MatGraphError):
        ctx.mg_knn_graph(pos, lat, ptr, 65, out)
    small = mg.Edges.allocate(b.n_atoms, 3, "cuda")
    with pytest.raises(mg.MatGraphError):     # capacity < k * n_atoms
        ctx.mg_knn_graph(pos, lat, ptr, 4, small)


def test_count_matches_graph(mg, ctx):
    b = C.small_batch(64, seed=9)
    pos, lat, ptr = mg.to_device(b)
    n = ctx.mg_cutoff_count(pos, lat, ptr, 5.5)
    assert n == oracle.cutoff_graph(b.pos, b.lattice, b.struct_ptr, 5.5)["n_edges"]


def test_host_entry_points(mg, ctx):
    b = C.small_batch(32, seed=5)
    ref = oracle.cutoff_graph(b.pos, b.lattice, b.struct_ptr, 5.0)
    got = ctx.mg_cutoff_graph_host(b.pos, b.lattice, b.struct_ptr, 5.0, ref["n_edges"] + 10, dist=True)
    assert got["status"] == 0
    rep = check.check_cutoff(b, 5.0, got, ref)
    assert rep["extra"] == 0 and rep["missing"] == 0
    gk = ctx.mg_knn_graph_host(b.pos, b.lattice, b.struct_ptr, 12, dist=True)
    assert gk["status"] == 0
    check.check_knn(b, 12, gk)


def test_repeated_calls_are_deterministic_sets(mg, ctx):
    b = C.small_batch(128, seed=6)
    a, _ = _run_cutoff(mg, ctx, b, 6.0)
    c, _ = _run_cutoff(mg, ctx, b, 6.0)
    assert a["n_edges"] == c["n_edges"] and np.array_equal(a["row_ptr"], c["row_ptr"])
    ka = check._keys(a["src"], a["dst"], a["offset"])
    kc = check._keys(c["src"], c["dst"], c["offset"])
    assert np.array_equal(np.sort(ka), np.sort(kc))


# ------------------------------------------------------------------ the one-launch scan kernel on every kind of batch
# mg_cutoff_graph picks its kernels per call (cut_scan.cuh for batches of large structures, the count +
# emit pair otherwise); MATGRAPH_FUSED=1 sends every batch through the scan kernel.
@pytest.fixture()
def scan_ctx(mg, monkeypatch):
    monkeypatch.setenv("MATGRAPH_FUSED", "1")
    c = mg.Context(0)
    yield c
    c.close()


def test_scan_kernel_small_cells_and_mixed_batches(mg, scan_ctx):
    small = C.small_batch(40, seed=8)
    rng = np.random.default_rng(3)
    cell = (np.diag([9.0, 10.0, 11.0]) + rng.uniform(-1, 1, (3, 3))).astype(np.float32)
    big = C.Batch(pos=rng.random((150, 3), dtype=np.float32), lattice=cell[None], struct_ptr=np.array([0, 150], np.int32))
    empty = C.Batch(pos=np.zeros((0, 3), np.float32), lattice=np.eye(3, dtype=np.float32)[None], struct_ptr=np.array([0, 0], np.int32))
    for b, rc in ((C.config_batch(0), 5.0), (C.concat([small, empty, big, small]), 6.5), (C.config_batch(2, n_struct=300), 6.0)):
        pos, lat, ptr = mg.to_device(b)
        got = scan_ctx.cutoff_graph(pos, lat, ptr, rc, dist=True).to_numpy()
        assert scan_ctx.mg_check() == 0
        rep = check.check_cutoff(b, rc, got)
        assert rep["extra"] == 0 and rep["missing"] == 0, rep


def test_scan_kernel_pool_exhausted_and_dense_rows(mg, monkeypatch):
    # a pool of a few chunks (test knob): warps whose codes do not fit list their rows a second time and write edge
    # by edge; dense cells: blocks with more hits than the stash holds go in passes of consecutive lanes
    monkeypatch.setenv("MATGRAPH_FUSED", "1")
    items = []
    for s in range(4):
        rng = np.random.default_rng(200 + s)
        n = int(rng.integers(3, 21))
        cell = np.diag(rng.uniform(3.0, 4.0, 3)).astype(np.float32)
        cell[1, 0] = np.float32(rng.uniform(-1, 1))
        items.append((cell, rng.random((n, 3), dtype=np.float32)))
    dense = C._assemble(items)
    b = C.concat([C.small_batch(30, seed=6), dense])
    ref = None
    for words in ("0", "3", "40", "4096"):
        monkeypatch.setenv("MATGRAPH_MASK_WORDS", words)
        c = mg.Context(0)
        try:
            pos, lat, ptr = mg.to_device(b)
            got = c.cutoff_graph(pos, lat, ptr, 7.0, dist=True).to_numpy()
            assert c.mg_check() == 0
            rep = check.check_cutoff(b, 7.0, got)
            assert rep["extra"] == 0 and rep["missing"] == 0, (words, rep)
            key = (got["n_edges"], got["row_ptr"].tobytes())
            ref = ref or key
            assert key == ref
        finally:
            c.close()


def test_scan_kernel_capacity_and_count(mg, scan_ctx):
    b = C.small_batch(16, seed=2)
    pos, lat, ptr = mg.to_device(b)
    need = scan_ctx.mg_cutoff_count(pos, lat, ptr, 5.0)
    full = scan_ctx.cutoff_graph(pos, lat, ptr, 5.0, capacity=need).to_numpy()
    assert scan_ctx.mg_check() == 0 and full["n_edges"] == need
    got = scan_ctx.cutoff_graph(pos, lat, ptr, 5.0, capacity=need // 2 + 1).to_numpy()
    assert scan_ctx.mg_check() == 6 and got["n_edges"] == need
    assert np.array_equal(got["row_ptr"], full["row_ptr"])
    m = need // 2 + 1
    assert np.array_equal(got["src"], full["src"][:m])
    kg = check._keys(got["src"], got["dst"], got["offset"])
    assert set(kg.tolist()) <= set(check._keys(full["src"], full["dst"], full["offset"]).tolist())


# ---- K2: the cell list of large structures (csrc/cut_bins.cuh) --------------------------------------
def _big_cell(rng, lengths, n, skew=0.0, shift=0.0):
    cell = np.diag(np.asarray(lengths, np.float64))
    cell[1, 0] = skew * lengths[0]
    cell[2, 1] = -0.5 * skew * lengths[1]
    x = rng.random((n, 3), dtype=np.float32) + np.float32(shift)
    return cell.astype(np.float32), x.astype(np.float32)


def test_cell_list_shapes_and_wraps(mg, ctx):
    # slabs on three, two, one and no axis (cell lengths from 3 to 12 cutoffs), skewed cells, coordinates on the
    # boundary of the cell (0, 1 - ulp, exactly representable slab edges) and outside it, in one batch with small
    # structures: every structure above 64 atoms in the minimum-image regime goes through the binned rows
    rng = np.random.default_rng(77)
    rc = 4.0
    items = [_big_cell(rng, (50.0, 40.0, 30.0), 900),               # 12 / 10 / 7 cutoffs: slabs on all axes
             _big_cell(rng, (45.0, 13.0, 36.0), 500, skew=0.3),     # middle axis short: one slab there
             _big_cell(rng, (12.0, 11.0, 48.0), 300),               # only the last axis has slabs
             _big_cell(rng, (11.0, 12.0, 13.0), 200, skew=0.2),     # no slabs: one bin
             _big_cell(rng, (64.0, 64.0, 64.0), 150),               # more bins than atoms: slabs are merged
             _big_cell(rng, (40.0, 40.0, 40.0), 700, shift=-2.0)]   # coordinates in [-2, -1): wrapped
    edge = np.array([[0.0, 0.0, 0.0], [1.0 - 2.0 ** -24, 0.5, 0.25], [0.125, 0.875, 1.0 - 2.0 ** -24],
                     [0.5, 0.0, 0.75], [2.0 ** -24, 0.999999, 0.0]], np.float32)
    items[0][1][:5] = edge
    b = C.concat([C.small_batch(5, seed=4), C._assemble(items), C.small_batch(3, seed=5)])
    got, status = _run_cutoff(mg, ctx, b, rc)
    assert status == 0
    rep = check.check_cutoff(b, rc, got)
    assert rep["extra"] == 0 and rep["missing"] == 0 and rep["n_edges"] > 10000, rep
    # the same call again: same arrays, bit for bit (the cell list is built in index order, no atomics race)
    again, _ = _run_cutoff(mg, ctx, b, rc)
    for k in ("row_ptr", "src", "dst", "offset", "vec", "dist"):
        assert np.array_equal(got[k], again[k]), k


def test_cell_list_far_atoms_radii_and_small_pool(mg, monkeypatch):
    rng = np.random.default_rng(78)
    cell, x = _big_cell(rng, (30.0, 32.0, 34.0), 400, skew=0.1)
    far = x.copy()
    far[7, 0] += np.float32(70.0)                                   # 70 cells away: the structure takes the generic rows
    near = C._assemble([(cell, x)])
    b_far = C._assemble([(cell, far)])
    mid = x.copy()
    mid[11, 1] += np.float32(20.0)                                  # 20 cells away: outside the 15 cells a sorted entry can pack
    mid[12, 2] -= np.float32(15.0)                                  # ... and exactly at its edge
    b_mid = C._assemble([(cell, mid)])
    c = mg.Context(0)
    try:
        pos, lat, ptr = mg.to_device(b_far)
        got = c.cutoff_graph(pos, lat, ptr, 4.5, dist=True).to_numpy()
        assert c.mg_check() == 0                                    # |tau| = 70 still fits int8
        rep = check.check_cutoff(b_far, 4.5, got)
        assert rep["extra"] == 0 and rep["missing"] == 0 and np.abs(got["offset"]).max() >= 69
        pos, lat, ptr = mg.to_device(b_mid)
        got = c.cutoff_graph(pos, lat, ptr, 4.5, dist=True).to_numpy()
        assert c.mg_check() == 0
        rep = check.check_cutoff(b_mid, 4.5, got)
        assert rep["extra"] == 0 and rep["missing"] == 0 and np.abs(got["offset"]).max() >= 19
        bad = far.copy()
        bad[9, 1] = np.float32(np.nan)
        pos, lat, ptr = mg.to_device(C._assemble([(cell, bad)]))
        c.cutoff_graph(pos, lat, ptr, 4.5, dist=True)
        assert c.mg_check() != 0                                    # a NaN coordinate is reported
        # per-atom cutoffs on a binned structure
        radii = rng.uniform(2.0, 4.5, size=near.n_atoms).astype(np.float32)
        pos, lat, ptr = mg.to_device(near)
        import torch
        ref = oracle.cutoff_graph_radii(near.pos, near.lattice, near.struct_ptr, radii)
        out = mg.Edges.allocate(near.n_atoms, int(ref["n_edges"]) + 8, pos.device, dist=True)
        got = c.mg_cutoff_graph_radii(pos, lat, ptr, torch.from_numpy(radii).to(pos.device), out).to_numpy()
        assert c.mg_check() == 0
        kg = np.sort(check._keys(got["src"], got["dst"], got["offset"]))
        kr = np.sort(check._keys(ref["src"], ref["dst"], ref["tau"]))
        assert np.array_equal(kg, kr) and np.array_equal(got["row_ptr"], ref["row_ptr"])
    finally:
        c.close()
    # a pool of three chunks: the warps list their rows again and write edge by edge
    monkeypatch.setenv("MATGRAPH_MASK_WORDS", "3")
    c = mg.Context(0)
    try:
        pos, lat, ptr = mg.to_device(near)
        got = c.cutoff_graph(pos, lat, ptr, 6.0, dist=True).to_numpy()
        assert c.mg_check() == 0
        rep = check.check_cutoff(near, 6.0, got)
        assert rep["extra"] == 0 and rep["missing"] == 0 and rep["n_edges"] > 3 * 512, rep
    finally:
        c.close()


def test_knn_atoms_more_than_127_cells_apart(mg, ctx):
    # two atoms in a 3 A cube, the second one given 100 / 130 cells along x: the nearest neighbours of atom 0 are images
    # of atom 1 at 2.6 A, ahead of its own images at 3 A.  At 100 cells their offsets fit int8 and the rows are the
    # oracle's; at 130 they do not, and the call must say so — k = 6 is the case where atom 0's own six images would
    # fill the row and hide the missing pair.
    cell = np.diag([3.0, 3.0, 3.0]).astype(np.float32)
    for shift, expect in ((100.0, 0), (130.0, 5)):
        x = np.array([[0.0, 0.0, 0.0], [0.5 + shift, 0.5, 0.5]], np.float32)
        b = C._assemble([(cell, x)])
        pos, lat, ptr = mg.to_device(b)
        for k in (6, 8, 14):
            got = ctx.knn_graph(pos, lat, ptr, k, dist=True).to_numpy()
            assert ctx.mg_check() == expect, (shift, k)              # 5: MG_ERR_OFFSET_RANGE
            if expect == 0:
                check.check_knn(b, k, got)
                assert np.abs(got["offset"]).max() >= 100


@pytest.mark.parametrize("env", [{"MATGRAPH_NO_PDL": "1"}, {"MATGRAPH_LEGACY": "1"},
                                 {"MATGRAPH_FUSED": "1", "MATGRAPH_WRITE_KERNEL": "1"},
                                 {"MATGRAPH_FUSED": "1", "MATGRAPH_NO_COOP": "1"},
                                 {"MATGRAPH_FUSED": "1", "MATGRAPH_NO_PDL": "1"}])
def test_launch_knobs_give_the_same_graphs(mg, monkeypatch, env):
    # the knobs of include/matgraph.h pick other launches for the same graphs: small cells, a supercell (cell list) and a
    # dense cell in one batch, cutoff and KNN against the oracle under each of them
    for key, val in env.items():
        monkeypatch.setenv(key, val)
    rng = np.random.default_rng(12)
    dense = C._assemble([(np.diag([3.2, 3.4, 3.6]).astype(np.float32), rng.random((9, 3), dtype=np.float32))])
    batches = [C.concat([C.small_batch(20, seed=21), dense, C.small_batch(4, seed=22)]), C.supercell_batch(2, seed=3)]
    c = mg.Context(0)
    try:
        for b, rc, k in ((batches[0], 6.0, 12), (batches[1], 5.0, 0)):
            pos, lat, ptr = mg.to_device(b)
            got = c.cutoff_graph(pos, lat, ptr, rc, dist=True).to_numpy()
            assert c.mg_check() == 0
            rep = check.check_cutoff(b, rc, got)
            assert rep["extra"] == 0 and rep["missing"] == 0 and rep["n_edges"] > 0, (env, rep)
            if k:
                gk = c.knn_graph(pos, lat, ptr, k, dist=True).to_numpy()
                assert c.mg_check() == 0
                check.check_knn(b, k, gk)
    finally:
        c.close()
