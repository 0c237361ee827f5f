"""GPU parity: the CUDA path (through the C ABI binding) against the FP64 oracle, element by
element on the same seeded inputs, with the acceptance rules of BASELINE.json north_star
(oracle/check.py): bit-exact canonical edge sets outside a 1e-5 A band around r_c (the kernels
decide the band in FP64, so in practice the sets are identical), KNN rows in oracle order up to
the 1e-5 A tie band, vec / dist within 1e-5 A absolute."""
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


def _cutoff(mg, ctx, batch, r_c, dist=True, capacity=None):
    pos, lat, ptr = mg.to_device(batch)
    out = ctx.cutoff_graph(pos, lat, ptr, r_c, capacity=capacity, dist=dist)
    got = out.to_numpy()
    status = ctx.mg_check()
    return got, status


def _knn(mg, ctx, batch, k, dist=True):
    pos, lat, ptr = mg.to_device(batch)
    out = ctx.knn_graph(pos, lat, ptr, k, dist=dist)
    got = out.to_numpy()
    status = ctx.mg_check()
    return got, status


# ------------------------------------------------------------------ the BASELINE.json configs
def test_config0_cutoff(mg, ctx):
    b = C.config_batch(0)
    got, status = _cutoff(mg, ctx, b, 5.0)
    assert status == 0
    rep = check.check_cutoff(b, 5.0, got)
    assert rep["extra"] == 0 and rep["missing"] == 0, rep    # FP64 window => identical sets
    assert rep["n_edges"] == rep["n_ref"] > 0


def test_config1_knn(mg, ctx):
    b = C.config_batch(1)
    got, status = _knn(mg, ctx, b, 12)
    assert status == 0
    rep = check.check_knn(b, 12, got)
    assert rep["n_edges"] == 12 * b.n_atoms


@pytest.fixture(scope="module")
def batch2():
    return C.config_batch(2)


def test_config2_cutoff_full(mg, ctx, batch2):
    got, status = _cutoff(mg, ctx, batch2, 6.0)
    assert status == 0
    rep = check.check_cutoff(batch2, 6.0, got)
    assert rep["extra"] == 0 and rep["missing"] == 0, rep
    assert rep["n_edges"] > 3_000_000


def test_config2_knn_full(mg, ctx, batch2):
    got, status = _knn(mg, ctx, batch2, 12)
    assert status == 0
    rep = check.check_knn(batch2, 12, got)
    assert rep["n_edges"] == 12 * batch2.n_atoms
    # FP64 re-ranking of the selected entries: nearly every row is identical to the oracle's
    assert rep["exact_rows"] >= 0.999 * batch2.n_atoms, rep


def test_config3_cutoff_supercells(mg, ctx):
    # 16 cells of 500-2000 atoms, r_c = 8 A: plane spacings > 2 r_c, so every ordered pair has a
    # single candidate image (the minimum-image limit of the per-pair sub-box)
    b = C.config_batch(3)
    assert b.n_struct == 16 and 500 <= np.diff(b.struct_ptr).min() and np.diff(b.struct_ptr).max() <= 2000
    got, status = _cutoff(mg, ctx, b, 8.0)
    assert status == 0
    rep = check.check_cutoff(b, 8.0, got)
    assert rep["extra"] == 0 and rep["missing"] == 0, rep
    assert rep["n_edges"] == rep["n_ref"] > 1_000_000


def test_mixed_small_and_large_structures(mg, ctx):
    # structures above and below the shared-memory staging limit in one batch, dense enough that
    # the large one has several images per pair
    small = C.small_batch(12, seed=21)
    rng = np.random.default_rng(7)
    cell = (np.diag([9.0, 10.0, 11.0]) + rng.uniform(-1, 1, (3, 3))).astype(np.float32)
    big = C.Batch(pos=rng.random((150, 3), dtype=np.float32), lattice=cell[None],
                  struct_ptr=np.array([0, 150], np.int32))
    b = C.concat([small, big, small])
    got, status = _cutoff(mg, ctx, b, 6.5)
    assert status == 0
    rep = check.check_cutoff(b, 6.5, got)
    assert rep["extra"] == 0 and rep["missing"] == 0, rep


def test_knn_large_structures(mg, ctx):
    # structures above the shared-memory staging limit take the growing-radius routine row by row
    small = C.small_batch(6, seed=31)
    rng = np.random.default_rng(11)
    cell = (np.diag([11.0, 12.0, 13.0]) + rng.uniform(-1, 1, (3, 3))).astype(np.float32)
    big = C.Batch(pos=rng.random((200, 3), dtype=np.float32), lattice=cell[None],
                  struct_ptr=np.array([0, 200], np.int32))
    b = C.concat([small, big, small])
    got, status = _knn(mg, ctx, b, 12)
    assert status == 0
    check.check_knn(b, 12, got)


@pytest.mark.parametrize("n_big", [300, 600, 1500])
def test_knn_structures_above_256_atoms(mg, ctx, n_big):
    # the growing-radius routine carries dst in a tie word that must not wrap above 256 atoms
    small = C.small_batch(4, seed=33)
    rng = np.random.default_rng(n_big)
    side = (n_big / 0.08) ** (1.0 / 3.0)
    cell = (np.diag([side, 1.1 * side, 0.9 * side]) + rng.uniform(-1, 1, (3, 3))).astype(np.float32)
    big = C.Batch(pos=rng.random((n_big, 3), dtype=np.float32), lattice=cell[None],
                  struct_ptr=np.array([0, n_big], np.int32))
    b = C.concat([small, big, small])
    got, status = _knn(mg, ctx, b, 12)
    assert status == 0
    rep = check.check_knn(b, 12, got)
    assert rep["exact_rows"] >= 0.99 * b.n_atoms, rep


def test_knn_supercell_config3_sized(mg, ctx):
    # one BASELINE configs[3]-sized supercell (500-2000 atoms) through the KNN call
    b = C.config_batch(3, n_struct=2)
    got, status = _knn(mg, ctx, b, 12)
    assert status == 0
    check.check_knn(b, 12, got)


def test_cutoff_graph_many_calls_no_count_between(mg, ctx):
    # back-to-back mg_cutoff_graph calls on one context with no mg_cutoff_count in between: nothing in
    # the library may depend on how many calls were made (a per-call ticket once grew without bound)
    b = C.small_batch(64, seed=5)
    pos, lat, ptr = mg.to_device(b)
    ref = oracle.cutoff_graph(b.pos, b.lattice, b.struct_ptr, 5.0)
    cap = int(ref["n_edges"])
    out = mg.Edges.allocate(b.n_atoms, cap, "cuda", dist=True)
    for _ in range(3000):
        ctx.mg_cutoff_graph(pos, lat, ptr, 5.0, out)
    got = out.to_numpy()
    assert ctx.mg_check() == 0
    rep = check.check_cutoff(b, 5.0, got, ref=ref)
    assert rep["extra"] == 0 and rep["missing"] == 0


def test_config4_full_size_walk(mg, ctx):
    # BASELINE configs[4] at full size: 1024 crystals, 100 update steps; steps 1, 25, 50, 75, 100 are
    # checked against the oracle and against a fresh mg_knn_graph call on the same inputs (R17)
    import torch
    k = 24
    b0 = C.config_batch(4)
    assert b0.n_struct == 1024
    ptr = torch.from_numpy(b0.struct_ptr).cuda()
    graph = ctx.mg_graph_create(mg.MG_KIND_KNN, ptr, b0.n_atoms, k=k)
    out = mg.Edges.allocate(b0.n_atoms, k * b0.n_atoms, "cuda", dist=True)
    for step, b in enumerate(C.walk(b0, 100, seed=0), start=1):
        pos, lat, _ = mg.to_device(b)
        ctx.mg_update_graph(graph, pos, lat, out)
        if step not in (1, 25, 50, 75, 100):
            continue
        got = out.to_numpy()
        assert ctx.mg_check() == 0
        rep = check.check_knn(b, k, got)
        assert rep["n_edges"] == k * b.n_atoms
        fresh, _ = _knn(mg, ctx, b, k)
        for key in ("src", "dst", "offset", "vec", "dist", "row_ptr"):
            assert np.array_equal(fresh[key], got[key]), (step, key)
    assert ctx.mg_check() == 0
    graph.close()


def test_config4_update_steps(mg, ctx):
    import torch
    k = 24
    b0 = C.config_batch(4, n_struct=256)
    ptr = torch.from_numpy(b0.struct_ptr).cuda()
    graph = ctx.mg_graph_create(mg.MG_KIND_KNN, ptr, b0.n_atoms, k=k)
    out = mg.Edges.allocate(b0.n_atoms, k * b0.n_atoms, "cuda", dist=True)
    for step, b in enumerate(C.walk(b0, 6, seed=0)):
        pos, lat, _ = mg.to_device(b)
        ctx.mg_update_graph(graph, pos, lat, out)
        got = out.to_numpy()
        assert ctx.mg_check() == 0
        rep = check.check_knn(b, k, got)
        assert rep["n_edges"] == k * b.n_atoms
        # R17: identical to a fresh build on the same inputs
        fresh, _ = _knn(mg, ctx, b, k)
        for key in ("src", "dst", "offset", "vec", "dist", "row_ptr"):
            assert np.array_equal(fresh[key], got[key]), (step, key)
    graph.close()


@pytest.mark.parametrize("cfg,n_struct,k,sigma", [(4, 128, 12, 0.02), (4, 128, 24, 0.02), (3, 2, 12, 0.004)])
def test_update_graph_in_a_cuda_graph(mg, ctx, cfg, n_struct, k, sigma):
    # mg_update_graph allocates nothing and never synchronises: capture one step in a CUDA graph,
    # replay it on new geometry written into the captured input buffers, compare with fresh calls
    # (the pair-lane kernel, the one for k > 16 in its own module, the one for batches of large structures in its own)
    import torch
    b0 = C.config_batch(cfg, n_struct=n_struct)
    steps = list(C.walk(b0, 4, seed=3, sigma=sigma))
    ptr = torch.from_numpy(b0.struct_ptr).cuda()
    pos_buf = torch.from_numpy(steps[0].pos).cuda()
    lat_buf = torch.from_numpy(steps[0].lattice).cuda()
    graph = ctx.mg_graph_create(mg.MG_KIND_KNN, ptr, b0.n_atoms, k=k)
    out = mg.Edges.allocate(b0.n_atoms, k * b0.n_atoms, "cuda", dist=True)
    ctx.mg_update_graph(graph, pos_buf, lat_buf, out)            # warm-up outside the capture
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    cg = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        with torch.cuda.graph(cg, stream=side):
            ctx.mg_update_graph(graph, pos_buf, lat_buf, out)
    for b in steps[1:]:
        pos_buf.copy_(torch.from_numpy(b.pos))
        lat_buf.copy_(torch.from_numpy(b.lattice))
        cg.replay()
        torch.cuda.synchronize()
        got = out.to_numpy()
        assert ctx.mg_check() == 0
        check.check_knn(b, k, got)
        fresh, _ = _knn(mg, ctx, b, k)
        for key in ("dst", "offset", "vec", "dist"):
            assert np.array_equal(fresh[key], got[key]), key
    graph.close()


def test_update_cutoff_matches_fresh(mg, ctx):
    import torch
    b0 = C.config_batch(4, n_struct=64)
    ptr = torch.from_numpy(b0.struct_ptr).cuda()
    graph = ctx.mg_graph_create(mg.MG_KIND_CUTOFF, ptr, b0.n_atoms, r_c=5.0)
    for b in C.walk(b0, 3, seed=1):
        pos, lat, _ = mg.to_device(b)
        cap = ctx.mg_cutoff_count(pos, lat, ptr, 5.0)
        out = mg.Edges.allocate(b.n_atoms, cap, "cuda", dist=True)
        ctx.mg_update_graph(graph, pos, lat, out)
        got = out.to_numpy()
        assert ctx.mg_check() == 0
        rep = check.check_cutoff(b, 5.0, got)
        assert rep["extra"] == 0 and rep["missing"] == 0
    graph.close()


# ------------------------------------------------------------------ closed forms through the GPU
@pytest.mark.parametrize("name,rc,count", [("sc", 1.01, 6), ("sc", 1.42, 18), ("sc", 2.01, 32),
                                            ("fcc_conv", 0.7072, 12), ("fcc_prim", 0.7072, 12),
                                            ("bcc_conv", 0.8661, 8), ("bcc_prim", 0.8661, 8),
                                            ("diamond", 0.4331, 4), ("hcp", 1.0001, 12)])
def test_textbook_coordination(mg, ctx, name, rc, count):
    b = C.textbook(name)
    got, status = _cutoff(mg, ctx, b, rc)
    assert status == 0
    assert np.all(np.diff(got["row_ptr"]) == count)
    check.check_cutoff(b, rc, got)


def test_strict_inequality_exact(mg, ctx):
    # d == r_c exactly is not an edge (Def. 3 strict '<'): decided by the FP64 window path
    b = C.textbook("sc")
    got, _ = _cutoff(mg, ctx, b, 1.0)
    assert got["n_edges"] == 0
    got, _ = _cutoff(mg, ctx, b, float(np.nextafter(np.float32(1.0), np.float32(2.0))))
    assert got["n_edges"] == 6


def test_knn_sc_tiebreak_order(mg, ctx):
    b = C.textbook("sc")
    got, _ = _knn(mg, ctx, b, 12)
    first6 = [(-1, 0, 0), (0, -1, 0), (0, 0, -1), (0, 0, 1), (0, 1, 0), (1, 0, 0)]
    next6 = [(-1, -1, 0), (-1, 0, -1), (-1, 0, 1), (-1, 1, 0), (0, -1, -1), (0, -1, 1)]
    assert list(map(tuple, got["offset"].tolist())) == first6 + next6
    check.check_knn(b, 12, got)


@pytest.mark.parametrize("k", [1, 6, 12, 24, 32, 33, 48, 64])
def test_knn_k_sweep(mg, ctx, k):
    b = C.small_batch(48, seed=3)
    got, status = _knn(mg, ctx, b, k)
    assert status == 0
    check.check_knn(b, k, got)


# ------------------------------------------------------------------ paper-scale workloads
@pytest.fixture(scope="module")
def batch_paper():
    return C.paper_scale_batch(256)          # cells of up to 64 atoms, the paper's batch size


@pytest.mark.parametrize("k", [16, 32, 64])
def test_paper_scale_knn(mg, ctx, batch_paper, k):
    # the columns of the paper's Table 1: KNN 16 / 32 / 64
    got, status = _knn(mg, ctx, batch_paper, k)
    assert status == 0
    rep = check.check_knn(batch_paper, k, got)
    assert rep["exact_rows"] >= 0.995 * batch_paper.n_atoms, rep


@pytest.mark.parametrize("rc", [3.0, 5.0, 8.0])
def test_paper_scale_cutoff(mg, ctx, batch_paper, rc):
    got, status = _cutoff(mg, ctx, batch_paper, rc)
    assert status == 0
    rep = check.check_cutoff(batch_paper, rc, got)
    assert rep["extra"] == 0 and rep["missing"] == 0, rep


@pytest.mark.parametrize("name,k", [("fcc_conv", 24), ("fcc_prim", 24), ("bcc_conv", 20), ("diamond", 10), ("hcp", 15), ("rocksalt", 30)])
def test_knn_inside_a_degenerate_shell(mg, ctx, name, k):
    # k ends in the middle of a symmetric shell (e.g. FCC: 12 + 6 + 24 neighbours, k = 24 cuts the third shell):
    # many images share the k-th distance exactly, the oracle breaks the tie by (dst, tau); whatever subset the
    # library returns must be k distinct images, all inside the 1e-5 A tie band of the oracle's (check_knn)
    b = C.textbook(name, a=3.61)
    got, status = _knn(mg, ctx, b, k)
    assert status == 0
    rep = check.check_knn(b, k, got)
    assert rep["n_edges"] == k * b.n_atoms


@pytest.mark.parametrize("k", [24, 32])
def test_knn_sheared_cells_with_tables_above_256_cells(mg, ctx, k):
    # strongly sheared cells: the per-pair sub-box has hundreds to thousands of cells, the warp's table holds 256.
    # The pair-lane kernel walks such a structure one source row at a time, the table tile by tile
    # (mg_knn_find_tiled); above 4096 cells the growing-radius routine takes the rows.  Mixed with ordinary
    # skewed cells (BASELINE configs[4] family), which hold a few such structures of their own.
    rng = np.random.default_rng(31)
    items = []
    for s, n in ((1.0, 1), (1.0, 3), (0.7, 2), (0.7, 5), (0.5, 1), (0.5, 4), (0.4, 1), (0.33, 2)):
        cell = np.array([[14.0, 0.0, 0.0], [13.8, s, 0.0], [13.7, 0.5 * s, s]], np.float32)
        items.append((cell, rng.random((n, 3), dtype=np.float32)))
    b = C.concat([C.skewed_batch(120, seed=11), C._assemble(items), C.small_batch(6, seed=3)])
    got, status = _knn(mg, ctx, b, k)
    assert status == 0
    rep = check.check_knn(b, k, got)
    assert rep["n_edges"] == k * b.n_atoms


@pytest.mark.parametrize("k", [33, 40, 64])
def test_knn_above_32_neighbours_on_structures_above_64_atoms(mg, ctx, k):
    # k > 32 takes the warp-per-atom kernel of knn_small.cuh; structures above its staging limit of 64 atoms are read in
    # place (they used to be refused with MG_ERR_UNSUPPORTED)
    rng = np.random.default_rng(41)
    items = []
    for n, lens in ((100, (9.0, 10.0, 11.0)), (300, (14.0, 15.0, 13.0)), (65, (7.0, 7.5, 8.0))):
        cell = (np.diag(lens) + rng.uniform(-0.8, 0.8, (3, 3))).astype(np.float32)
        items.append((cell, rng.random((n, 3), dtype=np.float32)))
    b = C.concat([C.small_batch(5, seed=51), C._assemble(items), C.small_batch(3, seed=52)])
    got, status = _knn(mg, ctx, b, k)
    assert status == 0
    rep = check.check_knn(b, k, got)
    assert rep["n_edges"] == k * b.n_atoms
    # ... and under mg_update_graph (per-atom radius hints), against a fresh call on the moved atoms
    import torch
    pos, lat, ptr = mg.to_device(b)
    graph = ctx.mg_graph_create(mg.MG_KIND_KNN, ptr, b.n_atoms, k=k)
    out = mg.Edges.allocate(b.n_atoms, k * b.n_atoms, "cuda", dist=True)
    for t in C.walk(b, 2, seed=9):
        ctx.mg_update_graph(graph, torch.from_numpy(t.pos).cuda(), torch.from_numpy(t.lattice).cuda(), out)
        assert ctx.mg_check() == 0
        check.check_knn(t, k, out.to_numpy())
    graph.close()


def test_cutoff_1500_atoms_with_spacings_below_two_cutoffs(mg, ctx):
    # one structure of 1500 atoms in a cell of 25-27 A, r_c = 14 A: plane spacings below 2 r_c, so an ordered pair has up
    # to eight candidate images (no minimum-image regime, no cell list): the generic rows of the scan kernel, lanes over
    # (target, cell); about 1.5 M edges, compared with the oracle edge by edge
    rng = np.random.default_rng(15)
    cell = (np.diag([25.0, 26.0, 27.0]) + rng.uniform(-1.5, 1.5, (3, 3))).astype(np.float32)
    big = C.Batch(pos=rng.random((1500, 3), dtype=np.float32), lattice=cell[None], struct_ptr=np.array([0, 1500], np.int32))
    b = C.concat([big, C.small_batch(4, seed=17)])
    got, status = _cutoff(mg, ctx, b, 14.0)
    assert status == 0
    rep = check.check_cutoff(b, 14.0, got)
    assert rep["extra"] == 0 and rep["missing"] == 0 and rep["n_edges"] > 1_000_000, rep
    assert np.abs(got["offset"]).max() >= 1                      # images of other cells are among the edges


def _random_structure(rng, n, lens, jitter=1.0):
    cell = (np.diag(np.asarray(lens, np.float64)) + rng.uniform(-jitter, jitter, (3, 3))).astype(np.float32)
    return cell, rng.random((n, 3), dtype=np.float32)


@pytest.mark.parametrize("k", [1, 12, 27, 32, 33, 64])
def test_knn_batches_of_large_structures_through_the_cell_list(mg, ctx, k):
    # batches whose structures average more than 64 atoms take knn_bins.cu: one warp per row, candidates from the cell list
    # where the structure has one (large cell, R / h < 1/2), the growing-radius routine for everything else in the batch
    rng = np.random.default_rng(61 + k)
    items = [_random_structure(rng, 700, (24.0, 26.0, 22.0)),       # cell list on all axes
             _random_structure(rng, 400, (40.0, 9.0, 30.0)),        # one short axis: no slabs there
             _random_structure(rng, 90, (6.0, 6.5, 7.0), 0.3),      # dense: several images per pair, no cell list
             _random_structure(rng, 3, (4.0, 5.0, 6.0), 0.2),       # a small one among them
             (np.eye(3, dtype=np.float32), np.zeros((0, 3), np.float32)),   # an empty one
             _random_structure(rng, 70, (20.0, 21.0, 19.0))]
    items[5][1][17] += np.float32(16.0)                             # an atom 16 cells away: that structure's cell list is not used
    items[0][1][:3] = np.array([[0.0, 0.0, 0.0], [1.0 - 2.0 ** -24, 0.5, 0.5], [0.5, 0.0, 1.0 - 2.0 ** -24]], np.float32)
    b = C._assemble(items)
    assert b.n_atoms / b.n_struct > 64
    got, status = _knn(mg, ctx, b, k)
    assert status == 0
    rep = check.check_knn(b, k, got)
    assert rep["n_edges"] == k * b.n_atoms


@pytest.mark.parametrize("k", [12, 40])
def test_knn_update_graph_on_large_structures(mg, ctx, k):
    import torch
    b = C.config_batch(3, n_struct=3)
    pos, lat, ptr = mg.to_device(b)
    graph = ctx.mg_graph_create(mg.MG_KIND_KNN, ptr, b.n_atoms, k=k)
    out = mg.Edges.allocate(b.n_atoms, k * b.n_atoms, "cuda", dist=True)
    for t in C.walk(b, 3, seed=4, sigma=0.004):
        ctx.mg_update_graph(graph, torch.from_numpy(t.pos).cuda(), torch.from_numpy(t.lattice).cuda(), out)
        assert ctx.mg_check() == 0
        check.check_knn(t, k, out.to_numpy())
    graph.close()
    # an invalid lattice among large structures: placeholder rows there, the error from mg_check, the others right
    bad = C.Batch(pos=b.pos, lattice=b.lattice.copy(), struct_ptr=b.struct_ptr)
    bad.lattice.reshape(-1, 9)[1, :] = 0.0
    pos, lat, ptr = mg.to_device(bad)
    g = ctx.knn_graph(pos, lat, ptr, k, dist=True).to_numpy()
    assert ctx.mg_check() == 3                                     # MG_ERR_SINGULAR_LATTICE
    lo, hi = bad.struct_ptr[1], bad.struct_ptr[2]
    assert np.array_equal(g["dst"][k * lo:k * hi], np.repeat(np.arange(lo, hi), k))
    first = C.Batch(pos=b.pos[:b.struct_ptr[1]], lattice=b.lattice[:1], struct_ptr=b.struct_ptr[:2])
    ref = oracle.knn_graph(first.pos, first.lattice, first.struct_ptr, k)
    assert np.array_equal(g["dst"][:k * lo], ref["dst"])


@pytest.mark.parametrize("k", [1, 12, 16, 17, 32])
def test_knn_large_structures_inside_a_batch_of_small_cells(mg, ctx, k):
    # the batch averages at most 64 atoms per structure, so it takes the pair-lane kernels (k <= 16 and k > 16), whose rows of
    # a structure above the staging limit go a warp per row over every target and the pair's sub-box (mg_knn_row_box):
    # one image per pair, several images per pair, coordinates outside the cell, a cluster whose rows overflow the
    # warp's hit buffer (those fall through to the growing-radius routine)
    import torch
    rng = np.random.default_rng(71 + k)
    items = [C.small_crystal(5, s) for s in range(24)]
    items.insert(3, _random_structure(rng, 130, (22.0, 25.0, 21.0)))              # sparse: one cell per pair
    items.insert(9, _random_structure(rng, 90, (6.0, 6.5, 7.0), 0.3))             # dense: a sub-box of several cells
    items.insert(15, _random_structure(rng, 300, (30.0, 9.0, 28.0)))
    far = _random_structure(rng, 70, (12.0, 13.0, 11.0))
    far[1][:] = (far[1] * np.float32(5.0) - np.float32(2.0)).astype(np.float32)   # coordinates in [-2, 3)
    items.insert(20, far)
    blob = _random_structure(rng, 120, (18.0, 18.0, 18.0))
    blob[1][:100] = blob[1][0] + rng.normal(0, 0.002, (100, 3)).astype(np.float32)
    if k >= 12: items.append(blob)                                                # (with k = 1 its rows are a tie in FP32)
    b = C._assemble(items)
    assert b.n_atoms / b.n_struct <= 64
    got, status = _knn(mg, ctx, b, k)
    assert status == 0
    rep = check.check_knn(b, k, got)
    assert rep["n_edges"] == k * b.n_atoms
    # and as a sequence of updates: the hint these rows leave is the next call's radius
    pos, lat, ptr = mg.to_device(b)
    graph = ctx.mg_graph_create(mg.MG_KIND_KNN, ptr, b.n_atoms, k=k)
    out = mg.Edges.allocate(b.n_atoms, k * b.n_atoms, "cuda", dist=True)
    for t in C.walk(b, 2, seed=9, sigma=0.01):
        ctx.mg_update_graph(graph, torch.from_numpy(t.pos).cuda(), torch.from_numpy(t.lattice).cuda(), out)
        assert ctx.mg_check() == 0
        check.check_knn(t, k, out.to_numpy())
    graph.close()
