"""Randomised parity against the oracle, fixed seeds: inputs no hand-written case thought of.  Three generators —
large structures for the cutoff graph (cell list and generic rows), sheared / shifted / tiny cells, batches of large
structures and large structures among small cells for KNN, and
whole batches through every entry point (cutoff, per-atom cutoffs, KNN, symmetrize, triplets, update sequences)."""
import numpy as np
import pytest

import oracle
from oracle import check
from oracle import graph_ops as G
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


@pytest.mark.parametrize("seed", [101, 102])
def test_soak_cutoff_large_structures(mg, ctx, seed):
    rng = np.random.default_rng(seed)
    for case in range(10):
        items = []
        rc = float(rng.uniform(2.5, 6.0))
        for s in range(int(rng.integers(1, 4))):
            n = int(rng.integers(65, 400))
            lens = rc * rng.uniform(1.5, 14.0, 3) * (1.0 if rng.random() < 0.8 else 0.6)   # 1 to 14 cutoffs per axis
            ang = rng.uniform(65, 115, 3)
            cell = np.asarray(C.cell_from_parameters(lens[0], lens[1], lens[2], ang[0], ang[1], ang[2]), np.float32)
            x = rng.random((n, 3), dtype=np.float32)
            mode = rng.integers(0, 5)
            if mode == 1: x = (x * np.float32(4.0) - np.float32(2.0)).astype(np.float32)   # outside the cell
            if mode == 2: x[: n // 4] = np.round(x[: n // 4] * 8) / 8                        # on slab boundaries
            if mode == 3: x[: n // 8, 0] = np.float32(1.0) - np.float32(2.0 ** -24)          # just below 1
            if mode == 4: x = (x + np.float32(rng.integers(-14, 15))).astype(np.float32)     # whole cells away
            items.append((cell, x.astype(np.float32)))
        if rng.random() < 0.5:
            items.insert(0, C.small_crystal(int(rng.integers(1 << 30)), 0))
        b = C._assemble(items)
        pos, lat, ptr = mg.to_device(b)
        got = ctx.cutoff_graph(pos, lat, ptr, rc, dist=True).to_numpy()
        assert ctx.mg_check() == 0, (seed, case)
        rep = check.check_cutoff(b, rc, got)
        assert rep["extra"] == 0 and rep["missing"] == 0, (seed, case, rep)


@pytest.mark.parametrize("seed", [201, 202])
def test_soak_knn_sheared_and_shifted_cells(mg, ctx, seed):
    rng = np.random.default_rng(seed)
    for case in range(14):
        items = []
        k = int(rng.choice([1, 4, 12, 24, 32]))
        for s in range(int(rng.integers(1, 6))):
            n = int(rng.integers(1, 14))
            mode = rng.integers(0, 4)
            if mode == 0:      # sheared: one long vector, the others nearly parallel to it (tables of 100s to 1000s of cells)
                L = float(rng.uniform(6, 16)); sc = float(rng.uniform(0.35, 1.2))
                cell = np.array([[L, 0, 0], [L - rng.uniform(0.1, 0.5), sc, 0],
                                 [L - rng.uniform(0.1, 0.6), rng.uniform(0.2, 0.8) * sc, sc]], np.float32)
            else:
                lens = rng.uniform(3, 12, 3); ang = rng.uniform(40, 140, 3)
                cell = C.cell_from_parameters(lens[0], lens[1], lens[2], ang[0], ang[1], ang[2])   # None: no such cell
                if cell is None or not np.isfinite(cell).all() or abs(np.linalg.det(np.asarray(cell, np.float64))) < 1.0:
                    cell = np.diag(lens)
                cell = np.asarray(cell, np.float32)
            x = rng.random((n, 3), dtype=np.float32)
            if mode == 2: x = (x + rng.integers(-30, 31, size=(n, 3))).astype(np.float32)
            if mode == 3: x[0] += np.float32(rng.integers(41, 90))      # beyond the 40-cell guard of the pair-lane kernel
            items.append((cell, x.astype(np.float32)))
        b = C._assemble(items)
        pos, lat, ptr = mg.to_device(b)
        got = ctx.knn_graph(pos, lat, ptr, k, dist=True).to_numpy()
        assert ctx.mg_check() == 0, (seed, case, k)
        check.check_knn(b, k, got)


@pytest.mark.parametrize("seed", [401, 402])
def test_soak_knn_batches_of_large_structures(mg, ctx, seed):
    # batches that average more than 64 atoms per structure: a warp per row through the cell list (knn_bins.cu), with the
    # densities, cell shapes and coordinate ranges that decide whether a structure has one, and a dense cluster whose rows
    # overflow the warp's hit buffer
    rng = np.random.default_rng(seed)
    for case in range(10):
        items = []
        k = int(rng.choice([1, 2, 6, 12, 20, 32, 40, 64]))
        for s in range(int(rng.integers(1, 4))):
            n = int(rng.integers(65, 500))
            side = (n / float(rng.uniform(0.02, 0.12))) ** (1 / 3)
            lens = side * rng.uniform(0.6, 1.6, 3)
            ang = rng.uniform(70, 110, 3)
            cell = C.cell_from_parameters(lens[0], lens[1], lens[2], ang[0], ang[1], ang[2])
            cell = np.asarray(cell if cell is not None else np.diag(lens), np.float32)
            x = rng.random((n, 3), dtype=np.float32)
            mode = rng.integers(0, 5)
            if mode == 1: x = (x * np.float32(3.0) - np.float32(1.0)).astype(np.float32)
            if mode == 2: x[: n // 4] = np.round(x[: n // 4] * 8) / 8
            if mode == 3: x = (x + np.float32(rng.integers(-14, 15))).astype(np.float32)
            if mode == 4: x[: n // 3] = x[0] + rng.normal(0, 0.01, (n // 3, 3)).astype(np.float32)
            items.append((cell, x.astype(np.float32)))
        if rng.random() < 0.3:
            items.append(C.small_crystal(int(rng.integers(1 << 30)), 0))
        b = C._assemble(items)
        pos, lat, ptr = mg.to_device(b)
        got = ctx.knn_graph(pos, lat, ptr, k, dist=True).to_numpy()
        assert ctx.mg_check() == 0, (seed, case, k)
        check.check_knn(b, k, got)


@pytest.mark.parametrize("seed", [501, 502])
def test_soak_knn_large_structures_among_small_cells(mg, ctx, seed):
    # batches that average at most 64 atoms per structure with one or two structures above the staging limit: their rows
    # go a warp per row over every target and the pair's sub-box (mg_knn_row_box of knn_pairs.cuh), in both pair-lane kernels
    rng = np.random.default_rng(seed)
    for case in range(10):
        k = int(rng.choice([1, 3, 12, 16, 20, 32]))
        items = [C.small_crystal(int(rng.integers(1 << 30)), 0) for _ in range(int(rng.integers(12, 30)))]
        for s in range(int(rng.integers(1, 3))):
            n = int(rng.integers(65, 260))
            side = (n / float(rng.uniform(0.01, 0.25))) ** (1 / 3)
            lens = side * rng.uniform(0.5, 1.7, 3)
            ang = rng.uniform(65, 115, 3)
            cell = C.cell_from_parameters(lens[0], lens[1], lens[2], ang[0], ang[1], ang[2])
            cell = np.asarray(cell if cell is not None else np.diag(lens), np.float32)
            x = rng.random((n, 3), dtype=np.float32)
            mode = rng.integers(0, 5)
            if mode == 1: x = (x * np.float32(3.0) - np.float32(1.0)).astype(np.float32)
            if mode == 2: x = (x + np.float32(rng.integers(-30, 31))).astype(np.float32)   # the whole structure, cells away
            if mode == 3: x[: n // 4] = np.round(x[: n // 4] * 8) / 8
            if mode == 4 and k > 1: x[: n // 2] = x[0] + rng.normal(0, 0.01, (n // 2, 3)).astype(np.float32)
            items.insert(int(rng.integers(0, len(items) + 1)), (cell, x.astype(np.float32)))
        b = C._assemble(items)
        while b.n_atoms / b.n_struct > 64:
            items.append(C.small_crystal(int(rng.integers(1 << 30)), 0))
            b = C._assemble(items)
        pos, lat, ptr = mg.to_device(b)
        got = ctx.knn_graph(pos, lat, ptr, k, dist=True).to_numpy()
        assert ctx.mg_check() == 0, (seed, case, k)
        check.check_knn(b, k, got)


@pytest.mark.parametrize("seed", [301, 302])
def test_soak_every_entry_point(mg, ctx, seed):
    import torch
    rng = np.random.default_rng(seed)
    for case in range(8):
        sd = int(rng.integers(1 << 30))
        kind = case % 4
        if kind == 0: b = C.small_batch(int(rng.integers(1, 120)), seed=sd)
        elif kind == 1: b = C.skewed_batch(int(rng.integers(1, 60)), seed=sd)
        elif kind == 2: b = C.paper_scale_batch(int(rng.integers(1, 24)), seed=sd)
        else: b = C.concat([C.small_batch(int(rng.integers(1, 30)), seed=sd), C.supercell_batch(1, seed=sd % 7),
                            C.small_batch(3, seed=sd + 1)])
        pos, lat, ptr = mg.to_device(b)
        rc = float(rng.uniform(2.5, 7.0)); k = int(rng.choice([1, 3, 6, 12, 16, 24, 32, 40, 64]))
        if kind == 3: k, rc = min(k, 12), min(rc, 5.0)
        g = ctx.cutoff_graph(pos, lat, ptr, rc, dist=True).to_numpy()
        assert ctx.mg_check() == 0
        rep = check.check_cutoff(b, rc, g)
        assert rep["extra"] == 0 and rep["missing"] == 0, (seed, case, rep)
        if kind != 3:                                                 # per-atom cutoffs (Def. 3's c_i)
            radii = rng.uniform(1.5, rc, b.n_atoms).astype(np.float32)
            ref = oracle.cutoff_graph_radii(b.pos, b.lattice, b.struct_ptr, radii)
            out = mg.Edges.allocate(b.n_atoms, int(ref["n_edges"]) + 4, "cuda", dist=True)
            ctx.mg_cutoff_graph_radii(pos, lat, ptr, torch.from_numpy(radii).cuda(), out)
            gr = out.to_numpy()
            assert ctx.mg_check() == 0
            assert np.array_equal(np.sort(check._keys(gr["src"], gr["dst"], gr["offset"])),
                                  np.sort(check._keys(ref["src"], ref["dst"], ref["tau"])))
            assert np.array_equal(gr["row_ptr"], ref["row_ptr"])
        kn = ctx.knn_graph(pos, lat, ptr, k, dist=True)
        gk = kn.to_numpy()
        assert ctx.mg_check() == 0
        check.check_knn(b, k, gk)
        if b.n_atoms * k < 20000:                                     # symmetric graph and triplets of the KNN graph
            sym = mg.Edges.allocate(b.n_atoms, 2 * k * b.n_atoms, "cuda", dist=True)
            ctx.mg_symmetrize(kn, b.n_atoms, sym)
            gs = sym.to_numpy()
            assert ctx.mg_check() == 0
            ref = G.symmetrize(b.n_atoms, gk["src"], gk["dst"], gk["offset"], vec=gk["vec"], dist=gk["dist"])
            assert gs["n_edges"] == ref["n_edges"] and np.array_equal(gs["row_ptr"], ref["row_ptr"])
            assert np.array_equal(np.sort(check._keys(gs["src"], gs["dst"], gs["offset"])),
                                  np.sort(check._keys(np.asarray(ref["src"]), np.asarray(ref["dst"]), np.asarray(ref["tau"]))))
            d = np.diff(gs["row_ptr"]).astype(np.int64)
            nt = int((d * (d - 1)).sum())
            tri = ctx.mg_triplets_graph(sym.row_ptr, b.n_atoms, nt)
            assert ctx.mg_check() == 0 and int(tri["n_triplets"]) == nt
            reft = G.triplets(gs["row_ptr"])
            assert np.array_equal(tri["edge_a"].cpu().numpy()[:nt], np.asarray(reft["edge_a"]))
            assert np.array_equal(tri["edge_b"].cpu().numpy()[:nt], np.asarray(reft["edge_b"]))
        if kind in (0, 1):                                            # an update sequence equals fresh calls
            graph = ctx.mg_graph_create(mg.MG_KIND_KNN, ptr, b.n_atoms, k=k)
            out = mg.Edges.allocate(b.n_atoms, k * b.n_atoms, "cuda", dist=True)
            for t in C.walk(b, 3, seed=sd, sigma=float(rng.choice([0.01, 0.03, 0.08]))):
                ctx.mg_update_graph(graph, torch.from_numpy(t.pos).cuda(), torch.from_numpy(t.lattice).cuda(), out)
                assert ctx.mg_check() == 0
                check.check_knn(t, k, out.to_numpy())
            graph.close()
