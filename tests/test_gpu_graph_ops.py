"""GPU parity of mg_symmetrize and mg_triplets_graph against
oracle/graph_ops.py, through the C ABI binding, on the library's own KNN / cutoff graphs."""
import numpy as np
import pytest

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


def _rows_as_sets(g, n_atoms):
    tau = np.asarray(g["offset"] if "offset" in g else g["tau"]).reshape(-1, 3).astype(np.int64)
    keys = [(int(d), int(t[0]), int(t[1]), int(t[2])) for d, t in zip(g["dst"], tau)]
    rp = np.asarray(g["row_ptr"])
    return [sorted(keys[rp[i]:rp[i + 1]]) for i in range(n_atoms)]


@pytest.mark.parametrize("cfg,k", [(1, 12), (2, 12), (4, 24)])
def test_symmetrize_knn(mg, ctx, cfg, k):
    b = C.config_batch(cfg, n_struct=512 if cfg == 2 else None)
    pos, lat, ptr = mg.to_device(b)
    knn = ctx.knn_graph(pos, lat, ptr, k, dist=True)
    out = mg.Edges.allocate(b.n_atoms, 2 * k * b.n_atoms, "cuda", dist=True)
    ctx.mg_symmetrize(knn, b.n_atoms, out)
    got = out.to_numpy()
    assert ctx.mg_check() == 0
    kn = knn.to_numpy()
    ref = G.symmetrize(b.n_atoms, kn["src"], kn["dst"], kn["offset"], vec=kn["vec"], dist=kn["dist"])
    assert got["n_edges"] == ref["n_edges"] and np.array_equal(got["row_ptr"], ref["row_ptr"])
    assert np.array_equal(got["src"], np.repeat(np.arange(b.n_atoms), np.diff(got["row_ptr"])))
    assert _rows_as_sets(got, b.n_atoms) == _rows_as_sets(ref, b.n_atoms)            # bit-exact edge sets
    # the old rows keep their place and order; vec / dist of every edge equal the oracle's (exact: copies and negations)
    look = {(int(s), int(d), *map(int, t)): (v, dd) for s, d, t, v, dd in zip(ref["src"], ref["dst"], ref["tau"], ref["vec"], ref["dist"])}
    for s, d, t, v, dd in zip(got["src"], got["dst"], got["offset"], got["vec"], got["dist"]):
        rv, rd = look[(int(s), int(d), *map(int, t))]
        assert np.array_equal(np.asarray(rv, np.float32), v) and np.float32(rd) == dd
    rp_in, rp = kn["row_ptr"], got["row_ptr"]
    for i in range(0, b.n_atoms, max(1, b.n_atoms // 200)):
        assert np.array_equal(got["dst"][rp[i]:rp[i] + k], kn["dst"][rp_in[i]:rp_in[i + 1]])


def test_symmetrize_cutoff_is_identity_and_capacity_is_reported(mg, ctx):
    b = C.config_batch(0)
    pos, lat, ptr = mg.to_device(b)
    cut = ctx.cutoff_graph(pos, lat, ptr, 5.0, dist=True)
    e = int(cut.n_edges.item())
    out = mg.Edges.allocate(b.n_atoms, e, "cuda", dist=True)
    ctx.mg_symmetrize(cut, b.n_atoms, out)
    got, cin = out.to_numpy(), cut.to_numpy()
    assert ctx.mg_check() == 0 and got["n_edges"] == e
    for key in ("row_ptr", "src", "dst", "offset", "vec", "dist"):
        assert np.array_equal(got[key], cin[key]), key
    # a KNN graph needs more room than it has edges: the required count comes back with MG_ERR_CAPACITY
    knn = ctx.knn_graph(pos, lat, ptr, 4, dist=True)
    small = mg.Edges.allocate(b.n_atoms, 4 * b.n_atoms, "cuda", dist=True)
    ctx.mg_symmetrize(knn, b.n_atoms, small)
    need = int(small.n_edges.item())
    assert ctx.mg_check() == 6 and need > 4 * b.n_atoms
    kn = knn.to_numpy()
    assert need == G.symmetrize(b.n_atoms, kn["src"], kn["dst"], kn["offset"])["n_edges"]


@pytest.mark.parametrize("kind", ["knn", "cutoff", "empty"])
def test_triplets(mg, ctx, kind):
    import torch
    b = C.config_batch(1) if kind != "empty" else C.Batch(pos=np.zeros((0, 3), np.float32), lattice=np.zeros((0, 3, 3), np.float32),
                                                           struct_ptr=np.zeros(1, np.int32))
    if kind == "empty":
        row_ptr = torch.zeros(1, dtype=torch.int32, device="cuda")
    else:
        pos, lat, ptr = mg.to_device(b)
        g = ctx.knn_graph(pos, lat, ptr, 12) if kind == "knn" else ctx.cutoff_graph(pos, lat, ptr, 4.0)
        row_ptr = g.row_ptr
    ref = G.triplets(row_ptr.cpu().numpy())
    out = ctx.mg_triplets_graph(row_ptr, b.n_atoms, ref["n_triplets"])
    assert ctx.mg_check() == 0
    assert int(out["n_triplets"].item()) == ref["n_triplets"]
    assert np.array_equal(out["tri_ptr"].cpu().numpy(), ref["tri_ptr"])
    n = ref["n_triplets"]
    assert np.array_equal(out["edge_a"][:n].cpu().numpy(), ref["edge_a"]) and np.array_equal(out["edge_b"][:n].cpu().numpy(), ref["edge_b"])
    if kind == "knn":
        assert n == 12 * 11 * b.n_atoms
        short = ctx.mg_triplets_graph(row_ptr, b.n_atoms, n // 2)            # too small: count still reported
        assert ctx.mg_check() == 6 and int(short["n_triplets"].item()) == n
        assert np.array_equal(short["edge_a"][:n // 2].cpu().numpy(), ref["edge_a"][:n // 2])


# ------------------------------------------------------------------ per-atom cutoffs
@pytest.mark.parametrize("cfg", [0, 2, 3])
def test_cutoff_graph_radii(mg, ctx, cfg):
    import torch
    import oracle
    from oracle import check
    b = C.config_batch(cfg, n_struct={0: None, 2: 512, 3: 2}[cfg])
    rng = np.random.default_rng(17 + cfg)
    radii = rng.uniform(2.0, 6.5, b.n_atoms).astype(np.float32)      # "covalent-like": one cutoff per atom
    ref = oracle.cutoff_graph_radii(b.pos, b.lattice, b.struct_ptr, radii)
    pos, lat, ptr = mg.to_device(b)
    out = mg.Edges.allocate(b.n_atoms, ref["n_edges"], "cuda", dist=True)
    ctx.mg_cutoff_graph_radii(pos, lat, ptr, torch.from_numpy(radii).cuda(), out)
    got = out.to_numpy()
    assert ctx.mg_check() == 0
    assert got["n_edges"] == ref["n_edges"] and np.array_equal(got["row_ptr"], ref["row_ptr"])
    kg = np.sort(check._keys(got["src"], got["dst"], got["offset"]))
    ko = np.sort(check._keys(ref["src"], ref["dst"], ref["tau"]))
    assert np.array_equal(kg, ko)                                     # bit-exact edge sets (FP64 window decision)
    d64, v64 = oracle.edge_distance(b.pos, b.lattice, b.struct_ptr, got["src"], got["dst"], got["offset"])
    assert np.abs(got["vec"] - v64).max() <= 1e-5 and np.abs(got["dist"] - d64).max() <= 1e-5
    assert np.all(d64 < radii[got["src"]].astype(np.float64))


def test_cutoff_graph_radii_constant_equals_cutoff_graph(mg, ctx):
    import torch
    b = C.config_batch(0)
    pos, lat, ptr = mg.to_device(b)
    a = ctx.cutoff_graph(pos, lat, ptr, 5.0, dist=True).to_numpy()
    out = mg.Edges.allocate(b.n_atoms, a["n_edges"], "cuda", dist=True)
    ctx.mg_cutoff_graph_radii(pos, lat, ptr, torch.full((b.n_atoms,), 5.0, device="cuda"), out)
    g = out.to_numpy()
    assert ctx.mg_check() == 0 and g["n_edges"] == a["n_edges"] and np.array_equal(g["row_ptr"], a["row_ptr"])
    from oracle import check
    assert np.array_equal(np.sort(check._keys(g["src"], g["dst"], g["offset"])), np.sort(check._keys(a["src"], a["dst"], a["offset"])))
    bad = torch.full((b.n_atoms,), 5.0, device="cuda")
    bad[3] = -1.0
    ctx.mg_cutoff_graph_radii(pos, lat, ptr, bad, out)
    assert ctx.mg_check() == 7                                         # MG_ERR_UNSUPPORTED


def test_symmetrize_of_an_incomplete_graph_reads_nothing_past_its_arrays(mg, ctx):
    # a KNN graph cut off by hand: n_edges says more edges than the arrays hold (what a cutoff call with too
    # small a capacity leaves behind).  mg_symmetrize reads the edges that are there and reports MG_ERR_CAPACITY.
    import torch
    b, k = C.config_batch(1), 12
    pos, lat, ptr = mg.to_device(b)
    knn = ctx.knn_graph(pos, lat, ptr, k, dist=True)
    keep = (k * b.n_atoms) // 3
    cut = mg.Edges(row_ptr=knn.row_ptr, src=knn.src[:keep].clone(), dst=knn.dst[:keep].clone(),
                   offset=knn.offset[:keep].clone(), vec=knn.vec[:keep].clone(), dist=knn.dist[:keep].clone(),
                   n_edges=knn.n_edges, capacity=keep)
    out = mg.Edges.allocate(b.n_atoms, 2 * k * b.n_atoms, "cuda", dist=True)
    ctx.mg_symmetrize(cut, b.n_atoms, out)
    torch.cuda.synchronize()
    assert ctx.mg_check() == 6                                     # MG_ERR_CAPACITY
    # and the context is fine afterwards
    ctx.mg_symmetrize(knn, b.n_atoms, out)
    assert ctx.mg_check() == 0 and int(out.n_edges.item()) > k * b.n_atoms


def test_graph_ops_row_offsets_at_full_size(mg, ctx):
    # BASELINE configs[2] (43 578 atoms: the scans of graph_ops.cuh run over six chunks of 8192 rows): the row offsets of
    # both calls against their definitions written in numpy, sampled rows of the triplets against Def. 3's Gamma_2
    import torch
    b, k = C.config_batch(2), 12
    pos, lat, ptr = mg.to_device(b)
    knn = ctx.knn_graph(pos, lat, ptr, k, dist=True)
    out = mg.Edges.allocate(b.n_atoms, 2 * k * b.n_atoms, "cuda", dist=True)
    ctx.mg_symmetrize(knn, b.n_atoms, out)
    assert ctx.mg_check() == 0
    kn, got = knn.to_numpy(), out.to_numpy()

    def key(s, d, t):
        t = t.astype(np.int64) + 128
        return ((s.astype(np.int64) * b.n_atoms + d.astype(np.int64)) << 24) | (t[:, 0] << 16) | (t[:, 1] << 8) | t[:, 2]
    fwd = key(kn["src"], kn["dst"], kn["offset"])
    rev = key(kn["dst"], kn["src"], -kn["offset"].astype(np.int64))
    missing = ~np.isin(rev, fwd)
    extra = np.bincount(kn["dst"][missing], minlength=b.n_atoms)        # a missing reverse edge lands in the row of its dst
    want = np.concatenate([[0], np.cumsum(k + extra)])
    assert np.array_equal(got["row_ptr"], want) and got["n_edges"] == want[-1]
    assert np.array_equal(np.sort(key(got["src"], got["dst"], got["offset"])), np.sort(np.concatenate([fwd, rev[missing]])))
    # triplets of the symmetric graph (rows of different lengths)
    tri = ctx.mg_triplets_graph(out.row_ptr, b.n_atoms, 1)
    n_tri = int(tri["n_triplets"])
    assert ctx.mg_check() == 6                                     # one slot was not enough: MG_ERR_CAPACITY, count known
    d = np.diff(got["row_ptr"]).astype(np.int64)
    want_t = np.concatenate([[0], np.cumsum(d * (d - 1))])
    assert n_tri == want_t[-1]
    tri = ctx.mg_triplets_graph(out.row_ptr, b.n_atoms, n_tri)
    assert ctx.mg_check() == 0
    tp = tri["tri_ptr"].cpu().numpy()
    assert np.array_equal(tp, want_t)
    ea, eb = tri["edge_a"].cpu().numpy(), tri["edge_b"].cpu().numpy()
    for i in (0, 1, 8191, 8192, 8193, 16384, 24575, 32768, b.n_atoms - 1):
        e0, di = got["row_ptr"][i], int(d[i])
        pairs = [(e0 + a, e0 + c) for a in range(di) for c in range(di) if a != c]
        assert list(zip(ea[tp[i]:tp[i + 1]], eb[tp[i]:tp[i + 1]])) == pairs
