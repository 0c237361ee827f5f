"""mg_symmetrize_static (include/matgraph.h): the symmetric graph for callers that cannot
allocate — no context, no cudaMalloc, scratch in a static device array — against the existing
mg_symmetrize on the library's own KNN graphs, on calls in a row that share the static array.
Collected last on purpose (the suite runs with pytest -x); passes alone in a fresh process and after the
other tests."""
import numpy as np
import pytest

from workloads import crystals as C

pytestmark = pytest.mark.gpu

TOL = 1e-5      # Angstrom: the tolerance of the parity tests (BASELINE.json north_star)


@pytest.fixture(scope="module")
def mg():
    import paper_2307_05380_b200 as m
    return m


@pytest.fixture(scope="module")
def ctx(mg):
    c = mg.Context(0)
    yield c
    c.close()


def _canonical(g):
    """Edges sorted by (src, dst, tau): the appended reverse edges of a row come in no particular order."""
    tau = g["offset"].reshape(-1, 3).astype(np.int64)
    order = np.lexsort((tau[:, 2], tau[:, 1], tau[:, 0], g["dst"], g["src"]))
    return {k: g[k].reshape(len(order), -1)[order] for k in ("src", "dst", "offset", "vec", "dist")}


def _same_graph(got, ref, deg_in):
    assert got["n_edges"] == ref["n_edges"] and np.array_equal(got["row_ptr"], ref["row_ptr"])
    a, b = _canonical(got), _canonical(ref)
    for k in ("src", "dst", "offset"):
        assert np.array_equal(a[k], b[k]), k                       # integer work: bit-exact
    assert np.abs(a["vec"] - b["vec"]).max() <= TOL and np.abs(a["dist"] - b["dist"]).max() <= TOL
    # the rows of the input keep their place and order in both
    rp = got["row_ptr"]
    for i in range(0, len(deg_in), max(1, len(deg_in) // 300)):
        s = slice(rp[i], rp[i] + deg_in[i])
        assert np.array_equal(got["dst"][s], ref["dst"][s]) and np.array_equal(got["offset"][s], ref["offset"][s])


def _knn_and_reference(mg, ctx, b, k):
    pos, lat, ptr = mg.to_device(b)
    knn = ctx.knn_graph(pos, lat, ptr, k, dist=True)
    ref = mg.Edges.allocate(b.n_atoms, 2 * k * b.n_atoms, "cuda", dist=True)
    ctx.mg_symmetrize(knn, b.n_atoms, ref)
    assert ctx.mg_check() == 0
    return knn, ref.to_numpy()


def test_static_symmetrize_matches_mg_symmetrize_on_calls_in_a_row(mg, ctx):
    import torch
    ba, ka = C.config_batch(1), 12                                   # 256 crystals, KNN k = 12
    bb, kb = C.config_batch(2, n_struct=700), 6                      # another batch, other sizes
    knn_a, ref_a = _knn_and_reference(mg, ctx, ba, ka)
    knn_b, ref_b = _knn_and_reference(mg, ctx, bb, kb)
    assert ref_a["n_edges"] > ka * ba.n_atoms and ref_b["n_edges"] > kb * bb.n_atoms   # reverse edges were added
    outs = [mg.Edges.allocate(ba.n_atoms, 2 * ka * ba.n_atoms, "cuda", dist=True),
            mg.Edges.allocate(bb.n_atoms, 2 * kb * bb.n_atoms, "cuda", dist=True),
            mg.Edges.allocate(ba.n_atoms, 2 * ka * ba.n_atoms, "cuda", dist=True)]
    # two calls in a row on one stream, no synchronisation between them: the second starts from the first one's scratch
    mg.mg_symmetrize_static(knn_a, ba.n_atoms, outs[0])
    mg.mg_symmetrize_static(knn_b, bb.n_atoms, outs[1])
    torch.cuda.synchronize()
    free_before = torch.cuda.mem_get_info()[0]
    # ... and the first graph again, after the scratch held a graph of other sizes
    mg.mg_symmetrize_static(knn_a, ba.n_atoms, outs[2])
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before              # nothing was allocated on the device
    deg_a, deg_b = np.full(ba.n_atoms, ka), np.full(bb.n_atoms, kb)
    _same_graph(outs[0].to_numpy(), ref_a, deg_a)
    _same_graph(outs[1].to_numpy(), ref_b, deg_b)
    _same_graph(outs[2].to_numpy(), ref_a, deg_a)


def test_static_symmetrize_capacity_and_limits(mg, ctx):
    import torch
    b, k = C.config_batch(0), 8
    knn, ref = _knn_and_reference(mg, ctx, b, k)
    # too small an output: the required count comes back in n_edges, rows are cut off at the capacity
    small = mg.Edges.allocate(b.n_atoms, k * b.n_atoms, "cuda", dist=True)
    mg.mg_symmetrize_static(knn, b.n_atoms, small)
    torch.cuda.synchronize()
    got = small.to_numpy()
    assert got["n_edges"] == ref["n_edges"] > k * b.n_atoms
    assert np.array_equal(got["row_ptr"], ref["row_ptr"])
    # the next call is not affected by the overflow of the last one
    full = mg.Edges.allocate(b.n_atoms, 2 * k * b.n_atoms, "cuda", dist=True)
    mg.mg_symmetrize_static(knn, b.n_atoms, full)
    torch.cuda.synchronize()
    _same_graph(full.to_numpy(), ref, np.full(b.n_atoms, k))
    # sizes beyond the static scratch are refused with their own status, nothing is launched
    big_atoms = mg.Edges.allocate(mg.MG_STATIC_MAX_ATOMS + 1, 16, "cuda", dist=True)
    big_atoms.n_edges.zero_()
    with pytest.raises(mg.MatGraphError) as e:
        mg.mg_symmetrize_static(big_atoms, mg.MG_STATIC_MAX_ATOMS + 1, big_atoms)
    assert e.value.code == 8 and "static scratch" in str(e.value)
    big_edges = mg.Edges.allocate(4, mg.MG_STATIC_MAX_EDGES + 1, "cuda", dist=True)
    big_edges.n_edges.zero_()
    with pytest.raises(mg.MatGraphError) as e:
        mg.mg_symmetrize_static(big_edges, 4, big_edges)
    assert e.value.code == 8
    # at the limits themselves the call is accepted (an empty graph of the largest sizes)
    edge_case = mg.Edges.allocate(mg.MG_STATIC_MAX_ATOMS, mg.MG_STATIC_MAX_EDGES, "cuda", dist=True)
    edge_case.row_ptr.zero_()
    edge_case.n_edges.zero_()
    out = mg.Edges.allocate(mg.MG_STATIC_MAX_ATOMS, 16, "cuda", dist=True)
    mg.mg_symmetrize_static(edge_case, mg.MG_STATIC_MAX_ATOMS, out)
    torch.cuda.synchronize()
    assert int(out.n_edges.item()) == 0 and int(out.row_ptr.abs().max().item()) == 0
