"""Host logic of the multi-GPU path, world_size 2 over gloo on CPU: the
batch is sharded by structures, every rank builds the graph of its shard (here with the oracle —
no GPU in this test), one all_gather of the counts stitches the CSRs; the result must equal the
graph of the whole batch."""
import os
import socket

import numpy as np
import pytest

from workloads import crystals as C
from paper_2307_05380_b200 import shard


def test_shard_ranges_cover_and_balance():
    b = C.small_batch(300, seed=4)
    for world in (1, 2, 3, 8):
        rs = shard.shard_ranges(b.struct_ptr, world)
        assert rs[0][0] == 0 and rs[-1][1] == b.n_struct
        assert all(rs[i][1] == rs[i + 1][0] for i in range(world - 1))
        n = np.diff(b.struct_ptr).astype(np.int64)
        w = np.array([np.sum(n[a:c] ** 2) for a, c in rs], float)
        assert w.max() <= 1.2 * w.mean() + 400 + 1e-9
    # more ranks than structures: empty shards are legal
    rs = shard.shard_ranges(np.array([0, 3, 5], np.int32), 4)
    assert rs[0][0] == 0 and rs[-1][1] == 2 and sum(c - a for a, c in rs) == 2


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out_dir):
    import torch.distributed as dist
    import oracle
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    b = C.small_batch(40, seed=12)
    pos, lat, ptr, a0, s0 = shard.shard_batch(b.pos, b.lattice, b.struct_ptr, rank, world)
    g = oracle.cutoff_graph(pos, lat, ptr, 5.0)
    st = shard.stitch(g, pos.shape[0], None)
    assert st["atom_offset"] == a0
    np.savez(os.path.join(out_dir, f"r{rank}.npz"), row_ptr=st["row_ptr"], src=st["src"], dst=st["dst"],
             tau=g["tau"], n_edges_global=st["n_edges_global"], n_atoms_global=st["n_atoms_global"])
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.timeout(300)
def test_two_rank_stitch_equals_whole_batch(tmp_path):
    import torch.multiprocessing as mp
    import oracle
    world = 2
    mp.spawn(_worker, args=(world, _free_port(), str(tmp_path)), nprocs=world, join=True)
    b = C.small_batch(40, seed=12)
    ref = oracle.cutoff_graph(b.pos, b.lattice, b.struct_ptr, 5.0)
    parts = [np.load(os.path.join(str(tmp_path), f"r{r}.npz")) for r in range(world)]
    assert int(parts[0]["n_edges_global"]) == ref["n_edges"] and int(parts[0]["n_atoms_global"]) == b.n_atoms
    src = np.concatenate([p["src"] for p in parts])
    dst = np.concatenate([p["dst"] for p in parts])
    tau = np.concatenate([p["tau"] for p in parts])
    row_ptr = np.concatenate([parts[0]["row_ptr"][:-1], parts[1]["row_ptr"]])
    assert np.array_equal(src, ref["src"]) and np.array_equal(dst, ref["dst"]) and np.array_equal(tau, ref["tau"])
    assert np.array_equal(row_ptr, ref["row_ptr"])
