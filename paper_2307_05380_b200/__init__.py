"""paper_2307_05380_b200 — thin Python binding of libmatgraph.so (include/matgraph.h).

Argument marshalling only: torch supplies device memory and the current CUDA stream; every step
of the graph construction (search bounds, image enumeration, distance filter, scan, emission,
top-k) runs in the sm_100a kernels under csrc/.  There is no CPU path: importing works anywhere
(the library is built and its symbols are checked), but creating a `Context` without a CUDA device
raises.  The functions mirror the C ABI one to one (`mg_cutoff_graph`, `mg_knn_graph`,
`mg_update_graph`, ...); `Context` wraps them for convenience.
"""
from __future__ import annotations

import ctypes
import dataclasses
import os
from typing import Optional

import numpy as np

from ._build import LIB, build

MG_KIND_CUTOFF, MG_KIND_KNN = 0, 1
MG_MAX_K = 64
EXPORTS = ["mg_create", "mg_destroy", "mg_reserve", "mg_cutoff_graph", "mg_cutoff_count",
           "mg_knn_graph", "mg_graph_create", "mg_graph_destroy", "mg_update_graph",
           "mg_cutoff_graph_host", "mg_knn_graph_host", "mg_check", "mg_launch_count",
           "mg_status_string", "mg_set_profile", "mg_profile_read", "mg_symmetrize", "mg_triplets_graph", "mg_cutoff_graph_radii",
           "mg_symmetrize_static"]


class MatGraphError(RuntimeError):
    def __init__(self, code: int, what: str):
        super().__init__(f"{what}: {_lib().mg_status_string(code).decode()} (mg_status {code})")
        self.code = code


class _Edges(ctypes.Structure):
    _fields_ = [("row_ptr", ctypes.c_void_p), ("src", ctypes.c_void_p), ("dst", ctypes.c_void_p),
                ("offset", ctypes.c_void_p), ("vec", ctypes.c_void_p), ("dist", ctypes.c_void_p),
                ("capacity", ctypes.c_int64), ("n_edges", ctypes.c_void_p)]


_LIBH = None


class _Triplets(ctypes.Structure):
    _fields_ = [("tri_ptr", ctypes.c_void_p), ("edge_a", ctypes.c_void_p), ("edge_b", ctypes.c_void_p),
                ("capacity", ctypes.c_int64), ("n_triplets", ctypes.c_void_p)]


def _lib():
    """Load (building first if needed) libmatgraph.so; fails loudly when it cannot be had."""
    global _LIBH
    if _LIBH is None:
        path = build()
        lib = ctypes.CDLL(path)
        vp, i32, i64, f32 = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_float
        ep = ctypes.POINTER(_Edges)
        lib.mg_create.argtypes = [ctypes.POINTER(vp), ctypes.c_int]
        lib.mg_destroy.argtypes = [vp]
        lib.mg_destroy.restype = None
        lib.mg_reserve.argtypes = [vp, i32, i32]
        lib.mg_cutoff_graph.argtypes = [vp, vp, vp, vp, i32, i32, f32, ep, vp]
        lib.mg_cutoff_count.argtypes = [vp, vp, vp, vp, i32, i32, f32, ctypes.POINTER(i64), vp]
        lib.mg_knn_graph.argtypes = [vp, vp, vp, vp, i32, i32, i32, ep, vp]
        lib.mg_graph_create.argtypes = [vp, ctypes.c_int, f32, i32, vp, i32, i32, ctypes.POINTER(vp)]
        lib.mg_graph_destroy.argtypes = [vp]
        lib.mg_graph_destroy.restype = None
        lib.mg_update_graph.argtypes = [vp, vp, vp, vp, ep, vp]
        lib.mg_cutoff_graph_host.argtypes = [vp, vp, vp, vp, i32, i32, f32, ep]
        lib.mg_knn_graph_host.argtypes = [vp, vp, vp, vp, i32, i32, i32, ep]
        lib.mg_check.argtypes = [vp, vp]
        lib.mg_launch_count.argtypes = [vp]
        lib.mg_launch_count.restype = i64
        lib.mg_set_profile.argtypes = [vp, ctypes.c_int]
        lib.mg_profile_read.argtypes = [vp, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(i64)]
        lib.mg_cutoff_graph_radii.argtypes = [vp, vp, vp, vp, i32, i32, vp, ep, vp]
        lib.mg_symmetrize.argtypes = [vp, ep, i32, ep, vp]
        lib.mg_symmetrize_static.argtypes = [i32, ep, i32, ep, vp]
        lib.mg_triplets_graph.argtypes = [vp, vp, i32, ctypes.POINTER(_Triplets), vp]
        lib.mg_status_string.argtypes = [ctypes.c_int]
        lib.mg_status_string.restype = ctypes.c_char_p
        _LIBH = lib
    return _LIBH


def library_path() -> str:
    return LIB


def _torch():
    import torch
    return torch


@dataclasses.dataclass
class Edges:
    """Caller-owned output buffers of one graph call (device tensors)."""
    row_ptr: "torch.Tensor"   # int32 [n_atoms+1]
    src: "torch.Tensor"       # int32 [capacity]
    dst: "torch.Tensor"       # int32 [capacity]
    offset: "torch.Tensor"    # int8  [capacity,3]
    vec: "torch.Tensor"       # float32 [capacity,3]
    dist: Optional["torch.Tensor"]
    n_edges: "torch.Tensor"   # int64 [1]
    capacity: int

    @staticmethod
    def allocate(n_atoms: int, capacity: int, device, dist: bool = False) -> "Edges":
        torch = _torch()
        cap = max(int(capacity), 1)
        return Edges(row_ptr=torch.empty(n_atoms + 1, dtype=torch.int32, device=device),
                     src=torch.empty(cap, dtype=torch.int32, device=device),
                     dst=torch.empty(cap, dtype=torch.int32, device=device),
                     offset=torch.empty((cap, 3), dtype=torch.int8, device=device),
                     vec=torch.empty((cap, 3), dtype=torch.float32, device=device),
                     dist=torch.empty(cap, dtype=torch.float32, device=device) if dist else None,
                     n_edges=torch.zeros(1, dtype=torch.int64, device=device), capacity=int(capacity))

    def _c(self) -> _Edges:
        return _Edges(self.row_ptr.data_ptr(), self.src.data_ptr(), self.dst.data_ptr(),
                      self.offset.data_ptr(), self.vec.data_ptr(),
                      self.dist.data_ptr() if self.dist is not None else None,
                      self.capacity, self.n_edges.data_ptr())

    def to_numpy(self) -> dict:
        """Synchronises; returns the valid prefix of every array as numpy."""
        e = int(self.n_edges.item())
        m = min(e, self.capacity)
        return dict(n_edges=e, row_ptr=self.row_ptr.cpu().numpy(), src=self.src[:m].cpu().numpy(),
                    dst=self.dst[:m].cpu().numpy(), offset=self.offset[:m].cpu().numpy(),
                    vec=self.vec[:m].cpu().numpy(),
                    dist=self.dist[:m].cpu().numpy() if self.dist is not None else None)


def _check_inputs(pos, lattice, struct_ptr):
    torch = _torch()
    assert pos.is_cuda and lattice.is_cuda and struct_ptr.is_cuda, "inputs must be CUDA tensors"
    assert pos.dtype == torch.float32 and lattice.dtype == torch.float32 and struct_ptr.dtype == torch.int32
    assert pos.is_contiguous() and lattice.is_contiguous() and struct_ptr.is_contiguous()
    n_struct = struct_ptr.numel() - 1
    n_atoms = pos.shape[0] if pos.dim() == 2 else pos.numel() // 3
    assert lattice.numel() == 9 * n_struct and pos.numel() == 3 * n_atoms
    return n_struct, n_atoms


def _stream():
    return ctypes.c_void_p(_torch().cuda.current_stream().cuda_stream)


class Graph:
    """mg_graph handle: fixed (kind, r_c | k, struct_ptr), regenerated by Context.update_graph."""

    def __init__(self, ctx: "Context", handle, kind, struct_ptr, n_struct, n_atoms, r_c, k):
        self.ctx, self._h, self.kind = ctx, handle, kind
        self.struct_ptr, self.n_struct, self.n_atoms, self.r_c, self.k = struct_ptr, n_struct, n_atoms, r_c, k

    def close(self):
        if self._h is not None:
            _lib().mg_graph_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Context:
    """mg_ctx handle.  One context serves one stream at a time."""

    def __init__(self, device: int = 0):
        torch = _torch()
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2307_05380_b200 needs a CUDA device (sm_100a); there is no CPU fallback")
        self.device = torch.device("cuda", device)
        h = ctypes.c_void_p()
        rc = _lib().mg_create(ctypes.byref(h), device)
        if rc != 0:
            raise MatGraphError(rc, "mg_create")
        self._h = h

    def close(self):
        if getattr(self, "_h", None) is not None:
            _lib().mg_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- C ABI, one to one -------------------------------------------------------------
    def mg_reserve(self, n_struct: int, n_atoms: int):
        rc = _lib().mg_reserve(self._h, n_struct, n_atoms)
        if rc != 0:
            raise MatGraphError(rc, "mg_reserve")

    def mg_cutoff_count(self, pos, lattice, struct_ptr, r_c: float) -> int:
        n_struct, n_atoms = _check_inputs(pos, lattice, struct_ptr)
        out = ctypes.c_int64(0)
        rc = _lib().mg_cutoff_count(self._h, pos.data_ptr(), lattice.data_ptr(), struct_ptr.data_ptr(),
                                    n_struct, n_atoms, float(r_c), ctypes.byref(out), _stream())
        if rc != 0:
            raise MatGraphError(rc, "mg_cutoff_count")
        return int(out.value)

    def mg_cutoff_graph(self, pos, lattice, struct_ptr, r_c: float, out: Edges) -> Edges:
        n_struct, n_atoms = _check_inputs(pos, lattice, struct_ptr)
        assert out.row_ptr.numel() == n_atoms + 1
        rc = _lib().mg_cutoff_graph(self._h, pos.data_ptr(), lattice.data_ptr(), struct_ptr.data_ptr(),
                                    n_struct, n_atoms, float(r_c), ctypes.byref(out._c()), _stream())
        if rc != 0:
            raise MatGraphError(rc, "mg_cutoff_graph")
        return out

    def mg_knn_graph(self, pos, lattice, struct_ptr, k: int, out: Edges) -> Edges:
        n_struct, n_atoms = _check_inputs(pos, lattice, struct_ptr)
        assert out.row_ptr.numel() == n_atoms + 1
        rc = _lib().mg_knn_graph(self._h, pos.data_ptr(), lattice.data_ptr(), struct_ptr.data_ptr(),
                                 n_struct, n_atoms, int(k), ctypes.byref(out._c()), _stream())
        if rc != 0:
            raise MatGraphError(rc, "mg_knn_graph")
        return out

    def mg_graph_create(self, kind: int, struct_ptr, n_atoms: int, r_c: float = 0.0, k: int = 0) -> Graph:
        n_struct = struct_ptr.numel() - 1
        h = ctypes.c_void_p()
        rc = _lib().mg_graph_create(self._h, kind, float(r_c), int(k), struct_ptr.data_ptr(), n_struct,
                                    n_atoms, ctypes.byref(h))
        if rc != 0:
            raise MatGraphError(rc, "mg_graph_create")
        return Graph(self, h, kind, struct_ptr, n_struct, n_atoms, r_c, k)

    def mg_update_graph(self, graph: Graph, pos, lattice, out: Edges) -> Edges:
        _check_inputs(pos, lattice, graph.struct_ptr)
        rc = _lib().mg_update_graph(self._h, graph._h, pos.data_ptr(), lattice.data_ptr(),
                                    ctypes.byref(out._c()), _stream())
        if rc != 0:
            raise MatGraphError(rc, "mg_update_graph")
        return out

    def mg_cutoff_graph_radii(self, pos, lattice, struct_ptr, radii, out: Edges) -> Edges:
        n_struct, n_atoms = _check_inputs(pos, lattice, struct_ptr)
        assert radii.is_cuda and radii.dtype == _torch().float32 and radii.numel() == n_atoms and radii.is_contiguous()
        rc = _lib().mg_cutoff_graph_radii(self._h, pos.data_ptr(), lattice.data_ptr(), struct_ptr.data_ptr(),
                                          n_struct, n_atoms, radii.data_ptr(), ctypes.byref(out._c()), _stream())
        if rc != 0:
            raise MatGraphError(rc, "mg_cutoff_graph_radii")
        return out

    def mg_symmetrize(self, inp: Edges, n_atoms: int, out: Edges) -> Edges:
        rc = _lib().mg_symmetrize(self._h, ctypes.byref(inp._c()), n_atoms, ctypes.byref(out._c()), _stream())
        if rc != 0:
            raise MatGraphError(rc, "mg_symmetrize")
        return out

    def mg_triplets_graph(self, row_ptr, n_atoms: int, capacity: int) -> dict:
        """Allocates tri_ptr / edge_a / edge_b (device tensors) and runs mg_triplets_graph."""
        torch = _torch()
        cap = max(int(capacity), 1)
        out = dict(tri_ptr=torch.empty(n_atoms + 1, dtype=torch.int64, device=row_ptr.device),
                   edge_a=torch.empty(cap, dtype=torch.int32, device=row_ptr.device),
                   edge_b=torch.empty(cap, dtype=torch.int32, device=row_ptr.device),
                   n_triplets=torch.zeros(1, dtype=torch.int64, device=row_ptr.device), capacity=int(capacity))
        c = _Triplets(out["tri_ptr"].data_ptr(), out["edge_a"].data_ptr(), out["edge_b"].data_ptr(), int(capacity),
                      out["n_triplets"].data_ptr())
        rc = _lib().mg_triplets_graph(self._h, row_ptr.data_ptr(), n_atoms, ctypes.byref(c), _stream())
        if rc != 0:
            raise MatGraphError(rc, "mg_triplets_graph")
        return out

    def mg_check(self) -> int:
        """Synchronises the current stream; returns the mg_status recorded by the kernels."""
        return int(_lib().mg_check(self._h, _stream()))

    def mg_launch_count(self) -> int:
        return int(_lib().mg_launch_count(self._h))

    def mg_set_profile(self, on: bool):
        rc = _lib().mg_set_profile(self._h, 1 if on else 0)
        if rc != 0:
            raise MatGraphError(rc, "mg_set_profile")

    def mg_profile_read(self) -> dict:
        """Mean kernel durations (ms) since mg_set_profile(True): prep, count, emit, knn."""
        ms = (ctypes.c_double * 4)()
        n = (ctypes.c_int64 * 4)()
        rc = _lib().mg_profile_read(self._h, ms, n)
        if rc != 0:
            raise MatGraphError(rc, "mg_profile_read")
        names = ("prep", "count", "emit", "knn")
        return {k: dict(ms=float(ms[i]), calls=int(n[i])) for i, k in enumerate(names)}

    # ---- host-buffer calls (numpy in, numpy out; copies inside the call) ----------------
    def _host(self, fn, pos, lattice, struct_ptr, param, capacity, dist):
        pos = np.ascontiguousarray(pos, np.float32).reshape(-1, 3)
        lattice = np.ascontiguousarray(lattice, np.float32).reshape(-1, 3, 3)
        struct_ptr = np.ascontiguousarray(struct_ptr, np.int32)
        n_struct, n_atoms = lattice.shape[0], pos.shape[0]
        cap = max(int(capacity), 1)
        o = dict(row_ptr=np.empty(n_atoms + 1, np.int32), src=np.empty(cap, np.int32),
                 dst=np.empty(cap, np.int32), offset=np.empty((cap, 3), np.int8),
                 vec=np.empty((cap, 3), np.float32), dist=np.empty(cap, np.float32) if dist else None,
                 n_edges=np.zeros(1, np.int64))
        ce = _Edges(o["row_ptr"].ctypes.data, o["src"].ctypes.data, o["dst"].ctypes.data,
                    o["offset"].ctypes.data, o["vec"].ctypes.data,
                    o["dist"].ctypes.data if dist else None, int(capacity), o["n_edges"].ctypes.data)
        rc = fn(self._h, pos.ctypes.data, lattice.ctypes.data, struct_ptr.ctypes.data, n_struct, n_atoms,
                param, ctypes.byref(ce))
        e = int(o["n_edges"][0])
        m = min(e, int(capacity))
        res = dict(status=int(rc), n_edges=e, row_ptr=o["row_ptr"], src=o["src"][:m], dst=o["dst"][:m],
                   offset=o["offset"][:m], vec=o["vec"][:m], dist=o["dist"][:m] if dist else None)
        return res

    def mg_cutoff_graph_host(self, pos, lattice, struct_ptr, r_c: float, capacity: int, dist=False) -> dict:
        return self._host(_lib().mg_cutoff_graph_host, pos, lattice, struct_ptr, ctypes.c_float(r_c), capacity, dist)

    def mg_knn_graph_host(self, pos, lattice, struct_ptr, k: int, dist=False) -> dict:
        n_atoms = np.asarray(pos).reshape(-1, 3).shape[0]
        return self._host(_lib().mg_knn_graph_host, pos, lattice, struct_ptr, ctypes.c_int32(k), k * n_atoms, dist)

    # ---- conveniences -------------------------------------------------------------------
    def cutoff_graph(self, pos, lattice, struct_ptr, r_c: float, capacity: Optional[int] = None,
                     dist: bool = False) -> Edges:
        """Allocates the outputs (exact size via mg_cutoff_count when capacity is None) and runs
        mg_cutoff_graph."""
        _, n_atoms = _check_inputs(pos, lattice, struct_ptr)
        if capacity is None:
            capacity = self.mg_cutoff_count(pos, lattice, struct_ptr, r_c)
        out = Edges.allocate(n_atoms, capacity, pos.device, dist)
        return self.mg_cutoff_graph(pos, lattice, struct_ptr, r_c, out)

    def knn_graph(self, pos, lattice, struct_ptr, k: int, dist: bool = False) -> Edges:
        _, n_atoms = _check_inputs(pos, lattice, struct_ptr)
        out = Edges.allocate(n_atoms, k * n_atoms, pos.device, dist)
        return self.mg_knn_graph(pos, lattice, struct_ptr, k, out)


# limits of mg_symmetrize_static (include/matgraph.h)
MG_STATIC_MAX_ATOMS = 65536
MG_STATIC_MAX_EDGES = 4194304


def mg_symmetrize_static(inp: Edges, n_atoms: int, out: Edges, device: int = 0) -> Edges:
    """mg_symmetrize without a context and without any allocation by the library (static device scratch;
    n_atoms <= MG_STATIC_MAX_ATOMS, inp.capacity <= MG_STATIC_MAX_EDGES).  Calls on one device must not
    overlap on the GPU."""
    rc = _lib().mg_symmetrize_static(device, ctypes.byref(inp._c()), n_atoms, ctypes.byref(out._c()), _stream())
    if rc != 0:
        raise MatGraphError(rc, "mg_symmetrize_static")
    return out


def to_device(batch, device="cuda"):
    """(pos, lattice, struct_ptr) device tensors of a workloads.crystals.Batch-like object."""
    torch = _torch()
    return (torch.from_numpy(np.ascontiguousarray(batch.pos)).to(device),
            torch.from_numpy(np.ascontiguousarray(batch.lattice)).to(device),
            torch.from_numpy(np.ascontiguousarray(batch.struct_ptr)).to(device))
