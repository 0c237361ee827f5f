"""ctypes front end of the FP64 CPU oracle (oracle/mg_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It imports nothing from the CUDA package and the CUDA package never imports
it.  `build()` compiles the C file with gcc (-O2 -fopenmp -ffp-contract=off) next to the source.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mg_oracle.c")
_LIB = os.path.join(_HERE, "libmgoracle.so")
_lib = None


class _Graph(ctypes.Structure):
    _fields_ = [("n_edges", ctypes.c_int64), ("n_atoms", ctypes.c_int64),
                ("row_ptr", ctypes.POINTER(ctypes.c_int64)),
                ("src", ctypes.POINTER(ctypes.c_int32)), ("dst", ctypes.POINTER(ctypes.c_int32)),
                ("tau", ctypes.POINTER(ctypes.c_int32)), ("vec", ctypes.POINTER(ctypes.c_double)),
                ("dist", ctypes.POINTER(ctypes.c_double)), ("n_box", ctypes.c_double),
                ("n_evaluated", ctypes.c_int64), ("kth_dist", ctypes.POINTER(ctypes.c_double)),
                ("max_abs_tau", ctypes.c_int32 * 3), ("bad_struct", ctypes.c_int32)]


def build(force: bool = False) -> str:
    """Compile the oracle if the .so is missing or older than the source."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB)
        fp = ctypes.POINTER(ctypes.c_float)
        ip = ctypes.POINTER(ctypes.c_int32)
        lib.mgo_cutoff_graph.argtypes = [fp, fp, ip, ctypes.c_int32, ctypes.c_double, ctypes.POINTER(_Graph)]
        lib.mgo_cutoff_graph.restype = ctypes.c_int
        lib.mgo_knn_graph.argtypes = [fp, fp, ip, ctypes.c_int32, ctypes.c_int32, ctypes.POINTER(_Graph)]
        lib.mgo_knn_graph.restype = ctypes.c_int
        lib.mgo_free.argtypes = [ctypes.POINTER(_Graph)]
        lib.mgo_free.restype = None
        lib.mgo_cutoff_graph_radii.argtypes = [fp, fp, ip, ctypes.c_int32, fp, ctypes.POINTER(_Graph)]
        lib.mgo_cutoff_graph_radii.restype = ctypes.c_int
        lib.mgo_num_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def num_threads() -> int:
    return int(_load().mgo_num_threads())


def _prep(pos, lattice, struct_ptr):
    pos = np.ascontiguousarray(pos, dtype=np.float32).reshape(-1, 3)
    lattice = np.ascontiguousarray(lattice, dtype=np.float32).reshape(-1, 3, 3)
    struct_ptr = np.ascontiguousarray(struct_ptr, dtype=np.int32)
    assert struct_ptr.shape[0] == lattice.shape[0] + 1
    assert struct_ptr[0] == 0 and struct_ptr[-1] == pos.shape[0]
    return pos, lattice, struct_ptr


def _ptr(a, ct):
    return a.ctypes.data_as(ctypes.POINTER(ct))


def _take(g: _Graph, knn: bool) -> dict:
    e, n = int(g.n_edges), int(g.n_atoms)

    def arr(p, count, dtype):
        if count == 0:
            return np.zeros(0, dtype=dtype)
        return np.ctypeslib.as_array(p, shape=(count,)).astype(dtype, copy=True)

    out = dict(
        n_edges=e,
        row_ptr=arr(g.row_ptr, n + 1, np.int64),
        src=arr(g.src, e, np.int32), dst=arr(g.dst, e, np.int32),
        tau=arr(g.tau, 3 * e, np.int32).reshape(-1, 3),
        vec=arr(g.vec, 3 * e, np.float64).reshape(-1, 3),
        dist=arr(g.dist, e, np.float64),
        n_box=float(g.n_box), n_evaluated=int(g.n_evaluated),
        max_abs_tau=np.array(list(g.max_abs_tau), dtype=np.int32),
    )
    if knn:
        out["kth_dist"] = arr(g.kth_dist, n, np.float64)
    return out


def cutoff_graph(pos, lattice, struct_ptr, r_c: float) -> dict:
    """Def. 3 by brute force.  Edges come back in canonical order
    (src, dst, tau_x, tau_y, tau_z).  r_c is compared as (double)(float)r_c (R15)."""
    lib = _load()
    pos, lattice, struct_ptr = _prep(pos, lattice, struct_ptr)
    g = _Graph()
    rc = float(np.float32(r_c))
    rcode = lib.mgo_cutoff_graph(_ptr(pos, ctypes.c_float), _ptr(lattice, ctypes.c_float),
                                 _ptr(struct_ptr, ctypes.c_int32), lattice.shape[0], rc, ctypes.byref(g))
    if rcode != 0:
        raise ValueError(f"singular or non-finite lattice in structure {g.bad_struct}")
    try:
        return _take(g, knn=False)
    finally:
        lib.mgo_free(ctypes.byref(g))


def cutoff_graph_radii(pos, lattice, struct_ptr, radii) -> dict:
    """Def. 3 with one cutoff per SOURCE atom ("c_i > 0"): edge (i, j, tau) iff d < c_i."""
    lib = _load()
    pos, lattice, struct_ptr = _prep(pos, lattice, struct_ptr)
    radii = np.ascontiguousarray(radii, dtype=np.float32)
    assert radii.shape == (pos.shape[0],)
    g = _Graph()
    rcode = lib.mgo_cutoff_graph_radii(_ptr(pos, ctypes.c_float), _ptr(lattice, ctypes.c_float),
                                       _ptr(struct_ptr, ctypes.c_int32), lattice.shape[0],
                                       _ptr(radii, ctypes.c_float), ctypes.byref(g))
    if rcode == 2:
        raise ValueError("a radius is not a positive finite number")
    if rcode != 0:
        raise ValueError(f"singular or non-finite lattice in structure {g.bad_struct}")
    try:
        return _take(g, knn=False)
    finally:
        lib.mgo_free(ctypes.byref(g))


def knn_graph(pos, lattice, struct_ptr, k: int) -> dict:
    """Exactly k edges per atom, rows sorted by (distance, dst, tau) (Alg. 2; R2, R8)."""
    lib = _load()
    pos, lattice, struct_ptr = _prep(pos, lattice, struct_ptr)
    g = _Graph()
    rcode = lib.mgo_knn_graph(_ptr(pos, ctypes.c_float), _ptr(lattice, ctypes.c_float),
                              _ptr(struct_ptr, ctypes.c_int32), lattice.shape[0], int(k), ctypes.byref(g))
    if rcode != 0:
        raise ValueError(f"singular or non-finite lattice in structure {g.bad_struct}")
    try:
        return _take(g, knn=True)
    finally:
        lib.mgo_free(ctypes.byref(g))


def edge_distance(pos, lattice, struct_ptr, src, dst, tau):
    """FP64 distance and vector of given (src, dst, tau) triples, oracle operation order.
    Vectorised numpy restatement used by the parity checker for edges the oracle did not emit."""
    pos, lattice, struct_ptr = _prep(pos, lattice, struct_ptr)
    src = np.asarray(src, dtype=np.int64)
    dst = np.asarray(dst, dtype=np.int64)
    tau = np.asarray(tau, dtype=np.float64).reshape(-1, 3)
    s_of = np.searchsorted(struct_ptr, src, side="right") - 1
    A = lattice.astype(np.float64)[s_of]                         # [E,3,3]
    f = (pos.astype(np.float64)[dst] - pos.astype(np.float64)[src]) + tau
    v = f[:, 0, None] * A[:, 0, :] + f[:, 1, None] * A[:, 1, :] + f[:, 2, None] * A[:, 2, :]
    d = np.sqrt(v[:, 0] * v[:, 0] + v[:, 1] * v[:, 1] + v[:, 2] * v[:, 2])
    return d, v
