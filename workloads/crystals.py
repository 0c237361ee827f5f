"""Seeded synthetic crystal batches — the ONLY module shared by the oracle side and the CUDA side.

It produces inputs (FP32 fractional positions, FP32 lattices, int32 struct_ptr) shaped like the
paper's Materials-Project workload (small triclinic cells with a few to tens of atoms) and
like the five BASELINE.json configs.  The Materials Project records themselves are not in this
container and none of them is reproduced here; these batches stand in for them.

It holds none of the graph method's arithmetic: no search bounds, no edge predicate, no k-nearest
selection.  The only geometry in here is what the *input recipe* itself needs — building a cell
from lengths/angles, the "valid cell" rejection and the minimum-distance
rejection of atom placements (R19) — written locally in numpy so that neither `oracle/` nor the
CUDA library is imported.

Per-structure random streams are keyed by (seed, family, structure index): a smaller batch is a
prefix of a larger batch of the same family.
"""
from __future__ import annotations

import dataclasses
from typing import Iterator

import numpy as np

# ----------------------------------------------------------------------------- families
FAMILY_SMALL = 0      # BASELINE.json configs[0..2]
FAMILY_SUPERCELL = 1  # configs[3]
FAMILY_SKEWED = 2     # configs[4] initial states
FAMILY_WALK = 3       # configs[4] per-step noise streams
FAMILY_PAPER = 4      # cells of up to 64 atoms, the shape of the paper's own workload


@dataclasses.dataclass
class Batch:
    """One batch of crystals in the layout the C-ABI takes (include/matgraph.h)."""
    pos: np.ndarray         # float32 [n_atoms, 3] fractional coordinates (Def. 1)
    lattice: np.ndarray     # float32 [n_struct, 3, 3] row-major, ROWS = lattice vectors
    struct_ptr: np.ndarray  # int32   [n_struct + 1]

    @property
    def n_struct(self) -> int:
        return int(self.struct_ptr.shape[0] - 1)

    @property
    def n_atoms(self) -> int:
        return int(self.pos.shape[0])


# ----------------------------------------------------------------------------- cell helpers
def cell_from_parameters(a, b, c, alpha_deg, beta_deg, gamma_deg) -> np.ndarray:
    """Rows a1,a2,a3 of the cell in the standard orientation (a1 along x, a2 in the xy plane)."""
    al, be, ga = np.deg2rad([alpha_deg, beta_deg, gamma_deg])
    ca, cb, cg = np.cos(al), np.cos(be), np.cos(ga)
    sg = np.sin(ga)
    g = 1.0 - ca * ca - cb * cb - cg * cg + 2.0 * ca * cb * cg  # Gram factor, R18
    if g <= 0.0 or sg <= 0.0:
        return None
    a3y = (ca - cb * cg) / sg
    a3z = np.sqrt(g) / sg
    return np.array([[a, 0.0, 0.0],
                     [b * cg, b * sg, 0.0],
                     [c * cb, c * a3y, c * a3z]], dtype=np.float64)


def gram_factor(alpha_deg, beta_deg, gamma_deg) -> float:
    ca, cb, cg = np.cos(np.deg2rad([alpha_deg, beta_deg, gamma_deg]))
    return float(1.0 - ca * ca - cb * cb - cg * cg + 2.0 * ca * cb * cg)


def _spacings(cell: np.ndarray) -> np.ndarray:
    """Distances between opposite faces of the cell(s); cell [...,3,3] float64 -> [...,3]."""
    a1, a2, a3 = cell[..., 0, :], cell[..., 1, :], cell[..., 2, :]
    c23, c31, c12 = np.cross(a2, a3), np.cross(a3, a1), np.cross(a1, a2)
    vol = np.abs(np.sum(a1 * c23, axis=-1))
    norms = np.stack([np.linalg.norm(c23, axis=-1), np.linalg.norm(c31, axis=-1),
                      np.linalg.norm(c12, axis=-1)], axis=-1)
    return vol[..., None] / norms


def _draw_cell(rng, len_lo, len_hi, ang_lo, ang_hi, g_min=1e-3, h_min=1.0):
    """R18: redraw until the Gram factor > g_min and every face spacing >= h_min on the
    FP32-rounded cell."""
    while True:
        a, b, c = rng.uniform(len_lo, len_hi, 3)
        al, be, ga = rng.uniform(ang_lo, ang_hi, 3)
        if gram_factor(al, be, ga) <= g_min:
            continue
        cell = cell_from_parameters(a, b, c, al, be, ga)
        if cell is None:
            continue
        cell32 = cell.astype(np.float32)
        if not np.all(np.isfinite(cell32)):
            continue
        if _spacings(cell32.astype(np.float64)).min() < h_min:
            continue
        return cell32


def _too_close(x_new, x_old, cell64, dmin, reach):
    """True if the candidate fractional point x_new has any periodic image of any point in x_old
    (or of itself) closer than dmin.  reach[a] = images to scan along axis a."""
    r0, r1, r2 = (np.arange(-m, m + 1) for m in reach)
    tau = np.stack(np.meshgrid(r0, r1, r2, indexing="ij"), axis=-1).reshape(-1, 3).astype(np.float64)
    shifts = tau @ cell64                                   # [T,3]
    if x_old.shape[0]:
        d = (x_old - x_new) @ cell64                        # [n,3]
        v = d[:, None, :] + shifts[None, :, :]
        if np.min(np.einsum("ntc,ntc->nt", v, v)) < dmin * dmin:
            return True
    nz = np.any(tau != 0.0, axis=1)
    s = shifts[nz]
    return bool(np.min(np.einsum("tc,tc->t", s, s)) < dmin * dmin)


def _place_atoms(rng, n, cell32, dmin, max_tries=200):
    """R19: sequential insertion, <= max_tries uniform tries per atom; None if an atom cannot be
    placed (the caller then redraws the cell, keeping n)."""
    cell64 = cell32.astype(np.float64)
    h = _spacings(cell64)
    reach = [int(np.ceil(dmin / hh)) + 1 for hh in h]
    if dmin < 0.5 * h.min():        # nearest image suffices
        return _place_atoms_minimage(rng, n, cell64, dmin, max_tries)
    x = np.zeros((n, 3), dtype=np.float32)
    for i in range(n):
        for _ in range(max_tries):
            cand = rng.random(3, dtype=np.float32)
            if not _too_close(cand.astype(np.float64), x[:i].astype(np.float64), cell64, dmin, reach):
                x[i] = cand
                break
        else:
            return None
    return x


def _place_atoms_minimage(rng, n, cell64, dmin, max_tries):
    x = np.zeros((n, 3), dtype=np.float32)
    x64 = np.zeros((n, 3), dtype=np.float64)
    for i in range(n):
        for _ in range(max_tries):
            cand = rng.random(3, dtype=np.float32)
            if i:
                df = x64[:i] - cand.astype(np.float64)
                df -= np.rint(df)
                v = df @ cell64
                if np.min(np.einsum("nc,nc->n", v, v)) < dmin * dmin:
                    continue
            x[i] = cand
            x64[i] = cand
            break
        else:
            return None
    return x


def _rng(seed, family, index):
    return np.random.default_rng(np.random.SeedSequence([int(seed), int(family), int(index)]))


# ----------------------------------------------------------------------------- families
def small_crystal(seed: int, index: int, family=FAMILY_SMALL, n_lo=1, n_hi=20, len_lo=3.0,
                  len_hi=10.0, ang_lo=60.0, ang_hi=120.0, dmin=1.0):
    """One crystal of BASELINE.json configs[0..2] (and, with other ranges, configs[4])."""
    rng = _rng(seed, family, index)
    n = int(rng.integers(n_lo, n_hi + 1))
    while True:
        cell32 = _draw_cell(rng, len_lo, len_hi, ang_lo, ang_hi)
        x = _place_atoms(rng, n, cell32, dmin)
        if x is not None:
            return cell32, x


def supercell(seed: int, index: int, density=0.08, n_lo=500, n_hi=2000, dmin=1.2):
    """One crystal of configs[3]: N = round(density*V) must land in [n_lo, n_hi] (R21)."""
    rng = _rng(seed, FAMILY_SUPERCELL, index)
    while True:
        cell32 = _draw_cell(rng, 20.0, 35.0, 75.0, 105.0)
        vol = abs(np.linalg.det(cell32.astype(np.float64)))
        n = int(round(density * vol))
        if not (n_lo <= n <= n_hi):
            continue
        x = _place_atoms(rng, n, cell32, dmin)
        if x is not None:
            return cell32, x


def paper_scale_crystal(seed: int, index: int, n_hi=64, vol_per_atom=18.0, dmin=1.0):
    """One crystal shaped like the paper's workload (Materials Project structures of at
    most 64 atoms; NOT a record of that dataset): N ~ U{1..n_hi}, cell lengths (0.8 .. 1.5) x the cube root
    of vol_per_atom * N (>= 3 A), angles U(60, 120) degrees, 1.0 A periodic minimum distance."""
    rng = _rng(seed, FAMILY_PAPER, index)
    n = int(rng.integers(1, n_hi + 1))
    side = float(np.cbrt(vol_per_atom * n))
    while True:
        cell32 = _draw_cell(rng, max(3.0, 0.8 * side), max(3.6, 1.5 * side), 60.0, 120.0)
        x = _place_atoms(rng, n, cell32, dmin)
        if x is not None:
            return cell32, x


def _assemble(items) -> Batch:
    cells = np.stack([c for c, _ in items]).astype(np.float32)
    counts = np.array([x.shape[0] for _, x in items], dtype=np.int64)
    ptr = np.zeros(len(items) + 1, dtype=np.int32)
    ptr[1:] = np.cumsum(counts)
    pos = np.concatenate([x for _, x in items], axis=0).astype(np.float32) if len(items) else \
        np.zeros((0, 3), np.float32)
    return Batch(pos=np.ascontiguousarray(pos), lattice=np.ascontiguousarray(cells), struct_ptr=ptr)


def small_batch(n_struct: int, seed: int = 0) -> Batch:
    return _assemble([small_crystal(seed, s) for s in range(n_struct)])


def paper_scale_batch(n_struct: int, seed: int = 0) -> Batch:
    """batches of up to 64-atom cells for k = 16 / 32 / 64 and cutoffs 3 / 5 / 8 A
    (the columns of the paper's Tables 1-2)."""
    return _assemble([paper_scale_crystal(seed, s) for s in range(n_struct)])


def supercell_batch(n_struct: int, seed: int = 0) -> Batch:
    return _assemble([supercell(seed, s) for s in range(n_struct)])


def skewed_batch(n_struct: int, seed: int = 0) -> Batch:
    return _assemble([small_crystal(seed, s, family=FAMILY_SKEWED, n_lo=2, n_hi=20, len_lo=3.0,
                                    len_hi=12.0, ang_lo=35.0, ang_hi=145.0, dmin=1.0)
                      for s in range(n_struct)])


def walk(batch: Batch, n_steps: int, seed: int = 0, sigma=0.02, strain=0.02, h_floor=0.5
         ) -> Iterator[Batch]:
    """configs[4] trajectory (R20): cumulative random walk, FP64 state, each step cast to FP32.
    Yields n_steps batches (the initial state is NOT yielded)."""
    x = batch.pos.astype(np.float64)
    cell = batch.lattice.astype(np.float64)
    ptr = batch.struct_ptr
    s_count = cell.shape[0]
    eye = np.eye(3)[None]
    for step in range(n_steps):
        rng = _rng(seed, FAMILY_WALK, step)
        x = x + rng.normal(0.0, sigma, size=x.shape)
        x -= np.floor(x)
        eps = rng.uniform(-strain, strain, size=(s_count, 3, 3))
        new = cell @ (eye + eps)
        bad = _spacings(new.astype(np.float32).astype(np.float64)).min(axis=-1) < h_floor
        while np.any(bad):
            idx = np.nonzero(bad)[0]
            eps_r = rng.uniform(-strain, strain, size=(idx.size, 3, 3))
            new[idx] = cell[idx] @ (eye + eps_r)
            bad = _spacings(new.astype(np.float32).astype(np.float64)).min(axis=-1) < h_floor
        cell = new
        x32 = x.astype(np.float32)
        x32[x32 >= 1.0] = 0.0
        yield Batch(pos=x32, lattice=cell.astype(np.float32), struct_ptr=ptr)


# ----------------------------------------------------------------------------- the five configs
CONFIGS = {
    0: dict(kind="cutoff", r_c=5.0, n_struct=8, family="small"),
    1: dict(kind="knn", k=12, n_struct=256, family="small"),
    2: dict(kind="cutoff+knn", r_c=6.0, k=12, n_struct=4096, family="small"),
    3: dict(kind="cutoff", r_c=8.0, n_struct=16, family="supercell"),
    4: dict(kind="knn-update", k=24, n_struct=1024, n_steps=100, family="skewed"),
}


def config_batch(cfg: int, n_struct: int | None = None, seed: int = 0) -> Batch:
    """Initial batch of BASELINE.json configs[cfg]; n_struct overrides the batch size (prefix)."""
    c = CONFIGS[cfg]
    n = c["n_struct"] if n_struct is None else n_struct
    return {"small": small_batch, "supercell": supercell_batch, "skewed": skewed_batch}[c["family"]](n, seed)


# ----------------------------------------------------------------------------- textbook cells (tests)
def textbook(name: str, a: float = 1.0) -> Batch:
    """Exactly-known crystals for the closed-form pins; one structure each."""
    s3 = np.sqrt(3.0)
    table = {
        "sc": (np.eye(3), [[0, 0, 0]]),
        "fcc_conv": (np.eye(3), [[0, 0, 0], [0, .5, .5], [.5, 0, .5], [.5, .5, 0]]),
        "fcc_prim": (0.5 * np.array([[0, 1, 1], [1, 0, 1], [1, 1, 0]], float), [[0, 0, 0]]),
        "bcc_conv": (np.eye(3), [[0, 0, 0], [.5, .5, .5]]),
        "bcc_prim": (0.5 * np.array([[-1, 1, 1], [1, -1, 1], [1, 1, -1]], float), [[0, 0, 0]]),
        "diamond": (np.eye(3), [[0, 0, 0], [0, .5, .5], [.5, 0, .5], [.5, .5, 0],
                                [.25, .25, .25], [.25, .75, .75], [.75, .25, .75], [.75, .75, .25]]),
        "hcp": (np.array([[1, 0, 0], [-0.5, s3 / 2, 0], [0, 0, np.sqrt(8.0 / 3.0)]]),
                [[1 / 3, 2 / 3, 0.25], [2 / 3, 1 / 3, 0.75]]),
        "rocksalt": (np.eye(3), [[0, 0, 0], [0, .5, .5], [.5, 0, .5], [.5, .5, 0],
                                 [.5, .5, .5], [.5, 0, 0], [0, .5, 0], [0, 0, .5]]),
    }
    cell, frac = table[name]
    return Batch(pos=np.asarray(frac, dtype=np.float32).reshape(-1, 3),
                 lattice=(a * cell).astype(np.float32)[None],
                 struct_ptr=np.array([0, len(frac)], dtype=np.int32))


def concat(batches) -> Batch:
    pos = np.concatenate([b.pos for b in batches], axis=0)
    lat = np.concatenate([b.lattice for b in batches], axis=0)
    counts = np.concatenate([np.diff(b.struct_ptr) for b in batches])
    ptr = np.zeros(counts.size + 1, np.int32)
    ptr[1:] = np.cumsum(counts)
    return Batch(pos=np.ascontiguousarray(pos, np.float32), lattice=np.ascontiguousarray(lat, np.float32),
                 struct_ptr=ptr)
