"""Seeded synthetic "water-like" block-sparse Hamiltonians (inputs only).

This module serves BOTH the CUDA path and the CPU oracle and therefore holds
none of the submatrix method's arithmetic: it only draws random numbers and
lays them out as a block-CSR matrix.  Neither `oracle/` nor the CUDA package
is imported here.

The paper's workload is bulk liquid water run through CP2K (PAPER.md:77
Fig. 1, :94 "double-zeta valence polarization basis", :112); those geometries
and Hamiltonians are not available, so this generator stands in for them with
the recipe BASELINE.json `configs` states (readings G1-G8):

  G1  cubic periodic box, L = (N / rho)^(1/3), rho = 0.0334 molecules/A^3
      (33.4 nm^-3); positions i.i.d. uniform in [0, L)^3.
  G2  block (i, j) is stored iff the minimum-image distance r_ij < cutoff
      (strict); the diagonal block is always stored.
  G3  diagonal block: diag(onsite) + G, onsite = -1 for the first n_occ
      orbitals and +1 for the rest; G symmetric, independent entries of the
      upper triangle (incl. diagonal) ~ N(0, 0.05), mirrored.
  G4  off-diagonal block, i < j: 0.3 * exp(-r_ij / 2 A) * N(0,1)^{b_i x b_j};
      H_ji := H_ij^T ("symmetrised").
  G5  block-CSR, row-major blocks, fp64 master values.
  G6  numpy Generator(PCG64(seed)); draw order: positions (N x 3), diagonal
      upper triangles for i = 0..N-1, off-diagonal blocks over pairs sorted
      lexicographically (i < j).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

RHO = 0.0334  # molecules per cubic Angstrom (liquid water, 33.4 nm^-3)

# BASELINE.json `configs`, in order.  `x_dtypes` are the working precisions the
# config names; `max_iter`/`tol` the stopping rule (tol <= 0: fixed count).
CONFIGS = [
    dict(name="cfg0", n_mol=32, b=6, n_occ=3, cutoff=4.0, seed=1000,
         runs=[dict(x_dtype="f64", max_iter=100, tol=1e-8)]),
    dict(name="cfg1", n_mol=1000, b=6, n_occ=3, cutoff=6.0, seed=1001,
         runs=[dict(x_dtype="f64", max_iter=100, tol=1e-8),
               dict(x_dtype="f32", max_iter=100, tol=1e-5)]),
    dict(name="cfg2", n_mol=3000, b=23, n_occ=4, cutoff=5.0, seed=1002,
         runs=[dict(x_dtype="bf16", max_iter=20, tol=0.0)]),
    dict(name="cfg3", n_mol=10000, b=6, n_occ=3, cutoff=6.0, seed=1003,
         runs=[dict(x_dtype="f16", max_iter=20, tol=0.0)]),
    dict(name="cfg4", n_mol=2000, b=23, n_occ=4, cutoff=8.0, seed=1004,
         runs=[dict(x_dtype="bf16", max_iter=25, tol=0.0),
               dict(x_dtype="f16", max_iter=25, tol=0.0),
               dict(x_dtype="f64", max_iter=25, tol=0.0)]),
]


@dataclass
class Workload:
    """Block-CSR symmetric matrix H plus the geometry it came from."""
    n_blk: int
    blk_size: np.ndarray      # int32 [N]
    row_ptr: np.ndarray       # int32 [N+1]
    col_idx: np.ndarray       # int32 [nnzb], strictly ascending per row
    val_ptr: np.ndarray       # int64 [nnzb+1], element offset of each block
    vals: np.ndarray          # float64 [val_ptr[-1]], row-major b_i x b_j blocks
    box: float
    positions: np.ndarray     # float64 [N,3]
    meta: dict = field(default_factory=dict)

    @property
    def nnzb(self) -> int:
        return int(self.col_idx.shape[0])

    @property
    def n(self) -> int:
        return int(self.blk_size.sum())

    def dense(self) -> np.ndarray:
        """Dense n x n copy (tests on small inputs only)."""
        off = np.concatenate([[0], np.cumsum(self.blk_size)]).astype(np.int64)
        out = np.zeros((self.n, self.n))
        for i in range(self.n_blk):
            for p in range(self.row_ptr[i], self.row_ptr[i + 1]):
                j = int(self.col_idx[p])
                bi, bj = int(self.blk_size[i]), int(self.blk_size[j])
                out[off[i]:off[i] + bi, off[j]:off[j] + bj] = \
                    self.vals[self.val_ptr[p]:self.val_ptr[p + 1]].reshape(bi, bj)
        return out


def _min_image_pairs(pos: np.ndarray, box: float, cutoff: float):
    """All pairs i<j with minimum-image distance r < cutoff, lexicographic order."""
    n = pos.shape[0]
    if not np.isfinite(cutoff):
        ii, jj = np.triu_indices(n, k=1)
    elif n <= 4096 or cutoff >= 0.5 * box:
        ii, jj = np.triu_indices(n, k=1)
    else:
        from scipy.spatial import cKDTree
        tree = cKDTree(pos, boxsize=box)
        pr = tree.query_pairs(cutoff * (1.0 + 1e-9), output_type="ndarray")
        ii, jj = pr[:, 0].astype(np.int64), pr[:, 1].astype(np.int64)
        sw = ii > jj
        ii, jj = np.where(sw, jj, ii), np.where(sw, ii, jj)
    d = pos[ii] - pos[jj]
    d -= box * np.round(d / box)
    r = np.sqrt((d * d).sum(axis=1))
    keep = r < cutoff
    ii, jj, r = ii[keep], jj[keep], r[keep]
    o = np.lexsort((jj, ii))
    return ii[o].astype(np.int64), jj[o].astype(np.int64), r[o]


def make_workload(n_mol: int, b, n_occ, cutoff: float, seed: int,
                  name: str = "custom", pos=None, coupling: float = 0.3) -> Workload:
    """Build one seeded workload.  `b`/`n_occ` may be ints or per-molecule arrays.  `pos` (N x 3, inside the box) and
    `coupling` (amplitude of the off-diagonal blocks, BASELINE: 0.3) are overridden only by make_workload_gapped."""
    rng = np.random.Generator(np.random.PCG64(seed))
    box = (n_mol / RHO) ** (1.0 / 3.0)
    if pos is None:
        pos = rng.random((n_mol, 3)) * box

    blk = np.broadcast_to(np.asarray(b, dtype=np.int32), (n_mol,)).copy()
    occ = np.broadcast_to(np.asarray(n_occ, dtype=np.int32), (n_mol,)).copy()
    uniform = bool((blk == blk[0]).all())

    ii, jj, r = _min_image_pairs(pos, box, cutoff)
    npairs = ii.shape[0]

    # ---- block-CSR structure: (i,i), (i,j), (j,i) sorted by (row, col)
    rows = np.concatenate([np.arange(n_mol, dtype=np.int64), ii, jj])
    cols = np.concatenate([np.arange(n_mol, dtype=np.int64), jj, ii])
    # source: kind 0 = diagonal i, 1 = pair p as stored, 2 = pair p transposed
    kind = np.concatenate([np.zeros(n_mol, np.int8), np.ones(npairs, np.int8),
                           np.full(npairs, 2, np.int8)])
    src = np.concatenate([np.arange(n_mol), np.arange(npairs), np.arange(npairs)])
    o = np.lexsort((cols, rows))
    rows, cols, kind, src = rows[o], cols[o], kind[o], src[o]
    nnzb = rows.shape[0]
    row_ptr = np.zeros(n_mol + 1, dtype=np.int64)
    np.add.at(row_ptr, rows + 1, 1)
    row_ptr = np.cumsum(row_ptr)
    sizes = blk[rows].astype(np.int64) * blk[cols].astype(np.int64)
    val_ptr = np.concatenate([[0], np.cumsum(sizes)]).astype(np.int64)
    vals = np.empty(int(val_ptr[-1]), dtype=np.float64)

    if uniform:
        bb = int(blk[0])
        iu = np.triu_indices(bb)
        g = rng.standard_normal((n_mol, iu[0].shape[0])) * 0.05
        diag = np.zeros((n_mol, bb, bb))
        diag[:, iu[0], iu[1]] = g
        diag[:, iu[1], iu[0]] = g
        onsite = np.where(np.arange(bb)[None, :] < occ[:, None], -1.0, 1.0)
        diag[:, np.arange(bb), np.arange(bb)] += onsite
        offd = rng.standard_normal((npairs, bb, bb))
        offd *= (coupling * np.exp(-r / 2.0))[:, None, None]
        v3 = vals.reshape(nnzb, bb, bb)
        k0, k1, k2 = kind == 0, kind == 1, kind == 2
        v3[k0] = diag[src[k0]]
        v3[k1] = offd[src[k1]]
        v3[k2] = offd[src[k2]].transpose(0, 2, 1)
    else:
        diag_blocks = []
        for i in range(n_mol):
            bb = int(blk[i])
            iu = np.triu_indices(bb)
            g = rng.standard_normal(iu[0].shape[0]) * 0.05
            d = np.zeros((bb, bb))
            d[iu] = g
            d[(iu[1], iu[0])] = g
            d[np.arange(bb), np.arange(bb)] += np.where(np.arange(bb) < occ[i], -1.0, 1.0)
            diag_blocks.append(d)
        off_blocks = []
        for p in range(npairs):
            bi, bj = int(blk[ii[p]]), int(blk[jj[p]])
            off_blocks.append(rng.standard_normal((bi, bj)) * (coupling * np.exp(-r[p] / 2.0)))
        for q in range(nnzb):
            s = int(src[q])
            if kind[q] == 0:
                blkv = diag_blocks[s]
            elif kind[q] == 1:
                blkv = off_blocks[s]
            else:
                blkv = off_blocks[s].T
            vals[val_ptr[q]:val_ptr[q + 1]] = np.ascontiguousarray(blkv).ravel()

    return Workload(
        n_blk=n_mol, blk_size=blk.astype(np.int32), row_ptr=row_ptr.astype(np.int32),
        col_idx=cols.astype(np.int32), val_ptr=val_ptr, vals=vals, box=box,
        positions=pos,
        meta=dict(name=name, n_mol=n_mol, cutoff=cutoff, seed=seed, n_pairs=int(npairs)))


def make_config(index: int, **overrides) -> Workload:
    """Workload of BASELINE.json configs[index] (overrides: n_mol, cutoff, seed, ...)."""
    c = dict(CONFIGS[index])
    c.update(overrides)
    return make_workload(c["n_mol"], c["b"], c["n_occ"], c["cutoff"], c["seed"], name=c["name"])


def sample_columns(wl: Workload, count: int, seed: int) -> np.ndarray:
    """Seeded, sorted subset of block-column ids (oracle subsets on the large configs)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    count = min(count, wl.n_blk)
    return np.sort(rng.choice(wl.n_blk, size=count, replace=False)).astype(np.int32)


def make_overlap(wl: Workload, seed: int = None, amp: float = 0.05, noise: float = 0.02) -> Workload:
    """Seeded overlap matrix S with H's block pattern, for the non-orthogonal rows of SURVEY.md 8(f) f2 (PAPER.md:83-91,
    Eq. 12-14): diagonal blocks I + symmetric N(0, noise) noise, off-diagonal blocks amp * exp(-r / 2 A) * N(0, 1) for the
    same molecule pairs as H, S_ji = S_ij^T.  The amplitudes keep S symmetric positive definite (spectrum ~ 1 +- 0.4 on
    the BASELINE geometries; the oracle asserts it).  Own RNG stream: seed + 500000 of the workload's seed."""
    seed = int(wl.meta.get("seed", 0)) + 500000 if seed is None else seed
    rng = np.random.Generator(np.random.PCG64(seed))
    blk = np.asarray(wl.blk_size)
    vp = np.asarray(wl.val_ptr, dtype=np.int64)
    vals = np.zeros(int(vp[-1]))
    box = wl.box
    pos = wl.positions
    for i in range(wl.n_blk):
        bi = int(blk[i])
        for p in range(int(wl.row_ptr[i]), int(wl.row_ptr[i + 1])):
            j = int(wl.col_idx[p])
            if j < i:
                continue
            bj = int(blk[j])
            if j == i:
                g = rng.standard_normal((bi, bi)) * noise
                b_ = np.eye(bi) + 0.5 * (g + g.T)
                vals[vp[p]:vp[p + 1]] = b_.ravel()
            else:
                d = pos[i] - pos[j]
                d -= box * np.round(d / box)
                r = float(np.sqrt((d * d).sum()))
                b_ = rng.standard_normal((bi, bj)) * (amp * np.exp(-r / 2.0))
                vals[vp[p]:vp[p + 1]] = b_.ravel()
                row = wl.col_idx[wl.row_ptr[j]:wl.row_ptr[j + 1]]
                q = int(wl.row_ptr[j]) + int(np.searchsorted(row, i))
                vals[vp[q]:vp[q + 1]] = b_.T.ravel()
    return Workload(n_blk=wl.n_blk, blk_size=wl.blk_size, row_ptr=wl.row_ptr, col_idx=wl.col_idx, val_ptr=wl.val_ptr,
                    vals=vals, box=wl.box, positions=wl.positions, meta=dict(wl.meta, overlap_seed=seed))


def make_workload_gapped(n_mol: int, b, n_occ, cutoff: float, seed: int, coupling: float = 0.04, jitter: float = 0.15,
                         name: str = "gapped") -> Workload:
    """Second workload of SURVEY.md 8(f) f4: the same block structure and value recipe as make_workload, but with
    NON-OVERLAPPING molecules (a jittered simple-cubic lattice at the same number density: nearest distances ~ 2.2-3.9 A
    instead of down to 0.06 A) and weaker couplings, so that the spectrum of H keeps the gap between the onsite levels
    -1 and +1 around mu = 0 and a fixed Newton-Schulz count converges (reading A13: the BASELINE generator is gapless).
    Seeded: lattice sites drawn without replacement, then the jitter, then the blocks as in make_workload."""
    rng = np.random.Generator(np.random.PCG64(seed + 700000))
    box = (n_mol / RHO) ** (1.0 / 3.0)
    side = int(np.ceil(n_mol ** (1.0 / 3.0) - 1e-9))
    a = box / side
    sites = rng.choice(side ** 3, size=n_mol, replace=False)
    ijk = np.stack([sites // (side * side), (sites // side) % side, sites % side], axis=1).astype(np.float64)
    pos = (ijk + 0.5 + (rng.random((n_mol, 3)) - 0.5) * 2.0 * jitter) * a
    return make_workload(n_mol, b, n_occ, cutoff, seed, name=name, pos=pos, coupling=coupling)
