"""ctypes front end of the CPU fp64 oracle (submatrix_oracle.c).

TEST INFRASTRUCTURE ONLY: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this.  It imports nothing from
the CUDA package; inputs come from workloads/generator.py.

Every function takes the block-CSR arrays of a `Workload`-like object (fields
n_blk, blk_size, row_ptr, col_idx, val_ptr, vals) and follows PAPER.md:110
(Fig. 2, the three steps), :87 (Eq. 13) and :91 (Eq. 14 with S = I); see the
header of submatrix_oracle.c for the passage behind each C function.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from types import SimpleNamespace

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liborc.so")
_SRC = os.path.join(_HERE, "submatrix_oracle.c")


def build(force: bool = False) -> str:
    """Compile submatrix_oracle.c with gcc (building the checker is not using it)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fPIC", "-shared", "-pthread", "-o", _SO, _SRC, "-lm"])
    return _SO


_lib = None


def lib():
    global _lib
    if _lib is None:
        # ORC_SO: an alternative build of the same source (the address/UB-sanitizer build of tests/test_oracle_pins.py)
        _lib = C.CDLL(os.environ.get("ORC_SO") or build())
        _lib.orc_gershgorin.restype = C.c_double
        _lib.orc_trace.restype = C.c_double
    return _lib


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t)) if a is not None else None


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _csr(w):
    return (C.c_int32(w.n_blk), _p(_i32(w.blk_size), C.c_int32), _p(_i32(w.row_ptr), C.c_int32),
            _p(_i32(w.col_idx), C.c_int32))


def check_pattern(w) -> int:
    return lib().orc_check_pattern(C.c_int32(w.n_blk), _p(_i32(w.row_ptr), C.c_int32),
                                   _p(_i32(w.col_idx), C.c_int32))


def pattern_sizes(w, pad_to: int):
    out = np.zeros(5, dtype=np.int64)
    rc = lib().orc_pattern_sizes(*_csr(w), C.c_int32(pad_to), _p(out, C.c_int64))
    if rc:
        raise ValueError(f"orc_pattern_sizes: {rc}")
    return SimpleNamespace(nbr_len=int(out[0]), gmap_len=int(out[1]), packed_elems=int(out[2]),
                           max_dim=int(out[3]), max_dim_pad=int(out[4]))


def build_pattern(w, pad_to: int):
    """Integer pattern arrays of PAPER.md:110 step 1 (see include/submatrix.h for names)."""
    sz = pattern_sizes(w, pad_to)
    n = w.n_blk
    P = SimpleNamespace(
        nbr_ptr=np.zeros(n + 1, np.int32), nbr_idx=np.zeros(sz.nbr_len, np.int32),
        own_pos=np.zeros(n, np.int32), dim=np.zeros(n, np.int32), dim_pad=np.zeros(n, np.int32),
        row_off=np.zeros(sz.nbr_len, np.int32), sub_off=np.zeros(n + 1, np.int64),
        gmap_ptr=np.zeros(n + 1, np.int64), gmap=np.zeros(sz.gmap_len, np.int32),
        tmap=np.zeros(w.nnzb, np.int32), order=np.zeros(n, np.int32), sizes=sz)
    rc = lib().orc_build_pattern(
        *_csr(w), C.c_int32(pad_to), _p(P.nbr_ptr, C.c_int32), _p(P.nbr_idx, C.c_int32),
        _p(P.own_pos, C.c_int32), _p(P.dim, C.c_int32), _p(P.dim_pad, C.c_int32),
        _p(P.row_off, C.c_int32), _p(P.sub_off, C.c_int64), _p(P.gmap_ptr, C.c_int64),
        _p(P.gmap, C.c_int32), _p(P.tmap, C.c_int32), _p(P.order, C.c_int32))
    if rc:
        raise ValueError(f"orc_build_pattern: status {rc}")
    return P


def gather(w, i: int, mu: float = 0.0) -> np.ndarray:
    """T_i(H) - mu*I as a dense m x m fp64 array."""
    nb = w.col_idx[w.row_ptr[i]:w.row_ptr[i + 1]]
    m = int(np.asarray(w.blk_size)[nb].sum())
    T = np.zeros((m, m))
    vp = np.ascontiguousarray(w.val_ptr, dtype=np.int64)
    vals = np.ascontiguousarray(w.vals, dtype=np.float64)
    lib().orc_gather(*_csr(w), _p(vp, C.c_int64), _p(vals, C.c_double), C.c_int32(i),
                     C.c_double(mu), _p(T, C.c_double))
    return T


def gershgorin(T: np.ndarray) -> float:
    T = np.ascontiguousarray(T, dtype=np.float64)
    return float(lib().orc_gershgorin(C.c_int32(T.shape[0]), _p(T, C.c_double)))


def jacobi_eigh(T: np.ndarray, max_sweeps: int = 30, rel_tol: float = 1e-15):
    """(w, V, sweeps): T = V diag(w) V^T, columns of V are eigenvectors (own cyclic Jacobi)."""
    A = np.array(T, dtype=np.float64, order="C", copy=True)
    m = A.shape[0]
    Vt = np.zeros((m, m))
    w = np.zeros(m)
    sw = lib().orc_jacobi(C.c_int32(m), _p(A, C.c_double), _p(Vt, C.c_double), _p(w, C.c_double),
                          C.c_int32(max_sweeps), C.c_double(rel_tol))
    return w, Vt.T.copy(), int(sw)


def sign(T: np.ndarray) -> np.ndarray:
    """sign(T) for symmetric T by Eq. 13's definition on the spectrum."""
    w, V, _ = jacobi_eigh(T)
    m = T.shape[0]
    S = np.zeros((m, m))
    Vt = np.ascontiguousarray(V.T)
    lib().orc_sign_from_eig(C.c_int32(m), _p(Vt, C.c_double), _p(w, C.c_double), _p(S, C.c_double))
    return S


def ns_polynomial(T: np.ndarray, scale: float, k: int, order: int = 2) -> np.ndarray:
    """Exact-arithmetic result of k Newton-Schulz steps from T/scale (reading A13).  order 3 (f3, reading A22):
    k steps of x <- x (15 - 10 x^2 + 3 x^4) / 8 instead of x <- x (3 - x^2) / 2."""
    w, V, _ = jacobi_eigh(T)
    m = T.shape[0]
    S = np.zeros((m, m))
    Vt = np.ascontiguousarray(V.T)
    fn = {2: lib().orc_nsk_from_eig, 3: lib().orc_ns3k_from_eig}[order]
    fn(C.c_int32(m), _p(Vt, C.c_double), _p(w, C.c_double), C.c_double(scale), C.c_int32(k), _p(S, C.c_double))
    return S


def density_columns(w, mu: float = 0.0, cols=None, mode: str = "exact", k_fixed: int = 0,
                    scale=None, n_threads: int = 1):
    """Raw D = 1/2 (I - sign(T_i - mu I)) blocks of the listed block columns (all if None).

    Returns (d_vals in H's block-CSR layout with only the listed columns' blocks
    written, stats).  mode "nsk": the NS-k polynomial at scale (Gershgorin if None); "ns3k": k_fixed steps of the
    third-order iteration (f3, reading A22).
    """
    vp = np.ascontiguousarray(w.val_ptr, dtype=np.int64)
    vals = np.ascontiguousarray(w.vals, dtype=np.float64)
    d = np.zeros_like(vals)
    cols_a = None if cols is None else _i32(cols)
    nc = w.n_blk if cols is None else int(cols_a.shape[0])
    st = SimpleNamespace(min_abs_eig=np.zeros(nc), scale=np.zeros(nc), sweeps=np.zeros(nc, np.int32),
                         n_neg=np.zeros(nc, np.int32))
    sc = None if scale is None else np.ascontiguousarray(scale, dtype=np.float64)
    rc = lib().orc_density_columns(
        *_csr(w), _p(vp, C.c_int64), _p(vals, C.c_double), C.c_double(mu), C.c_int32(nc),
        _p(cols_a, C.c_int32), C.c_int32({"exact": 0, "nsk": 1, "ns3k": 2}[mode]), C.c_int32(k_fixed),
        _p(sc, C.c_double), _p(d, C.c_double), _p(st.min_abs_eig, C.c_double),
        _p(st.scale, C.c_double), _p(st.sweeps, C.c_int32), _p(st.n_neg, C.c_int32),
        C.c_int32(n_threads))
    if rc:
        raise ValueError(f"orc_density_columns: status {rc}")
    return d, st


def mu_search(w, n_target: float, mu_lo: float, mu_hi: float, tol_n: float = 1e-6, mu_tol: float = 1e-12,
              max_trials: int = 60, n_threads: int = 1):
    """Chemical potential for a fixed electron count: Eq. 14 carries mu,
    PAPER.md:89-92 relate D to the occupied states; with S = I, Tr D(mu) counts the eigenvalues below mu and is
    non-decreasing, so mu solves Tr D(mu) = n_target by bisection.  Step by step: the two ends of the bracket
    (upper first), then midpoints until |Tr D - n_target| <= tol_n, the bracket is narrower than mu_tol, or
    max_trials evaluations.  Each evaluation is the whole submatrix method with the exact sign (density_columns).
    Returns (mu, Tr D(mu), trials, d_vals of the last trial)."""
    def count(mu):
        d, _ = density_columns(w, mu=mu, n_threads=n_threads)
        return trace(w, d), d
    trials = 0
    n_hi, d = count(mu_hi); trials += 1
    if n_hi < n_target - tol_n:
        raise ValueError("bracket: Tr D(mu_hi) < n_target")
    n_lo, d = count(mu_lo); trials += 1
    if n_lo > n_target + tol_n:
        raise ValueError("bracket: Tr D(mu_lo) > n_target")
    if abs(n_lo - n_target) <= tol_n:
        return mu_lo, n_lo, trials, d
    lo, hi, mu, n_mid = mu_lo, mu_hi, mu_lo, n_lo
    while trials < max_trials:
        mu = 0.5 * (lo + hi)
        n_mid, d = count(mu); trials += 1
        if abs(n_mid - n_target) <= tol_n:
            break
        if n_mid < n_target:
            lo = mu
        else:
            hi = mu
        if hi - lo <= mu_tol:
            break
    return mu, n_mid, trials, d


def symmetrise(w, d_raw: np.ndarray) -> np.ndarray:
    vp = np.ascontiguousarray(w.val_ptr, dtype=np.int64)
    d_raw = np.ascontiguousarray(d_raw, dtype=np.float64)
    out = np.zeros_like(d_raw)
    rc = lib().orc_symmetrise(*_csr(w), _p(vp, C.c_int64), _p(d_raw, C.c_double), _p(out, C.c_double))
    if rc:
        raise ValueError(f"orc_symmetrise: status {rc}")
    return out


def trace(w, d_vals: np.ndarray) -> float:
    vp = np.ascontiguousarray(w.val_ptr, dtype=np.int64)
    d_vals = np.ascontiguousarray(d_vals, dtype=np.float64)
    return float(lib().orc_trace(*_csr(w), _p(vp, C.c_int64), _p(d_vals, C.c_double)))


def column_mask(w, cols) -> np.ndarray:
    """Boolean mask over d_vals elements that belong to blocks in the listed block columns."""
    sel = np.zeros(w.n_blk, dtype=bool)
    sel[np.asarray(cols)] = True
    blk_sel = sel[np.asarray(w.col_idx)]
    sizes = np.diff(np.asarray(w.val_ptr))
    return np.repeat(blk_sel, sizes)


def density_columns_lapack(w, mu: float = 0.0, cols=None, mode: str = "exact", k_fixed: int = 0, scale=None):
    """Same result as density_columns, with LAPACK's symmetric eigensolver (numpy.linalg.eigh, a
    library primitive used as one step) in place of the Jacobi sweeps.  For the large submatrices
    of configs[4] (m ~ 1650), where cyclic Jacobi needs ~10 min per submatrix.  Pinned to the Jacobi
    path in tests/test_oracle_pins.py.  Steps: PAPER.md:110 (gather, f, insert columns), Eq. 13 on
    the spectrum, Eq. 14 with S = I."""
    blk = np.asarray(w.blk_size)
    vp = np.asarray(w.val_ptr, dtype=np.int64)
    d = np.zeros(int(vp[-1]))
    col_list = list(range(w.n_blk)) if cols is None else [int(c) for c in cols]
    st = SimpleNamespace(min_abs_eig=np.zeros(len(col_list)), scale=np.zeros(len(col_list)),
                         n_neg=np.zeros(len(col_list), np.int32))
    for ci, i in enumerate(col_list):
        T = gather(w, i, mu)
        m = T.shape[0]
        gs = float(np.abs(T).sum(axis=1).max())
        lam, V = np.linalg.eigh(T)
        if mode == "exact":
            f = np.sign(lam)
        else:
            x = lam / (gs if scale is None else float(scale[ci]))
            for _ in range(k_fixed):
                x = x * (15.0 - 10.0 * x * x + 3.0 * x ** 4) / 8.0 if mode == "ns3k" else 0.5 * x * (3.0 - x * x)
            f = x
        S = (V * f) @ V.T
        nb = np.asarray(w.col_idx[w.row_ptr[i]:w.row_ptr[i + 1]])
        offs = np.concatenate([[0], np.cumsum(blk[nb])])
        own = int(np.where(nb == i)[0][0])
        bi = int(blk[i])
        for a, j in enumerate(nb):
            row = w.col_idx[w.row_ptr[j]:w.row_ptr[j + 1]]
            p = int(w.row_ptr[j]) + int(np.searchsorted(row, i))
            blk_s = S[offs[a]:offs[a + 1], offs[own]:offs[own + 1]]
            ident = np.eye(bi) if a == own else 0.0
            d[vp[p]:vp[p + 1]] = (0.5 * (ident - blk_s)).ravel()
        st.min_abs_eig[ci] = np.abs(lam).min()
        st.scale[ci] = gs
        st.n_neg[ci] = int((lam < 0).sum())
    return d, st


# ---- non-orthogonal basis (PAPER.md:83 Eq. 12, :87 Eq. 13, :91 Eq. 14) --------------------
# Reading A20: Eq. 12 as printed has "sign" on both sides; the matrix [[0, A^1/2], [A^-1/2, 0]] squares to
# the identity, so it is its own sign and the printed relation is the known identity
#     sign([[0, A], [I, 0]]) = [[0, A^1/2], [A^-1/2, 0]]      (A without eigenvalues on the closed negative real axis).

def sign_block_matrix(T: np.ndarray) -> np.ndarray:
    """sign(M), M = [[0, T], [I, 0]] (2m x 2m, NOT symmetric), by Eq. 13 written out on M itself:
    sign(M) = M (M^2)^(-1/2).  M^2 = diag(T, T) is symmetric, so its inverse square root comes from the oracle's own
    Jacobi eigendecomposition: (M^2)^(-1/2) = V diag(w^-1/2) V^T.  T must be symmetric positive definite."""
    m = T.shape[0]
    M = np.zeros((2 * m, 2 * m))
    M[:m, m:] = T
    M[m:, :m] = np.eye(m)
    M2 = M @ M
    w, V, _ = jacobi_eigh(0.5 * (M2 + M2.T))
    if w.min() <= 0.0:
        raise ValueError("sign_block_matrix: T is not positive definite")
    return M @ ((V / np.sqrt(w)) @ V.T)


def inv_sqrt_blocks(T: np.ndarray):
    """(T^-1/2, T^1/2) = the lower-left and upper-right blocks of sign([[0, T], [I, 0]]) (Eq. 12), computed from the
    Jacobi eigendecomposition of T itself (the same function of the same matrix as sign_block_matrix at an eighth of
    the cost; tests/test_oracle_pins.py pins one against the other)."""
    w, V, _ = jacobi_eigh(T)
    if w.min() <= 0.0:
        raise ValueError("inv_sqrt_blocks: T is not positive definite")
    return (V / np.sqrt(w)) @ V.T, (V * np.sqrt(w)) @ V.T


def _scatter_owned(w, i, Si, out):
    """Insert the owned block column of the dense m x m result Si of column i into block-CSR values (PAPER.md:110 step 3)."""
    blk = np.asarray(w.blk_size)
    vp = np.asarray(w.val_ptr, dtype=np.int64)
    nb = np.asarray(w.col_idx[w.row_ptr[i]:w.row_ptr[i + 1]])
    offs = np.concatenate([[0], np.cumsum(blk[nb])])
    own = int(np.where(nb == i)[0][0])
    for a, j in enumerate(nb):
        row = w.col_idx[w.row_ptr[j]:w.row_ptr[j + 1]]
        p = int(w.row_ptr[j]) + int(np.searchsorted(row, i))
        out[vp[p]:vp[p + 1]] = Si[offs[a]:offs[a + 1], offs[own]:offs[own + 1]].ravel()


def inv_sqrt_columns(wS, cols=None, literal: bool = False):
    """Submatrix method with f = the blocks of Eq. 12: for every listed block column i gather T_i(S),
    evaluate sign([[0, T_i], [I, 0]]), and insert the owned columns of its lower-left block (T_i^-1/2) and of its
    upper-right block (T_i^1/2) into two block-sparse results with S's pattern.  Returns (z_vals ~ S^-1/2,
    y_vals ~ S^1/2, min eigenvalue of T_i per column).  literal=True evaluates Eq. 13 on the 2m x 2m matrix itself."""
    vp = np.asarray(wS.val_ptr, dtype=np.int64)
    z = np.zeros(int(vp[-1])); y = np.zeros(int(vp[-1]))
    col_list = list(range(wS.n_blk)) if cols is None else [int(c) for c in cols]
    lam_min = np.zeros(len(col_list))
    for ci, i in enumerate(col_list):
        T = gather(wS, i, 0.0)
        m = T.shape[0]
        if literal:
            Sg = sign_block_matrix(T)
            Zi, Yi = Sg[m:, :m], Sg[:m, m:]
        else:
            Zi, Yi = inv_sqrt_blocks(T)
        lam_min[ci] = np.linalg.eigvalsh(T).min()
        _scatter_owned(wS, i, Zi, z)
        _scatter_owned(wS, i, Yi, y)
    return z, y, lam_min


def density_nonorth_columns(wH, wS, mu: float = 0.0, cols=None):
    """Eq. 14, P = 1/2 (I - sign(S^-1 H - mu I)) S^-1, by the submatrix method on the pair (H, S) (same
    block pattern): for every listed block column i, with T_H = T_i(H), T_S = T_i(S) gathered on the same index set,
        Z = T_S^-1/2 (Eq. 12),  S^-1 = Z Z,  A = S^-1 T_H - mu I  (not symmetric),
        sign(A) = Z sign(Z T_H Z - mu I) Z^-1   (A = Z (Z T_H Z - mu I) Z^-1 is similar to a symmetric matrix, whose
                                                 sign is Eq. 13 on the spectrum, own Jacobi),
        P_i = 1/2 (I - sign(A)) S^-1,
    and the owned columns of P_i are inserted.  tests/test_oracle_pins.py pins sign(A) against Eq. 13 written out with
    scipy.linalg.sqrtm on A itself."""
    vp = np.asarray(wH.val_ptr, dtype=np.int64)
    out = np.zeros(int(vp[-1]))
    col_list = list(range(wH.n_blk)) if cols is None else [int(c) for c in cols]
    for i in col_list:
        TH = gather(wH, i, 0.0)
        TS = gather(wS, i, 0.0)
        Z, Y = inv_sqrt_blocks(TS)
        Ht = Z @ TH @ Z
        Ht = 0.5 * (Ht + Ht.T) - mu * np.eye(Ht.shape[0])
        sgA = Z @ sign(Ht) @ Y                       # Y = T_S^1/2 = Z^-1
        Pi = 0.5 * (np.eye(TH.shape[0]) - sgA) @ (Z @ Z)
        _scatter_owned(wH, i, Pi, out)
    return out
