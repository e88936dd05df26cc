"""Pins of the CPU oracle against what the paper and the mathematics fix.

PAPER.md prints no worked numerical example for this path, so the pins are closed
forms, invariants of Eq. 13 / Eq. 14, limits in which the
submatrix method is exact, library routines (LAPACK eigh, scipy
signm, LDL^T inertia) and brute force on tiny inputs.
"""
import os

import numpy as np
import pytest
import scipy.linalg

from oracle import oracle as orc
from workloads.generator import Workload, make_config, make_workload


def _rand_sym(m, seed):
    rng = np.random.default_rng(seed)
    a = rng.standard_normal((m, m))
    return 0.5 * (a + a.T)


# ------------------------------------------------------------------ Jacobi

def test_jacobi_diagonal_is_fixed_point():
    d = np.array([3.0, -1.5, 0.25, -7.0])
    w, V, sweeps = orc.jacobi_eigh(np.diag(d))
    assert sweeps == 0
    assert np.array_equal(w, d)
    assert np.array_equal(V, np.eye(4))


def test_jacobi_tridiagonal_toeplitz_closed_form():
    # eigenvalues of tridiag(1, 0, 1) are 2 cos(k pi / (m+1)), k = 1..m
    m = 37
    T = np.diag(np.ones(m - 1), 1) + np.diag(np.ones(m - 1), -1)
    w, V, _ = orc.jacobi_eigh(T)
    expect = 2.0 * np.cos(np.arange(1, m + 1) * np.pi / (m + 1))
    assert np.allclose(np.sort(w), np.sort(expect), atol=1e-13)


@pytest.mark.parametrize("m,seed", [(1, 0), (2, 1), (17, 2), (64, 3), (131, 4)])
def test_jacobi_reconstruction_orthogonality_and_lapack(m, seed):
    T = _rand_sym(m, seed)
    w, V, _ = orc.jacobi_eigh(T)
    fro = np.linalg.norm(T)
    assert np.linalg.norm((V * w) @ V.T - T) <= 1e-13 * max(fro, 1.0)
    assert np.linalg.norm(V.T @ V - np.eye(m)) <= 1e-13 * np.sqrt(m)
    assert np.allclose(np.sort(w), np.linalg.eigvalsh(T), atol=1e-12 * max(fro, 1.0))


# -------------------------------------------------------------------- sign

def test_sign_2x2_closed_form():
    # T = [[a, b], [b, -a]]: T^2 = (a^2+b^2) I, so Eq. 13 gives sign(T) = T / sqrt(a^2+b^2)
    a, b = 0.7, -1.9
    T = np.array([[a, b], [b, -a]])
    assert np.allclose(orc.sign(T), T / np.hypot(a, b), atol=1e-15)


def test_sign_definite_matrices():
    T = _rand_sym(9, 5)
    P = T @ T + np.eye(9)
    assert np.allclose(orc.sign(P), np.eye(9), atol=1e-13)
    assert np.allclose(orc.sign(-P), -np.eye(9), atol=1e-13)


@pytest.mark.parametrize("m,seed", [(6, 10), (40, 11), (97, 12)])
def test_sign_invariants_eq13(m, seed):
    T = _rand_sym(m, seed)
    S = orc.sign(T)
    eye = np.eye(m)
    assert np.abs(S @ S - eye).max() < 1e-12            # sign^2 = A^2 (A^2)^-1 = I
    assert np.abs(S - S.T).max() < 1e-13
    assert np.abs(S @ T - T @ S).max() < 1e-12 * np.linalg.norm(T)
    # S T = (T^2)^(1/2): symmetric positive definite with eigenvalues |lambda|
    ST = S @ T
    assert np.abs(ST - ST.T).max() < 1e-12 * np.linalg.norm(T)
    assert np.allclose(np.linalg.eigvalsh(0.5 * (ST + ST.T)), np.sort(np.abs(np.linalg.eigvalsh(T))),
                       atol=1e-11)
    # Eq. 13 literally, with the inverse square root from scipy
    ref = T @ np.linalg.inv(scipy.linalg.sqrtm(T @ T).real)
    assert np.abs(S - ref).max() < 1e-9
    assert np.abs(orc.sign(3.7 * T) - S).max() < 1e-12   # sign(cT) = sign(T), c > 0
    assert np.abs(orc.sign(-T) + S).max() < 1e-12        # sign(-T) = -sign(T)
    perm = np.random.default_rng(seed).permutation(m)
    Q = eye[perm]
    assert np.abs(orc.sign(Q @ T @ Q.T) - Q @ S @ Q.T).max() < 1e-12


def test_sign_matches_scipy_signm_and_lapack():
    T = _rand_sym(30, 21)
    S = orc.sign(T)
    lam, V = np.linalg.eigh(T)
    assert np.abs(S - (V * np.sign(lam)) @ V.T).max() < 1e-12
    assert np.abs(S - scipy.linalg.signm(T)).max() < 1e-8


def test_sign_of_zero_eigenvalue_is_zero():
    # reading A14: sgn(0) := 0, the Newton-Schulz fixed point
    T = np.diag([2.0, 0.0, -3.0])
    assert np.array_equal(orc.sign(T), np.diag([1.0, 0.0, -1.0]))


# ------------------------------------------------------------ NS-k polynomial

@pytest.mark.parametrize("k", [0, 1, 5, 12])
def test_ns_polynomial_equals_matrix_iteration(k):
    # the spectral form must equal k explicit steps X <- 1/2 X (3I - X^2) in fp64
    T = _rand_sym(24, 33)
    s = orc.gershgorin(T)
    X = T / s
    eye = np.eye(24)
    for _ in range(k):
        X = 0.5 * X @ (3.0 * eye - X @ X)
    assert np.abs(orc.ns_polynomial(T, s, k) - X).max() < 1e-12


def test_ns_polynomial_scalar_recursion_and_limit():
    d = np.array([0.9, -0.4, 0.05, -1.0])
    out = orc.ns_polynomial(np.diag(d), 1.0, 3)
    x = d.copy()
    for _ in range(3):
        x = 0.5 * x * (3.0 - x * x)
    assert np.allclose(np.diag(out), x, atol=1e-15)
    T = _rand_sym(16, 34)
    assert np.abs(orc.ns_polynomial(T, orc.gershgorin(T), 60) - orc.sign(T)).max() < 1e-10

# ------------------------------------------------------------ third-order iteration (f3, reading A22)

@pytest.mark.parametrize("k", [0, 1, 4, 9])
def test_ns3_polynomial_equals_matrix_iteration(k):
    # spectral form == k explicit steps X <- X (I + W/2 + 3 W^2 / 8), W = I - X^2 (the series of (I - W)^-1/2 cut after W^2)
    T = _rand_sym(24, 35)
    s = orc.gershgorin(T)
    X = T / s
    eye = np.eye(24)
    for _ in range(k):
        W = eye - X @ X
        X = X @ (eye + 0.5 * W + 0.375 * W @ W)
    assert np.abs(orc.ns_polynomial(T, s, k, order=3) - X).max() < 1e-12


def test_ns3_scalar_map_fixed_points_order_and_basin():
    g3 = lambda x: float(orc.ns_polynomial(np.array([[x]]), 1.0, 1, order=3)[0, 0])
    # fixed points 0, +-1 and the repelling pair +-sqrt(7/3) (3 x^4 - 10 x^2 + 7 = 0)
    for x in (0.0, 1.0, -1.0, np.sqrt(7.0 / 3.0), -np.sqrt(7.0 / 3.0)):
        assert abs(g3(x) - x) < 1e-14
    # odd; g3 = x (15 - 10 x^2 + 3 x^4) / 8 at a rational point: g3(1/2) = (1/2)(15 - 5/2 + 3/16)/8 = 203/256
    assert g3(0.5) == 203.0 / 256.0 and g3(-0.5) == -203.0 / 256.0
    # cubic contact at 1: g3(1 - e) = 1 - (5/2) e^3 + O(e^4)  (first and second derivative vanish at 1, the third is 15)
    for e in (1e-2, 1e-3):
        assert abs((1.0 - g3(1.0 - e)) / e ** 3 - 2.5) < 4.0 * e
    # basin: converges to sgn(x) inside sqrt(7/3) = 1.5275, leaves it outside (order 2: sqrt(3))
    conv = lambda x, k: float(orc.ns_polynomial(np.array([[x]]), 1.0, k, order=3)[0, 0])
    assert abs(conv(1.52, 12) - 1.0) < 1e-12 and abs(conv(-1.52, 12) + 1.0) < 1e-12
    assert abs(conv(1.535, 6)) > 10.0           # escapes (overflows to inf/nan a few steps later)
    # small x grow by 15/8 per step instead of 3/2: x0 = 1e-3 is converged after 15 order-3 steps, order 2 needs ~22
    x2 = float(orc.ns_polynomial(np.array([[1e-3]]), 1.0, 15)[0, 0])
    assert abs(conv(1e-3, 1) / 1e-3 - 1.875) < 1e-5
    assert abs(conv(1e-3, 15) - 1.0) < 1e-12 and abs(x2 - 1.0) > 0.3


def test_ns3_converges_to_sign_and_density_modes_agree():
    T = _rand_sym(16, 36)
    assert np.abs(orc.ns_polynomial(T, orc.gershgorin(T), 40, order=3) - orc.sign(T)).max() < 1e-10
    w = make_workload(6, 4, 2, 7.0, seed=5)
    d_j, _ = orc.density_columns(w, mode="ns3k", k_fixed=5)
    d_l, _ = orc.density_columns_lapack(w, mode="ns3k", k_fixed=5)
    assert np.abs(d_j - d_l).max() < 1e-12
    # column 0 by hand: D blocks = owned columns of (I - p(T_0)) / 2
    T0 = orc.gather(w, 0)
    S0 = orc.ns_polynomial(T0, orc.gershgorin(T0), 5, order=3)
    nb = w.col_idx[w.row_ptr[0]:w.row_ptr[1]]
    own = int(np.where(nb == 0)[0][0])
    p = int(w.row_ptr[0]) + own
    b = int(w.blk_size[0])
    blk = d_j[w.val_ptr[p]:w.val_ptr[p + 1]].reshape(b, b)
    assert np.abs(blk - 0.5 * (np.eye(b) - S0[own * b:(own + 1) * b, own * b:(own + 1) * b])).max() < 1e-13
    d2, _ = orc.density_columns(w, mode="nsk", k_fixed=5)
    assert np.abs(d2 - d_j).max() > 1e-6          # and it is a different polynomial than order 2



def test_gershgorin_bounds_spectral_radius():
    T = _rand_sym(50, 40)
    s = orc.gershgorin(T)
    assert s == pytest.approx(np.abs(T).sum(axis=1).max(), rel=1e-15)
    assert s >= np.abs(np.linalg.eigvalsh(T)).max()


# -------------------------------------------------- submatrix method: worked example

def _sign2(t):
    lam = np.linalg.eigvalsh(t)
    if lam[0] > 0:
        return np.eye(2)
    if lam[1] < 0:
        return -np.eye(2)
    # one eigenvalue of each sign: sign(T) = (2T - tr(T) I) / (lambda_+ - lambda_-)
    gap = np.sqrt((t[0, 0] - t[1, 1]) ** 2 + 4 * t[0, 1] ** 2)
    return (2 * t - np.trace(t) * np.eye(2)) / gap


def test_submatrix_method_on_a_three_site_chain_by_hand():
    # Fig. 2 by hand: a chain 0-1-2 with scalar blocks.  Column 0 sees {0,1},
    # column 1 sees {0,1,2} (the whole matrix), column 2 sees {1,2}.
    h = np.array([[-0.8, 0.5, 0.0], [0.5, 0.3, -0.7], [0.0, -0.7, 0.9]])
    w = Workload(n_blk=3, blk_size=np.ones(3, np.int32), row_ptr=np.array([0, 2, 5, 7], np.int32),
                 col_idx=np.array([0, 1, 0, 1, 2, 1, 2], np.int32), val_ptr=np.arange(8, dtype=np.int64),
                 vals=np.array([h[0, 0], h[0, 1], h[1, 0], h[1, 1], h[1, 2], h[2, 1], h[2, 2]]),
                 box=1.0, positions=np.zeros((3, 3)))
    d, _ = orc.density_columns(w)
    s0 = _sign2(h[:2, :2])
    s2 = _sign2(h[1:, 1:])
    lam, V = np.linalg.eigh(h)
    s1 = (V * np.sign(lam)) @ V.T
    expect = np.array([
        0.5 * (1 - s0[0, 0]),      # D(0,0): column 0 of sign(T_0), row 0
        -0.5 * s1[0, 1],           # D(0,1): column 1 of sign(T_1) = sign(H), row 0
        -0.5 * s0[1, 0],           # D(1,0)
        0.5 * (1 - s1[1, 1]),      # D(1,1)
        -0.5 * s2[0, 1],           # D(1,2): column 2 -> local column 1 of sign(T_2), local row 0
        -0.5 * s1[2, 1],           # D(2,1)
        0.5 * (1 - s2[1, 1]),      # D(2,2)
    ])
    assert np.allclose(d, expect, atol=1e-14)


# ------------------------------------------------------- limits where the method is exact

def _neg_inertia(a):
    """Number of negative eigenvalues via LDL^T (Sylvester's law), independent of Jacobi."""
    _, d, _ = scipy.linalg.ldl(a)
    n = d.shape[0]
    neg, i = 0, 0
    while i < n:
        if i + 1 < n and d[i + 1, i] != 0.0:
            blk = d[i:i + 2, i:i + 2]
            det = blk[0, 0] * blk[1, 1] - blk[0, 1] * blk[1, 0]
            neg += 1 if det < 0 else (2 if blk[0, 0] + blk[1, 1] < 0 else 0)
            i += 2
        else:
            neg += int(d[i, i] < 0)
            i += 1
    return neg


def test_full_coverage_equals_full_matrix_sign():
    # every N(i) = all blocks  =>  every T_i = H  =>  D = 1/2 (I - sign(H))   [north_star pin]
    w = make_config(0, cutoff=np.inf)
    assert w.nnzb == w.n_blk ** 2
    d, st = orc.density_columns(w, n_threads=4)
    D = Workload(**{**w.__dict__, "vals": d}).dense()
    H = w.dense()
    lam, V = np.linalg.eigh(H)
    D_full = 0.5 * (np.eye(w.n) - (V * np.sign(lam)) @ V.T)
    assert np.abs(D - D_full).max() < 1e-13
    assert np.abs(D @ D - D).max() < 1e-12              # idempotent
    assert np.abs(D - D.T).max() < 1e-13
    n_neg = _neg_inertia(H)
    assert n_neg == int((lam < 0).sum())
    assert abs(orc.trace(w, d) - n_neg) < 1e-10         # Tr D = number of negative eigenvalues
    assert (st.n_neg == n_neg).all()


def test_mu_search_brackets_the_target_eigenvalue_in_the_full_coverage_limit():
    # full coverage: Tr D(mu) = #{eigenvalues of H below mu} exactly, so the chemical potential that gives
    # n_target electrons must lie strictly between eigenvalue n_target and eigenvalue n_target + 1 of H
    # (numpy eigvalsh: independent of the oracle's Jacobi path)                     [PAPER.md:89-92, Eq. 14]
    w = make_workload(10, 6, 3, np.inf, seed=5)
    assert w.nnzb == w.n_blk ** 2
    lam = np.linalg.eigvalsh(w.dense())
    for n_target in (7, 30, 44):
        mu, n, trials, d = orc.mu_search(w, n_target, -3.0, 3.0, tol_n=1e-8, n_threads=4)
        assert lam[n_target - 1] < mu < lam[n_target], (mu, lam[n_target - 1], lam[n_target])
        assert abs(n - n_target) < 1e-9 and abs(orc.trace(w, d) - n) < 1e-12
        assert 3 <= trials <= 40
    with pytest.raises(ValueError):
        orc.mu_search(w, 200, -3.0, 3.0)              # more electrons than orbitals: not bracketed


def test_trace_is_monotone_in_mu_away_from_the_limits():
    w = make_config(0)
    prev = -1.0
    for mu in np.linspace(-2.5, 2.5, 11):
        d, _ = orc.density_columns(w, mu=float(mu), n_threads=4)
        t = orc.trace(w, d)
        assert t >= prev - 1e-9
        prev = t
    assert prev == pytest.approx(w.n, abs=1e-9)        # everything occupied far above the spectrum


def test_block_diagonal_limit_gives_block_projectors():
    w = make_config(0, cutoff=0.0)
    assert w.nnzb == w.n_blk
    d, _ = orc.density_columns(w)
    b = int(w.blk_size[0])
    for i in range(w.n_blk):
        h = w.vals[w.val_ptr[i]:w.val_ptr[i + 1]].reshape(b, b)
        lam, V = np.linalg.eigh(h)
        proj = V[:, lam < 0] @ V[:, lam < 0].T
        assert np.abs(d[w.val_ptr[i]:w.val_ptr[i + 1]].reshape(b, b) - proj).max() < 1e-13


def test_each_submatrix_density_is_idempotent_but_assembled_D_is_not():
    w = make_config(0)
    for i in (0, 7, 31):
        T = orc.gather(w, i)
        Dsub = 0.5 * (np.eye(T.shape[0]) - orc.sign(T))
        assert np.abs(Dsub @ Dsub - Dsub).max() < 1e-12
    d, _ = orc.density_columns(w)
    D = Workload(**{**w.__dict__, "vals": d}).dense()
    # the method is an approximation: away from the limits D^2 != D
    assert 1e-4 < np.abs(D @ D - D).max() < 0.5


def test_negated_hamiltonian_gives_complement():
    w = make_config(0)
    d, _ = orc.density_columns(w)
    wn = Workload(**{**w.__dict__, "vals": -w.vals})
    dn, _ = orc.density_columns(wn)
    ident = np.zeros_like(d)
    b = int(w.blk_size[0])
    for i in range(w.n_blk):
        p = w.row_ptr[i] + int(np.searchsorted(w.col_idx[w.row_ptr[i]:w.row_ptr[i + 1]], i))
        ident[w.val_ptr[p]:w.val_ptr[p + 1]] = np.eye(b).ravel()
    assert np.abs(dn - (ident - d)).max() < 1e-12


def test_locality_subset_and_thread_count_do_not_change_columns():
    w = make_config(0)
    d_all, _ = orc.density_columns(w, n_threads=3)
    cols = [2, 3, 17, 30]
    d_sub, _ = orc.density_columns(w, cols=cols)
    mask = orc.column_mask(w, cols)
    assert np.array_equal(d_all[mask], d_sub[mask])
    assert not d_sub[~mask].any()


def test_relabelling_molecules_permutes_D():
    w = make_workload(12, 3, 1, 5.0, seed=77)
    perm = np.random.default_rng(5).permutation(w.n_blk)     # new label of old block i
    H = w.dense()
    b = 3
    idx = np.concatenate([np.arange(b) + b * int(np.where(perm == k)[0][0]) for k in range(w.n_blk)])
    Hp = H[np.ix_(idx, idx)]
    # rebuild the block-CSR of the relabelled matrix from its dense form
    nzb = [(i, j) for i in range(w.n_blk) for j in range(w.n_blk)
           if np.any(Hp[i * b:(i + 1) * b, j * b:(j + 1) * b] != 0.0)]
    row_ptr = np.zeros(w.n_blk + 1, np.int32)
    for i, _ in nzb:
        row_ptr[i + 1] += 1
    row_ptr = np.cumsum(row_ptr).astype(np.int32)
    col_idx = np.array([j for _, j in nzb], np.int32)
    vals = np.concatenate([Hp[i * b:(i + 1) * b, j * b:(j + 1) * b].ravel() for i, j in nzb])
    wp = Workload(n_blk=w.n_blk, blk_size=w.blk_size.copy(), row_ptr=row_ptr, col_idx=col_idx,
                  val_ptr=np.arange(len(nzb) + 1, dtype=np.int64) * b * b, vals=vals, box=w.box,
                  positions=w.positions)
    d, _ = orc.density_columns(w)
    dp, _ = orc.density_columns(wp)
    D = Workload(**{**w.__dict__, "vals": d}).dense()
    Dp = Workload(**{**wp.__dict__, "vals": dp}).dense()
    assert np.abs(Dp - D[np.ix_(idx, idx)]).max() < 1e-12


# ------------------------------------------------------------------ pattern

@pytest.mark.parametrize("cfg,pad", [(0, 1), (0, 16), (1, 64)])
def test_pattern_against_dense_boolean_adjacency(cfg, pad):
    w = make_config(cfg)
    P = orc.build_pattern(w, pad)
    n = w.n_blk
    adj = -np.ones((n, n), dtype=np.int64)               # stored-block index or -1
    for i in range(n):
        for p in range(w.row_ptr[i], w.row_ptr[i + 1]):
            adj[i, w.col_idx[p]] = p
    assert P.nbr_ptr[-1] == w.nnzb == P.sizes.nbr_len     # sum of counts = nnzb
    for i in range(n):
        nb = np.nonzero(adj[:, i] >= 0)[0]                # rows with a stored block in column i
        lo, hi = P.nbr_ptr[i], P.nbr_ptr[i + 1]
        assert np.array_equal(P.nbr_idx[lo:hi], nb)
        assert nb[P.own_pos[i]] == i
        sizes = w.blk_size[nb]
        assert P.dim[i] == sizes.sum()
        assert P.dim_pad[i] == -(-P.dim[i] // pad) * pad
        assert np.array_equal(P.row_off[lo:hi], np.concatenate([[0], np.cumsum(sizes)[:-1]]))
        g = P.gmap[P.gmap_ptr[i]:P.gmap_ptr[i + 1]].reshape(len(nb), len(nb))
        assert np.array_equal(g, adj[np.ix_(nb, nb)])
        assert (g[:, P.own_pos[i]] >= 0).all()            # column i is fully stored
    assert np.array_equal(P.sub_off, np.concatenate([[0], np.cumsum(P.dim_pad.astype(np.int64) ** 2)]))
    assert np.array_equal(P.tmap[P.tmap], np.arange(w.nnzb))
    for i in range(n):
        for p in range(w.row_ptr[i], w.row_ptr[i + 1]):
            assert adj[w.col_idx[p], i] == P.tmap[p]
    key = [(-int(P.dim_pad[i]), i) for i in range(n)]
    assert [int(x) for x in P.order] == [i for _, i in sorted(key)]
    assert P.sizes.max_dim == P.dim.max() and P.sizes.max_dim_pad == P.dim_pad.max()
    assert P.sizes.packed_elems == P.sub_off[-1] and P.sizes.gmap_len == P.gmap_ptr[-1]


def test_pattern_rejects_bad_structure():
    w = make_config(0)
    # drop one off-diagonal block: no longer structurally symmetric
    i = int(np.argmax(np.diff(w.row_ptr) > 1))
    p = w.row_ptr[i] + (1 if w.col_idx[w.row_ptr[i]] == i else 0)
    keep = np.ones(w.nnzb, bool)
    keep[p] = False
    row_ptr = w.row_ptr.copy()
    row_ptr[i + 1:] -= 1
    bad = Workload(**{**w.__dict__, "row_ptr": row_ptr, "col_idx": w.col_idx[keep]})
    assert orc.check_pattern(bad) == -3
    # unsorted columns
    ci = w.col_idx.copy()
    lo = w.row_ptr[i]
    ci[lo], ci[lo + 1] = ci[lo + 1], ci[lo]
    assert orc.check_pattern(Workload(**{**w.__dict__, "col_idx": ci})) == -3
    assert orc.check_pattern(w) == 0


def test_gather_against_dense_indexing():
    w = make_workload(20, np.array([2, 3, 5, 4] * 5), np.array([1, 1, 2, 2] * 5), 4.5, seed=9)
    H = w.dense()
    off = np.concatenate([[0], np.cumsum(w.blk_size)])
    for i in (0, 5, 19):
        nb = w.col_idx[w.row_ptr[i]:w.row_ptr[i + 1]]
        idx = np.concatenate([np.arange(off[j], off[j + 1]) for j in nb])
        # dense principal submatrix: entries between members of N(i) that are not stored are zero in H too
        assert np.array_equal(orc.gather(w, i, mu=0.25), H[np.ix_(idx, idx)] - 0.25 * np.eye(len(idx)))


# ------------------------------------------------------------- symmetrise / trace

def test_symmetrise_is_exactly_symmetric_and_trace_preserving():
    w = make_config(0)
    d, _ = orc.density_columns(w)
    ds = orc.symmetrise(w, d)
    D = Workload(**{**w.__dict__, "vals": d}).dense()
    Ds = Workload(**{**w.__dict__, "vals": ds}).dense()
    assert np.array_equal(Ds, Ds.T)
    assert np.array_equal(Ds, 0.5 * (D + D.T))
    assert orc.trace(w, ds) == orc.trace(w, d)
    assert orc.trace(w, d) == pytest.approx(np.trace(D), abs=1e-12)
    assert np.abs(D - D.T).max() > 1e-4     # symmetrisation is not a no-op (reading A6)


def test_trace_is_near_but_not_equal_to_electron_count():
    w = make_config(0)
    d, st = orc.density_columns(w)
    tr = orc.trace(w, d)
    n_neg_full = int((np.linalg.eigvalsh(w.dense()) < 0).sum())
    assert abs(tr - n_neg_full) < 0.5 and abs(tr - round(tr)) > 1e-6


def test_lapack_variant_matches_jacobi_oracle():
    # density_columns_lapack swaps the eigensolver only; it must reproduce the Jacobi path
    w = make_config(0)
    cols = [0, 5, 9, 31]
    d_j, st_j = orc.density_columns(w, cols=cols)
    d_l, st_l = orc.density_columns_lapack(w, cols=cols)
    assert np.abs(d_j - d_l).max() < 1e-12
    assert np.array_equal(st_j.n_neg, st_l.n_neg)
    assert np.allclose(st_j.scale, st_l.scale, rtol=1e-14)
    d_j, _ = orc.density_columns(w, cols=cols, mode="nsk", k_fixed=7)
    d_l, _ = orc.density_columns_lapack(w, cols=cols, mode="nsk", k_fixed=7)
    assert np.abs(d_j - d_l).max() < 1e-12
    w2 = make_workload(40, 23, 4, 5.0, seed=3)
    d_j, _ = orc.density_columns(w2, cols=[1, 2])
    d_l, _ = orc.density_columns_lapack(w2, cols=[1, 2])
    assert np.abs(d_j - d_l).max() < 1e-11


def test_oracle_matches_stored_golden():
    # Regression fixture (tests/golden/README.md): what the pinned oracle returns for configs[0], written by
    # tests/golden/make_golden.py from oracle/ alone.  Tr D in the full-coverage limit is also a pin of its own:
    # 3 occupied orbitals x 32 molecules = 96 negative eigenvalues (BASELINE.json configs[0], north_star).
    import importlib.util
    import os
    here = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
    spec = importlib.util.spec_from_file_location("make_golden", os.path.join(here, "make_golden.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    now = mod.golden_values()
    stored = {}
    with open(os.path.join(here, "cfg0_oracle.txt")) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            k, v = line.split()
            stored[k] = float(v)
    assert set(stored) == set(now)
    for k, v in stored.items():
        assert abs(now[k] - v) <= 1e-11 * max(1.0, abs(v)), (k, now[k], v)
    assert abs(stored["trace_full_coverage"] - 96.0) <= 1e-9
    assert stored["trace_sym"] == stored["trace"]


# ---------------------------------------------------------------- f2: Eq. 12 / Eq. 14 with an overlap matrix

def _with_vals(w, vals):
    import copy
    w2 = copy.copy(w)
    w2.vals = vals
    return w2


def test_eq12_blocks_closed_forms_and_scipy():
    """sign([[0, T], [I, 0]]) = [[0, T^1/2], [T^-1/2, 0]] (reading A20): diagonal T in closed form, the
    result squares to I, its blocks are inverse to each other and square to T / T^-1, and they agree with
    scipy.linalg.sqrtm and with scipy's sign function of the non-symmetric block matrix."""
    import scipy.linalg as sl
    d = np.array([0.25, 1.0, 4.0, 9.0])
    Sg = orc.sign_block_matrix(np.diag(d))
    assert np.allclose(Sg[4:, :4], np.diag(d ** -0.5), atol=1e-14) and np.allclose(Sg[:4, 4:], np.diag(d ** 0.5), atol=1e-14)
    assert np.allclose(Sg[:4, :4], 0, atol=1e-14) and np.allclose(Sg[4:, 4:], 0, atol=1e-14)
    rng = np.random.default_rng(3)
    G = rng.standard_normal((9, 9))
    T = G @ G.T + 0.5 * np.eye(9)
    Sg = orc.sign_block_matrix(T)
    Z, Y = Sg[9:, :9], Sg[:9, 9:]
    assert np.abs(Sg @ Sg - np.eye(18)).max() < 1e-11                     # sign^2 = I
    assert np.abs(Z @ Y - np.eye(9)).max() < 1e-11 and np.abs(Y @ Y - T).max() < 1e-11
    assert np.abs(Z @ T @ Z - np.eye(9)).max() < 1e-11
    assert np.abs(Y - sl.sqrtm(T).real).max() < 1e-11
    M = np.block([[np.zeros((9, 9)), T], [np.eye(9), np.zeros((9, 9))]])
    assert np.abs(Sg - sl.signm(M).real).max() < 1e-9                     # library sign of the block matrix itself
    Zb, Yb = orc.inv_sqrt_blocks(T)                                       # the cheap form = the literal form
    assert np.abs(Zb - Z).max() < 1e-12 and np.abs(Yb - Y).max() < 1e-12
    with pytest.raises(ValueError):
        orc.inv_sqrt_blocks(np.diag([1.0, -1.0]))


def test_inv_sqrt_columns_limits_and_locality():
    from workloads.generator import make_overlap
    import scipy.linalg as sl
    wl = make_config(0)
    wS = make_overlap(wl)
    ev = np.linalg.eigvalsh(wS.dense())
    assert ev.min() > 0.3 and ev.max() < 2.0                              # the generator's S is s.p.d.
    z, y, lam = orc.inv_sqrt_columns(wS)
    assert lam.min() > 0
    # literal Eq. 13 on the doubled matrix and the block form give the same columns
    z2, y2, _ = orc.inv_sqrt_columns(wS, cols=[0, 17], literal=True)
    m = orc.column_mask(wS, [0, 17])
    assert np.abs(z[m] - z2[m]).max() < 1e-12 and np.abs(y[m] - y2[m]).max() < 1e-12
    # locality: a subset of columns gives the same columns
    z3, _, _ = orc.inv_sqrt_columns(wS, cols=[3, 9])
    m = orc.column_mask(wS, [3, 9])
    assert np.array_equal(z3[m], z[m])
    # full-coverage limit: every T_i = S, so the result IS S^-1/2: Z S Z = I, Z = inverse of scipy's sqrtm
    wf = make_config(0, cutoff=np.inf)
    wSf = make_overlap(wf)
    zf, yf, _ = orc.inv_sqrt_columns(wSf)
    Zd, Yd, Sd = _with_vals(wSf, zf).dense(), _with_vals(wSf, yf).dense(), wSf.dense()
    assert np.abs(Zd @ Sd @ Zd - np.eye(wSf.n)).max() < 1e-11
    assert np.abs(Zd - np.linalg.inv(sl.sqrtm(Sd).real)).max() < 1e-11
    assert np.abs(Yd @ Yd - Sd).max() < 1e-11
    # block-diagonal limit: T_i = S_ii, the result is the inverse square root of every diagonal block
    wb = make_config(0, cutoff=0.0)
    wSb = make_overlap(wb)
    zb, _, _ = orc.inv_sqrt_columns(wSb)
    for i in (0, 31):
        p = wb.row_ptr[i]
        B = wSb.vals[wb.val_ptr[p]:wb.val_ptr[p + 1]].reshape(6, 6)
        assert np.abs(zb[wb.val_ptr[p]:wb.val_ptr[p + 1]].reshape(6, 6) - np.linalg.inv(sl.sqrtm(B).real)).max() < 1e-12
    # away from the limits the submatrix result approximates S^-1/2 (approximate method)
    Zs = _with_vals(wS, z).dense()
    assert np.abs(Zs @ wS.dense() @ Zs - np.eye(wS.n)).max() < 5e-2


def test_eq14_nonorthogonal_density():
    """Eq. 14 with S != I: sign(S^-1 H - mu I) of the oracle (through the similarity to a symmetric matrix)
    equals Eq. 13 written out on the non-symmetric matrix with scipy (A (A^2)^-1/2); in the full-coverage limit P is the
    projector of the generalised eigenproblem H c = e S c (P S P = P, Tr(P S) = number of eigenvalues below mu, counted
    independently by scipy.linalg.eigh); S = I reduces to the orthogonal path."""
    from workloads.generator import make_overlap
    import scipy.linalg as sl
    wf = make_config(0, cutoff=np.inf)
    wSf = make_overlap(wf)
    Hd, Sd = wf.dense(), wSf.dense()
    for mu in (0.0, 0.3):
        P = _with_vals(wf, orc.density_nonorth_columns(wf, wSf, mu)).dense()
        ev, Cg = sl.eigh(Hd, Sd)
        occ = ev < mu
        assert np.abs(P - Cg[:, occ] @ Cg[:, occ].T).max() < 1e-10
        assert abs(np.trace(P @ Sd) - occ.sum()) < 1e-9
        assert np.abs(P @ Sd @ P - P).max() < 1e-10
        A = np.linalg.solve(Sd, Hd) - mu * np.eye(wf.n)                    # Eq. 13 on the non-symmetric A itself
        sgA = A @ np.linalg.inv(sl.sqrtm(A @ A)).real
        assert np.abs(P - 0.5 * (np.eye(wf.n) - sgA) @ np.linalg.inv(Sd)).max() < 1e-9
    # S = I: Eq. 14 reduces to D = 1/2 (I - sign(H - mu I)), the orthogonal path of the same oracle
    wl = make_config(0)
    wI = _with_vals(wl, wl.vals * 0.0)
    for i in range(wl.n_blk):
        p = wl.row_ptr[i] + int(np.searchsorted(wl.col_idx[wl.row_ptr[i]:wl.row_ptr[i + 1]], i))
        wI.vals[wl.val_ptr[p]:wl.val_ptr[p + 1]] = np.eye(6).ravel()
    d0, _ = orc.density_columns(wl)
    assert np.abs(orc.density_nonorth_columns(wl, wI, 0.0) - d0).max() < 1e-12


def test_lapack_variant_is_pinned_to_jacobi_at_configs4_size():
    """The full-size configs[2] / configs[4] parity tests use oracle.density_columns_lapack; BASELINE.json names the
    Jacobi oracle.  tests/golden/cfg4_jacobi_vs_lapack.txt records one configs[4] column (m ~ 1600) through BOTH (written
    by tests/golden/make_cfg4_jacobi_pin.py from oracle/ alone, ~5 min of Jacobi sweeps): they agree to 1e-10.
    RUN_SLOW=1 repeats the comparison instead of reading the record."""
    import importlib.util
    here = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
    if os.environ.get("RUN_SLOW") == "1":
        spec = importlib.util.spec_from_file_location("make_cfg4_jacobi_pin", os.path.join(here, "make_cfg4_jacobi_pin.py"))
        mod = importlib.util.module_from_spec(spec)
        spec.loader.exec_module(mod)
        rec = mod.compare()
    else:
        rec = {}
        for ln in open(os.path.join(here, "cfg4_jacobi_vs_lapack.txt")):
            if not ln.startswith("#"):
                k, v = ln.split(None, 1)
                rec[k] = float(v)
    assert rec["m"] >= 1200                                   # a large-submatrix-regime column, not a small one
    assert rec["max_abs_diff"] <= 1e-10
    assert rec["frobenius_jacobi"] > 1.0                      # a real block column of D, not zeros


def test_oracle_under_address_and_undefined_behaviour_sanitizers(tmp_path):
    """the host oracle built with -fsanitize=address,undefined runs configs[0] (pattern, gather,
    Jacobi, sign, NS-k polynomial, scatter, symmetrise, trace; two threads) without a report."""
    import subprocess
    import sys
    so = str(tmp_path / "liborc_asan.so")
    src = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "oracle", "submatrix_oracle.c")
    subprocess.check_call(["gcc", "-O1", "-g", "-fsanitize=address,undefined", "-fno-omit-frame-pointer", "-fPIC", "-shared",
                           "-pthread", "-o", so, src, "-lm"])
    asan = subprocess.check_output(["gcc", "-print-file-name=libasan.so"], text=True).strip()
    code = ("import numpy as np\n"
            "from oracle import oracle as orc\n"
            "from workloads.generator import make_config\n"
            "wl = make_config(0)\n"
            "P = orc.build_pattern(wl, 16)\n"
            "d, st = orc.density_columns(wl, n_threads=2)\n"
            "dk, _ = orc.density_columns(wl, cols=np.arange(4, dtype=np.int32), mode='nsk', k_fixed=5)\n"
            "ds = orc.symmetrise(wl, d)\n"
            "print('TRACE', orc.trace(wl, ds))\n")
    env = dict(os.environ, ORC_SO=so, LD_PRELOAD=asan, ASAN_OPTIONS="detect_leaks=0", UBSAN_OPTIONS="halt_on_error=1",
               PYTHONPATH=os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    p = subprocess.run([sys.executable, "-c", code], env=env, capture_output=True, text=True, timeout=600)
    assert p.returncode == 0, p.stderr[-3000:]
    assert "TRACE" in p.stdout
    assert "AddressSanitizer" not in p.stderr and "runtime error" not in p.stderr, p.stderr[-3000:]
