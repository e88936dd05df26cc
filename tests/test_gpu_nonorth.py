"""GPU parity of SURVEY.md 8(f) f2 -- non-orthogonal basis: S^-1/2 through Eq. 12 and Eq. 14 with an
overlap matrix -- against the oracle functions of oracle/oracle.py (inv_sqrt_columns,
density_nonorth_columns), on seeded (H, S) pairs with one block pattern (workloads.generator.make_overlap)."""
import numpy as np
import pytest

from oracle import oracle as orc
from workloads.generator import make_config, make_overlap, make_workload

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def sm():
    import paper_2205_14741_b200.binding as b
    return b


_ORACLE = {}


def oracle_cached(name, kind, fn):
    """Oracle results are reused by the tests of one workload (the Jacobi sweeps of the 23-orbital pair take 35-70 s)."""
    if (name, kind) not in _ORACLE:
        _ORACLE[(name, kind)] = fn()
    return _ORACLE[(name, kind)]


def pair(kind):
    wl = {"cfg0": lambda: make_config(0), "mid6": lambda: make_workload(150, 6, 3, 6.0, seed=71),
          "mid23": lambda: make_workload(24, 23, 4, 5.0, seed=72),
          "ragged": lambda: make_workload(40, np.array([2, 3, 5, 4, 7] * 8), np.array([1, 1, 2, 2, 3] * 8), 5.5, seed=11)}[kind]()
    return wl, make_overlap(wl)


@pytest.mark.parametrize("kind", ["cfg0", "mid6", "ragged"])
def test_inv_sqrt_fp64_all_columns(sm, kind):
    wl, wS = pair(kind)
    z_or, y_or, lam = oracle_cached("inv_sqrt", kind, lambda: orc.inv_sqrt_columns(wS))
    S = sm.Bcsr(wS)
    P = sm.sm_build_pattern(S, 16)
    Z, Y, iters, res, scale = sm.sm_inv_sqrt(S, P, "f64", max_iter=100, tol=1e-9, want_sqrt=True)
    torch.cuda.synchronize()
    assert sm.sm_sign_status(res, 1e-9) == sm.SM_OK
    assert np.abs(Z.cpu().numpy() - z_or).max() <= 1e-10
    assert np.abs(Y.cpu().numpy() - y_or).max() <= 1e-10
    # chunked (several chunks of doubled images) gives the same numbers
    tot2, big2 = sm._doubled_elems(P)
    Z2, _, _, _, _ = sm.sm_inv_sqrt(S, P, "f64", max_iter=100, tol=1e-9, max_chunk_elems2=max(big2, tot2 // 3))
    torch.cuda.synchronize()
    assert np.abs(Z2.cpu().numpy() - z_or).max() <= 1e-10


def test_inv_sqrt_fp32(sm):
    wl, wS = pair("mid6")
    z_or, _, _ = oracle_cached("inv_sqrt", "mid6", lambda: orc.inv_sqrt_columns(wS))
    S = sm.Bcsr(wS)
    P = sm.sm_build_pattern(S, 16)
    Z, _, iters, res, _ = sm.sm_inv_sqrt(S, P, "f32", max_iter=100, tol=1e-5)
    torch.cuda.synchronize()
    assert np.abs(Z.cpu().numpy() - z_or).max() <= 1e-4


@pytest.mark.parametrize("x_dtype,kind", [("bf16", "mid23"), ("f16", "mid23"), ("f16", "mid6"), ("bf16", "cfg0")])
def test_inv_sqrt_16bit(sm, x_dtype, kind):
    # doubled images up to 2 * 500 = 1000 rows: non-symmetric tcgen05 path (true products, MN-major B operand)
    wl, wS = pair(kind)
    z_or, _, _ = oracle_cached("inv_sqrt", kind, lambda: orc.inv_sqrt_columns(wS))
    S = sm.Bcsr(wS)
    P = sm.sm_build_pattern(S, 64)
    Z, _, iters, res, _ = sm.sm_inv_sqrt(S, P, x_dtype, max_iter=12, tol=0.0)
    torch.cuda.synchronize()
    Zh = Z.cpu().numpy()
    rel = np.linalg.norm(Zh - z_or) / np.linalg.norm(z_or)
    print(kind, x_dtype, "relF", rel)
    assert np.isfinite(Zh).all() and rel <= 2e-2


@pytest.mark.parametrize("x_dtype,lim,kind", [("f64", 1e-10, "cfg0"), ("f64", 1e-10, "mid6"), ("f32", 1e-4, "mid6"), ("f64", 1e-10, "ragged")])
def test_density_nonorth_matches_the_oracle(sm, x_dtype, lim, kind):
    wl, wS = pair(kind)
    mu = 0.05
    p_or = oracle_cached("nonorth%g" % mu, kind, lambda: orc.density_nonorth_columns(wl, wS, mu))
    A = sm.Bcsr(wl)
    Sd = sm.Bcsr(wS)
    P = sm.sm_build_pattern(A, 16)
    tol = 1e-9 if x_dtype == "f64" else 1e-5
    Pv, tr, iters, res, _ = sm.sm_density_nonorth(A, Sd.vals, P, x_dtype, mu=mu, max_iter=100, tol=tol)
    torch.cuda.synchronize()
    assert sm.sm_sign_status(res, tol) == sm.SM_OK
    Ph = Pv.double().cpu().numpy()
    assert np.abs(Ph - p_or).max() <= lim
    assert abs(tr.item() - float((p_or * wS.vals).sum())) <= (1e-9 if x_dtype == "f64" else 1e-3) * wl.n


def test_density_nonorth_full_coverage_is_the_generalised_projector(sm):
    import scipy.linalg as sl
    wl = make_config(0, cutoff=np.inf)
    wS = make_overlap(wl)
    A, Sd = sm.Bcsr(wl), sm.Bcsr(wS)
    P = sm.sm_build_pattern(A, 16)
    Pv, tr, _, res, _ = sm.sm_density_nonorth(A, Sd.vals, P, "f64", mu=0.0, max_iter=100, tol=1e-9, symmetrise=True)
    torch.cuda.synchronize()
    ev = sl.eigh(wl.dense(), wS.dense(), eigvals_only=True)
    assert abs(tr.item() - (ev < 0).sum()) <= 1e-8            # Tr(P S) = number of generalised eigenvalues below mu


# 16-bit Eq. 14 chains five 16-bit-rounded stages (sign of the doubled matrix, Z Z, S^-1 T_H, sign, (I - sign) S^-1 / 2): fp16
# stays far inside the hot path's relF limit 2e-2; bf16 (8 significand bits) is given twice that limit on the 23-orbital
# workload (measured 2.5e-2), the price of two chained sign iterations.
@pytest.mark.parametrize("x_dtype,kind,val_dtype,lim", [("f16", "mid23", "f64", 2e-2), ("bf16", "mid23", "f64", 4e-2),
                                                         ("f16", "mid6", "f32", 2e-2), ("bf16", "cfg0", "f32", 2e-2),
                                                         ("f16", "ragged", "f64", 2e-2)])
def test_density_nonorth_16bit(sm, x_dtype, kind, val_dtype, lim):
    """Eq. 14 with S != I on the tcgen05 kernels: S^-1/2 by the non-symmetric sign of the doubled matrix, the three dense
    products by the non-symmetric update kernel without its identity term (umma_product), the sign of S^-1 H - mu I."""
    wl, wS = pair(kind)
    mu = 0.05
    p_or = oracle_cached("nonorth%g" % mu, kind, lambda: orc.density_nonorth_columns(wl, wS, mu))
    A = sm.Bcsr(wl, val_dtype=val_dtype)
    Sd = sm.Bcsr(wS, val_dtype=val_dtype)
    P = sm.sm_build_pattern(A, 64)
    Pv, tr, iters, res, _ = sm.sm_density_nonorth(A, Sd.vals, P, x_dtype, mu=mu, max_iter=30, tol=0.0)
    torch.cuda.synchronize()
    Ph = Pv.cpu().numpy()
    rel = np.linalg.norm(Ph - p_or) / np.linalg.norm(p_or)
    dtr = abs(tr.item() - float((p_or * wS.vals).sum())) / wl.n
    print(kind, x_dtype, "relF", rel, "maxabs", np.abs(Ph - p_or).max(), "dTr/n", dtr)
    assert np.isfinite(Ph).all() and rel <= lim and dtr <= 1.5e-3
    assert (iters == 30).all()
    # chunked (buffer stride not a multiple of the image size) = unchunked, bit for bit
    tot2, big2 = sm._doubled_elems(P)
    Pc, _, _, _, _ = sm.sm_density_nonorth(A, Sd.vals, P, x_dtype, mu=mu, max_iter=30, tol=0.0, max_chunk_elems2=max(big2, tot2 // 3 + 1))
    torch.cuda.synchronize()
    assert torch.equal(Pc, Pv)
