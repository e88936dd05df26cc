"""sm_sign_ns_static -- the allocation-free variant of sm_sign_ns (workspace in a file-scope device array, no_alloc.cu) --
against the existing path (sm_sign_ns with a caller workspace) on the same gathered submatrices, and against the oracle's
NS-k polynomial.  Collected last on purpose (pytest -x must not hide other tests behind it); passes
alone in a fresh process and after the other tests."""
import gc

import numpy as np
import pytest

from oracle import oracle as orc
from workloads.generator import make_config, make_workload

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


@pytest.fixture(scope="module")
def sm():
    import paper_2205_14741_b200.binding as b   # raises if libsubmatrix.so is missing: no fallback
    return b


def _gathered(sm, wl, x_dtype, mu):
    A = sm.Bcsr(wl)
    P = sm.sm_build_pattern(A, 16)
    cols, col_off, n = sm.sm_plan_columns(P, P.order)
    X, scale = sm.sm_gather(A, P, cols, col_off, n, mu, "gershgorin", x_dtype)
    return A, P, cols, col_off, n, X


@pytest.mark.parametrize("x_dtype,tol_abs", [("f64", 1e-12), ("f32", 1e-5)])
def test_static_workspace_matches_the_existing_path_on_two_calls_in_a_row(sm, x_dtype, tol_abs):
    wl = make_config(0)
    # call 2 runs on different matrices (shifted by mu), with a different step count (odd: the result is copied back from
    # the scratch image) and finds call 1's contents in the shared array
    for call, (mu, k, tol) in enumerate([(0.0, 6, 0.0), (0.07, 9, 0.0), (0.0, 100, 1e-8 if x_dtype == "f64" else 1e-5)]):
        A, P, cols, col_off, n, X = _gathered(sm, wl, x_dtype, mu)
        assert sm.sm_sign_ws_bytes(P, n, P.packed_elems, x_dtype) <= sm.sm_sign_ns_static_capacity()
        X_ref = X.clone()
        it_ref, res_ref = sm.sm_sign_ns(P, cols, col_off, n, P.packed_elems, x_dtype, X_ref, k, tol)
        # everything the new entry point touches is allocated BEFORE the call; the call itself must not allocate
        iters = torch.full((n,), -7, dtype=torch.int32, device=X.device)
        residual = torch.full((n,), -1.0, dtype=torch.float64, device=X.device)
        gc.collect()        # tensors of earlier tests must not be freed between the two readings
        torch.cuda.synchronize()
        before, free_before = torch.cuda.memory_allocated(), torch.cuda.mem_get_info()[0]
        sm.sm_sign_ns_static(P, cols, col_off, n, P.packed_elems, x_dtype, X, k, tol, iters, residual)
        torch.cuda.synchronize()
        assert torch.cuda.memory_allocated() <= before, "torch allocated device memory inside the call"
        if call > 0:        # (the first call may still load the kernels' module and asks for the array's address)
            assert torch.cuda.mem_get_info()[0] >= free_before, "device memory was allocated inside the call"
        # same kernels, same order of operations: bit-identical to the existing path, and within the parity tolerance
        assert torch.equal(X, X_ref), call
        assert torch.equal(iters, it_ref) and torch.equal(residual, res_ref), call
        assert float((X.double() - X_ref.double()).abs().max()) <= tol_abs
        if tol == 0.0:
            assert (iters == k).all()
            # ... and the oracle's NS-k polynomial for a few submatrices (first, middle, last of P.order)
            Ph = sm.pattern_to_host(P)
            order = P.order.cpu().numpy()
            off = col_off.cpu().numpy()
            for pos in (0, n // 2, n - 1):
                i = int(order[pos])
                T = orc.gather(wl, i, mu)
                m, Pd = T.shape[0], int(Ph.dim_pad[i])
                x = X[off[pos]:off[pos] + Pd * Pd].double().cpu().numpy().reshape(Pd, Pd)
                assert np.abs(x[:m, :m] - orc.ns_polynomial(T, orc.gershgorin(T), k)).max() <= tol_abs
                assert not x[m:].any() and not x[:, m:].any()
        else:
            assert sm.sm_sign_status(residual, tol) == sm.SM_OK


def test_static_workspace_rejects_what_does_not_fit_or_would_allocate(sm):
    # 40 submatrices of dimension ~ 500: two fp64 images of 40 * 512^2 * 8 B = 84 MB each > the 16 MiB array
    wl = make_workload(40, 23, 4, 9.0, seed=5)
    A, P, cols, col_off, n, X = _gathered(sm, wl, "f64", 0.0)
    assert sm.sm_sign_ws_bytes(P, n, P.packed_elems, "f64") > sm.sm_sign_ns_static_capacity()
    iters = torch.zeros(n, dtype=torch.int32, device=X.device)
    residual = torch.zeros(n, dtype=torch.float64, device=X.device)
    X0 = X.clone()
    with pytest.raises(sm.SmError) as e:
        sm.sm_sign_ns_static(P, cols, col_off, n, P.packed_elems, "f64", X, 3, 0.0, iters, residual)
    assert e.value.status == sm.SM_ERR_SPACE
    torch.cuda.synchronize()
    assert torch.equal(X, X0)                                  # nothing was launched
    # 16-bit types keep a lazily allocated pinned error word: refused
    wl0 = make_config(0)
    A = sm.Bcsr(wl0)
    P = sm.sm_build_pattern(A, 64)
    cols, col_off, n = sm.sm_plan_columns(P, P.order)
    Xh, _ = sm.sm_gather(A, P, cols, col_off, n, 0.0, "gershgorin", "f16")
    iters = torch.zeros(n, dtype=torch.int32, device=Xh.device)
    residual = torch.zeros(n, dtype=torch.float64, device=Xh.device)
    with pytest.raises(sm.SmError) as e:
        sm.sm_sign_ns_static(P, cols, col_off, n, P.packed_elems, "f16", Xh, 3, 0.0, iters, residual)
    assert e.value.status == sm.SM_ERR_UNSUPPORTED
