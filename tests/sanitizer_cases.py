"""Small invocations of every kernel family for `compute-sanitizer` (tier 3):

    compute-sanitizer --tool memcheck  python tests/sanitizer_cases.py
    compute-sanitizer --tool racecheck python tests/sanitizer_cases.py
    compute-sanitizer --tool synccheck python tests/sanitizer_cases.py

Not collected by pytest (no test_ prefix); results are checked loosely (finite, symmetric) -- parity lives in the
test_gpu_*.py files.  One tool per gpurun call (B200_PROFILING.md)."""
import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import paper_2205_14741_b200.binding as sm                      # noqa: E402
from workloads.generator import make_config, make_overlap, make_workload      # noqa: E402


def density(wl, x_dtype, pad, max_iter, tol, scale="gershgorin", **opts):
    for k, v in opts.items():
        sm.set_option(k, v)
    A = sm.Bcsr(wl)
    P = sm.sm_build_pattern(A, pad)
    plan = sm.DensityPlan(A, P, x_dtype)
    sm.sm_density(A, P, plan, mu=0.0, scale_mode=scale, max_iter=max_iter, tol=tol, symmetrise=True)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(plan.D).all())
    print("ok", x_dtype, opts, "Tr D", plan.trace.item())
    for k in opts:
        sm.set_option(k, {"umma.resident": 1}.get(k, 0) if k != "umma.sym" else 1)


def main():
    small = make_config(0)                                   # m <= 78: resident kernel (16-bit), DFMA tiles (fp64)
    mid = make_workload(16, 23, 4, 5.0, seed=33)             # m ~ 250-450: grouped tiles
    mixed = make_workload(60, 6, 3, 6.0, seed=33)            # Pd 64 .. 256
    density(small, "f64", 16, 30, 1e-8)
    density(small, "f32", 16, 30, 1e-5)
    density(mid, "f64", 16, 4, 0.0)                          # DMMA tiles
    density(small, "bf16", 64, 6, 0.0)                       # k_umma_resident
    density(mixed, "f16", 64, 6, 0.0, scale="global")
    density(mixed, "f16", 64, 12, 1e-3)                      # resident kernel, convergence mode
    density(mid, "bf16", 64, 3, 0.0, scale="global")         # k_umma_gemm, dynamic deal
    density(mid, "bf16", 64, 3, 0.0, **{"umma.dyn": 0})
    density(mid, "f16", 64, 3, 0.0, **{"umma.stream": 1})
    density(mid, "bf16", 64, 3, 0.0, **{"umma.epi": 1})
    density(mid, "bf16", 64, 3, 0.0, **{"umma.epi": 1, "umma.lt": 1})
    density(mid, "f16", 64, 3, 0.0, **{"umma.sym": 0})
    density(mixed, "bf16", 64, 3, 0.0, **{"gather.tma": 1})
    # f2: Eq. 12 at doubled dimension (non-symmetric kernels) and Eq. 14 with an overlap matrix
    wS = make_overlap(small)
    S = sm.Bcsr(wS)
    for x_dtype, pad in (("f64", 16), ("bf16", 64)):
        P = sm.sm_build_pattern(S, pad)
        Z, _, _, res, _ = sm.sm_inv_sqrt(S, P, x_dtype, max_iter=8, tol=0.0)
        torch.cuda.synchronize()
        assert bool(torch.isfinite(Z).all())
    A = sm.Bcsr(small)
    P = sm.sm_build_pattern(A, 16)
    Pv, tr, _, _, _ = sm.sm_density_nonorth(A, S.vals, P, "f64", mu=0.0, max_iter=30, tol=1e-8)
    torch.cuda.synchronize()
    print("ok nonorth Tr(PS)", tr.item())
    print("SANITIZER CASES DONE")


if __name__ == "__main__":
    main()
