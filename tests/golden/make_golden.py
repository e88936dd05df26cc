"""Writes tests/golden/cfg0_oracle.txt from the CPU oracle alone (never from the CUDA path)."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from oracle import oracle as orc                      # noqa: E402
from workloads.generator import make_config           # noqa: E402

SAMPLE = (0, 1, 7, 36, 100, 1000, 5000, -1)          # stored-element indices of D recorded in the fixture


def golden_values():
    wl = make_config(0)
    d, _ = orc.density_columns(wl)
    d_sym = orc.symmetrise(wl, d)
    full = make_config(0, cutoff=np.inf)              # full coverage: D is the exact projector, Tr D an integer
    d_full, _ = orc.density_columns(full)
    out = {"n": int(wl.n), "n_blk": int(wl.n_blk), "nnzb": int(wl.nnzb), "n_vals": int(d.size),
           "trace": orc.trace(wl, d), "trace_sym": orc.trace(wl, d_sym), "trace_full_coverage": orc.trace(full, d_full),
           "frobenius": float(np.linalg.norm(d)), "sum": float(d.sum())}
    for k in SAMPLE:
        out["d[%d]" % k] = float(d[k])
    return out


if __name__ == "__main__":
    vals = golden_values()
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfg0_oracle.txt")
    with open(path, "w") as f:
        f.write("# configs[0] through oracle/ (exact sign by cyclic Jacobi); written by tests/golden/make_golden.py\n")
        for k, v in vals.items():
            f.write("%s %s\n" % (k, repr(v)))
    print(path)
