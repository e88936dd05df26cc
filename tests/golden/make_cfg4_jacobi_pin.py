"""Writes tests/golden/cfg4_jacobi_vs_lapack.txt from the CPU oracle alone: ONE configs[4] block column (m ~ 1650)
through the Jacobi oracle (oracle.density_columns, the definition BASELINE.json names) and through the LAPACK variant
(oracle.density_columns_lapack) that the full-size configs[2] / configs[4] parity tests use, and their agreement.
About 10 minutes on one core; tests/test_oracle_pins.py checks the recorded agreement and re-runs the comparison
itself when RUN_SLOW=1."""
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from oracle import oracle as orc                      # noqa: E402
from workloads.generator import make_config, sample_columns           # noqa: E402


def compare(col=None):
    wl = make_config(4)
    col = int(sample_columns(wl, 1, 4242)[0]) if col is None else col
    t0 = time.perf_counter()
    d_j, st_j = orc.density_columns(wl, cols=np.array([col], dtype=np.int32), n_threads=1)
    t_j = time.perf_counter() - t0
    d_l, st_l = orc.density_columns_lapack(wl, cols=[col])
    mask = orc.column_mask(wl, [col])
    m = int(wl.blk_size[wl.col_idx[wl.row_ptr[col]:wl.row_ptr[col + 1]]].sum())
    return dict(column=col, m=m, max_abs_diff=float(np.abs(d_j[mask] - d_l[mask]).max()),
                frobenius_jacobi=float(np.linalg.norm(d_j[mask])), min_abs_eig_lapack=float(st_l.min_abs_eig[0]),
                jacobi_seconds=t_j)


if __name__ == "__main__":
    vals = compare()
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfg4_jacobi_vs_lapack.txt")
    with open(path, "w") as f:
        f.write("# one configs[4] column: oracle.density_columns (cyclic Jacobi) vs oracle.density_columns_lapack; "
                "written by tests/golden/make_cfg4_jacobi_pin.py (oracle/ only)\n")
        for k, v in vals.items():
            f.write("%s %s\n" % (k, repr(v)))
    print(path, vals)
