"""Writes tests/golden/config0_Pu_true.txt: P u_true of BASELINE.json configs[0].

Calls only oracle/ (and the seeded model recipe in workloads/).  u_true is the
complex128 solution of A(m_true) u = q, q = unit point source at (16,16,4), in
the model with the +10 % Gaussian anomaly (sigma = 3 cells) at the centre.  It is
obtained with the oracle's own LSQR on the square system (no receivers, lambda = 1)
run to a normal-equations residual of 1e-12 relative; the true residual
||A u - q|| is printed (4e-12 when this file was written).

Usage:  python tests/golden/make_config0.py
Output: 16 lines "re im" (float64 repr), receiver order = workloads.config0 order
        (iy-major lattice {4,12,20,28}^2 at iz = 2).
"""
import math
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import oracle as O  # noqa: E402
from workloads.configs import config0_true_model, _grid_nodes, _lattice  # noqa: E402


def main():
    n = 32
    op = O.Operator(n, n, n, 10.0, 2.0 * math.pi * 5.0, 8)
    m_true = config0_true_model()
    q = np.zeros(op.ng, dtype=np.complex128)
    q[(4 * n + 16) * n + 16] = 1.0
    none = np.zeros(0, dtype=np.int64)
    out = O.lsqr(op, m_true, 1.0, none, q, np.zeros(0), tol=1e-12, maxit=5000)
    u = out["x"]
    print("iters", out["iters"], "||A u - q|| =", np.linalg.norm(O.apply_A(op, m_true, u) - q))
    xs = _lattice(n, 4)
    rec = O.rec_cells(n, n, n, _grid_nodes(xs, xs, 2))
    pu = u[rec]
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "config0_Pu_true.txt")
    with open(path, "w") as f:
        f.write("# P u_true for BASELINE.json configs[0]; written by tests/golden/make_config0.py\n")
        for z in pu:
            f.write("%r %r\n" % (float(z.real), float(z.imag)))
    print("wrote", path)


if __name__ == "__main__":
    main()
