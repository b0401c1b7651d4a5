#!/usr/bin/env python
"""Writes tests/golden/cfg3_lowest_eigs.txt: the lowest eigenvalues of the tangent Hessian of the FULL-SIZE
BASELINE.json configs[3] instance (1000x1000 periodic, ~200 skyrmions, seed 1003; 2,000,000 unknowns) and of its
same-density 316x316 instance, from the CPU oracle alone (oracle/spin_oracle.py: explicit sparse tangent Hessian
O1-O7 + ARPACK shift-invert, the O-sparse route of SURVEY.md 8(c); PAPER.md:162 explicit-Hessian procedure).

Nothing here touches the CUDA path.  Two passes, both over a sparse LU of (H_t - sigma I):
  pass 1  sigma = -0.5 (below the spectrum), 4 pairs, tol 1e-6   -> crude lambda_1
  pass 2  sigma = lambda_1 - 2e-3, 12 pairs, tol 0 (machine precision; relative gaps are now O(1e-2))
Cost at L = 1000 on 8 cores: ~20 min per LU (1.55e9 nonzeros in L+U, 35 GB RSS), ~17 + ~7 min ARPACK.

    python tests/golden/make_cfg3_eigs.py [316] [1000]
"""
import os
import sys
import time

import numpy as np
import scipy.sparse as sp
import scipy.sparse.linalg as spla

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle import spin_oracle as so  # noqa: E402
from paper_2509_26269_b200 import workloads as wl  # noqa: E402  (seeded input generator only)


def lowest(L: int, nev: int = 12):
    w = wl.config3() if L == 1000 else wl.config3_scaled(L)
    model = so.SpinModel(w.Lx, w.Ly, w.pbc_x, w.pbc_y, w.J, w.D, w.K, w.B, w.mu)
    Ht, _ = so.tangent_hessian(model, w.spins, dense=False)
    Ht = (0.5 * (Ht + Ht.T)).tocsc()
    n = Ht.shape[0]
    lam = None
    for sigma, k, tol in ((-0.5, 4, 1e-6), (None, nev, 0.0)):
        if sigma is None:
            sigma = float(lam[0]) - 2e-3
        t0 = time.time()
        lu = spla.splu((Ht - sigma * sp.identity(n, format="csc")).tocsc())
        op = spla.LinearOperator(Ht.shape, matvec=lu.solve, dtype=np.float64)
        lam = np.sort(spla.eigsh(Ht, k=k, sigma=sigma, which="LM", OPinv=op, tol=tol, ncv=max(4 * k, 32))[0])
        print(f"L={L} sigma={sigma:.6f} k={k}: {time.time() - t0:.0f} s", lam[:4], flush=True)
        del lu, op
    return w, lam


def main():
    sizes = [int(a) for a in sys.argv[1:]] or [316]
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "cfg3_lowest_eigs.txt")
    old = {}
    if os.path.exists(out):
        for line in open(out):
            if line.startswith("L="):
                old[int(line.split()[0][2:])] = line
    for L in sizes:
        w, lam = lowest(L)
        old[L] = f"L={L} seed={w.seed} " + " ".join(f"{x:.15e}" for x in lam) + "\n"
    with open(out, "w") as f:
        f.write("# lowest 12 eigenvalues of the tangent Hessian, BASELINE.json configs[3] recipe (workloads.config3 /\n"
                "# config3_scaled), written by tests/golden/make_cfg3_eigs.py from oracle/spin_oracle.py only\n"
                "# (PAPER.md:162 explicit Hessian; SURVEY.md 8(c) O-sparse: ARPACK shift-invert on the explicit sparse H_t)\n")
        for L in sorted(old):
            f.write(old[L])


if __name__ == "__main__":
    main()
