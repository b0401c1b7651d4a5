"""CPU ORACLE (test infrastructure, NOT the product) -- outer minimum-mode-following loop with a conjugate-gradient step rule
(Alg. 1 l.9-14: "x <- R_x(x + alpha F_mmf)   > Lbfgs/CG").

The paper names the optimiser class for the outer layer and nothing else.  F_mmf is not the gradient of a function, so an
energy line search does not apply; the reading taken (A28) is the translation step of the dimer method
(Henkelman & Jonsson, J. Chem. Phys. 111, 7010 (1999)): Polak-Ribiere+ conjugate directions on the reflected force with a
one-trial secant line search on the force component along the direction:

  (lam, v) = MinMode(x);  F = F_mmf(x) = F - 2 (F.v_1) v_1  (Eq. 2);  d = F
  repeat:  stop if |F|_2 <= tau_F and lam_1 < 0 < lam_2
           dh = d / |d|;  f0 = F.dh
           trial  x_t = R(x + delta dh);  F_t = F_mmf(x_t) (MinMode at x_t);  f1 = F_t.T(dh)
           C = (f0 - f1) / delta                       (curvature of the effective landscape along dh)
           s = f0 / C  if C > 0 else smax;   s = min(max(s, -smax), smax)      (zero of the force along dh, capped)
           x <- R(x + s dh);  F_new = F_mmf(x) (MinMode at x)
           beta = max(0, F_new.(F_new - T(F)) / (F.F));   d = F_new + beta T(d);   F = F_new
  T = projection onto the tangent space at the new point (spins) / identity (atoms); R = retraction (spins) / identity.

Written against callables so that the loop can be pinned on a plain 2-D function with an analytic Hessian
(tests/test_oracle_relax.py) and on the spin lattice, where it must reach the saddle the fixed-step loop
(spin_oracle.mmf_run) reaches.  Parity status: pinned step by step on the quadratic saddle x^T diag(-1, 2, 3) x / 2 with its
analytic minimum mode (the secant step in closed form, its clip at smax, the negative-curvature branch, beta of linear CG,
exactness after three steps) and at the end point on the lattice.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline legs may import this file.
"""
from __future__ import annotations

import numpy as np


def mmf_run_cg(minmode, force, retract, transport, x0, delta, smax, max_steps, tau_F, trace=None):
    """minmode(x) -> (lam [k>=2], V [k][...]);  force(x) -> F = -grad (tangent-projected / masked).
    Returns (x, lam, steps, converged, |F_mmf|, evals) with evals = number of MinMode solves."""
    def fmmf(x):
        lam, V = minmode(x)
        F = force(x)
        return lam, F - 2.0 * np.sum(F * V[0]) * V[0]

    x = np.array(x0, dtype=np.float64, copy=True)
    lam, F = fmmf(x)
    evals = 1
    d = F.copy()
    steps = 0
    while True:
        fn = float(np.linalg.norm(F))
        if fn <= tau_F and lam[0] < 0.0 < lam[1]:
            return x, lam, steps, True, fn, evals
        if steps >= max_steps:
            return x, lam, steps, False, fn, evals
        dh = d / np.linalg.norm(d)
        f0 = float(np.sum(F * dh))
        xt = retract(x + delta * dh)
        _, Ft = fmmf(xt)
        f1 = float(np.sum(Ft * transport(xt, dh)))
        C = (f0 - f1) / delta
        s = f0 / C if C > 0.0 else smax
        s = min(max(s, -smax), smax)
        xn = retract(x + s * dh)
        lam, Fn = fmmf(xn)
        evals += 2
        beta = max(0.0, float(np.sum(Fn * (Fn - transport(xn, F)))) / float(np.sum(F * F)))
        d = Fn + beta * transport(xn, d)
        x, F = xn, Fn
        steps += 1
        if trace is not None:
            trace.append((float(np.linalg.norm(F)), s, beta, lam[0], lam[1]))
