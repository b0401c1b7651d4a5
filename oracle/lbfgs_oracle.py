"""CPU ORACLE (test infrastructure, NOT the product) -- the L-BFGS variants of the two optimiser loops of the bilayer kernel
(SURVEY 8(f) f2).

  PAPER.md:163  "We employ a GPU implementation of LBFGS (... LBFGS-B) ... and a nonlinear conjugate-gradient (CG) variant
                 for comparison"                                             -> L-BFGS is the paper's PRIMARY outer optimiser
  PAPER.md:262  Alg. 1 l.12  "x <- R_x(x + alpha F_mmf)   > Lbfgs/CG"       -> step rule of the climb          (mmf_run_lbfgs)
  PAPER.md:275  Alg. 1 l.17  RelaxDownHill; "a deterministic optimizer (e.g., L-BFGS/CG)"  (relax_downhill_lbfgs)

The paper calls a library routine and prints no algorithm, memory size, line search or safeguard.  Readings (A29, A30):

A29  RelaxDownHill, Riemannian L-BFGS.  History of at most M pairs (s_i, y_i), both TRANSPORTED to the current tangent space by
     projection at every accepted step (spins; identity for atoms): s = T(a d), y = g_new - T(g_old).  Direction d = -H g from
     the standard two-loop recursion (Nocedal 1980) with H_0 = gamma I, gamma = s.y / y.y of the newest pair; no history:
     d = -g.  A pair is stored only if s.y > CURV_EPS |s| |y| (else H stays positive definite without it).  Line search: the
     acceptance test of the CG loop (relax_oracle, reading A26: g_t.d <= SIGMA |g.d| and (Armijo or E_t <= E + EPS_E |E|)) with
     trial steps a = a_0, a_0/2, ... where a_0 = alpha0 while the history is empty and 1 (the quasi-Newton step) afterwards.
     If d is not a descent direction, or every trial along it is rejected, the history is dropped and the step retried along
     -g (a_0 = the last accepted first-step length); rejected there too: stalled.  Stop: |g|_2 <= tau_F, max_steps.

A30  Outer climb, L-BFGS on the reflected force.  F_mmf is not the gradient of a function, so there is no energy line search:
     x <- R(x + p),  p = H F_mmf  (two-loop recursion as above on pairs s = T(p), y = -(F_new - T(F_old)), H_0 = alpha0 I while
     the history is empty), |p|_2 capped at smax (the whole step is rescaled).  ONE MinMode solve per iteration (the CG rule,
     mmf_cg_oracle, spends two).  A pair is stored only if s.y > CURV_EPS |s| |y|; if F.p <= 0 the history is dropped and
     p = alpha0 F.  Stop: |F_mmf|_2 <= tau_F and lambda_1 < 0 < lambda_2, max_steps.

Pins (tests/test_oracle_lbfgs.py): the two-loop recursion against the explicit dense BFGS inverse update
H+ = (I - rho s y^T) H (I - rho y s^T) + rho s s^T applied pair by pair to gamma I (a textbook closed form that shares nothing
with the recursion), the secant equation H y_new = s_new, a 1-D sequence computed by hand, minimiser of an SPD quadratic =
numpy.linalg.solve, the quadratic saddle with an analytic minimum mode (the reflected force is then the gradient of
x^T |A| x / 2, whose stationary point is the saddle), the step cap, and the closed-form ferromagnet energy.
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline legs may import this file; it shares no code with the CUDA path.
"""
from __future__ import annotations

import numpy as np

from .relax_oracle import C1, EPS_E, MAX_BACKTRACKS, SIGMA

M_DEFAULT = 8
CURV_EPS = 1e-10


def two_loop(q, S, Y, gamma0):
    """r = H q for the L-BFGS inverse Hessian defined by the pairs (S[i], Y[i]), oldest first, H_0 = gamma I with
    gamma = s.y / y.y of the newest pair (gamma0 if there is none).  Nocedal's two-loop recursion."""
    q = np.array(q, dtype=np.float64, copy=True)
    n = len(S)
    if n == 0:
        return gamma0 * q
    rho = [1.0 / float(np.sum(S[i] * Y[i])) for i in range(n)]
    al = [0.0] * n
    for i in range(n - 1, -1, -1):
        al[i] = rho[i] * float(np.sum(S[i] * q))
        q -= al[i] * Y[i]
    gamma = float(np.sum(S[-1] * Y[-1])) / float(np.sum(Y[-1] * Y[-1]))
    r = gamma * q
    for i in range(n):
        be = rho[i] * float(np.sum(Y[i] * r))
        r += (al[i] - be) * S[i]
    return r


def _push(S, Y, s, y, M):
    """Store the pair if it has positive curvature; keep the newest M.  Returns True if stored."""
    sy = float(np.sum(s * y))
    if not sy > CURV_EPS * float(np.linalg.norm(s)) * float(np.linalg.norm(y)):
        return False
    S.append(s)
    Y.append(y)
    if len(S) > M:
        S.pop(0)
        Y.pop(0)
    return True


def relax_downhill_lbfgs(energy, gradient, retract, transport, x0, max_steps, tau_F, alpha0, M=M_DEFAULT, trace=None):
    """Reading A29.  Returns (x, info) with info = dict(steps, converged, evals, energy, gnorm, alpha, pairs).
    trace: optional list, receives (E, |g|, a, number of pairs used for the step) after every accepted step."""
    x = np.array(x0, dtype=np.float64, copy=True)
    E = energy(x)
    g = gradient(x)
    evals = 1
    S, Y = [], []
    alpha = float(alpha0)        # first-trial length along -g (used whenever the history is empty)
    steps = 0
    converged = False
    while True:
        gg = float(np.sum(g * g))
        if np.sqrt(gg) <= tau_F:
            converged = True
            break
        if steps >= max_steps:
            break
        accepted = False
        while True:
            npairs = len(S)
            d = -two_loop(g, S, Y, 1.0) if npairs else -g
            slope = float(np.sum(g * d))
            if npairs and not slope < 0.0:           # not a descent direction: drop the history
                S, Y = [], []
                continue
            a = 1.0 if npairs else alpha
            first = True
            for _ in range(MAX_BACKTRACKS):
                xt = retract(x + a * d)
                Et = energy(xt)
                gt = gradient(xt)
                evals += 1
                gtd = float(np.sum(gt * d))
                if gtd <= SIGMA * abs(slope) and (Et <= E + C1 * a * slope or Et <= E + EPS_E * abs(E)):
                    accepted = True
                    break
                a *= 0.5
                first = False
            if accepted or not npairs:
                break
            S, Y = [], []                            # every trial along the quasi-Newton direction rejected: retry along -g
        if not accepted:
            break                                    # stalled along -g
        if not npairs:
            alpha = 2.0 * a if first else a
        s = transport(xt, a * d)
        y = gt - transport(xt, g)
        S = [transport(xt, v) for v in S]
        Y = [transport(xt, v) for v in Y]
        _push(S, Y, s, y, M)
        x, E, g = xt, Et, gt
        steps += 1
        if trace is not None:
            trace.append((E, float(np.linalg.norm(g)), a, npairs))
    info = dict(steps=steps, converged=converged, evals=evals, energy=E, gnorm=float(np.sqrt(np.sum(g * g))), alpha=alpha,
                pairs=len(S))
    return x, info


def mmf_run_lbfgs(minmode, force, retract, transport, x0, alpha0, smax, max_steps, tau_F, M=M_DEFAULT, trace=None):
    """Reading A30.  minmode(x) -> (lam [k >= 2], V [k][...]);  force(x) -> F = -grad (tangent-projected / masked).
    Returns (x, lam, steps, converged, |F_mmf|, evals) with evals = number of MinMode solves."""
    def fmmf(x):
        lam, V = minmode(x)
        F = force(x)
        return lam, F - 2.0 * np.sum(F * V[0]) * V[0]

    x = np.array(x0, dtype=np.float64, copy=True)
    lam, F = fmmf(x)
    evals = 1
    S, Y = [], []
    steps = 0
    while True:
        fn = float(np.linalg.norm(F))
        if fn <= tau_F and lam[0] < 0.0 < lam[1]:
            return x, lam, steps, True, fn, evals
        if steps >= max_steps:
            return x, lam, steps, False, fn, evals
        p = two_loop(F, S, Y, alpha0)
        if S and not float(np.sum(F * p)) > 0.0:
            S, Y = [], []
            p = alpha0 * F
        pn = float(np.linalg.norm(p))
        if pn > smax:
            p = p * (smax / pn)
        xn = retract(x + p)
        lam, Fn = fmmf(xn)
        evals += 1
        s = transport(xn, p)
        y = -(Fn - transport(xn, F))
        S = [transport(xn, v) for v in S]
        Y = [transport(xn, v) for v in Y]
        _push(S, Y, s, y, M)
        x, F = xn, Fn
        steps += 1
        if trace is not None:
            trace.append((float(np.linalg.norm(F)), float(np.linalg.norm(p)), len(S), lam[0], lam[1]))
