"""CPU ORACLE (test infrastructure, NOT the product) -- two-sided minimum-mode descent.

  seeds            x_seed = R(x_saddle + s * eta * v_min), s in {+1, -1}      PAPER.md:271-274 (Alg. 1 l.15-16), :307
  RelaxDownHill    "relax downhill to local minima using a deterministic optimizer (e.g., L-BFGS/CG)"
                   PAPER.md:275 (Alg. 1 l.17), :307 (Suppl. Note 1 b(iii))

The paper names the optimiser class and nothing else (no line search, no constants), so the algorithm below is the
reading DESIGN.md lists as A26 -- Riemannian Polak-Ribiere+ nonlinear conjugate gradients with backtracking:

  d_0 = -g_0                                   g = tangent-projected / masked gradient
  trial  x_t = R(x + a d),  a = alpha, alpha/2, alpha/4, ...  (at most MAX_BACKTRACKS)
  accept if   g_t.d <= SIGMA |g.d|            (no overshoot: the directional derivative at the trial point is not
                                               strongly positive; one-sided strong-Wolfe test, rounding-robust)
        and ( E_t <= E + C1 a (g.d)            (Armijo)
           or E_t <= E + EPS_E |E| )           (the energy test is blind once the decrease drops below the rounding of
                                               E; then the derivative test alone decides, as in Hager & Zhang's
                                               approximate Wolfe conditions)
  beta = max(0, (g_t.g_t - g_t.g) / (g.g))     (PR+; g_t is tangent at x_t, so transporting g by projection leaves
                                                g_t.g unchanged)
  d   <- -g_t + beta T(d),  T = projection onto the tangent space at x_t (spins) / identity (atoms; d is masked)
       if the new d is not a descent direction (g_t.d >= 0) it is reset to -g_t
  alpha <- 2a if the first trial was accepted, else a
  stop: |g|_2 <= tau_F (converged) | max_steps | every trial along -g rejected (stalled)

Written against four callables (energy, gradient, retract, transport) so that the same loop can be pinned on a plain
quadratic in R^n (tests/test_oracle_relax.py: minimiser == numpy.linalg.solve), on the ferromagnet (closed-form
energy -N(6J + K + mu B)), on a Morse trimer (bond lengths r0) and on a 2-D double well for the two-sided descent.
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline legs may import this file; it shares no code with
the CUDA path.  Parity status: pinned -- end points as above, and step by step (tests/test_oracle_relax.py): a 1-D sequence
derived by hand from the rule (a rejected overshoot, a doubled step, two restarts to steepest descent, evaluation counts),
and the direction update against textbook linear CG after an exact step (beta, signs).  The trajectory is compared with the
CUDA path only while the accept/reject decisions sit well above rounding.
"""
from __future__ import annotations

import numpy as np

C1 = 1e-4
EPS_E = 1e-10
SIGMA = 0.5
MAX_BACKTRACKS = 40


def relax_downhill(energy, gradient, retract, transport, x0, max_steps, tau_F, alpha0, trace=None):
    """Returns (x, info) with info = dict(steps, converged, evals, energy, gnorm, alpha).
    trace: optional list, receives (E, |g|, a) after every accepted step."""
    x = np.array(x0, dtype=np.float64, copy=True)
    E = energy(x)
    g = gradient(x)
    evals = 1
    d = -g
    gg = float(np.sum(g * g))
    slope = -gg
    steepest = True
    alpha = float(alpha0)
    steps = 0
    converged = False
    while True:
        if np.sqrt(gg) <= tau_F:
            converged = True
            break
        if steps >= max_steps:
            break
        a = alpha
        accepted = False
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
        if not accepted:
            if steepest:
                break                         # stalled: no acceptable step along -g
            d = -g
            slope = -gg
            steepest = True
            continue
        gtgt = float(np.sum(gt * gt))
        gtg = float(np.sum(gt * g))
        beta = max(0.0, (gtgt - gtg) / gg)
        new_slope = -gtgt + beta * gtd
        if new_slope >= 0.0:
            beta = 0.0
            new_slope = -gtgt
        d = -gt + beta * transport(xt, d)
        steepest = beta == 0.0
        x, E, g, gg, slope = xt, Et, gt, gtgt, new_slope
        alpha = 2.0 * a if first else a
        steps += 1
        if trace is not None:
            trace.append((E, np.sqrt(gg), a))
    info = dict(steps=steps, converged=converged, evals=evals, energy=E, gnorm=float(np.sqrt(gg)), alpha=alpha)
    return x, info


def two_sided_descent(energy, gradient, retract, transport, x_saddle, v_min, eta, max_steps, tau_F, alpha0):
    """Alg. 1 l.15-18: for s in (+1, -1): seed = R(x_saddle + s eta v_min), relax downhill.
    Returns [(x_min, info) for s = +1, (x_min, info) for s = -1]."""
    out = []
    for s in (1.0, -1.0):
        seed = retract(x_saddle + s * eta * v_min)
        out.append(relax_downhill(energy, gradient, retract, transport, seed, max_steps, tau_F, alpha0))
    return out


# ---- the four callables for the two model families (thin adaptors; the physics stays in spin_oracle / cart_oracle)
def spin_ops(model):
    from . import spin_oracle as so

    def retract(x):
        return x / np.linalg.norm(x, axis=1, keepdims=True)            # A7

    def transport(x, d):
        return d - np.sum(x * d, axis=1, keepdims=True) * x             # A17: projection onto the tangent space at x

    return (lambda m: so.energy(model, m)), (lambda m: so.projected_gradient(model, m)), retract, transport


def cart_ops(model):
    from . import cart_oracle as co

    return (lambda x: co.energy(model, x)), (lambda x: co.gradient(model, x, masked=True)), (lambda x: x), (lambda x, d: d)
