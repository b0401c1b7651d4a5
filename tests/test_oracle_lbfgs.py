"""Pins for oracle/lbfgs_oracle.py (no GPU): the L-BFGS variants of RelaxDownHill and of the outer climb (readings A29, A30;
PAPER.md:163, :262, :275) against things that are not the loops themselves: the dense BFGS inverse-update formula, the
secant equation, a 1-D sequence computed by hand, a library linear solve, a quadratic saddle with an analytic minimum mode,
the closed-form ferromagnet energy."""
import numpy as np

from oracle import lbfgs_oracle as lo
from oracle import spin_oracle as so
from paper_2509_26269_b200 import workloads as wl


def _flat(f, grad):
    return f, grad, (lambda x: x), (lambda x, d: d)


def _dense_bfgs_inverse(S, Y):
    """H after applying H+ = (I - rho s y^T) H (I - rho y s^T) + rho s s^T pair by pair (oldest first) to gamma I,
    gamma = s.y / y.y of the NEWEST pair -- the definition the two-loop recursion is an O(mn) evaluation of."""
    n = S[0].size
    gamma = float(S[-1] @ Y[-1]) / float(Y[-1] @ Y[-1])
    H = gamma * np.eye(n)
    for s, y in zip(S, Y):
        rho = 1.0 / float(s @ y)
        A = np.eye(n) - rho * np.outer(s, y)
        H = A @ H @ A.T + rho * np.outer(s, s)
    return H


def test_two_loop_is_the_dense_bfgs_inverse():
    rng = np.random.default_rng(3)
    n = 12
    Q = rng.standard_normal((n, n)); A = Q @ Q.T + np.eye(n)          # pairs of an SPD quadratic: s.y = s^T A s > 0
    for m in (1, 2, 5, 8):
        S = [rng.standard_normal(n) for _ in range(m)]
        Y = [A @ s for s in S]
        H = _dense_bfgs_inverse(S, Y)
        q = rng.standard_normal(n)
        r = lo.two_loop(q, S, Y, 123.0)
        assert np.max(np.abs(r - H @ q)) <= 1e-12 * np.max(np.abs(H @ q))
        assert np.max(np.abs(lo.two_loop(Y[-1], S, Y, 1.0) - S[-1])) <= 1e-12 * np.max(np.abs(S[-1]))   # secant equation
        assert np.max(np.abs(H - H.T)) <= 1e-12 and np.linalg.eigvalsh(H).min() > 0.0
    q = rng.standard_normal(n)
    assert np.array_equal(lo.two_loop(q, [], [], 0.25), 0.25 * q)      # no history: H = gamma0 I


def test_one_dimensional_sequence_by_hand():
    # f = x^2/2, x0 = 1, alpha0 = 1/4 (every number below is an exact binary fraction).
    # step 1: no history, d = -1, a = 1/4: x = 3/4; g_t.d = -3/4 <= 1/2, E 9/32 <= 1/2 - 1e-4/4: accepted at the first trial,
    #         alpha <- 1/2; pair s = -1/4, y = -1/4 (s.y > 0, stored), gamma = 1 = the exact inverse Hessian.
    # step 2: d = -H g = -3/4, a = 1 (quasi-Newton step): x = 0, g = 0: converged; its pair s = y = -3/4 is stored as well.
    #         evals = 1 + 1 + 1, pairs = 2.
    trace = []
    x, info = lo.relax_downhill_lbfgs(*_flat(lambda x: float(0.5 * x @ x), lambda x: x.copy()), np.array([1.0]), 10, 1e-14, 0.25,
                                      trace=trace)
    assert info["converged"] and info["steps"] == 2 and info["evals"] == 3 and info["alpha"] == 0.5 and info["pairs"] == 2
    assert x[0] == 0.0
    assert trace == [(0.28125, 0.75, 0.25, 0), (0.0, 0.0, 1.0, 1)]
    # a first trial that overshoots: alpha0 = 3: x_t = -2, g_t.d = 2 > 1/2: rejected; a = 3/2: x_t = -1/2, g_t.d = 1/2 <= 1/2,
    # E 1/8 <= 1/2 - 1.5e-4: accepted at the SECOND trial, so alpha stays 3/2; pair s = -3/2, y = -3/2; step 2 lands on 0.
    trace = []
    x, info = lo.relax_downhill_lbfgs(*_flat(lambda x: float(0.5 * x @ x), lambda x: x.copy()), np.array([1.0]), 10, 1e-14, 3.0,
                                      trace=trace)
    assert info["steps"] == 2 and info["evals"] == 4 and info["alpha"] == 1.5 and x[0] == 0.0
    assert trace == [(0.125, 0.5, 1.5, 0), (0.0, 0.0, 1.0, 1)]


def test_quadratic_minimiser_is_linear_solve_and_negative_curvature_pairs_are_skipped():
    rng = np.random.default_rng(0)
    n = 30
    Q = rng.standard_normal((n, n)); A = Q @ Q.T + 0.5 * np.eye(n)
    b = rng.standard_normal(n)
    ops = _flat(lambda x: float(0.5 * x @ A @ x - b @ x), lambda x: A @ x - b)
    trace = []
    x, info = lo.relax_downhill_lbfgs(*ops, np.zeros(n), 500, 1e-10, 0.1, trace=trace)
    assert info["converged"] and np.max(np.abs(x - np.linalg.solve(A, b))) < 1e-9
    E = np.array([t[0] for t in trace])
    assert np.all(np.diff(E) <= 1e-10 * np.abs(E[:-1]))
    assert max(t[3] for t in trace) == lo.M_DEFAULT                    # the history fills up and is capped
    # a pair with s.y <= 0 must not be stored: concave direction of x^4/4 - x^2/2 between its inflection points
    S, Y = [], []
    assert not lo._push(S, Y, np.array([0.1]), np.array([-0.05]), 8) and S == []
    assert lo._push(S, Y, np.array([0.1]), np.array([0.05]), 8) and len(S) == 1


def test_ferromagnet_closed_form_energy_lbfgs():
    w = wl.config0()
    mdl = so.SpinModel(w.Lx, w.Ly, w.pbc_x, w.pbc_y, w.J, w.D, w.K, w.B, w.mu)
    from oracle import relax_oracle as ro
    m, info = lo.relax_downhill_lbfgs(*ro.spin_ops(mdl), w.spins, 500, 1e-10, 0.05)
    assert info["converged"]
    assert np.max(np.abs(np.linalg.norm(m, axis=1) - 1.0)) < 1e-14
    assert abs(info["energy"] - (-w.N * (6 * w.J + w.K + w.mu * w.B[2]))) < 1e-10
    _, icg = ro.relax_downhill(*ro.spin_ops(mdl), w.spins, 2000, 1e-10, 0.05)
    assert info["evals"] <= icg["evals"]                               # not a pin: the point of having it


# ---- outer climb on a quadratic saddle with an analytic minimum mode: f = x^T A x / 2, A = diag(-1, 2, 3), v_1 = e_1,
# lambda = (-1, 2): F = -A x, F_mmf = F - 2 (F.e_1) e_1 = -|A| x, the gradient flow of the SPD quadratic x^T |A| x / 2 whose
# stationary point is the saddle x = 0
A_SADDLE = np.diag([-1.0, 2.0, 3.0])
ABS_A = np.diag([1.0, 2.0, 3.0])


def _saddle_ops(v=np.array([1.0, 0.0, 0.0])):
    minmode = lambda x: (np.array([-1.0, 2.0]), np.stack([v, np.array([0.0, 1.0, 0.0])]))
    return minmode, (lambda x: -A_SADDLE @ x), (lambda x: x), (lambda x, d: d)


def test_mmf_lbfgs_first_steps_closed_form_and_cap():
    x0 = np.array([0.5, -0.25, 0.125])
    # step 1: no history, p = alpha0 F_mmf = -alpha0 |A| x0
    x1, lam, steps, conv, fn, evals = lo.mmf_run_lbfgs(*_saddle_ops(), x0, 0.125, 10.0, 1, 0.0)
    assert steps == 1 and evals == 2 and not conv
    assert np.array_equal(x1, x0 - 0.125 * (ABS_A @ x0))
    # step 2: one pair s = x1 - x0, y = |A| s; p = H F(x1) with the dense BFGS inverse of that pair
    x2, *_ = lo.mmf_run_lbfgs(*_saddle_ops(), x0, 0.125, 10.0, 2, 0.0)
    s = x1 - x0; y = ABS_A @ s
    H = _dense_bfgs_inverse([s], [y])
    assert np.max(np.abs(x2 - (x1 + H @ (-ABS_A @ x1)))) <= 1e-15
    # cap: a step longer than smax is rescaled to length smax exactly, direction kept
    xc, *_ = lo.mmf_run_lbfgs(*_saddle_ops(), x0, 0.125, 0.01, 1, 0.0)
    p = xc - x0
    assert abs(np.linalg.norm(p) - 0.01) <= 1e-17
    assert np.max(np.abs(p / np.linalg.norm(p) + (ABS_A @ x0) / np.linalg.norm(ABS_A @ x0))) <= 1e-15
    # end point: the saddle, index test from the analytic eigenvalues, in few MinMode solves
    xs, lam, steps, conv, fn, evals = lo.mmf_run_lbfgs(*_saddle_ops(), x0, 0.125, 10.0, 100, 1e-12)
    assert conv and fn <= 1e-12 and np.max(np.abs(xs)) <= 1e-12 and evals == steps + 1 and steps <= 12


def test_mmf_lbfgs_drops_history_when_the_step_opposes_the_force():
    # a WRONG minimum mode (e_2 instead of e_1) makes the reflected force that of diag(-1, -2, 3): pairs along the first two
    # axes have s.y < 0 and are never stored, so every step is alpha0 F (history empty) and the iteration runs away from 0
    # along them at the rate (1 + alpha0 |lambda|) per step -- closed form
    x0 = np.array([0.5, -0.25, 0.0])
    x, lam, steps, conv, fn, evals = lo.mmf_run_lbfgs(*_saddle_ops(v=np.array([0.0, 1.0, 0.0])), x0, 0.125, 100.0, 3, 0.0)
    assert np.max(np.abs(x - x0 * np.array([1.125 ** 3, 1.25 ** 3, 1.0]))) <= 1e-15
