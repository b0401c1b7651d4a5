"""Pins for oracle/relax_oracle.py (no GPU): the relax-downhill loop and the two-sided descent (Alg. 1 l.15-18,
PAPER.md:271-276) against things that are not the loop itself: a library linear solve, the closed-form ferromagnet
energy, Morse equilibrium bond lengths, and the two minima of a double well."""
import numpy as np

from oracle import cart_oracle as co
from oracle import relax_oracle as ro
from oracle import spin_oracle as so
from paper_2509_26269_b200 import workloads as wl


def _flat_ops(f, grad):
    return f, grad, (lambda x: x), (lambda x, d: d)


def test_quadratic_minimiser_is_linear_solve():
    # flat space, SPD quadratic: the minimiser is A^{-1} b (numpy.linalg.solve), whatever the line search does
    rng = np.random.default_rng(0)
    n = 30
    Q = rng.standard_normal((n, n))
    A = Q @ Q.T + 0.5 * np.eye(n)
    b = rng.standard_normal(n)
    ops = _flat_ops(lambda x: float(0.5 * x @ A @ x - b @ x), lambda x: A @ x - b)
    trace = []
    x, info = ro.relax_downhill(*ops, np.zeros(n), 5000, 1e-10, 0.1, trace=trace)
    assert info["converged"] and info["gnorm"] <= 1e-10
    assert np.max(np.abs(x - np.linalg.solve(A, b))) < 1e-9
    E = np.array([t[0] for t in trace])
    assert np.all(np.diff(E) <= ro.EPS_E * np.abs(E[:-1]))          # monotone down to the rounding allowance
    assert info["steps"] == len(trace) and info["evals"] >= info["steps"] + 1


def test_max_steps_and_already_converged():
    ops = _flat_ops(lambda x: float(0.5 * x @ x), lambda x: x.copy())
    x, info = ro.relax_downhill(*ops, np.ones(4), 0, 1e-12, 0.1)
    assert info["steps"] == 0 and not info["converged"] and np.all(x == 1.0)
    x, info = ro.relax_downhill(*ops, np.zeros(4), 10, 1e-12, 0.1)
    assert info["steps"] == 0 and info["converged"] and info["evals"] == 1
    # alpha0 far too large: the backtracking must still find a step (exact minimiser of x^2/2 is a = 1)
    x, info = ro.relax_downhill(*ops, np.ones(4), 200, 1e-12, 1e6)
    assert info["converged"] and np.max(np.abs(x)) < 1e-12


def test_ferromagnet_closed_form_energy():
    # perturbed +z ferromagnet (cfg 0) relaxes to m = +z: E = -N (6J + K + mu B) with the ordered-pair sum of Eq. 4 (A1);
    # the DMI term vanishes for a uniform state
    w = wl.config0()
    mdl = so.SpinModel(w.Lx, w.Ly, w.pbc_x, w.pbc_y, w.J, w.D, w.K, w.B, w.mu)
    m, info = ro.relax_downhill(*ro.spin_ops(mdl), w.spins, 2000, 1e-10, 0.05)
    assert info["converged"]
    assert np.max(np.abs(np.linalg.norm(m, axis=1) - 1.0)) < 1e-14
    assert np.max(np.abs(m - np.array([0.0, 0.0, 1.0]))) < 1e-9
    assert abs(info["energy"] - (-w.N * (6 * w.J + w.K + w.mu * w.B[2]))) < 1e-10


def test_morse_trimer_bond_lengths():
    # three free atoms, all pair distances inside the cut-off: the minimum is the equilateral triangle with edge r0,
    # E = 3 (-De - phi(rc))
    mdl = co.MorseModel(np.eye(2) * 60, 0.4205, 1.4199, 2.78, 6.0)
    x0 = np.array([[20.0, 20.0, 20.0], [23.1, 20.2, 19.9], [21.3, 22.9, 20.3]])
    x, info = ro.relax_downhill(*ro.cart_ops(mdl), x0, 5000, 1e-10, 0.1)
    assert info["converged"]
    r = [np.linalg.norm(x[i] - x[j]) for i, j in ((0, 1), (0, 2), (1, 2))]
    assert np.max(np.abs(np.array(r) - 2.78)) < 1e-8
    assert abs(info["energy"] - 3 * (-0.4205 - mdl.phi(6.0))) < 1e-12


def test_fixed_atoms_do_not_move():
    w = wl.small_cluster(9, seed=3)
    fixed = np.zeros(9, dtype=bool)
    fixed[:3] = True
    mdl = co.MorseModel(w.cell, w.De, w.alpha, w.r0, w.rc, fixed)
    x, info = ro.relax_downhill(*ro.cart_ops(mdl), w.positions, 300, 1e-7, 0.1)
    assert np.all(x[:3] == w.positions[:3])
    assert info["energy"] < co.energy(mdl, w.positions)


def test_two_sided_descent_double_well():
    # f = (x^2 - 1)^2 + y^2: index-1 saddle at the origin, v_min = e_x, the two branches end in (+1, 0) and (-1, 0)
    f = lambda p: float((p[0] ** 2 - 1.0) ** 2 + p[1] ** 2)
    g = lambda p: np.array([4.0 * p[0] * (p[0] ** 2 - 1.0), 2.0 * p[1]])
    res = ro.two_sided_descent(*_flat_ops(f, g), np.zeros(2), np.array([1.0, 0.0]), 0.05, 2000, 1e-11, 0.1)
    (xp, ip), (xm, im) = res
    assert ip["converged"] and im["converged"]
    assert np.max(np.abs(xp - [1.0, 0.0])) < 1e-10 and np.max(np.abs(xm - [-1.0, 0.0])) < 1e-10


def test_two_sided_descent_spin_seeds_on_manifold():
    # spins: the seeds are retracted (unit length) and both branches end at stationary points below the start energy
    w = wl.config1(L=12)
    mdl = so.SpinModel(w.Lx, w.Ly, w.pbc_x, w.pbc_y, w.J, w.D, w.K, w.B, w.mu)
    lam, V = so.lowest_modes(mdl, w.spins, 1)
    E0 = so.energy(mdl, w.spins)
    res = ro.two_sided_descent(*ro.spin_ops(mdl), w.spins, V[0], 0.1, 3000, 1e-6, 0.05)   # (a 1e-7 translation mode of the skyrmion limits what is reachable)
    for x, info in res:
        assert info["converged"] and info["energy"] < E0
        assert np.max(np.abs(np.linalg.norm(x, axis=1) - 1.0)) < 1e-14
        assert np.linalg.norm(so.projected_gradient(mdl, x)) <= 1e-6


def test_certified_edge_skyrmion_collapse():
    # Alg. 1 l.9-18 end to end on the oracle side: minimum-mode following from a small skyrmion climbs to the collapse saddle
    # (lambda_1 < 0 < lambda_2, |F_mmf| <= tau_F), the two-sided descent from it ends in two different minima, one of which
    # is the ferromagnet with the closed-form energy -N (6J + K + mu B).  12 x 12 periodic, configs[0] parameters.
    w = wl.config1(L=12, R=2.0, sigma=0.0)
    mdl = so.SpinModel(w.Lx, w.Ly, w.pbc_x, w.pbc_y, w.J, w.D, w.K, w.B, w.mu)
    m, lam, steps, conv, fn = so.mmf_run(mdl, w.spins, 2, 0.1, 4000, 1e-4)
    assert conv and fn <= 1e-4 and lam[0] < 0.0 < lam[1]
    E_saddle = so.energy(mdl, m)
    lam2, V = so.lowest_modes(mdl, m, 2)
    res = ro.two_sided_descent(*ro.spin_ops(mdl), m, V[0], 0.1, 6000, 1e-6, 0.05)
    E = sorted(info["energy"] for _, info in res)
    assert all(info["converged"] for _, info in res)
    E_fm = -w.N * (6 * w.J + w.K + w.mu * w.B[2])
    assert abs(E[0] - E_fm) < 1e-9                       # one branch: the ferromagnet (closed form)
    assert E[1] < E_saddle - 1.0 and E[1] > E_fm + 1.0   # the other: a distinct minimum below the saddle (the skyrmion)
    fm = min(res, key=lambda r: r[1]["energy"])[0]
    assert np.max(np.abs(fm - np.array([0.0, 0.0, 1.0]))) < 1e-5


def test_cg_mmf_double_well_and_same_saddle_as_fixed_step():
    # oracle/mmf_cg_oracle.py (outer loop with the CG step rule, reading A28).  (i) 2-D double well with the analytic Hessian as
    # MinMode: from (0.4, 0.3) the loop must reach the index-1 saddle at the origin.  (ii) on the 12 x 12 lattice it must reach the
    # saddle the fixed-step loop reaches (same energy and curvatures), in an order of magnitude fewer MinMode solves.
    from oracle import mmf_cg_oracle as mc

    def minmode(p):
        lam, U = np.linalg.eigh(np.array([[12.0 * p[0] ** 2 - 4.0, 0.0], [0.0, 2.0]]))
        return lam, U.T
    force = lambda p: -np.array([4.0 * p[0] * (p[0] ** 2 - 1.0), 2.0 * p[1]])
    x, lam, steps, conv, fn, evals = mc.mmf_run_cg(minmode, force, lambda x: x, lambda x, d: d, np.array([0.4, 0.3]), 0.01, 0.2, 100, 1e-10)
    assert conv and steps < 20 and evals == 2 * steps + 1
    assert np.max(np.abs(x)) < 1e-10 and abs(lam[0] + 4.0) < 1e-9 and abs(lam[1] - 2.0) < 1e-12
    w = wl.config1(L=12, R=2.0, sigma=0.0)
    mdl = so.SpinModel(w.Lx, w.Ly, w.pbc_x, w.pbc_y, w.J, w.D, w.K, w.B, w.mu)
    _, _, retract, transport = ro.spin_ops(mdl)
    x, lam, steps, conv, fn, evals = mc.mmf_run_cg(lambda m: so.lowest_modes(mdl, m, 2), lambda m: -so.projected_gradient(mdl, m), retract,
                                                   transport, w.spins, 0.05, 1.0, 400, 1e-4)
    assert conv and fn <= 1e-4 and steps < 200
    m_fix, lam_fix, steps_fix, conv_fix, _ = so.mmf_run(mdl, w.spins, 2, 0.1, 4000, 1e-4)
    assert conv_fix and evals < steps_fix / 5
    assert abs(so.energy(mdl, x) - so.energy(mdl, m_fix)) < 1e-6
    assert np.max(np.abs(lam - lam_fix) / np.abs(lam_fix)) < 1e-3
    assert np.max(np.abs(x - m_fix)) < 1e-2


# ---------------------------------------------------------------------------------------------------------------------
# Step-level pins of the two conjugate-gradient loops (readings A26, A28).  End-point pins alone cannot see a wrong beta, a
# wrong sign in the restart test, a wrong step-doubling rule or a wrong secant clip (all still converge); these do.
def test_relax_one_dimensional_sequence_by_hand():
    # f = x^2/2 from x0 = 1 with alpha0 = 3; every number is an exact binary fraction, derived by hand from the rule of A26:
    # step 1  g = 1, d = -1, slope = -1.  a = 3: x_t = -2, g_t.d = 2 > 1/2 |slope|: REJECTED (overshoot).  a = 3/2: x_t = -1/2,
    #         g_t.d = 1/2 <= 1/2, E_t = 1/8 <= 1/2 - 1.5e-4: accepted at the SECOND trial -> alpha stays 3/2.  evals = 3.
    #         beta = (1/4 + 1/2)/1 = 3/4; new slope = -1/4 + 3/4 * 1/2 = +1/8 >= 0 -> restart: beta = 0, d = +1/2, slope = -1/4.
    # step 2  a = 3/2: x_t = 1/4, g_t.d = 1/8 <= 1/8, E_t = 1/32 <= 1/8 - 3.75e-5: accepted at the FIRST trial -> alpha = 3.  evals = 4.
    #         beta = (1/16 + 1/8)/(1/4) = 3/4; new slope = -1/16 + 3/4 * 1/8 = +1/32 >= 0 -> restart: d = -1/4, slope = -1/16.
    # step 3  a = 3: x_t = -1/2, g_t.d = 1/8 > 1/32: rejected.  a = 3/2: x_t = -1/8, g_t.d = 1/32 <= 1/32, E_t = 1/128: accepted at
    #         the second trial -> alpha = 3/2.  evals = 6.
    ops = _flat_ops(lambda x: float(0.5 * x @ x), lambda x: x.copy())
    want_x = [-0.5, 0.25, -0.125]
    want_alpha = [1.5, 3.0, 1.5]
    want_evals = [3, 4, 6]
    for n in (1, 2, 3):
        trace = []
        x, info = ro.relax_downhill(*ops, np.array([1.0]), n, 0.0, 3.0, trace=trace)
        assert x[0] == want_x[n - 1] and info["alpha"] == want_alpha[n - 1] and info["evals"] == want_evals[n - 1]
        assert info["steps"] == n and info["energy"] == 0.5 * want_x[n - 1] ** 2 and info["gnorm"] == abs(want_x[n - 1])
    assert trace == [(0.125, 0.5, 1.5), (0.03125, 0.25, 1.5), (0.0078125, 0.125, 1.5)]


def test_relax_direction_update_is_linear_cg_after_an_exact_step():
    # On an SPD quadratic with an EXACT first step (alpha0 = g.g / g^T A g, accepted at the first trial: g_1.d_0 = 0) the new
    # gradient is orthogonal to the old one, so PR+ beta = g_1.g_1 / g_0.g_0 = the beta of LINEAR conjugate gradients and
    # d_1 = -g_1 + beta_1 d_0 is the CG direction.  x_1 and the direction of x_2 - x_1 are pinned against the textbook
    # recurrence written out below (numpy only); the second step's length is one of 2 alpha0 / 2^j.
    rng = np.random.default_rng(5)
    n = 9
    Q = rng.standard_normal((n, n)); A = Q @ Q.T + np.eye(n)
    b = rng.standard_normal(n)
    x0 = rng.standard_normal(n)
    ops = _flat_ops(lambda x: float(0.5 * x @ A @ x - b @ x), lambda x: A @ x - b)
    r0 = b - A @ x0                                  # linear CG (Hestenes-Stiefel), two steps
    p0 = r0
    a0 = (r0 @ r0) / (p0 @ A @ p0)
    x1_cg = x0 + a0 * p0
    r1 = r0 - a0 * (A @ p0)
    beta1 = (r1 @ r1) / (r0 @ r0)
    p1 = r1 + beta1 * p0
    x1, i1 = ro.relax_downhill(*ops, x0, 1, 0.0, a0)
    assert i1["evals"] == 2 and i1["alpha"] == 2.0 * a0                   # first trial accepted -> doubled
    assert np.max(np.abs(x1 - x1_cg)) <= 1e-14 * np.max(np.abs(x1_cg))
    trace = []
    x2, i2 = ro.relax_downhill(*ops, x0, 2, 0.0, a0, trace=trace)
    step = x2 - x1
    a1 = trace[1][2]
    assert any(a1 == 2.0 * a0 / 2 ** j for j in range(8))
    assert np.max(np.abs(step / a1 - p1)) <= 1e-12 * np.max(np.abs(p1))    # beta and the sign of every term of d_1
    # and with exact steps throughout (a 2-D quadratic where 2 alpha0 happens to be exact is not needed: restart the loop from
    # x_1 with the exact CG step length instead) the iterates are those of linear CG
    a1_cg = (r1 @ r1) / (p1 @ A @ p1)
    assert ops[0](x1 + a1_cg * p1) <= ops[0](x2) + 1e-15                  # the exact CG step is at least as good as the accepted one


def test_mmf_cg_secant_step_closed_form_clip_and_negative_curvature():
    # Quadratic saddle f = x^T A x / 2, A = diag(-1, 2, 3), analytic MinMode v_1 = e_1: F_mmf = -|A| x is LINEAR, so the secant
    # estimate C = (f0 - f1)/delta equals dh^T |A| dh whatever delta is and s = f0 / C is the exact zero of the force along dh:
    # x_1 = x_0 + [(F.dh)/(dh^T |A| dh)] dh with dh = F/|F| -- the first step of linear CG on |A|.  Three such steps reach the
    # saddle (3-D).  With smax below that length the step is exactly smax dh.  With a wrong mode (e_2) the effective Hessian
    # along dh = e_1 is negative, C < 0, and the step is +smax along dh.
    from oracle import mmf_cg_oracle as mo
    A = np.diag([-1.0, 2.0, 3.0]); absA = np.diag([1.0, 2.0, 3.0])
    mm = lambda x: (np.array([-1.0, 2.0]), np.stack([np.array([1.0, 0.0, 0.0]), np.array([0.0, 1.0, 0.0])]))
    force = lambda x: -A @ x
    flat = ((lambda x: x), (lambda x, d: d))
    x0 = np.array([0.5, -0.25, 0.125])
    F0 = -absA @ x0
    dh = F0 / np.linalg.norm(F0)
    s_exact = (F0 @ dh) / (dh @ absA @ dh)
    for delta in (1e-3, 0.05):
        trace = []
        x1, lam, steps, conv, fn, evals = mo.mmf_run_cg(mm, force, *flat, x0, delta, 10.0, 1, 0.0, trace=trace)
        assert steps == 1 and evals == 3
        assert abs(trace[0][1] - s_exact) <= 1e-10 * s_exact
        assert np.max(np.abs(x1 - (x0 + s_exact * dh))) <= 1e-10
    r1 = -absA @ (x0 + s_exact * dh)                                        # linear CG beta on |A| (gradient of the next point)
    assert abs(trace[0][2] - (r1 @ r1) / (F0 @ F0)) <= 1e-9                 # PR+ = FR after an exact step (F_1 . F_0 = 0)
    x3, lam, steps, conv, fn, evals = mo.mmf_run_cg(mm, force, *flat, x0, 1e-3, 10.0, 3, 0.0)
    assert np.max(np.abs(x3)) <= 1e-9                                       # n = 3: CG is exact after three steps
    xc, *_ = mo.mmf_run_cg(mm, force, *flat, x0, 1e-3, 0.01, 1, 0.0)
    assert np.max(np.abs(xc - (x0 + 0.01 * dh))) <= 1e-16                   # clipped to smax
    mm_wrong = lambda x: (np.array([-1.0, 2.0]), np.stack([np.array([0.0, 1.0, 0.0]), np.array([1.0, 0.0, 0.0])]))
    xe = np.array([0.5, 0.0, 0.0])                                          # F = (0.5, 0, 0): dh = e_1, effective curvature -1
    trace = []
    xn, *_ = mo.mmf_run_cg(mm_wrong, force, *flat, xe, 1e-3, 0.02, 1, 0.0, trace=trace)
    assert trace[0][1] == 0.02 and np.max(np.abs(xn - np.array([0.52, 0.0, 0.0]))) <= 1e-16
