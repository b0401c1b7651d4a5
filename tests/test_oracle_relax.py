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
