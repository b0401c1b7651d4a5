"""Pins for oracle/spin_oracle.py against things it does not itself define (no GPU).

Each test is chosen so that a plausible mistake in the oracle (dropped term, wrong sign/index,
transposed block, missing factor 2) fails at least one of them.
"""
import numpy as np
import pytest
import scipy.linalg

from oracle import spin_oracle as so
from paper_2509_26269_b200 import workloads as wl


def magnon_dispersion(L, J, K, muB):
    """Closed-form spin-wave energies of the +z ferromagnet on the periodic LxL triangular lattice
    (textbook linear spin-wave theory; BASELINE.json north_star pin (a); with Eq. 4's ordered-pair
    counting the bond coupling is 2J):  lam(q) = 2 * 2J * sum_{3 bond dirs} (1 - cos q.delta) + 2K + mu B."""
    n = np.arange(L)
    q1, q2 = np.meshgrid(2 * np.pi * n / L, 2 * np.pi * n / L, indexing="ij")
    lam = 4.0 * J * (3.0 - np.cos(q1) - np.cos(q2) - np.cos(q2 - q1)) + 2.0 * K + muB
    return np.sort(np.repeat(lam.ravel(), 2))


def model_of(w):
    return so.SpinModel(w.Lx, w.Ly, w.pbc_x, w.pbc_y, w.J, w.D, w.K, w.B, w.mu)


def rand_model(L=6, pbc=(1, 1), seed=0, **kw):
    p = dict(J=1.0, D=0.3, K=0.05, B=(0.01, -0.02, 0.03), mu=1.0)
    p.update(kw)
    return so.SpinModel(L, L + 2, pbc[0], pbc[1], **p), wl.random_spins(L, L + 2, seed)


def test_energy_loops_equals_vectorised():
    for pbc in [(1, 1), (0, 0), (1, 0)]:
        model, m = rand_model(pbc=pbc, seed=3)
        assert abs(so.energy_loops(model, m) - so.energy(model, m)) < 1e-12


def test_ferromagnet_energy_closed_form():
    # all spins +z on periodic LxL: E = -N*6*J - N*mu*Bz - N*K (six ordered neighbours per site; DMI vanishes)
    L = 6
    model = so.SpinModel(L, L, 1, 1, 1.3, 0.4, 0.07, (0, 0, 0.05))
    m = np.zeros((L * L, 3)); m[:, 2] = 1
    assert abs(so.energy_loops(model, m) - (-L * L * (6 * 1.3 + 0.05 + 0.07))) < 1e-11


def test_two_site_dmi_sign():
    # 2x1 open lattice: one bond along +x. E = -2J m0.m1 - 2 D (z x x).(m0 x m1) = ... - 2 D y.(m0 x m1)
    model = so.SpinModel(2, 1, 0, 0, 0.0, 0.5, 0.0, (0, 0, 0))
    m0 = np.array([0.0, 0.0, 1.0]); m1 = np.array([1.0, 0.0, 0.0])
    # y . (z x x) = y . y = 1  -> E = -2*0.5*1 = -1
    assert abs(so.energy_loops(model, np.stack([m0, m1])) - (-1.0)) < 1e-14
    # swapped spins flip the sign of the DMI energy (chirality)
    assert abs(so.energy_loops(model, np.stack([m1, m0])) - (+1.0)) < 1e-14


def test_open_boundary_bond_count():
    model = so.SpinModel(5, 4, 0, 0, 1, 0, 0, (0, 0, 0))
    I, J, R = model.bonds()
    # undirected bonds on an open rhombic Lx x Ly triangular patch: (Lx-1)Ly + Lx(Ly-1) + (Lx-1)(Ly-1)
    assert I.size == 2 * (4 * 4 + 5 * 3 + 4 * 3)
    assert np.allclose(np.linalg.norm(R, axis=1), 1.0)
    model = so.SpinModel(5, 4, 1, 1, 1, 0, 0, (0, 0, 0))
    assert model.bonds()[0].size == 6 * 20


def test_bond_vectors_match_geometry():
    # rhat_ij must equal r_j - r_i for interior sites (positions from the workload generator)
    Lx, Ly = 6, 5
    pos = wl.site_positions(Lx, Ly)
    model = so.SpinModel(Lx, Ly, 0, 0, 1, 0.3, 0, (0, 0, 0))
    I, J, R = model.bonds()
    assert np.allclose(pos[J] - pos[I], R[:, :2], atol=1e-14)
    assert np.all(R[:, 2] == 0)


@pytest.mark.parametrize("pbc", [(1, 1), (0, 0), (0, 1)])
def test_gradient_vs_central_fd_of_literal_energy(pbc):
    # E is quadratic + linear in m => central differences are exact up to rounding for any eps
    model, m = rand_model(pbc=pbc, seed=5)
    g = so.gradient(model, m)
    rng = np.random.default_rng(0)
    for _ in range(4):
        d = rng.standard_normal(m.shape)
        eps = 0.37
        fd = (so.energy_loops(model, m + eps * d) - so.energy_loops(model, m - eps * d)) / (2 * eps)
        assert abs(fd - np.sum(g * d)) < 1e-10 * max(1.0, abs(fd))


def test_energy_quadratic_form():
    # E = 1/2 m^T H m - mu B . sum m   with H the bond-assembled Euclidean Hessian
    model, m = rand_model(pbc=(1, 0), seed=7)
    H = so.euclid_hessian(model)
    mf = m.ravel()
    E = 0.5 * mf @ (H @ mf) - model.mu * np.sum(m @ model.B)
    assert abs(E - so.energy_loops(model, m)) < 1e-11


def test_euclid_hessian_is_gradient_jacobian_and_symmetric():
    model, m = rand_model(pbc=(1, 1), seed=9)
    H = so.euclid_hessian(model).toarray()
    assert np.max(np.abs(H - H.T)) < 1e-15
    d = np.random.default_rng(1).standard_normal(m.shape)
    jv = so.gradient(model, m + d) - so.gradient(model, m)  # gradient is affine in m
    assert np.allclose(H @ d.ravel(), jv.ravel(), atol=1e-12)


def test_graph_laplacian_special_case():
    # D = K = B = 0: H = -2J * adjacency of the triangular lattice graph
    model = so.SpinModel(5, 6, 1, 1, 0.7, 0.0, 0.0, (0, 0, 0))
    H = so.euclid_hessian(model).toarray()
    N = 30
    A = np.zeros((N, N))
    for iy in range(6):
        for ix in range(5):
            for dx, dy in [(1, 0), (-1, 0), (0, 1), (0, -1), (-1, 1), (1, -1)]:
                A[iy * 5 + ix, ((iy + dy) % 6) * 5 + (ix + dx) % 5] += 1
    assert np.allclose(H, np.kron(-2 * 0.7 * A, np.eye(3)))


def test_magnon_dispersion_full_spectrum():
    # BASELINE.json north_star pin (a): uniform +z ferromagnet => tangent-Hessian spectrum = spin-wave energies
    L, J, D, K, Bz = 8, 1.0, 0.3, 0.05, 0.02
    model = so.SpinModel(L, L, 1, 1, J, D, K, (0, 0, Bz))
    m = np.zeros((L * L, 3)); m[:, 2] = 1
    Ht, _ = so.tangent_hessian(model, m)
    lam = np.linalg.eigvalsh(Ht)
    ref = magnon_dispersion(L, J, K, Bz)
    assert np.max(np.abs(lam - ref)) < 1e-12
    assert abs(lam[0] - (2 * K + Bz)) < 1e-13  # = 0.12
    # non-square lattice and other couplings
    model = so.SpinModel(6, 6, 1, 1, 0.8, 0.0, 0.1, (0, 0, 0.3))
    m = np.zeros((36, 3)); m[:, 2] = 1
    lam = np.linalg.eigvalsh(so.tangent_hessian(model, m)[0])
    assert np.max(np.abs(lam - magnon_dispersion(6, 0.8, 0.1, 0.3))) < 1e-12


@pytest.mark.parametrize("pbc", [(1, 1), (0, 0)])
def test_tangent_hessian_symmetry_and_basis(pbc):
    model, m = rand_model(pbc=pbc, seed=11)
    Ht, Bm = so.tangent_hessian(model, m)
    assert np.max(np.abs(Ht - Ht.T)) < 1e-14 * np.max(np.abs(Ht))
    BtB = (Bm.T @ Bm).toarray()
    assert np.allclose(BtB, np.eye(2 * model.N), atol=1e-14)
    assert np.allclose(Bm.T @ m.ravel(), 0, atol=1e-14)


def _retract(m, v, eps):
    x = m + eps * v
    return x / np.linalg.norm(x, axis=1, keepdims=True)


def test_riemannian_hvp_vs_fd_of_projected_gradient():
    # pins O7/O9: P * d/de [P g](R_m(e v)) = Hess[v] on tangent v, along the retraction
    model, m = rand_model(pbc=(1, 1), seed=13)
    rng = np.random.default_rng(2)
    v = rng.standard_normal(m.shape)
    v -= np.sum(v * m, 1, keepdims=True) * m
    eps = 1e-5
    gp = so.projected_gradient(model, _retract(m, v, eps))
    gm = so.projected_gradient(model, _retract(m, v, -eps))
    fd = (gp - gm) / (2 * eps)
    fd -= np.sum(fd * m, 1, keepdims=True) * m
    hv = so.hvp(model, m, v[None])[0]
    assert np.max(np.abs(fd - hv)) < 2e-8
    assert np.max(np.abs(np.sum(hv * m, 1))) < 1e-13  # output is tangent


def test_hvp_projects_input():
    model, m = rand_model(pbc=(0, 0), seed=15)
    V = wl.random_block(model.N, 2, 4)
    Vt = V - np.sum(V * m[None], 2, keepdims=True) * m[None]
    assert np.allclose(so.hvp(model, m, V), so.hvp(model, m, Vt), atol=1e-13)


def test_rotation_identity_pins_curvature_term():
    # D = 0, B || z, anisotropy along z: E invariant under rotation about z.  Differentiating
    # grad_R E(R_t m) = R_t grad_R E(m) at t=0 gives Hess[z x m] = P(z x P g) at ANY m (not only
    # stationary points) -- fails if the -(m.g) v term is dropped or has the wrong sign.
    model, m = rand_model(pbc=(1, 1), seed=17, D=0.0, B=(0, 0, 0.04))
    z = np.array([0.0, 0.0, 1.0])
    v = np.cross(np.broadcast_to(z, m.shape), m)
    Pg = so.projected_gradient(model, m)
    rhs = np.cross(np.broadcast_to(z, m.shape), Pg)
    rhs -= np.sum(rhs * m, 1, keepdims=True) * m
    lhs = so.hvp(model, m, v[None])[0]
    assert np.max(np.abs(lhs - rhs)) < 1e-13


def test_single_spin_closed_forms():
    # one spin in a field, at the minimum m = B/|B|: both tangent eigenvalues = mu |B|
    model = so.SpinModel(1, 1, 0, 0, 1.0, 0.3, 0.0, (0.3, -0.4, 1.2), mu=1.5)
    Bn = np.linalg.norm(model.B)
    m = (model.B / Bn)[None, :]
    lam = np.linalg.eigvalsh(so.tangent_hessian(model, m)[0])
    assert np.allclose(lam, 1.5 * Bn, atol=1e-13)
    # anisotropy only, m = z: both = 2K; m in-plane (maximum of -K mz^2): eigenvalues {0, -2K}
    model = so.SpinModel(1, 1, 0, 0, 1.0, 0.0, 0.2, (0, 0, 0))
    lam = np.linalg.eigvalsh(so.tangent_hessian(model, np.array([[0.0, 0.0, 1.0]]))[0])
    assert np.allclose(lam, 0.4, atol=1e-14)
    lam = np.linalg.eigvalsh(so.tangent_hessian(model, np.array([[1.0, 0.0, 0.0]]))[0])
    assert np.allclose(lam, [-0.4, 0.0], atol=1e-14)


def test_lowest_modes_bruteforce_8x8():
    # BASELINE.json north_star pin (d): brute-force dense eigendecomposition on the 8x8 config
    w = wl.config0()
    model = model_of(w)
    lam, V = so.lowest_modes(model, w.spins, 2, extra=2)
    Ht, Bm = so.tangent_hessian(model, w.spins)
    full = np.linalg.eigvalsh(Ht)
    assert Ht.shape == (128, 128)
    assert np.allclose(lam, full[:4], atol=1e-13)
    # eigen-equation through the independent HVP route, orthonormality, tangency
    HV = so.hvp(model, w.spins, V)
    for a in range(4):
        assert np.linalg.norm(HV[a] - lam[a] * V[a]) < 1e-12
    G = V.reshape(4, -1) @ V.reshape(4, -1).T
    assert np.allclose(G, np.eye(4), atol=1e-13)
    assert np.max(np.abs(np.sum(V * w.spins[None], 2))) < 1e-14
    # noise-free limit of the same recipe recovers the 2K+B gap exactly (doubly degenerate)
    w0 = wl.config0(sigma=0.0)
    lam0, _ = so.lowest_modes(model, w0.spins, 2)
    assert np.allclose(lam0, 0.12, atol=1e-13)


def test_sparse_route_matches_dense():
    w = wl.config1(L=20)
    model = model_of(w)
    lam_d, V_d = so.lowest_modes(model, w.spins, 3)
    lam_s, V_s = so.lowest_modes_sparse(model, w.spins, 3)
    assert np.allclose(lam_d, lam_s, atol=1e-11)
    ang = scipy.linalg.subspace_angles(V_d.reshape(3, -1).T, V_s.reshape(3, -1).T)
    assert ang.max() < 1e-7
    assert lam_d[0] < 0  # a skyrmion ansatz on this lattice has negative curvature modes


def test_mmf_step_householder_invariants():
    w = wl.config0()
    model = model_of(w)
    lam, V = so.lowest_modes(model, w.spins, 2)
    F = -so.projected_gradient(model, w.spins)
    Fm = so.mmf_force(model, w.spins, V[:1])
    assert abs(np.linalg.norm(Fm) - np.linalg.norm(F)) < 1e-13
    assert abs(np.sum(Fm * V[0]) + np.sum(F * V[0])) < 1e-13
    # component orthogonal to v untouched
    Fo = F - np.sum(F * V[0]) * V[0]
    Fmo = Fm - np.sum(Fm * V[0]) * V[0]
    assert np.allclose(Fo, Fmo, atol=1e-14)
    m2 = so.mmf_step(model, w.spins, V[:1], 0.05)
    assert np.allclose(np.linalg.norm(m2, axis=1), 1.0, atol=1e-15)
    # first-order: m2 - m = dt*Fm + O(dt^2) (Fm tangent)
    assert np.max(np.abs(m2 - w.spins - 0.05 * Fm)) < 0.05 ** 2 * np.max(np.sum(Fm ** 2, 1)) + 1e-12
    # k=2 subspace variant reflects both
    Fm2 = so.mmf_force(model, w.spins, V)
    assert abs(np.sum(Fm2 * V[1]) + np.sum(F * V[1])) < 1e-13


def test_mmf_force_vanishes_only_at_stationary_point():
    # at the FM ground state F = 0 => F_mmf = 0 and the step is the identity
    model = so.SpinModel(4, 4, 1, 1, 1, 0.3, 0.05, (0, 0, 0.02))
    m = np.zeros((16, 3)); m[:, 2] = 1
    v = np.zeros((1, 16, 3)); v[0, :, 0] = 0.25
    assert np.max(np.abs(so.mmf_step(model, m, v, 0.1) - m)) < 1e-15


def test_transformed_operator_definition_pins():
    # Chebyshev T_d against numpy's own evaluation and closed forms; -p_1(H) = -(H - c0)/(a_L - c0) exactly
    x = np.linspace(-2.5, 2.5, 41)
    for d in (1, 2, 3, 7):
        ref = np.polynomial.chebyshev.chebval(x, [0] * d + [1])
        assert np.max(np.abs(so.chebyshev_T(d, x) - ref) / np.maximum(1, np.abs(ref))) < 1e-12
    assert np.allclose(so.chebyshev_T(2, x), 2 * x * x - 1)
    w = wl.config0()
    model = so.SpinModel(w.Lx, w.Ly, w.pbc_x, w.pbc_y, w.J, w.D, w.K, w.B, w.mu)
    V = wl.random_block(w.N, 2, seed=3)
    a, b, aL = 0.3, 19.0, 0.1
    HV = so.hvp(model, w.spins, V)
    PV = V - np.sum(V * w.spins[None], axis=2, keepdims=True) * w.spins[None]
    c0 = 0.5 * (a + b)
    ref1 = -(HV - c0 * PV) / (aL - c0)
    assert np.max(np.abs(so.transformed_operator_apply(model, w.spins, V, 1, a, b, aL) - ref1)) < 1e-12
    # p_d(a_L) = 1: an eigenvector with eigenvalue a_L is mapped to minus itself
    lam, Vm = so.lowest_modes(model, w.spins, 1)
    out = so.transformed_operator_apply(model, w.spins, Vm, 5, lam[0] + 0.2, 19.0, lam[0])
    assert np.max(np.abs(out + Vm)) < 1e-10


def test_mmf_run_termination_logic():
    # the loop is the composition of pinned pieces; here: the test is evaluated BEFORE a step, the cap counts applied
    # steps, and a state without a negative mode can never be declared a saddle
    w = wl.config1(L=12, R=2.5)
    model = so.SpinModel(w.Lx, w.Ly, w.pbc_x, w.pbc_y, w.J, w.D, w.K, w.B, w.mu)
    lam0, V0 = so.lowest_modes(model, w.spins, 2)
    m1, lam1, steps, conv, fn = so.mmf_run(model, w.spins, 2, 0.05, 3, 0.0)
    assert steps == 3 and not conv
    ref = w.spins
    for _ in range(3):
        _, V = so.lowest_modes(model, ref, 2)
        ref = so.mmf_step(model, ref, V[:1], 0.05)
    assert np.max(np.abs(m1 - ref)) < 1e-12
    if lam0[0] < 0.0 < lam0[1]:
        m2, _, steps2, conv2, _ = so.mmf_run(model, w.spins, 2, 0.05, 3, 1e9)
        assert steps2 == 0 and conv2 and np.array_equal(m2, w.spins)
    wf = wl.config0(sigma=0.05)                     # tilted ferromagnet: all curvatures positive
    mf = so.SpinModel(wf.Lx, wf.Ly, 1, 1, wf.J, wf.D, wf.K, wf.B, wf.mu)
    assert so.lowest_modes(mf, wf.spins, 2)[0][0] > 0
    _, _, steps3, conv3, _ = so.mmf_run(mf, wf.spins, 2, 0.05, 2, 1e9)
    assert steps3 == 2 and not conv3
