"""Pins for oracle/shell_oracle.py (no GPU): the general-neighbour-shell restatement of Eq. 4 against the already pinned
nearest-neighbour oracle, the closed-form spin-wave spectrum with several shells and out-of-plane DMI, finite differences
of the literal-loop energy, symmetry, open boundaries."""
import numpy as np
import pytest

from oracle import shell_oracle as sh
from oracle import spin_oracle as so
from paper_2509_26269_b200 import workloads as wl


def shell_model(L, rcut, pbc=(1, 1), K=0.05, B=(0.01, -0.02, 0.03), Lx=None, **kw):
    offs, J, D = wl.shell_table(rcut, **kw)
    return sh.ShellModel(Lx or L, L, pbc[0], pbc[1], offs, J, D, K, B)


@pytest.mark.parametrize("pbc", [(1, 1), (0, 0), (1, 0)])
def test_nearest_neighbour_table_reproduces_spin_oracle(pbc):
    # rcut = 1, Dz = 0: exactly the six-neighbour model of spin_oracle (D_ij = D z x rhat_ij)
    L = 6
    mdl = shell_model(L, 1.0, pbc, Dz1=0.0, Lx=7)
    ref = so.SpinModel(7, L, pbc[0], pbc[1], 1.0, 0.3, 0.05, (0.01, -0.02, 0.03))
    m = wl.random_spins(7, L, 5)
    assert abs(sh.energy(mdl, m) - so.energy(ref, m)) < 1e-12
    assert np.max(np.abs(sh.gradient(mdl, m) - so.gradient(ref, m))) < 1e-13
    assert abs(sh.euclid_hessian(mdl) - so.euclid_hessian(ref)).max() < 1e-14
    V = wl.random_block(7 * L, 2, 3)
    assert np.max(np.abs(sh.hvp(mdl, m, V) - so.hvp(ref, m, V))) < 1e-12


def test_closed_form_spin_wave_spectrum_many_shells():
    # m = +z, periodic L x L: lambda_pm(q) = 2 sum_d J_d (1 - cos q.d) + 2K + mu B +- 2 sum_d Dz_d sin q.d
    L, K, Bz = 9, 0.05, 0.02
    offs, J, D = wl.shell_table(3.0)
    assert len(offs) == 36
    mdl = sh.ShellModel(L, L, 1, 1, offs, J, D, K, (0.0, 0.0, Bz))
    m = np.zeros((L * L, 3))
    m[:, 2] = 1.0
    Ht, _ = sh.tangent_hessian(mdl, m)
    lam = np.sort(np.linalg.eigvalsh(0.5 * (Ht + Ht.T)))
    n1, n2 = np.meshgrid(np.arange(L), np.arange(L), indexing="ij")
    A = np.full((L, L), 2 * K + Bz)
    S = np.zeros((L, L))
    for (dx, dy), Jd, Dd in zip(offs, J, D):
        ph = 2 * np.pi * (n1 * dx + n2 * dy) / L
        A += 2 * Jd * (1 - np.cos(ph))
        S += 2 * Dd[2] * np.sin(ph)
    ref = np.sort(np.concatenate([(A + S).ravel(), (A - S).ravel()]))
    assert np.max(np.abs(lam - ref)) < 1e-12
    assert np.max(np.abs(S)) > 1e-2            # the non-reciprocal term is really exercised
    # in-plane DMI alone drops out at linear order: spectrum = A(q), each twice
    mdl0 = sh.ShellModel(L, L, 1, 1, *wl.shell_table(3.0, Dz1=0.0), K, (0.0, 0.0, Bz))
    Ht0, _ = sh.tangent_hessian(mdl0, m)
    assert np.max(np.abs(np.sort(np.linalg.eigvalsh(0.5 * (Ht0 + Ht0.T))) - np.sort(np.concatenate([A.ravel(), A.ravel()])))) < 1e-12


def test_gradient_is_fd_of_literal_energy_and_hessian_symmetric():
    mdl = shell_model(7, 2.0, (1, 0))
    m = wl.random_spins(7, 7, 11)
    rng = np.random.default_rng(2)
    d = rng.standard_normal(m.shape)
    g = sh.gradient(mdl, m)
    for eps in (1e-3, 1.0):                    # E is quadratic + linear in m: the central difference is exact for any eps
        fd = (sh.energy_loops(mdl, m + eps * d) - sh.energy_loops(mdl, m - eps * d)) / (2 * eps)
        assert abs(fd - np.sum(g * d)) < 1e-10 * max(1.0, abs(fd))
    assert abs(sh.energy(mdl, m) - sh.energy_loops(mdl, m)) < 1e-11
    H = sh.euclid_hessian(mdl)
    assert abs(H - H.T).max() < 1e-15
    Ht, _ = sh.tangent_hessian(mdl, m)
    assert np.max(np.abs(Ht - Ht.T)) < 1e-13
    # E = 1/2 m^T H m - mu B . sum m  (H holds the whole quadratic part)
    mv = m.ravel()
    assert abs(0.5 * mv @ (H @ mv) - np.sum(m @ mdl.B) - sh.energy(mdl, m)) < 1e-10


def test_projected_hvp_is_fd_of_projected_gradient():
    mdl = shell_model(6, 2.0)
    m = wl.random_spins(6, 6, 4)
    V = wl.random_block(36, 1, 9)
    v = V[0] - np.sum(V[0] * m, axis=1, keepdims=True) * m
    eps = 1e-5
    ret = lambda x: x / np.linalg.norm(x, axis=1, keepdims=True)
    mp, mm = ret(m + eps * v), ret(m - eps * v)
    fd = (sh.projected_gradient(mdl, mp) - sh.projected_gradient(mdl, mm)) / (2 * eps)
    fd -= np.sum(fd * m, axis=1, keepdims=True) * m
    assert np.max(np.abs(sh.hvp(mdl, m, v[None])[0] - fd)) < 1e-8


def test_open_boundaries_drop_bonds_and_table_validation():
    offs, J, D = wl.shell_table(2.0)
    per = sh.ShellModel(5, 5, 1, 1, offs, J, D, 0.0, (0, 0, 0))
    opn = sh.ShellModel(5, 5, 0, 0, offs, J, D, 0.0, (0, 0, 0))
    assert per.bonds()[0].size == 25 * len(offs)
    inside = sum(1 for x in range(5) for y in range(5) for dx, dy in offs if 0 <= x + dx < 5 and 0 <= y + dy < 5)
    assert opn.bonds()[0].size == inside < 25 * len(offs)
    with pytest.raises(AssertionError):
        sh.ShellModel(5, 5, 1, 1, offs[:-1], J[:-1], D[:-1], 0.0, (0, 0, 0))       # inversion partner missing
    D2 = D.copy(); D2[0, 2] += 0.1
    with pytest.raises(AssertionError):
        sh.ShellModel(5, 5, 1, 1, offs, J, D2, 0.0, (0, 0, 0))                      # D(-d) != -D(d)


def test_transformed_operator_spectral_definition():
    # the Chebyshev transformation -p_d(Hess) on a shell table (the operator the transformed shell solver iterates on)
    mdl = shell_model(8, 3.0, (1, 0), Lx=9)
    m = wl.random_spins(9, 8, 4)
    V = wl.random_block(72, 2, 6)
    a, b, aL = -0.4, 40.0, -1.5
    # degree 1 in closed form: p_1(x) = (x - c0) / (a_L - c0), applied through the pinned HVP
    PV = V - np.sum(V * m[None], axis=2, keepdims=True) * m[None]
    c0 = 0.5 * (a + b)
    ref1 = -(sh.hvp(mdl, m, V) - c0 * PV) / (aL - c0)
    assert np.max(np.abs(sh.transformed_operator_apply(mdl, m, V, 1, a, b, aL) - ref1)) < 1e-12
    # p_d(a_L) = 1: an eigenvector with eigenvalue a_L goes to minus itself; every other eigenvector is scaled by
    # -T_d(l(lambda)) / T_d(l(a_L)) with T_d from numpy.polynomial (not the oracle's cos / cosh form)
    lam, Vm = sh.lowest_modes(mdl, m, 3)
    out = sh.transformed_operator_apply(mdl, m, Vm[:1], 7, lam[0] + 0.3, 40.0, lam[0])
    assert np.max(np.abs(out + Vm[:1])) < 1e-10
    d, a2, b2 = 6, lam[1] + 0.05, 40.0
    ell = lambda x: (2.0 * x - a2 - b2) / (b2 - a2)
    Td = np.polynomial.chebyshev.Chebyshev.basis(d)
    out3 = sh.transformed_operator_apply(mdl, m, Vm, d, a2, b2, lam[0])
    for j in range(3):
        assert np.max(np.abs(out3[j] + Td(ell(lam[j])) / Td(ell(lam[0])) * Vm[j])) < 1e-9
    # the nearest-neighbour table gives the pinned spin oracle's operator
    mdl1 = shell_model(6, 1.0, (1, 1), Dz1=0.0, Lx=7)
    ref = so.SpinModel(7, 6, 1, 1, 1.0, 0.3, 0.05, (0.01, -0.02, 0.03))
    m1 = wl.random_spins(7, 6, 5)
    V1 = wl.random_block(42, 2, 3)
    assert np.max(np.abs(sh.transformed_operator_apply(mdl1, m1, V1, 5, -0.2, 15.0, -0.9)
                         - so.transformed_operator_apply(ref, m1, V1, 5, -0.2, 15.0, -0.9))) < 1e-10
