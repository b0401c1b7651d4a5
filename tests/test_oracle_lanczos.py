"""Pins for oracle/lanczos_oracle.py against things it does not itself define (no GPU)."""
import numpy as np
import pytest
import scipy.linalg

from oracle import lanczos_oracle as lo
from oracle import spin_oracle as so
from paper_2509_26269_b200 import workloads as wl


def sym(n, seed, spread=None):
    rng = np.random.default_rng(seed)
    if spread is None:
        A = rng.standard_normal((n, n))
        return 0.5 * (A + A.T)
    Q = np.linalg.qr(rng.standard_normal((n, n)))[0]
    return (Q * spread) @ Q.T


@pytest.mark.parametrize("n,k,m,seed", [(60, 2, 12, 0), (200, 3, 15, 1), (200, 1, 8, 2), (90, 6, 20, 3)])
def test_matches_lapack_on_random_symmetric(n, k, m, seed):
    A = sym(n, seed)
    v0 = np.random.default_rng(100 + seed).standard_normal(n)
    theta, X, info = lo.thick_restart_lanczos(lambda x: A @ x, v0, k, m, 1e-10, 200000)
    ref, Y = scipy.linalg.eigh(A)
    assert info["converged"]
    assert np.max(np.abs(theta - ref[:k])) <= 1e-9
    assert np.max(np.abs(X.T @ X - np.eye(k))) <= 1e-12
    # true residuals agree with the estimates the stop test used, and meet the tolerance
    R = A @ X - X * theta
    assert np.max(np.linalg.norm(R, axis=0)) <= 1e-10 * (1 + 1e-3) + 1e-13
    assert np.max(np.abs(np.linalg.norm(R, axis=0) - info["resid_est"])) <= 1e-12
    ang = scipy.linalg.subspace_angles(X, Y[:, :k])
    assert ang.max() <= 1e-7


def test_ritz_values_of_unrestarted_run_equal_brute_force_krylov_projection():
    # m steps without restart span K_m(A, v); the Ritz values are the eigenvalues of Q^T A Q for ANY orthonormal basis Q
    n, m = 40, 9
    A = sym(n, 7, spread=np.linspace(0.5, 3.0, n))        # well conditioned so the explicit Krylov matrix is usable
    v0 = np.random.default_rng(8).standard_normal(n)
    K = np.empty((n, m)); x = v0.copy()
    for j in range(m):
        K[:, j] = x / np.linalg.norm(x); x = A @ K[:, j]
    Q = np.linalg.qr(K)[0]
    ref = scipy.linalg.eigvalsh(Q.T @ A @ Q)
    V = np.zeros((n, m + 1)); T = np.zeros((m, m)); V[:, 0] = v0 / np.linalg.norm(v0)
    lo.lanczos_steps(lambda x: A @ x, V, T, 0, m)
    assert np.max(np.abs(scipy.linalg.eigvalsh(T) - ref)) <= 1e-9
    # T is tridiagonal with positive off-diagonals, and equals V^T A V
    assert np.max(np.abs(np.triu(T, 2))) == 0.0 and np.all(np.diag(T, 1) > 0)
    assert np.max(np.abs(V[:, :m].T @ A @ V[:, :m] - T)) <= 1e-12


def test_lanczos_relation_and_bordered_shape_after_restart():
    n, k, m = 80, 3, 10
    A = sym(n, 11)
    calls = []
    def op(x):
        calls.append(1); return A @ x
    # run exactly one restart: max_steps = m + (m - k)
    theta, X, info = lo.thick_restart_lanczos(op, np.ones(n), k, m, 0.0, m + (m - k))
    assert info["restarts"] == 1 and info["steps"] == m + (m - k) == len(calls)
    # re-create the state after the restart by hand and check A V = V T + beta v_m e_m^T with T bordered-diagonal
    V = np.zeros((n, m + 1)); T = np.zeros((m, m)); V[:, 0] = 1.0 / np.sqrt(n)
    beta = lo.lanczos_steps(lambda x: A @ x, V, T, 0, m)
    th, S = np.linalg.eigh(T)
    Vr = np.zeros((n, m + 1)); Tr = np.zeros((m, m))
    Vr[:, :k] = V[:, :m] @ S[:, :k]; Vr[:, k] = V[:, m]
    Tr[np.arange(k), np.arange(k)] = th[:k]; Tr[k, :k] = Tr[:k, k] = beta * S[m - 1, :k]
    beta2 = lo.lanczos_steps(lambda x: A @ x, Vr, Tr, k, m)
    E = A @ Vr[:, :m] - Vr[:, :m] @ Tr
    E[:, m - 1] -= beta2 * Vr[:, m]
    assert np.max(np.abs(E)) <= 1e-12 * np.linalg.norm(A, 2) * 10
    assert np.max(np.abs(Vr.T @ Vr - np.eye(m + 1))) <= 1e-13
    assert np.max(np.abs(Vr[:, :m].T @ A @ Vr[:, :m] - Tr)) <= 1e-12
    # and the second cycle of the driver is exactly this state
    th2 = np.linalg.eigvalsh(Tr)[:k]
    assert np.max(np.abs(th2 - theta)) <= 1e-13


def test_diagonal_matrix_is_exact_after_n_minus_1_dimensional_krylov_space():
    d = np.array([3.0, -1.0, 0.5, 2.0, -0.25, 7.0, 1.5])
    n = d.size
    theta, X, info = lo.thick_restart_lanczos(lambda x: d * x, np.ones(n), 2, n - 1, 1e-12, 10000)
    assert info["converged"]
    assert np.max(np.abs(theta - np.array([-1.0, -0.25]))) <= 1e-12
    assert abs(abs(X[1, 0]) - 1.0) <= 1e-10 and abs(abs(X[4, 1]) - 1.0) <= 1e-10


def test_argument_checks():
    with pytest.raises(ValueError):
        lo.thick_restart_lanczos(lambda x: x, np.ones(5), 2, 2, 1e-8, 10)
    with pytest.raises(ValueError):
        lo.thick_restart_lanczos(lambda x: x, np.ones(5), 2, 5, 1e-8, 10)


def test_spin_hessian_config0_matches_dense():
    w = wl.config0()
    model = so.SpinModel(w.Lx, w.Ly, w.pbc_x, w.pbc_y, w.J, w.D, w.K, w.B, w.mu)
    lam_ref, V_ref = so.lowest_modes(model, w.spins, 2)
    v0 = wl.random_block(w.N, 1, seed=5)[0]
    theta, V, info = lo.lowest_modes_lanczos(model, w.spins, 2, v0, 15, 1e-10)
    assert info["converged"]
    assert np.max(np.abs(theta - lam_ref)) <= 1e-9 * np.max(np.abs(lam_ref))
    ang = scipy.linalg.subspace_angles(V.reshape(2, -1).T, V_ref.reshape(2, -1).T)
    assert ang.max() <= 1e-6
    # tangent: m_i . v_i = 0
    assert np.max(np.abs(np.einsum("nc,knc->kn", w.spins, V))) <= 1e-12
    # and the HVP oracle's own residual
    HV = so.hvp(model, w.spins, V)
    assert np.max(np.linalg.norm((HV - theta[:, None, None] * V).reshape(2, -1), axis=1)) <= 2e-10
