"""CPU oracle for the HVP-Lanczos variant of the inner eigen-solve (TEST INFRASTRUCTURE, not product code).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this module; the CUDA
path shares no code with it.

What it restates.  PAPER.md:54-60 and :160: the lowest-k curvature eigenpairs are obtained by handing the HVP callback to a
Krylov eigensolver "(Lanczos or LOBPCG) in operator mode"; "Lanczos performs better at larger sizes, so we use
it for the remaining experiments"; ref. [26] (Lanczos 1950).  The paper calls a library routine and prints no
algorithm, so this file follows the published thick-restart Lanczos method (Wu and Simon, SIAM J. Matrix Anal. Appl. 22,
602 (2000)), the method behind the library call the paper names, step by step in that paper's order:

    1. Lanczos steps j = k0 .. m-1 on the basis V = [v_0 .. v_j]:
           u = A v_j;   alpha_j = v_j . u;   u <- u - V (V^T u), twice (full re-orthogonalisation, classical Gram-Schmidt
           applied twice);   beta_j = ||u||;   v_{j+1} = u / beta_j
       T[j][j] = alpha_j, T[j][j+1] = T[j+1][j] = beta_j.
    2. Rayleigh-Ritz on the m x m projected matrix T: T = S diag(theta) S^T, keep the k smallest theta_i, Ritz vectors
       x_i = V s_i, residual norms |beta_{m-1} S[m-1][i]| (the Lanczos relation A V = V T + beta_{m-1} v_m e_m^T).
    3. Stop when all k residual norms are <= tol (absolute, ||x_i|| = 1; reading A9), else thick restart:
           V <- [x_1 .. x_k, v_m],   T <- diag(theta_1..theta_k) bordered by row/column k with entries beta_{m-1} S[m-1][i],
       and continue at step 1 with k0 = k.

Readings (A25): basis size m ("ncv") is a parameter (the paper gives none); the start vector is an input; the
iteration count reported is the number of Lanczos steps (= operator applications).

Pins (tests/test_oracle_lanczos.py): dense LAPACK eigenpairs on random symmetric matrices; the Ritz values of an m-step
run without restart against the eigenvalues of Q^T A Q for Q from a QR factorisation of the explicit Krylov matrix
[v, Av, .., A^{m-1} v] (brute force); the Lanczos relation and the bordered-diagonal shape of T after a restart; exactness
after n steps on a diagonal matrix; the spin tangent Hessian of config 0 against its dense eigendecomposition.
"""
from __future__ import annotations

import numpy as np


def lanczos_steps(apply_A, V: np.ndarray, T: np.ndarray, k0: int, m: int):
    """Steps j = k0 .. m-1 of item 1.  V: (n, m+1) with columns 0..k0 filled (orthonormal); T: (m, m) with the leading
    k0 x k0 block (and, after a restart, row/column k0) filled.  Returns beta_{m-1}; fills V[:, k0+1 .. m] and T."""
    beta = 0.0
    for j in range(k0, m):
        u = apply_A(V[:, j])
        alpha = float(V[:, j] @ u)
        for _ in range(2):                      # classical Gram-Schmidt against every basis vector, twice
            h = V[:, : j + 1].T @ u
            u = u - V[:, : j + 1] @ h
        beta = float(np.linalg.norm(u))
        T[j, j] = alpha
        if j + 1 < m:
            T[j, j + 1] = beta
            T[j + 1, j] = beta
        V[:, j + 1] = u / beta
    return beta


def thick_restart_lanczos(apply_A, v0: np.ndarray, k: int, m: int, tol: float, max_steps: int):
    """Smallest-k eigenpairs of the symmetric operator apply_A by thick-restart Lanczos with basis size m.
    Returns (theta[k] ascending, X[n, k] orthonormal, info) with info = dict(steps, converged, resid_est[k], restarts)."""
    n = v0.shape[0]
    if not (1 <= k < m <= n - 1):
        raise ValueError("need 1 <= k < m <= n - 1")
    V = np.zeros((n, m + 1))
    T = np.zeros((m, m))
    V[:, 0] = v0 / np.linalg.norm(v0)
    k0, steps, restarts = 0, 0, 0
    while True:
        beta = lanczos_steps(apply_A, V, T, k0, m)
        steps += m - k0
        theta, S = np.linalg.eigh(T)                       # item 2 (ascending)
        theta_k, S_k = theta[:k], S[:, :k]
        resid = np.abs(beta * S_k[m - 1, :])
        X = V[:, :m] @ S_k
        converged = bool(np.all(resid <= tol))
        if converged or steps >= max_steps:
            return theta_k.copy(), X, dict(steps=steps, converged=converged, resid_est=resid, restarts=restarts)
        # item 3: thick restart
        V[:, :k] = X
        V[:, k] = V[:, m]
        T[:, :] = 0.0
        T[np.arange(k), np.arange(k)] = theta_k
        T[k, :k] = beta * S_k[m - 1, :]
        T[:k, k] = beta * S_k[m - 1, :]
        k0 = k
        restarts += 1


def lowest_modes_lanczos(model, spins: np.ndarray, k: int, v0: np.ndarray, m: int, tol: float, max_steps: int = 100000):
    """The spin-lattice instance: A = Riemannian Hessian B H_t B^T in the ambient 3N coordinates (the operator of
    oracle.spin_oracle.hvp, with H_t and the tangent basis B built once), start vector projected onto the tangent space.
    v0: (N, 3).  Returns (theta[k], V[k, N, 3], info)."""
    from oracle import spin_oracle as so
    N = spins.shape[0]
    Ht, Bm = so.tangent_hessian(model, spins, dense=False)
    Ht = 0.5 * (Ht + Ht.T)

    def apply_A(x):
        return Bm @ (Ht @ (Bm.T @ x))

    x0 = Bm @ (Bm.T @ v0.reshape(-1))
    theta, X, info = thick_restart_lanczos(apply_A, x0, k, m, tol, max_steps)
    return theta, np.ascontiguousarray(X.T).reshape(k, N, 3), info
