"""CPU ORACLE (test infrastructure, NOT the product) -- spin lattice with GENERAL neighbour shells.

Eq. 4 is written for arbitrary pairs: E = -sum_{i != j} [J_ij m_i.m_j + D_ij.(m_i x m_j)]
- sum_i mu B.m_i - sum_i K (m_i.e_z)^2; the paper's Pd/Fe/Ir(111) workload tabulates J_ij and the full three-component
D_ij over many shells (Tables I/II PAPER.md:328-616, ~340 neighbours per site, 100x100 periodic).  Here the
couplings are a translation-invariant table over lattice offsets delta = (dx, dy):  J_ij = J_delta, D_ij = D_delta for
j = i + delta, ordered pairs counted as printed (reading A1).  The table must be inversion symmetric
(J_{-delta} = J_delta, D_{-delta} = -D_delta: the same bond seen from its other end, reading A2), otherwise Eq. 4 has no
symmetric Hessian; the constructor checks it.

Same steps as oracle/spin_oracle.py (O1-O9), restated for the table: literal double loop for the energy, gradient
g_i = -2 sum_delta [J_delta m_j + m_j x D_delta] - mu B - 2 K m_iz z, Euclidean Hessian assembled bond by bond
(H_ij = -2 J_delta I3 + 2 [D_delta]x, H_ii = -2 K z z^T), tangent Hessian B^T (H - diag(c_i I3)) B, LAPACK eigh,
HVP = B H_t B^T V.  The model-independent pieces (tangent basis, c_i) are taken from spin_oracle.

Pins (tests/test_oracle_shell.py): the nearest-neighbour table reproduces the pinned spin_oracle; closed-form spin-wave
spectrum at m = +z on the periodic L x L lattice,
    lambda_pm(q) = 2 sum_delta J_delta (1 - cos q.delta) + 2K + mu B  +-  2 sum_delta D^z_delta sin q.delta ,
    q.delta = 2 pi (n1 dx + n2 dy)/L   (in-plane DMI components drop out at linear order; the z components give the
    non-reciprocal term);  central differences of the literal-loop energy;  Hessian symmetry;  open boundaries drop bonds.
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline legs may import this file; it shares no code with the
CUDA path.
"""
from __future__ import annotations

import numpy as np
import scipy.linalg
import scipy.sparse as sp

from . import spin_oracle as so


class ShellModel:
    def __init__(self, Lx, Ly, pbc_x, pbc_y, offsets, Jd, Dd, K, B, mu=1.0):
        self.Lx, self.Ly, self.pbc_x, self.pbc_y = int(Lx), int(Ly), bool(pbc_x), bool(pbc_y)
        self.offsets = np.asarray(offsets, dtype=np.int64).reshape(-1, 2)
        self.Jd = np.asarray(Jd, dtype=np.float64).reshape(-1)
        self.Dd = np.asarray(Dd, dtype=np.float64).reshape(-1, 3)
        self.K, self.mu = float(K), float(mu)
        self.B = np.asarray(B, dtype=np.float64).reshape(3)
        self.N = self.Lx * self.Ly
        n = self.offsets.shape[0]
        assert self.Jd.shape[0] == n and self.Dd.shape[0] == n
        index = {(int(dx), int(dy)): t for t, (dx, dy) in enumerate(self.offsets)}
        assert len(index) == n and (0, 0) not in index, "offsets must be distinct and non-zero"
        for (dx, dy), t in index.items():
            u = index.get((-dx, -dy))
            assert u is not None and self.Jd[u] == self.Jd[t] and np.all(self.Dd[u] == -self.Dd[t]), \
                "table must be inversion symmetric: J(-d) = J(d), D(-d) = -D(d)"
        self._bonds = None

    # O1: ordered pairs (i, j = i + delta, shell index); open boundaries drop the neighbour
    def bonds(self):
        if self._bonds is None:
            I, Jn, T = [], [], []
            ix = np.arange(self.Lx)[None, :].repeat(self.Ly, 0)
            iy = np.arange(self.Ly)[:, None].repeat(self.Lx, 1)
            for t, (dx, dy) in enumerate(self.offsets):
                jx, jy = ix + dx, iy + dy
                ok = np.ones_like(ix, dtype=bool)
                if self.pbc_x:
                    jx = jx % self.Lx
                else:
                    ok &= (jx >= 0) & (jx < self.Lx)
                if self.pbc_y:
                    jy = jy % self.Ly
                else:
                    ok &= (jy >= 0) & (jy < self.Ly)
                I.append((iy * self.Lx + ix)[ok])
                Jn.append((jy * self.Lx + jx)[ok])
                T.append(np.full(int(ok.sum()), t))
            self._bonds = (np.concatenate(I), np.concatenate(Jn), np.concatenate(T))
        return self._bonds


# O2: energy, literally Eq. 4
def energy_loops(model: ShellModel, m: np.ndarray) -> float:
    I, Jn, T = model.bonds()
    E = 0.0
    for b in range(I.size):
        mi, mj = m[I[b]], m[Jn[b]]
        E -= model.Jd[T[b]] * float(mi @ mj)
        E -= float(model.Dd[T[b]] @ np.cross(mi, mj))
    for i in range(model.N):
        E -= model.mu * float(model.B @ m[i])
        E -= model.K * float(m[i, 2]) ** 2
    return E


def energy(model: ShellModel, m: np.ndarray) -> float:
    I, Jn, T = model.bonds()
    mi, mj = m[I], m[Jn]
    e_ex = -np.sum(model.Jd[T] * np.sum(mi * mj, axis=1))
    e_dm = -np.sum(model.Dd[T] * np.cross(mi, mj))
    return float(e_ex + e_dm - model.mu * np.sum(m @ model.B) - model.K * np.sum(m[:, 2] ** 2))


# O3: g_i = -2 sum_j [J_ij m_j + m_j x D_ij] - mu B - 2 K m_iz z
def gradient(model: ShellModel, m: np.ndarray) -> np.ndarray:
    I, Jn, T = model.bonds()
    contrib = -2.0 * (model.Jd[T][:, None] * m[Jn] + np.cross(m[Jn], model.Dd[T]))
    g = np.zeros_like(m)
    np.add.at(g, I, contrib)
    g -= model.mu * model.B[None, :]
    g[:, 2] -= 2.0 * model.K * m[:, 2]
    return g


def projected_gradient(model: ShellModel, m: np.ndarray) -> np.ndarray:
    g = gradient(model, m)
    return g - so.curvature_scalar(m, g)[:, None] * m


# O5: H_ij = -2 J_ij I3 + 2 [D_ij]x, H_ii = -2 K z z^T, one 3x3 block per ordered bond
def euclid_hessian(model: ShellModel) -> sp.csr_matrix:
    I, Jn, T = model.bonds()
    blocks = np.empty((model.offsets.shape[0], 3, 3))
    for t in range(blocks.shape[0]):
        blocks[t] = -2.0 * model.Jd[t] * np.eye(3) + 2.0 * so._cross_matrix(model.Dd[t])
    rows, cols, vals = [], [], []
    for a in range(3):
        for b in range(3):
            rows.append(3 * I + a)
            cols.append(3 * Jn + b)
            vals.append(blocks[T, a, b])
    ii = np.arange(model.N)
    rows.append(3 * ii + 2)
    cols.append(3 * ii + 2)
    vals.append(np.full(model.N, -2.0 * model.K))
    H = sp.coo_matrix((np.concatenate(vals), (np.concatenate(rows), np.concatenate(cols))), shape=(3 * model.N, 3 * model.N))
    return H.tocsr()


# O7: H_t = B^T (H - diag(c_i I3)) B
def tangent_hessian(model: ShellModel, m: np.ndarray, dense: bool = True):
    H = euclid_hessian(model)
    c = so.curvature_scalar(m, gradient(model, m))
    Bm = so.tangent_basis(m)
    Ht = Bm.T @ (H - sp.diags(np.repeat(c, 3))) @ Bm
    return (Ht.toarray() if dense else Ht.tocsc()), Bm


def lowest_modes(model: ShellModel, m: np.ndarray, k: int, extra: int = 0):
    Ht, Bm = tangent_hessian(model, m, dense=True)
    lam, Y = scipy.linalg.eigh(0.5 * (Ht + Ht.T), subset_by_index=[0, k + extra - 1])
    return lam, np.ascontiguousarray((Bm @ Y).T).reshape(k + extra, model.N, 3)


def hvp(model: ShellModel, m: np.ndarray, V: np.ndarray) -> np.ndarray:
    Ht, Bm = tangent_hessian(model, m, dense=False)
    k = V.shape[0]
    out = Bm @ (Ht @ (Bm.T @ V.reshape(k, -1).T))
    return np.ascontiguousarray(out.T).reshape(k, model.N, 3)


def transformed_operator_apply(model: ShellModel, m: np.ndarray, V: np.ndarray, d: int, a: float, b: float, a_L: float):
    """-p_d(Hess) V for tangent-projected V ([k][N][3]): the Chebyshev spectral transformation of the solver (DESIGN.md 5,
    Zhou-Saad filter p_d(x) = T_d(l(x)) / T_d(l(a_L)), l(x) = (2x - a - b)/(b - a)) written out by its SPECTRAL definition --
    eigh of the explicit tangent Hessian, the polynomial applied to the eigenvalues -- as spin_oracle.transformed_operator_apply
    does for the stencil model.  Pins: degree 1 in closed form, p_d(a_L) = 1 on an eigenvector, the nearest-neighbour table
    against the pinned spin oracle, T_d against numpy.polynomial (tests/test_oracle_shell.py)."""
    Ht, Bm = tangent_hessian(model, m, dense=True)
    lam, Y = scipy.linalg.eigh(0.5 * (Ht + Ht.T))
    ell = lambda x: (2.0 * x - a - b) / (b - a)
    pl = so.chebyshev_T(d, ell(lam)) / so.chebyshev_T(d, np.array([ell(a_L)]))[0]
    k = V.shape[0]
    coeff = Y.T @ (Bm.T @ V.reshape(k, -1).T)
    out = -(Bm @ (Y @ (pl[:, None] * coeff)))
    return np.ascontiguousarray(out.T).reshape(k, model.N, 3)


def mmf_step(model: ShellModel, m: np.ndarray, v: np.ndarray, dt: float) -> np.ndarray:
    """Eq. 2 + retraction, as spin_oracle.mmf_step."""
    F = -projected_gradient(model, m)
    out = F.copy()
    for a in range(v.shape[0]):
        out -= 2.0 * np.sum(F * v[a]) * v[a]
    x = m + dt * out
    return x / np.linalg.norm(x, axis=1, keepdims=True)
