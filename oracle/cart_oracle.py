"""CPU ORACLE (test infrastructure, NOT the product) -- Cartesian-atom path.

Plain all-pairs O(Na^2) numpy restatement of the Ni(111) portability case of arxiv 2509.26269
("only the projector switched to Cartesian updates") with the Morse pair
potential and parameters BASELINE.json configs[4] fixes (the paper's EAM tables are not available):

  phi(r) = De [exp(-2 alpha (r - r0)) - 2 exp(-alpha (r - r0))]  for r < rc, 0 otherwise
  energy reported with the constant shift phi(r) - phi(rc) (reading A21; leaves g and H unchanged)
  minimum image in the 2-D periodic in-plane cell, open in z; no cell list here (that is the GPU's)
  masked Hessian = rows/cols of the free atoms, dense LAPACK eigen-solve  ("masked")
  reflected-force step with identity retraction on the free atoms

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline / ``--impl reference``
legs may import this file.  It shares no code with the CUDA path.  Pins (tests/test_oracle_cart.py):
central finite differences of the energy / gradient, Hessian symmetry, acoustic sum rule, isolated
dimer closed form 2 phi''(r0) = 4 alpha^2 De.  The multi-step MMF trajectory is "parity unpinned"
beyond one step (neighbour set changes at the cut-off, reading H11).
"""
from __future__ import annotations

import numpy as np
import scipy.linalg


class MorseModel:
    def __init__(self, cell, De, alpha, r0, rc, fixed=None):
        self.cell = np.asarray(cell, dtype=np.float64).reshape(2, 2)  # rows = in-plane cell vectors
        self.De, self.alpha, self.r0, self.rc = float(De), float(alpha), float(r0), float(rc)
        self.fixed = None if fixed is None else np.asarray(fixed).astype(bool)
        self._inv = np.linalg.inv(self.cell)

    def phi(self, r):
        e = np.exp(-self.alpha * (r - self.r0))
        return self.De * (e * e - 2.0 * e)

    def dphi(self, r):
        e = np.exp(-self.alpha * (r - self.r0))
        return self.De * (-2.0 * self.alpha * e * e + 2.0 * self.alpha * e)

    def d2phi(self, r):
        e = np.exp(-self.alpha * (r - self.r0))
        return self.De * (4.0 * self.alpha ** 2 * e * e - 2.0 * self.alpha ** 2 * e)

    def min_image(self, d):
        """d[...,3] -> minimum-image displacement (in-plane periodic, z open)."""
        s = d[..., :2] @ self._inv
        s -= np.round(s)
        out = d.copy()
        out[..., :2] = s @ self.cell
        return out

    def pairs(self, x):
        """All ordered pairs (i, j), i != j, with r_ij < rc: returns i, j, d_ij = x_i - x_j (min image), r."""
        Na = x.shape[0]
        I, Jn, Dv, R = [], [], [], []
        for i in range(Na):
            d = self.min_image(x[i][None, :] - x)
            r = np.linalg.norm(d, axis=1)
            ok = (r < self.rc)
            ok[i] = False
            j = np.nonzero(ok)[0]
            I.append(np.full(j.size, i))
            Jn.append(j)
            Dv.append(d[j])
            R.append(r[j])
        return np.concatenate(I), np.concatenate(Jn), np.concatenate(Dv, 0), np.concatenate(R)


def energy(model: MorseModel, x: np.ndarray) -> float:
    """E = 1/2 sum_{i != j, r<rc} [phi(r_ij) - phi(rc)]."""
    _, _, _, r = model.pairs(x)
    return float(0.5 * np.sum(model.phi(r) - model.phi(model.rc)))


def gradient(model: MorseModel, x: np.ndarray, masked: bool = True) -> np.ndarray:
    """g_i = sum_j phi'(r_ij) n_ij, n_ij = (x_i - x_j)/r_ij; rows of fixed atoms zeroed when masked."""
    I, _, d, r = model.pairs(x)
    contrib = (model.dphi(r) / r)[:, None] * d
    g = np.zeros_like(x)
    np.add.at(g, I, contrib)
    if masked and model.fixed is not None:
        g[model.fixed] = 0.0
    return g


def hessian(model: MorseModel, x: np.ndarray) -> np.ndarray:
    """Unmasked dense 3Na x 3Na Hessian: K_ij = phi'' n n^T + (phi'/r)(I - n n^T); H_ii += K_ij, H_ij = -K_ij."""
    Na = x.shape[0]
    H = np.zeros((3 * Na, 3 * Na))
    I, Jn, d, r = model.pairs(x)
    n = d / r[:, None]
    nn = n[:, :, None] * n[:, None, :]
    Kb = model.d2phi(r)[:, None, None] * nn + (model.dphi(r) / r)[:, None, None] * (np.eye(3)[None] - nn)
    for b in range(I.size):
        i, j = I[b], Jn[b]
        H[3 * i:3 * i + 3, 3 * i:3 * i + 3] += Kb[b]
        H[3 * i:3 * i + 3, 3 * j:3 * j + 3] -= Kb[b]
    return H


def free_dofs(model: MorseModel, Na: int) -> np.ndarray:
    free = np.ones(Na, dtype=bool) if model.fixed is None else ~model.fixed
    return (3 * np.nonzero(free)[0][:, None] + np.arange(3)[None, :]).ravel()


def hvp(model: MorseModel, x: np.ndarray, V: np.ndarray) -> np.ndarray:
    """Masked HVP: fixed atoms have v = 0 on input and a zero row on output (reading A21)."""
    Na = x.shape[0]
    H = hessian(model, x)
    idx = free_dofs(model, Na)
    k = V.shape[0]
    Vf = V.reshape(k, -1)
    out = np.zeros_like(Vf)
    out[:, idx] = (H[np.ix_(idx, idx)] @ Vf[:, idx].T).T
    return out.reshape(k, Na, 3)


def lowest_modes(model: MorseModel, x: np.ndarray, k: int, extra: int = 0):
    Na = x.shape[0]
    H = hessian(model, x)
    idx = free_dofs(model, Na)
    Hm = H[np.ix_(idx, idx)]
    Hm = 0.5 * (Hm + Hm.T)
    lam, Y = scipy.linalg.eigh(Hm, subset_by_index=[0, k + extra - 1])
    V = np.zeros((k + extra, 3 * Na))
    V[:, idx] = Y.T
    return lam, V.reshape(k + extra, Na, 3)


def mmf_force(model: MorseModel, x: np.ndarray, v: np.ndarray) -> np.ndarray:
    F = -gradient(model, x, masked=True)
    out = F.copy()
    for a in range(v.shape[0]):
        out -= 2.0 * np.sum(F * v[a]) * v[a]
    if model.fixed is not None:
        out[model.fixed] = 0.0
    return out


def mmf_step(model: MorseModel, x: np.ndarray, v: np.ndarray, dt: float) -> np.ndarray:
    """x' = x + dt F_mmf on the free atoms; identity retraction."""
    return x + dt * mmf_force(model, x, v)
