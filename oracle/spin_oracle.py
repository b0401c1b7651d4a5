"""CPU ORACLE (test infrastructure, NOT the product) -- spin-lattice path.

Plain, slow, obviously-correct numpy/scipy restatement of what the hot path of
arxiv 2509.26269 ("MOTO") computes on a 2-D triangular spin lattice, fp64 throughout:

  energy                 PAPER.md:136-138  (Eq. 4), ordered pairs i != j counted as written (reading A1)
  gradient               derivative of Eq. 4 ("forces ... tangent-projected")
  explicit Hessian       PAPER.md:162 (Sec. III.B.b): Jacobian of the tangent-projected gradient,
                         restricted to the tangent space, dense symmetric eigen-solve
  HVP                    PAPER.md:156 (H v = d/de grad E(m + e v)), applied in the tangent space with
                         the -(m_i . g_i) v_i curvature term (BASELINE.json north_star; reading A5)
  reflected-force step   PAPER.md:64 (Eq. 2), PAPER.md:262 (Alg. 1 l.12), retraction = renormalise (A7)

The method reaches exactly the lowest-k eigenpairs of a well-defined symmetric matrix, so the
oracle is that definition written out: assemble the explicit tangent Hessian bond by bond and call
LAPACK (dense) or ARPACK shift-invert (sparse, for lattices whose dense matrix does not fit).

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline / ``--impl reference``
legs may import this file.  It shares no code with the CUDA path and imports nothing from the
package.  Pins (tests/test_oracle_spin.py): closed-form magnon dispersion, finite differences of the
literal Eq.-4 energy, Hessian symmetry, rotation identity, single-spin closed forms, graph-adjacency
special case, brute force on 8x8.  Parity status: every function below is pinned except the
multi-step MMF *trajectory* (per-step only) -- see DESIGN.md "Pins".
"""
from __future__ import annotations

import numpy as np
import scipy.linalg
import scipy.sparse as sp
import scipy.sparse.linalg as spla

SQRT3_2 = np.sqrt(3.0) / 2.0
# O1: the six nearest-neighbour offsets (dix, diy) of the rhombic triangular lattice and their
# un-wrapped unit bond vectors rhat = dix*a1 + diy*a2 with a1=(1,0), a2=(1/2, sqrt3/2).
NN_OFFSETS = [(1, 0), (-1, 0), (0, 1), (0, -1), (-1, 1), (1, -1)]


def bond_vector(dix: int, diy: int) -> np.ndarray:
    return np.array([dix * 1.0 + diy * 0.5, diy * SQRT3_2, 0.0])


class SpinModel:
    """Lattice + Eq.-4 parameters.  D_ij = D (z x rhat_ij), rhat_ij = r_j - r_i (reading A2)."""

    def __init__(self, Lx, Ly, pbc_x, pbc_y, J, D, K, B, mu=1.0):
        self.Lx, self.Ly, self.pbc_x, self.pbc_y = int(Lx), int(Ly), bool(pbc_x), bool(pbc_y)
        self.J, self.D, self.K, self.mu = float(J), float(D), float(K), float(mu)
        self.B = np.asarray(B, dtype=np.float64).reshape(3)
        self.N = self.Lx * self.Ly
        self._bonds = None

    # ---- O1 neighbour table: ordered pairs (i, j, rhat_ij); open boundaries drop the neighbour
    def bonds(self):
        if self._bonds is None:
            I, Jn, R = [], [], []
            ix = np.arange(self.Lx)[None, :].repeat(self.Ly, 0)
            iy = np.arange(self.Ly)[:, None].repeat(self.Lx, 1)
            for (dx, dy) in NN_OFFSETS:
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
                i = (iy * self.Lx + ix)[ok]
                j = (jy * self.Lx + jx)[ok]
                I.append(i)
                Jn.append(j)
                R.append(np.broadcast_to(bond_vector(dx, dy), (i.size, 3)))
            self._bonds = (np.concatenate(I), np.concatenate(Jn), np.concatenate(R, 0))
        return self._bonds

    def dmi_vectors(self):
        """D_ij = D (z x rhat_ij) for every ordered bond."""
        _, _, R = self.bonds()
        z = np.array([0.0, 0.0, 1.0])
        return self.D * np.cross(np.broadcast_to(z, R.shape), R)


# ---- O2 energy, literally Eq. 4
def energy_loops(model: SpinModel, m: np.ndarray) -> float:
    """Pure-Python double loop over ordered pairs; small lattices only."""
    I, Jn, _ = model.bonds()
    Dv = model.dmi_vectors()
    E = 0.0
    for b in range(I.size):
        mi, mj = m[I[b]], m[Jn[b]]
        E -= model.J * float(mi @ mj)
        E -= float(Dv[b] @ np.cross(mi, mj))
    for i in range(model.N):
        E -= model.mu * float(model.B @ m[i])
        E -= model.K * float(m[i, 2]) ** 2
    return E


def energy(model: SpinModel, m: np.ndarray) -> float:
    """Eq. 4 with the pair sums written as array sums over the ordered-bond list."""
    I, Jn, _ = model.bonds()
    Dv = model.dmi_vectors()
    mi, mj = m[I], m[Jn]
    e_ex = -model.J * np.sum(mi * mj)
    e_dm = -np.sum(Dv * np.cross(mi, mj))
    e_ze = -model.mu * np.sum(m @ model.B)
    e_an = -model.K * np.sum(m[:, 2] ** 2)
    return float(e_ex + e_dm + e_ze + e_an)


# ---- O3 Euclidean gradient  g_i = -2 sum_j [J m_j + m_j x D_ij] - mu B - 2 K m_iz z
def gradient(model: SpinModel, m: np.ndarray) -> np.ndarray:
    I, Jn, _ = model.bonds()
    Dv = model.dmi_vectors()
    contrib = -2.0 * (model.J * m[Jn] + np.cross(m[Jn], Dv))
    g = np.zeros_like(m)
    np.add.at(g, I, contrib)
    g -= model.mu * model.B[None, :]
    g[:, 2] -= 2.0 * model.K * m[:, 2]
    return g


# ---- O4 c_i = m_i . g_i ; Riemannian gradient P g = g - c m
def curvature_scalar(m: np.ndarray, g: np.ndarray) -> np.ndarray:
    return np.sum(m * g, axis=1)


def projected_gradient(model: SpinModel, m: np.ndarray) -> np.ndarray:
    g = gradient(model, m)
    return g - curvature_scalar(m, g)[:, None] * m


def _cross_matrix(d: np.ndarray) -> np.ndarray:
    """[d]x with [d]x u = d x u."""
    return np.array([[0.0, -d[2], d[1]], [d[2], 0.0, -d[0]], [-d[1], d[0], 0.0]])


# ---- O5 explicit Euclidean Hessian (3N x 3N), bond by bond.  Constant in m.
#      H_ij = -2 J I3 + 2 [D_ij]x ,  H_ii = -2 K z z^T
def euclid_hessian(model: SpinModel) -> sp.csr_matrix:
    I, Jn, _ = model.bonds()
    Dv = model.dmi_vectors()
    rows, cols, vals = [], [], []
    # group bonds by DMI vector (six distinct ones) to keep this assembly short but explicit
    for a in range(3):
        for b in range(3):
            blk = np.zeros(I.size)
            if a == b:
                blk += -2.0 * model.J
            # 2 [D]x entry (a, b)
            e = np.zeros(I.size)
            if (a, b) == (0, 1):
                e = -Dv[:, 2]
            elif (a, b) == (0, 2):
                e = Dv[:, 1]
            elif (a, b) == (1, 0):
                e = Dv[:, 2]
            elif (a, b) == (1, 2):
                e = -Dv[:, 0]
            elif (a, b) == (2, 0):
                e = -Dv[:, 1]
            elif (a, b) == (2, 1):
                e = Dv[:, 0]
            blk = blk + 2.0 * e
            rows.append(3 * I + a)
            cols.append(3 * Jn + b)
            vals.append(blk)
    ii = np.arange(model.N)
    rows.append(3 * ii + 2)
    cols.append(3 * ii + 2)
    vals.append(np.full(model.N, -2.0 * model.K))
    H = sp.coo_matrix((np.concatenate(vals), (np.concatenate(rows), np.concatenate(cols))),
                      shape=(3 * model.N, 3 * model.N))
    return H.tocsr()


# ---- O6 tangent basis B (3N x 2N): e1 = normalize(m x a), a = axis with smallest |m.a|, e2 = m x e1
def tangent_basis(m: np.ndarray) -> sp.csr_matrix:
    N = m.shape[0]
    ax = np.argmin(np.abs(m), axis=1)
    a = np.zeros_like(m)
    a[np.arange(N), ax] = 1.0
    e1 = np.cross(m, a)
    e1 /= np.linalg.norm(e1, axis=1, keepdims=True)
    e2 = np.cross(m, e1)
    rows = (3 * np.arange(N)[:, None] + np.arange(3)[None, :])
    r = np.concatenate([rows.ravel(), rows.ravel()])
    c = np.concatenate([np.repeat(2 * np.arange(N), 3), np.repeat(2 * np.arange(N) + 1, 3)])
    v = np.concatenate([e1.ravel(), e2.ravel()])
    return sp.coo_matrix((v, (r, c)), shape=(3 * N, 2 * N)).tocsr()


# ---- O7 tangent Hessian  H_t = B^T (H - diag(c_i I3)) B   (2N x 2N)
def tangent_hessian(model: SpinModel, m: np.ndarray, dense: bool = True):
    H = euclid_hessian(model)
    c = curvature_scalar(m, gradient(model, m))
    Bm = tangent_basis(m)
    A = H - sp.diags(np.repeat(c, 3))
    Ht = (Bm.T @ A @ Bm)
    if dense:
        return Ht.toarray(), Bm
    return Ht.tocsc(), Bm


# ---- O8 lowest-k eigenpairs; ambient modes V = B Y  ([k][N][3], orthonormal)
def lowest_modes(model: SpinModel, m: np.ndarray, k: int, extra: int = 0):
    """Dense LAPACK solve of the explicit tangent Hessian. Returns (lam[k+extra], V[k+extra][N][3])."""
    Ht, Bm = tangent_hessian(model, m, dense=True)
    Ht = 0.5 * (Ht + Ht.T)  # "Hermitian part"; Ht is already symmetric to rounding
    lam, Y = scipy.linalg.eigh(Ht, subset_by_index=[0, k + extra - 1])
    V = np.ascontiguousarray((Bm @ Y).T).reshape(k + extra, model.N, 3)
    return lam, V


def lowest_modes_sparse(model: SpinModel, m: np.ndarray, k: int, extra: int = 0, sigma: float | None = None,
                        tol: float = 0.0):
    """O-sparse: same H_t in CSC, ARPACK shift-invert with sigma below the spectrum."""
    Ht, Bm = tangent_hessian(model, m, dense=False)
    Ht = (0.5 * (Ht + Ht.T)).tocsc()
    if sigma is None:
        sigma = -1.0  # spectrum is bounded below by about -|c|max - small; all configs have lam_min > -0.5
    lam, Y = spla.eigsh(Ht, k=k + extra, sigma=sigma, which="LM", tol=tol)
    order = np.argsort(lam)
    lam, Y = lam[order], Y[:, order]
    V = np.ascontiguousarray((Bm @ Y).T).reshape(k + extra, model.N, 3)
    return lam, V


# ---- O9 HVP oracle  HV = B H_t B^T V  (input projected by construction)
def hvp(model: SpinModel, m: np.ndarray, V: np.ndarray) -> np.ndarray:
    Ht, Bm = tangent_hessian(model, m, dense=False)
    k = V.shape[0]
    Vf = V.reshape(k, -1).T  # 3N x k
    out = Bm @ (Ht @ (Bm.T @ Vf))
    return np.ascontiguousarray(out.T).reshape(k, model.N, 3)


# ---- O10 reflected-force MMF step with renormalisation retraction
def mmf_force(model: SpinModel, m: np.ndarray, v: np.ndarray) -> np.ndarray:
    """F_mmf = F - 2 sum_a (F.v_a) v_a with F = -P g (Eq. 2; subspace variant for kr > 1)."""
    F = -projected_gradient(model, m)
    out = F.copy()
    for a in range(v.shape[0]):
        out -= 2.0 * np.sum(F * v[a]) * v[a]
    return out


def mmf_step(model: SpinModel, m: np.ndarray, v: np.ndarray, dt: float) -> np.ndarray:
    x = m + dt * mmf_force(model, m, v)
    return x / np.linalg.norm(x, axis=1, keepdims=True)


# ---- O11 the spectral transformation the GPU solver runs LOBPCG on (a solver device, not in the paper: DESIGN.md 5):
#      -p_d(H_t), p_d(x) = T_d(l(x)) / T_d(l(a_L)),  l(x) = (2x - a - b)/(b - a),  T_d the Chebyshev polynomial.
#      Written here as the DEFINITION through the dense eigen-decomposition (no three-term recurrence).
def chebyshev_T(d: int, x: np.ndarray) -> np.ndarray:
    x = np.asarray(x, dtype=np.float64)
    out = np.empty_like(x)
    inside = np.abs(x) <= 1.0
    out[inside] = np.cos(d * np.arccos(x[inside]))
    xo = x[~inside]
    out[~inside] = np.sign(xo) ** d * np.cosh(d * np.arccosh(np.abs(xo)))
    return out


def transformed_operator_apply(model: SpinModel, m: np.ndarray, V: np.ndarray, d: int, a: float, b: float, a_L: float):
    """-p_d(Hess) V for tangent-projected V ([k][N][3]), via eigh of the explicit tangent Hessian."""
    Ht, Bm = tangent_hessian(model, m, dense=True)
    lam, Y = scipy.linalg.eigh(0.5 * (Ht + Ht.T))
    ell = lambda x: (2.0 * x - a - b) / (b - a)
    pl = chebyshev_T(d, ell(lam)) / chebyshev_T(d, np.array([ell(a_L)]))[0]
    k = V.shape[0]
    coeff = Y.T @ (Bm.T @ V.reshape(k, -1).T)            # 2N x k
    out = -(Bm @ (Y @ (pl[:, None] * coeff)))
    return np.ascontiguousarray(out.T).reshape(k, model.N, 3)


# ---- O12 outer MMF loop with the paper's termination test (Alg. 1 l.9-14), fixed step dt
def mmf_run(model: SpinModel, m: np.ndarray, k: int, dt: float, max_steps: int, tau_F: float):
    """repeat: lowest-k modes (dense eigh) -> F_mmf with v_1 -> stop if |F_mmf| <= tau_F and lam_1 < 0 < lam_2 -> step.
    Returns (m, lam, steps applied, converged, |F_mmf| at the returned state)."""
    m = m.copy()
    for step in range(max_steps + 1):
        lam, V = lowest_modes(model, m, k)
        F = mmf_force(model, m, V[:1])
        fn = float(np.linalg.norm(F))
        if fn <= tau_F and lam[0] < 0.0 < lam[1]:
            return m, lam, step, True, fn
        if step == max_steps:
            return m, lam, step, False, fn
        m = mmf_step(model, m, V[:1], dt)
