"""GPU parity tests (spin lattice): the CUDA path, called through the C ABI, against the CPU oracle on the
same seeded inputs.  Tolerances are BASELINE.json north_star's: HVP relative L2 <= 1e-11, eigenvalues
relative <= 1e-8, lowest-k subspace principal angle <= 1e-6."""
import numpy as np
import pytest
import scipy.linalg

from oracle import spin_oracle as so
from paper_2509_26269_b200 import workloads as wl

pytestmark = pytest.mark.gpu

HVP_TOL = 1e-11
EIG_TOL = 1e-8
ANGLE_TOL = 1e-6


def model_of(w):
    return so.SpinModel(w.Lx, w.Ly, w.pbc_x, w.pbc_y, w.J, w.D, w.K, w.B, w.mu)


def dev(a):
    import torch
    return torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64).cuda()


def rel_l2(a, b):
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


def custom(Lx, Ly, px, py, seed, B=(0.01, -0.02, 0.03), k=2):
    m = wl.random_spins(Lx, Ly, seed)
    return wl.SpinWorkload(f"rand{Lx}x{Ly}", Lx, Ly, px, py, 1.0, 0.3, 0.05, B, 1.0, k, seed, m)


CASES = [
    lambda: wl.config0(),
    lambda: wl.config1(),
    lambda: custom(37, 23, 0, 0, 1),    # odd sizes, open, ragged tail
    lambda: custom(64, 50, 1, 0, 2),    # mixed boundaries
    lambda: custom(130, 70, 0, 1, 3),   # spans several tiles
    lambda: custom(1, 1, 0, 0, 4),      # degenerate: single spin
    lambda: custom(2, 3, 1, 1, 5),      # tiny periodic (neighbours alias)
    lambda: wl.config3_scaled(100),
]


@pytest.mark.parametrize("case", range(len(CASES)))
def test_energy_grad_parity(moto, case):
    w = CASES[case]()
    model = model_of(w)
    ctx = moto.spin_context(w)
    E, g = ctx.energy_grad(dev(w.spins))
    E_ref = so.energy(model, w.spins)
    g_ref = so.projected_gradient(model, w.spins)
    assert abs(E.item() - E_ref) <= 1e-12 * max(1.0, abs(E_ref))
    assert np.max(np.abs(g.cpu().numpy() - g_ref)) <= 1e-12


@pytest.mark.parametrize("case", range(len(CASES)))
@pytest.mark.parametrize("k", [1, 2, 6])
def test_hvp_parity(moto, case, k):
    w = CASES[case]()
    model = model_of(w)
    ctx = moto.spin_context(w, kmax=8)
    V = wl.random_block(w.N, k, seed=100 + case)       # NOT tangent: the call must project
    HV = ctx.hvp(dev(w.spins), dev(V)).cpu().numpy()
    ref = so.hvp(model, w.spins, V)
    assert rel_l2(HV, ref) <= HVP_TOL
    assert np.max(np.abs(np.sum(HV * w.spins[None], axis=2))) <= 1e-12   # tangent output


# lattices for the TMA-staged K1 path (even Lx >= 8), forced on with hvp_path=2 so that oracle-sized cases run it:
# several strips + ragged last strip, every boundary combination, segments shorter than a chunk, tiny Ly.
TMA_CASES = [
    lambda: wl.config0(),                 # 8x8 periodic: one strip, both wrap side boxes, Ly == chunk
    lambda: wl.config1(),                 # 70x70 periodic: two strips
    lambda: custom(64, 50, 1, 0, 2),      # periodic x, open y
    lambda: custom(130, 70, 0, 1, 3),     # open x, periodic y, three strips
    lambda: custom(126, 41, 0, 0, 6),     # open, strip boundary at a multiple of 62 + 2
    lambda: custom(200, 9, 1, 1, 7),      # rows barely more than one chunk
    lambda: custom(62, 3, 1, 1, 8),       # Ly = 3: wrapped halo rows alias the segment's own rows
    lambda: custom(10, 2, 1, 1, 9),       # Ly = 2
    lambda: custom(250, 130, 1, 1, 10),   # > 148 segments' worth of work: CTAs span strip boundaries
    lambda: wl.config3_scaled(100),
]


@pytest.mark.parametrize("case", range(len(TMA_CASES)))
@pytest.mark.parametrize("k", [1, 2, 3, 5, 6])      # k >= 4: all column pairs in one launch (+ a single-column launch for odd k)
def test_hvp_tma_parity(moto, case, k):
    w = TMA_CASES[case]()
    model = model_of(w)
    ctx = moto.spin_context(w, kmax=8)
    ctx.set_solver(hvp_path=2)
    V = wl.random_block(w.N, k, seed=200 + case)
    HV = ctx.hvp(dev(w.spins), dev(V)).cpu().numpy()
    ref = so.hvp(model, w.spins, V)
    assert rel_l2(HV, ref) <= HVP_TOL
    assert np.max(np.abs(np.sum(HV * w.spins[None], axis=2))) <= 1e-12
    # generic path on the same input: the two CUDA kernels agree to rounding
    ctx.set_solver(hvp_path=1)
    HV1 = ctx.hvp(dev(w.spins), dev(V)).cpu().numpy()
    assert rel_l2(HV, HV1) <= 1e-13


@pytest.mark.parametrize("case", range(len(TMA_CASES)))
def test_energy_grad_tma_parity(moto, case):
    # moto_energy_grad through the TMA-staged kernel (energy / gradient mode: only m in the ring) against the oracle, and
    # against the generic kernel; E alone and g alone take the same path
    w = TMA_CASES[case]()
    model = model_of(w)
    ctx = moto.spin_context(w)
    ctx.set_solver(hvp_path=2)
    n0 = ctx.launch_count
    E, g = ctx.energy_grad(dev(w.spins))
    assert ctx.launch_count - n0 == 1                       # one launch: the CTA that finishes last sums the energy partials
    E_ref = so.energy(model, w.spins)
    g_ref = so.projected_gradient(model, w.spins)
    assert abs(E.item() - E_ref) <= 1e-12 * max(1.0, abs(E_ref))
    assert np.max(np.abs(g.cpu().numpy() - g_ref)) <= 1e-12
    for _ in range(3):                                      # the arrival counter is left at 0: repeated calls, bit-identical
        E2, none = ctx.energy_grad(dev(w.spins), want_grad=False)
        assert none is None and E2.item() == E.item()
    ctx.set_solver(hvp_path=1)
    E1, g1 = ctx.energy_grad(dev(w.spins))
    assert abs(E1.item() - E.item()) <= 1e-13 * max(1.0, abs(E_ref)) and np.max(np.abs((g1 - g).cpu().numpy())) <= 1e-13


@pytest.mark.parametrize("case", [0, 1, 2, 3, 5, 8])
def test_lowest_modes_tma_path(moto, case):
    # solver mode of the TMA kernel (c given, fused V^T HV partials) inside the LOBPCG
    w = TMA_CASES[case]()
    if w.N > 12000:
        pytest.skip("dense oracle too large")
    lam_ref, V_ref = so.lowest_modes(model_of(w), w.spins, 2, extra=1)
    ctx = moto.spin_context(w)
    ctx.set_solver(hvp_path=2)
    lam, V, info = ctx.lowest_modes(dev(w.spins), 2, tol=1e-9, max_iter=4000)
    assert info["converged"], info
    lam = lam.cpu().numpy()
    assert np.max(np.abs(lam - lam_ref[:2]) / np.maximum(np.abs(lam_ref[:2]), 1e-3)) <= EIG_TOL
    if lam_ref[2] - lam_ref[1] > 1e-3:
        ang = scipy.linalg.subspace_angles(V.cpu().numpy().reshape(2, -1).T, V_ref[:2].reshape(2, -1).T)
        assert ang.max() <= ANGLE_TOL


def test_hvp_kmax_and_arg_errors(moto):
    w = wl.config0()
    ctx = moto.spin_context(w, kmax=8)
    V = wl.random_block(w.N, 8, seed=7)
    HV = ctx.hvp(dev(w.spins), dev(V)).cpu().numpy()
    assert rel_l2(HV, so.hvp(model_of(w), w.spins, V)) <= HVP_TOL
    import torch
    with pytest.raises(moto.MotoError):
        ctx.hvp(dev(w.spins), dev(wl.random_block(w.N, 9, seed=7)))
    with pytest.raises(moto.MotoError):
        v = dev(V)
        ctx.hvp(dev(w.spins), v, out=v)


def test_gram_parity(moto):
    w = custom(50, 41, 1, 1, 9)
    ctx = moto.spin_context(w, kmax=8)
    S = wl.random_block(w.N, 6, seed=1)
    T = wl.random_block(w.N, 12, seed=2)
    G = ctx.gram(dev(S), dev(T)).cpu().numpy()
    ref = S.reshape(6, -1) @ T.reshape(12, -1).T
    assert np.max(np.abs(G - ref)) <= 1e-11 * np.max(np.abs(ref)) + 1e-10


@pytest.mark.parametrize("n,nev", [(3, 1), (6, 2), (9, 3), (18, 6), (24, 8)])
def test_rayleigh_ritz_vs_lapack(moto, n, nev):
    rng = np.random.default_rng(n)
    Q = rng.standard_normal((n, n))
    GB = Q @ Q.T + 0.1 * np.eye(n)
    GA = rng.standard_normal((n, n)); GA = GA + GA.T
    w = wl.config0()
    ctx = moto.spin_context(w, kmax=8)
    th, Cm = ctx.rayleigh_ritz(dev(GA), dev(GB), nev)
    th, Cm = th.cpu().numpy(), Cm.cpu().numpy()
    ref, Y = scipy.linalg.eigh(GA, GB)
    assert np.max(np.abs(th - ref[:nev])) <= 1e-11 * np.max(np.abs(ref))
    assert np.max(np.abs(Cm.T @ GB @ Cm - np.eye(nev))) <= 1e-11
    assert np.max(np.abs(Cm.T @ GA @ Cm - np.diag(th))) <= 1e-10 * np.max(np.abs(ref))


def test_rayleigh_ritz_drops_null_directions(moto):
    # rank-deficient G_B (duplicate + zero basis vectors), as on the first LOBPCG iteration (P = 0)
    rng = np.random.default_rng(0)
    S = rng.standard_normal((40, 6)); S[:, 4] = 0.0; S[:, 5] = S[:, 1]
    Aop = rng.standard_normal((40, 40)); Aop = Aop + Aop.T
    GA, GB = S.T @ Aop @ S, S.T @ S
    w = wl.config0()
    ctx = moto.spin_context(w, kmax=8)
    th, Cm = ctx.rayleigh_ritz(dev(GA), dev(GB), 2)
    Sr = S[:, :4]
    ref = scipy.linalg.eigh(Sr.T @ Aop @ Sr, Sr.T @ Sr, eigvals_only=True)
    assert np.max(np.abs(th.cpu().numpy() - ref[:2])) <= 1e-10 * np.max(np.abs(ref))


@pytest.mark.parametrize("n,nbad", [(18, 3), (21, 1), (24, 6), (9, 2), (15, 0)])
def test_rayleigh_ritz_wide_pencils_rank_deficient(moto, n, nbad):
    # n > 8 takes the one-thread-per-entry path: Cholesky whitening when G_B is well conditioned, the truncating
    # eigen-decomposition when it is not (nbad dependent basis vectors: zero columns and duplicates)
    rng = np.random.default_rng(100 + n)
    S = rng.standard_normal((60, n))
    for b in range(nbad):
        if b % 2 == 0: S[:, n - 1 - b] = 0.0
        else: S[:, n - 1 - b] = S[:, b] * 1.5
    Aop = rng.standard_normal((60, 60)); Aop = Aop + Aop.T
    GA, GB = S.T @ Aop @ S, S.T @ S
    nev = n // 3
    w = wl.config0()
    ctx = moto.spin_context(w, kmax=8)
    th, Cm = ctx.rayleigh_ritz(dev(GA), dev(GB), nev)
    th, Cm = th.cpu().numpy(), Cm.cpu().numpy()
    Sr = S[:, :n - nbad]
    ref = scipy.linalg.eigh(Sr.T @ Aop @ Sr, Sr.T @ Sr, eigvals_only=True)
    assert np.max(np.abs(th - ref[:nev])) <= 1e-10 * np.max(np.abs(ref))
    assert np.max(np.abs(Cm.T @ GB @ Cm - np.eye(nev))) <= 1e-10
    assert np.max(np.abs(Cm.T @ GA @ Cm - np.diag(th))) <= 1e-9 * np.max(np.abs(ref))


def _check_modes(w, lam, V, lam_ref, V_ref, k):
    lam = lam.cpu().numpy(); V = V.cpu().numpy()
    relerr = np.abs(lam - lam_ref[:k]) / np.maximum(np.abs(lam_ref[:k]), 1e-3)
    assert relerr.max() <= EIG_TOL, (lam, lam_ref)
    ang = scipy.linalg.subspace_angles(V.reshape(k, -1).T, V_ref[:k].reshape(k, -1).T)
    assert ang.max() <= ANGLE_TOL, ang
    G = V.reshape(k, -1) @ V.reshape(k, -1).T
    assert np.max(np.abs(G - np.eye(k))) <= 1e-10
    assert np.max(np.abs(np.sum(V * w.spins[None], axis=2))) <= 1e-10
    for a in range(k):   # sign convention: largest-|component| entry positive
        f = V[a].ravel()
        assert f[np.argmax(np.abs(f))] > 0


def test_lowest_modes_cfg0(moto):
    w = wl.config0()
    lam_ref, V_ref = so.lowest_modes(model_of(w), w.spins, 2, extra=1)
    ctx = moto.spin_context(w)
    lam, V, info = ctx.lowest_modes(dev(w.spins), 2, tol=1e-9, max_iter=500)
    assert info["converged"] and max(info["resid"]) <= 1e-9
    _check_modes(w, lam, V, lam_ref, V_ref, 2)
    # oracle-side residual of the GPU pair
    HV = so.hvp(model_of(w), w.spins, V.cpu().numpy())
    for a in range(2):
        assert np.linalg.norm(HV[a] - lam[a].item() * V[a].cpu().numpy()) <= 2e-9


def test_lowest_modes_cfg1(moto):
    w = wl.config1()
    lam_ref, V_ref = so.lowest_modes(model_of(w), w.spins, 2, extra=1)
    ctx = moto.spin_context(w)
    lam, V, info = ctx.lowest_modes(dev(w.spins), 2, tol=1e-9, max_iter=2000)
    assert info["converged"], info
    _check_modes(w, lam, V, lam_ref, V_ref, 2)


def test_lowest_modes_guard_and_warm_start(moto):
    w = wl.config1(L=40)
    lam_ref, V_ref = so.lowest_modes(model_of(w), w.spins, 3, extra=1)
    ctx = moto.spin_context(w, kmax=6)
    ctx.set_solver(guard=3)
    lam, V, info = ctx.lowest_modes(dev(w.spins), 3, tol=1e-9, max_iter=2000)
    assert info["converged"]
    _check_modes(w, lam, V, lam_ref, V_ref, 3)
    # warm start from the converged block: converges at once
    lam2, V2, info2 = ctx.lowest_modes(dev(w.spins), 3, tol=1e-8, max_iter=50, V0=V)
    assert info2["converged"] and info2["iters"] <= 2
    _check_modes(w, lam2, V2, lam_ref, V_ref, 3)


def test_lowest_modes_not_converged_status(moto):
    w = wl.config1(L=40)
    ctx = moto.spin_context(w)
    with pytest.raises(moto.MotoError) as e:
        ctx.lowest_modes(dev(w.spins), 2, tol=1e-12, max_iter=3)
    assert e.value.status == moto.ENOTCONV
    lam, V, info = ctx.lowest_modes(dev(w.spins), 2, tol=1e-12, max_iter=3, allow_notconv=True)
    assert not info["converged"] and info["iters"] == 3 and np.isfinite(lam.cpu().numpy()).all()


def test_ferromagnet_degenerate_pair(moto):
    # uniform +z: lowest eigenvalue 2K+B exactly doubly degenerate -> compare the 2-d subspace
    w = wl.config0(sigma=0.0)
    ctx = moto.spin_context(w)
    lam, V, info = ctx.lowest_modes(dev(w.spins), 2, tol=1e-10, max_iter=500)
    assert np.allclose(lam.cpu().numpy(), 0.12, atol=1e-9)


def test_mmf_step_parity(moto):
    for w in (wl.config0(), wl.config1(L=30), custom(37, 23, 0, 0, 1)):
        model = model_of(w)
        _, V_ref = so.lowest_modes(model, w.spins, 2)
        ctx = moto.spin_context(w)
        for kr in (1, 2):
            out, fn = ctx.mmf_step(dev(w.spins), dev(V_ref[:kr]), 0.05)
            ref = so.mmf_step(model, w.spins, V_ref[:kr], 0.05)
            assert np.max(np.abs(out.cpu().numpy() - ref)) <= 1e-13
            assert abs(fn.item() - np.linalg.norm(so.mmf_force(model, w.spins, V_ref[:kr]))) <= 1e-12
        # in place
        s = dev(w.spins)
        ctx.mmf_step(s, dev(V_ref[:1]), 0.05, out=s)
        assert np.max(np.abs(s.cpu().numpy() - so.mmf_step(model, w.spins, V_ref[:1], 0.05))) <= 1e-13


@pytest.mark.parametrize("case", range(len(TMA_CASES)))
def test_mmf_step_tma_parity(moto, case):
    # moto_mmf_step with one mode: pass 1 (F = -P g, alpha = F . v) through the TMA-staged kernel, |F_mmf| out of pass 2 itself (two
    # launches in all); a random tangent unit vector stands for v (the step is defined for any v); in place; repeated calls
    w = TMA_CASES[case]()
    model = model_of(w)
    v = wl.random_block(w.N, 2, seed=700 + case)
    v = v - np.sum(v * w.spins[None], axis=2, keepdims=True) * w.spins[None]
    v /= np.linalg.norm(v.reshape(2, -1), axis=1)[:, None, None]
    ctx = moto.spin_context(w)
    ctx.set_solver(hvp_path=2)
    for kr in (1, 2):
        n0 = ctx.launch_count
        out, fn = ctx.mmf_step(dev(w.spins), dev(v[:kr]), 0.05)
        assert ctx.launch_count - n0 == 2
        ref = so.mmf_step(model, w.spins, v[:kr], 0.05)
        assert np.max(np.abs(out.cpu().numpy() - ref)) <= 1e-13
        fref = np.linalg.norm(so.mmf_force(model, w.spins, v[:kr]))
        assert abs(fn.item() - fref) <= 1e-12 * max(1.0, fref)
        out2, fn2 = ctx.mmf_step(dev(w.spins), dev(v[:kr]), 0.05)          # arrival counters back at 0: bit-identical
        assert np.array_equal(out.cpu().numpy(), out2.cpu().numpy()) and fn.item() == fn2.item()
    s = dev(w.spins)
    ctx.mmf_step(s, dev(v[:1]), 0.05, out=s)
    assert np.max(np.abs(s.cpu().numpy() - so.mmf_step(model, w.spins, v[:1], 0.05))) <= 1e-13


def test_transport(moto):
    w = wl.config1(L=30)
    model = model_of(w)
    _, V = so.lowest_modes(model, w.spins, 2)
    m2 = so.mmf_step(model, w.spins, V[:1], 0.05)
    ctx = moto.spin_context(w)
    Vt = ctx.transport(dev(m2), dev(V)).cpu().numpy()
    assert np.max(np.abs(np.sum(Vt * m2[None], axis=2))) <= 1e-13
    G = Vt.reshape(2, -1) @ Vt.reshape(2, -1).T
    assert np.max(np.abs(G - np.eye(2))) <= 1e-12
    Pv = V - np.sum(V * m2[None], 2, keepdims=True) * m2[None]
    ang = scipy.linalg.subspace_angles(Vt.reshape(2, -1).T, Pv.reshape(2, -1).T)
    assert ang.max() <= 1e-10


def test_host_variants(moto):
    w = wl.config1(L=30)
    model = model_of(w)
    ctx = moto.spin_context(w)
    E, g = ctx.energy_grad_host(w.spins, np.zeros_like(w.spins))
    assert abs(E - so.energy(model, w.spins)) <= 1e-12 * abs(E)
    assert np.max(np.abs(g - so.projected_gradient(model, w.spins))) <= 1e-12
    V = wl.random_block(w.N, 2, seed=3)
    HV = ctx.hvp_host(w.spins, V, np.zeros_like(V))
    assert rel_l2(HV, so.hvp(model, w.spins, V)) <= HVP_TOL
    lam = np.zeros(2); Vh = np.zeros((2, w.N, 3))
    info = ctx.lowest_modes_host(w.spins, 2, 1e-9, 2000, lam, Vh)
    lam_ref, V_ref = so.lowest_modes(model, w.spins, 2)
    assert info["converged"] and np.max(np.abs(lam - lam_ref)) <= 1e-8 * np.max(np.abs(lam_ref))
    out, fn = ctx.mmf_step_host(w.spins, V_ref[:1], 0.05, np.zeros_like(w.spins))
    assert np.max(np.abs(out - so.mmf_step(model, w.spins, V_ref[:1], 0.05))) <= 1e-13


def test_determinism(moto):
    w = wl.config1(L=40)
    ctx = moto.spin_context(w)
    a = ctx.lowest_modes(dev(w.spins), 2, tol=1e-8, max_iter=1000)
    b = ctx.lowest_modes(dev(w.spins), 2, tol=1e-8, max_iter=1000)
    assert np.array_equal(a[0].cpu().numpy(), b[0].cpu().numpy())
    assert np.array_equal(a[1].cpu().numpy(), b[1].cpu().numpy())
    assert ctx.launch_count > 0


# ---------------------------------------------------------------- full size: BASELINE.json configs[3], the bench configuration
@pytest.fixture(scope="module")
def cfg3_full():
    return wl.config3()


def _golden_eigs(L):
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "cfg3_lowest_eigs.txt")
    for line in open(path):
        if line.startswith(f"L={L} "):
            return np.array([float(x) for x in line.split()[2:]])
    raise KeyError(L)


def test_cfg3_full_size_hvp_parity(moto, cfg3_full):
    # the launch configuration bench.py times (TMA path, k = 2, 10^6 spins) against the oracle's explicit sparse Hessian
    w = cfg3_full
    ctx = moto.spin_context(w, kmax=2)
    V = wl.random_block(w.N, 2, seed=33)
    HV = ctx.hvp(dev(w.spins), dev(V)).cpu().numpy()
    ref = so.hvp(model_of(w), w.spins, V)
    assert rel_l2(HV, ref) <= HVP_TOL
    assert np.max(np.abs(HV - ref)) <= 1e-11 * np.max(np.abs(ref))


def test_cfg3_full_size_lowest_modes_vs_golden(moto, cfg3_full):
    # eigenvalues against the oracle's ARPACK shift-invert values stored by tests/golden/make_cfg3_eigs.py;
    # lambda_3 - lambda_2 = 1.0e-4, so the subspace test is the oracle-side residual (reading A10), not an angle
    w = cfg3_full
    gold = _golden_eigs(1000)
    ctx = moto.spin_context(w, kmax=2)
    lam, V, info = ctx.lowest_modes(dev(w.spins), 2, tol=1e-6, max_iter=20000)
    assert info["converged"], info
    lam = lam.cpu().numpy(); V = V.cpu().numpy()
    assert np.max(np.abs(lam - gold[:2]) / np.abs(gold[:2])) <= EIG_TOL, (lam, gold[:2])
    HV = so.hvp(model_of(w), w.spins, V)
    for a in range(2):
        assert np.linalg.norm(HV[a] - lam[a] * V[a]) <= 1e-6 * (1 + 1e-3)      # the stated tol; 1e-3 for the oracle's own rounding
    assert np.max(np.abs(V.reshape(2, -1) @ V.reshape(2, -1).T - np.eye(2))) <= 1e-10
    assert np.max(np.abs(np.sum(V * w.spins[None], axis=2))) <= 1e-10


def test_cfg3_scaled_316_vs_golden(moto):
    w = wl.config3_scaled(316)
    gold = _golden_eigs(316)
    ctx = moto.spin_context(w, kmax=2)
    lam, V, info = ctx.lowest_modes(dev(w.spins), 2, tol=1e-7, max_iter=20000)
    assert info["converged"], info
    assert np.max(np.abs(lam.cpu().numpy() - gold[:2]) / np.abs(gold[:2])) <= EIG_TOL


@pytest.mark.parametrize("case", [1, 2, 3, 5, 6, 8])
@pytest.mark.parametrize("path", [1, 2])
def test_hvp_three_term_parity(moto, case, path):
    # the recurrence step of the transformed solver: out = alpha (Hess[V] - c0 V) + beta U, tangent V, solver mode
    w = TMA_CASES[case]()
    model = model_of(w)
    ctx = moto.spin_context(w, kmax=8)
    ctx.set_solver(hvp_path=path)
    rng = np.random.default_rng(case)
    for k in (1, 2, 3, 5):                    # 5 on the TMA path: two pairs in one grouped launch + a single-column launch
        V = wl.random_block(w.N, k, seed=300 + case)
        V = V - np.sum(V * w.spins[None], axis=2, keepdims=True) * w.spins[None]     # tangent input
        U = wl.random_block(w.N, k, seed=400 + case)
        alpha, c0, beta = rng.uniform(-2, 2), rng.uniform(-1, 20), rng.uniform(-2, 2)
        HV = so.hvp(model, w.spins, V)
        ref = alpha * (HV - c0 * V) + beta * U
        out = ctx.hvp_three_term(dev(w.spins), dev(V), alpha, c0, beta, U=dev(U)).cpu().numpy()
        assert rel_l2(out, ref) <= HVP_TOL
        # no operand, cached c
        out2 = ctx.hvp_three_term(dev(w.spins), dev(V), alpha, c0, 0.0, refresh_c=False).cpu().numpy()
        assert rel_l2(out2, alpha * (HV - c0 * V)) <= HVP_TOL
        # in place over the operand (what the solver does from the third step on)
        Ud = dev(U)
        ctx.hvp_three_term(dev(w.spins), dev(V), alpha, c0, beta, U=Ud, out=Ud, refresh_c=False)
        assert rel_l2(Ud.cpu().numpy(), ref) <= HVP_TOL


@pytest.mark.parametrize("case", range(len(TMA_CASES)))
def test_multistep_recurrence_matches_the_stepwise_one(moto, case):
    # The three ways the degree-d recurrence is launched (moto_solver_opts.cheb_mode): 3 = two steps per pass with the
    # intermediate step kept in shared memory and a redundantly computed halo ring (spin_cheb2_tma.cu; plus one single
    # step when d is odd), 1 = one step per pass in one cooperative launch (neighbour-flag synchronisation, every second
    # step swept bottom-up on the point-reflected stencil), 2 = d dependent launches.  Same arithmetic per site up to the
    # summation order inside the stencil of a reversed sweep, so agreement to rounding, and the same solve.
    w = TMA_CASES[case]()
    outs, sols = {}, {}
    for mode in (1, 2, 3):
        ctx = moto.spin_context(w)
        ctx.set_solver(hvp_path=2, precond_degree=24, cheb_mode=mode)
        for k in (1, 2):
            V = wl.random_block(w.N, k, seed=77 + k)
            V = V - np.sum(V * w.spins[None], axis=2, keepdims=True) * w.spins[None]
            for d in (2, 3, 24, 25):
                outs[mode, k, d] = ctx.cheb_apply(dev(w.spins), dev(V), d, -0.1, 18.6, -0.16).cpu().numpy()
        if w.N >= 400:
            lam, Vm, info = ctx.lowest_modes(dev(w.spins), 2, tol=1e-8, max_iter=400, allow_notconv=True)
            sols[mode] = (lam.cpu().numpy(), info)
    for (mode, k, d), o in outs.items():
        assert np.isfinite(o).all()
        assert rel_l2(o, outs[2, k, d]) <= 1e-13, (mode, k, d, rel_l2(o, outs[2, k, d]))
    for mode in sols:
        assert sols[mode][1]["converged"] == sols[2][1]["converged"]
        assert np.max(np.abs(sols[mode][0] - sols[2][0])) <= 1e-9 * np.max(np.abs(sols[2][0]))


@pytest.mark.parametrize("path", [1, 2])
def test_lowest_mode_k1_and_zero_iterations(moto, path):
    # block size 1 (the paper's default single minimum mode) on both K1 paths; max_iter = 0 returns the
    # Rayleigh-Ritz of the start block with ENOTCONV and finite outputs
    w = wl.config1(L=40)
    lam_ref, V_ref = so.lowest_modes(model_of(w), w.spins, 1, extra=1)
    ctx = moto.spin_context(w)
    ctx.set_solver(hvp_path=path)
    lam, V, info = ctx.lowest_modes(dev(w.spins), 1, tol=1e-9, max_iter=4000)
    assert info["converged"], info
    assert abs(lam.item() - lam_ref[0]) <= EIG_TOL * abs(lam_ref[0])
    ang = scipy.linalg.subspace_angles(V.cpu().numpy().reshape(1, -1).T, V_ref[:1].reshape(1, -1).T)
    assert ang.max() <= ANGLE_TOL
    lam0, V0, info0 = ctx.lowest_modes(dev(w.spins), 1, tol=1e-9, max_iter=0, allow_notconv=True)
    assert not info0["converged"] and info0["iters"] == 0 and np.isfinite(lam0.cpu().numpy()).all()


CHEB_CASES = [lambda: wl.config0(), lambda: custom(24, 16, 1, 0, 21), lambda: custom(62, 10, 0, 1, 22), lambda: custom(130, 6, 1, 1, 23)]


@pytest.mark.parametrize("case", range(len(CHEB_CASES)))
@pytest.mark.parametrize("d", [1, 2, 3, 8, 40, 128, 256])
def test_cheb_apply_parity(moto, case, d):
    # the transformed operator -p_d(Hess) of the solver (one persistent multi-step launch for d >= 2) against its
    # definition through the oracle's dense eigen-decomposition (lattices small enough for a full dense eigh).  The library
    # applies the filter in product form over its Leja-ordered roots: d = 40 .. 256 (the largest degree allowed) are the cases
    # where any other root order loses every digit
    w = CHEB_CASES[case]()
    model = model_of(w)
    ctx = moto.spin_context(w, kmax=2)
    ctx.set_solver(hvp_path=2)
    lam_ref, _ = so.lowest_modes(model, w.spins, 2)
    a, b, aL = lam_ref[1] + 0.05, lam_ref[1] + 25.0, lam_ref[0]
    for k in (1, 2):
        V = wl.random_block(w.N, k, seed=500 + case)
        V = V - np.sum(V * w.spins[None], axis=2, keepdims=True) * w.spins[None]
        out = ctx.cheb_apply(dev(w.spins), dev(V), d, a, b, aL).cpu().numpy()
        ref = so.transformed_operator_apply(model, w.spins, V, d, a, b, aL)
        assert rel_l2(out, ref) <= 1e-10, rel_l2(out, ref)


def test_transformed_generic_path_kb_gt_2(moto):
    # block sizes above 2 (guard columns) on the transformed operator: opt-in through precond_degree > 0
    w = wl.config1(L=40)
    lam_ref, V_ref = so.lowest_modes(model_of(w), w.spins, 3, extra=1)
    ctx = moto.spin_context(w, kmax=5)
    ctx.set_solver(guard=2, hvp_path=2, precond_degree=16)
    lam, V, info = ctx.lowest_modes(dev(w.spins), 3, tol=1e-9, max_iter=2000)
    assert info["converged"], info
    _check_modes(w, lam, V, lam_ref, V_ref, 3)


@pytest.mark.parametrize("case,k,kmax", [(lambda: custom(64, 50, 1, 0, 2), 4, 4), (lambda: custom(70, 40, 0, 1, 3), 3, 3),
                                         (lambda: wl.config1(L=40), 6, 6)])
def test_generic_path_transformed_default(moto, case, k, kmax):
    # block sizes above 2 where the TMA K1 applies run on -p_32(A) by default (soft locking, A-residual test every second
    # iteration); precond_degree = -1 is plain LOBPCG.  Both against the dense oracle.
    w = case()
    lam_ref, V_ref = so.lowest_modes(model_of(w), w.spins, k, extra=1)
    res = {}
    for name, deg in (("default", 0), ("d16", 16), ("plain", -1)):
        ctx = moto.spin_context(w, kmax=kmax)
        ctx.set_solver(hvp_path=2, precond_degree=deg)
        lam, V, info = ctx.lowest_modes(dev(w.spins), k, tol=1e-9, max_iter=20000)
        assert info["converged"], (name, info)
        _check_modes(w, lam, V, lam_ref, V_ref, k)
        res[name] = info
    assert res["plain"]["hvp_count"] == kmax * (res["plain"]["iters"] + 1)      # plain: one HVP per column and iteration
    assert res["default"]["hvp_count"] > kmax * (res["default"]["iters"] + 2) and res["default"]["iters"] < res["plain"]["iters"]


@pytest.mark.parametrize("deg", [16, 32, 64])
def test_transformed_guard_columns_on_a_dense_spectrum(moto, deg):
    # random spins, k = 3 with two guard columns: before soft locking and the interval above the whole block (a = theta_kb +
    # margin) degree 32 bounced between 1e-9 and 1e-2 for thousands of iterations; the oracle recomputes the residuals
    w = custom(70, 40, 0, 1, 3)
    model = model_of(w)
    lam_ref, V_ref = so.lowest_modes(model, w.spins, 3, extra=1)
    ctx = moto.spin_context(w, kmax=5)
    ctx.set_solver(guard=2, hvp_path=2, precond_degree=deg)
    lam, V, info = ctx.lowest_modes(dev(w.spins), 3, tol=1e-9, max_iter=400)
    assert info["converged"] and info["iters"] <= 60, info
    _check_modes(w, lam, V, lam_ref, V_ref, 3)
    Vh, lh = V.cpu().numpy(), lam.cpu().numpy()
    R = so.hvp(model, w.spins, Vh) - lh[:, None, None] * Vh
    assert np.max(np.linalg.norm(R.reshape(3, -1), axis=1)) <= 1e-9 * (1 + 1e-3)


def test_warm_started_resolve_kb6_transformed(moto):
    # the re-solve of an MMF loop at block size 6 (warm start, transported block) runs transformed too: same eigenpairs as the
    # plain solver from the same start, in fewer iterations
    w = wl.config1(L=40)
    model = model_of(w)
    x = dev(w.spins)
    out = {}
    for name, deg in (("default", 0), ("plain", -1)):
        ctx = moto.spin_context(w, kmax=6)
        ctx.set_solver(hvp_path=2, precond_degree=deg)
        lam, V, info = ctx.lowest_modes(x, 6, tol=1e-9, max_iter=20000)
        assert info["converged"], (name, info)
        x2, _ = ctx.mmf_step(x, V[:1].contiguous(), 0.05)
        ctx.transport(x2, V)
        lam2, V2, info2 = ctx.lowest_modes(x2, 6, tol=1e-9, max_iter=20000, V0=V)
        assert info2["converged"], (name, info2)
        out[name] = (x2.cpu().numpy(), lam2.cpu().numpy(), V2.cpu().numpy(), info2)
    import dataclasses
    lam_ref, V_ref = so.lowest_modes(model, out["default"][0], 6, extra=1)
    _check_modes(dataclasses.replace(w, spins=out["default"][0]), dev(out["default"][1]), dev(out["default"][2]), lam_ref, V_ref, 6)
    assert out["default"][3]["iters"] < out["plain"][3]["iters"]


@pytest.mark.parametrize("case,k,guard", [(lambda: wl.config1(L=40), 6, 0), (lambda: custom(70, 40, 0, 1, 3), 3, 2),
                                           (lambda: custom(64, 50, 1, 0, 2), 4, 0), (lambda: custom(130, 70, 0, 0, 3), 8, 0)])
def test_grouped_recurrence_launch_equals_pairwise(moto, case, k, guard):
    # block sizes above 2: all column pairs in one two-steps-per-pass launch (cheb_mode auto), each pair on its own CTAs, against
    # one launch per pair of the one-step-per-pass kernel (cheb_mode 1) -- bit for bit; odd block sizes add a single-column launch
    w = case()
    out = {}
    for mode in (0, 1):
        ctx = moto.spin_context(w, kmax=k + guard)
        ctx.set_solver(guard=guard, hvp_path=2, cheb_mode=mode)
        lam, V, info = ctx.lowest_modes(dev(w.spins), k, tol=1e-9, max_iter=2000)
        assert info["converged"], (mode, info)
        out[mode] = (lam.cpu().numpy(), V.cpu().numpy(), info)
    assert out[0][2]["iters"] == out[1][2]["iters"]
    assert np.array_equal(out[0][0], out[1][0]) and np.array_equal(out[0][1], out[1][1])
    assert out[0][2]["launches"] < out[1][2]["launches"] if "launches" in out[0][2] else True


def test_building_block_argument_errors_and_fallbacks(moto):
    import torch
    w = custom(37, 23, 0, 0, 1)              # odd Lx: the TMA path does not apply
    ctx = moto.spin_context(w, kmax=3)
    x = dev(w.spins)
    V = wl.random_block(w.N, 3, seed=5)
    V = V - np.sum(V * w.spins[None], axis=2, keepdims=True) * w.spins[None]
    # three-term step falls back to the generic kernel and still matches the oracle
    out = ctx.hvp_three_term(x, dev(V), 0.5, 3.0, -0.25, U=dev(V)).cpu().numpy()
    HV = so.hvp(model_of(w), w.spins, V)
    assert rel_l2(out, 0.5 * (HV - 3.0 * V) - 0.25 * V) <= HVP_TOL
    # the transformed operator needs the TMA path: a status code, never a silent CPU fallback
    with pytest.raises(moto.MotoError) as e:
        ctx.cheb_apply(x, dev(V[:2]), 4, -0.1, 18.0, -0.2)
    assert e.value.status == moto.ESTATE
    w2 = wl.config1(L=40)
    ctx2 = moto.spin_context(w2, kmax=2)
    V2 = dev(wl.random_block(w2.N, 2, seed=6))
    for bad in (dict(d=0), dict(d=300), dict(a=-0.3), dict(b=-0.5)):     # degree range, a_L < a < b
        kw = dict(d=4, a=-0.1, b=18.0, a_L=-0.2); kw.update(bad)
        with pytest.raises(moto.MotoError):
            ctx2.cheb_apply(dev(w2.spins), V2, kw["d"], kw["a"], kw["b"], kw["a_L"])
    with pytest.raises(moto.MotoError):
        ctx2.cheb_apply(dev(w2.spins), V2, 4, -0.1, 18.0, -0.2, out=V2)   # aliasing


def test_guard_column_on_the_fused_path(moto):
    # k = 1 with one guard column: block size 2 on the fused (and, with hvp_path=2, transformed) path; only column 0 is returned
    w = wl.config1(L=40)
    lam_ref, V_ref = so.lowest_modes(model_of(w), w.spins, 1, extra=1)
    ctx = moto.spin_context(w, kmax=2)
    ctx.set_solver(guard=1, hvp_path=2)
    lam, V, info = ctx.lowest_modes(dev(w.spins), 1, tol=1e-9, max_iter=3000)
    assert info["converged"], info
    assert V.shape[0] == 1 and abs(lam.item() - lam_ref[0]) <= EIG_TOL * abs(lam_ref[0])
    ang = scipy.linalg.subspace_angles(V.cpu().numpy().reshape(1, -1).T, V_ref[:1].reshape(1, -1).T)
    assert ang.max() <= ANGLE_TOL


def test_mmf_run_outer_loop(moto):
    # moto_mmf_run against the oracle's loop: a few steps on small lattices (the trajectory is only compared while the
    # modes are well separated), and the termination semantics
    w = wl.config1(L=12, R=2.5)
    model = model_of(w)
    m_ref, lam_ref, steps_ref, conv_ref, fn_ref = so.mmf_run(model, w.spins, 2, 0.05, 3, 0.0)
    ctx = moto.spin_context(w, kmax=2)
    x = dev(w.spins)
    V, info = ctx.mmf_run(x, 2, 0.05, 3, 0.0, tol=1e-11, max_iter=5000)
    assert info["steps"] == 3 and not info["converged"] and info["status"] == moto.ENOTCONV
    assert np.max(np.abs(x.cpu().numpy() - m_ref)) <= 1e-7
    assert np.max(np.abs(np.array(info["lam"]) - lam_ref)) <= 1e-7 and abs(info["fnorm"] - fn_ref) <= 1e-6 * fn_ref
    # huge tau_F: a state with lambda_1 < 0 < lambda_2 is accepted at once and left untouched ...
    lam0, _ = so.lowest_modes(model, w.spins, 2)
    if lam0[0] < 0.0 < lam0[1]:
        x2 = dev(w.spins)
        _, info2 = ctx.mmf_run(x2, 2, 0.05, 5, 1e9, tol=1e-9, max_iter=5000)
        assert info2["converged"] and info2["steps"] == 0 and info2["status"] == moto.OK
        assert np.array_equal(x2.cpu().numpy(), w.spins)
    # ... and a state with only positive curvatures never is
    wf = wl.config0(sigma=0.05)
    ctxf = moto.spin_context(wf, kmax=2)
    _, info3 = ctxf.mmf_run(dev(wf.spins), 2, 0.05, 2, 1e9, tol=1e-9, max_iter=2000)
    assert not info3["converged"] and info3["steps"] == 2
    with pytest.raises(moto.MotoError):
        ctx.mmf_run(dev(w.spins), 1, 0.05, 2, 1e-3, tol=1e-9)      # k = 1: no lambda_2


@pytest.mark.parametrize("params", [(-0.7, -0.5, -0.2, (0.3, -0.1, 0.2), 1.7), (0.4, 1.1, 0.3, (0.0, 0.0, -0.5), 0.6)])
def test_other_parameter_signs(moto, params):
    # antiferromagnetic exchange, negative / dominant DMI, easy-plane anisotropy, tilted field, mu != 1: HVP parity on both
    # K1 paths, and the transformed solver (whose upper spectral bound b = max(-c) + lambda_max(L) must hold for any signs)
    J, D, K, B, mu = params
    m = wl.random_spins(40, 30, 11)
    w = wl.SpinWorkload("signs", 40, 30, 1, 0, J, D, K, B, mu, 2, 11, m)
    model = model_of(w)
    V = wl.random_block(w.N, 2, seed=12)
    ref = so.hvp(model, w.spins, V)
    for path in (1, 2):
        ctx = moto.spin_context(w, kmax=2)
        ctx.set_solver(hvp_path=path)
        assert rel_l2(ctx.hvp(dev(w.spins), dev(V)).cpu().numpy(), ref) <= HVP_TOL
        E, g = ctx.energy_grad(dev(w.spins))
        assert abs(E.item() - so.energy(model, w.spins)) <= 1e-12 * abs(so.energy(model, w.spins))
    lam_ref, V_ref = so.lowest_modes(model, w.spins, 2, extra=1)
    lam, Vm, info = ctx.lowest_modes(dev(w.spins), 2, tol=1e-9, max_iter=6000)
    assert info["converged"], info
    assert np.max(np.abs(lam.cpu().numpy() - lam_ref[:2]) / np.maximum(np.abs(lam_ref[:2]), 1e-3)) <= EIG_TOL
    # the bound itself: the whole spectrum lies below max(-c) + lambda_max(L) evaluated by the oracle's pieces
    Ht, _ = so.tangent_hessian(model, w.spins, dense=True)
    lam_max = np.linalg.eigvalsh(0.5 * (Ht + Ht.T))[-1]
    c = so.curvature_scalar(w.spins, so.gradient(model, w.spins))
    Lmax = np.linalg.eigvalsh(so.euclid_hessian(model).toarray())[-1]
    assert lam_max <= np.max(-c) + Lmax + 1e-9


# ---------------------------------------------------------------------------------------------------------------------
# BASELINE.json configs[2] at full size: 256x256 OPEN lattice, two skyrmions, k = 6, then MMF steps with a re-solve per
# step (8(c) "O-sparse (cfg 2, 3)").  65 536 sites takes the TMA K1 path with open boundaries on both
# axes (out-of-range box coordinates zero-fill) and the generic kb > 2 LOBPCG (k_gram_sym, k_update, k_residual, 18x18 pencils).
@pytest.fixture(scope="module")
def cfg2_full():
    w = wl.config2()
    lam_ref, V_ref = so.lowest_modes_sparse(model_of(w), w.spins, 6, extra=2)
    return w, lam_ref, V_ref


def test_cfg2_full_size_hvp_parity_k6(moto, cfg2_full):
    w, _, _ = cfg2_full
    model = model_of(w)
    ctx = moto.spin_context(w, kmax=8)
    V = wl.random_block(w.N, 6, seed=44)               # not tangent: the call projects
    ref = so.hvp(model, w.spins, V)
    for path in (0, 2, 1):                              # auto (= TMA at this size), TMA forced, generic
        ctx.set_solver(hvp_path=path)
        HV = ctx.hvp(dev(w.spins), dev(V)).cpu().numpy()
        assert rel_l2(HV, ref) <= HVP_TOL, path
        assert np.max(np.abs(HV - ref)) <= 1e-11 * np.max(np.abs(ref)), path
        assert np.max(np.abs(np.sum(HV * w.spins[None], axis=2))) <= 1e-12
    E, g = ctx.energy_grad(dev(w.spins))
    assert abs(E.item() - so.energy(model, w.spins)) <= 1e-12 * abs(so.energy(model, w.spins))
    assert np.max(np.abs(g.cpu().numpy() - so.projected_gradient(model, w.spins))) <= 1e-12


def test_cfg2_full_size_lowest_modes_k6(moto, cfg2_full):
    # eigenvalues one by one at 1e-8 relative (floor 1e-3, reading A23); eigenvectors as subspaces (reading A10): the angle to
    # the oracle's lowest-6 space where the gap after mode 6 allows it, containment in the oracle's lowest-8 space otherwise;
    # and the oracle-side residual of every returned pair
    w, lam_ref, V_ref = cfg2_full
    ctx = moto.spin_context(w, kmax=8)
    ctx.set_solver(guard=2)
    lam, V, info = ctx.lowest_modes(dev(w.spins), 6, tol=w.tol, max_iter=20000)
    assert info["converged"], info
    lam = lam.cpu().numpy(); V = V.cpu().numpy()
    assert np.max(np.abs(lam - lam_ref[:6]) / np.maximum(np.abs(lam_ref[:6]), 1e-3)) <= EIG_TOL, (lam, lam_ref)
    Vf = V.reshape(6, -1).T
    gap = lam_ref[6] - lam_ref[5]
    if gap > 1e-2 * abs(lam_ref[5]):
        assert scipy.linalg.subspace_angles(Vf, V_ref[:6].reshape(6, -1).T).max() <= ANGLE_TOL
    else:
        Q = np.linalg.qr(V_ref.reshape(8, -1).T)[0]
        assert np.linalg.norm(Vf - Q @ (Q.T @ Vf), 2) <= ANGLE_TOL
    HV = so.hvp(model_of(w), w.spins, V)
    for a in range(6):
        assert np.linalg.norm(HV[a] - lam[a] * V[a]) <= w.tol * (1 + 1e-3), a
    assert np.max(np.abs(Vf.T @ Vf - np.eye(6))) <= 1e-10
    assert np.max(np.abs(np.sum(V * w.spins[None], axis=2))) <= 1e-10


def test_cfg2_full_size_first_mmf_steps(moto, cfg2_full):
    # the first 3 of configs[2]'s 100 MMF steps (dt = 0.05, re-solve per step, warm start from the transported block): per
    # step the oracle is fed the GPU's own v_1 (SURVEY 8(c) "MMF trajectory": only single steps are pinned) and must
    # reproduce the new state to 1e-13 and |F_mmf|; the re-solved pairs are checked by their oracle-side residuals
    w, lam_ref, _ = cfg2_full
    model = model_of(w)
    ctx = moto.spin_context(w, kmax=8)
    ctx.set_solver(guard=2)
    x = dev(w.spins)
    V0 = None
    for step in range(3):
        lam, V, info = ctx.lowest_modes(x, 6, tol=w.tol, max_iter=20000, V0=V0)
        assert info["converged"], (step, info)
        xh, Vh, lh = x.cpu().numpy(), V.cpu().numpy(), lam.cpu().numpy()
        if step == 0:
            assert np.max(np.abs(lh - lam_ref[:6]) / np.maximum(np.abs(lam_ref[:6]), 1e-3)) <= EIG_TOL
        HV = so.hvp(model, xh, Vh[:2])
        for a in range(2):
            assert np.linalg.norm(HV[a] - lh[a] * Vh[a]) <= w.tol * (1 + 1e-3)
        xn, fn = ctx.mmf_step(x, V[:1].contiguous(), w.dt)
        ref = so.mmf_step(model, xh, Vh[:1], w.dt)
        assert np.max(np.abs(xn.cpu().numpy() - ref)) <= 1e-13
        assert abs(fn.item() - np.linalg.norm(so.mmf_force(model, xh, Vh[:1]))) <= 1e-12 * max(1.0, fn.item())
        x = xn
        V0 = V.clone()
        ctx.transport(x, V0)


def test_transformed_solve_oracle_side_residual_at_1e9(moto):
    # LOBPCG on -p_d(A) (the default fused path where the TMA K1 applies) decides convergence on |A x - theta x| of A itself.
    # At tol = 1e-9 that decision sits far below what an expanded-form residual could resolve (tt - 2 theta xt + theta^2 xx
    # has a rounding floor ~1e-8): the oracle recomputes the residual of every returned pair and it must meet the tolerance.
    for w in (wl.config3_scaled(100), wl.config1()):
        model = model_of(w)
        ctx = moto.spin_context(w, kmax=2)
        ctx.set_solver(hvp_path=2)
        lam, V, info = ctx.lowest_modes(dev(w.spins), 2, tol=1e-9, max_iter=20000)
        assert info["converged"], info
        lam = lam.cpu().numpy(); V = V.cpu().numpy()
        HV = so.hvp(model, w.spins, V)
        for a in range(2):
            r = np.linalg.norm(HV[a] - lam[a] * V[a])
            assert r <= 1e-9 * (1 + 1e-3), (w.name, a, r, info["resid"])
            assert abs(r - info["resid"][a]) <= 1e-3 * 1e-9 + 1e-3 * r      # the reported residual is the true one
        lam_ref, _ = so.lowest_modes(model, w.spins, 2)
        assert np.max(np.abs(lam - lam_ref[:2]) / np.maximum(np.abs(lam_ref[:2]), 1e-3)) <= EIG_TOL


@pytest.mark.parametrize("n,nev", [(6, 2), (3, 1), (18, 6), (24, 8)])
@pytest.mark.parametrize("cond", [1e3, 1e6, 1e10, 1e13])
def test_rayleigh_ritz_ill_conditioned_basis(moto, n, nev, cond):
    # K4 on the kind of pencil a converging LOBPCG produces: S = [X, W, P] with nearly dependent columns (W, P -> span X),
    # cond(S) up to 1e13 before the rank truncation at 1e-10 of the largest eigenvalue of the scaled G_B sets in.  Truth:
    # Ritz values of A on span(S) from a QR of S itself (backward stable, never forms S^T S).  Forming the Gram matrices
    # costs cond(S)^2 eps in the small directions, which the kernel must turn into a dropped direction, not into garbage:
    # the lowest Ritz values may then only move UP (a subspace of span S), by at most what the dropped directions held.
    rng = np.random.default_rng(int(np.log10(cond)) * 100 + n)
    N = 80
    Q0 = np.linalg.qr(rng.standard_normal((N, n)))[0]
    sv = np.logspace(0, -np.log10(cond), n)
    S = (Q0 * sv) @ np.linalg.qr(rng.standard_normal((n, n)))[0]
    Aop = rng.standard_normal((N, N)); Aop = Aop + Aop.T
    GA, GB = S.T @ Aop @ S, S.T @ S
    w = wl.config0()
    ctx = moto.spin_context(w, kmax=8)
    th, Cm = ctx.rayleigh_ritz(dev(GA), dev(GB), nev)
    th, Cm = th.cpu().numpy(), Cm.cpu().numpy()
    assert np.isfinite(th).all() and np.isfinite(Cm).all()
    Qs = np.linalg.qr(S)[0]
    full = np.linalg.eigvalsh(Qs.T @ Aop @ Qs)
    # every returned pair is a genuine Ritz pair of span(S): orthonormal in the S metric, Rayleigh quotient = theta
    Y = S @ Cm
    assert np.max(np.abs(Y.T @ Y - np.eye(nev))) <= 1e-6
    assert np.max(np.abs(np.diag(Y.T @ Aop @ Y) - th)) <= 1e-6 * np.max(np.abs(full))
    assert np.all(th >= full[:nev] - 1e-8 * np.max(np.abs(full)))             # Cauchy interlacing: never below the truth
    if cond <= 1e3:                  # cond(G_B) = 1e6 < 1e10: no direction is dropped, the answer is the truth itself
        assert np.max(np.abs(th - full[:nev])) <= 1e-8 * np.max(np.abs(full))
