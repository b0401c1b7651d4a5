"""GPU tests of moto_lowest_modes_batch (Alg. 1 l.3-5): P independent problems solved at
once must give exactly what P separate calls give, and what the dense oracle gives."""
import numpy as np
import pytest

from oracle import spin_oracle as so
from paper_2509_26269_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def dev(a):
    import torch
    return torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64).cuda()


def population(P, L, R=3.0):
    """P perturbed copies of one skyrmion state (Alg. 1 l.1: x_0 + P_Omega delta_i), different seeds."""
    return [wl.config1(seed=2000 + p, L=L, R=R, sigma=0.05) for p in range(P)]


@pytest.mark.parametrize("L,P", [(16, 6), (64, 3)])       # generic K1 / TMA K1 + Chebyshev transformation (cooperative launches)
def test_batch_equals_separate_calls_and_oracle(moto, L, P):
    import torch
    ws = population(P, L)
    hvp_path = 2 if L == 64 else 0
    ctxs = [moto.spin_context(w, kmax=2, stream=torch.cuda.Stream()) for w in ws]
    for c in ctxs:
        c.set_solver(hvp_path=hvp_path)
    xs = [dev(w.spins) for w in ws]
    lams, Vs, infos = moto.lowest_modes_batch(ctxs, xs, 2, 1e-9, max_iter=20000)
    torch.cuda.synchronize()
    for p, w in enumerate(ws):
        assert infos[p]["converged"] and infos[p]["status"] == 0
        ref = moto.spin_context(w, kmax=2)
        ref.set_solver(hvp_path=hvp_path)
        lam1, V1, info1 = ref.lowest_modes(xs[p], 2, tol=1e-9, max_iter=20000)
        assert np.array_equal(lam1.cpu().numpy(), lams[p].cpu().numpy())          # bit-identical: same kernels, same order
        assert np.array_equal(V1.cpu().numpy(), Vs[p].cpu().numpy())
        assert info1["iters"] == infos[p]["iters"]
        if L == 16:
            mdl = so.SpinModel(w.Lx, w.Ly, w.pbc_x, w.pbc_y, w.J, w.D, w.K, w.B, w.mu)
            lam_ref, _ = so.lowest_modes(mdl, w.spins, 2)
            assert np.max(np.abs(lams[p].cpu().numpy() - lam_ref) / np.maximum(np.abs(lam_ref), 1e-3)) <= 1e-8


def test_batch_mixed_lattices_notconv_and_errors(moto):
    import ctypes as C
    import torch
    ws = [wl.config0(), wl.config1(L=12), wl.config1(L=20)]
    ctxs = [moto.spin_context(w, kmax=2, stream=torch.cuda.Stream()) for w in ws]
    xs = [dev(w.spins) for w in ws]
    lams, Vs, infos = moto.lowest_modes_batch(ctxs, xs, 2, 1e-12, max_iter=3, allow_notconv=True)
    assert all(i["status"] == moto.binding.ENOTCONV and not i["converged"] for i in infos)
    lams, Vs, infos = moto.lowest_modes_batch(ctxs, xs, 2, 1e-8, max_iter=5000)
    assert all(i["converged"] for i in infos)
    lib = moto.load_library()
    H = (C.c_void_p * 2)(ctxs[0]._h, ctxs[0]._h)
    S = (C.c_void_p * 2)(xs[0].data_ptr(), xs[0].data_ptr())
    assert lib.moto_lowest_modes_batch(H, 2, S, 2, 1e-8, 10, 0, S, S, None, None) == moto.binding.EINVAL    # same context twice
    assert lib.moto_lowest_modes_batch(None, 2, S, 2, 1e-8, 10, 0, S, S, None, None) == moto.binding.EINVAL
    assert lib.moto_lowest_modes_batch(H, 0, S, 2, 1e-8, 10, 0, S, S, None, None) == moto.binding.EINVAL


def test_batch_more_problems_than_threads(moto):
    # P = 40 > 32 host threads: the worker queue must hand every problem out exactly once
    import torch
    ws = [wl.config0(seed=5000 + p) for p in range(40)]
    ctxs = [moto.spin_context(w, kmax=2, stream=torch.cuda.Stream()) for w in ws]
    xs = [dev(w.spins) for w in ws]
    lams, Vs, infos = moto.lowest_modes_batch(ctxs, xs, 2, 1e-9, max_iter=5000)
    for p, w in enumerate(ws):
        mdl = so.SpinModel(w.Lx, w.Ly, w.pbc_x, w.pbc_y, w.J, w.D, w.K, w.B, w.mu)
        lam_ref, _ = so.lowest_modes(mdl, w.spins, 2)
        assert infos[p]["converged"]
        assert np.max(np.abs(lams[p].cpu().numpy() - lam_ref) / np.maximum(np.abs(lam_ref), 1e-3)) <= 1e-8


# ---------------------------------------------------------------- the persistent kernel on the Chebyshev-transformed operator
# From 128 sites on (and up to 148 x 256 sites) the persistent kernel runs LOBPCG on -p_16(A) (lobpcg_persistent.cu): plain
# start, transformed phases closed by a restart on A, convergence decided on true A-residuals only.

def open_lattice(p):
    m = wl.random_spins(37, 33, 300 + p)
    return wl.SpinWorkload("rand37x33_open", 37, 33, 0, 0, 1.0, 0.3, 0.05, (0.01, -0.02, 0.03), 1.0, 2, 300 + p, m)


@pytest.mark.parametrize("make,P", [(lambda p: wl.config1(seed=2000 + p, L=40, R=3.0, sigma=0.05), 5), (open_lattice, 3)])
def test_persistent_transformed_batch_equals_separate_and_oracle(moto, make, P):
    import torch
    ws = [make(p) for p in range(P)]
    assert ws[0].N >= 128
    ctxs = [moto.spin_context(w, kmax=2) for w in ws]
    xs = [dev(w.spins) for w in ws]
    lams, Vs, infos = moto.lowest_modes_batch(ctxs, xs, 2, 1e-9, max_iter=20000)
    for p, w in enumerate(ws):
        assert infos[p]["converged"] and infos[p]["status"] == 0
        ref = moto.spin_context(w, kmax=2)
        lam1, V1, info1 = ref.lowest_modes(xs[p], 2, tol=1e-9, max_iter=20000)
        assert np.array_equal(lam1.cpu().numpy(), lams[p].cpu().numpy())          # bit-identical: chunk-ordered sums
        assert np.array_equal(V1.cpu().numpy(), Vs[p].cpu().numpy())
        assert info1["iters"] == infos[p]["iters"] and info1["hvp_count"] == infos[p]["hvp_count"]
        assert info1["hvp_count"] > 2 * (info1["iters"] + 1)                       # the transformation was on: > 1 HVP per column and iteration
        mdl = so.SpinModel(w.Lx, w.Ly, w.pbc_x, w.pbc_y, w.J, w.D, w.K, w.B, w.mu)
        lam_ref, V_ref = so.lowest_modes(mdl, w.spins, 2)
        lam = lams[p].cpu().numpy()
        assert np.max(np.abs(lam - lam_ref) / np.maximum(np.abs(lam_ref), 1e-3)) <= 1e-8
        V = Vs[p].cpu().numpy().reshape(2, -1)
        assert np.max(np.abs(V @ V.T - np.eye(2))) <= 1e-9
        assert np.max(np.abs(np.einsum("kic,ic->ki", Vs[p].cpu().numpy(), w.spins))) <= 1e-12      # tangent
        # true A-residual of what came back, recomputed with K1, against the reported one and the tolerance
        HV = ref.hvp(xs[p], Vs[p]).cpu().numpy().reshape(2, -1)
        for j in range(2):
            r = np.linalg.norm(HV[j] - lam[j] * V[j])
            assert r <= 1.01e-9 and abs(r - infos[p]["resid"][j]) <= 1e-11


def test_persistent_operator_options_agree(moto):
    w = wl.config1(L=40)
    x = dev(w.spins)
    out = {}
    for name, kw in (("auto", dict()), ("plain", dict(precond_degree=-1)), ("d8", dict(precond_degree=8, persistent=1)),
                     ("d32", dict(precond_degree=32, persistent=1)), ("multi-launch", dict(persistent=2))):
        ctx = moto.spin_context(w, kmax=2)
        ctx.set_solver(**kw)
        lam, V, info = ctx.lowest_modes(x, 2, tol=1e-9, max_iter=20000)
        assert info["converged"], name
        out[name] = (lam.cpu().numpy(), info)
    for name, (lam, info) in out.items():
        assert np.max(np.abs(lam - out["multi-launch"][0])) <= 1e-8 * np.max(np.abs(lam)), name
    assert out["plain"][1]["hvp_count"] == 2 * (out["plain"][1]["iters"] + 2)      # A X, then one HVP per column and iteration (the last one unused)
    assert out["auto"][1]["iters"] < out["plain"][1]["iters"] // 3                 # far fewer Rayleigh-Ritz steps when transformed
    assert out["d32"][1]["iters"] <= out["d8"][1]["iters"]
    # k = 1 takes the same kernel (kb = 1)
    ctx = moto.spin_context(w, kmax=2)
    lam1, V1, info1 = ctx.lowest_modes(x, 1, tol=1e-9, max_iter=20000)
    assert info1["converged"] and abs(float(lam1[0]) - out["multi-launch"][0][0]) <= 1e-8 * abs(out["multi-launch"][0][0])


def test_persistent_transformed_max_iter_and_warm_start(moto):
    import torch
    w = wl.config3_scaled(100)                       # clustered spectrum: 2155 plain iterations, ~50 transformed
    ctx = moto.spin_context(w, kmax=2)
    x = dev(w.spins)
    # cut off inside a transformed phase: ENOTCONV, and what is reported are true A-Ritz values and A-residuals
    lam, V, info = ctx.lowest_modes(x, 2, tol=1e-12, max_iter=14, allow_notconv=True)
    assert info["status"] == moto.binding.ENOTCONV and not info["converged"] and info["iters"] == 14
    Vn, lamn = V.cpu().numpy().reshape(2, -1), lam.cpu().numpy()
    HV = ctx.hvp(x, V).cpu().numpy().reshape(2, -1)
    for j in range(2):
        assert abs(lamn[j] - Vn[j] @ HV[j]) <= 1e-12
        r = np.linalg.norm(HV[j] - lamn[j] * Vn[j])
        assert r > 1e-12 and abs(r - info["resid"][j]) <= 1e-9 * max(1.0, r) + 1e-3 * r
    # converged solve, then a warm start from the perturbed solution: same eigenvalues for fewer HVPs
    lam0, V0, info0 = ctx.lowest_modes(x, 2, tol=w.tol, max_iter=20000)
    assert info0["converged"] and info0["iters"] < 200
    g = torch.Generator(device="cuda").manual_seed(5)
    Vp = V0 + 1e-4 * torch.randn(V0.shape, dtype=torch.float64, device="cuda", generator=g)
    lam2, V2, info2 = ctx.lowest_modes(x, 2, tol=w.tol, max_iter=20000, V0=Vp)
    assert info2["converged"] and info2["hvp_count"] < info0["hvp_count"]
    assert np.max(np.abs(lam2.cpu().numpy() - lam0.cpu().numpy())) <= 1e-8 * abs(float(lam0[0]))
