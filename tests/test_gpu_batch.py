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
