"""GPU parity tests of the general-neighbour-shell path (moto_set_shells) against oracle/shell_oracle.py,
and against the library's own nearest-neighbour kernels on the six-neighbour table."""
import ctypes as C

import numpy as np
import pytest
import scipy.linalg

from oracle import relax_oracle as ro
from oracle import shell_oracle as sh
from oracle import spin_oracle as so
from paper_2509_26269_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def dev(a):
    import torch
    return torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64).cuda()


def rel_l2(a, b):
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


def model_of(w):
    return sh.ShellModel(w.Lx, w.Ly, w.pbc_x, w.pbc_y, w.offsets, w.Jd, w.Dd, w.K, w.B, w.mu)


def shell_workload(Lx, Ly, pbc, rcut, seed, B=(0.01, -0.02, 0.03), **kw):
    offs, J, D = wl.shell_table(rcut, **kw)
    return wl.ShellWorkload(f"sh{Lx}x{Ly}", Lx, Ly, pbc[0], pbc[1], offs, J, D, K=0.05, B=B, mu=1.0, k=2, seed=seed,
                            spins=wl.random_spins(Lx, Ly, seed))


@pytest.mark.parametrize("Lx,Ly,pbc,rcut", [(12, 12, (1, 1), 3.0), (13, 9, (0, 0), 3.0), (16, 7, (1, 0), 2.0), (5, 4, (1, 1), 3.0),
                                             (40, 33, (0, 1), 4.5)])
def test_energy_grad_hvp_parity(moto, Lx, Ly, pbc, rcut):
    # random spins (the paper's "random spin configurations"); 5x4 periodic with rcut 3: offsets wrap more than once
    w = shell_workload(Lx, Ly, pbc, rcut, seed=Lx + Ly)
    mdl = model_of(w)
    ctx = moto.shell_context(w, kmax=8)
    E, g = ctx.energy_grad(dev(w.spins))
    E_ref = sh.energy(mdl, w.spins)
    assert abs(E.item() - E_ref) <= 1e-12 * max(1.0, abs(E_ref))
    assert np.max(np.abs(g.cpu().numpy() - sh.projected_gradient(mdl, w.spins))) <= 1e-12
    for k in (1, 2, 5):
        V = wl.random_block(w.N, k, seed=k)          # not tangent: the API projects
        HV = ctx.hvp(dev(w.spins), dev(V)).cpu().numpy()
        assert rel_l2(HV, sh.hvp(mdl, w.spins, V)) <= 1e-11
        assert np.max(np.abs(np.sum(HV * w.spins[None], axis=2))) <= 1e-12     # output tangent


def test_six_neighbour_table_equals_nearest_neighbour_kernels(moto):
    # rcut = 1, Dz = 0 is the model of configs[0..3]: the table path must agree with the stencil kernels (generic and TMA)
    for L, path in ((14, 1), (64, 2)):
        base = wl.config1(L=L)
        offs, J, D = wl.shell_table(1.0, Dz1=0.0)
        w = wl.ShellWorkload("nn", L, L, 1, 1, offs, J, D, base.K, base.B, base.mu, 2, 0, base.spins)
        nn = moto.spin_context(base, kmax=2)
        nn.set_solver(hvp_path=path)
        st = moto.shell_context(w, kmax=2)
        x, V = dev(base.spins), dev(wl.random_block(base.N, 2, 4))
        E0, g0 = nn.energy_grad(x)
        E1, g1 = st.energy_grad(x)
        assert abs(E0.item() - E1.item()) <= 1e-12 * abs(E0.item())
        assert np.max(np.abs((g0 - g1).cpu().numpy())) <= 1e-12
        assert rel_l2(st.hvp(x, V).cpu().numpy(), nn.hvp(x, V).cpu().numpy()) <= 1e-12
        # n = 0 switches the table off again: bit-identical to the nearest-neighbour context?  J = D = 0 there, so compare
        # against a context created with J, D and an emptied table instead
        nn2 = moto.spin_context(base, kmax=2)
        nn2.set_solver(hvp_path=path)
        nn2.set_shells(offs, J, D)
        nn2.set_shells(np.zeros((0, 2), np.int32), np.zeros(0), np.zeros((0, 3)))
        assert np.array_equal(nn2.hvp(x, V).cpu().numpy(), nn.hvp(x, V).cpu().numpy())


@pytest.mark.parametrize("method", [0, 1])
def test_lowest_modes_vs_dense_oracle(moto, method):
    w = wl.config_shells(L=18, rcut=3.0)
    mdl = model_of(w)
    lam_ref, V_ref = sh.lowest_modes(mdl, w.spins, 2, extra=1)
    ctx = moto.shell_context(w, kmax=2)
    ctx.set_solver(method=method)
    lam, V, info = ctx.lowest_modes(dev(w.spins), 2, tol=1e-9, max_iter=20000)
    assert info["converged"]
    lam, V = lam.cpu().numpy(), V.cpu().numpy()
    assert np.max(np.abs(lam - lam_ref[:2]) / np.maximum(np.abs(lam_ref[:2]), 1e-3)) <= 1e-8
    gap = lam_ref[2] - lam_ref[1]
    ang = scipy.linalg.subspace_angles(V.reshape(2, -1).T, V_ref[:2].reshape(2, -1).T)
    if gap > 1e-3:
        assert np.max(ang) <= 1e-6
    res = sh.hvp(mdl, w.spins, V) - lam[:, None, None] * V            # oracle-side residual of the GPU's pairs
    assert np.max(np.linalg.norm(res.reshape(2, -1), axis=1)) <= 2e-9


def test_mmf_step_and_relax_parity(moto):
    w = wl.config_shells(L=14, rcut=3.0)
    mdl = model_of(w)
    lam, V = sh.lowest_modes(mdl, w.spins, 1)
    ctx = moto.shell_context(w, kmax=2)
    out, fn = ctx.mmf_step(dev(w.spins), dev(V), 0.05)
    assert np.max(np.abs(out.cpu().numpy() - sh.mmf_step(mdl, w.spins, V, 0.05))) <= 1e-13
    ops = ((lambda m: sh.energy(mdl, m)), (lambda m: sh.projected_gradient(mdl, m))) + ro.spin_ops(so.SpinModel(1, 1, 0, 0, 0, 0, 0, (0, 0, 0)))[2:]
    ref, iref = ro.relax_downhill(*ops, w.spins, 6, 0.0, 0.05)
    x = dev(w.spins)
    info = ctx.relax(x, 6, 0.0, 0.05)
    assert info["steps"] == 6 and info["evals"] == iref["evals"] and info["alpha"] == iref["alpha"]
    assert abs(info["energy"] - iref["energy"]) <= 1e-12 * abs(iref["energy"])
    assert np.max(np.abs(x.cpu().numpy() - ref)) <= 1e-11


def test_full_size_366_neighbours(moto):
    # the paper's workload class: 100 x 100 periodic, every shell within 10 lattice constants (366 neighbours)
    w = wl.config_shells()
    assert len(w.offsets) == 366 and w.N == 10000
    mdl = model_of(w)
    ctx = moto.shell_context(w, kmax=2)
    x = dev(w.spins)
    E, g = ctx.energy_grad(x)
    assert abs(E.item() - sh.energy(mdl, w.spins)) <= 1e-12 * abs(E.item())
    assert np.max(np.abs(g.cpu().numpy() - sh.projected_gradient(mdl, w.spins))) <= 1e-12
    V = wl.random_block(w.N, 2, 8)
    assert rel_l2(ctx.hvp(x, dev(V)).cpu().numpy(), sh.hvp(mdl, w.spins, V)) <= 1e-11
    lam, Vm, info = ctx.lowest_modes(x, 2, tol=1e-8, max_iter=20000)
    assert info["converged"]
    lam, Vm = lam.cpu().numpy(), Vm.cpu().numpy()
    res = sh.hvp(mdl, w.spins, Vm) - lam[:, None, None] * Vm
    assert np.max(np.linalg.norm(res.reshape(2, -1), axis=1)) <= 2e-8
    # "lowest-ness" at this size is not pinned (shift-invert on the 14.7 M-nonzero explicit Hessian takes minutes): it is
    # checked with the same 366-neighbour table on a 36 x 36 lattice, where the dense oracle is exact
    w2 = wl.config_shells(L=36)
    mdl2 = model_of(w2)
    lam_ref, V_ref = sh.lowest_modes(mdl2, w2.spins, 2, extra=1)
    ctx2 = moto.shell_context(w2, kmax=2)
    lam2, V2, info2 = ctx2.lowest_modes(dev(w2.spins), 2, tol=1e-9, max_iter=20000)
    assert info2["converged"]
    assert np.max(np.abs(lam2.cpu().numpy() - lam_ref[:2]) / np.maximum(np.abs(lam_ref[:2]), 1e-3)) <= 1e-8
    if lam_ref[2] - lam_ref[1] > 1e-3:
        assert np.max(scipy.linalg.subspace_angles(V2.cpu().numpy().reshape(2, -1).T, V_ref[:2].reshape(2, -1).T)) <= 1e-6


def test_set_shells_errors(moto):
    w = shell_workload(8, 8, (1, 1), 2.0, seed=1)
    ctx = moto.shell_context(w, kmax=2)
    lib = moto.load_library()
    with pytest.raises(moto.binding.MotoError):
        ctx.set_shells(w.offsets[:-1], w.Jd[:-1], w.Dd[:-1])                # inversion partner missing
    D2 = w.Dd.copy(); D2[0, 2] += 0.1
    with pytest.raises(moto.binding.MotoError):
        ctx.set_shells(w.offsets, w.Jd, D2)                                 # D(-d) != -D(d)
    with pytest.raises(moto.binding.MotoError):
        ctx.set_shells(np.vstack([w.offsets, [[0, 0]]]), np.append(w.Jd, 1.0), np.vstack([w.Dd, [[0, 0, 0]]]))
    assert lib.moto_set_shells(ctx._h, 513, None, None, None) == moto.binding.EINVAL
    with pytest.raises(moto.binding.MotoError):                             # the Chebyshev building block needs the TMA path
        ctx.cheb_apply(dev(w.spins), dev(wl.random_block(w.N, 1, 1)), 4, 0.0, 20.0, -1.0)
    cart = moto.cart_context(wl.small_cluster(5, seed=2))
    off = np.ascontiguousarray(w.offsets, np.int32)
    assert lib.moto_set_shells(cart._h, len(off), off.ctypes.data, w.Jd.ctypes.data, np.ascontiguousarray(w.Dd).ctypes.data) == moto.binding.ESTATE


# ---------------------------------------------------------------- the register-blocked kernel (spin_shells_dense.cu)
# Lx >= 32 and k <= 2 take k_shell_dense: fields staged in shared memory with the boundary handled there, R = 2 or 3 output
# rows per thread (R = 3 when that leaves the fullest SM less work: 96 x 100 gives 150 CTAs at R = 2, 102 at R = 3).
@pytest.mark.parametrize("Lx,Ly,pbc,rcut", [(70, 50, (0, 0), 5.0),      # R = 2, open: zeros beyond every edge, runs A + B in most CTAs
                                             (33, 47, (1, 0), 4.5),      # R = 2, odd sizes: last row group has one row
                                             (96, 100, (0, 0), 3.0),     # R = 3, open, last row group has one row (100 = 33 x 3 + 1)
                                             (96, 100, (0, 1), 3.0),     # R = 3, open x / periodic y
                                             (32, 40, (1, 1), 10.0)])    # halo (11) wraps a 32-wide lattice; 366 taps
def test_dense_kernel_parity_api_and_three_term(moto, Lx, Ly, pbc, rcut):
    w = shell_workload(Lx, Ly, pbc, rcut, seed=Lx + 3 * Ly)
    mdl = model_of(w)
    ctx = moto.shell_context(w, kmax=2)
    x = dev(w.spins)
    # energy / gradient through the same kernel (m the only staged field); c reaches the three-term calls below
    E, g = ctx.energy_grad(x)
    E_ref = sh.energy(mdl, w.spins)
    assert abs(E.item() - E_ref) <= 1e-12 * max(1.0, abs(E_ref))
    assert np.max(np.abs(g.cpu().numpy() - sh.projected_gradient(mdl, w.spins))) <= 1e-12
    E2, _ = ctx.energy_grad(x, want_grad=False)
    assert E2.item() == E.item()
    for k in (1, 2):
        V = wl.random_block(w.N, k, seed=10 + k)                       # not tangent: the API projects the neighbours
        HV = ctx.hvp(x, dev(V)).cpu().numpy()
        assert rel_l2(HV, sh.hvp(mdl, w.spins, V)) <= 1e-11
        assert np.max(np.abs(np.sum(HV * w.spins[None], axis=2))) <= 1e-12
        # solver mode (tangent input, c from the context): out = alpha (Hess[V] - c0 V) + beta U
        Vt = V - np.sum(V * w.spins[None], axis=2, keepdims=True) * w.spins[None]
        U = wl.random_block(w.N, k, seed=20 + k)
        alpha, c0, beta = 0.37, -0.8, 1.9
        out = ctx.hvp_three_term(x, dev(Vt), alpha, c0, beta, dev(U)).cpu().numpy()
        ref = alpha * (sh.hvp(mdl, w.spins, Vt) - c0 * Vt) + beta * U
        assert rel_l2(out, ref) <= 1e-11
        out0 = ctx.hvp_three_term(x, dev(Vt), 1.0, 0.0, 0.0, None, refresh_c=False).cpu().numpy()
        assert rel_l2(out0, sh.hvp(mdl, w.spins, Vt)) <= 1e-11
    # reruns are bit-identical (fixed summation order)
    a = ctx.hvp(x, dev(V)).cpu().numpy()
    assert np.array_equal(a, HV)


def test_cheb_apply_and_transformed_solve_on_shells(moto):
    # the Chebyshev transformation on the shell path: d launches of k_shell_dense with device-side coefficients
    w = shell_workload(36, 30, (1, 0), 4.5, seed=77)
    mdl = model_of(w)
    ctx = moto.shell_context(w, kmax=2)
    x = dev(w.spins)
    lam_ref, V_ref = sh.lowest_modes(mdl, w.spins, 2, extra=1)
    a, b, aL = lam_ref[1] + 0.05, 60.0, lam_ref[0]
    for k, d in ((1, 1), (2, 2), (2, 7), (1, 12)):
        V = wl.random_block(w.N, k, seed=30 + d)
        Vt = V - np.sum(V * w.spins[None], axis=2, keepdims=True) * w.spins[None]
        out = ctx.cheb_apply(x, dev(Vt), d, a, b, aL).cpu().numpy()
        ref = sh.transformed_operator_apply(mdl, w.spins, Vt, d, a, b, aL)
        assert rel_l2(out, ref) <= 1e-10, (k, d)
    # the solver on -p_16(A) (default on shells where the dense kernel applies) against the dense oracle, and against the plain solve
    res = {}
    for name, deg in (("auto", 0), ("plain", -1), ("d8", 8)):
        ctx.set_solver(precond_degree=deg)
        lam, Vm, info = ctx.lowest_modes(x, 2, tol=1e-9, max_iter=20000)
        assert info["converged"], name
        res[name] = info
        lam, Vm = lam.cpu().numpy(), Vm.cpu().numpy()
        assert np.max(np.abs(lam - lam_ref[:2]) / np.maximum(np.abs(lam_ref[:2]), 1e-3)) <= 1e-8, name
        r = sh.hvp(mdl, w.spins, Vm) - lam[:, None, None] * Vm
        assert np.max(np.linalg.norm(r.reshape(2, -1), axis=1)) <= 1.01e-9, name
        if lam_ref[2] - lam_ref[1] > 1e-3:
            assert np.max(scipy.linalg.subspace_angles(Vm.reshape(2, -1).T, V_ref[:2].reshape(2, -1).T)) <= 1e-6, name
    assert res["auto"]["iters"] < res["plain"]["iters"] and res["auto"]["hvp_count"] > 2 * (res["auto"]["iters"] + 2)
    # thick-restart Lanczos on the same transformed operator (method = 1; k = 2 and k = 1)
    for k in (2, 1):
        ctx.set_solver(method=1, precond_degree=0)
        lam, Vm, info = ctx.lowest_modes(x, k, tol=1e-9, max_iter=20000)
        assert info["converged"]
        lam, Vm = lam.cpu().numpy(), Vm.cpu().numpy()
        assert np.max(np.abs(lam - lam_ref[:k]) / np.maximum(np.abs(lam_ref[:k]), 1e-3)) <= 1e-8
        r = sh.hvp(mdl, w.spins, Vm) - lam[:, None, None] * Vm
        assert np.max(np.linalg.norm(r.reshape(k, -1), axis=1)) <= 1.01e-9
        assert info["hvp_count"] > 4 * info["iters"]                    # transformed: many HVPs per Lanczos step


@pytest.mark.parametrize("L,pbc", [(316, 1), (250, 0)])
def test_dense_and_warp_per_site_kernels_agree_beyond_oracle_sizes(moto, L, pbc):
    # 10^5 sites x 366 neighbours: the explicit Hessian of the oracle does not fit a test; the two kernels share no code
    # (k = 3 takes the warp-per-site kernel of spin_shells.cu, k = 2 the register-blocked one), both are oracle-checked at
    # 100 x 100 and below, and must agree here on every output (many CTA waves, runs A + B, R = 2)
    w = wl.config_shells(L=L, pbc=pbc)
    ctx = moto.shell_context(w, kmax=3)
    x = dev(w.spins)
    V = dev(wl.random_block(w.N, 3, seed=5))
    ref = ctx.hvp(x, V).cpu().numpy()
    new = ctx.hvp(x, V[:2].contiguous()).cpu().numpy()
    assert np.max(np.abs(new - ref[:2])) <= 1e-12 * np.max(np.abs(ref))
