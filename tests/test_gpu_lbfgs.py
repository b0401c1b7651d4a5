"""GPU parity tests of the L-BFGS variants (moto_relax_lbfgs, moto_mmf_run_lbfgs; readings A29, A30)
against oracle/lbfgs_oracle.py: the first steps of the trajectory step for step (decisions far above rounding), the end
points (energies, stationarity and index recomputed by the oracle on the GPU's states), closed forms, and the point of
having them: fewer evaluations / minimum-mode solves than the conjugate-gradient rule."""
import numpy as np
import pytest

from oracle import cart_oracle as co
from oracle import lbfgs_oracle as lo
from oracle import relax_oracle as ro
from oracle import spin_oracle as so
from paper_2509_26269_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def spin_model(w):
    return so.SpinModel(w.Lx, w.Ly, w.pbc_x, w.pbc_y, w.J, w.D, w.K, w.B, w.mu)


def dev(a):
    import torch
    return torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64).cuda()


@pytest.mark.parametrize("steps", [1, 2, 4, 9])
@pytest.mark.parametrize("L", [14, 40])
def test_relax_lbfgs_first_steps_match_oracle_spins(moto, steps, L):
    w = wl.config1(L=L, R=3.0)
    mdl = spin_model(w)
    ref, iref = lo.relax_downhill_lbfgs(*ro.spin_ops(mdl), w.spins, steps, 0.0, 0.05, M=4)
    ctx = moto.spin_context(w, kmax=2)
    x = dev(w.spins)
    info = ctx.relax_lbfgs(x, steps, 0.0, 0.05, m=4)
    assert info["steps"] == iref["steps"] == steps and info["evals"] == iref["evals"] and info["alpha"] == iref["alpha"]
    assert abs(info["energy"] - iref["energy"]) <= 1e-12 * abs(iref["energy"])
    assert abs(info["gnorm"] - iref["gnorm"]) <= 1e-9 * iref["gnorm"]
    assert np.max(np.abs(x.cpu().numpy() - ref)) <= 1e-10


def test_relax_lbfgs_end_points_and_fewer_evaluations(moto):
    # ferromagnet (closed form), and the 40x40 skyrmion minimum (same energy as the oracle's and the CG loop's; stationarity
    # checked by the oracle on the GPU's end point); L-BFGS needs fewer evaluations than CG on both
    w = wl.config0()
    ctx = moto.spin_context(w, kmax=2)
    x = dev(w.spins)
    info = ctx.relax_lbfgs(x, 2000, 1e-10, 0.05)
    assert info["converged"] and abs(info["energy"] - (-w.N * (6 * w.J + w.K + w.mu * w.B[2]))) <= 1e-10
    assert np.max(np.abs(x.cpu().numpy() - np.array([0.0, 0.0, 1.0]))) <= 1e-9
    w = wl.config1(L=40)
    mdl = spin_model(w)
    ctx = moto.spin_context(w, kmax=2)
    x = dev(w.spins)
    info = ctx.relax_lbfgs(x, 4000, 1e-6, 0.05)
    y = dev(w.spins)
    icg = ctx.relax(y, 4000, 1e-6, 0.05)
    ref, iref = lo.relax_downhill_lbfgs(*ro.spin_ops(mdl), w.spins, 4000, 1e-6, 0.05)
    assert info["converged"] and icg["converged"] and iref["converged"]
    xh = x.cpu().numpy()
    assert np.max(np.abs(np.linalg.norm(xh, axis=1) - 1.0)) <= 1e-14
    assert abs(info["energy"] - iref["energy"]) <= 1e-11 * abs(iref["energy"])
    assert abs(info["energy"] - icg["energy"]) <= 1e-11 * abs(icg["energy"])
    assert np.linalg.norm(so.projected_gradient(mdl, xh)) <= 1.01e-6
    assert info["evals"] < icg["evals"]


def test_relax_lbfgs_cartesian(moto):
    w = wl.config4()
    mdl = co.MorseModel(w.cell, w.De, w.alpha, w.r0, w.rc, w.fixed)
    ref, iref = lo.relax_downhill_lbfgs(*ro.cart_ops(mdl), w.positions, 3, 0.0, 0.05, M=4)
    ctx = moto.cart_context(w)
    x = dev(w.positions)
    info = ctx.relax_lbfgs(x, 3, 0.0, 0.05, m=4)
    assert info["steps"] == 3 and info["evals"] == iref["evals"]
    assert abs(info["energy"] - iref["energy"]) <= 1e-12 * abs(iref["energy"])
    xh = x.cpu().numpy()
    assert np.max(np.abs(xh - ref)) <= 1e-10
    assert np.all(xh[w.fixed == 1] == w.positions[w.fixed == 1])
    info = ctx.relax_lbfgs(x, 5000, 1e-6, 0.05)
    assert info["converged"] and np.linalg.norm(co.gradient(mdl, x.cpu().numpy())) <= 1.01e-6
    y = dev(w.positions)
    icg = ctx.relax(y, 5000, 1e-6, 0.05)
    assert abs(info["energy"] - icg["energy"]) <= 1e-10 * abs(icg["energy"]) and info["evals"] < icg["evals"]


def _mm_ops(mdl):
    _, _, retract, transport = ro.spin_ops(mdl)
    return (lambda m: so.lowest_modes(mdl, m, 2)), (lambda m: -so.projected_gradient(mdl, m)), retract, transport


@pytest.mark.parametrize("steps", [1, 2, 3])
def test_mmf_run_lbfgs_first_steps_match_oracle(moto, steps):
    w = wl.config1(L=12, R=2.0, sigma=0.0)
    mdl = spin_model(w)
    ref, lam_ref, steps_ref, conv_ref, fn_ref, evals_ref = lo.mmf_run_lbfgs(*_mm_ops(mdl), w.spins, 0.1, 0.5, steps, 0.0, M=4)
    ctx = moto.spin_context(w, kmax=2)
    x = dev(w.spins)
    V, info = ctx.mmf_run_lbfgs(x, 2, 0.1, 0.5, steps, 0.0, tol=1e-11, max_iter=20000, m=4)
    assert info["steps"] == steps and not info["converged"] and info["status"] == moto.binding.ENOTCONV
    assert np.max(np.abs(x.cpu().numpy() - ref)) <= 1e-8
    assert abs(info["fnorm"] - fn_ref) <= 1e-7 * fn_ref
    assert np.max(np.abs(np.array(info["lam"]) - lam_ref) / np.abs(lam_ref)) <= 1e-7


def test_mmf_run_lbfgs_reaches_the_saddle_in_fewer_solves_than_cg(moto):
    # the skyrmion-collapse saddle of test_certified_edge_skyrmion_collapse: same saddle (energy, oracle-side stationarity and
    # index of the GPU's state), one minimum-mode solve per iteration -> fewer solves than the CG rule's 2 per iteration
    w = wl.config1(L=12, R=2.0, sigma=0.0)
    mdl = spin_model(w)
    ref, lam_ref, steps_ref, conv_ref, fn_ref, evals_ref = lo.mmf_run_lbfgs(*_mm_ops(mdl), w.spins, 0.1, 0.5, 600, 1e-4)
    ctx = moto.spin_context(w, kmax=2)
    x = dev(w.spins)
    V, info = ctx.mmf_run_lbfgs(x, 2, 0.1, 0.5, 600, 1e-4, tol=1e-9, max_iter=20000)
    assert conv_ref and info["converged"] and info["lam"][0] < 0.0 < info["lam"][1] and info["fnorm"] <= 1e-4
    xs = x.cpu().numpy()
    assert abs(so.energy(mdl, xs) - so.energy(mdl, ref)) <= 1e-7 * abs(so.energy(mdl, ref))
    lam_chk, V_chk = so.lowest_modes(mdl, xs, 2)
    assert np.linalg.norm(so.mmf_force(mdl, xs, V_chk[:1])) <= 1.1e-4 and lam_chk[0] < 0.0 < lam_chk[1]
    assert np.max(np.abs(np.array(info["lam"]) - lam_chk) / np.abs(lam_chk)) <= 1e-6
    y = dev(w.spins)
    Vc, icg = ctx.mmf_run_cg(y, 2, 0.05, 1.0, 400, 1e-4, tol=1e-9, max_iter=20000)
    assert icg["converged"] and info["steps"] + 1 < 2 * icg["steps"] + 1          # MinMode solves: steps + 1 vs 2 steps + 1


def test_mmf_run_lbfgs_heptamer(moto):
    w = wl.config4()
    mdl = co.MorseModel(w.cell, w.De, w.alpha, w.r0, w.rc, w.fixed)
    ctx = moto.cart_context(w)
    x = dev(w.positions)
    assert ctx.relax_lbfgs(x, 5000, 1e-6, 0.05)["converged"]
    d = np.zeros_like(w.positions)
    top = np.arange(w.Na - 7, w.Na)
    d[top] = 0.15 * np.random.default_rng(5).standard_normal((7, 3))
    d[top, 2] *= 0.2
    x = x + dev(d)
    V, info = ctx.mmf_run_lbfgs(x, 2, 0.04, 0.3, 600, 1e-4, tol=1e-8, max_iter=5000)
    assert info["converged"] and info["steps"] < 233                                # the CG rule spends 233 solves on this start
    xs = x.cpu().numpy()
    lam_ref, V_ref = co.lowest_modes(mdl, xs, 2)
    assert lam_ref[0] < 0.0 < lam_ref[1] and np.max(np.abs(np.array(info["lam"]) - lam_ref) / np.abs(lam_ref)) <= 1e-6
    assert np.linalg.norm(co.mmf_force(mdl, xs, V_ref[:1])) <= 1.1e-4
    assert np.all(xs[w.fixed == 1] == w.positions[w.fixed == 1])


def test_lbfgs_argument_errors(moto):
    import ctypes as C
    w = wl.config0()
    ctx = moto.spin_context(w, kmax=2)
    x = dev(w.spins)
    lib = moto.load_library()
    b = moto.binding
    assert lib.moto_relax_lbfgs(ctx._h, x.data_ptr(), 10, 1e-6, 0.05, 9, x.data_ptr(), None) == b.EINVAL     # m > 8
    assert lib.moto_relax_lbfgs(ctx._h, x.data_ptr(), 10, 1e-6, 0.0, 4, x.data_ptr(), None) == b.EINVAL      # alpha0 = 0
    assert lib.moto_relax_lbfgs(ctx._h, x.data_ptr(), 10, 1e-6, 0.05, 4, None, None) == b.EINVAL             # no scratch
    assert lib.moto_mmf_run_lbfgs(ctx._h, x.data_ptr(), 1, 0.1, 0.5, 10, 1e-4, 1e-8, 100, 0, 4, x.data_ptr(), x.data_ptr(), None) == b.EINVAL
