"""GPU parity tests (Cartesian atoms, Morse over a cell list) against the all-pairs CPU oracle."""
import numpy as np
import pytest
import scipy.linalg

from oracle import cart_oracle as co
from paper_2509_26269_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def model_of(w):
    return co.MorseModel(w.cell, w.De, w.alpha, w.r0, w.rc, w.fixed)


def dev(a):
    import torch
    return torch.as_tensor(np.ascontiguousarray(a), dtype=torch.float64).cuda()


def rel_l2(a, b):
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


@pytest.fixture(scope="module")
def slab():
    w = wl.config4()
    mdl = model_of(w)
    return w, mdl


def test_energy_grad_parity(moto, slab):
    w, mdl = slab
    ctx = moto.cart_context(w)
    E, g = ctx.energy_grad(dev(w.positions))
    E_ref = co.energy(mdl, w.positions)
    assert abs(E.item() - E_ref) <= 1e-11 * abs(E_ref)
    assert np.max(np.abs(g.cpu().numpy() - co.gradient(mdl, w.positions))) <= 1e-11


@pytest.mark.parametrize("k", [1, 2, 5])
def test_hvp_parity(moto, slab, k):
    w, mdl = slab
    ctx = moto.cart_context(w, kmax=8)
    V = wl.random_block(w.Na, k, seed=11)   # non-zero on fixed atoms: must be ignored
    HV = ctx.hvp(dev(w.positions), dev(V)).cpu().numpy()
    ref = co.hvp(mdl, w.positions, V)
    assert rel_l2(HV, ref) <= 1e-11
    assert np.all(HV[:, w.fixed == 1, :] == 0)


def test_small_cluster_and_periodic_wrap(moto):
    w = wl.small_cluster(9, seed=3)
    # move the cluster across the periodic boundary so minimum-image pairs matter
    w.positions[:, :2] -= 22.0
    mdl = model_of(w)
    ctx = moto.cart_context(w, kmax=4)
    V = wl.random_block(w.Na, 3, seed=1)
    assert rel_l2(ctx.hvp(dev(w.positions), dev(V)).cpu().numpy(), co.hvp(mdl, w.positions, V)) <= 1e-11
    E, g = ctx.energy_grad(dev(w.positions))
    assert abs(E.item() - co.energy(mdl, w.positions)) <= 1e-12
    assert np.max(np.abs(g.cpu().numpy() - co.gradient(mdl, w.positions))) <= 1e-12


def test_lowest_modes_parity(moto, slab):
    w, mdl = slab
    lam_ref, V_ref = co.lowest_modes(mdl, w.positions, 2, extra=1)
    ctx = moto.cart_context(w, kmax=4)
    ctx.set_solver(guard=2)
    lam, V, info = ctx.lowest_modes(dev(w.positions), 2, tol=1e-9, max_iter=3000)
    assert info["converged"], info
    lam = lam.cpu().numpy(); V = V.cpu().numpy()
    assert np.max(np.abs(lam - lam_ref[:2]) / np.maximum(np.abs(lam_ref[:2]), 1e-3)) <= 1e-8
    ang = scipy.linalg.subspace_angles(V.reshape(2, -1).T, V_ref[:2].reshape(2, -1).T)
    assert ang.max() <= 1e-6
    assert np.all(V[:, w.fixed == 1, :] == 0)


def test_mmf_step_parity(moto, slab):
    w, mdl = slab
    _, V_ref = co.lowest_modes(mdl, w.positions, 2)
    ctx = moto.cart_context(w)
    out, fn = ctx.mmf_step(dev(w.positions), dev(V_ref[:1]), 0.05)
    ref = co.mmf_step(mdl, w.positions, V_ref[:1], 0.05)
    assert np.max(np.abs(out.cpu().numpy() - ref)) <= 1e-13
    assert np.array_equal(out.cpu().numpy()[w.fixed == 1], w.positions[w.fixed == 1])
    assert abs(fn.item() - np.linalg.norm(co.mmf_force(mdl, w.positions, V_ref[:1]))) <= 1e-12


def test_bad_geometry_rejected(moto):
    w = wl.small_cluster(4, seed=1)
    w.cell = np.array([[10.0, 0.0], [0.0, 10.0]])   # rc = 6 > half the cell width
    with pytest.raises(moto.MotoError):
        moto.cart_context(w)


def test_mmf_run_cartesian_matches_stepwise_calls(moto, slab):
    # the outer loop on Cartesian atoms (identity retraction, masked modes): moto_mmf_run == the same calls made one by one,
    # and its first step == the oracle's step fed the same mode
    w, mdl = slab
    ctx = moto.cart_context(w, kmax=4)
    ctx.set_solver(guard=2)
    x = dev(w.positions)
    V, info = ctx.mmf_run(x, 2, 0.05, 2, 0.0, tol=1e-9, max_iter=5000)
    assert info["steps"] == 2 and not info["converged"]
    y = dev(w.positions)
    lam, Vs, _ = ctx.lowest_modes(y, 2, tol=1e-9, max_iter=5000)
    first = co.mmf_step(mdl, w.positions, Vs[:1].cpu().numpy(), 0.05)
    for s in range(2):
        y, _ = ctx.mmf_step(y, Vs[:1].contiguous(), 0.05)
        if s == 0:
            assert np.max(np.abs(y.cpu().numpy() - first)) <= 1e-12
        ctx.transport(y, Vs)
        lam, Vs, _ = ctx.lowest_modes(y, 2, tol=1e-9, max_iter=5000, V0=Vs)
    assert np.max(np.abs(x.cpu().numpy() - y.cpu().numpy())) <= 1e-9
    assert np.array_equal(x.cpu().numpy()[w.fixed == 1], w.positions[w.fixed == 1])
