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


def test_heptamer_certified_edge(moto, slab):
    # The paper's portability case end to end (Alg. 1 l.9-18): relax the Ni(111) slab + heptamer to its
    # reference minimum, displace the heptamer (seeded), climb with moto_mmf_run to an index-1 saddle, descend on both sides.
    # The oracle cannot follow 2000 outer steps (a dense 2421^2 eigen-solve each), so it checks what is unique about the
    # three end states: stationarity (its own gradient / reflected force), the index (its own dense eigenvalues, which must
    # equal the GPU's), and that one branch returns to the reference minimum.
    w, mdl = slab
    ctx = moto.cart_context(w)
    x = dev(w.positions)
    rinfo = ctx.relax(x, 5000, 1e-6, 0.05)
    assert rinfo["converged"]
    x0 = x.clone()
    rng = np.random.default_rng(5)
    d = np.zeros_like(w.positions)
    top = np.arange(w.Na - 7, w.Na)                       # the heptamer atoms
    d[top] = 0.15 * rng.standard_normal((7, 3))
    d[top, 2] *= 0.2
    x = x0 + dev(d)
    V, info = ctx.mmf_run(x, 2, 0.04, 6000, 1e-4, tol=1e-8, max_iter=5000)
    assert info["converged"] and info["lam"][0] < 0.0 < info["lam"][1]
    xs = x.cpu().numpy()
    lam_ref, V_ref = co.lowest_modes(mdl, xs, 2)
    assert lam_ref[0] < 0.0 < lam_ref[1]
    assert np.max(np.abs(np.array(info["lam"]) - lam_ref) / np.abs(lam_ref)) <= 1e-6
    assert np.linalg.norm(co.mmf_force(mdl, xs, V_ref[:1])) <= 1.1e-4
    E_saddle, E_min = co.energy(mdl, xs), co.energy(mdl, x0.cpu().numpy())
    assert abs(E_min - rinfo["energy"]) <= 1e-11 * abs(E_min)
    assert 0.05 < E_saddle - E_min < 1.0                  # a barrier of a few tenths of an eV
    xp, xm, infos = ctx.two_sided_descent(x, V[0].contiguous(), 0.1, 8000, 1e-6, 0.05)
    assert all(i["converged"] for i in infos)
    ends = sorted(zip([i["energy"] for i in infos], [xp.cpu().numpy(), xm.cpu().numpy()]), key=lambda t: t[0])
    for E, y in ends:
        assert np.linalg.norm(co.gradient(mdl, y)) <= 1.1e-6 and abs(co.energy(mdl, y) - E) <= 1e-11 * abs(E)
        assert E < E_saddle - 0.01
        assert np.all(y[w.fixed == 1] == w.positions[w.fixed == 1])
    assert abs(ends[0][0] - E_min) <= 1e-9 and np.max(np.abs(ends[0][1] - x0.cpu().numpy())) <= 1e-4   # back to the reference minimum
    assert np.max(np.abs(ends[1][1] - x0.cpu().numpy())) > 0.5                                          # a different minimum


def test_transformed_solver_on_atoms(moto, slab):
    # Cartesian atoms take the Chebyshev-transformed LOBPCG by default (degree 24; the upper end of the interval is the block
    # Gershgorin bound of the stored pair coefficients): same eigenpairs as the plain solver and as the all-pairs oracle, in fewer
    # Rayleigh-Ritz steps, on the slab (fixed bottom layers) and on a free cluster
    wc = wl.small_cluster(38, seed=3)
    for w, mdl in (slab, (wc, model_of(wc))):
        pos = w.positions
        lam_ref, V_ref = co.lowest_modes(mdl, pos, 2, extra=1)
        res = {}
        for name, deg in (("auto", 0), ("plain", -1), ("d8", 8), ("d40", 40)):
            ctx = moto.cart_context(w, kmax=2)
            ctx.set_solver(precond_degree=deg)
            lam, V, info = ctx.lowest_modes(dev(pos), 2, tol=1e-9, max_iter=20000)
            assert info["converged"], name
            res[name] = info
            lam, V = lam.cpu().numpy(), V.cpu().numpy()
            assert np.max(np.abs(lam - lam_ref[:2]) / np.maximum(np.abs(lam_ref[:2]), 1e-3)) <= 1e-8, name
            if lam_ref[2] - lam_ref[1] > 1e-3:
                assert np.max(scipy.linalg.subspace_angles(V.reshape(2, -1).T, V_ref[:2].reshape(2, -1).T)) <= 1e-6, name
            r = co.hvp(mdl, pos, V) - lam[:, None, None] * V                    # oracle-side residual
            assert np.max(np.linalg.norm(r.reshape(2, -1), axis=1)) <= 1.01e-9, name
            if w.fixed is not None:
                assert np.all(V[:, w.fixed == 1, :] == 0)                        # masked rows stay zero through the recurrence
        assert res["auto"]["iters"] < res["plain"]["iters"] and res["auto"]["hvp_count"] > 2 * (res["auto"]["iters"] + 2)
