"""Thin ctypes binding over libmoto.so (include/moto.h): argument marshalling only.

torch is used for device memory and the CUDA stream handle; every step of the path runs inside the
library's kernels.  There is no CPU fallback: if the library is missing or no CUDA device is
present, calls raise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

KMAX = 8
NSMAX = 24
OK, EINVAL, ENOMEM, ECUDA, ENOTCONV, ESTATE = range(6)
KIND_TRI2D, KIND_CARTESIAN = 0, 1

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmoto.so")
_lib = None


class MotoError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"moto status {status}: {msg}")
        self.status = status


class Lattice(C.Structure):
    _fields_ = [("kind", C.c_int32), ("Lx", C.c_int32), ("Ly", C.c_int32), ("pbc_x", C.c_int32), ("pbc_y", C.c_int32),
                ("n_atoms", C.c_int32), ("cell", (C.c_double * 2) * 2), ("d_fixed", C.c_void_p)]


class SpinParams(C.Structure):
    _fields_ = [("J", C.c_double), ("D", C.c_double), ("K", C.c_double), ("B", C.c_double * 3), ("mu", C.c_double)]


class MorseParams(C.Structure):
    _fields_ = [("De", C.c_double), ("alpha", C.c_double), ("r0", C.c_double), ("rc", C.c_double)]


class SolverOpts(C.Structure):
    _fields_ = [("guard", C.c_int32), ("check_every", C.c_int32), ("precond_degree", C.c_int32), ("hvp_path", C.c_int32),
                ("precond_lo", C.c_double), ("precond_hi", C.c_double), ("seed", C.c_uint64), ("method", C.c_int32), ("ncv", C.c_int32),
                ("cheb_mode", C.c_int32), ("persistent", C.c_int32)]


class MmfInfo(C.Structure):
    _fields_ = [("steps", C.c_int32), ("converged", C.c_int32), ("fnorm", C.c_double), ("lam", C.c_double * KMAX),
                ("hvp_count", C.c_int64), ("solver_iters", C.c_int64)]


class RelaxInfo(C.Structure):
    _fields_ = [("steps", C.c_int32), ("converged", C.c_int32), ("evals", C.c_int32), ("pad_", C.c_int32),
                ("energy", C.c_double), ("gnorm", C.c_double), ("alpha", C.c_double)]

    def as_dict(self, status=0):
        return dict(steps=self.steps, converged=bool(self.converged), evals=self.evals, energy=self.energy, gnorm=self.gnorm,
                    alpha=self.alpha, status=status)


class SolveInfo(C.Structure):
    _fields_ = [("iters", C.c_int32), ("converged", C.c_int32), ("resid", C.c_double * KMAX), ("hvp_count", C.c_int64)]


_SIGS = {
    "moto_version": (C.c_char_p, []),
    "moto_workspace_bytes": (C.c_size_t, [C.POINTER(Lattice), C.c_int]),
    "moto_create": (C.c_int, [C.POINTER(Lattice), C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p, C.c_int,
                              C.POINTER(C.c_void_p)]),
    "moto_destroy": (None, [C.c_void_p]),
    "moto_set_solver": (C.c_int, [C.c_void_p, C.POINTER(SolverOpts)]),
    "moto_last_error": (C.c_char_p, [C.c_void_p]),
    "moto_set_shells": (C.c_int, [C.c_void_p, C.c_int, C.c_void_p, C.c_void_p, C.c_void_p]),
    "moto_check_overflow": (C.c_int, [C.c_void_p]),
    "moto_energy_grad": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]),
    "moto_hvp": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p]),
    "moto_lowest_modes": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int, C.c_double, C.c_int, C.c_int, C.c_void_p, C.c_void_p,
                                    C.POINTER(SolveInfo)]),
    "moto_lowest_modes_batch": (C.c_int, [C.c_void_p, C.c_int, C.c_void_p, C.c_int, C.c_double, C.c_int, C.c_int, C.c_void_p, C.c_void_p,
                                          C.c_void_p, C.c_void_p]),
    "moto_mmf_step": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_double, C.c_void_p, C.c_void_p]),
    "moto_hvp_three_term": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_double, C.c_double, C.c_double, C.c_void_p,
                                      C.c_void_p, C.c_int]),
    "moto_cheb_apply": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, C.c_void_p, C.c_int]),
    "moto_mmf_run": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int, C.c_double, C.c_int, C.c_double, C.c_double, C.c_int, C.c_int,
                               C.c_void_p, C.POINTER(MmfInfo)]),
    "moto_relax": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int, C.c_double, C.c_double, C.POINTER(RelaxInfo)]),
    "moto_two_sided_descent": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_double, C.c_int, C.c_double, C.c_double,
                                         C.c_void_p, C.c_void_p, C.POINTER(RelaxInfo)]),
    "moto_mmf_run_cg": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int, C.c_double, C.c_double, C.c_int, C.c_double, C.c_double, C.c_int, C.c_int,
                                  C.c_void_p, C.c_void_p, C.POINTER(MmfInfo)]),
    "moto_relax_lbfgs": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int, C.c_double, C.c_double, C.c_int, C.c_void_p, C.POINTER(RelaxInfo)]),
    "moto_mmf_run_lbfgs": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int, C.c_double, C.c_double, C.c_int, C.c_double, C.c_double, C.c_int, C.c_int,
                                     C.c_int, C.c_void_p, C.c_void_p, C.POINTER(MmfInfo)]),
    "moto_transport": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int]),
    "moto_gram": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_int, C.c_void_p]),
    "moto_rayleigh_ritz": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_int, C.c_void_p, C.c_void_p]),
    "moto_energy_grad_host": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]),
    "moto_hvp_host": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_void_p]),
    "moto_lowest_modes_host": (C.c_int, [C.c_void_p, C.c_void_p, C.c_int, C.c_double, C.c_int, C.c_int, C.c_void_p,
                                         C.c_void_p, C.POINTER(SolveInfo)]),
    "moto_mmf_step_host": (C.c_int, [C.c_void_p, C.c_void_p, C.c_void_p, C.c_int, C.c_double, C.c_void_p, C.c_void_p]),
    "moto_launch_count": (C.c_int64, [C.c_void_p]),
    "moto_gram_static": (C.c_int, [C.c_void_p, C.c_int, C.c_void_p, C.c_int, C.c_int64, C.c_void_p, C.c_void_p]),
    "moto_gram_static_last_error": (C.c_char_p, []),
}
EXPORTS = tuple(_SIGS)


def load_library(path: str | None = None):
    """dlopen libmoto.so and set the prototypes.  Raises (never falls back) if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    path = path or LIB_PATH
    if not os.path.exists(path):
        raise RuntimeError(f"{path} not found: build it with `python -m paper_2509_26269_b200.build` "
                           "(there is no CPU fallback)")
    lib = C.CDLL(path)
    for name, (res, args) in _SIGS.items():
        fn = getattr(lib, name)
        fn.restype = res
        fn.argtypes = args
    _lib = lib
    return lib


def _ptr(t):
    """Device/host address of a torch tensor or numpy array (None -> NULL)."""
    if t is None:
        return None
    if isinstance(t, np.ndarray):
        assert t.dtype == np.float64 and t.flags.c_contiguous
        return t.ctypes.data
    assert t.is_contiguous()
    return t.data_ptr()


def _dev_f64(t, shape=None):
    import torch
    assert isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous(), \
        "expected a contiguous CUDA float64 tensor"
    if shape is not None:
        assert tuple(t.shape) == tuple(shape), f"shape {tuple(t.shape)} != {tuple(shape)}"
    return t


class Context:
    """A moto_ctx plus the torch-owned workspace it points into."""

    def __init__(self, lattice: Lattice, params, kmax: int = 2, device="cuda:0", stream=None, fixed=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("moto: no CUDA device (there is no CPU fallback)")
        self.lib = load_library()
        self.device = torch.device(device)
        self.kmax = int(kmax)
        self._fixed = None
        if fixed is not None:
            self._fixed = torch.as_tensor(np.asarray(fixed, dtype=np.uint8)).to(self.device).contiguous()
            lattice.d_fixed = self._fixed.data_ptr()
        self.lattice = lattice
        self.params = params
        self.N = lattice.Lx * lattice.Ly if lattice.kind == KIND_TRI2D else lattice.n_atoms
        nbytes = self.lib.moto_workspace_bytes(C.byref(lattice), self.kmax)
        if nbytes == 0:
            raise MotoError(EINVAL, "bad lattice or kmax")
        self.workspace_bytes = int(nbytes)
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            base = self.workspace.data_ptr()
            self._ws_ptr = (base + 255) & ~255
            self.stream = stream if stream is not None else torch.cuda.current_stream(self.device)
            h = C.c_void_p()
            st = self.lib.moto_create(C.byref(lattice), C.addressof(params), self._ws_ptr, nbytes,
                                      self.stream.cuda_stream, self.kmax, C.byref(h))
        if st != OK:
            raise MotoError(st, "moto_create failed")
        self._h = h

    # -- helpers
    def _check(self, st, allow=()):
        if st != OK and st not in allow:
            raise MotoError(st, self.lib.moto_last_error(self._h).decode())
        return st

    def close(self):
        if getattr(self, "_h", None):
            self.lib.moto_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_solver(self, guard=0, check_every=0, precond_degree=0, precond_lo=0.0, precond_hi=0.0, seed=0, hvp_path=0,
                   method=0, ncv=0, cheb_mode=0, persistent=0):
        """method: 0 block LOBPCG, 1 thick-restart Lanczos (ncv = basis size, 0 = largest the workspace holds)."""
        o = SolverOpts(guard, check_every, precond_degree, hvp_path, precond_lo, precond_hi, seed, method, ncv, cheb_mode, persistent)
        self._check(self.lib.moto_set_solver(self._h, C.byref(o)))

    def set_shells(self, offsets, J, D):
        """moto_set_shells: host tables offsets [n][2] int32, J [n], D [n][3] (n = 0 / empty: back to nearest neighbours)."""
        off = np.ascontiguousarray(offsets, dtype=np.int32).reshape(-1, 2)
        Jh = np.ascontiguousarray(J, dtype=np.float64).reshape(-1)
        Dh = np.ascontiguousarray(D, dtype=np.float64).reshape(-1, 3)
        assert off.shape[0] == Jh.shape[0] == Dh.shape[0]
        self._check(self.lib.moto_set_shells(self._h, int(off.shape[0]), off.ctypes.data, Jh.ctypes.data, Dh.ctypes.data))

    @property
    def launch_count(self) -> int:
        return int(self.lib.moto_launch_count(self._h))

    def _empty(self, *shape):
        import torch
        return torch.empty(*shape, dtype=torch.float64, device=self.device)

    # -- device-pointer API (names follow include/moto.h)
    def check_overflow(self):
        self._check(self.lib.moto_check_overflow(self._h))

    def energy_grad(self, spins, want_grad=True):
        """moto_energy_grad -> (E [1] device tensor, g [N][3] device tensor or None)."""
        _dev_f64(spins, (self.N, 3))
        E = self._empty(1)
        g = self._empty(self.N, 3) if want_grad else None
        self._check(self.lib.moto_energy_grad(self._h, _ptr(spins), _ptr(E), _ptr(g)))
        return E, g

    def hvp(self, spins, V, out=None):
        """moto_hvp: V [k][N][3] -> HV [k][N][3]."""
        _dev_f64(spins, (self.N, 3))
        k = V.shape[0]
        _dev_f64(V, (k, self.N, 3))
        HV = out if out is not None else self._empty(k, self.N, 3)
        self._check(self.lib.moto_hvp(self._h, _ptr(spins), _ptr(V), k, _ptr(HV)))
        return HV

    def hvp_three_term(self, spins, V, alpha, c0, beta, U=None, out=None, refresh_c=True):
        """moto_hvp_three_term: out = alpha (Hess[V] - c0 V) + beta U for tangent V (solver mode)."""
        _dev_f64(spins, (self.N, 3))
        k = V.shape[0]
        _dev_f64(V, (k, self.N, 3))
        if U is not None:
            _dev_f64(U, (k, self.N, 3))
        out = out if out is not None else self._empty(k, self.N, 3)
        self._check(self.lib.moto_hvp_three_term(self._h, _ptr(spins), _ptr(V), k, float(alpha), float(c0), float(beta), _ptr(U),
                                                 _ptr(out), int(bool(refresh_c))))
        return out

    def cheb_apply(self, spins, V, d, a, b, a_L, out=None, refresh_c=True):
        """moto_cheb_apply: out = -p_d(Hess) V (the transformed operator of the solver), tangent V, k <= 2."""
        _dev_f64(spins, (self.N, 3))
        k = V.shape[0]
        _dev_f64(V, (k, self.N, 3))
        out = out if out is not None else self._empty(k, self.N, 3)
        self._check(self.lib.moto_cheb_apply(self._h, _ptr(spins), _ptr(V), k, int(d), float(a), float(b), float(a_L), _ptr(out),
                                             int(bool(refresh_c))))
        return out

    def lowest_modes(self, spins, k, tol, max_iter=200, V0=None, allow_notconv=False):
        """moto_lowest_modes -> (lam [k], V [k][N][3], info dict)."""
        _dev_f64(spins, (self.N, 3))
        lam = self._empty(k)
        if V0 is not None:
            V = _dev_f64(V0, (k, self.N, 3)).clone()
            warm = 1
        else:
            V = self._empty(k, self.N, 3)
            warm = 0
        info = SolveInfo()
        st = self._check(self.lib.moto_lowest_modes(self._h, _ptr(spins), k, float(tol), int(max_iter), warm, _ptr(lam),
                                                    _ptr(V), C.byref(info)), allow=(ENOTCONV,) if allow_notconv else ())
        return lam, V, dict(iters=info.iters, converged=bool(info.converged), resid=list(info.resid)[:k],
                            hvp_count=info.hvp_count, status=st)

    def mmf_step(self, spins, v, dt, out=None, want_fnorm=True):
        """moto_mmf_step -> (spins', |F_mmf| [1] device tensor or None)."""
        _dev_f64(spins, (self.N, 3))
        kr = v.shape[0]
        _dev_f64(v, (kr, self.N, 3))
        out = out if out is not None else self._empty(self.N, 3)
        fn = self._empty(1) if want_fnorm else None
        self._check(self.lib.moto_mmf_step(self._h, _ptr(spins), _ptr(v), kr, float(dt), _ptr(out), _ptr(fn)))
        return out, fn

    def mmf_run(self, state, k, dt, max_steps, tau_F, tol, max_iter=20000, V0=None):
        """moto_mmf_run: outer MMF loop with the saddle test; `state` is updated in place.  -> (V, info dict)."""
        _dev_f64(state, (self.N, 3))
        if V0 is not None:
            V, warm = _dev_f64(V0, (k, self.N, 3)).clone(), 1
        else:
            V, warm = self._empty(k, self.N, 3), 0
        info = MmfInfo()
        st = self._check(self.lib.moto_mmf_run(self._h, _ptr(state), k, float(dt), int(max_steps), float(tau_F), float(tol),
                                               int(max_iter), warm, _ptr(V), C.byref(info)), allow=(ENOTCONV,))
        return V, dict(steps=info.steps, converged=bool(info.converged), fnorm=info.fnorm, lam=list(info.lam)[:k],
                       hvp_count=info.hvp_count, solver_iters=info.solver_iters, status=st)

    def mmf_run_cg(self, state, k, delta, smax, max_steps, tau_F, tol, max_iter=20000, V0=None):
        """moto_mmf_run_cg: outer MMF loop with the CG step rule; `state` is updated in place.  -> (V, info dict)."""
        _dev_f64(state, (self.N, 3))
        if V0 is not None:
            V, warm = _dev_f64(V0, (k, self.N, 3)).clone(), 1
        else:
            V, warm = self._empty(k, self.N, 3), 0
        scratch = self._empty(4, self.N, 3)
        info = MmfInfo()
        st = self._check(self.lib.moto_mmf_run_cg(self._h, _ptr(state), k, float(delta), float(smax), int(max_steps), float(tau_F),
                                                  float(tol), int(max_iter), warm, _ptr(V), _ptr(scratch), C.byref(info)), allow=(ENOTCONV,))
        return V, dict(steps=info.steps, converged=bool(info.converged), fnorm=info.fnorm, lam=list(info.lam)[:k],
                       hvp_count=info.hvp_count, solver_iters=info.solver_iters, status=st)

    def mmf_run_lbfgs(self, state, k, alpha0, smax, max_steps, tau_F, tol, max_iter=20000, V0=None, m=8):
        """moto_mmf_run_lbfgs: outer MMF loop with the L-BFGS step rule; `state` is updated in place.  -> (V, info dict)."""
        _dev_f64(state, (self.N, 3))
        if V0 is not None:
            V, warm = _dev_f64(V0, (k, self.N, 3)).clone(), 1
        else:
            V, warm = self._empty(k, self.N, 3), 0
        scratch = self._empty(2 * m + 4, self.N, 3)
        info = MmfInfo()
        st = self._check(self.lib.moto_mmf_run_lbfgs(self._h, _ptr(state), k, float(alpha0), float(smax), int(max_steps), float(tau_F),
                                                     float(tol), int(max_iter), warm, int(m), _ptr(V), _ptr(scratch), C.byref(info)),
                         allow=(ENOTCONV,))
        return V, dict(steps=info.steps, converged=bool(info.converged), fnorm=info.fnorm, lam=list(info.lam)[:k],
                       hvp_count=info.hvp_count, solver_iters=info.solver_iters, status=st)

    def relax_lbfgs(self, state, max_steps, tau_F, alpha0, m=8):
        """moto_relax_lbfgs: relax `state` downhill in place (L-BFGS, history m).  -> info dict."""
        _dev_f64(state, (self.N, 3))
        scratch = self._empty(2 * m + 5, self.N, 3)
        info = RelaxInfo()
        st = self._check(self.lib.moto_relax_lbfgs(self._h, _ptr(state), int(max_steps), float(tau_F), float(alpha0), int(m), _ptr(scratch),
                                                   C.byref(info)), allow=(ENOTCONV,))
        return info.as_dict(st)

    def relax(self, state, max_steps, tau_F, alpha0):
        """moto_relax: relax `state` downhill in place (CG + backtracking).  -> info dict."""
        _dev_f64(state, (self.N, 3))
        info = RelaxInfo()
        st = self._check(self.lib.moto_relax(self._h, _ptr(state), int(max_steps), float(tau_F), float(alpha0), C.byref(info)),
                         allow=(ENOTCONV,))
        return info.as_dict(st)

    def two_sided_descent(self, saddle, vmin, eta, max_steps, tau_F, alpha0):
        """moto_two_sided_descent -> (x_min(+eta), x_min(-eta), [info dict, info dict])."""
        _dev_f64(saddle, (self.N, 3))
        _dev_f64(vmin, (self.N, 3))
        xp, xm = self._empty(self.N, 3), self._empty(self.N, 3)
        info = (RelaxInfo * 2)()
        st = self._check(self.lib.moto_two_sided_descent(self._h, _ptr(saddle), _ptr(vmin), float(eta), int(max_steps), float(tau_F),
                                                         float(alpha0), _ptr(xp), _ptr(xm), info), allow=(ENOTCONV,))
        return xp, xm, [info[0].as_dict(st), info[1].as_dict(st)]

    def transport(self, spins_new, V):
        k = V.shape[0]
        _dev_f64(V, (k, self.N, 3))
        self._check(self.lib.moto_transport(self._h, _ptr(spins_new), _ptr(V), k))
        return V

    def gram(self, S, T):
        ns, nt = S.shape[0], T.shape[0]
        _dev_f64(S, (ns, self.N, 3)); _dev_f64(T, (nt, self.N, 3))
        G = self._empty(ns, nt)
        self._check(self.lib.moto_gram(self._h, _ptr(S), ns, _ptr(T), nt, _ptr(G)))
        return G

    def rayleigh_ritz(self, GA, GB, nev):
        n = GA.shape[0]
        _dev_f64(GA, (n, n)); _dev_f64(GB, (n, n))
        theta = self._empty(nev)
        Cm = self._empty(n, nev)
        self._check(self.lib.moto_rayleigh_ritz(self._h, _ptr(GA), _ptr(GB), n, nev, _ptr(theta), _ptr(Cm)))
        return theta, Cm

    # -- host-buffer API (numpy arrays, pinned or pageable)
    def energy_grad_host(self, h_spins, h_g=None):
        E = np.zeros(1)
        self._check(self.lib.moto_energy_grad_host(self._h, _ptr(h_spins), _ptr(E), _ptr(h_g)))
        return float(E[0]), h_g

    def hvp_host(self, h_spins, h_V, h_HV):
        self._check(self.lib.moto_hvp_host(self._h, _ptr(h_spins), _ptr(h_V), h_V.shape[0], _ptr(h_HV)))
        return h_HV

    def lowest_modes_host(self, h_spins, k, tol, max_iter, h_lam, h_V, warm=False, allow_notconv=False):
        info = SolveInfo()
        st = self._check(self.lib.moto_lowest_modes_host(self._h, _ptr(h_spins), k, float(tol), int(max_iter), int(warm),
                                                         _ptr(h_lam), _ptr(h_V), C.byref(info)),
                         allow=(ENOTCONV,) if allow_notconv else ())
        return dict(iters=info.iters, converged=bool(info.converged), resid=list(info.resid)[:k],
                    hvp_count=info.hvp_count, status=st)

    def mmf_step_host(self, h_spins, h_v, dt, h_out):
        fn = np.zeros(1)
        self._check(self.lib.moto_mmf_step_host(self._h, _ptr(h_spins), _ptr(h_v), h_v.shape[0], float(dt), _ptr(h_out),
                                                _ptr(fn)))
        return h_out, float(fn[0])


def lowest_modes_batch(ctxs, spins, k, tol, max_iter=200, V0=None, allow_notconv=False):
    """moto_lowest_modes_batch over P contexts (each on its own stream) -> ([lam_p], [V_p], [info dict_p]).
    Synchronises the device first: the contexts' streams are not ordered against the stream that produced the inputs."""
    import torch
    P = len(ctxs)
    lib = load_library()
    lams = [c._empty(k) for c in ctxs]
    Vs = [(_dev_f64(V0[p], (k, c.N, 3)).clone() if V0 is not None else c._empty(k, c.N, 3)) for p, c in enumerate(ctxs)]
    for p, c in enumerate(ctxs):
        _dev_f64(spins[p], (c.N, 3))
    torch.cuda.synchronize()
    H = (C.c_void_p * P)(*[c._h for c in ctxs])
    S = (C.c_void_p * P)(*[_ptr(s) for s in spins])
    L = (C.c_void_p * P)(*[_ptr(t) for t in lams])
    VV = (C.c_void_p * P)(*[_ptr(t) for t in Vs])
    infos = (SolveInfo * P)()
    sts = (C.c_int32 * P)()
    st = lib.moto_lowest_modes_batch(H, P, S, k, float(tol), int(max_iter), 1 if V0 is not None else 0, L, VV, infos, sts)
    for p, c in enumerate(ctxs):
        c._check(sts[p], allow=(ENOTCONV,) if allow_notconv else ())
    if st not in (OK, ENOTCONV):
        raise MotoError(st, "moto_lowest_modes_batch failed")
    out = [dict(iters=i.iters, converged=bool(i.converged), resid=list(i.resid)[:k], hvp_count=i.hvp_count, status=sts[p])
           for p, i in enumerate(infos)]
    return lams, Vs, out


def gram_static(S, T, G, stream=None):
    """moto_gram_static: G [ns][nt] <- S [ns][...] . T [nt][...] with no context, no workspace and no allocation (the caller
    passes the output; ns <= 6, nt <= 12).  stream: a raw cudaStream_t handle (int) or None for the default stream."""
    lib = load_library()
    ns, nt = S.shape[0], T.shape[0]
    _dev_f64(S); _dev_f64(T); _dev_f64(G, (ns, nt))
    n3 = S[0].numel()
    assert T[0].numel() == n3, "S and T rows differ in length"
    st = lib.moto_gram_static(_ptr(S), ns, _ptr(T), nt, n3, _ptr(G), stream)
    if st != OK:
        raise MotoError(st, lib.moto_gram_static_last_error().decode())
    return G


def spin_context(w, kmax=None, device="cuda:0", stream=None) -> Context:
    """Context for a workloads.SpinWorkload."""
    lat = Lattice(KIND_TRI2D, w.Lx, w.Ly, w.pbc_x, w.pbc_y, 0)
    p = SpinParams(w.J, w.D, w.K, (C.c_double * 3)(*w.B), w.mu)
    return Context(lat, p, kmax=kmax or w.k, device=device, stream=stream)


def cart_context(w, kmax=None, device="cuda:0", stream=None) -> Context:
    """Context for a workloads.CartWorkload."""
    lat = Lattice(KIND_CARTESIAN, 0, 0, 1, 1, w.Na)
    for a in range(2):
        for b in range(2):
            lat.cell[a][b] = float(w.cell[a][b])
    p = MorseParams(w.De, w.alpha, w.r0, w.rc)
    return Context(lat, p, kmax=kmax or w.k, device=device, stream=stream, fixed=w.fixed)


def shell_context(w, kmax=None, device="cuda:0", stream=None) -> Context:
    """Context for a workloads.ShellWorkload: a spin lattice whose couplings come from the neighbour table (moto_set_shells)."""
    lat = Lattice(KIND_TRI2D, w.Lx, w.Ly, w.pbc_x, w.pbc_y, 0)
    p = SpinParams(0.0, 0.0, w.K, (C.c_double * 3)(*w.B), w.mu)
    ctx = Context(lat, p, kmax=kmax or w.k, device=device, stream=stream)
    ctx.set_shells(w.offsets, w.Jd, w.Dd)
    return ctx
