"""Thin ctypes binding of libhqmc.so (include/hqmc.h).  Argument marshalling only: every step of the
hot path runs in the library's CUDA kernels.  PyTorch is used for device memory and streams.

There is NO CPU fallback: importing this module raises if libhqmc.so is missing, and every compute
call raises HqmcError if the library reports an error (e.g. no CUDA device).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libhqmc.so")

HQMC_OK, HQMC_EINVAL, HQMC_ECUDA, HQMC_ENOCONV, HQMC_ENOMEM = 0, -1, -2, -3, -4
K_MDAGM, K_AXPY, K_PRECOND, K_DUPDATE, K_M, K_FORCE, K_PHASE, K_MISC, K_COUNT = range(9)
MDAGM_AUTO, MDAGM_REGISTER, MDAGM_CLUSTER, MDAGM_STREAM = 0, 1, 2, 3
CG_AUTO, CG_TEXTBOOK, CG_DEFERRED_X = 0, 1, 2
PERSIST_AUTO, PERSIST_OFF, PERSIST_ON = 0, 1, 2
KERNEL_CLASSES = ["mdagm", "cg_axpy", "precond", "cg_dupdate", "apply_M", "force", "phase", "misc"]

# every symbol include/hqmc.h and include/hqmc_tuning.h declare
SYMBOLS = [
    "hqmc_create", "hqmc_destroy", "hqmc_set_precond", "hqmc_get_precond", "hqmc_set_theta", "hqmc_apply_M",
    "hqmc_apply_Mdag", "hqmc_apply_MdagM", "hqmc_precond", "hqmc_cg_solve", "hqmc_force", "hqmc_force_boson",
    "hqmc_energies", "hqmc_leapfrog_trajectory", "hqmc_hqmc_step", "hqmc_rng_raw", "hqmc_rng_gauss", "hqmc_rng_uniform", "hqmc_sweep", "hqmc_sweep_batched", "hqmc_cg_solve_batched", "hqmc_leapfrog_trajectory_batched", "hqmc_refresh_batched", "hqmc_hqmc_step_batched", "hqmc_set_green_batch", "hqmc_green_apply", "hqmc_translation_average", "hqmc_green_2pt",
    "hqmc_pair_correlator", "hqmc_apply_MdagM_host", "hqmc_refresh_host", "hqmc_cg_solve_host",
    "hqmc_leapfrog_trajectory_host", "hqmc_action_boson_noalloc", "hqmc_slab_dot", "hqmc_slab_axpy", "hqmc_slab_dupdate",
    "hqmc_slab_scale", "hqmc_slab_sum_rows", "hqmc_slab_field_axpy", "hqmc_slab_action_boson", "hqmc_set_profiling", "hqmc_reset_stats", "hqmc_get_kernel_stats",
    "hqmc_set_time_tile", "hqmc_set_mdagm_kernel", "hqmc_set_precond_tile", "hqmc_set_cg_variant", "hqmc_set_cg_persistent", "hqmc_set_md_graph", "hqmc_set_pdl", "hqmc_set_debug_skip", "hqmc_strerror", "hqmc_last_error", "hqmc_version",
]


class HqmcError(RuntimeError):
    pass


class _Params(C.Structure):
    _fields_ = [("L", C.c_int), ("Ntau", C.c_int), ("dtau", C.c_double), ("t", C.c_double), ("c_tau", C.c_double),
                ("K", C.c_double), ("compact", C.c_int), ("precond_W", C.c_int), ("prec", C.c_int)]


if not os.path.exists(LIB_PATH):
    raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2508_16298_b200.build` "
                      "(there is no CPU fallback)")
_lib = C.CDLL(LIB_PATH)
_lib.hqmc_strerror.restype = C.c_char_p
_lib.hqmc_last_error.restype = C.c_char_p
_lib.hqmc_rng_uniform.restype = C.c_double
for _s in SYMBOLS:
    getattr(_lib, _s)  # raises AttributeError if a declared symbol is not exported


def _check(status: int, allow_noconv: bool = False) -> int:
    if status == HQMC_OK or (allow_noconv and status == HQMC_ENOCONV):
        return status
    raise HqmcError(f"{_lib.hqmc_strerror(status).decode()} ({status}): {_lib.hqmc_last_error().decode()}")


def _ptr(t: torch.Tensor) -> C.c_void_p:
    return C.c_void_p(t.data_ptr())


class HQMC:
    """One lattice + couplings on one GPU.  Vectors are torch complex tensors [Ntau, L, L] on the device,
    theta / p / forces are float64 tensors [Ntau, 2, L, L]."""

    def __init__(self, L, Ntau, dtau=0.1, t=1.0, c_tau=1.0, K=1.0, compact=True, W=6, prec="c128", device="cuda:0"):
        self.L, self.Ntau, self.N = L, Ntau, L * L * Ntau
        self.device = torch.device(device)
        self.cdtype = torch.complex128 if prec == "c128" else torch.complex64
        self.np_cdtype = np.complex128 if prec == "c128" else np.complex64
        p = _Params(L, Ntau, dtau, t, c_tau, K, int(compact), W, 0 if prec == "c128" else 1)
        self._ctx = C.c_void_p()
        if self.device.type == "cuda":
            torch.cuda.set_device(self.device)
            stream = torch.cuda.current_stream(self.device).cuda_stream
        else:
            stream = 0
        _check(_lib.hqmc_create(C.byref(p), C.c_void_p(stream), C.byref(self._ctx)))

    def close(self):
        if self._ctx:
            _lib.hqmc_destroy(self._ctx)
            self._ctx = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- helpers ------------------------------------------------------------------------------
    def _vec(self, v):
        assert v.is_cuda and v.dtype == self.cdtype and v.numel() == self.N and v.is_contiguous()
        return v

    def _field(self, f):
        assert f.is_cuda and f.dtype == torch.float64 and f.numel() == 2 * self.N and f.is_contiguous()
        return f

    def new_vec(self):
        return torch.empty((self.Ntau, self.L, self.L), dtype=self.cdtype, device=self.device)

    def new_field(self):
        return torch.empty((self.Ntau, 2, self.L, self.L), dtype=torch.float64, device=self.device)

    # ---- setup --------------------------------------------------------------------------------
    def set_theta(self, theta):
        _check(_lib.hqmc_set_theta(self._ctx, _ptr(self._field(theta))))

    def set_precond(self, taps):
        taps = np.ascontiguousarray(taps, dtype=np.float64)
        _check(_lib.hqmc_set_precond(self._ctx, C.c_int(len(taps) - 1), taps.ctypes.data_as(C.c_void_p)))

    def get_precond(self):
        W = C.c_int(0)
        taps = np.zeros(33)
        _check(_lib.hqmc_get_precond(self._ctx, C.byref(W), taps.ctypes.data_as(C.c_void_p)))
        return taps[: W.value + 1].copy()

    def set_time_tile(self, tt: int):
        _check(_lib.hqmc_set_time_tile(self._ctx, C.c_int(tt)))

    def set_mdagm_kernel(self, which: int):
        """MDAGM_AUTO / MDAGM_REGISTER / MDAGM_CLUSTER / MDAGM_STREAM (include/hqmc_tuning.h)."""
        _check(_lib.hqmc_set_mdagm_kernel(self._ctx, C.c_int(which)))

    def set_precond_tile(self, slices_per_run: int):
        _check(_lib.hqmc_set_precond_tile(self._ctx, C.c_int(slices_per_run)))

    def set_cg_variant(self, which: int):
        """CG_AUTO / CG_TEXTBOOK / CG_DEFERRED_X (include/hqmc_tuning.h)."""
        _check(_lib.hqmc_set_cg_variant(self._ctx, C.c_int(int(which))))

    def set_cg_persistent(self, mode: int):
        """PERSIST_AUTO / PERSIST_OFF / PERSIST_ON: the whole-solve persistent kernel (include/hqmc_tuning.h)."""
        _check(_lib.hqmc_set_cg_persistent(self._ctx, C.c_int(int(mode))))

    def set_md_graph(self, on: bool):
        _check(_lib.hqmc_set_md_graph(self._ctx, C.c_int(int(on))))

    def set_pdl(self, on: int):
        _check(_lib.hqmc_set_pdl(self._ctx, C.c_int(int(on))))

    def set_debug_skip(self, mask: int):
        """Timing only: do not launch the kernel classes whose bit is set (results become meaningless)."""
        _check(_lib.hqmc_set_debug_skip(self._ctx, C.c_uint(mask)))

    # ---- operators ----------------------------------------------------------------------------
    def _apply(self, fn, v, out):
        out = self.new_vec() if out is None else out
        _check(fn(self._ctx, _ptr(self._vec(v)), _ptr(self._vec(out))))
        return out

    def apply_M(self, v, out=None):
        return self._apply(_lib.hqmc_apply_M, v, out)

    def apply_Mdag(self, v, out=None):
        return self._apply(_lib.hqmc_apply_Mdag, v, out)

    def apply_MdagM(self, v, out=None):
        return self._apply(_lib.hqmc_apply_MdagM, v, out)

    def precond(self, v, out=None):
        return self._apply(_lib.hqmc_precond, v, out)

    def cg_solve(self, rhs, tol=1e-10, max_iter=1000000, x=None):
        """-> (x, iterations, relative recurrence residual, converged)."""
        x = self.new_vec() if x is None else x
        it, rel = C.c_longlong(0), C.c_double(0.0)
        s = _check(_lib.hqmc_cg_solve(self._ctx, _ptr(self._vec(rhs)), _ptr(self._vec(x)), C.c_double(tol),
                                      C.c_longlong(max_iter), C.byref(it), C.byref(rel)), allow_noconv=True)
        return x, it.value, rel.value, s == HQMC_OK

    def force(self, x, out=None):
        out = self.new_field() if out is None else out
        _check(_lib.hqmc_force(self._ctx, _ptr(self._vec(x)), _ptr(self._field(out))))
        return out

    def force_boson(self, out=None):
        out = self.new_field() if out is None else out
        _check(_lib.hqmc_force_boson(self._ctx, _ptr(self._field(out))))
        return out

    def energies(self, p=None, phi=None, x=None):
        """-> (S_B, sum p^2, S_F) at the context's theta."""
        SB, p2, SF = C.c_double(0), C.c_double(0), C.c_double(0)
        _check(_lib.hqmc_energies(self._ctx, _ptr(self._field(p)) if p is not None else None,
                                  _ptr(self._vec(phi)) if phi is not None else None,
                                  _ptr(self._vec(x)) if x is not None else None, C.byref(SB), C.byref(p2), C.byref(SF)))
        return SB.value, p2.value, SF.value

    def trajectory(self, theta, p, phi, nsteps, eps, cg_tol=1e-10, cg_max_iter=1000000):
        """In place on theta, p.  -> dict(H0, H1, cg_iters, converged)."""
        H0, H1, it = C.c_double(0), C.c_double(0), C.c_longlong(0)
        s = _check(_lib.hqmc_leapfrog_trajectory(self._ctx, _ptr(self._field(theta)), _ptr(self._field(p)),
                                                 _ptr(self._vec(phi)), C.c_int(nsteps), C.c_double(eps), C.c_double(cg_tol),
                                                 C.c_longlong(cg_max_iter), C.byref(H0), C.byref(H1), C.byref(it)),
                   allow_noconv=True)
        return dict(H0=H0.value, H1=H1.value, cg_iters=it.value, converged=(s == HQMC_OK))

    def hqmc_step(self, theta, p, eta, u, nsteps, eps, cg_tol=1e-10, cg_max_iter=1000000):
        """One HQMC update, in place on theta (restored on rejection) and p.
        -> dict(H0, H1, accepted, cg_iters, converged)."""
        H0, H1, it, acc = C.c_double(0), C.c_double(0), C.c_longlong(0), C.c_int(0)
        s = _check(_lib.hqmc_hqmc_step(self._ctx, _ptr(self._field(theta)), _ptr(self._field(p)), _ptr(self._vec(eta)),
                                       C.c_double(u), C.c_int(nsteps), C.c_double(eps), C.c_double(cg_tol), C.c_longlong(cg_max_iter),
                                       C.byref(H0), C.byref(H1), C.byref(acc), C.byref(it)), allow_noconv=True)
        return dict(H0=H0.value, H1=H1.value, accepted=bool(acc.value), cg_iters=it.value, converged=(s == HQMC_OK))

    # ---- on-device random numbers and the sweep loop --------------------------
    def rng_raw(self, seed, update, stream, n):
        """The four Philox4x32-10 words of elements 0..n-1 -> uint32 tensor [n, 4] (bit-identical to the CPU twin)."""
        out = torch.empty((n, 4), dtype=torch.int32, device=self.device)
        _check(_lib.hqmc_rng_raw(self._ctx, C.c_ulonglong(seed), C.c_uint(update), C.c_uint(stream), C.c_longlong(n), _ptr(out)))
        return out

    def rng_gauss(self, seed, update, stream, n):
        """n pairs of independent N(0, 1/2) -> float64 tensor [n, 2]."""
        out = torch.empty((n, 2), dtype=torch.float64, device=self.device)
        _check(_lib.hqmc_rng_gauss(self._ctx, C.c_ulonglong(seed), C.c_uint(update), C.c_uint(stream), C.c_longlong(n), _ptr(out)))
        return out

    @staticmethod
    def rng_uniform(seed, update):
        return float(_lib.hqmc_rng_uniform(C.c_ulonglong(seed), C.c_uint(update)))

    def sweep(self, theta, seed, first_update, n_updates, nsteps, eps, cg_tol=1e-10, cg_max_iter=1000000):
        """n_updates HQMC updates in place on theta, every random number drawn by the library
        -> dict(H0[], H1[], accepted[], cg_iters[], converged)."""
        n = n_updates
        H0, H1, it, acc = (C.c_double * n)(), (C.c_double * n)(), (C.c_longlong * n)(), (C.c_int * n)()
        s = _check(_lib.hqmc_sweep(self._ctx, _ptr(self._field(theta)), C.c_ulonglong(seed), C.c_uint(first_update), C.c_int(n),
                                   C.c_int(nsteps), C.c_double(eps), C.c_double(cg_tol), C.c_longlong(cg_max_iter), H0, H1, acc, it),
                   allow_noconv=True)
        return dict(H0=list(H0), H1=list(H1), accepted=[bool(a) for a in acc], cg_iters=list(it), converged=(s == HQMC_OK))

    def sweep_batched(self, theta, seed, first_update, n_updates, nsteps, eps, cg_tol=1e-10, cg_max_iter=1000000):
        """n_updates HQMC updates of the n chains stacked in theta [n][Ntau][2][L][L] (in place); chain b draws what `sweep` draws
        from seed + b -> dict(H0, H1, accepted, cg_iters: lists [update][chain], converged)."""
        assert theta.is_cuda and theta.dtype == torch.float64 and theta.is_contiguous() and theta.numel() % (2 * self.N) == 0
        n, m = theta.numel() // (2 * self.N), n_updates
        H0, H1, it, acc = (C.c_double * (n * m))(), (C.c_double * (n * m))(), (C.c_longlong * (n * m))(), (C.c_int * (n * m))()
        s = _check(_lib.hqmc_sweep_batched(self._ctx, _ptr(theta), C.c_ulonglong(seed), C.c_uint(first_update), C.c_int(m), C.c_int(n),
                                           C.c_int(nsteps), C.c_double(eps), C.c_double(cg_tol), C.c_longlong(cg_max_iter), H0, H1, acc, it),
                   allow_noconv=True)
        rows = lambda a, f: [[f(a[k * n + b]) for b in range(n)] for k in range(m)]
        return dict(H0=rows(H0, float), H1=rows(H1, float), accepted=rows(acc, bool), cg_iters=rows(it, int), converged=(s == HQMC_OK))

    # ---- stochastic estimator -------------------------------------------------
    def _vecs(self, v):
        assert v.is_cuda and v.dtype == self.cdtype and v.is_contiguous() and v.numel() % self.N == 0 and v.numel() >= self.N
        return v, v.numel() // self.N

    def refresh_batched(self, theta, eta, out=None):
        """phi_b = M^+(theta_b) eta_b for stacked chains: theta [n][Ntau][2][L][L], eta [n][Ntau][L][L]."""
        eta, n = self._vecs(eta)
        assert theta.is_cuda and theta.dtype == torch.float64 and theta.is_contiguous() and theta.numel() == 2 * self.N * n
        out = torch.empty_like(eta) if out is None else out
        _check(_lib.hqmc_refresh_batched(self._ctx, _ptr(theta), _ptr(eta), _ptr(out), C.c_int(n)))
        return out

    def trajectory_batched(self, theta, p, phi, nsteps, eps, cg_tol=1e-10, cg_max_iter=1000000):
        """n independent chains advanced together; theta, p [n][Ntau][2][L][L] are updated in place
        -> dict(H0[n], H1[n], cg_iters[n], converged)."""
        phi, n = self._vecs(phi)
        for f in (theta, p):
            assert f.is_cuda and f.dtype == torch.float64 and f.is_contiguous() and f.numel() == 2 * self.N * n
        H0, H1, it = (C.c_double * n)(), (C.c_double * n)(), (C.c_longlong * n)()
        s = _check(_lib.hqmc_leapfrog_trajectory_batched(self._ctx, _ptr(theta), _ptr(p), _ptr(phi), C.c_int(n), C.c_int(nsteps),
                                                         C.c_double(eps), C.c_double(cg_tol), C.c_longlong(cg_max_iter), H0, H1, it),
                   allow_noconv=True)
        return dict(H0=list(H0), H1=list(H1), cg_iters=list(it), converged=(s == HQMC_OK))

    def hqmc_step_batched(self, theta, p, eta, u, nsteps, eps, cg_tol=1e-10, cg_max_iter=1000000):
        """One HQMC update of n chains (refresh, trajectory, Metropolis with the uniforms u[n], restore on rejection)."""
        eta, n = self._vecs(eta)
        for f in (theta, p):
            assert f.is_cuda and f.dtype == torch.float64 and f.is_contiguous() and f.numel() == 2 * self.N * n
        assert len(u) == n
        H0, H1, it, acc = (C.c_double * n)(), (C.c_double * n)(), (C.c_longlong * n)(), (C.c_int * n)()
        s = _check(_lib.hqmc_hqmc_step_batched(self._ctx, _ptr(theta), _ptr(p), _ptr(eta), (C.c_double * n)(*[float(v) for v in u]),
                                               C.c_int(n), C.c_int(nsteps), C.c_double(eps), C.c_double(cg_tol), C.c_longlong(cg_max_iter),
                                               H0, H1, acc, it), allow_noconv=True)
        return dict(H0=list(H0), H1=list(H1), accepted=[bool(a) for a in acc], cg_iters=list(it), converged=(s == HQMC_OK))

    def cg_solve_batched(self, rhs, tol=1e-10, max_iter=1000000, x=None):
        """M^+M x_b = rhs_b for the stacked right-hand sides [n][Ntau][L][L], all advancing in the same launches
        -> (x, iterations[n], relative recurrence residuals[n], all converged)."""
        rhs, n = self._vecs(rhs)
        x = torch.empty_like(rhs) if x is None else x
        it, rel = (C.c_longlong * n)(), (C.c_double * n)()
        s = _check(_lib.hqmc_cg_solve_batched(self._ctx, _ptr(rhs), _ptr(x), C.c_int(n), C.c_double(tol), C.c_longlong(max_iter),
                                              it, rel), allow_noconv=True)
        return x, list(it), list(rel), s == HQMC_OK

    def set_green_batch(self, n: int):
        """Vectors green_apply solves per launch (0 = by L2 footprint, 1 = one at a time)."""
        _check(_lib.hqmc_set_green_batch(self._ctx, C.c_int(n)))

    def green_apply(self, xi, tol=1e-10, max_iter=1000000, out=None):
        """g_k = (M^+M)^{-1} M^+ xi_k for the stacked vectors xi [n_rv][Ntau][L][L] -> (g, total iterations, converged)."""
        xi, n = self._vecs(xi)
        out = torch.empty_like(xi) if out is None else out
        it = C.c_longlong(0)
        s = _check(_lib.hqmc_green_apply(self._ctx, _ptr(xi), _ptr(out), C.c_int(n), C.c_double(tol), C.c_longlong(max_iter),
                                         C.byref(it)), allow_noconv=True)
        return out, it.value, s == HQMC_OK

    def translation_average(self, a, b, out=None):
        """Eq.17-19: C(Delta) = (1/N) sum_i a_i b_{i+Delta}."""
        out = self.new_vec() if out is None else out
        _check(_lib.hqmc_translation_average(self._ctx, _ptr(self._vec(a)), _ptr(self._vec(b)), _ptr(self._vec(out))))
        return out

    def green_2pt(self, g, xi, out=None):
        g, n = self._vecs(g)
        xi, n2 = self._vecs(xi)
        assert n == n2
        out = self.new_vec() if out is None else out
        _check(_lib.hqmc_green_2pt(self._ctx, _ptr(g), _ptr(xi), C.c_int(n), _ptr(self._vec(out))))
        return out

    def pair_correlator(self, g, xi, out=None):
        g, n = self._vecs(g)
        xi, n2 = self._vecs(xi)
        assert n == n2 and n >= 2
        out = self.new_vec() if out is None else out
        _check(_lib.hqmc_pair_correlator(self._ctx, _ptr(g), _ptr(xi), C.c_int(n), _ptr(self._vec(out))))
        return out

    # ---- vector steps of the tau-slab PCG (include/hqmc.h "tau-slab sharding"; the loop is slab.py) --------------
    def slab_dot(self, a, b, out):
        """out[0] = Re <a, b> over the (contiguous) views a, b; out: a device float64 view."""
        assert a.is_contiguous() and b.is_contiguous() and a.numel() == b.numel() and a.dtype == b.dtype == self.cdtype
        _check(_lib.hqmc_slab_dot(self._ctx, _ptr(a), _ptr(b), C.c_longlong(a.numel()), _ptr(out)))

    def slab_axpy(self, x, r, d, Od, num, den, rr_out):
        for v in (x, r, d, Od):
            assert v.is_contiguous() and v.dtype == self.cdtype and v.numel() == x.numel()
        _check(_lib.hqmc_slab_axpy(self._ctx, _ptr(x), _ptr(r), _ptr(d), _ptr(Od), C.c_longlong(x.numel()), _ptr(num), _ptr(den),
                                   _ptr(rr_out)))

    def slab_dupdate(self, d, z, num, den):
        assert d.is_contiguous() and z.is_contiguous() and d.numel() == z.numel() and d.dtype == z.dtype == self.cdtype
        _check(_lib.hqmc_slab_dupdate(self._ctx, _ptr(d), _ptr(z), C.c_longlong(d.numel()), _ptr(num), _ptr(den)))

    def slab_scale(self, v, s):
        assert v.is_contiguous() and v.dtype == self.cdtype
        _check(_lib.hqmc_slab_scale(self._ctx, _ptr(v), C.c_longlong(v.numel()), C.c_double(s)))

    def slab_field_axpy(self, y, x, a):
        """y += a x on float64 views (drift and kicks of a slab's owned slices)."""
        assert y.is_contiguous() and x.is_contiguous() and y.dtype == x.dtype == torch.float64 and y.numel() == x.numel()
        _check(_lib.hqmc_slab_field_axpy(self._ctx, _ptr(y), _ptr(x), C.c_double(a), C.c_longlong(y.numel())))

    def slab_action_boson(self, first_slice, n_slices, out):
        """out[0] = the share of S_B of slices [first_slice, first_slice + n_slices) of the context's theta."""
        _check(_lib.hqmc_slab_action_boson(self._ctx, C.c_int(first_slice), C.c_int(n_slices), _ptr(out)))

    def slab_sum_rows(self, rows, c0, c1, out):
        """out[c0:c1] = sum over the rows (in order) of rows[:, c0:c1]; rows [k, m] and out [m]: device float64."""
        assert rows.dim() == 2 and rows.is_contiguous() and rows.dtype == out.dtype == torch.float64 and 0 <= c0 < c1 <= rows.shape[1]
        _check(_lib.hqmc_slab_sum_rows(self._ctx, C.c_void_p(rows.data_ptr() + 8 * c0), C.c_int(rows.shape[0]),
                                       C.c_int(rows.shape[1]), C.c_int(c1 - c0), C.c_void_p(out.data_ptr() + 8 * c0)))

    # ---- host-buffer entry points (numpy arrays, pageable or pinned) ----------------------------
    def apply_MdagM_host(self, h_in: np.ndarray, h_out: np.ndarray):
        assert h_in.dtype == self.np_cdtype and h_out.dtype == self.np_cdtype and h_in.size == self.N == h_out.size
        _check(_lib.hqmc_apply_MdagM_host(self._ctx, h_in.ctypes.data_as(C.c_void_p), h_out.ctypes.data_as(C.c_void_p)))
        return h_out

    def refresh_host(self, h_theta, h_eta, h_phi):
        th = h_theta.ctypes.data_as(C.c_void_p) if h_theta is not None else None
        _check(_lib.hqmc_refresh_host(self._ctx, th, h_eta.ctypes.data_as(C.c_void_p), h_phi.ctypes.data_as(C.c_void_p)))
        return h_phi

    def cg_solve_host(self, h_theta, h_rhs, h_x, tol=1e-10, max_iter=1000000):
        it, rel = C.c_longlong(0), C.c_double(0.0)
        th = h_theta.ctypes.data_as(C.c_void_p) if h_theta is not None else None
        s = _check(_lib.hqmc_cg_solve_host(self._ctx, th, h_rhs.ctypes.data_as(C.c_void_p), h_x.ctypes.data_as(C.c_void_p),
                                           C.c_double(tol), C.c_longlong(max_iter), C.byref(it), C.byref(rel)), allow_noconv=True)
        return h_x, it.value, rel.value, s == HQMC_OK

    def trajectory_host(self, h_theta, h_p, h_phi, nsteps, eps, cg_tol=1e-10, cg_max_iter=1000000):
        H0, H1, it = C.c_double(0), C.c_double(0), C.c_longlong(0)
        s = _check(_lib.hqmc_leapfrog_trajectory_host(self._ctx, h_theta.ctypes.data_as(C.c_void_p),
                                                      h_p.ctypes.data_as(C.c_void_p), h_phi.ctypes.data_as(C.c_void_p),
                                                      C.c_int(nsteps), C.c_double(eps), C.c_double(cg_tol),
                                                      C.c_longlong(cg_max_iter), C.byref(H0), C.byref(H1), C.byref(it)),
                   allow_noconv=True)
        return dict(H0=H0.value, H1=H1.value, cg_iters=it.value, converged=(s == HQMC_OK))

    # ---- instrumentation ----------------------------------------------------------------------
    def set_profiling(self, on: bool):
        _check(_lib.hqmc_set_profiling(self._ctx, C.c_int(int(on))))

    def reset_stats(self):
        _check(_lib.hqmc_reset_stats(self._ctx))

    def kernel_stats(self):
        """-> {class: (launches, summed device ms)}"""
        out = {}
        for i, name in enumerate(KERNEL_CLASSES):
            n, ms = C.c_longlong(0), C.c_double(0)
            _check(_lib.hqmc_get_kernel_stats(self._ctx, C.c_int(i), C.byref(n), C.byref(ms)))
            out[name] = (n.value, ms.value)
        return out


def version() -> int:
    return int(_lib.hqmc_version())


NOALLOC_MAX_LINKS = 1 << 25


def action_boson_noalloc(theta: torch.Tensor, L: int, Nt: int, c_tau: float, K: float, compact: bool, out: torch.Tensor,
                         stream=None) -> torch.Tensor:
    """S_B(theta) into the caller's device double out[0] through hqmc_action_boson_noalloc (include/hqmc.h): no context and
    no allocation anywhere -- the caller brings theta (fp64 [Nt][2][L][L], CUDA, contiguous) AND out (fp64, >= 1 element,
    CUDA).  Enqueued on `stream` (default: torch's current stream), not synchronised.  Lattices beyond NOALLOC_MAX_LINKS
    raise HqmcError; calls that overlap on the GPU race on the library's shared static scratch."""
    if not (theta.is_cuda and out.is_cuda and theta.dtype == torch.float64 and out.dtype == torch.float64
            and theta.is_contiguous() and out.numel() >= 1 and theta.numel() == 2 * L * L * Nt):
        raise ValueError("theta: contiguous CUDA fp64 [Nt][2][L][L]; out: CUDA fp64 with at least one element")
    st = torch.cuda.current_stream(theta.device).cuda_stream if stream is None else int(stream)
    with torch.cuda.device(theta.device):
        _check(_lib.hqmc_action_boson_noalloc(_ptr(theta), C.c_int(L), C.c_int(Nt), C.c_double(c_tau), C.c_double(K),
                                              C.c_int(1 if compact else 0), _ptr(out), C.c_void_p(st)))
    return out
