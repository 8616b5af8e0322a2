"""ctypes wrapper around oracle/hqmc_oracle.c -- the CPU ORACLE.  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference` legs may import
this.  It holds no arithmetic of its own: every function marshals numpy arrays into the C oracle
(see the header of hqmc_oracle.c for citations, readings and pins).  It never imports the CUDA package.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "hqmc_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain -O2, OpenMP over independent time slices)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=gnu11", "-fopenmp", "-fPIC", "-shared", "-o", _LIB, _SRC, "-lm"])
    return _LIB


class _Params(C.Structure):
    _fields_ = [("L", C.c_int), ("Ntau", C.c_int), ("dtau", C.c_double), ("t", C.c_double),
                ("c_tau", C.c_double), ("K", C.c_double), ("compact", C.c_int), ("W", C.c_int),
                ("taps", C.c_double * 33)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_pcg.restype = C.c_long
        _lib.orc_trajectory.restype = C.c_long
        _lib.orc_action_boson.restype = C.c_double
        _lib.orc_sum_p2.restype = C.c_double
        _lib.orc_max_threads.restype = C.c_int
        _lib.orc_get_threads.restype = C.c_int
        _lib.orc_hqmc_step.restype = C.c_int
    return _lib


def _c(a):  # complex128 contiguous
    a = np.ascontiguousarray(a, dtype=np.complex128)
    return a, a.ctypes.data_as(C.c_void_p)


def _d(a):
    a = np.ascontiguousarray(a, dtype=np.float64)
    return a, a.ctypes.data_as(C.c_void_p)


def set_threads(n: int) -> None:
    lib().orc_set_threads(C.c_int(int(n)))


def max_threads() -> int:
    return int(lib().orc_max_threads())


def get_threads() -> int:
    return int(lib().orc_get_threads())


def philox4x32_10(ctr, key):
    """One block of the counter-based generator both sides use (hqmc_oracle.c): 4 counter words, 2 key words -> 4 words."""
    c = (C.c_uint32 * 4)(*[int(x) & 0xFFFFFFFF for x in ctr]); k = (C.c_uint32 * 2)(*[int(x) & 0xFFFFFFFF for x in key])
    out = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, out)
    return [int(x) for x in out]


def rng_raw(seed: int, update: int, stream: int, n: int) -> np.ndarray:
    out = np.empty(4 * n, dtype=np.uint32)
    lib().orc_rng_raw(C.c_uint64(seed), C.c_uint32(update), C.c_uint32(stream), C.c_long(n), out.ctypes.data_as(C.c_void_p))
    return out.reshape(n, 4)


def rng_uniform(seed: int, update: int, stream: int, n: int) -> np.ndarray:
    out = np.empty(2 * n)
    lib().orc_rng_uniform(C.c_uint64(seed), C.c_uint32(update), C.c_uint32(stream), C.c_long(n), out.ctypes.data_as(C.c_void_p))
    return out.reshape(n, 2)


def rng_gauss(seed: int, update: int, stream: int, n: int) -> np.ndarray:
    """n pairs of independent N(0, 1/2) (reading C6): stream 0 = R as (re, im), stream 1 = p in pairs."""
    out = np.empty(2 * n)
    lib().orc_rng_gauss(C.c_uint64(seed), C.c_uint32(update), C.c_uint32(stream), C.c_long(n), out.ctypes.data_as(C.c_void_p))
    return out.reshape(n, 2)


def precond_taps(L: int, dtau: float = 0.1, t: float = 1.0, W: int = 6):
    """(c_0..c_W, p_0..p_W) of reading C10, from the oracle's own B at pi-flux."""
    c = np.zeros(W + 1)
    p = np.zeros(W + 1)
    lib().orc_precond_taps(C.c_int(L), C.c_double(dtau * t), C.c_int(W), c.ctypes.data_as(C.c_void_p),
                           p.ctypes.data_as(C.c_void_p))
    return c, p


class Oracle:
    """One lattice + couplings.  theta is passed per call (arrays [Ntau][2][L][L], float64)."""

    def __init__(self, L: int, Ntau: int, dtau: float = 0.1, t: float = 1.0, c_tau: float = 1.0, K: float = 1.0,
                 compact: bool = True, W: int = 6, taps=None):
        assert L % 2 == 0 and L >= 4 and Ntau >= 2
        self.L, self.Ntau, self.Vs, self.N = L, Ntau, L * L, L * L * Ntau
        self.dtau, self.t = dtau, t
        self.P = _Params()
        self.P.L, self.P.Ntau, self.P.dtau, self.P.t = L, Ntau, dtau, t
        self.P.c_tau, self.P.K, self.P.compact, self.P.W = c_tau, K, int(compact), W
        if W > 0:
            if taps is None:
                taps = precond_taps(L, dtau, t, W)[1]
            assert len(taps) == W + 1 and W <= 32
            for i, v in enumerate(taps):
                self.P.taps[i] = float(v)
        self.taps = np.array([self.P.taps[i] for i in range(W + 1)]) if W > 0 else np.zeros(0)
        self._p = C.byref(self.P)

    # ---- single-slice pieces (for pins) -------------------------------------------------------
    def sweep(self, theta_slice, fam: int, a: float, v):
        th, thp = _d(theta_slice)
        out = np.array(v, dtype=np.complex128).reshape(-1).copy()
        lib().orc_sweep(C.c_int(self.L), thp, C.c_int(fam), C.c_double(a), out.ctypes.data_as(C.c_void_p))
        return out.reshape(np.shape(v))

    def apply_B(self, theta_slice, v):
        th, thp = _d(theta_slice)
        vin, vp = _c(np.reshape(v, -1))
        out = np.empty_like(vin)
        lib().orc_apply_B(C.c_int(self.L), thp, C.c_double(self.dtau * self.t), vp, out.ctypes.data_as(C.c_void_p))
        return out.reshape(np.shape(v))

    # ---- full-lattice operators ---------------------------------------------------------------
    def _op(self, fn, theta, v, extra=()):
        th, thp = _d(theta)
        vin, vp = _c(np.reshape(v, -1))
        assert vin.size == self.N and th.size == 2 * self.N
        out = np.empty_like(vin)
        fn(self._p, thp, vp, out.ctypes.data_as(C.c_void_p), *extra)
        return out.reshape(np.shape(v))

    def apply_M(self, theta, v):
        return self._op(lib().orc_apply_M, theta, v)

    def apply_Mdag(self, theta, v):
        return self._op(lib().orc_apply_Mdag, theta, v)

    def apply_MdagM(self, theta, v):
        tmp = np.empty(self.N, dtype=np.complex128)
        return self._op(lib().orc_apply_MdagM, theta, v, (tmp.ctypes.data_as(C.c_void_p),))

    def precond(self, v):
        vin, vp = _c(np.reshape(v, -1))
        out = np.empty_like(vin)
        lib().orc_precond(self._p, vp, out.ctypes.data_as(C.c_void_p))
        return out.reshape(np.shape(v))

    def pcg(self, theta, rhs, tol: float = 1e-10, max_iter: int = 100000):
        """-> (x, iterations, recurrence relative residual)."""
        th, thp = _d(theta)
        b, bp = _c(np.reshape(rhs, -1))
        x = np.zeros_like(b)
        rel = C.c_double(0.0)
        it = lib().orc_pcg(self._p, thp, bp, x.ctypes.data_as(C.c_void_p), C.c_double(tol), C.c_long(max_iter),
                           C.byref(rel))
        return x.reshape(np.shape(rhs)), int(it), float(rel.value)

    def force_fermion(self, theta, X):
        th, thp = _d(theta)
        x, xp = _c(np.reshape(X, -1))
        g = np.empty(2 * self.N)
        lib().orc_force_fermion(self._p, thp, xp, g.ctypes.data_as(C.c_void_p))
        return g.reshape(self.Ntau, 2, self.L, self.L)

    def force_boson(self, theta):
        th, thp = _d(theta)
        g = np.empty(2 * self.N)
        lib().orc_force_boson(self._p, thp, g.ctypes.data_as(C.c_void_p))
        return g.reshape(self.Ntau, 2, self.L, self.L)

    def action_boson(self, theta) -> float:
        th, thp = _d(theta)
        return float(lib().orc_action_boson(self._p, thp))

    def sum_p2(self, p) -> float:
        pp, ppp = _d(p)
        return float(lib().orc_sum_p2(self._p, ppp))

    def trajectory(self, theta, p, phi, nsteps: int, eps: float, cg_tol: float = 1e-13, cg_max_iter: int = 1000000):
        """-> dict(theta, p, H0, H1, cg_iters, parts).  Inputs are not modified."""
        th = np.array(theta, dtype=np.float64, order="C").copy()
        pp = np.array(p, dtype=np.float64, order="C").copy()
        f, fp = _c(np.reshape(phi, -1))
        H0, H1 = C.c_double(0), C.c_double(0)
        parts = np.zeros(6)
        it = lib().orc_trajectory(self._p, th.ctypes.data_as(C.c_void_p), pp.ctypes.data_as(C.c_void_p), fp,
                                  C.c_int(nsteps), C.c_double(eps), C.c_double(cg_tol), C.c_long(cg_max_iter),
                                  C.byref(H0), C.byref(H1), parts.ctypes.data_as(C.c_void_p))
        return dict(theta=th, p=pp, H0=H0.value, H1=H1.value, cg_iters=int(it), parts=parts)

    def hqmc_step(self, theta, p, eta, u: float, nsteps: int, eps: float, cg_tol: float = 1e-13, cg_max_iter: int = 1000000):
        """One HQMC update -> dict(theta, p, H0, H1, accepted, cg_iters).  Inputs are not modified."""
        th = np.array(theta, dtype=np.float64, order="C").copy()
        pp = np.array(p, dtype=np.float64, order="C").copy()
        e, ep = _c(np.reshape(eta, -1))
        H0, H1, it = C.c_double(0), C.c_double(0), C.c_long(0)
        acc = lib().orc_hqmc_step(self._p, th.ctypes.data_as(C.c_void_p), pp.ctypes.data_as(C.c_void_p), ep, C.c_double(u),
                                  C.c_int(nsteps), C.c_double(eps), C.c_double(cg_tol), C.c_long(cg_max_iter), C.byref(H0),
                                  C.byref(H1), C.byref(it))
        return dict(theta=th, p=pp, H0=H0.value, H1=H1.value, accepted=bool(acc), cg_iters=int(it.value))

    def hqmc_sweep(self, theta, seed: int, first: int, n_updates: int, nsteps: int, eps: float, cg_tol: float = 1e-13,
                   cg_max_iter: int = 1000000):
        """n_updates HQMC updates with the oracle's own counter-based draws -> dict(theta, H0, H1, accepted,
        cg_iters), one entry per update.  theta is not modified."""
        th = np.array(theta, dtype=np.float64, order="C").copy()
        H0, H1 = np.zeros(n_updates), np.zeros(n_updates)
        acc, it = np.zeros(n_updates, dtype=np.int32), np.zeros(n_updates, dtype=np.int64)
        lib().orc_hqmc_sweep(self._p, th.ctypes.data_as(C.c_void_p), C.c_uint64(seed), C.c_uint32(first), C.c_int(n_updates),
                             C.c_int(nsteps), C.c_double(eps), C.c_double(cg_tol), C.c_long(cg_max_iter),
                             H0.ctypes.data_as(C.c_void_p), H1.ctypes.data_as(C.c_void_p), acc.ctypes.data_as(C.c_void_p),
                             it.ctypes.data_as(C.c_void_p))
        return dict(theta=th, H0=H0, H1=H1, accepted=acc.astype(bool), cg_iters=it)
