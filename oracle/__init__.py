"""oracle/ -- TEST INFRASTRUCTURE: the plain CPU oracle of the e-ph collision integral.

`ephc_oracle.c` (oracle B, list based, plain C) and `brute.py` (oracle A, brute force, numpy).
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs import
this package; the product (paper_2511_03683_b200/) never does and shares no code with it.

This module is the ctypes binding of ephc_oracle.c plus the gcc build step.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ephc_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


def build_lib(force: bool = False) -> str:
    """gcc -O2 (no fast-math, no -march: keeps the selection predicate free of FMA contraction)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".{os.getpid()}.tmp"
        subprocess.check_call(["gcc", "-O2", "-fPIC", "-shared", "-fopenmp", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


_i32p = np.ctypeslib.ndpointer(dtype=np.int32, flags="C_CONTIGUOUS")
_f64p = np.ctypeslib.ndpointer(dtype=np.float64, flags="C_CONTIGUOUS")


def _load():
    global _lib
    if _lib is not None:
        return _lib
    lib = C.CDLL(build_lib())
    prob_args = [_i32p, C.c_int, C.c_int, C.c_int, _i32p, _f64p, C.c_double, C.c_double, _f64p,
                 C.c_double, C.c_double, C.c_double, C.c_int64, _i32p, _i32p, _f64p]
    lib.orc_build.restype = C.c_void_p
    lib.orc_build.argtypes = prob_args
    lib.orc_free.argtypes = [C.c_void_p]
    for name in ("orc_nch", "orc_ndiag", "orc_nw"):
        getattr(lib, name).restype = C.c_int64
        getattr(lib, name).argtypes = [C.c_void_p]
    lib.orc_export.argtypes = [C.c_void_p] + [_i32p] * 6 + [_f64p] * 2
    lib.orc_export_diag.argtypes = [C.c_void_p] + [_i32p] * 3 + [_f64p] * 2
    lib.orc_collision.argtypes = [C.c_void_p, _f64p, _f64p, _f64p]
    lib.orc_collision_omp.argtypes = [C.c_void_p, _f64p, _f64p, _f64p]
    lib.orc_threads.restype = C.c_int
    lib.orc_transport_setup.argtypes = [C.c_void_p, _f64p, _f64p, _f64p]
    lib.orc_transport_iter.argtypes = [C.c_void_p, _f64p, _f64p, _f64p, _f64p, _f64p, _f64p]
    lib.orc_rt_step.restype = C.c_int
    lib.orc_rt_step.argtypes = [C.c_void_p, _f64p, _f64p, C.c_double, C.c_int, _f64p]
    lib.orc_collision_sampled.argtypes = prob_args + [_f64p, _f64p, C.c_int, _i32p, _f64p]
    lib.orc_drift.restype = C.c_int
    lib.orc_drift.argtypes = [_i32p, C.c_int, C.c_int, _i32p, _f64p, _f64p, _f64p]
    lib.orc_rt_step_field.restype = C.c_int
    lib.orc_rt_step_field.argtypes = [C.c_void_p, _i32p, _f64p, _f64p, _f64p, C.c_double, C.c_int, _f64p]
    _lib = lib
    return lib


def _prob_args(p):
    grid = np.asarray(p.grid, dtype=np.int32)
    return (grid, p.nk, p.nb, p.nnu, np.ascontiguousarray(p.kfull, dtype=np.int32),
            np.ascontiguousarray(p.E, dtype=np.float64).reshape(-1), p.emin, p.emax,
            np.ascontiguousarray(p.hw, dtype=np.float64).reshape(-1), p.sigma, p.ncut, p.g2_cut,
            p.npair, np.ascontiguousarray(p.pair_ik, dtype=np.int32),
            np.ascontiguousarray(p.pair_ikq, dtype=np.int32),
            np.ascontiguousarray(p.g2, dtype=np.float64).reshape(-1))


def _f(x):
    return np.ascontiguousarray(x, dtype=np.float64).reshape(-1)


class OracleList:
    """Canonical unordered channel list of one problem + the three drivers built on it."""

    def __init__(self, prob):
        self._lib = _load()
        self.ns = prob.nk * prob.nb
        self._h = self._lib.orc_build(*_prob_args(prob))
        if not self._h:
            raise MemoryError("orc_build failed")
        self.nch = int(self._lib.orc_nch(self._h))
        self.ndiag = int(self._lib.orc_ndiag(self._h))

    def close(self):
        if getattr(self, "_h", None):
            self._lib.orc_free(self._h)
            self._h = None

    __del__ = close

    @property
    def nw(self):
        return int(self._lib.orc_nw(self._h))

    def export(self):
        n = max(self.nch, 1)
        ints = [np.zeros(n, np.int32) for _ in range(6)]
        w = [np.zeros(n, np.float64) for _ in range(2)]
        self._lib.orc_export(self._h, *ints, *w)
        keys = ("ik", "ikq", "iq", "n", "m", "nu", "w_abs", "w_em")
        return {k: a[: self.nch] for k, a in zip(keys, ints + w)}

    def export_diag(self):
        n = max(self.ndiag, 1)
        ints = [np.zeros(n, np.int32) for _ in range(3)]
        w = [np.zeros(n, np.float64) for _ in range(2)]
        self._lib.orc_export_diag(self._h, *ints, *w)
        keys = ("s", "iq", "nu", "w_abs", "w_em")
        return {k: a[: self.ndiag] for k, a in zip(keys, ints + w)}

    def collision(self, f, N, omp=False):
        I = np.zeros(self.ns)
        (self._lib.orc_collision_omp if omp else self._lib.orc_collision)(self._h, _f(f), _f(N), I)
        return I

    def transport_setup(self, f0, N):
        G = np.zeros(self.ns)
        self._lib.orc_transport_setup(self._h, _f(f0), _f(N), G)
        return G

    def transport_iter(self, f0, N, F, v, tau):
        out = np.zeros(3 * self.ns)
        self._lib.orc_transport_iter(self._h, _f(f0), _f(N), _f(F), _f(v), _f(tau), out)
        return out.reshape(3, self.ns)

    def rt_step(self, f, N, dt, nsteps):
        f = _f(f).copy()
        sumf = np.zeros(nsteps + 1)
        rc = self._lib.orc_rt_step(self._h, f, _f(N), float(dt), int(nsteps), sumf)
        if rc != 0:
            raise MemoryError("orc_rt_step failed")
        return f, sumf


def drift(prob, f, field):
    """Drift term of Eq. 1, D = -(1/hbar) F . grad_k f (reading R-25), for every state slot."""
    out = np.zeros(prob.nk * prob.nb)
    rc = _load().orc_drift(np.asarray(prob.grid, dtype=np.int32), prob.nk, prob.nb,
                           np.ascontiguousarray(prob.kfull, dtype=np.int32), _f(f), _f(field), out)
    if rc != 0:
        raise MemoryError("orc_drift failed")
    return out


def rt_step_field(L, prob, f, N, field, dt, nsteps):
    """RK4 on df/dt = D[f] + I[f] (Eq. 1 as printed)."""
    f = _f(f).copy()
    sumf = np.zeros(nsteps + 1)
    rc = _load().orc_rt_step_field(L._h, np.ascontiguousarray(prob.kfull, dtype=np.int32), f, _f(N), _f(field),
                                   float(dt), int(nsteps), sumf)
    if rc != 0:
        raise MemoryError("orc_rt_step_field failed")
    return f, sumf


def transport_moments(f0, v, F):
    """Post-processing of the transport solution (reading R-26): S[al][be] = sum_s f0_s (1 - f0_s) v[al][s] F[be][s]
    (-df0/dE = f0 (1 - f0) / k_B T for a Fermi-Dirac f0) and n = sum_s f0_s.  The conductivity is
    sigma = e^2 / (Omega N_k k_B T) * S and the mobility e S / (k_B T n); the constants are the caller's."""
    f0 = _f(f0)
    ns = f0.size
    v, F = _f(v).reshape(3, ns), _f(F).reshape(3, ns)
    S = np.zeros((3, 3))
    for a in range(3):
        for b in range(3):
            S[a, b] = np.sum(f0 * (1.0 - f0) * v[a] * F[b])
    return S, float(np.sum(f0))


def threads() -> int:
    return int(_load().orc_threads())


def collision_sampled(prob, f, N, states):
    """I[s] for the listed states, straight from the problem definition (no list)."""
    states = np.ascontiguousarray(states, dtype=np.int32)
    out = np.zeros(len(states))
    _load().orc_collision_sampled(*_prob_args(prob), _f(f), _f(N), len(states), states, out)
    return out
