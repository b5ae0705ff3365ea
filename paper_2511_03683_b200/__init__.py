"""paper_2511_03683_b200 -- thin Python binding of the C ABI in include/ephc.h (libephc.so).

Argument marshalling only: every step of the hot path (collision integral of Eq. 2; transport
iteration; RK4 real-time stepping) runs in the CUDA kernels of csrc/.  PyTorch
is used by callers for device memory and streams; this module only reads `data_ptr()` of tensors (or takes
raw integer addresses) and passes them through.  There is no CPU fallback: if libephc.so is missing, or no
CUDA device is present, the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

from . import _build

__all__ = ["EphcError", "Handle", "build_channels", "lib_path", "HOST_ONLY", "SELECT_GPU", "TRANSPORT_COLLAPSE", "version",
           "noalloc_init", "noalloc_max_states", "sum_states_noalloc"]

HOST_ONLY = 1
SELECT_GPU = 2
TRANSPORT_COLLAPSE = 4
_HERE = os.path.dirname(os.path.abspath(__file__))
_lib = None


class EphcError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"ephc error {code}: {msg}")
        self.code = code


class _Problem(C.Structure):
    _fields_ = [("grid", C.c_int32 * 3), ("nk", C.c_int32), ("nb", C.c_int32), ("nnu", C.c_int32),
                ("flags", C.c_uint32), ("kfull", C.c_void_p), ("E", C.c_void_p), ("emin", C.c_double),
                ("emax", C.c_double), ("hw", C.c_void_p), ("sigma", C.c_double), ("ncut", C.c_double),
                ("g2_cut", C.c_double), ("npair", C.c_int64), ("pair_ik", C.c_void_p),
                ("pair_ikq", C.c_void_p), ("g2", C.c_void_p)]


class Counts(C.Structure):
    _fields_ = [(n, C.c_int64) for n in (
        "ns", "npair_active", "nch", "nw", "ndiag", "gather_entries", "gather_halfpairs", "scatter_entries",
        "scatter_pairs", "store_bytes_gather", "store_bytes_scatter", "store_bytes_transport",
        "alg_bytes_collision", "alg_bytes_transport")] + [
        ("n_workunits", C.c_int32), ("n_rounds", C.c_int32), ("n_tasks", C.c_int32), ("reserved", C.c_int32),
        ("store_bytes_paper", C.c_int64)]

    def asdict(self):
        return {n: int(getattr(self, n)) for n, _ in self._fields_ if n != "reserved"}


def lib_path() -> str:
    return _build.LIB


def _load():
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    if not os.path.exists(path):
        raise RuntimeError(f"{path} is not built: run `python -m paper_2511_03683_b200._build` "
                           "(or __graft_entry__.build()); there is no fallback path")
    lib = C.CDLL(path)
    vp, i64, dbl, i32 = C.c_void_p, C.c_int64, C.c_double, C.c_int
    sig = {
        "ephc_build_channels": (i32, [C.POINTER(_Problem), C.POINTER(vp)]),
        "ephc_build_channels_range": (i32, [C.POINTER(_Problem), i32, i32, C.POINTER(vp)]),
        "ephc_owned_states": (i32, [vp, C.POINTER(i64), C.POINTER(i64)]),
        "ephc_rt_stage": (i32, [vp, vp, vp, vp, dbl, i32, vp, vp]),
        "ephc_drift": (i32, [vp, vp, C.POINTER(dbl), vp, vp]),
        "ephc_rt_step_field": (i32, [vp, vp, vp, C.POINTER(dbl), dbl, i32, vp, vp]),
        "ephc_transport_moments": (i32, [vp, vp, vp, vp, vp, vp]),
        "ephc_query": (i32, [vp, C.POINTER(Counts)]),
        "ephc_export_channels": (i32, [vp] * 9),
        "ephc_export_diag": (i32, [vp] * 6),
        "ephc_export_gather": (i32, [vp] * 8),
        "ephc_export_tiles": (i32, [vp] * 8),
        "ephc_export_stream": (i32, [vp] * 7),
        "ephc_stream_entries": (i64, [vp]),
        "ephc_export_res": (i32, [vp] * 7),
        "ephc_export_rows": (i32, [vp] * 4),
        "ephc_export_rows_collapsed": (i32, [vp] * 4),
        "ephc_res_entries": (i64, [vp]),
        "ephc_set_variant": (i32, [vp, i32]),
        "ephc_get_variant": (i32, [vp]),
        "ephc_get_transport_variant": (i32, [vp]),
        "ephc_collision": (i32, [vp, vp, vp, vp, vp]),
        "ephc_transport_setup": (i32, [vp, vp, vp, vp, vp]),
        "ephc_transport_start": (i32, [vp, vp, vp, vp, vp, vp]),
        "ephc_transport_iter": (i32, [vp, vp, vp, vp, vp, vp]),
        "ephc_transport_iters": (i32, [vp, vp, vp, vp, vp, i32, vp]),
        "ephc_noalloc_init": (i32, []),
        "ephc_noalloc_max_states": (i64, []),
        "ephc_sum_states_noalloc": (i32, [vp, i64, vp, vp]),
        "ephc_transport_collapse": (i32, [vp, vp]),
        "ephc_set_transport_collapsed": (i32, [vp, i32]),
        "ephc_collapsed_entries": (i64, [vp]),
        "ephc_rt_step": (i32, [vp, vp, vp, dbl, i32, vp, vp]),
        "ephc_collision_host": (i32, [vp, vp, vp, vp]),
        "ephc_transport_solve_host": (i32, [vp, vp, vp, vp, i32, vp, vp]),
        "ephc_rt_step_host": (i32, [vp, vp, vp, dbl, i32, vp]),
        "ephc_launch_count": (i64, [vp]),
        "ephc_destroy": (i32, [vp]),
        "ephc_last_error": (C.c_char_p, []),
        "ephc_version": (C.c_char_p, []),
    }
    for name, (res, args) in sig.items():
        fn = getattr(lib, name)
        fn.restype = res
        fn.argtypes = args
    _lib = lib
    return lib


def version() -> str:
    return _load().ephc_version().decode()


def _check(rc: int):
    if rc != 0:
        raise EphcError(rc, _load().ephc_last_error().decode())


def _dev_ptr(x, nelem: Optional[int] = None, name: str = "tensor") -> int:
    """Device address of a CUDA float64 tensor (or a raw int address, passed through)."""
    if x is None:
        return 0
    if isinstance(x, int):
        return x
    if not (hasattr(x, "data_ptr") and x.is_cuda):
        raise TypeError(f"{name}: expected a CUDA tensor (device entry points take device buffers)")
    if str(x.dtype) != "torch.float64" or not x.is_contiguous():
        raise TypeError(f"{name}: expected a contiguous float64 tensor")
    if nelem is not None and x.numel() != nelem:
        raise ValueError(f"{name}: expected {nelem} elements, got {x.numel()}")
    return x.data_ptr()


def _host_ptr(x, nelem: Optional[int], name: str, writable: bool = False):
    """(address, keep-alive) of a host float64 buffer: numpy array or CPU (pinned) torch tensor."""
    if x is None:
        return 0, None
    if hasattr(x, "data_ptr"):
        if x.is_cuda or str(x.dtype) != "torch.float64" or not x.is_contiguous():
            raise TypeError(f"{name}: expected a contiguous CPU float64 tensor")
        if nelem is not None and x.numel() != nelem:
            raise ValueError(f"{name}: expected {nelem} elements")
        return x.data_ptr(), x
    a = x if writable else np.ascontiguousarray(x, dtype=np.float64)
    if a.dtype != np.float64 or not a.flags["C_CONTIGUOUS"] or (writable and not a.flags["WRITEABLE"]):
        raise TypeError(f"{name}: expected a C-contiguous float64 array")
    if nelem is not None and a.size != nelem:
        raise ValueError(f"{name}: expected {nelem} elements, got {a.size}")
    return a.ctypes.data, a


def _stream_ptr(stream) -> int:
    if stream is None:
        return 0
    if isinstance(stream, int):
        return stream
    return int(stream.cuda_stream)


class Handle:
    """Owner of one channel store (ephc_handle*)."""

    def __init__(self, ptr: int, nk: int, nb: int, nnu: int, nq: int):
        self._h = C.c_void_p(ptr)
        self.nk, self.nb, self.nnu, self.nq = nk, nb, nnu, nq
        self.ns = nk * nb

    def close(self):
        if getattr(self, "_h", None):
            _load().ephc_destroy(self._h)
            self._h = None

    __del__ = close

    def query(self) -> dict:
        c = Counts()
        _check(_load().ephc_query(self._h, C.byref(c)))
        return c.asdict()

    def export_channels(self) -> dict:
        nch = self.query()["nch"]
        n = max(nch, 1)
        ints = [np.zeros(n, np.int32) for _ in range(6)]
        w = [np.zeros(n, np.float64) for _ in range(2)]
        _check(_load().ephc_export_channels(self._h, *[a.ctypes.data for a in ints + w]))
        keys = ("ik", "ikq", "iq", "n", "m", "nu", "w_abs", "w_em")
        return {k: a[:nch] for k, a in zip(keys, ints + w)}

    def export_diag(self) -> dict:
        nd = self.query()["ndiag"]
        n = max(nd, 1)
        ints = [np.zeros(n, np.int32) for _ in range(3)]
        w = [np.zeros(n, np.float64) for _ in range(2)]
        _check(_load().ephc_export_diag(self._h, *[a.ctypes.data for a in ints + w]))
        keys = ("s", "iq", "nu", "w_abs", "w_em")
        return {k: a[:nd] for k, a in zip(keys, ints + w)}

    def export_gather(self) -> dict:
        ne = self.query()["gather_entries"]
        n = max(ne, 1)
        ints = [np.zeros(n, np.int32) for _ in range(6)]
        w = np.zeros(n, np.float64)
        _check(_load().ephc_export_gather(self._h, *[a.ctypes.data for a in ints], w.ctypes.data))
        keys = ("dest", "partner", "iq", "nu", "kind", "diag", "w")
        return {k: a[:ne] for k, a in zip(keys, ints + [w])}

    def export_tiles(self) -> dict:
        ne = self.query()["scatter_entries"]
        n = max(ne, 1)
        ints = [np.zeros(n, np.int32) for _ in range(6)]
        w = np.zeros(n, np.float64)
        _check(_load().ephc_export_tiles(self._h, *[a.ctypes.data for a in ints], w.ctypes.data))
        keys = ("a", "b", "iq", "nu", "kind", "diag", "w")
        return {k: a[:ne] for k, a in zip(keys, ints + [w])}

    def export_stream(self) -> dict:
        ne = int(_load().ephc_stream_entries(self._h))
        n = max(ne, 1)
        ints = [np.zeros(n, np.int32) for _ in range(5)]
        w = np.zeros(n, np.float64)
        _check(_load().ephc_export_stream(self._h, *[a.ctypes.data for a in ints], w.ctypes.data))
        keys = ("a", "b", "iq", "nu", "kind", "w")
        return {k: a[:ne] for k, a in zip(keys, ints + [w])}

    def export_res(self) -> dict:
        ne = int(_load().ephc_res_entries(self._h))
        n = max(ne, 1)
        ints = [np.zeros(n, np.int32) for _ in range(5)]
        w = np.zeros(n, np.float64)
        _check(_load().ephc_export_res(self._h, *[a.ctypes.data for a in ints], w.ctypes.data))
        keys = ("a", "b", "iq", "nu", "kind", "w")
        return {k: a[:ne] for k, a in zip(keys, ints + [w])}

    def export_rows(self) -> dict:
        ne = self.query()["gather_entries"]
        n = max(ne, 1)
        dest, partner, pos = np.zeros(n, np.int32), np.zeros(n, np.int32), np.zeros(n, np.int64)
        _check(_load().ephc_export_rows(self._h, dest.ctypes.data, partner.ctypes.data, pos.ctypes.data))
        return {"dest": dest[:ne], "partner": partner[:ne], "gather_pos": pos[:ne]}

    def export_rows_collapsed(self) -> dict:
        nc = self.collapsed_entries()
        n = max(nc, 1)
        dest, partner, count = (np.zeros(n, np.int32) for _ in range(3))
        _check(_load().ephc_export_rows_collapsed(self._h, dest.ctypes.data, partner.ctypes.data, count.ctypes.data))
        return {"dest": dest[:nc], "partner": partner[:nc], "count": count[:nc]}

    def set_variant(self, variant: int):
        _check(_load().ephc_set_variant(self._h, int(variant)))

    def get_variant(self) -> int:
        """Variant ephc_collision / ephc_rt_step will use (0 gather, 1 tiles, 2 stream, 3 resident tiles)."""
        v = int(_load().ephc_get_variant(self._h))
        _check(min(v, 0))
        return v

    def get_transport_variant(self) -> int:
        """Variant ephc_transport_setup / ephc_transport_iter will use."""
        v = int(_load().ephc_get_transport_variant(self._h))
        _check(min(v, 0))
        return v

    def launch_count(self) -> int:
        return int(_load().ephc_launch_count(self._h))

    # ---- device entry points -----------------------------------------------------------------------------
    def collision(self, f, N, I, stream=None):
        _check(_load().ephc_collision(self._h, _dev_ptr(f, self.ns, "f"), _dev_ptr(N, self.nq * self.nnu, "N"),
                                      _dev_ptr(I, self.ns, "I"), _stream_ptr(stream)))

    def transport_setup(self, f0, N, Gamma, stream=None):
        _check(_load().ephc_transport_setup(self._h, _dev_ptr(f0, self.ns, "f0"),
                                            _dev_ptr(N, self.nq * self.nnu, "N"),
                                            _dev_ptr(Gamma, self.ns, "Gamma"), _stream_ptr(stream)))

    def transport_start(self, Gamma, v, tau, F0, stream=None):
        _check(_load().ephc_transport_start(self._h, _dev_ptr(Gamma, self.ns, "Gamma"), _dev_ptr(v, 3 * self.ns, "v"),
                                            _dev_ptr(tau, self.ns, "tau"), _dev_ptr(F0, 3 * self.ns, "F0"),
                                            _stream_ptr(stream)))

    def transport_iter(self, F, v, tau, Fout, stream=None):
        _check(_load().ephc_transport_iter(self._h, _dev_ptr(F, 3 * self.ns, "F"), _dev_ptr(v, 3 * self.ns, "v"),
                                           _dev_ptr(tau, self.ns, "tau"), _dev_ptr(Fout, 3 * self.ns, "Fout"),
                                           _stream_ptr(stream)))

    def transport_iters(self, F, v, tau, Fout, niter: int, stream=None):
        _check(_load().ephc_transport_iters(self._h, _dev_ptr(F, 3 * self.ns, "F"), _dev_ptr(v, 3 * self.ns, "v"),
                                            _dev_ptr(tau, self.ns, "tau"), _dev_ptr(Fout, 3 * self.ns, "Fout"),
                                            int(niter), _stream_ptr(stream)))

    def transport_collapse(self, stream=None):
        _check(_load().ephc_transport_collapse(self._h, _stream_ptr(stream)))

    def set_transport_collapsed(self, on: bool):
        _check(_load().ephc_set_transport_collapsed(self._h, 1 if on else 0))

    def collapsed_entries(self) -> int:
        return int(_load().ephc_collapsed_entries(self._h))

    def owned_states(self):
        lo, hi = C.c_int64(), C.c_int64()
        _check(_load().ephc_owned_states(self._h, C.byref(lo), C.byref(hi)))
        return int(lo.value), int(hi.value)

    def rt_stage(self, f, y_in, N, dt_fs: float, stage: int, y_out=None, stream=None):
        _check(_load().ephc_rt_stage(self._h, _dev_ptr(f, self.ns, "f"), _dev_ptr(y_in, self.ns, "y_in"),
                                     _dev_ptr(N, self.nq * self.nnu, "N"), float(dt_fs), int(stage),
                                     _dev_ptr(y_out, self.ns, "y_out"), _stream_ptr(stream)))

    def drift(self, f, field, out, stream=None):
        fld = (C.c_double * 3)(*[float(x) for x in field])
        _check(_load().ephc_drift(self._h, _dev_ptr(f, self.ns, "f"), fld, _dev_ptr(out, self.ns, "out"), _stream_ptr(stream)))

    def rt_step_field(self, f, N, field, dt_fs: float, nsteps: int, sumf=None, stream=None):
        fld = (C.c_double * 3)(*[float(x) for x in field])
        _check(_load().ephc_rt_step_field(self._h, _dev_ptr(f, self.ns, "f"), _dev_ptr(N, self.nq * self.nnu, "N"), fld,
                                          float(dt_fs), int(nsteps), _dev_ptr(sumf, nsteps + 1, "sumf"), _stream_ptr(stream)))

    def transport_moments(self, f0, v, F, out10, stream=None):
        _check(_load().ephc_transport_moments(self._h, _dev_ptr(f0, self.ns, "f0"), _dev_ptr(v, 3 * self.ns, "v"),
                                              _dev_ptr(F, 3 * self.ns, "F"), _dev_ptr(out10, 10, "out10"), _stream_ptr(stream)))

    def rt_step(self, f, N, dt_fs: float, nsteps: int, sumf=None, stream=None):
        _check(_load().ephc_rt_step(self._h, _dev_ptr(f, self.ns, "f"), _dev_ptr(N, self.nq * self.nnu, "N"),
                                    float(dt_fs), int(nsteps), _dev_ptr(sumf, nsteps + 1, "sumf"),
                                    _stream_ptr(stream)))

    # ---- host-buffer entry points (end-to-end) -------------------------------------------------------------
    def collision_host(self, f, N, I):
        pf, k1 = _host_ptr(f, self.ns, "f")
        pN, k2 = _host_ptr(N, self.nq * self.nnu, "N")
        pI, k3 = _host_ptr(I, self.ns, "I", writable=True)
        _check(_load().ephc_collision_host(self._h, pf, pN, pI))

    def transport_solve_host(self, f0, N, v, niter: int, F, Gamma=None):
        pf, k1 = _host_ptr(f0, self.ns, "f0")
        pN, k2 = _host_ptr(N, self.nq * self.nnu, "N")
        pv, k3 = _host_ptr(v, 3 * self.ns, "v")
        pF, k4 = _host_ptr(F, 3 * self.ns, "F", writable=True)
        pG, k5 = _host_ptr(Gamma, self.ns, "Gamma", writable=True)
        _check(_load().ephc_transport_solve_host(self._h, pf, pN, pv, int(niter), pF, pG))

    def rt_step_host(self, f, N, dt_fs: float, nsteps: int, sumf=None):
        pf, k1 = _host_ptr(f, self.ns, "f", writable=True)
        pN, k2 = _host_ptr(N, self.nq * self.nnu, "N")
        ps, k3 = _host_ptr(sumf, nsteps + 1, "sumf", writable=True)
        _check(_load().ephc_rt_step_host(self._h, pf, pN, float(dt_fs), int(nsteps), ps))


def noalloc_init() -> None:
    """Looks up the device address of the library's fixed scratch array for the current device (once per device)."""
    _check(_load().ephc_noalloc_init())


def noalloc_max_states() -> int:
    return int(_load().ephc_noalloc_max_states())


def sum_states_noalloc(f, out, n: Optional[int] = None, stream=None) -> None:
    """out[0] = sum of the first n (default: all) elements of the device vector f; allocates nothing (include/ephc.h)."""
    if n is None:
        n = f.numel()
    _check(_load().ephc_sum_states_noalloc(_dev_ptr(f, None, "f"), int(n), _dev_ptr(out, None, "out"), _stream_ptr(stream)))


def build_channels(prob, flags: int = 0, k_range=None) -> Handle:
    """ephc_build_channels (or, with k_range = (k_lo, k_hi), ephc_build_channels_range) on an object with the fields of
    ephc_problem (e.g. ephc_inputs.Problem)."""
    lib = _load()
    keep = dict(
        kfull=np.ascontiguousarray(prob.kfull, dtype=np.int32),
        E=np.ascontiguousarray(prob.E, dtype=np.float64).reshape(-1),
        hw=np.ascontiguousarray(prob.hw, dtype=np.float64).reshape(-1),
        pair_ik=np.ascontiguousarray(prob.pair_ik, dtype=np.int32),
        pair_ikq=np.ascontiguousarray(prob.pair_ikq, dtype=np.int32),
        g2=np.ascontiguousarray(prob.g2, dtype=np.float64).reshape(-1),
    )
    nk, nb, nnu = int(prob.nk), int(prob.nb), int(prob.nnu)
    nq = int(prob.grid[0]) * int(prob.grid[1]) * int(prob.grid[2])
    npair = int(keep["pair_ik"].shape[0])
    if keep["kfull"].size != nk or keep["E"].size != nk * nb or keep["hw"].size != nq * nnu or \
            keep["pair_ikq"].size != npair or keep["g2"].size != npair * nnu * nb * nb:
        raise ValueError("array sizes do not match nk, nb, nnu, grid, npair")
    p = _Problem()
    p.grid = (C.c_int32 * 3)(*[int(g) for g in prob.grid])
    p.nk, p.nb, p.nnu, p.flags = nk, nb, nnu, int(flags)
    p.emin, p.emax = float(prob.emin), float(prob.emax)
    p.sigma, p.ncut, p.g2_cut = float(prob.sigma), float(prob.ncut), float(prob.g2_cut)
    p.npair = npair
    for k, a in keep.items():
        setattr(p, k, a.ctypes.data if a.size else None)
    out = C.c_void_p()
    if k_range is None:
        _check(lib.ephc_build_channels(C.byref(p), C.byref(out)))
    else:
        _check(lib.ephc_build_channels_range(C.byref(p), int(k_range[0]), int(k_range[1]), C.byref(out)))
    return Handle(out.value, nk, nb, nnu, nq)
