"""CPU oracle -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

ctypes loader for ``cs_oracle.c`` (plain single-threaded fp64 C written from the paper).  Only
``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import this package.  It imports nothing from ``paper_2103_00736_b200`` (the seeded input
generators are handed in by the caller as plain arrays) and the CUDA path imports nothing from here.

This file holds no arithmetic of the method: it compiles the C file with gcc, marshals numpy arrays
and returns numpy arrays.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "cs_oracle.c")
_LIB = os.path.join(_HERE, "libcs_oracle.so")
_lib = None

RESID_FIELDS = ("pres_abs", "pres_rel", "dres_abs", "dres_rel", "gap_abs", "gap_rel",
                "cone_viol_rel", "kkt_rel", "pobj", "dobj", "fp_res")


def build(force: bool = False) -> str:
    """gcc -O2 (no fast-math, no OpenMP: sums stay sequential and IEEE)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        dp, ip, i64 = C.POINTER(C.c_double), C.POINTER(C.c_int32), C.c_int64
        lib.orc_create.restype = C.c_void_p
        lib.orc_create.argtypes = [i64, i64, ip, ip, dp, dp, dp, i64, i64, ip,
                                   C.c_double, C.c_double, C.c_double, C.c_int, C.c_double, i64]
        lib.orc_destroy.argtypes = [C.c_void_p]
        lib.orc_set_point.argtypes = [C.c_void_p, dp, dp]
        lib.orc_set_scaling.argtypes = [C.c_void_p, dp]
        lib.orc_set_scaling.restype = C.c_int
        lib.orc_run.argtypes = [C.c_void_p, i64, C.POINTER(i64), i64]
        lib.orc_run.restype = C.c_int
        lib.orc_run_fixed.argtypes = [C.c_void_p, i64]
        lib.orc_run_stall.argtypes = [C.c_void_p, i64, i64, i64, C.c_double, C.c_double, dp, C.POINTER(i64), i64]
        lib.orc_run_stall.restype = i64
        lib.orc_ruiz.argtypes = [C.c_void_p, i64, dp, dp]
        lib.orc_get.argtypes = [C.c_void_p] + [dp] * 7
        lib.orc_counters.argtypes = [C.c_void_p, C.POINTER(i64)]
        lib.orc_residuals.argtypes = [C.c_void_p, dp]
        lib.orc_pinv_apply.argtypes = [C.c_void_p, dp, dp]
        lib.orc_abs_range.argtypes = [C.c_void_p, dp, dp]
        lib.orc_mat_vec.argtypes = [C.c_void_p, dp, dp]
        lib.orc_mat_tvec.argtypes = [C.c_void_p, dp, dp]
        for f in (lib.orc_proj_cone, lib.orc_abs_cone):
            f.argtypes = [dp, dp, i64, i64, ip]
        _lib = lib
    return _lib


def _d(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _i(a):
    return a.ctypes.data_as(C.POINTER(C.c_int32))


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    a = np.ascontiguousarray(a, dtype=np.int32)
    return a if a.size else np.zeros(1, np.int32)


def proj_cone(v, n_lin, soc_size):
    v = _f64(v); out = np.empty_like(v); ss = _i32(soc_size)
    _load().orc_proj_cone(_d(v), _d(out), int(n_lin), int(len(soc_size)), _i(ss))
    return out


def abs_cone(v, n_lin, soc_size):
    v = _f64(v); out = np.empty_like(v); ss = _i32(soc_size)
    _load().orc_abs_cone(_d(v), _d(out), int(n_lin), int(len(soc_size)), _i(ss))
    return out


class Oracle:
    """Stateful Algorithm 2.  ``run(k, L)`` continues the iteration counter l."""

    def __init__(self, m, n, row_ptr, col_idx, val, b, c, n_lin, soc_size, mu=1.0, t=9.2,
                 o_floor=1e-16, solve_mode=0, pcg_tol=1e-14, pcg_max=20000):
        lib = _load()
        self.m, self.n = int(m), int(n)
        self._keep = (_i32(row_ptr), _i32(col_idx), _f64(val), _f64(b), _f64(c), _i32(soc_size))
        rp, ci, va, bb, cc, ss = self._keep
        self._h = lib.orc_create(self.m, self.n, _i(rp), _i(ci), _d(va), _d(bb), _d(cc), int(n_lin),
                                 int(len(soc_size)), _i(ss), float(mu), float(t), float(o_floor),
                                 int(solve_mode), float(pcg_tol), int(pcg_max))
        if not self._h:
            raise ValueError("orc_create rejected the problem")

    @classmethod
    def from_problem(cls, p, **kw):
        kw.setdefault("mu", p.mu)
        kw.setdefault("t", p.t)
        return cls(p.m, p.n, p.row_ptr, p.col_idx, p.val, p.b, p.c, p.n_lin, p.soc_size, **kw)

    def close(self):
        if getattr(self, "_h", None):
            _load().orc_destroy(self._h)
            self._h = None

    __del__ = close

    def set_point(self, x, z):
        x, z = _f64(x), _f64(z)
        _load().orc_set_point(self._h, _d(x), _d(z))

    def set_scaling(self, O):
        O = _f64(O)
        rc = _load().orc_set_scaling(self._h, _d(O))
        if rc:
            raise RuntimeError(f"oracle solve failed (code {rc})")

    def run(self, k, L=()):
        L = np.ascontiguousarray(sorted(L), dtype=np.int64)
        Lp = L.ctypes.data_as(C.POINTER(C.c_int64)) if L.size else None
        rc = _load().orc_run(self._h, int(k), Lp, int(L.size))
        if rc:
            raise RuntimeError(f"oracle solve failed (code {rc})")

    def run_fixed(self, k):
        _load().orc_run_fixed(self._h, int(k))

    def run_stall(self, k, window, lag, ratio, f_floor=0.0):
        """orc_run_stall: k more passes of Algorithm 2 with the stall criterion in place of a set L.
        Returns the list of iterations that conditioned during this call."""
        l0 = self.counters()["l"]
        f = getattr(self, "_f_hist", np.zeros(1))
        if f.size < l0 + int(k) + 1:
            f = np.concatenate([f, np.zeros(l0 + int(k) + 1 - f.size)])
        self._f_hist = f
        out = np.zeros(int(k) + 1, np.int64)
        nc = _load().orc_run_stall(self._h, int(k), int(window), int(lag), float(ratio), float(f_floor), _d(f),
                                   out.ctypes.data_as(C.POINTER(C.c_int64)), out.size)
        if nc < 0:
            raise RuntimeError("oracle stall-criterion run failed (bad arguments or solve error)")
        return [int(v) for v in out[:nc]]

    def ruiz(self, n_iter):
        """orc_ruiz: (D, E) of the l2 Ruiz equilibration of the pristine A after n_iter sweeps."""
        D, E = np.empty(self.m), np.empty(self.n)
        _load().orc_ruiz(self._h, int(n_iter), _d(D), _d(E))
        return D, E

    def get(self):
        n, m = self.n, self.m
        out = {k: np.empty(n) for k in ("x", "z", "s", "O", "p", "d")}
        out["y"] = np.empty(m)
        _load().orc_get(self._h, _d(out["x"]), _d(out["z"]), _d(out["y"]), _d(out["s"]), _d(out["O"]),
                        _d(out["p"]), _d(out["d"]))
        return out

    def counters(self):
        a = (C.c_int64 * 6)()
        _load().orc_counters(self._h, a)
        return dict(l=a[0], n_cond=a[1], pcg_steps_total=a[2], pcg_steps_last=a[3], solve_mode=a[4],
                    pcg_fail=a[5])

    def residuals(self):
        out = np.empty(11)
        _load().orc_residuals(self._h, _d(out))
        return dict(zip(RESID_FIELDS, out.tolist()))

    def pinv_apply(self, rhs):
        rhs = _f64(rhs); out = np.empty(self.n)
        _load().orc_pinv_apply(self._h, _d(rhs), _d(out))
        return out

    def abs_range(self, v):
        v = _f64(v); out = np.empty(self.n)
        _load().orc_abs_range(self._h, _d(v), _d(out))
        return out

    def mat_vec(self, v):
        v = _f64(v); out = np.empty(self.m)
        _load().orc_mat_vec(self._h, _d(v), _d(out))
        return out

    def mat_tvec(self, y):
        y = _f64(y); out = np.empty(self.n)
        _load().orc_mat_tvec(self._h, _d(y), _d(out))
        return out
