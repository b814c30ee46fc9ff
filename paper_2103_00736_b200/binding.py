"""ctypes binding of libcs.so (include/cs.h, diagnostics in include/cs_diag.h): same names, argument marshalling only.

Arrays may be numpy arrays (host memory) or torch tensors (host or CUDA memory); the binding passes
their raw pointers with the matching ``cs_mem`` tag.  There is NO fallback: if ``libcs.so`` is missing
or cannot be loaded, importing the symbols raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libcs.so")

CS_OK, CS_EINVAL, CS_ENOMEM, CS_ECUDA, CS_ESTATE, CS_ECGMAX = range(6)
CS_HOST, CS_DEVICE = 0, 1
STATUS_NAMES = {0: "CS_OK", 1: "CS_EINVAL", 2: "CS_ENOMEM", 3: "CS_ECUDA", 4: "CS_ESTATE", 5: "CS_ECGMAX"}


class cs_csr(C.Structure):
    _fields_ = [("m", C.c_int64), ("n", C.c_int64), ("nnz", C.c_int64), ("row_ptr", C.c_void_p),
                ("col_idx", C.c_void_p), ("val", C.c_void_p), ("where", C.c_int)]


class cs_cones(C.Structure):
    _fields_ = [("n_lin", C.c_int64), ("n_soc", C.c_int64), ("soc_size", C.c_void_p)]


class cs_params(C.Structure):
    _fields_ = [("mu", C.c_double), ("t", C.c_double), ("o_floor", C.c_double), ("cg_tol", C.c_double),
                ("cg_reduce", C.c_double), ("cg_max_iter", C.c_int32), ("precond", C.c_int32),
                ("dense_m_threshold", C.c_int32), ("reserved", C.c_int32)]


class cs_resid(C.Structure):
    _fields_ = [("iter", C.c_int64), ("cg_steps_total", C.c_int64), ("cg_steps_cond", C.c_int64), ("cg_steps_last", C.c_int32),
                ("n_conditionings", C.c_int32), ("cg_hit_max", C.c_int32), ("dense_refine2", C.c_int32)] + \
               [(k, C.c_double) for k in ("pres_abs", "pres_rel", "dres_abs", "dres_rel", "gap_abs", "gap_rel",
                                          "cone_viol_rel", "kkt_rel", "pobj", "dobj", "fp_res")]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_ if k != "reserved"}


class cs_schedule(C.Structure):
    _fields_ = [("max_iter", C.c_int64), ("check_every", C.c_int64), ("tol", C.c_double), ("rule", C.c_int32),
                ("reserved", C.c_int32), ("first", C.c_int64), ("every", C.c_int64), ("window", C.c_int64),
                ("lag", C.c_int64), ("ratio", C.c_double), ("f_floor", C.c_double)]


CS_RULE_SET, CS_RULE_STALL = 0, 1

_INT_STATUS = ("cs_create", "cs_set_params", "cs_get_params", "cs_set_point", "cs_set_dual", "cs_iterate", "cs_condition",
               "cs_set_scaling", "cs_equilibrate", "cs_solve", "cs_residuals", "cs_solution", "cs_diag_phase_times",
               "cs_diag_gather_probe", "cs_diag_barrier_probe", "cs_diag_l2_probe", "cs_diag_create", "cs_diag_layout_digest",
               "cs_cone_violation_static")
EXPORTS = _INT_STATUS + ("cs_kernel_launches", "cs_last_error", "cs_destroy")

_lib = None


def lib():
    """Load libcs.so (fails loudly when it has not been built: run ``__graft_entry__.build()``)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2103_00736_b200.build`; "
                               "there is no CPU fallback")
        L = C.CDLL(LIB_PATH)
        vp = C.c_void_p
        L.cs_create.argtypes = [C.POINTER(vp), C.POINTER(cs_csr), vp, vp, C.c_int, C.POINTER(cs_cones), vp]
        L.cs_set_params.argtypes = [vp, C.POINTER(cs_params)]
        L.cs_get_params.argtypes = [vp, C.POINTER(cs_params)]
        L.cs_set_point.argtypes = [vp, vp, vp, C.c_int]
        L.cs_set_dual.argtypes = [vp, vp, C.c_int]
        L.cs_iterate.argtypes = [vp, C.c_int64]
        L.cs_condition.argtypes = [vp]
        L.cs_set_scaling.argtypes = [vp, vp, C.c_int]
        L.cs_residuals.argtypes = [vp, C.POINTER(cs_resid)]
        L.cs_solution.argtypes = [vp, vp, vp, vp, vp, vp, C.c_int]
        L.cs_kernel_launches.argtypes = [vp]
        L.cs_kernel_launches.restype = C.c_int64
        L.cs_last_error.argtypes = [vp]
        L.cs_last_error.restype = C.c_char_p
        L.cs_destroy.argtypes = [vp]
        L.cs_destroy.restype = None
        L.cs_diag_phase_times.argtypes = [vp, C.POINTER(C.c_double)]
        L.cs_diag_barrier_probe.argtypes = [vp, C.c_int32, C.POINTER(C.c_double)]
        L.cs_diag_gather_probe.argtypes = [C.c_int64, C.c_int64, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.cs_equilibrate.argtypes = [vp, C.c_int32]
        L.cs_solve.argtypes = [vp, C.POINTER(cs_schedule), C.POINTER(cs_resid), C.POINTER(C.c_int64), C.c_int64,
                               C.POINTER(C.c_int64)]
        L.cs_diag_l2_probe.argtypes = [C.c_int64, C.c_int32, C.POINTER(C.c_double)]
        L.cs_diag_create.argtypes = [C.POINTER(vp), C.POINTER(cs_csr), vp, vp, C.c_int, C.POINTER(cs_cones), vp, C.c_int32]
        L.cs_diag_layout_digest.argtypes = [vp, C.POINTER(C.c_uint64)]
        L.cs_cone_violation_static.argtypes = [vp, vp, C.c_int64, C.POINTER(cs_cones), vp, C.c_int, vp]
        for name in _INT_STATUS:
            getattr(L, name).restype = C.c_int
        _lib = L
    return _lib


class CsError(RuntimeError):
    def __init__(self, status, text):
        super().__init__(f"{STATUS_NAMES.get(status, status)}: {text}")
        self.status = status


def _ptr(a, dtype=None):
    """(pointer, cs_mem) of a numpy array or torch tensor; None -> (None, host)."""
    if a is None:
        return None, CS_HOST
    if isinstance(a, np.ndarray):
        if dtype is not None and a.dtype != dtype:
            raise TypeError(f"expected {dtype}, got {a.dtype}")
        if not a.flags["C_CONTIGUOUS"]:
            raise ValueError("array must be contiguous")
        return a.ctypes.data, CS_HOST
    # torch tensor (duck-typed so that torch stays optional for host-only use)
    if not a.is_contiguous():
        raise ValueError("tensor must be contiguous")
    if dtype is not None and np.dtype(str(a.dtype).replace("torch.", "")) != dtype:
        raise TypeError(f"expected {dtype}, got {a.dtype}")
    return a.data_ptr(), (CS_DEVICE if a.is_cuda else CS_HOST)


def _same_space(*tags):
    tags = [t for p, t in tags if p is not None]
    if tags and any(t != tags[0] for t in tags):
        raise ValueError("all arrays of one call must live in the same memory space")
    return tags[0] if tags else CS_HOST


def gather_probe(n_vec, n_idx):
    """(us with gathers, us without) of n_idx random 8-byte gathers from an n_vec vector (cs_diag_gather_probe)."""
    a, b = C.c_double(), C.c_double()
    st = lib().cs_diag_gather_probe(int(n_vec), int(n_idx), C.byref(a), C.byref(b))
    if st != CS_OK:
        raise CsError(st, "cs_diag_gather_probe failed")
    return a.value, b.value


def l2_probe(nbytes=32 * 2**20, reps=50):
    """L2 -> SM read bandwidth in GB/s (cs_diag_l2_probe)."""
    g = C.c_double()
    st = lib().cs_diag_l2_probe(int(nbytes), int(reps), C.byref(g))
    if st != CS_OK:
        raise CsError(st, "cs_diag_l2_probe failed")
    return g.value


def cone_violation_static(x, z, n_lin, soc_size=None, out=None, stream=None):
    """cs_cone_violation_static: x, z = CUDA tensors [n]; returns the 5 doubles (numpy) or fills the CUDA tensor `out`."""
    xp, zp = _ptr(x, np.float64), _ptr(z, np.float64)
    if xp[1] != CS_DEVICE or zp[1] != CS_DEVICE:
        raise ValueError("x and z must live in device memory")
    soc = np.ascontiguousarray(soc_size if soc_size is not None else [], dtype=np.int32)
    K = cs_cones(int(n_lin), int(soc.shape[0]), soc.ctypes.data if soc.size else None)
    res = np.empty(5) if out is None else out
    op = _ptr(res, np.float64)
    st = lib().cs_cone_violation_static(xp[0], zp[0], int(x.shape[0]), C.byref(K), op[0], op[1],
                                        C.c_void_p(int(stream)) if stream else None)
    if st != CS_OK:
        raise CsError(st, lib().cs_last_error(None).decode())
    return res


class Solver:
    """One ``cs_solver`` handle.  Method names mirror the C ABI without the ``cs_`` prefix."""

    def __init__(self, m, n, row_ptr, col_idx, val, b, c, n_lin, soc_size=None, stream=None, build_mode=None):
        """build_mode (diagnostic, cs_diag_create): None = cs_create, 1 = layout built on the host, 2 = on the device."""
        L = lib()
        rp, ci, va = _ptr(row_ptr, np.int32), _ptr(col_idx, np.int32), _ptr(val, np.float64)
        where_A = _same_space(rp, ci, va)
        bp, cp = _ptr(b, np.float64), _ptr(c, np.float64)
        where_v = _same_space(bp, cp)
        nnz = int(val.shape[0])
        A = cs_csr(int(m), int(n), nnz, rp[0], ci[0], va[0], where_A)
        soc = np.ascontiguousarray(soc_size if soc_size is not None else [], dtype=np.int32)
        K = cs_cones(int(n_lin), int(soc.shape[0]), soc.ctypes.data if soc.size else None)
        h = C.c_void_p()
        sp = C.c_void_p(int(stream)) if stream else None
        if build_mode is None:
            st = L.cs_create(C.byref(h), C.byref(A), bp[0], cp[0], where_v, C.byref(K), sp)
        else:
            st = L.cs_diag_create(C.byref(h), C.byref(A), bp[0], cp[0], where_v, C.byref(K), sp, int(build_mode))
        if st != CS_OK:
            raise CsError(st, L.cs_last_error(None).decode())
        self._h, self.m, self.n = h, int(m), int(n)

    @classmethod
    def from_problem(cls, p, device=None, stream=None, build_mode=None):
        """Build from a ``workloads.Problem``; ``device`` = torch device to stage the inputs on first
        (inputs resident in HBM), None = pass the host arrays."""
        arrs = [p.row_ptr, p.col_idx, p.val, p.b, p.c]
        if device is not None:
            import torch
            arrs = [torch.from_numpy(np.ascontiguousarray(a)).to(device) for a in arrs]
        S = cls(p.m, p.n, arrs[0], arrs[1], arrs[2], arrs[3], arrs[4], p.n_lin, p.soc_size, stream=stream, build_mode=build_mode)
        S.set_params(mu=p.mu, t=p.t)
        return S

    def _check(self, st, ok=(CS_OK,)):
        if st not in ok:
            raise CsError(st, lib().cs_last_error(self._h).decode())
        return st

    def destroy(self):
        if getattr(self, "_h", None):
            try:
                lib().cs_destroy(self._h)
            except TypeError:       # interpreter shutdown: the module globals are gone, the process frees the device memory
                pass
            self._h = None

    __del__ = destroy

    def get_params(self):
        p = cs_params()
        self._check(lib().cs_get_params(self._h, C.byref(p)))
        return {k: getattr(p, k) for k, _ in p._fields_}

    def set_params(self, **kw):
        cur = self.get_params()
        unknown = set(kw) - set(cur)
        if unknown:
            raise TypeError(f"unknown parameter(s): {sorted(unknown)}")
        cur.update(kw)
        p = cs_params(cur["mu"], cur["t"], cur["o_floor"], cur["cg_tol"], cur["cg_reduce"], int(cur["cg_max_iter"]),
                      int(cur["precond"]),
                      int(cur["dense_m_threshold"]), 0)
        self._check(lib().cs_set_params(self._h, C.byref(p)))

    def set_point(self, x, z):
        xp, zp = _ptr(x, np.float64), _ptr(z, np.float64)
        self._check(lib().cs_set_point(self._h, xp[0], zp[0], _same_space(xp, zp)))

    def set_dual(self, y):
        """cs_set_dual: warm start of the inner solve from a dual vector y[m] (cs_solution's y of an earlier run)."""
        yp = _ptr(y, np.float64)
        self._check(lib().cs_set_dual(self._h, yp[0], yp[1]))

    def iterate(self, k):
        self._check(lib().cs_iterate(self._h, int(k)))

    def condition(self):
        self._check(lib().cs_condition(self._h))

    def set_scaling(self, O):
        op = _ptr(O, np.float64)
        self._check(lib().cs_set_scaling(self._h, op[0], op[1]))

    def equilibrate(self, n_sweeps):
        """cs_equilibrate: fixed l2 Ruiz equilibration E installed as O."""
        self._check(lib().cs_equilibrate(self._h, int(n_sweeps)))

    def solve(self, max_iter, tol=0.0, check_every=0, first=0, every=0, stall=None, strict=False):
        """cs_solve: Algorithm 2 with L = {first, first+every, ...} or, with stall=(window, lag, ratio[, f_floor]), the stall
        rule.  Returns (residual dict, list of the iterations that conditioned)."""
        sch = cs_schedule(max_iter=int(max_iter), check_every=int(check_every), tol=float(tol),
                          rule=CS_RULE_STALL if stall else CS_RULE_SET, reserved=0, first=int(first),
                          every=int(every), window=int(stall[0]) if stall else 0, lag=int(stall[1]) if stall else 0,
                          ratio=float(stall[2]) if stall else 0.0,
                          f_floor=float(stall[3]) if stall and len(stall) > 3 else 0.0)
        cap = 4096
        conds = (C.c_int64 * cap)()
        nc = C.c_int64(0)
        r = cs_resid()
        self._check(lib().cs_solve(self._h, C.byref(sch), C.byref(r), conds, cap, C.byref(nc)),
                    ok=(CS_OK,) if strict else (CS_OK, CS_ECGMAX))
        return r.as_dict(), [int(conds[i]) for i in range(min(cap, nc.value))]

    def residuals(self, strict=False):
        r = cs_resid()
        self._check(lib().cs_residuals(self._h, C.byref(r)), ok=(CS_OK,) if strict else (CS_OK, CS_ECGMAX))
        return r.as_dict()

    def solution_into(self, x=None, z=None, y=None, s=None, O=None):
        ps = [_ptr(a, np.float64) for a in (x, z, y, s, O)]
        self._check(lib().cs_solution(self._h, *[p[0] for p in ps], _same_space(*ps)))

    def solution(self):
        """x, z, y, s, O as host numpy arrays."""
        out = {k: np.empty(self.n) for k in ("x", "z", "s", "O")}
        out["y"] = np.empty(self.m)
        self.solution_into(out["x"], out["z"], out["y"], out["s"], out["O"])
        return out

    def phase_times(self):
        """Device time per phase of k_iterate so far (ns): cone, rhs, K1, K2, update, reduce, precond."""
        a = (C.c_double * 8)()
        self._check(lib().cs_diag_phase_times(self._h, a))
        names = ("cone", "rhs", "K1", "K2", "update", "reduce", "precond", "r7")
        return dict(zip(names, [float(x) for x in a]))

    def barrier_probe(self, n=1000):
        us = C.c_double()
        self._check(lib().cs_diag_barrier_probe(self._h, int(n), C.byref(us)))
        return us.value

    def layout_digest(self):
        """cs_diag_layout_digest: 32 words identifying the handle's layout (diagnostic; copies the arrays to the host)."""
        a = (C.c_uint64 * 32)()
        self._check(lib().cs_diag_layout_digest(self._h, a))
        return [int(v) for v in a]

    def kernel_launches(self):
        return int(lib().cs_kernel_launches(self._h))

    def run(self, k, L=()):
        """Algorithm 2 with the schedule L: continues the iteration counter kept by the caller
        in ``self.l``.  cs_iterate / cs_condition calls only."""
        l = getattr(self, "l", 0)
        end = l + int(k)
        for cond_at in sorted(x for x in L if l < x <= end):
            if cond_at - 1 > l:
                self.iterate(cond_at - 1 - l)
                l = cond_at - 1
            if cond_at > 1:
                self.condition()
        if end > l:
            self.iterate(end - l)
        self.l = end
