"""Seeded synthetic conic programs  min c'x  s.t.  Ax=b, x in K  (eq.(1)).

This module is DATA ONLY: it draws random sparse matrices and builds (b, c) from a constructed
complementary primal/dual pair, so that the optimal value c'x0 = b'y0 is known by construction
(BASELINE.json configs 0-4; SURVEY.md section 8(d) recipes).  It contains none of the solver's
arithmetic (no projections, no splitting iteration, no conditioning rule) and is the one module the
CPU oracle's tests and the CUDA path's tests/bench both use.

The inputs stand in for the paper's dense random LP/SOCP workloads of section V-A / V-D
(PAPER.md:342-346, 368-371); no public benchmark or dataset is involved.

K is described as ``n_lin`` leading orthant coordinates (size-1 Lorentz cones, PAPER.md:52-56 with
n_i = 1) followed by ``soc_size[i]``-sized Lorentz cones.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np
import scipy.sparse as sp

BASE_SEED = 210300736  # seed = BASE_SEED + config index


@dataclass
class Problem:
    name: str
    m: int
    n: int
    row_ptr: np.ndarray  # int32 [m+1]
    col_idx: np.ndarray  # int32 [nnz], sorted and unique within a row
    val: np.ndarray  # float64 [nnz]
    b: np.ndarray  # float64 [m]
    c: np.ndarray  # float64 [n]
    n_lin: int
    soc_size: np.ndarray  # int32 [n_soc]
    x0: np.ndarray  # constructed primal optimum (NOT unique in general, SURVEY 8(c) v)
    y0: np.ndarray  # constructed dual multiplier
    s0: np.ndarray  # constructed dual slack z (unique)
    mu: float = 1.0
    t: float = 9.2  # PAPER.md:352 (LP); 1.7 for SOCP
    L_first: int = 300  # PAPER.md:348-350 (LP); 200 for SOCP
    L_every: int = 100
    meta: dict = field(default_factory=dict)

    @property
    def nnz(self) -> int:
        return int(self.row_ptr[-1])

    @property
    def n_soc(self) -> int:
        return int(self.soc_size.shape[0])

    def csr(self) -> sp.csr_matrix:
        return sp.csr_matrix((self.val, self.col_idx, self.row_ptr), shape=(self.m, self.n))

    def opt_value(self) -> float:
        return float(self.c @ self.x0)

    def schedule(self, k_iter: int) -> list[int]:
        """The paper's L = {L_first, L_first+L_every, ...} truncated to k_iter (eq.(17),(18))."""
        return list(range(self.L_first, k_iter + 1, self.L_every))


# --------------------------------------------------------------------------------------------
# sparse patterns
# --------------------------------------------------------------------------------------------

def _finish_csr(rows, cols, vals, m, n, rng, min_row_nnz=1):
    """COO -> canonical CSR (sorted, unique).  Every row is topped up to at least `min_row_nnz` entries
    with N(0,1) values in uniform random columns (BASELINE.json is silent on empty / very short rows;
    DESIGN.md "Input recipe": with fewer than ~3 entries per row the Zipf matrices are rank-deficient
    w.h.p. -- singleton rows sharing a column -- which breaks the paper's full-row-rank assumption)."""
    A = sp.csr_matrix((vals, (rows, cols)), shape=(m, n))
    A.sum_duplicates()
    for _ in range(50):
        counts = np.diff(A.indptr)
        short = np.flatnonzero(counts < min_row_nnz)
        if not short.size:
            break
        rr = np.repeat(short, min_row_nnz - counts[short])
        cc = rng.integers(0, n, size=rr.size)
        vv = rng.standard_normal(rr.size)
        A = (A + sp.csr_matrix((vv, (rr, cc)), shape=(m, n))).tocsr()
        A.sum_duplicates()
    A.sort_indices()
    A.eliminate_zeros()
    return A


def _distinct_rows_uniform(rng, m, n, k):
    """k distinct uniform rows for each of n columns -> int64 [n, k]."""
    if k > m:
        raise ValueError("more non-zeros per column than rows")
    r = rng.integers(0, m, size=(n, k))
    for _ in range(200):
        r.sort(axis=1)
        dup = np.zeros_like(r, dtype=bool)
        dup[:, 1:] = r[:, 1:] == r[:, :-1]
        nd = int(dup.sum())
        if nd == 0:
            return r
        r[dup] = rng.integers(0, m, size=nd)
    raise RuntimeError("could not de-duplicate rows")


def _distinct_rows_zipf(rng, m, n, k, s_exp):
    """k distinct rows per column drawn Zipf(s_exp) over a random permutation of the rows."""
    w = np.arange(1, m + 1, dtype=np.float64) ** (-s_exp)
    cdf = np.cumsum(w)
    cdf /= cdf[-1]
    draw = lambda size: np.minimum(np.searchsorted(cdf, rng.random(size)), m - 1)
    r = draw((n, k)).reshape(n, k)
    for _ in range(500):
        r.sort(axis=1)
        dup = np.zeros_like(r, dtype=bool)
        dup[:, 1:] = r[:, 1:] == r[:, :-1]
        nd = int(dup.sum())
        if nd == 0:
            break
        r[dup] = draw(nd)
    else:
        raise RuntimeError("could not de-duplicate rows")
    perm = rng.permutation(m)
    return perm[r]


def sparse_fixed_per_column(rng, m, n, k, zipf=None, min_row_nnz=1):
    rows = _distinct_rows_zipf(rng, m, n, k, zipf) if zipf else _distinct_rows_uniform(rng, m, n, k)
    cols = np.repeat(np.arange(n, dtype=np.int64), k)
    vals = rng.standard_normal(n * k)
    return _finish_csr(rows.reshape(-1), cols, vals, m, n, rng, min_row_nnz)


# --------------------------------------------------------------------------------------------
# complementary optimal pairs
# --------------------------------------------------------------------------------------------

def _lp_pair(rng, n, zero_frac):
    """x0 ~ U(0,1) with a random zero_frac of entries set to 0; s0 ~ U(0,1) on that zero set."""
    x0 = rng.random(n)
    zero = rng.random(n) < zero_frac
    # keep the drawn fraction exact-ish but never empty on either side
    if zero.all():
        zero[0] = False
    if not zero.any():
        zero[0] = True
    x0[zero] = 0.0
    s0 = np.where(zero, rng.random(n), 0.0)
    return x0, s0


def _soc_pair(rng, sizes):
    """Per Lorentz block one of: x0 interior & s0=0; x0=0 & s0 interior; both on the boundary with
    s0 = gamma*(x0_1, -x0_tail), gamma>0 (complementary: x0's0 = 0)."""
    n = int(sizes.sum())
    x0 = np.zeros(n)
    s0 = np.zeros(n)
    off = 0
    kinds = rng.integers(0, 3, size=sizes.shape[0])
    for sz, kind in zip(sizes.tolist(), kinds.tolist()):
        tail = rng.standard_normal(sz - 1)
        nt = float(np.linalg.norm(tail))
        if kind == 0:  # x0 strictly inside
            x0[off] = nt * (1.0 + rng.random()) + 0.1
            x0[off + 1:off + sz] = tail
        elif kind == 1:  # s0 strictly inside
            s0[off] = nt * (1.0 + rng.random()) + 0.1
            s0[off + 1:off + sz] = tail
        else:  # both on the boundary
            x0[off] = nt
            x0[off + 1:off + sz] = tail
            g = 0.25 + rng.random()
            s0[off] = g * nt
            s0[off + 1:off + sz] = -g * tail
        off += sz
    return x0, s0


def _assemble(name, A, x0, s0, rng, n_lin, soc_size, **kw):
    m, n = A.shape
    y0 = rng.standard_normal(m)
    b = A @ x0
    c = A.T @ y0 + s0
    return Problem(name=name, m=m, n=n,
                   row_ptr=A.indptr.astype(np.int32), col_idx=A.indices.astype(np.int32),
                   val=A.data.astype(np.float64), b=np.asarray(b, dtype=np.float64),
                   c=np.asarray(c, dtype=np.float64), n_lin=int(n_lin),
                   soc_size=np.asarray(soc_size, dtype=np.int32), x0=x0, y0=y0, s0=s0, **kw)


# --------------------------------------------------------------------------------------------
# generators (size-parametrised so the tests can use scaled-down replicas of each config)
# --------------------------------------------------------------------------------------------

def tiny_dense_lp(seed, m=50, n=100, density=0.2, zero_frac=0.4, name="cfg0_tiny_lp"):
    """BASELINE.json config 0: dense-stored CSR, each entry non-zero w.p. `density`, N(0,1);
    re-drawn until no empty row/column and full row rank."""
    rng = np.random.default_rng(seed)
    for _ in range(100):
        mask = rng.random((m, n)) < density
        M = np.where(mask, rng.standard_normal((m, n)), 0.0)
        if (mask.sum(0) > 0).all() and (mask.sum(1) > 0).all() and np.linalg.matrix_rank(M) == m:
            break
    else:
        raise RuntimeError("could not draw a full-rank pattern")
    A = sp.csr_matrix(M)
    A.sort_indices()
    x0, s0 = _lp_pair(rng, n, zero_frac)
    return _assemble(name, A, x0, s0, rng, n, np.zeros(0, np.int32), t=9.2, L_first=100, L_every=100)


def sparse_lp(seed, m, n, per_col, zero_frac=0.5, zipf=None, row_log10=None, col_log10=None,
              min_row_nnz=1, name="sparse_lp"):
    """BASELINE.json configs 1, 2, 4: fixed non-zeros per column at uniform (or Zipf) rows, N(0,1);
    optional row/column scaling 10^U(-a,a) (config 2); optimum built on the scaled matrix."""
    rng = np.random.default_rng(seed)
    A = sparse_fixed_per_column(rng, m, n, per_col, zipf=zipf, min_row_nnz=min_row_nnz)
    if row_log10 is not None:
        A = sp.diags(10.0 ** rng.uniform(-row_log10, row_log10, size=m)) @ A
    if col_log10 is not None:
        A = A @ sp.diags(10.0 ** rng.uniform(-col_log10, col_log10, size=n))
    A = sp.csr_matrix(A)
    A.sort_indices()
    x0, s0 = _lp_pair(rng, n, zero_frac)
    return _assemble(name, A, x0, s0, rng, n, np.zeros(0, np.int32), t=9.2, L_first=300, L_every=100)


def soc_sizes(rng, n_cones, n, lo=3, hi=40):
    """Block sizes ~U{lo..hi}; then the last blocks are adjusted so that the sum is exactly n
    (BASELINE.json config 3 fixes both 20,000 cones and n=400,000)."""
    if not (n_cones * lo <= n <= n_cones * hi):
        raise ValueError("n not reachable with these block sizes")
    sz = rng.integers(lo, hi + 1, size=n_cones).astype(np.int64)
    diff = int(n - sz.sum())
    i = n_cones - 1
    while diff != 0:
        if diff > 0:
            step = min(diff, hi - int(sz[i]))
        else:
            step = -min(-diff, int(sz[i]) - lo)
        sz[i] += step
        diff -= step
        i -= 1
        if i < 0:
            i = n_cones - 1
    return sz.astype(np.int32)


def sparse_socp(seed, m, n, n_cones, per_col, n_lin=0, lo=3, hi=40, name="sparse_socp"):
    """BASELINE.json config 3 (plus optional leading orthant coordinates for mixed-cone tests)."""
    rng = np.random.default_rng(seed)
    A = sparse_fixed_per_column(rng, m, n, per_col)
    sizes = soc_sizes(rng, n_cones, n - n_lin, lo, hi)
    xs, ss = _soc_pair(rng, sizes)
    if n_lin:
        xl, sl = _lp_pair(rng, n_lin, 0.5)
        x0, s0 = np.concatenate([xl, xs]), np.concatenate([sl, ss])
    else:
        x0, s0 = xs, ss
    return _assemble(name, A, x0, s0, rng, n_lin, sizes, t=1.7, L_first=200, L_every=100)


def gaussian_dense_lp(seed, m=80, n=100, name="sec4a_gaussian_lp"):
    """PAPER.md:315-320 (section IV-A): A ~ N(0,1) dense 80x100, b = A*xdot with xdot ~ U[0,1],
    c ~ N(0,1), K = R^100_+.  No constructed optimum (x0,y0,s0 are NaN)."""
    rng = np.random.default_rng(seed)
    M = rng.standard_normal((m, n))
    xdot = rng.random(n)
    A = sp.csr_matrix(M)
    A.sort_indices()
    nanv = lambda k: np.full(k, np.nan)
    return Problem(name=name, m=m, n=n, row_ptr=A.indptr.astype(np.int32),
                   col_idx=A.indices.astype(np.int32), val=A.data.copy(), b=M @ xdot,
                   c=rng.standard_normal(n), n_lin=n, soc_size=np.zeros(0, np.int32),
                   x0=nanv(n), y0=nanv(m), s0=nanv(n), t=9.2, L_first=300, L_every=100)


def dense_lp_sec5a(seed, n=100, name="sec5a_dense_lp"):
    """PAPER.md:342-346 (section V-A): m = floor(0.8 n), A ~ U[-1,1] dense, b = A |xdot| with xdot ~ N(0,1),
    c ~ N(0,1), K = R^n_+; schedule (17), t = 9.2, mu = 1.  No constructed optimum."""
    rng = np.random.default_rng(seed)
    m = int(0.8 * n)
    M = rng.uniform(-1.0, 1.0, size=(m, n))
    xdot = rng.standard_normal(n)
    A = sp.csr_matrix(M)
    A.sort_indices()
    nanv = lambda k: np.full(k, np.nan)
    return Problem(name=name, m=m, n=n, row_ptr=A.indptr.astype(np.int32),
                   col_idx=A.indices.astype(np.int32), val=A.data.copy(), b=M @ np.abs(xdot),
                   c=rng.standard_normal(n), n_lin=n, soc_size=np.zeros(0, np.int32),
                   x0=nanv(n), y0=nanv(m), s0=nanv(n), t=9.2, L_first=300, L_every=100)


def dense_socp_sec5d(seed, n=100, h=4, name="sec5d_dense_socp"):
    """PAPER.md:366-371 (section V-D) shape: m = floor(0.8 n), A ~ U[-1,1] dense, K = (K_h)^(n/h),
    c ~ U[0,1]; b = A * xfeas with xfeas in K.  The paper writes b = A*abs_K(xdot); here xfeas is
    built by the generator as (||tail|| + U(0,1), tail) per block, tail ~ U[0,1], so that this module
    holds no cone operator (feasibility is all the construction needs)."""
    if n % h:
        raise ValueError("n must be a multiple of h")
    rng = np.random.default_rng(seed)
    m = int(0.8 * n)
    M = rng.uniform(-1.0, 1.0, size=(m, n))
    xf = rng.random(n).reshape(n // h, h)
    xf[:, 0] = np.linalg.norm(xf[:, 1:], axis=1) + rng.random(n // h)
    xf = xf.reshape(-1)
    A = sp.csr_matrix(M)
    A.sort_indices()
    nanv = lambda k: np.full(k, np.nan)
    return Problem(name=name, m=m, n=n, row_ptr=A.indptr.astype(np.int32),
                   col_idx=A.indices.astype(np.int32), val=A.data.copy(), b=M @ xf,
                   c=rng.random(n), n_lin=0, soc_size=np.full(n // h, h, np.int32),
                   x0=nanv(n), y0=nanv(m), s0=nanv(n), t=1.7, L_first=200, L_every=100)


# --------------------------------------------------------------------------------------------
# the five BASELINE.json configs (scale < 1 gives a same-recipe replica for the parity tests)
# --------------------------------------------------------------------------------------------

CONFIG_SHAPES = {
    0: dict(m=50, n=100),
    1: dict(m=20_000, n=50_000, per_col=5),
    2: dict(m=100_000, n=250_000, per_col=8),
    3: dict(m=150_000, n=400_000, per_col=10, n_cones=20_000),
    4: dict(m=2_000_000, n=5_000_000, per_col=6),
}


def config(idx: int, scale: float = 1.0, seed: int | None = None) -> Problem:
    seed = BASE_SEED + idx if seed is None else seed
    sh = CONFIG_SHAPES[idx]
    sc = lambda v: max(8, int(round(v * scale)))
    if idx == 0:
        return tiny_dense_lp(seed)
    if idx == 1:
        return sparse_lp(seed, sc(sh["m"]), sc(sh["n"]), sh["per_col"], name=f"cfg1_sparse_lp_x{scale:g}")
    if idx == 2:
        return sparse_lp(seed, sc(sh["m"]), sc(sh["n"]), sh["per_col"], row_log10=3.0, col_log10=2.0,
                         name=f"cfg2_illcond_lp_x{scale:g}")
    if idx == 3:
        nc = sc(sh["n_cones"])
        n = int(round(nc * 20))  # 400,000 / 20,000
        return sparse_socp(seed, sc(sh["m"]), n, nc, sh["per_col"], name=f"cfg3_sparse_socp_x{scale:g}")
    if idx == 4:
        return sparse_lp(seed, sc(sh["m"]), sc(sh["n"]), sh["per_col"], zipf=1.1, min_row_nnz=4,
                         name=f"cfg4_zipf_lp_x{scale:g}")
    raise KeyError(idx)


# The 3x5 worked example printed in the paper: data only.
WORKED_A = np.array([[3.57, 3.45, 3.33, 64.24, -72.76],
                     [3.45, 3.33, 3.23, 95.14, -23.34],
                     [3.33, 3.23, 3.13, 93.53, -17.43]])
WORKED_B = np.array([-10.44, 20.65, 22.94])
WORKED_C = np.array([0.37, 1.93, -0.12, -0.38, 1.01])
WORKED_D_SK = np.array([0.0217, 0.0215, 0.0222])
WORKED_E_SK = np.full(5, 0.4722)
WORKED_E_AC = np.array([0.0792, 0.0884, 14.5484, 292.9524, 316.2179])


def worked_example() -> Problem:
    A = sp.csr_matrix(WORKED_A)
    A.sort_indices()
    nanv = lambda k: np.full(k, np.nan)
    return Problem(name="worked_example_3x5", m=3, n=5, row_ptr=A.indptr.astype(np.int32),
                   col_idx=A.indices.astype(np.int32), val=A.data.copy(), b=WORKED_B.copy(),
                   c=WORKED_C.copy(), n_lin=5, soc_size=np.zeros(0, np.int32),
                   x0=nanv(5), y0=nanv(3), s0=nanv(5), t=9.2)
