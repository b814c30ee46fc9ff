"""GPU parity over a sweep of seeded shapes chosen to hit every branch of the sliced layout and of the one-CTA /
multi-CTA split: all-orthant, all-Lorentz (block sizes 1..3 and large blocks), Zipf rows that become multi-chunk
segments, one entry per column, wide and nearly square matrices, one-CTA problems with and without the dense
factor-apply path.  Each case: 6 passes, a conditioning from the oracle's own iterate (protocol (ii-a)),
6 more passes; x, z, y, s to 1e-9, O to 1e-12."""
import numpy as np
import pytest

from paper_2103_00736_b200 import workloads as W

pytestmark = pytest.mark.gpu


def rel(a, b):
    nb = np.linalg.norm(b)
    return np.linalg.norm(a - b) / (nb if nb > 0 else 1.0)


SHAPES = {
    "lp_one_per_column": lambda: W.sparse_lp(11, 300, 2400, 1, min_row_nnz=2),
    "lp_nearly_square": lambda: W.sparse_lp(12, 900, 1000, 7),
    "lp_wide": lambda: W.sparse_lp(13, 40, 6000, 3),
    "lp_zipf_multichunk": lambda: W.sparse_lp(14, 1500, 9000, 6, zipf=1.1, min_row_nnz=4),
    "lp_zipf_steep": lambda: W.sparse_lp(15, 4000, 12000, 4, zipf=1.6, min_row_nnz=4),   # >= 4 per row: DESIGN.md 3 reading (x)
    # the same draw with 3,669 rows of 2-3 entries (full row rank, sigma_min 5e-3).  With min_row_nnz = 1 the draw is
    # rank-deficient (singleton rows sharing a column), outside reading (r); that is pinned on the CPU by
    # tests/test_oracle_algorithms.py::test_singleton_rows_make_the_zipf_draw_rank_deficient.
    "lp_zipf_steep_short_rows": lambda: W.sparse_lp(15, 4000, 12000, 4, zipf=1.6, min_row_nnz=2),
    # one dense column: every row's strongest column may be the same one; the FSAI build must stay bounded
    "lp_one_dense_column": lambda: _with_dense_column(W.sparse_lp(21, 3000, 9000, 5)),
    "socp_tiny_blocks": lambda: W.sparse_socp(16, 200, 900, 450, 4, lo=1, hi=3),
    "socp_large_blocks": lambda: W.sparse_socp(17, 300, 1500, 5, 5, lo=200, hi=400),
    "socp_plus_orthant": lambda: W.sparse_socp(18, 700, 2500, 60, 8, n_lin=1000, lo=2, hi=50),
    # Lorentz blocks of all three size classes of cone_sweep (sub-warp <= 64 < warp <= 4096 < CTA) plus orthant coordinates
    "socp_all_size_classes": lambda: _socp_with_sizes(23, 900, 150, [3, 40, 64, 65, 7, 300, 1000, 2, 4097, 33, 6000, 1, 12]),
    "one_cta_dense_path": lambda: W.sparse_socp(19, 60, 300, 20, 6, n_lin=100, lo=2, hi=20),
    "one_cta_cg_path": lambda: W.sparse_lp(20, 400, 1300, 5),
}


def _socp_with_sizes(seed, m, n_lin, sizes, per_col=6):
    """Mixed-cone problem with the given Lorentz block sizes (constructed complementary optimum, as workloads.sparse_socp)."""
    rng = np.random.default_rng(seed)
    sizes = np.asarray(sizes, np.int32)
    n = n_lin + int(sizes.sum())
    A = W.sparse_fixed_per_column(rng, m, n, per_col)
    xs, ss = W._soc_pair(rng, sizes)
    xl, sl = W._lp_pair(rng, n_lin, 0.5)
    return W._assemble("socp_sizes", A, np.concatenate([xl, xs]), np.concatenate([sl, ss]), rng, n_lin, sizes, t=1.7, L_first=200, L_every=100)


def _with_dense_column(p):
    """p with column 0 replaced by a dense column of large entries (b, c rebuilt from the constructed optimum)."""
    import scipy.sparse as sp
    rng = np.random.default_rng(99)
    A = p.csr().tolil()
    A[:, 0] = (5.0 + rng.random(p.m)).reshape(-1, 1)
    A = sp.csr_matrix(A)
    A.sort_indices()
    return W._assemble("lp_one_dense_column", A, p.x0, p.s0, rng, p.n, np.zeros(0, np.int32), t=9.2)


@pytest.mark.parametrize("name", list(SHAPES))
def test_shape_sweep_against_the_oracle(name):
    import oracle
    from paper_2103_00736_b200 import binding
    p = SHAPES[name]()
    mode = 1 if p.m <= 4000 else 0         # reading (s): the oracle's dense Cholesky + refinement where it is affordable
    O = oracle.Oracle.from_problem(p, solve_mode=mode)
    O.run(6)
    mid = O.get()
    O2 = oracle.Oracle.from_problem(p, solve_mode=mode)
    O2.set_point(mid["x"], mid["z"])
    O2.run(6, L=[1])                       # conditioning at l = 1 from (x, z) of the first leg: the rule on identical bits
    ref = O2.get()
    S = binding.Solver.from_problem(p, device="cuda:0")
    S.iterate(6)
    got = S.solution()
    for k in ("x", "z", "y", "s"):
        assert rel(got[k], mid[k]) <= 1e-9, (name, "leg 1", k, rel(got[k], mid[k]))
    S.destroy()
    S = binding.Solver.from_problem(p, device="cuda:0")
    S.set_point(mid["x"], mid["z"])
    S.run(6, L=[1])
    got = S.solution()
    assert rel(got["O"], ref["O"]) <= 1e-12, (name, "O", rel(got["O"], ref["O"]))
    for k in ("x", "z", "y", "s"):
        assert rel(got[k], ref[k]) <= 1e-9, (name, "leg 2", k, rel(got[k], ref[k]))
    r, q = S.residuals(), O2.residuals()
    for k in ("pres_abs", "dres_abs", "gap_abs", "kkt_rel"):
        assert abs(r[k] - q[k]) <= 1e-6 * abs(q[k]) + 1e-10 * (1 + np.linalg.norm(p.b)), (name, k, r[k], q[k])
    S.destroy()
