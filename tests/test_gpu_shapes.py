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
    # dense-stored inputs on many CTAs: the grid dense factor-apply path (csrc/cs_dense.cuh) with ragged sizes -- fewer rows
    # than one 64-row block; an odd m that is no multiple of any tile size (8-byte copies in the triangular inverse)
    "dense_grid_m40_wide": lambda: W.gaussian_dense_lp(24, m=40, n=400),
    "dense_grid_m203_ragged": lambda: W.gaussian_dense_lp(25, m=203, n=261),
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
    if name.startswith("dense_grid"):
        assert S.residuals()["cg_steps_total"] == 0            # the dense path ran, not CG
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


LAYOUT_CASES = dict(SHAPES)
LAYOUT_CASES.update({"cfg4_x0.02_fused_rows": lambda: W.config(4, 0.02), "cfg3_x0.1": lambda: W.config(3, 0.1), "cfg0": lambda: W.config(0),
                     "dense_sec5d_n400": lambda: W.dense_socp_sec5d(3, n=400, h=4)})


@pytest.mark.parametrize("name", list(LAYOUT_CASES))
def test_device_build_lays_the_matrix_out_exactly_as_the_host_build(name):
    """cs_create builds its layout on the device (csrc/cs_build.cuh: validation, two radix sorts, slice fill, fusion marks,
    fused rows' partition; automatic from 100,000 non-zeros on) or on the host.  Both, from host and from device inputs,
    must give the same bits in every layout array (slices, indices, pristine values, chunk tables, compressed views,
    fusion marks, permutations, b, c: cs_diag_layout_digest), and the same iterates bit for bit."""
    from paper_2103_00736_b200 import binding
    p = LAYOUT_CASES[name]()
    ref, sols = None, []
    for mode in (1, 2):
        for dev in (None, "cuda:0"):
            S = binding.Solver.from_problem(p, device=dev, build_mode=mode)
            d = S.layout_digest()
            ref = ref or d
            assert d == ref, (name, mode, dev, [i for i in range(32) if d[i] != ref[i]])
            if dev is None:
                S.run(5, L=[3])
                sols.append(S.solution())
            S.destroy()
    for k in sols[0]:
        assert np.array_equal(sols[0][k], sols[1][k]), (name, k)


def test_device_build_rejects_what_the_host_build_rejects():
    from paper_2103_00736_b200 import binding
    p = W.config(1, 0.05)
    bad_cols = p.col_idx.copy()
    bad_cols[[0, 1]] = bad_cols[[1, 0]]
    zero_row = p.val.copy()
    zero_row[p.row_ptr[7]:p.row_ptr[8]] = 0.0
    for kw in (dict(col_idx=bad_cols), dict(val=np.where(np.arange(p.nnz) == 3, np.nan, p.val)), dict(val=zero_row),
               dict(b=np.where(np.arange(p.m) == 2, np.inf, p.b))):
        for mode in (1, 2):
            a = dict(m=p.m, n=p.n, row_ptr=p.row_ptr, col_idx=p.col_idx, val=p.val, b=p.b, c=p.c, n_lin=p.n_lin, soc_size=p.soc_size)
            a.update(kw)
            with pytest.raises(binding.CsError) as ei:
                binding.Solver(build_mode=mode, **a)
            assert ei.value.status == binding.CS_EINVAL, (mode, list(kw))
