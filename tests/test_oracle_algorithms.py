"""Pins of the oracle's Algorithm 1 / Algorithm 2 against the paper's worked example, brute force,
HiGHS, hand-computed constants and equivariances (CPU only).  P:<line> = /root/reference/PAPER.md."""
import itertools
import os

import numpy as np
import pytest
import scipy.optimize as so
import scipy.sparse as sp

import oracle
from paper_2103_00736_b200 import workloads as W

HERE = os.path.dirname(os.path.abspath(__file__))


def _golden(name):
    out = {}
    with open(os.path.join(HERE, "golden", name)) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                k, v = line.split()
                out[k] = float(v)
    return out


def brute_force_lp(A, b, c):
    """min c'x s.t. Ax=b, x>=0 by enumerating all bases (tiny problems only)."""
    m, n = A.shape
    best = None
    for B in itertools.combinations(range(n), m):
        AB = A[:, B]
        if abs(np.linalg.det(AB)) < 1e-12:
            continue
        xB = np.linalg.solve(AB, b)
        if (xB < -1e-10).any():
            continue
        val = c[list(B)] @ xB
        if best is None or val < best[0] - 1e-12:
            x = np.zeros(n)
            x[list(B)] = xB
            y = np.linalg.solve(AB.T, c[list(B)])
            best = (val, x, y, c - A.T @ y)
    return best


def _problem_from_dense(A, b, c, n_lin, soc, **kw):
    S = sp.csr_matrix(A)
    S.sort_indices()
    nanv = lambda k: np.full(k, np.nan)
    return W.Problem(name="adhoc", m=A.shape[0], n=A.shape[1], row_ptr=S.indptr.astype(np.int32),
                     col_idx=S.indices.astype(np.int32), val=S.data.copy(), b=b, c=c, n_lin=n_lin,
                     soc_size=np.asarray(soc, np.int32), x0=nanv(A.shape[1]), y0=nanv(A.shape[0]),
                     s0=nanv(A.shape[1]), **kw)


# ------------------------------------------------------------------ worked example
def test_worked_example_condition_numbers_and_optimum():
    g = _golden("worked_example.txt")
    A = W.WORKED_A
    assert np.isclose(np.linalg.cond(A), g["cond_A"], rtol=1e-4)
    ASK = np.diag(W.WORKED_D_SK) @ A @ np.diag(W.WORKED_E_SK)      # A_hat = D A E, eq.(4)
    assert np.isclose(np.linalg.cond(ASK), g["cond_A_SK"], rtol=1e-3)  # D,E printed to 4 digits
    assert np.isclose(np.linalg.cond(A @ np.diag(W.WORKED_E_AC)), g["cond_A_AC"], rtol=1e-4)

    val, xs, ys, zs = brute_force_lp(A, W.WORKED_B, W.WORKED_C)
    res = so.linprog(W.WORKED_C, A_eq=A, b_eq=W.WORKED_B, bounds=(0, None), method="highs")
    assert np.isclose(res.fun, val, rtol=1e-8)

    p = W.worked_example()
    # Algorithm 1 (mu=1, s0=0): O = I throughout
    o = oracle.Oracle.from_problem(p)
    o.run(3000)
    gt = o.get()
    assert np.allclose(gt["x"], xs, atol=1e-8) and np.allclose(gt["z"], zs, atol=1e-8)
    assert np.allclose(gt["y"], ys, atol=1e-6)
    assert o.residuals()["kkt_rel"] < 1e-10
    # E^AC as a FIXED column scaling (eq.(4)-(5) with D=I, E=E^AC): same optimum, much faster (Fig.1(c))
    its = {}
    for name, E in (("none", np.ones(5)), ("ac", W.WORKED_E_AC)):
        o = oracle.Oracle.from_problem(p)
        o.set_point(np.zeros(5), np.zeros(5))     # s0 = 0 in either scaling
        o.set_scaling(E)
        k = 0
        while np.linalg.norm(o.get()["x"] - xs) > 1e-4 and k < 2000:
            o.run_fixed(1)
            k += 1
        its[name] = k
        assert k < 2000
    assert its["ac"] <= 5 and its["ac"] * 5 < its["none"]


# ------------------------------------------------------------------ tiny LPs vs brute force and HiGHS
@pytest.mark.parametrize("seed", [1, 2, 3])
def test_tiny_lp_matches_vertex_enumeration(seed):
    rng = np.random.default_rng(seed)
    m, n = 4, 9
    A = rng.standard_normal((m, n))
    x0, s0 = rng.random(n), np.zeros(n)
    zero = rng.permutation(n)[: n - m]         # non-degenerate vertex: exactly m positive entries
    x0[zero] = 0.0
    s0[zero] = rng.random(n - m) + 0.1
    b, c = A @ x0, A.T @ rng.standard_normal(m) + s0
    val, xs, ys, zs = brute_force_lp(A, b, c)
    p = _problem_from_dense(A, b, c, n, [])
    for L in ((), (50, 100, 150)):
        o = oracle.Oracle.from_problem(p)
        o.run(4000, L=L)
        g, r = o.get(), o.residuals()
        assert r["kkt_rel"] < 1e-9
        assert np.isclose(r["pobj"], val, atol=1e-8) and np.isclose(r["dobj"], val, atol=1e-8)
        assert np.allclose(g["x"], xs, atol=1e-7) and np.allclose(g["z"], zs, atol=1e-7)
        assert np.allclose(g["y"], ys, atol=1e-6)


def test_config0_reaches_constructed_optimum_and_highs_value():
    p = W.config(0)
    res = so.linprog(p.c, A_eq=p.csr().toarray(), b_eq=p.b, bounds=(0, None), method="highs")
    assert np.isclose(res.fun, p.opt_value(), rtol=1e-9)
    ends = {}
    for mode in (1, 2):
        o = oracle.Oracle.from_problem(p, solve_mode=mode)
        o.run(500, L=p.schedule(500))
        g, r = o.get(), o.residuals()
        assert r["kkt_rel"] < 1e-8
        assert np.isclose(r["pobj"], p.opt_value(), atol=1e-7)
        assert np.allclose(g["z"], p.s0, atol=1e-6) and np.allclose(g["y"], p.y0, atol=1e-6)  # unique
        ends[mode] = g
    assert np.linalg.norm(ends[1]["x"] - ends[2]["x"]) <= 1e-8 * np.linalg.norm(ends[1]["x"])  # Cholesky == PCG


# ------------------------------------------------------------------ conditioning rule, hand-computed
def test_conditioning_rule_hand_example():
    """K = R_+ x K_3.  x=(4 | 6,3,4), z=(0.5 | 2,.,.): o = (4/0.5, (6-5)/2) = (8, 0.5);
    spread = ln 16; t = ln 4 => alpha = 1/2 => O = (sqrt 8 | sqrt .5 x3)."""
    rng = np.random.default_rng(0)
    A = rng.standard_normal((2, 4))
    x = np.array([4.0, 6.0, 3.0, 4.0])
    z = np.array([0.5, 2.0, 0.3, -0.1])
    p = _problem_from_dense(A, A @ x, rng.standard_normal(4), 1, [3], t=np.log(4.0))
    o = oracle.Oracle.from_problem(p)
    o.set_point(x, z)
    o.run(1)
    O = o.get()["O"]
    assert np.allclose(O, [np.sqrt(8.0)] + [np.sqrt(0.5)] * 3, rtol=1e-14)
    # cap not active (t large): O = o exactly
    p2 = _problem_from_dense(A, A @ x, p.c, 1, [3], t=50.0)
    o2 = oracle.Oracle.from_problem(p2)
    o2.set_point(x, z)
    o2.run(1)
    assert np.allclose(o2.get()["O"], [8.0, 0.5, 0.5, 0.5], rtol=1e-14)
    # default start e_K gives O = I (reading (j),(h))
    o3 = oracle.Oracle.from_problem(p)
    o3.run(1)
    assert np.array_equal(o3.get()["O"], np.ones(4))


def test_step14_recast_keeps_xz_and_cap_holds():
    """Step 14 s = O^-1 x - mu O z continues 'current progress': right after a
    conditioning, abs_K(s) and s give back the same proj_K parts; and ln(max O/min O) <= t."""
    p = W.gaussian_dense_lp(3)
    o = oracle.Oracle.from_problem(p)
    o.run(40, L=[40])
    g = o.get()
    assert np.log(g["O"].max() / g["O"].min()) <= p.t * (1 + 1e-12)
    assert g["O"].min() > 0


# ------------------------------------------------------------------ row-scaling invariance (derived)
def test_row_scaling_is_inert():
    p = W.sparse_lp(21, 25, 60, 4)
    D = 10.0 ** np.random.default_rng(1).uniform(-2, 2, p.m)
    A = p.csr().toarray()
    p2 = _problem_from_dense(D[:, None] * A, D * p.b, p.c, p.n, [])
    runs = []
    for q in (p, p2):
        o = oracle.Oracle.from_problem(q)
        o.run(60, L=[30])
        runs.append(o.get())
    for k in ("s", "x", "z", "O"):
        assert np.linalg.norm(runs[0][k] - runs[1][k]) <= 1e-9 * np.linalg.norm(runs[0][k])


# ------------------------------------------------------------------ size-2 cones = rotated orthant
def test_size2_soc_equals_rotated_lp():
    """K_2 = {x1 >= |x2|} = Q R^2_+ with Q = [[1,1],[1,-1]]/sqrt2; Algorithm 1 is equivariant under the
    orthogonal change x -> Qx, A -> AQ', c -> Qc, so Q s_soc^l = s_lp^l for all l (L = {})."""
    rng = np.random.default_rng(5)
    m, n = 5, 12
    A = rng.standard_normal((m, n))
    Q = np.kron(np.eye(n // 2), np.array([[1.0, 1.0], [1.0, -1.0]]) / np.sqrt(2.0))
    xl = rng.random(n)                          # LP-feasible point => SOC-feasible Q'xl
    c_lp = (A @ Q.T).T @ rng.standard_normal(m) + rng.random(n)   # dual feasible => bounded LP
    c = Q.T @ c_lp
    # SOC problem (A, b, c, K_2^6) ; LP problem (A Q', b, Q c, R^12_+) with x_lp = Q x_soc
    ps = _problem_from_dense(A, A @ (Q.T @ xl), c, 0, [2] * 6)
    pl = _problem_from_dense(A @ Q.T, A @ (Q.T @ xl), Q @ c, n, [])
    os_, ol = oracle.Oracle.from_problem(ps), oracle.Oracle.from_problem(pl)
    # same start in both coordinate systems: s = 0  (x=z=e_K maps differently, so set points explicitly)
    x_soc = np.tile([1.0, 0.0], 6)
    os_.set_point(x_soc, x_soc)
    ol.set_point(Q @ x_soc, Q @ x_soc)
    os_.set_scaling(np.ones(n))
    ol.set_scaling(np.ones(n))
    for l in range(200):
        os_.run_fixed(1)
        ol.run_fixed(1)
        if l % 20 == 0 or l == 199:
            a, bq = Q @ os_.get()["s"], ol.get()["s"]
            assert np.linalg.norm(a - bq) <= 1e-10 * (1 + np.linalg.norm(bq))
    val = brute_force_lp(pl.csr().toarray(), pl.b, pl.c)[0]
    os_.run_fixed(5000)
    assert np.isclose(os_.residuals()["pobj"], val, atol=1e-7)


# ------------------------------------------------------------------ qualitative claims
def test_section4a_one_conditioning_helps():
    """L={} stalls, L={300} 'significant improvement', L={1..50} fast (Fig.2)."""
    worse = 0
    for seed in range(3):
        p = W.gaussian_dense_lp(100 + seed)
        res = {}
        for name, L, k in (("none", (), 1500), ("one", (300,), 1500), ("cont", tuple(range(1, 51)), 300)):
            o = oracle.Oracle.from_problem(p)
            ones = np.ones(p.n)
            o.set_point(ones, ones)
            o.run(k, L=L)
            res[name] = o.residuals()["pres_abs"]
        assert res["one"] < 1e-2 * res["none"]
        assert res["cont"] < 1e-2 * res["none"]


@pytest.mark.parametrize("h", [4, 10])
def test_section5d_socp_converges_with_and_without_conditioning(h):
    """P:364-377 shape (n=100): both schedules reach the same optimal value, KKT -> 0."""
    p = W.dense_socp_sec5d(7, n=100, h=h)
    vals = []
    for L in ((), tuple(range(200, 3001, 100))):
        o = oracle.Oracle.from_problem(p)
        o.run(3000, L=L)
        r = o.residuals()
        assert r["kkt_rel"] < 1e-7
        vals.append(r["pobj"])
    assert np.isclose(vals[0], vals[1], rtol=1e-6, atol=1e-7)


def test_constructed_socp_reaches_known_value():
    p = W.sparse_socp(9, 60, 160, 16, 5, n_lin=0, lo=3, hi=20)
    o = oracle.Oracle.from_problem(p)
    o.run(3000, L=p.schedule(3000))
    r = o.residuals()
    assert r["kkt_rel"] < 1e-7
    assert np.isclose(r["pobj"], p.opt_value(), rtol=1e-6, atol=1e-6)
    assert np.isclose(r["dobj"], p.opt_value(), rtol=1e-6, atol=1e-6)


# ------------------------------------------------------------------ criterion-driven conditioning
def _start_ones(p):
    o = oracle.Oracle.from_problem(p)
    ones = np.ones(p.n)
    o.set_point(ones, ones)
    return o


def test_stall_criterion_limits_reduce_to_a_set_L():
    """ratio = 0: every residual is a stall => conditions at every multiple of the window, i.e. the set
    L = {W+1, 2W+1, ...}; ratio = huge: never => L = {} (both bit for bit)."""
    p = W.gaussian_dense_lp(100)
    a = _start_ones(p)
    conds = a.run_stall(330, 50, 20, 0.0)
    assert conds == [1, 51, 101, 151, 201, 251, 301]
    b = _start_ones(p)
    b.run(330, L=(51, 101, 151, 201, 251, 301))
    assert np.array_equal(a.get()["x"], b.get()["x"]) and np.array_equal(a.get()["O"], b.get()["O"])
    a = _start_ones(p)
    assert a.run_stall(330, 50, 20, 1e300) == [1]
    b = _start_ones(p)
    b.run(330, L=())
    assert np.array_equal(a.get()["s"], b.get()["s"])


def test_stall_criterion_replayed_pass_by_pass():
    """The decisions of orc_run_stall re-taken outside it: one pass at a time through orc_run, the
    fixed-point residual read back through orc_residuals, the rule applied here (reading (y))."""
    p = W.gaussian_dense_lp(100)
    window, lag, ratio, floor = 20, 8, 0.7, 1e-8
    a = _start_ones(p)
    conds = a.run_stall(200, window, lag, ratio, floor) + a.run_stall(221, window, lag, ratio, floor)   # resumable
    b = _start_ones(p)
    f, mine = {}, []
    for l in range(1, 422):
        cond = l == 1 or ((l - 1) % window == 0 and f[l - 1] > ratio * f[l - 1 - lag] and f[l - 1] > floor)
        if cond:
            mine.append(l)
        b.run(1, L=(l,) if cond else ())
        f[l] = b.residuals()["fp_res"]
    assert mine == conds and 5 <= len(conds) < 12
    assert np.array_equal(a.get()["x"], b.get()["x"])
    # no decision was a near tie (so a device run in a different rounding order takes the same ones), and the
    # floor is what ends the conditionings once the run has converged
    for l in range(window + 1, 422, window):
        assert abs(f[l - 1] / floor - 1.0) > 1e-3
        if f[l - 1] > floor:
            assert abs(f[l - 1] / (ratio * f[l - 1 - lag]) - 1.0) > 1e-3
    assert f[420] < floor and max(conds) < 300
    c = _start_ones(p)
    assert len(c.run_stall(421, window, lag, ratio, 0.0)) > len(conds)     # without it: decisions on noise


def test_stall_criterion_beats_no_conditioning():
    """conditioning when the residual stalls does what L = {300} does in Fig. 2."""
    for seed in range(3):
        p = W.gaussian_dense_lp(100 + seed)
        a = _start_ones(p)
        a.run(1500, L=())
        b = _start_ones(p)
        conds = b.run_stall(1500, 50, 25, 0.5)
        assert len(conds) > 2
        assert b.residuals()["pres_abs"] < 1e-2 * a.residuals()["pres_abs"]


# ------------------------------------------------------------------ fixed equilibration
def test_ruiz_diagonal_matrix_closed_form():
    """A = diag(a): B = DAE is diagonal, one sweep gives D_i = E_i = |a_i|^{-1/2} and B_ii = sign(a_i)."""
    a = np.array([4.0, -9.0, 0.25, 100.0])
    n = a.size
    o = oracle.Oracle(n, n, np.arange(n + 1), np.arange(n), a, np.ones(n), np.ones(n), n, [])
    for sweeps in (1, 2, 7):
        D, E = o.ruiz(sweeps)
        assert np.allclose(D, np.abs(a) ** -0.5, rtol=1e-14) and np.allclose(E, D, rtol=1e-14)


def test_ruiz_equilibrates_rows_and_columns():
    """Fixed point: every row of DAE has l2 norm 1 and every column sqrt(m/n) (sparse LP pattern)."""
    p = W.sparse_lp(5, 40, 100, 16, row_log10=2, col_log10=1)   # dense enough for an exact equilibration to exist
    o = oracle.Oracle.from_problem(p)
    D, E = o.ruiz(400)
    B = sp.diags(D) @ p.csr() @ sp.diags(E)
    rn = np.sqrt(np.asarray(B.multiply(B).sum(axis=1)).ravel())
    cn = np.sqrt(np.asarray(B.multiply(B).sum(axis=0)).ravel())
    assert np.allclose(rn, 1.0, atol=1e-8) and np.allclose(cn, np.sqrt(40 / 100), atol=1e-8)
    assert (D > 0).all() and (E > 0).all()


def test_ruiz_undoes_a_diagonal_scaling_of_a_sign_matrix():
    """A = D0 S E0 with |S_ij| = 1: the only equilibrated scaling of the pattern is |B_ij| = 1/sqrt(n)."""
    rng = np.random.default_rng(3)
    m, n = 6, 9
    S = rng.choice([-1.0, 1.0], size=(m, n))
    A = sp.csr_matrix(np.diag(10 ** rng.uniform(-3, 3, m)) @ S @ np.diag(10 ** rng.uniform(-2, 2, n)))
    o = oracle.Oracle(m, n, A.indptr, A.indices, A.data, np.ones(m), np.ones(n), n, [])
    D, E = o.ruiz(60)
    B = np.diag(D) @ A.toarray() @ np.diag(E)
    assert np.allclose(np.abs(B), 1 / np.sqrt(n), rtol=1e-10)


def test_ruiz_is_constant_on_lorentz_blocks():
    """E commutes with K: one factor per block; the block MEAN of the squared column norms
    is what reaches m/n."""
    p = W.sparse_socp(11, 30, 90, 8, 4, n_lin=10, lo=3, hi=12)
    o = oracle.Oracle.from_problem(p)
    D, E = o.ruiz(300)
    B = sp.diags(D) @ p.csr() @ sp.diags(E)
    c2 = np.asarray(B.multiply(B).sum(axis=0)).ravel()
    a = p.n_lin
    assert np.allclose(c2[:a], 30 / 90, atol=1e-8)
    for sz in p.soc_size:
        assert np.ptp(E[a:a + sz]) == 0.0
        assert np.isclose(c2[a:a + sz].mean(), 30 / 90, atol=1e-8)
        a += sz
    # and the run on the equilibrated data reaches the same optimum (Algorithm 1 on scaled data)
    o.set_scaling(E)
    o.run_fixed(4000)
    r = o.residuals()
    assert r["kkt_rel"] < 1e-6 and np.isclose(r["pobj"], p.opt_value(), rtol=1e-5, atol=1e-6)


# ------------------------------------------------------------------ hand-computed 1 x 2 LP (tests/golden/hand_1x2_lp.txt)
def _hand_lp(mu=1.0, t=9.2):
    A = np.array([[1.0, 1.0]])
    return _problem_from_dense(A, np.array([2.0]), np.array([1.0, 3.0]), 2, [], mu=mu, t=t)


def test_residuals_hand_example_every_term():
    """orc_residuals term by term ((16a) P:332, (16b) P:335, (34) P:566-572) on a NON-optimal iterate whose x, z, y
    and every norm are rational numbers worked out by hand in the golden file: mu = 2 (a dropped 1/mu in y or z
    shows), ||b|| = 2 != ||c|| = sqrt(10) (a swapped normaliser shows), all four relative terms distinct and the
    maximum attained by the gap (a max over the wrong terms shows)."""
    g = _golden("hand_1x2_lp.txt")
    o = oracle.Oracle.from_problem(_hand_lp(mu=2.0))
    o.run(1)
    sol, r = o.get(), o.residuals()
    assert np.allclose(sol["x"], [g["mu2_x1"], g["mu2_x2"]], rtol=0, atol=1e-15)
    assert np.allclose(sol["z"], [g["mu2_z1"], g["mu2_z2"]], rtol=0, atol=1e-15)
    assert np.allclose(sol["y"], [g["mu2_y"]], rtol=0, atol=1e-15)
    for k in oracle.RESID_FIELDS:
        assert abs(r[k] - g["mu2_" + k]) <= 1e-15 * (1 + abs(g["mu2_" + k])), (k, r[k], g["mu2_" + k])
    terms = sorted(r[k] for k in ("pres_rel", "dres_rel", "gap_rel", "cone_viol_rel"))
    assert all(b - a > 1e-3 for a, b in zip(terms, terms[1:]))      # the pin can tell the four apart


def test_residuals_term_by_term_on_a_mixed_cone_iterate():
    """The same terms on a mid-run (non-optimal) iterate of a mixed orthant + Lorentz problem, evaluated with scipy
    sparse products and with the cone distance taken from Definition 1 as a constrained minimisation
    (SLSQP), not from the closed form the oracle uses."""
    p = W.sparse_socp(21, 30, 80, 8, 4, n_lin=20, lo=2, hi=12)
    p.mu = 1.7
    o = oracle.Oracle.from_problem(p)
    o.run(7, L=[4])
    s, r = o.get(), o.residuals()
    A, x, z, y = p.csr(), s["x"], s["z"], s["y"]

    def dist_K(v):
        tot, off = float(np.sum(np.minimum(v[:p.n_lin], 0.0) ** 2)), p.n_lin
        for sz in p.soc_size.tolist():
            blk = v[off:off + sz]
            if sz == 1:
                tot += min(blk[0], 0.0) ** 2
            else:
                cons = {"type": "ineq", "fun": lambda u: u[0] ** 2 - np.sum(u[1:] ** 2)}
                best = min((so.minimize(lambda u: np.sum((u - blk) ** 2), u0, constraints=[cons], bounds=[(0, None)] + [(None, None)] * (sz - 1),
                                        method="SLSQP", options={"ftol": 1e-15, "maxiter": 500}).fun
                            for u0 in (np.r_[np.linalg.norm(blk) + 1.0, blk[1:]], np.r_[1.0, np.zeros(sz - 1)])))
                tot += max(best, 0.0)
            off += sz
        return np.sqrt(tot)

    pres, dres = np.linalg.norm(A @ x - p.b), np.linalg.norm(p.c - z - A.T @ y)
    cx, by = float(p.c @ x), float(p.b @ y)
    exp = {"pres_abs": pres, "pres_rel": pres / (1 + np.linalg.norm(p.b)), "dres_abs": dres,
           "dres_rel": dres / (1 + np.linalg.norm(p.c)), "gap_abs": abs(cx - by),
           "gap_rel": abs(cx - by) / (1 + abs(cx) + abs(by)), "pobj": cx, "dobj": by}
    for k, v in exp.items():
        assert abs(r[k] - v) <= 1e-11 * (1 + abs(v)), (k, r[k], v)
    cv = (dist_K(x) + dist_K(z)) / (1 + np.linalg.norm(x) + np.linalg.norm(z))
    assert cv > 1e-3 and abs(r["cone_viol_rel"] - cv) <= 1e-6 * cv, (r["cone_viol_rel"], cv)   # SLSQP accuracy
    assert r["kkt_rel"] == max(r["pres_rel"], r["dres_rel"], r["gap_rel"], r["cone_viol_rel"])
    assert min(r["pres_rel"], r["dres_rel"], r["gap_rel"], r["cone_viol_rel"]) > 1e-6     # nothing is at its zero


def test_o_floor_branch_hand_example():
    """Step 7 with exact zeros, reading (g): numerator AND denominator are floored at o_floor, separately.
    K = R^3_+ x K_3 x K_2, o_floor = 1e-3:
        x = (0, 2, 5 | 5, 3, 4 | 0, 0),  z = (4, 0, 5 | 2, ., . | 0, .)
        o = (1e-3/4, 2/1e-3, 5/5 | |5 - 5| -> 1e-3, /2 | 1e-3/1e-3) = (2.5e-4, 2000, 1, 5e-4, 1)
    (flooring the ratio instead would give 1e-3, inf, 1, 1e-3, nan).  t = 50: alpha = 1 and O = o; t = ln 100:
    alpha = ln 100 / ln(2000/2.5e-4)."""
    rng = np.random.default_rng(4)
    x = np.array([0.0, 2.0, 5.0, 5.0, 3.0, 4.0, 0.0, 0.0])
    z = np.array([4.0, 0.0, 5.0, 2.0, 0.7, -0.2, 0.0, 0.3])
    o_exp = np.array([2.5e-4, 2000.0, 1.0, 5e-4, 5e-4, 5e-4, 1.0, 1.0])
    A = rng.standard_normal((2, 8))
    for t, alpha in ((50.0, 1.0), (np.log(100.0), np.log(100.0) / np.log(2000.0 / 2.5e-4))):
        p = _problem_from_dense(A, A @ np.abs(x), rng.standard_normal(8), 3, [3, 2], t=t)
        o = oracle.Oracle.from_problem(p, o_floor=1e-3)
        o.set_point(x, z)
        o.run(1)
        O = o.get()["O"]
        assert np.all(np.isfinite(O)) and np.allclose(O, o_exp ** alpha, rtol=1e-13), (t, O)
    # the default floor (1e-16) only guards exact zeros; the cap of step 11 then keeps O moderate
    o_def = np.array([1e-16 / 4, 2 / 1e-16, 1.0, 5e-17, 5e-17, 5e-17, 1.0, 1.0])
    alpha = np.log(100.0) / np.log(o_def.max() / o_def.min())
    p = _problem_from_dense(A, A @ np.abs(x), rng.standard_normal(8), 3, [3, 2], t=np.log(100.0))
    o = oracle.Oracle.from_problem(p)
    o.set_point(x, z)
    o.run(1)
    assert np.allclose(o.get()["O"], o_def ** alpha, rtol=1e-13)


def test_L_membership_timing_hand_example():
    """Step 4: l in L conditions at the START of iteration l, from the (x, z) left by iteration l-1.
    Hand-computed in the golden file: with L = {3} the rule sees (x2, z2) = ((5/2,-1/2), (-1/2,1/2)) => O = (5, 1)
    and iteration 3 ends at x = (240/26, -19/26), z = (6/26, 45/26); one iteration late it would see
    (x3, z3) = ((3,-1/2), (0, 3/2)) => o = (3/o_floor, 1/3)."""
    g = _golden("hand_1x2_lp.txt")
    o = oracle.Oracle.from_problem(_hand_lp())
    o.run(2, L=[3])
    assert np.array_equal(o.get()["O"], [1.0, 1.0])                 # not yet
    assert np.allclose(o.get()["x"], [2.5, -0.5], atol=1e-15) and np.allclose(o.get()["z"], [-0.5, 0.5], atol=1e-15)
    o.run(1, L=[3])
    s = o.get()
    assert np.allclose(s["O"], [g["L3_O1"], g["L3_O2"]], rtol=1e-14)
    assert np.allclose(s["x"], [g["L3_x1"], g["L3_x2"]], rtol=1e-13) and np.allclose(s["z"], [g["L3_z1"], g["L3_z2"]], rtol=1e-13)
    assert np.allclose(s["s"], [g["L3_s1"], g["L3_s2"]], rtol=1e-13)
    assert o.counters()["n_cond"] == 2
    o2 = oracle.Oracle.from_problem(_hand_lp())
    o2.run(3)                                                       # L = {}: a different third iterate
    s2 = o2.get()
    assert np.allclose(s2["x"], [g["noL_x1"], g["noL_x2"]], atol=1e-14) and np.allclose(s2["z"], [g["noL_z1"], g["noL_z2"]], atol=1e-14)
    o3 = oracle.Oracle.from_problem(_hand_lp())
    o3.run(4, L=[4])                                                # L = {4}: the rule sees (x3, z3); z3_1 = 0 hits the floor
    O3 = o3.get()["O"]
    assert O3[0] / O3[1] > 1e3 and not np.allclose(O3, [5.0, 1.0])


def test_exact_solve_resolves_the_projection_on_an_ill_conditioned_system():
    """Reading (s): the solve inside A^dagger is exact.  On the config-2 recipe (rows 10^U(-3,3), columns 10^U(-2,2))
    both solve modes must give A^dagger rhs to ~1e-13 of a reference obtained by iterative refinement with
    EXTENDED-precision residuals (numpy longdouble, dense): the dense Cholesky with its two refinement steps, and the
    Jacobi-PCG at its tight tolerance."""
    import scipy.linalg as sl
    p = W.config(2, 0.004)
    A = p.csr().toarray()
    Al = A.astype(np.longdouble)
    G = A @ A.T
    e = 1.0 / np.sqrt(np.diag(G))
    Lc = np.linalg.cholesky(G * np.outer(e, e))
    apply = lambda r: e * sl.solve_triangular(Lc.T, sl.solve_triangular(Lc, e * r, lower=True), lower=False)
    rhs = A @ np.random.default_rng(0).standard_normal(p.n)
    w = apply(rhs).astype(np.longdouble)
    for _ in range(8):
        w = w + apply(np.asarray(rhs - Al @ (Al.T @ w), dtype=np.float64)).astype(np.longdouble)
    ref = np.asarray(Al.T @ w, dtype=np.float64)
    assert np.linalg.cond(G) > 1e10
    for mode, tol, bound in ((1, 1e-14, 2e-14), (2, 1e-15, 5e-13)):
        o = oracle.Oracle.from_problem(p, solve_mode=mode, pcg_tol=tol, pcg_max=100000)
        o.run(1)                                                    # l = 1: O = I
        err = np.linalg.norm(o.pinv_apply(rhs) - ref) / np.linalg.norm(ref)
        assert err <= bound, (mode, err)


def test_singleton_rows_make_the_zipf_draw_rank_deficient():
    """Reading (r)/(x): the proofs use A A^dagger = I, i.e. full row rank.  The steep Zipf draw of the GPU shape
    sweep with rows topped up to ONE entry only has singleton rows that share a column -- two parallel rows, so A is
    rank-deficient whatever the values -- and the oracle's Cholesky refuses such a matrix; topped up to two entries
    the draw has no such pair (and thousands of 2-3-entry rows), which is the case the GPU sweep keeps."""
    def parallel_singletons(p):
        single = np.flatnonzero(np.diff(p.row_ptr) == 1)
        cols = p.col_idx[p.row_ptr[single]]
        return single.size, single.size - np.unique(cols).size
    bad = W.sparse_lp(15, 4000, 12000, 4, zipf=1.6, min_row_nnz=1)
    n_single, n_shared = parallel_singletons(bad)
    assert n_single > 1000 and n_shared > 10
    small = W.sparse_lp(15, 600, 1800, 4, zipf=1.6, min_row_nnz=1)
    assert parallel_singletons(small)[1] > 0
    with pytest.raises(RuntimeError):
        oracle.Oracle.from_problem(small, solve_mode=1).run(1)
    ok = W.sparse_lp(15, 4000, 12000, 4, zipf=1.6, min_row_nnz=2)
    assert parallel_singletons(ok) == (0, 0) and (np.diff(ok.row_ptr) < 4).sum() > 1000
