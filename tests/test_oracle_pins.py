"""Pins of the CPU oracle against things other than itself (CPU only, `-m "not gpu"`).

Each test names the passage of /root/reference/PAPER.md (P:<line>) or the mathematical fact it uses.
Independent referees used here: numpy.linalg (pinv, svd, solve), scipy.optimize (linprog/HiGHS,
SLSQP), brute-force vertex enumeration, hand-computed constants and the paper's printed numbers.
"""
import itertools
import os

import numpy as np
import pytest
import scipy.optimize as so

import oracle
from paper_2103_00736_b200 import workloads as W

RNG = np.random.default_rng(12345)


def _rand_cone_vec(rng, n_lin, sizes, scale=1.0):
    return scale * rng.standard_normal(n_lin + int(np.sum(sizes)))


# ------------------------------------------------------------------ 1. cone operators (Def.1)
@pytest.mark.parametrize("n_lin,sizes", [(5, []), (0, [3, 4, 2, 7]), (3, [1, 2, 40, 3])])
def test_cone_operators_invariants(n_lin, sizes):
    sizes = np.array(sizes, np.int32)
    for trial in range(50):
        v = _rand_cone_vec(RNG, n_lin, sizes, 10.0 ** RNG.uniform(-3, 3))
        P = oracle.proj_cone(v, n_lin, sizes)
        Pm = oracle.proj_cone(-v, n_lin, sizes)
        # idempotent
        assert np.allclose(oracle.proj_cone(P, n_lin, sizes), P, rtol=1e-14, atol=0)
        # Moreau: v = proj_K(v) - proj_K(-v), <proj_K(v), proj_K(-v)> = 0  (K self-dual)
        assert np.allclose(P - Pm, v, rtol=1e-13, atol=1e-13 * np.abs(v).max())
        assert abs(P @ Pm) <= 1e-12 * (v @ v)
        a = oracle.abs_cone(v, n_lin, sizes)
        # abs_K = proj_K(v) + proj_K(-v) ; norm preserving (eq.(20)) ; abs(abs(v)) = abs(v)
        assert np.allclose(a, P + Pm, rtol=1e-13, atol=1e-13 * np.abs(v).max())
        assert np.isclose(np.linalg.norm(a), np.linalg.norm(v), rtol=1e-13)
        assert np.allclose(oracle.abs_cone(a, n_lin, sizes), a, rtol=1e-13, atol=1e-13 * np.abs(v).max())
        # the result lies in K: first coordinate >= norm of the tail
        off = n_lin
        assert (a[:n_lin] >= 0).all()
        for sz in sizes:
            assert a[off] >= np.linalg.norm(a[off + 1:off + sz]) * (1 - 1e-13)
            off += sz


def test_size1_cone_is_abs_and_orthant():
    v = RNG.standard_normal(64)
    assert np.array_equal(oracle.abs_cone(v, 64, []), np.abs(v))
    assert np.array_equal(oracle.abs_cone(v, 0, np.ones(64, np.int32)), np.abs(v))
    assert np.array_equal(oracle.proj_cone(v, 64, []), np.maximum(v, 0.0))


def test_soc_projection_is_the_argmin():
    """Def.1: proj = argmin ||u-v|| over the cone, checked with a constrained optimiser."""
    for k in (2, 3, 5):
        for trial in range(8):
            v = RNG.standard_normal(k) * 3
            P = oracle.proj_cone(v, 0, np.array([k], np.int32))
            cons = {"type": "ineq", "fun": lambda u: u[0] ** 2 - u[1:] @ u[1:] if u[0] >= 0 else u[0]}
            best = None
            for start in (np.r_[np.linalg.norm(v) + 1, v[1:]], np.r_[1.0, np.zeros(k - 1)], P + 0.1):
                res = so.minimize(lambda u: 0.5 * (u - v) @ (u - v), start, jac=lambda u: u - v,
                                  constraints=[cons, {"type": "ineq", "fun": lambda u: u[0]}], method="SLSQP",
                                  options={"ftol": 1e-14, "maxiter": 500})
                if best is None or res.fun < best.fun:
                    best = res
            assert 0.5 * (P - v) @ (P - v) <= best.fun + 1e-7
            assert np.allclose(P, best.x, atol=2e-4)


def test_lemma1_inequality_21():
    """(21) P:466: <|u|*,|v|*> >= <u,v> with |.|* = abs_A(abs_K(.)) (19) P:457."""
    p = W.sparse_socp(7, 30, 60, 10, 4, n_lin=10, lo=2, hi=8)
    o = oracle.Oracle.from_problem(p)
    o.run(1)
    for trial in range(20):
        u, v = RNG.standard_normal(p.n), RNG.standard_normal(p.n)
        su = o.abs_range(oracle.abs_cone(u, p.n_lin, p.soc_size))
        sv = o.abs_range(oracle.abs_cone(v, p.n_lin, p.soc_size))
        assert su @ sv >= u @ v - 1e-10
        assert np.isclose(np.linalg.norm(su), np.linalg.norm(u), rtol=1e-11)  # (20)


# ------------------------------------------------------------------ 2/3. subspace reflector, affine projection
@pytest.mark.parametrize("mode", [1, 2])
def test_reflector_and_pinv_against_numpy(mode):
    p = W.sparse_lp(3, 40, 90, 4)
    o = oracle.Oracle.from_problem(p, solve_mode=mode)
    O = np.exp(RNG.uniform(-2, 2, p.n))
    o.set_scaling(O)
    Ahat = p.csr().toarray() * O[None, :]
    pinv = np.linalg.pinv(Ahat)  # independent library routine
    v = RNG.standard_normal(p.n)
    rhs = RNG.standard_normal(p.m)
    assert np.allclose(o.pinv_apply(rhs), pinv @ rhs, rtol=1e-9, atol=1e-11)
    refl = 2 * pinv @ (Ahat @ v) - v  # (2 A^dagger A - I) v, (37b) P:591
    got = o.abs_range(v)
    assert np.allclose(got, refl, rtol=1e-9, atol=1e-11)
    assert np.isclose(np.linalg.norm(got), np.linalg.norm(v), rtol=1e-12)
    assert np.allclose(o.abs_range(got), v, atol=1e-10)  # a reflector is an involution
    assert np.allclose(o.mat_vec(got), Ahat @ v, atol=1e-9)  # A(2P-I)v = Av
    assert np.allclose(o.mat_vec(v), Ahat @ v, rtol=1e-13, atol=1e-13)
    assert np.allclose(o.mat_tvec(rhs), Ahat.T @ rhs, rtol=1e-13, atol=1e-13)
    # affine projection Pi(x) = x - A^dagger(Ax - b) lands on {Ax=b} to 1e-10 (BASELINE north_star)
    x = RNG.standard_normal(p.n)
    pi = x - o.pinv_apply(Ahat @ x - p.b)
    assert np.linalg.norm(Ahat @ pi - p.b) <= 1e-10


# ------------------------------------------------------------------ 4. fixed point (22),(23) P:470-478
@pytest.mark.parametrize("kind", ["lp", "socp"])
def test_constructed_optimum_is_a_fixed_point_for_any_block_scaling(kind):
    p = W.sparse_lp(11, 30, 70, 4) if kind == "lp" else W.sparse_socp(11, 40, 90, 12, 5, n_lin=6, lo=2, hi=12)
    for trial in range(3):
        o = oracle.Oracle.from_problem(p)
        blocks = np.r_[np.ones(p.n_lin, np.int64), p.soc_size]
        Ob = np.exp(RNG.uniform(-1.5, 1.5, blocks.size)) if trial else np.ones(blocks.size)
        O = np.repeat(Ob, blocks)
        o.set_point(p.x0, p.s0)       # (x_opt, z_opt)
        o.set_scaling(O)              # steps 12-14: s = O^-1 x - mu O z = s_opt of the scaled problem
        s_opt = p.x0 / O - p.mu * O * p.s0
        g = o.get()
        assert np.allclose(g["s"], s_opt, rtol=1e-15, atol=0)
        # (23): d = (s_opt + |s_opt|*)/2
        star = o.abs_range(oracle.abs_cone(s_opt, p.n_lin, p.soc_size))
        assert np.allclose(g["d"], 0.5 * (s_opt + star), atol=1e-10 * (1 + np.abs(s_opt).max()))
        o.run_fixed(3)
        g = o.get()
        sc = 1 + np.abs(s_opt).max()
        assert np.linalg.norm(g["s"] - s_opt) <= 1e-10 * sc
        assert np.linalg.norm(g["x"] - p.x0) <= 1e-10 * sc
        assert np.linalg.norm(g["z"] - p.s0) <= 1e-10 * sc
        assert np.linalg.norm(g["y"] - p.y0) <= 1e-8 * (1 + np.abs(p.y0).max())  # derived y
        r = o.residuals()
        assert r["kkt_rel"] <= 1e-10
        assert np.isclose(r["pobj"], p.opt_value(), rtol=1e-10, atol=1e-10)


# ------------------------------------------------------------------ 5. Fejer monotonicity (30), summability (31)
def test_fejer_monotone_and_summable():
    p = W.sparse_socp(5, 40, 90, 12, 5, n_lin=6, lo=2, hi=12)
    o = oracle.Oracle.from_problem(p)
    s_opt = p.x0 - p.mu * p.s0
    o.run(1)
    prev_s = o.get()["s"]
    dist0 = None
    total = 0.0
    prev = np.linalg.norm(prev_s - s_opt)
    for l in range(150):
        if dist0 is None:
            dist0 = prev ** 2
        o.run(1)
        s = o.get()["s"]
        total += np.linalg.norm(s - prev_s) ** 2
        cur = np.linalg.norm(s - s_opt)
        assert cur <= prev * (1 + 1e-12) + 1e-12
        prev, prev_s = cur, s
    assert total <= dist0 * (1 + 1e-9)
