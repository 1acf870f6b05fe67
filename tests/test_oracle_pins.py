"""Pins of the CPU oracle against things that are NOT the oracle (CPU only, -m "not gpu").

The paper prints no worked numerical example for aprod1/aprod2/LSQR (PAPER.md has only
Eqs. 1-3 and the solver outline), so the oracle is pinned by: a dense brute-force matrix
built through a third, independent column map (tests/helpers.py); hand-worked integer
cases; the adjoint identity; += semantics; numpy.linalg.lstsq; scipy.sparse.linalg.lsqr
(an independent Paige-Saunders implementation); residual identities and closed forms.
Every plausible slip (dropped block, wrong axis offset, transposed operand, sign of a
rotation, wrong stopping rule) fails at least one of these.
"""
import numpy as np
import pytest

import oracle
from gaia_synth import host
from gaia_synth.configs import C1, SystemShape
from helpers import (columns_of, csr_matrix, dense_matrix, nonempty_columns, rhs, tiny_shape)


def _read_golden(name):
    """tests/golden/<name>: lines `key v v v ...` (ints; `|` separators ignored), repeated keys accumulate."""
    import os
    out = {}
    with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", name)) as f:
        for ln in f:
            ln = ln.split("#")[0].strip()
            if ln:
                k, *v = ln.replace("|", " ").split()
                out.setdefault(k, []).append([int(t) for t in v])
    return out


def _sys(shape):
    a, idx = host.make_rows(shape)
    return a, idx, oracle.layout_of(shape)


# ------------------------------------------------------------------ aprod: hand-worked case
def test_hand_worked_two_rows():
    """S=2, K=5, I=3, G=1 -> n = 10 + 15 + 3 + 1 = 29.  Integer data, results by hand.
    x[j] = j+1.  Row 0: star 0, att_start 1, instr (0,2,1,0,2,1); a[0][k] = 1 for all k.
      astro  cols 0..4            -> 1+2+3+4+5                = 15
      att    cols 10+{1..4}, 15+{1..4}, 20+{1..4} -> x = 12..15, 17..20, 22..25
                                   -> 54 + 74 + 94             = 222
      instr  cols 25+{0,2,1,0,2,1} -> x = 26,28,27,26,28,27    = 162
      glob   col 28               -> 29
      y[0] = 15 + 222 + 162 + 29 = 428
    Row 1: star 1, att_start 0, instr (1,1,1,1,1,1); a[1][k] = k (0..23).
      astro cols 5..9: 0*6+1*7+2*8+3*9+4*10                      = 90
      att: slots 5..8 cols 10..13 (x 11..14): 5*11+6*12+7*13+8*14 = 330
           slots 9..12 cols 15..18 (x 16..19): 9*16+10*17+11*18+12*19 = 740
           slots 13..16 cols 20..23 (x 21..24): 13*21+14*22+15*23+16*24 = 1310
      instr: col 26 (x 27) six times: (17+18+19+20+21+22)*27 = 117*27 = 3159
      glob: 23*29 = 667
      y[1] = 90+330+740+1310+3159+667 = 6296
    aprod2 with y = (1, 2), x0 = 0: x[26] = a0 part (slots 19 and 22 -> 1+1)*1 + 117*2 = 236;
      x[28] = 1*1 + 23*2 = 47; x[0] = 1; x[9] = 4*2 = 8; x[11] = row0 slot5 (1) + row1 slot6 (6*2) = 13.
    """
    g = _read_golden("two_rows.txt")
    S, K, I, G = g["layout"][0]
    L = oracle.layout(S, K, I, G)
    assert oracle.n_unknowns(L) == 29
    idx = np.array([r[:8] for r in g["row"]], dtype=np.int32)
    a = np.array([r[8:] for r in g["row"]], dtype=np.float64)
    assert a.shape == (2, 24) and a[1].tolist() == list(range(24))
    x = np.arange(1, 30, dtype=np.float64)
    y = oracle.aprod1(L, a, idx, x, np.zeros(2))
    assert y.tolist() == [float(v) for v in g["aprod1_y"][0]]
    x2 = oracle.aprod2(L, a, idx, np.array([1.0, 2.0]), np.zeros(29))
    for j, v in g["aprod2_x"]:
        assert x2[j] == float(v)
    # n_glob = 0: slot 23 is ignored and x has 28 entries
    L0 = oracle.layout(S, K, I, 0)
    y0 = oracle.aprod1(L0, a, idx, x[:28].copy(), np.zeros(2))
    assert y0.tolist() == [float(v) for v in g["aprod1_y_noglob"][0]]
    x0 = oracle.aprod2(L0, a, idx, np.array([1.0, 2.0]), np.zeros(28))
    assert x0.shape == (28,)
    for j, v in g["aprod2_x_noglob"]:
        assert x0[j] == float(v)


def test_col_map_matches_independent_map():
    shape = tiny_shape(n_stars=5, obs=7, n_knots=9, n_instr=11)
    a, idx, L = _sys(shape)
    cols = columns_of(shape, idx)
    for r in (0, 3, 17, idx.shape[0] - 1):
        for k in range(24):
            assert oracle.col(L, idx[r], k) == cols[r, k]
    shape0 = tiny_shape(n_glob=0)
    _, idx0 = host.make_rows(shape0)
    assert oracle.col(oracle.layout_of(shape0), idx0[0], 23) == -1


# ------------------------------------------------------------------ aprod: dense brute force
@pytest.mark.parametrize("n_glob", [1, 0])
def test_dense_brute_force(n_glob):
    shape = tiny_shape(n_stars=6, obs=9, n_knots=10, n_instr=7, n_glob=n_glob, seed=99)
    a, idx, L = _sys(shape)
    m, n = a.shape[0], shape.n_unknowns
    D = dense_matrix(shape, a, idx)
    x = host.test_vector(1, 1, n)
    y = host.test_vector(1, 2, m)
    y1 = oracle.aprod1(L, a, idx, x, np.zeros(m))
    x1 = oracle.aprod2(L, a, idx, y, np.zeros(n))
    np.testing.assert_allclose(y1, D @ x, rtol=0, atol=1e-13 * np.abs(D).dot(np.abs(x)).max())
    np.testing.assert_allclose(x1, D.T @ y, rtol=0, atol=1e-13 * np.abs(D.T).dot(np.abs(y)).max())
    # recover D entry by entry through the API: single products are bit-exact
    for j in range(n):
        e = np.zeros(n)
        e[j] = 1.0
        col_j = oracle.aprod1(L, a, idx, e, np.zeros(m))
        assert np.array_equal(col_j, D[:, j]) or np.allclose(col_j, D[:, j], rtol=0, atol=1e-15)
    for r in range(0, m, 5):
        e = np.zeros(m)
        e[r] = 1.0
        row_r = oracle.aprod2(L, a, idx, e, np.zeros(n))
        np.testing.assert_allclose(row_r, D[r], rtol=0, atol=1e-15)


def test_duplicate_instr_columns_accumulate():
    shape = tiny_shape(n_stars=2, obs=3, n_knots=6, n_instr=6)
    a, idx, L = _sys(shape)
    idx[:, 2:8] = np.array([1, 1, 3, 1, 0, 3], dtype=np.int32)   # repeated columns in a row
    D = dense_matrix(shape, a, idx)
    x = host.test_vector(2, 1, shape.n_unknowns)
    y = host.test_vector(2, 2, a.shape[0])
    np.testing.assert_allclose(oracle.aprod1(L, a, idx, x, np.zeros(a.shape[0])), D @ x, atol=1e-13)
    np.testing.assert_allclose(oracle.aprod2(L, a, idx, y, np.zeros(shape.n_unknowns)), D.T @ y, atol=1e-13)


def test_att_start_upper_edge_K_minus_4():
    shape = tiny_shape(n_stars=2, obs=2, n_knots=6, n_instr=6)
    a, idx, L = _sys(shape)
    idx[:, 1] = shape.n_knots - 4                     # natural upper bound (touches knot K-1)
    D = dense_matrix(shape, a, idx)
    x = host.test_vector(3, 1, shape.n_unknowns)
    np.testing.assert_allclose(oracle.aprod1(L, a, idx, x, np.zeros(4)), D @ x, atol=1e-13)
    xo = oracle.aprod2(L, a, idx, np.ones(4), np.zeros(shape.n_unknowns))
    for ax in range(3):                               # last knot of each axis is hit
        assert xo[shape.off_att + ax * shape.n_knots + shape.n_knots - 1] != 0.0


def test_single_star_astro_only_is_dense_5_columns():
    shape = tiny_shape(n_stars=1, obs=11, n_knots=5, n_instr=6)
    a, idx, L = _sys(shape)
    a[:, 5:] = 0.0
    x = host.test_vector(4, 1, shape.n_unknowns)
    y = oracle.aprod1(L, a, idx, x, np.zeros(11))
    np.testing.assert_allclose(y, a[:, :5] @ x[:5], rtol=1e-14, atol=1e-15)
    yv = host.test_vector(4, 2, 11)
    xo = oracle.aprod2(L, a, idx, yv, np.zeros(shape.n_unknowns))
    np.testing.assert_allclose(xo[:5], a[:, :5].T @ yv, rtol=1e-14, atol=1e-15)


def test_zero_block_leaves_x_untouched_bitwise():
    shape = tiny_shape()
    a, idx, L = _sys(shape)
    a[:, 5:17] = 0.0                                   # no attitude coefficients
    x0 = host.test_vector(5, 1, shape.n_unknowns)
    x1 = oracle.aprod2(L, a, idx, host.test_vector(5, 2, a.shape[0]), x0.copy())
    sl = slice(shape.off_att, shape.off_instr)
    assert np.array_equal(x1[sl], x0[sl])
    assert not np.array_equal(x1[:shape.off_att], x0[:shape.off_att])


# ------------------------------------------------------------------ aprod: identities at C1 size
def test_adjoint_identity_c1():
    a, idx, L = _sys(C1)
    m, n = a.shape[0], C1.n_unknowns
    for t in range(3):
        x = host.test_vector(10 + t, 1, n)
        y = host.test_vector(10 + t, 2, m)
        Ax = oracle.aprod1(L, a, idx, x, np.zeros(m))
        ATy = oracle.aprod2(L, a, idx, y, np.zeros(n))
        lhs, rhs_ = Ax @ y, x @ ATy
        assert abs(lhs - rhs_) <= 1e-13 * np.linalg.norm(Ax) * np.linalg.norm(y)


def test_accumulate_semantics_and_linearity():
    a, idx, L = _sys(C1)
    m, n = a.shape[0], C1.n_unknowns
    x = host.test_vector(20, 1, n)
    y0 = host.test_vector(20, 2, m)
    inc = oracle.aprod1(L, a, idx, x, np.zeros(m))
    once = oracle.aprod1(L, a, idx, x, y0.copy())
    twice = oracle.aprod1(L, a, idx, x, once.copy())
    scale = np.abs(y0) + 2 * np.abs(inc) + 1.0
    assert np.all(np.abs(once - (y0 + inc)) <= 1e-13 * scale)        # pre-filled y preserved
    assert np.all(np.abs(twice - (y0 + 2 * inc)) <= 1e-13 * scale)   # second call doubles the increment
    lin = oracle.aprod1(L, a, idx, 3.0 * x, np.zeros(m))
    assert np.all(np.abs(lin - 3.0 * inc) <= 1e-13 * (3 * np.abs(inc) + 1.0))
    yv = host.test_vector(20, 3, m)
    x0 = host.test_vector(20, 4, n)
    incx = oracle.aprod2(L, a, idx, yv, np.zeros(n))
    oncex = oracle.aprod2(L, a, idx, yv, x0.copy())
    np.testing.assert_allclose(oncex, x0 + incx, rtol=0, atol=1e-11 * np.abs(incx).max())


def test_csr_matches_oracle_c1():
    """scipy CSR mat-vec (library routine) on the matrix built through the independent map."""
    a, idx, L = _sys(C1)
    A = csr_matrix(C1, a, idx)
    x = host.test_vector(30, 1, C1.n_unknowns)
    y = host.test_vector(30, 2, a.shape[0])
    Ax = oracle.aprod1(L, a, idx, x, np.zeros(a.shape[0]))
    bound = abs(A).dot(np.abs(x))
    assert np.all(np.abs(Ax - A @ x) <= 1e-13 * bound)
    ATy = oracle.aprod2(L, a, idx, y, np.zeros(C1.n_unknowns))
    ref = A.T @ y
    assert np.linalg.norm(ATy - ref) <= 1e-13 * np.linalg.norm(ref)
    # three attitude columns (knot K-1 of each axis) are empty by construction (reading R3)
    empty = ~nonempty_columns(C1, idx)
    assert empty.sum() >= 3
    for ax in range(3):
        assert empty[C1.off_att + ax * C1.n_knots + C1.n_knots - 1]


def test_omp_and_compensated_variants_agree():
    a, idx, L = _sys(C1)
    m, n = a.shape[0], C1.n_unknowns
    x = host.test_vector(40, 1, n)
    y = host.test_vector(40, 2, m)
    s1 = oracle.aprod1(L, a, idx, x, np.zeros(m))
    p1 = oracle.aprod1(L, a, idx, x, np.zeros(m), threads=4)
    assert np.array_equal(s1, p1)                                  # same per-row arithmetic
    s2 = oracle.aprod2(L, a, idx, y, np.zeros(n))
    p2 = oracle.aprod2(L, a, idx, y, np.zeros(n), threads=4)
    assert np.linalg.norm(s2 - p2) <= 1e-13 * np.linalg.norm(s2)
    assert np.array_equal(s2[:C1.off_att], p2[:C1.off_att])        # astro part: same order
    xc, comp = np.zeros(n), np.zeros(n)
    oracle.aprod2_comp(L, a, idx, y, xc, comp)
    assert np.linalg.norm((xc + comp) - s2) <= 1e-13 * np.linalg.norm(s2)
    bound = oracle.aprod1_abs(L, a, idx, x)
    assert np.all(bound >= np.abs(s1) * (1 - 1e-12))


# ------------------------------------------------------------------ LSQR
def test_lsqr_matches_dense_least_squares():
    """Tiny well-conditioned system vs numpy.linalg.lstsq (min-norm, so empty columns agree)."""
    shape = tiny_shape(n_stars=8, obs=12, n_knots=8, n_instr=8, seed=7)
    a, idx, L = _sys(shape)
    D = dense_matrix(shape, a, idx)
    b = rhs(shape, a, idx, host.x_true(shape))
    xr = np.linalg.lstsq(D, b, rcond=None)[0]
    x, res = oracle.lsqr(L, a, idx, b, itnlim=2000, atol=1e-14, btol=1e-14, conlim=0)
    assert res["istop"] in (1, 2)
    assert np.linalg.norm(x - xr) <= 1e-10 * np.linalg.norm(xr)
    assert abs(res["r1norm"] - np.linalg.norm(b - D @ x)) <= 1e-8 * res["bnorm"]


def test_lsqr_matches_scipy_c1():
    from scipy.sparse.linalg import lsqr as sp_lsqr
    a, idx, L = _sys(C1)
    A = csr_matrix(C1, a, idx)
    xt = host.x_true(C1)
    b = rhs(C1, a, idx, xt)
    x, res = oracle.lsqr(L, a, idx, b, itnlim=5000, atol=1e-12, btol=1e-12, conlim=1e8)
    sx, sistop, sitn, sr1, sr2, sanorm, sacond, sarnorm, sxnorm, _ = sp_lsqr(
        A, b, atol=1e-12, btol=1e-12, conlim=1e8, iter_lim=5000)
    assert res["istop"] == sistop == 2
    assert abs(res["itn"] - sitn) <= max(2, 0.02 * sitn)
    assert np.linalg.norm(x - sx) <= 1e-9 * np.linalg.norm(sx)
    # Scalars at a forced equal iteration count.  Two correct LSQR codes drift apart once
    # the dominant Ritz value has converged and Lanczos orthogonality is lost (here after
    # ~6 iterations: the relative gap in x grows ~10x per iteration, each run still
    # matching its own true residual; reading R16), so the tight comparison is
    # made on the first iterations and a loose one at convergence.
    for k in (1, 2, 3, 4):
        x2, r2 = oracle.lsqr(L, a, idx, b, itnlim=k)
        s = sp_lsqr(A, b, atol=0, btol=0, conlim=0, iter_lim=k)
        assert r2["istop"] == 7 and r2["itn"] == k == s[2]
        for mine, theirs in ((r2["r1norm"], s[3]), (r2["anorm"], s[5]), (r2["acond"], s[6]),
                             (r2["arnorm"], s[7]), (r2["xnorm"], s[8])):
            assert abs(mine - theirs) <= 1e-10 * abs(theirs)
        assert np.linalg.norm(x2 - s[0]) <= 1e-11 * np.linalg.norm(s[0])
    for mine, theirs in ((res["r1norm"], sr1), (res["anorm"], sanorm), (res["acond"], sacond),
                         (res["xnorm"], sxnorm)):
        assert abs(mine - theirs) <= 2e-2 * abs(theirs)
    # noise level: r2norm ~ sigma * sqrt(M - rank)
    rank = nonempty_columns(C1, idx).sum()
    pred = C1.sigma * np.sqrt(a.shape[0] - rank)
    assert abs(res["r2norm"] - pred) <= 0.02 * pred
    # solution is close to x_true on the non-empty columns and exactly 0 on the empty ones
    ne = nonempty_columns(C1, idx)
    assert np.all(x[~ne] == 0.0)
    assert np.linalg.norm(x[ne] - xt[ne]) <= 1e-5 * np.linalg.norm(xt[ne])


def test_lsqr_invariants_and_residual_identities():
    a, idx, L = _sys(C1)
    b = rhs(C1, a, idx, host.x_true(C1))
    x, res, rh, ah = oracle.lsqr(L, a, idx, b, itnlim=150, history=True)
    assert res["istop"] == 7 and res["itn"] == 150
    assert np.all(np.diff(rh) <= 1e-12 * rh[:-1])                  # ||r_k|| never increases
    r = b - oracle.aprod1(L, a, idx, x, np.zeros_like(b))
    assert abs(np.linalg.norm(r) - res["r1norm"]) <= 1e-8 * np.linalg.norm(r)
    atr = oracle.aprod2(L, a, idx, r, np.zeros_like(x))
    assert abs(np.linalg.norm(atr) - res["arnorm"]) <= 1e-4 * res["arnorm"] + 1e-9 * res["anorm"] * res["r1norm"]
    assert abs(res["bnorm"] - np.linalg.norm(b)) <= 1e-14 * np.linalg.norm(b)
    # early Lanczos vectors are orthogonal: one step gives x1 along v1 = A^T b / ||A^T b||
    x1, r1 = oracle.lsqr(L, a, idx, b, itnlim=1)
    v1 = oracle.aprod2(L, a, idx, b, np.zeros_like(x))
    cosang = (x1 @ v1) / (np.linalg.norm(x1) * np.linalg.norm(v1))
    assert abs(cosang - 1.0) <= 1e-12


def test_lsqr_closed_forms():
    shape = tiny_shape(n_stars=20, obs=30, n_knots=12, n_instr=10, seed=5)
    a, idx, L = _sys(shape)
    m = a.shape[0]
    # b = 0 -> x = 0, istop 0, no iterations
    x, res = oracle.lsqr(L, a, idx, np.zeros(m), itnlim=10)
    assert res["istop"] == 0 and res["itn"] == 0 and not x.any()
    # the paper's synthetic systems "converge to the identity solution": b = A 1 -> x = 1
    ne = nonempty_columns(shape, idx)
    ones = np.ones(shape.n_unknowns)
    b1 = rhs(shape, a, idx, ones, noisy=False)
    x, res = oracle.lsqr(L, a, idx, b1, itnlim=5000, atol=1e-14, btol=1e-14)
    assert res["istop"] in (1, 2)
    # A has a 3-dimensional null space per attitude axis pair/astro gauge at this size, so compare A x
    assert np.linalg.norm(rhs(shape, a, idx, x, noisy=False) - b1) <= 1e-10 * np.linalg.norm(b1)
    D = dense_matrix(shape, a, idx)
    xmin = np.linalg.lstsq(D, b1, rcond=None)[0]
    assert np.linalg.norm(x - xmin) <= 1e-9 * np.linalg.norm(xmin)
    if np.linalg.matrix_rank(D) == ne.sum():
        assert np.linalg.norm(x[ne] - 1.0) <= 1e-9 * np.sqrt(ne.sum())
    # noise-free consistent system: x -> x_true on a full-column-rank system
    xt = host.x_true(shape)
    b = rhs(shape, a, idx, xt, noisy=False)
    x, res = oracle.lsqr(L, a, idx, b, itnlim=5000, atol=1e-14, btol=1e-14)
    if np.linalg.matrix_rank(D) == ne.sum():
        assert np.linalg.norm(x[ne] - xt[ne]) <= 1e-9 * np.linalg.norm(xt[ne])
    # itnlim exit
    x, res = oracle.lsqr(L, a, idx, b, itnlim=3)
    assert res["istop"] == 7 and res["itn"] == 3


def test_lsqr_omp_matches_serial():
    """Different summation order (OpenMP partials): identical early, identical at convergence,
    free to drift in between (reading R16)."""
    a, idx, L = _sys(C1)
    b = rhs(C1, a, idx, host.x_true(C1))
    xs, rs = oracle.lsqr(L, a, idx, b, itnlim=3)
    xp, rp = oracle.lsqr(L, a, idx, b, itnlim=3, threads=4)
    assert np.linalg.norm(xs - xp) <= 1e-12 * np.linalg.norm(xs)
    assert abs(rs["r1norm"] - rp["r1norm"]) <= 1e-12 * rs["r1norm"]
    xs, rs = oracle.lsqr(L, a, idx, b, itnlim=5000, atol=1e-12, btol=1e-12, conlim=1e8)
    xp, rp = oracle.lsqr(L, a, idx, b, itnlim=5000, atol=1e-12, btol=1e-12, conlim=1e8, threads=4)
    assert rs["istop"] == rp["istop"] == 2
    assert np.linalg.norm(xs - xp) <= 1e-9 * np.linalg.norm(xs)
    # one step from a shared state agrees to rounding
    st1 = oracle.lsqr_init(L, a, idx, b)
    for _ in range(40):
        oracle.lsqr_step(L, a, idx, st1)
    import copy
    st2 = copy.deepcopy(st1)
    oracle.lsqr_step(L, a, idx, st1)
    oracle.lsqr_step(L, a, idx, st2, threads=4)
    for k in ("u", "v", "w", "x"):
        assert np.linalg.norm(getattr(st1, k) - getattr(st2, k)) <= 1e-12 * np.linalg.norm(getattr(st1, k))
    for k, v1 in st1.scalars().items():
        assert abs(v1 - st2.scalars()[k]) <= 1e-11 * abs(v1) + 1e-300


def test_lsqr_step_api_equals_driver():
    """init + step replay == orc_lsqr, and a step restarted from a copied state is identical."""
    a, idx, L = _sys(C1)
    b = rhs(C1, a, idx, host.x_true(C1))
    x, res = oracle.lsqr(L, a, idx, b, itnlim=25)
    st = oracle.lsqr_init(L, a, idx, b)
    assert st.itn == 0 and abs(st.bnorm - np.linalg.norm(b)) <= 1e-13 * st.bnorm and abs(np.linalg.norm(st.u) - 1) < 1e-14
    assert abs(np.linalg.norm(st.v) - 1) < 1e-14 and np.array_equal(st.v, st.w) and not st.x.any()
    for _ in range(25):
        oracle.lsqr_step(L, a, idx, st, itnlim=25)
    assert st.istop == 7 and st.itn == 25
    assert np.array_equal(st.x, x) and st.rnorm == res["r1norm"] and st.anorm == res["anorm"]
    assert st.acond == res["acond"] and st.xnorm == res["xnorm"] and st.arnorm == res["arnorm"]
    # Golub-Kahan relations hold for the stored vectors: ||u|| = ||v|| = 1
    assert abs(np.linalg.norm(st.u) - 1) < 1e-13 and abs(np.linalg.norm(st.v) - 1) < 1e-13


# ------------------------------------------------------------------ column norms, variances, preconditioning
def test_colnorms_match_dense_columns():
    """Column 2-norms against the dense brute-force matrix, entry by entry; empty columns give 0."""
    for n_glob in (1, 0):
        shape = tiny_shape(n_glob=n_glob, seed=4321 + n_glob)
        a, idx = host.make_rows(shape)
        idx[::4, 2:8] = np.array([1, 1, 3, 0, 5, 3], dtype=np.int32)      # repeated columns inside a row
        D = dense_matrix(shape, a, idx)
        got = oracle.colnorms(oracle.layout_of(shape), a, idx)
        # a repeated column inside one row: the dense matrix holds the SUM of the two coefficients, the
        # column norm of A as an operator; the oracle must agree with that, not with the sum of squares
        ref = np.linalg.norm(D, axis=0)
        dup_cols = shape.off_instr + np.array([1, 3])
        assert np.allclose(got, ref, rtol=1e-14, atol=0)
        sumsq = np.sqrt(np.sum(a[:, 17:23] ** 2 * (idx[:, 2:8] == 1), axis=0).sum())   # what a per-slot sum would give
        assert abs(sumsq - ref[dup_cols[0]]) > 1e-3 * ref[dup_cols[0]]                  # (the case does discriminate)
        assert np.all(got[ref == 0.0] == 0.0)


def test_scale_columns_is_right_multiplication_by_a_diagonal():
    shape = tiny_shape(seed=99)
    a, idx = host.make_rows(shape)
    L = oracle.layout_of(shape)
    s = 0.5 + host.test_vector(5, 1, shape.n_unknowns) ** 2
    D = dense_matrix(shape, a, idx)
    Ds = dense_matrix(shape, oracle.scale_columns(L, a, idx, s), idx)
    assert np.allclose(Ds, D * s[None, :], rtol=1e-15, atol=0)


def test_lsqr_var_matches_scipy_and_the_normal_matrix():
    """var of Paige-Saunders against scipy's independent implementation at a forced equal iteration count
    (early, where the two trajectories are still the same to rounding), and, on a tiny full-rank system run
    long, against the definition it estimates: diag((A^T A)^-1)."""
    import scipy.sparse.linalg as spl
    shape = tiny_shape(seed=777)
    a, idx = host.make_rows(shape)
    L = oracle.layout_of(shape)
    b = rhs(shape, a, idx, host.x_true(shape))
    A = csr_matrix(shape, a, idx)
    for k in (1, 5, 12):
        x, var, res = oracle.lsqr_var(L, a, idx, b, k)
        r = spl.lsqr(A, b, atol=0, btol=0, conlim=0, iter_lim=k, calc_var=True)
        assert res["itn"] == k and np.allclose(x, r[0], rtol=0, atol=1e-12 * np.abs(r[0]).max())
        assert np.allclose(var, r[9], rtol=1e-10, atol=1e-14 * r[9].max())
    # var_k = sum_{i<=k} (w_i / rho_i)^2 grows towards diag((A^T A)^-1) from below while the Lanczos vectors
    # stay orthogonal (k well below the rank; in floating point it overshoots later, a known property of
    # LSQR's estimate, so no equality is asserted)
    keep = nonempty_columns(shape, idx)
    D = dense_matrix(shape, a, idx)[:, keep]
    exact = np.diag(np.linalg.inv(D.T @ D))
    prev = np.zeros(shape.n_unknowns)
    for k in (3, 10, 30):
        x, var, res = oracle.lsqr_var(L, a, idx, b, k)
        assert np.all(var >= prev) and np.all(var[~keep] == 0.0)
        assert np.all(var[keep] <= exact * (1 + 1e-8))
        prev = var
    assert np.max(prev[keep] / exact) > 0.5                  # and it does get there


def test_preconditioned_lsqr_gives_the_same_least_squares_solution_in_fewer_iterations():
    shape = tiny_shape(n_stars=10, obs=15, seed=31)
    a, idx = host.make_rows(shape)
    a[:, 17:23] *= 40.0                                       # badly scaled instrumental columns
    L = oracle.layout_of(shape)
    b = rhs(shape, a, idx, host.x_true(shape))
    D = dense_matrix(shape, a, idx)
    xl = np.linalg.lstsq(D, b, rcond=None)[0]
    x0, r0 = oracle.lsqr(L, a, idx, b, 5000, 1e-14, 1e-14)
    x1, var1, r1, d = oracle.lsqr_precond(L, a, idx, b, 5000, 1e-14, 1e-14)
    assert np.linalg.norm(x1 - xl) <= 1e-10 * np.linalg.norm(xl)
    assert np.linalg.norm(x0 - xl) <= 1e-10 * np.linalg.norm(xl)
    assert r1["itn"] < r0["itn"] and r1["istop"] in (1, 2)
    # the scaled matrix has unit columns, and the variances come back in the units of x
    assert np.allclose(oracle.colnorms(L, oracle.scale_columns(L, a, idx, 1.0 / d), idx)[d != 1.0], 1.0, rtol=1e-14)
    keep = nonempty_columns(shape, idx)
    assert np.all(var1[~keep] == 0.0) and np.all(var1[keep] > 0.0)


def test_covariances_of_pairs():
    """Eq. (4), reading R21.  Pins: a pair (j, j) is var[j] (pinned against scipy above);
    swapping j1 and j2 changes nothing; |cov| <= sqrt(var var) (the estimate is a sum of outer products);
    and on a single-star, astro-only system (5 unknowns) five iterations span the whole space, so the sum of
    outer products IS (A^T A)^-1, entry by entry."""
    shape = tiny_shape(seed=2024)
    a, idx = host.make_rows(shape)
    L = oracle.layout_of(shape)
    b = rhs(shape, a, idx, host.x_true(shape))
    n = shape.n_unknowns
    rng = np.random.default_rng(7)
    j1 = np.concatenate([np.arange(n), rng.integers(0, n, 200)])
    j2 = np.concatenate([np.arange(n), rng.integers(0, n, 200)])
    x, cov, res = oracle.lsqr_cov(L, a, idx, b, j1, j2, 15)
    x2, var, res2 = oracle.lsqr_var(L, a, idx, b, 15)
    assert np.array_equal(x, x2) and np.allclose(cov[:n], var, rtol=1e-13, atol=0)
    _, cov_sw, _ = oracle.lsqr_cov(L, a, idx, b, j2, j1, 15)
    assert np.allclose(cov, cov_sw, rtol=1e-13, atol=1e-18)     # (factor * a) * b vs (factor * b) * a: rounding only
    assert np.all(np.abs(cov[n:]) <= np.sqrt(var[j1[n:]] * var[j2[n:]]) * (1 + 1e-12))
    # single star, astro only: a dense 5-column problem
    one = SystemShape("one", n_stars=1, obs_per_star=40, n_knots=8, n_instr=8, n_glob=1, seed=5)
    a1, idx1 = host.make_rows(one)
    a1[:, 5:] = 0.0
    L1 = oracle.layout_of(one)
    b1 = host.test_vector(3, 1, a1.shape[0])
    p1, p2 = np.meshgrid(np.arange(5), np.arange(5), indexing="ij")
    _, c5, r5 = oracle.lsqr_cov(L1, a1, idx1, b1, p1.ravel(), p2.ravel(), 5)
    A5 = a1[:, :5]
    exact = np.linalg.inv(A5.T @ A5)
    assert r5["itn"] == 5 and np.allclose(c5.reshape(5, 5), exact, rtol=1e-8, atol=1e-10 * np.abs(exact).max())


# ------------------------------------------------------------------ the 23-coefficient production record
def _sys23(shape):
    """A system with N_Glob = 0 in both storages: 24 doubles per row (slot 23 holds junk, which G = 0 must ignore)
    and the 184-byte production record with the first 23 of them."""
    assert shape.n_glob == 0
    a24, idx = host.make_rows(shape)
    a24[:, 23] = host.test_vector(shape.seed, 9, a24.shape[0])     # junk in the unused global slot
    a23 = np.ascontiguousarray(a24[:, :23])
    L24 = oracle.layout_of(shape)
    L23 = oracle.layout(shape.n_stars, shape.n_knots, shape.n_instr, 0, coeffs_per_row=23)
    return a24, a23, idx, L24, L23


def test_coeff23_record_is_the_dense_matrix_of_its_23_slots():
    """PAPER.md:141 (N_Glob = 0): the record without the global slot.  Pinned on the dense matrix built by the
    test-side column map from the 23 stored coefficients alone, entry by entry; and bit-identical to the 24-slot
    storage of the same system (same slots, same order, only the stride differs)."""
    shape = tiny_shape(n_stars=6, obs=9, n_knots=10, n_instr=7, n_glob=0, seed=2323)
    a24, a23, idx, L24, L23 = _sys23(shape)
    m, n = a23.shape[0], shape.n_unknowns
    cols = columns_of(shape, idx)
    assert np.all(cols[:, 23] == -1)
    D = np.zeros((m, n))
    for r in range(m):
        for k in range(23):
            D[r, cols[r, k]] += a23[r, k]
    x, y = host.test_vector(2, 1, n), host.test_vector(2, 2, m)
    y1 = oracle.aprod1(L23, a23, idx, x, np.zeros(m))
    x1 = oracle.aprod2(L23, a23, idx, y, np.zeros(n))
    np.testing.assert_allclose(y1, D @ x, rtol=0, atol=1e-13 * np.abs(D).dot(np.abs(x)).max())
    np.testing.assert_allclose(x1, D.T @ y, rtol=0, atol=1e-13 * np.abs(D.T).dot(np.abs(y)).max())
    for j in range(n):                                   # a wrong stride shifts every row after the first
        e = np.zeros(n)
        e[j] = 1.0
        np.testing.assert_allclose(oracle.aprod1(L23, a23, idx, e, np.zeros(m)), D[:, j], rtol=0, atol=1e-15)
    for r in (0, 1, m // 2, m - 1):
        e = np.zeros(m)
        e[r] = 1.0
        np.testing.assert_allclose(oracle.aprod2(L23, a23, idx, e, np.zeros(n)), D[r], rtol=0, atol=1e-15)
    assert np.array_equal(y1, oracle.aprod1(L24, a24, idx, x, np.zeros(m)))
    assert np.array_equal(x1, oracle.aprod2(L24, a24, idx, y, np.zeros(n)))
    assert np.array_equal(oracle.colnorms(L23, a23, idx), oracle.colnorms(L24, a24, idx))
    np.testing.assert_allclose(oracle.colnorms(L23, a23, idx), np.linalg.norm(D, axis=0), rtol=1e-14, atol=0)
    with pytest.raises(AssertionError):                  # the binding refuses a 24-wide array for a 23-wide layout
        oracle.aprod1(L23, a24, idx, x, np.zeros(m))


def test_coeff23_omp_compensated_and_lsqr():
    shape = tiny_shape(n_stars=40, obs=17, n_knots=16, n_instr=9, n_glob=0, seed=2324)
    a24, a23, idx, L24, L23 = _sys23(shape)
    m, n = a23.shape[0], shape.n_unknowns
    x, y = host.test_vector(3, 1, n), host.test_vector(3, 2, m)
    for th in (2, 3):                                    # chunk offsets of the OpenMP partitions use the stride too
        assert np.array_equal(oracle.aprod1(L23, a23, idx, x, np.zeros(m), threads=th),
                              oracle.aprod1(L23, a23, idx, x, np.zeros(m)))
        np.testing.assert_allclose(oracle.aprod2(L23, a23, idx, y, np.zeros(n), threads=th),
                                   oracle.aprod2(L23, a23, idx, y, np.zeros(n)), rtol=0, atol=1e-12)
    comp = np.zeros(n)
    xc = oracle.aprod2_comp(L23, a23, idx, y, np.zeros(n), comp)
    np.testing.assert_allclose(xc + comp, oracle.aprod2(L23, a23, idx, y, np.zeros(n)), rtol=0, atol=1e-12)
    assert np.array_equal(oracle.aprod1_abs(L23, a23, idx, x), oracle.aprod1_abs(L24, a24, idx, x))
    s = 0.5 + np.abs(host.test_vector(3, 3, n))
    assert np.array_equal(oracle.scale_columns(L23, a23, idx, s), oracle.scale_columns(L24, a24, idx, s)[:, :23])
    # LSQR: the same iteration bit for bit in both storages, and the dense least-squares solution
    b = rhs(shape, a24, idx, host.x_true(shape))
    x23, r23 = oracle.lsqr(L23, a23, idx, b, itnlim=2000, atol=1e-14, btol=1e-14)
    x24, r24 = oracle.lsqr(L24, a24, idx, b, itnlim=2000, atol=1e-14, btol=1e-14)
    assert np.array_equal(x23, x24) and r23 == r24 and r23["istop"] in (1, 2)
    D = dense_matrix(shape, a24, idx)
    xr = np.linalg.lstsq(D, b, rcond=None)[0]
    assert np.linalg.norm(x23 - xr) <= 1e-10 * np.linalg.norm(xr)


# ------------------------------------------------------------------ randomised small layouts (hypothesis)
def test_random_layouts_against_the_dense_matrix():
    """Any small layout, with or without the global parameter, in either storage, repeated instrumental columns and
    edge attitude starts included: aprod 1 / aprod 2 / column norms equal the dense matrix built by the test-side
    column map, and the adjoint identity holds to 1e-13."""
    hyp = pytest.importorskip("hypothesis")
    st = pytest.importorskip("hypothesis.strategies")

    @hyp.settings(max_examples=60, deadline=None, derandomize=True)
    @hyp.given(S=st.integers(1, 5), obs=st.integers(1, 7), K=st.integers(4, 9), I=st.integers(1, 8),
               G=st.integers(0, 1), cpr=st.sampled_from([24, 23]), seed=st.integers(0, 2 ** 20))
    def run(S, obs, K, I, G, cpr, seed):
        if cpr == 23:
            G = 0
        rng = np.random.default_rng(seed)
        m = S * obs
        shape = SystemShape("rnd", n_stars=S, obs_per_star=obs, n_knots=K, n_instr=I, n_glob=G, seed=seed)
        a = rng.standard_normal((m, 24))
        idx = np.empty((m, 8), dtype=np.int32)
        idx[:, 0] = np.repeat(np.arange(S), obs)
        idx[:, 1] = rng.integers(0, K - 3, size=m)                # 0 .. K-4 inclusive (the natural bound, R3)
        idx[:, 2:8] = rng.integers(0, I, size=(m, 6))             # with replacement: repeated columns
        D = dense_matrix(shape, a, idx)
        L = oracle.layout(S, K, I, G, coeffs_per_row=cpr)
        av = np.ascontiguousarray(a[:, :cpr])
        n = shape.n_unknowns
        x, y = rng.standard_normal(n), rng.standard_normal(m)
        ax = oracle.aprod1(L, av, idx, x, np.zeros(m))
        aty = oracle.aprod2(L, av, idx, y, np.zeros(n))
        np.testing.assert_allclose(ax, D @ x, rtol=0, atol=1e-13 * (np.abs(D) @ np.abs(x)).max() + 1e-300)
        np.testing.assert_allclose(aty, D.T @ y, rtol=0, atol=1e-13 * (np.abs(D.T) @ np.abs(y)).max() + 1e-300)
        assert abs(ax @ y - x @ aty) <= 1e-13 * np.linalg.norm(ax) * np.linalg.norm(y) + 1e-300
        np.testing.assert_allclose(oracle.colnorms(L, av, idx), np.linalg.norm(D, axis=0), rtol=1e-13, atol=1e-300)

    run()
