"""GPU parity for SURVEY.md section 8(f1): column norms, Paige-Saunders variances and the column-norm
preconditioned solve (gsr_colnorms, gsr_lsqr_ex), against the CPU oracle on the same seeded inputs.

Tolerances: column norms 1e-12 relative per column (sums of <= a few thousand non-negative terms, fp64
atomics in any order); x as for plain LSQR (R16: <= 1e-9 for the first iterations and at
convergence); var <= 1e-9 relative (normwise) where the trajectories coincide (first iterations), and
<= 1e-6 at convergence, where it has accumulated a few hundred iterations of a drifting trajectory.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
import paper_2503_22863_b200 as gsr  # noqa: E402
from gaia_synth import host  # noqa: E402
from gaia_synth.configs import C1, C5  # noqa: E402
from helpers import rhs, tiny_shape  # noqa: E402

DEV = "cuda"


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).to(DEV)


def make(shape, a, idx):
    return gsr.gsr_create(shape.n_stars, shape.n_knots, shape.n_instr, shape.n_glob, dev(a), dev(idx))


def badly_scaled(shape, seed_scale=3):
    a, idx = host.make_rows(shape)
    a[:, 17:23] *= 40.0          # instrumental columns 40x, global 0.05x: what a column scaling is for
    a[:, 23] *= 0.05
    return a, idx


@pytest.mark.parametrize("shape", [tiny_shape(n_stars=9, obs=33, n_knots=12, n_instr=7, n_glob=0, seed=5),
                                   C1, C5.scaled(200, n_knots=300, n_instr=700, n_constraint_rows=40)],
                         ids=["tiny-noglob", "C1", "C5-small"])
def test_colnorms(shape):
    a, idx = badly_scaled(shape)
    # repeated instrumental columns inside a row (two pairs, and a triple): ||A e_j||_2 sums them before squaring
    idx[::4, 2:8] = np.array([1, 1, 3, 0, 5, 3], dtype=np.int32)
    idx[1::8, 2:8] = np.array([2, 4, 2, 6, 2, 0], dtype=np.int32)
    ref = oracle.colnorms(oracle.layout_of(shape), a, idx)
    with make(shape, a, idx) as s:
        out = torch.empty(s.n_unknowns, dtype=torch.float64, device=DEV)
        got = s.colnorms(out).cpu().numpy()
    assert np.all(got[ref == 0.0] == 0.0)
    nz = ref > 0
    assert np.max(np.abs(got[nz] - ref[nz]) / ref[nz]) <= 1e-12


def test_variances_plain_lsqr():
    shape = C1
    a, idx = host.make_rows(shape)
    L = oracle.layout_of(shape)
    b = rhs(shape, a, idx, host.x_true(shape))
    with make(shape, a, idx) as s:
        x = torch.empty(s.n_unknowns, dtype=torch.float64, device=DEV)
        var = torch.empty_like(x)
        for k in (1, 3, 5):
            res = s.lsqr_ex(dev(b), x, var=var, itnlim=k)
            xo, vo, ro = oracle.lsqr_var(L, a, idx, b, k)
            assert res.itn == k == ro["itn"]
            assert np.linalg.norm(x.cpu().numpy() - xo) <= 1e-9 * np.linalg.norm(xo)
            assert np.linalg.norm(var.cpu().numpy() - vo) <= 1e-9 * np.linalg.norm(vo)
        res = s.lsqr_ex(dev(b), x, var=var, itnlim=5000, atol=1e-12, btol=1e-12, conlim=1e8)
        xo, vo, ro = oracle.lsqr_var(L, a, idx, b, 5000, 1e-12, 1e-12, 1e8)
        assert res.istop == ro["istop"] and abs(res.itn - ro["itn"]) <= max(3, 0.05 * ro["itn"])
        assert np.linalg.norm(x.cpu().numpy() - xo) <= 1e-9 * np.linalg.norm(xo)
        vg = var.cpu().numpy()
        # the iteration counts may differ by a few at the stopping threshold: each extra iteration adds a term
        assert np.linalg.norm(vg - vo) <= 2e-2 * np.linalg.norm(vo) and np.all(vg >= 0)
        # asking for var does not change x (same run without it; atomics reorder sums, hence a tolerance)
        x2 = torch.empty_like(x)
        s.lsqr_ex(dev(b), x2, itnlim=3)
        s.lsqr_ex(dev(b), x, var=var, itnlim=3)
        assert np.linalg.norm((x2 - x).cpu().numpy()) <= 1e-10 * float(torch.linalg.norm(x))


@pytest.mark.parametrize("shape", [C1, C5.scaled(300, n_knots=400, n_instr=30, n_constraint_rows=60)], ids=["C1", "C5-small"])
def test_preconditioned_solve(shape):
    a, idx = badly_scaled(shape)
    L = oracle.layout_of(shape)
    b = rhs(shape, a, idx, host.x_true(shape))
    with make(shape, a, idx) as s:
        x = torch.empty(s.n_unknowns, dtype=torch.float64, device=DEV)
        var = torch.empty_like(x)
        for k in (1, 4):
            res = s.lsqr_ex(dev(b), x, var=var, precond=True, itnlim=k)
            xo, vo, ro, d = oracle.lsqr_precond(L, a, idx, b, k)
            assert res.itn == k
            assert np.linalg.norm(x.cpu().numpy() - xo) <= 1e-9 * np.linalg.norm(xo)
            assert np.linalg.norm(var.cpu().numpy() - vo) <= 1e-9 * np.linalg.norm(vo)
            for name in ("anorm", "acond", "arnorm", "xnorm"):      # norms of the scaled system
                assert abs(getattr(res, name) - ro[name]) <= 1e-9 * abs(ro[name])
            assert abs(res.r1norm - ro["rnorm"]) <= 1e-9 * ro["rnorm"]
        res = s.lsqr_ex(dev(b), x, var=var, precond=True, itnlim=5000, atol=1e-12, btol=1e-12, conlim=1e8)
        xo, vo, ro, d = oracle.lsqr_precond(L, a, idx, b, 5000, 1e-12, 1e-12, 1e8)
        assert res.istop == ro["istop"] and abs(res.itn - ro["itn"]) <= max(3, 0.05 * ro["itn"])
        assert np.linalg.norm(x.cpu().numpy() - xo) <= 1e-9 * np.linalg.norm(xo)
        # and it is worth it: fewer iterations than the plain solve of the same badly scaled system
        x0 = torch.empty_like(x)
        res0 = s.lsqr(dev(b), x0, 5000, 1e-12, 1e-12, 1e8)
        assert res.itn < res0.itn
        assert np.linalg.norm((x - x0).cpu().numpy()) <= 1e-7 * float(torch.linalg.norm(x0))
        # the two-pass schedule has no preconditioned operator
        s.set_option("fused", 0)
        with pytest.raises(Exception):
            s.lsqr_ex(dev(b), x, precond=True, itnlim=2)
        s.set_option("fused", 1)


def test_covariances_of_pairs():
    """SURVEY.md 8(f4), Eq. (4): pairs from every parameter block, plain and preconditioned."""
    shape = C5.scaled(120, n_knots=90, n_instr=25, n_constraint_rows=20)
    a, idx = badly_scaled(shape)
    L = oracle.layout_of(shape)
    b = rhs(shape, a, idx, host.x_true(shape))
    n = shape.n_unknowns
    rng = np.random.default_rng(11)
    j1 = np.concatenate([np.arange(n), rng.integers(0, n, 3000), rng.integers(shape.off_att, n, 3000)])
    j2 = np.concatenate([np.arange(n), rng.integers(0, n, 3000), rng.integers(shape.off_att, n, 3000)])
    with make(shape, a, idx) as s:
        x = torch.empty(n, dtype=torch.float64, device=DEV)
        var = torch.empty_like(x)
        cov = torch.full((j1.size,), 7.0, dtype=torch.float64, device=DEV)        # must be zeroed by the run
        s.set_cov_pairs(dev(j1), dev(j2), cov)
        for k in (1, 4):
            s.lsqr_ex(dev(b), x, var=var, itnlim=k)
            xo, co, ro = oracle.lsqr_cov(L, a, idx, b, j1, j2, k)
            cg = cov.cpu().numpy()
            assert np.linalg.norm(cg - co) <= 1e-9 * np.linalg.norm(co)
            assert np.linalg.norm(cg[:n] - var.cpu().numpy()) <= 1e-12 * np.linalg.norm(cg[:n])   # pair (j, j) = var[j]
            # preconditioned: the oracle on the scaled matrix, brought back to the units of x
            s.lsqr_ex(dev(b), x, precond=True, itnlim=k)
            d = oracle.colnorms(L, a, idx)
            d[d == 0.0] = 1.0
            zo, cz, rz = oracle.lsqr_cov(L, oracle.scale_columns(L, a, idx, 1.0 / d), idx, b, j1, j2, k)
            cp = cz / (d[j1] * d[j2])
            assert np.linalg.norm(cov.cpu().numpy() - cp) <= 1e-9 * np.linalg.norm(cp)
        # a plain gsr_lsqr leaves the registered accumulator alone; unregistering works; bad indices are refused
        before = cov.clone()
        s.lsqr(dev(b), x, 3)
        assert torch.equal(before, cov)
        bad = j2.copy()
        bad[5] = n
        with pytest.raises(Exception):
            s.set_cov_pairs(dev(j1), dev(bad), cov)
        s.set_cov_pairs(None, None, None)
        s.lsqr_ex(dev(b), x, itnlim=2)
        assert torch.equal(before, cov)
