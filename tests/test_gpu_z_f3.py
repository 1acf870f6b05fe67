"""GPU parity for SURVEY.md section 8(f3): the constraint equations as a section of their own (gsr_attach_constraints,
PAPER.md:41, 72), against the CPU oracle on the same seeded inputs (the 23-coefficient record: test_gpu_zzzz_coeff23.py).  The oracle sees ONE matrix [A_obs; A_con] (that is the
definition of "a section appended after the observation rows") in the storage under test.

Tolerances as everywhere (readings R14, R15, R16): aprod 1 per row 1e-13 of the forward bound, aprod 2
normwise 1e-11 overall and per block, LSQR x <= 1e-9 at equal early iteration counts and at convergence, one-step
replays 1e-11 / 1e-10.  (File name sorts last among the GPU tests.)
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
import paper_2503_22863_b200 as gsr  # noqa: E402
from gaia_synth import host  # noqa: E402
from gaia_synth.configs import C5  # noqa: E402
from gpu_helpers import replay_one_step  # noqa: E402
from helpers import rhs, tiny_shape  # noqa: E402

DEV = "cuda"


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).to(DEV)


def blocks_of(shape):
    return {"astro": slice(0, shape.off_att), "att": slice(shape.off_att, shape.off_instr),
            "instr": slice(shape.off_instr, shape.off_glob), "glob": slice(shape.off_glob, shape.n_unknowns)}


def check_products(shape, L, a, idx, s, seed):
    """aprod 1 (on a non-zero y) and aprod 2 (on a non-zero x) of system s against the oracle with layout L."""
    m, n = a.shape[0], shape.n_unknowns
    assert s.n_rows == m and s.n_unknowns == n
    x, y0 = host.test_vector(seed, 1, n), host.test_vector(seed, 2, m)
    ref = oracle.aprod1(L, a, idx, x, y0.copy())
    bound = oracle.aprod1_abs(L, a, idx, x, y0)
    yg = dev(y0)
    s.aprod1(dev(x), yg)
    err = np.abs(yg.cpu().numpy() - ref)
    assert np.all(err <= 1e-13 * bound), f"aprod1: {np.max(err / np.maximum(bound, 1e-300)):.3e}"
    y, x0 = host.test_vector(seed, 3, m), host.test_vector(seed, 4, n)
    ref2 = oracle.aprod2(L, a, idx, y, x0.copy())
    xg = dev(x0)
    s.aprod2(dev(y), xg)
    got = xg.cpu().numpy()
    assert np.linalg.norm(got - ref2) <= 1e-11 * np.linalg.norm(ref2)
    inc = ref2 - x0
    for name, b in blocks_of(shape).items():
        if b.stop > b.start and np.linalg.norm(inc[b]) > 0:
            e = np.linalg.norm(got[b] - ref2[b])
            assert e <= 1e-11 * np.linalg.norm(ref2[b]), f"aprod2 block {name}: {e / np.linalg.norm(ref2[b]):.3e}"


def check_colnorms(L, a, idx, s):
    ref = oracle.colnorms(L, a, idx)
    got = s.colnorms(torch.empty(s.n_unknowns, dtype=torch.float64, device=DEV)).cpu().numpy()
    assert np.all(got[ref == 0.0] == 0.0)
    nz = ref > 0
    assert np.max(np.abs(got[nz] - ref[nz]) / ref[nz]) <= 1e-12


def check_lsqr(shape, L, a, idx, s, early=(1, 2, 3, 5), with_replay=True):
    n = shape.n_unknowns
    b = rhs(shape, a if a.shape[1] == 24 else np.hstack([a, np.zeros((a.shape[0], 1))]), idx, host.x_true(shape))
    bd = dev(b)
    x = torch.empty(n, dtype=torch.float64, device=DEV)
    for k in early:                                             # literal equality while it is well-posed (R16 (i))
        xr, rr = oracle.lsqr(L, a, idx, b, itnlim=k)
        res = s.lsqr(bd, x, k)
        assert res.itn == k == rr["itn"]
        assert np.linalg.norm(x.cpu().numpy() - xr) <= 1e-9 * np.linalg.norm(xr)
    xr, rr = oracle.lsqr(L, a, idx, b, itnlim=5000, atol=1e-12, btol=1e-12, conlim=1e8)
    res = s.lsqr(bd, x, 5000, 1e-12, 1e-12, 1e8)               # at convergence (R16 (ii))
    assert res.istop == rr["istop"] and res.istop in (1, 2)
    assert abs(res.itn - rr["itn"]) <= max(3, 0.05 * rr["itn"])
    assert np.linalg.norm(x.cpu().numpy() - xr) <= 1e-9 * np.linalg.norm(xr)
    if with_replay and a.shape[1] == 24:                        # one-step replays (R16 (iii)); the helper's layout is the 24-slot one
        s.lsqr_init(bd)
        replay_one_step(shape, a, idx, s)
        s.lsqr_iterate(6)
        replay_one_step(shape, a, idx, s)


# ------------------------------------------------------------------ the constraint section
def constraint_system(n_glob):
    shape = C5.scaled(150, n_knots=200, n_instr=300, n_constraint_rows=46, n_glob=n_glob, name="C5-small")
    a, idx = host.make_rows(shape)
    m_obs = shape.n_stars * shape.obs_per_star
    assert a.shape[0] == m_obs + 46
    return shape, a, idx, m_obs


@pytest.mark.parametrize("n_glob", [1, 0])
def test_constraint_section_24(n_glob):
    """Observation rows through gsr_create, the 46 constraint rows attached as their own section: every product and
    the fused LSQR pass run over both sections and must equal the oracle on the one matrix [A_obs; A_con]."""
    shape, a, idx, m_obs = constraint_system(n_glob)
    L = oracle.layout_of(shape)
    av, iv = dev(a), dev(idx)
    with gsr.gsr_create(shape.n_stars, shape.n_knots, shape.n_instr, n_glob, av[:m_obs], iv[:m_obs]) as s:
        assert s.n_rows == m_obs
        s.attach_constraints(av[m_obs:], iv[m_obs:])
        assert s.n_rows == a.shape[0]
        check_products(shape, L, a, idx, s, seed=41)
        check_colnorms(L, a, idx, s)
        check_lsqr(shape, L, a, idx, s)
        # the two-pass schedule over two sections gives the same solve
        b = dev(rhs(shape, a, idx, host.x_true(shape)))
        x1 = torch.empty(shape.n_unknowns, dtype=torch.float64, device=DEV)
        x2 = torch.empty_like(x1)
        r1 = s.lsqr(b, x1, 5)                 # (5 iterations: later the two roundings drift apart chaotically, R16)
        s.set_option("fused", 0)
        r2 = s.lsqr(b, x2, 5)
        s.set_option("fused", 1)
        assert r1.itn == r2.itn == 5
        assert float(torch.linalg.norm(x1 - x2)) <= 1e-9 * float(torch.linalg.norm(x1))
        # detaching restores the observation rows alone
        s.attach_constraints(None, None)
        assert s.n_rows == m_obs
        check_products(shape, L, a[:m_obs], idx[:m_obs], s, seed=42)
