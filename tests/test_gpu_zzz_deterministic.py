"""The deterministic debug variant of aprod 2 (gsr_set_option("aprod2_variant", 2); SURVEY.md section 7 item 10;
csrc/aprod2_det.cu): every sum has one fixed order that depends on the sizes only.

* run to run the result is BIT-identical (the default kernels reduce with fp64 atomics and are reproducible to
  rounding only);
* with det_chunks = 1 the order is the CPU oracle's own (row by row, slot by slot, from x's initial value, no FMA
  contraction), so the result is bit-identical to oracle.aprod2 -- both record formats, repeated instrumental columns,
  a constraint section attached (the oracle then sees the one matrix [A_obs; A_con]); the 23-coefficient record:
  test_gpu_zzzz_coeff23.py;
* with any chunk count it meets the usual aprod 2 tolerance (reading R15);
* LSQR on the two-pass schedule with this aprod 2 follows the default solve (k = 5, reading R16).
(File name sorts last among the GPU tests.)"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
import paper_2503_22863_b200 as gsr  # noqa: E402
from gaia_synth import host  # noqa: E402
from gaia_synth.configs import C3, C5  # noqa: E402
from helpers import rhs, tiny_shape  # noqa: E402

DEV = "cuda"


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).to(DEV)


def aprod2_of(s, y, x0):
    x = dev(x0)
    s.aprod2(dev(y), x)
    return x.cpu().numpy()


def check_variant2(shape, L, a, idx, s, seed):
    m, n = a.shape[0], shape.n_unknowns
    assert s.n_rows == m and s.n_unknowns == n
    y, x0 = host.test_vector(seed, 3, m), host.test_vector(seed, 4, n)
    ref = oracle.aprod2(L, a, idx, y, x0.copy())
    s.set_option("aprod2_variant", 2)
    for chunks in (0, 7, 1):
        s.set_option("det_chunks", chunks)
        got = aprod2_of(s, y, x0)
        again = aprod2_of(s, y, x0)
        assert np.array_equal(got, again), f"det_chunks={chunks}: not bit-reproducible"
        assert np.linalg.norm(got - ref) <= 1e-11 * np.linalg.norm(ref)
        if chunks == 1:
            assert np.array_equal(got, ref), "det_chunks=1 must reproduce the oracle bit for bit"
    s.set_option("det_chunks", 0)
    s.set_option("aprod2_variant", 1)


@pytest.mark.parametrize("n_stars,obs", [(1, 1), (7, 37), (64, 64), (300, 1)])
def test_deterministic_aprod2(n_stars, obs):
    shape = tiny_shape(n_stars=n_stars, obs=obs, n_knots=40, n_instr=17, seed=900 + obs)
    a, idx = host.make_rows(shape)
    idx[::3, 2:8] = np.array([1, 1, 3, 0, 5, 3], dtype=np.int32)          # repeated columns inside a row
    with gsr.gsr_create(shape.n_stars, shape.n_knots, shape.n_instr, shape.n_glob, dev(a), dev(idx)) as s:
        check_variant2(shape, oracle.layout_of(shape), a, idx, s, seed=51)


def test_deterministic_aprod2_skewed_stars_and_sections():
    shape = C3.scaled(600)                                                 # power-law rows per star, hot knots
    a, idx = host.make_rows(shape)
    with gsr.gsr_create(shape.n_stars, shape.n_knots, shape.n_instr, shape.n_glob, dev(a), dev(idx)) as s:
        check_variant2(shape, oracle.layout_of(shape), a, idx, s, seed=52)
    # with the constraint rows as a section of their own (the oracle sees the one matrix [A_obs; A_con])
    shape = C5.scaled(40, n_knots=60, n_instr=30, n_constraint_rows=14, name="C5-tiny")
    a, idx = host.make_rows(shape)
    m_obs = shape.n_stars * shape.obs_per_star
    av, iv = dev(a), dev(idx)
    with gsr.gsr_create(shape.n_stars, shape.n_knots, shape.n_instr, shape.n_glob, av[:m_obs], iv[:m_obs]) as s:
        s.attach_constraints(av[m_obs:], iv[m_obs:])
        check_variant2(shape, oracle.layout_of(shape), a, idx, s, seed=53)


def test_lsqr_two_pass_with_deterministic_aprod2():
    shape = tiny_shape(n_stars=40, obs=30, n_knots=24, n_instr=12, seed=77)
    a, idx = host.make_rows(shape)
    b = dev(rhs(shape, a, idx, host.x_true(shape)))
    with gsr.gsr_create(shape.n_stars, shape.n_knots, shape.n_instr, shape.n_glob, dev(a), dev(idx)) as s:
        x1 = torch.empty(shape.n_unknowns, dtype=torch.float64, device=DEV)
        x2 = torch.empty_like(x1)
        r1 = s.lsqr(b, x1, 5)
        s.set_option("fused", 0)
        s.set_option("aprod2_variant", 2)
        r2 = s.lsqr(b, x2, 5)
        assert r1.itn == r2.itn == 5
        assert float(torch.linalg.norm(x1 - x2)) <= 1e-9 * float(torch.linalg.norm(x1))
        xr, rr = oracle.lsqr(oracle.layout_of(shape), a, idx, b.cpu().numpy(), itnlim=5)
        assert np.linalg.norm(x2.cpu().numpy() - xr) <= 1e-9 * np.linalg.norm(xr)
        with pytest.raises(gsr.GsrError) as ei:
            s.set_option("det_chunks", -1)
        assert ei.value.code == -1
