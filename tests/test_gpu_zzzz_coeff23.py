"""GPU parity for SURVEY.md section 8(f3): the 23-coefficient production record (GSR_LAYOUT_COEFF23, N_Glob = 0,
PAPER.md:141) through the tile kernels' Rec23 instances (tensor view of 4-row groups), against
the CPU oracle on the same seeded inputs -- products and column norms on row counts around the tile and the group,
LSQR plain and preconditioned against the oracle and against the 24-slot storage of the same system, the constraint
section in this storage, the deterministic aprod 2 variant on it.

Tolerances as everywhere (readings R14, R15, R16).  The file name sorts LAST among the GPU tests: these
kernels use a tensor-map shape that has not run on hardware yet (box 100 x 8 over a 92-column view), and a fault here
must not take other tests with it.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
import paper_2503_22863_b200 as gsr  # noqa: E402
from gaia_synth import host  # noqa: E402
from gaia_synth.configs import C5  # noqa: E402
from helpers import rhs, tiny_shape  # noqa: E402
import test_gpu_z_f3 as F  # noqa: E402  (the checks shared with the constraint-section tests)
import test_gpu_zzz_deterministic as D  # noqa: E402

DEV = "cuda"


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).to(DEV)


check_products, check_colnorms, check_lsqr, constraint_system = F.check_products, F.check_colnorms, F.check_lsqr, F.constraint_system


# ------------------------------------------------------------------ the 23-coefficient record
@pytest.mark.parametrize("n_stars,obs", [(1, 1), (1, 2), (1, 3), (1, 33), (1, 34), (1, 35), (3, 10), (3, 11), (7, 37),
                                         (5, 129), (64, 64), (40, 100), (300, 1), (41, 5)])
def test_coeff23_products(n_stars, obs):
    """Row counts around the 32-row tile and the 4-row group of the 184-byte record's tensor view (M mod 4 = 0 ... 3,
    a last tile that holds nothing but the tail), stars with 1-5 rows (the non-matrix-product astrometric path)."""
    shape = tiny_shape(n_stars=n_stars, obs=obs, n_knots=12, n_instr=9, n_glob=0, seed=230 + n_stars)
    a24, idx = host.make_rows(shape)
    a23 = np.ascontiguousarray(a24[:, :23])
    L23 = oracle.layout(shape.n_stars, shape.n_knots, shape.n_instr, 0, coeffs_per_row=23)
    with gsr.gsr_create(shape.n_stars, shape.n_knots, shape.n_instr, 0, dev(a23), dev(idx), coeffs_per_row=23) as s:
        check_products(shape, L23, a23, idx, s, seed=31)
        check_colnorms(L23, a23, idx, s)
    # duplicates inside a row, and the record refused with a global parameter
    idx2 = idx.copy()
    idx2[::3, 2:8] = np.array([1, 1, 3, 0, 5, 3], dtype=np.int32)
    with gsr.gsr_create(shape.n_stars, shape.n_knots, shape.n_instr, 0, dev(a23), dev(idx2), coeffs_per_row=23) as s:
        check_products(shape, L23, a23, idx2, s, seed=32)
        check_colnorms(L23, a23, idx2, s)
    with pytest.raises(gsr.GsrError) as ei:
        gsr.gsr_create(shape.n_stars, shape.n_knots, shape.n_instr, 1, dev(a23), dev(idx), coeffs_per_row=23)
    assert ei.value.code == -1


def test_coeff23_lsqr():
    shape = tiny_shape(n_stars=60, obs=25, n_knots=40, n_instr=12, n_glob=0, seed=2325)
    a24, idx = host.make_rows(shape)
    a23 = np.ascontiguousarray(a24[:, :23])
    L23 = oracle.layout(shape.n_stars, shape.n_knots, shape.n_instr, 0, coeffs_per_row=23)
    with gsr.gsr_create(shape.n_stars, shape.n_knots, shape.n_instr, 0, dev(a23), dev(idx), coeffs_per_row=23) as s:
        check_lsqr(shape, L23, a23, idx, s)
        # the same solve in the 24-slot storage of the same system gives the same solution
        x23 = torch.empty(shape.n_unknowns, dtype=torch.float64, device=DEV)
        b = dev(rhs(shape, a24, idx, host.x_true(shape)))
        s.lsqr(b, x23, 5000, 1e-12, 1e-12, 1e8)
        with gsr.gsr_create(shape.n_stars, shape.n_knots, shape.n_instr, 0, dev(a24), dev(idx)) as s24:
            x24 = torch.empty_like(x23)
            s24.lsqr(b, x24, 5000, 1e-12, 1e-12, 1e8)
            assert float(torch.linalg.norm(x23 - x24)) <= 1e-9 * float(torch.linalg.norm(x24))
            # column-norm preconditioning and variances run through the same fused pass in either storage
            xp23, xp24 = torch.empty_like(x23), torch.empty_like(x23)
            v23, v24 = torch.empty_like(x23), torch.empty_like(x23)
            r23 = s.lsqr_ex(b, xp23, var=v23, precond=True, itnlim=5000, atol=1e-12, btol=1e-12, conlim=1e8)
            r24 = s24.lsqr_ex(b, xp24, var=v24, precond=True, itnlim=5000, atol=1e-12, btol=1e-12, conlim=1e8)
            assert r23.istop == r24.istop and abs(r23.itn - r24.itn) <= max(3, 0.05 * r24.itn)
            assert float(torch.linalg.norm(xp23 - xp24)) <= 1e-9 * float(torch.linalg.norm(xp24))
        xo, _, ro, _ = oracle.lsqr_precond(L23, a23, idx, b.cpu().numpy(), itnlim=5000, atol=1e-12, btol=1e-12, conlim=1e8)
        assert r23.istop == ro["istop"]
        assert np.linalg.norm(xp23.cpu().numpy() - xo) <= 1e-9 * np.linalg.norm(xo)
        # the two-pass schedule and the one-thread-per-row kernels remain as cross-checks
        xv0, xv1 = torch.empty_like(x23), torch.empty_like(x23)
        for name in ("fused", "aprod1_variant", "aprod2_variant"):
            s.set_option(name, 0)
        s.lsqr(b, xv0, 5)
        for name in ("fused", "aprod1_variant", "aprod2_variant"):
            s.set_option(name, 1)
        s.lsqr(b, xv1, 5)
        assert float(torch.linalg.norm(xv0 - xv1)) <= 1e-9 * float(torch.linalg.norm(xv1))



def test_constraint_section_coeff23():
    shape, a, idx, m_obs = constraint_system(0)
    a23 = np.ascontiguousarray(a[:, :23])
    L23 = oracle.layout(shape.n_stars, shape.n_knots, shape.n_instr, 0, coeffs_per_row=23)
    av, iv = dev(a23), dev(idx)
    with gsr.gsr_create(shape.n_stars, shape.n_knots, shape.n_instr, 0, av[:m_obs], iv[:m_obs], coeffs_per_row=23) as s:
        s.attach_constraints(av[m_obs:], iv[m_obs:])
        assert s.n_rows == a.shape[0]
        check_products(shape, L23, a23, idx, s, seed=43)
        check_colnorms(L23, a23, idx, s)
        check_lsqr(shape, L23, a23, idx, s, early=(1, 3))


def test_deterministic_aprod2_coeff23_with_constraint_section():
    shape = C5.scaled(40, n_knots=60, n_instr=30, n_constraint_rows=14, n_glob=0, name="C5-tiny")
    a24, idx = host.make_rows(shape)
    a23 = np.ascontiguousarray(a24[:, :23])
    m_obs = shape.n_stars * shape.obs_per_star
    L23 = oracle.layout(shape.n_stars, shape.n_knots, shape.n_instr, 0, coeffs_per_row=23)
    av, iv = dev(a23), dev(idx)
    with gsr.gsr_create(shape.n_stars, shape.n_knots, shape.n_instr, 0, av[:m_obs], iv[:m_obs], coeffs_per_row=23) as s:
        s.attach_constraints(av[m_obs:], iv[m_obs:])
        D.check_variant2(shape, L23, a23, idx, s, seed=53)
