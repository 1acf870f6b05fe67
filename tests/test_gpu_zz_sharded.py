"""GPU parity for SURVEY.md section 8(f2): the row-sharded solve through the library's phase calls (gsr_shard_begin /
gsr_shard_phase / gsr_shard_poll) and the driver loop of paper_2503_22863_b200/sharded.py, with ALL shards driven by
this one process on one GPU (LocalComm: the sum over ranks is a tensor sum; no rank waits on another one's kernels).
Each shard is its own gsr_system over its range of rows with the global sizes; the constraint rows are attached to
shard 0 as a section of their own.  Compared with the CPU oracle's LSQR on the WHOLE system -- literally for the
first iterations, at convergence with the real tolerances (reading R16) -- and with the unsharded gsr_lsqr.
The host logic alone, under gloo with two processes: tests/test_sharded_cpu.py.  (File name sorts last.)"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

import oracle  # noqa: E402
import paper_2503_22863_b200 as gsr  # noqa: E402
from gaia_synth import host  # noqa: E402
from gaia_synth.configs import C5  # noqa: E402
from helpers import rhs  # noqa: E402
from paper_2503_22863_b200.sharded import LocalComm, ShardedLsqr, partition_stars  # noqa: E402

DEV = "cuda"


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).to(DEV)


def make_shards(shape, a, idx, b, world, n_con):
    """One gsr_system per rank over its star-aligned range of observation rows; rank 0 also gets the constraint
    section.  Returns (systems, right-hand sides, partition)."""
    m_obs = a.shape[0] - n_con
    parts = partition_stars(host.obs_counts(shape), world)
    systems, bs = [], []
    for k, p in enumerate(parts):
        av, iv = dev(a[p.row_lo:p.row_hi]), dev(idx[p.row_lo:p.row_hi])
        s = gsr.gsr_create(shape.n_stars, shape.n_knots, shape.n_instr, shape.n_glob, av, iv)
        bk = b[p.row_lo:p.row_hi]
        if k == 0 and n_con:
            s.attach_constraints(dev(a[m_obs:]), dev(idx[m_obs:]))
            bk = np.concatenate([bk, b[m_obs:]])
        assert s.n_unknowns == shape.n_unknowns and s.n_rows == len(bk)
        systems.append(s)
        bs.append(dev(bk))
    return systems, bs, parts


def solve_sharded(shape, systems, bs, itnlim, atol=0.0, btol=0.0, conlim=0.0, check_every=16):
    drv = ShardedLsqr(systems, LocalComm(len(systems)), check_every=check_every)
    res = drv.solve(bs, itnlim, atol, btol, conlim)
    xs = drv.solution([torch.zeros(shape.n_unknowns, dtype=torch.float64, device=DEV) for _ in systems])
    for x in xs[1:]:
        assert torch.equal(x, xs[0])
    return res, xs[0].cpu().numpy(), drv


@pytest.mark.parametrize("world,n_instr", [(1, 300), (2, 300), (3, 300), (2, 60_000)])
def test_sharded_lsqr_against_oracle(world, n_instr):
    # n_instr = 60,000: the accumulators live in the die-local L2 copies, as at C4.  With 12,046 rows that block is
    # five times under-determined and the trajectory amplifies rounding a few hundred times per iteration (4e-15 at
    # k = 1, 3e-13 at k = 3, 2e-9 at k = 5, oracle against itself in another summation order): reading R16 allows the
    # literal comparison only while it is well-posed, so that case stops at k = 3 and has no run to convergence.
    well_posed = n_instr <= 1000
    shape = C5.scaled(150, n_knots=200, n_instr=n_instr, n_constraint_rows=46, name="C5-small")
    a, idx = host.make_rows(shape)
    b = rhs(shape, a, idx, host.x_true(shape))
    L = oracle.layout_of(shape)
    systems, bs, parts = make_shards(shape, a, idx, b, world, 46)
    try:
        ns = shape.n_unknowns - shape.off_att
        for k in ((0, 1, 3, 5) if well_posed else (0, 1, 2, 3)):   # literal equality while it is well-posed (R16 (i))
            xr, rr = oracle.lsqr(L, a, idx, b, itnlim=k)
            res, x, drv = solve_sharded(shape, systems, bs, k)
            assert res.itn == k == rr["itn"] and res.istop == 7
            assert np.linalg.norm(x - xr) <= 1e-9 * max(np.linalg.norm(xr), 1e-300)
            for key in ("anorm", "acond", "xnorm", "bnorm", "r1norm"):
                assert abs(getattr(res, key) - rr[key]) <= 1e-9 * abs(rr[key]), key
            assert drv.exchanges == 3 + 2 * k and drv.exchanged_doubles == (ns + 2) + k * (ns + 3)
        if well_posed:
            xr, rr = oracle.lsqr(L, a, idx, b, itnlim=5000, atol=1e-12, btol=1e-12, conlim=1e8)
            res, x, _ = solve_sharded(shape, systems, bs, 5000, 1e-12, 1e-12, 1e8, check_every=7)   # at convergence (R16 (ii))
            assert res.istop == rr["istop"] and res.istop in (1, 2)
            assert abs(res.itn - rr["itn"]) <= max(3, 0.05 * rr["itn"])
            assert np.linalg.norm(x - xr) <= 1e-9 * np.linalg.norm(xr)
        # the astrometric block is distributed: a rank's own x is zero outside its stars
        for s, p in zip(systems, parts):
            xo = torch.empty(shape.n_unknowns, dtype=torch.float64, device=DEV)
            own = s.lsqr_result(xo)
            xa = xo[:shape.off_att].cpu().numpy()
            mask = np.ones(shape.off_att, dtype=bool)
            mask[5 * p.star_lo:5 * p.star_hi] = False
            assert not xa[mask].any()
            assert own.itn == res.itn
    finally:
        for s in systems:
            s.destroy()


def test_sharded_equals_unsharded_and_state_rules():
    shape = C5.scaled(120, n_knots=160, n_instr=90, n_constraint_rows=0, name="C5-small")
    a, idx = host.make_rows(shape)
    b = rhs(shape, a, idx, host.x_true(shape))
    with gsr.gsr_create(shape.n_stars, shape.n_knots, shape.n_instr, shape.n_glob, dev(a), dev(idx)) as whole:
        x1 = torch.empty(shape.n_unknowns, dtype=torch.float64, device=DEV)
        r1 = whole.lsqr(dev(b), x1, 5)
        systems, bs, _ = make_shards(shape, a, idx, b, 2, 0)
        try:
            r2, x2, _ = solve_sharded(shape, systems, bs, 5)
            assert r1.itn == r2.itn == 5
            assert np.linalg.norm(x2 - x1.cpu().numpy()) <= 1e-9 * float(torch.linalg.norm(x1))
            for key in ("anorm", "acond", "xnorm", "bnorm", "r1norm"):
                assert abs(getattr(r2, key) - getattr(r1, key)) <= 1e-9 * abs(getattr(r1, key))
            # while a sharded solve is in progress the plain stepping call is refused; a plain init ends it
            s0 = systems[0]
            with pytest.raises(gsr.GsrError) as ei:
                s0.lsqr_iterate(1)
            assert ei.value.code == -5
            s0.lsqr_init(bs[0])
            s0.lsqr_iterate(1)
            with pytest.raises(gsr.GsrError) as ei:
                s0.shard_phase()
            assert ei.value.code == -5
            # the two-pass schedule has no phases
            s0.set_option("fused", 0)
            with pytest.raises(gsr.GsrError) as ei:
                s0.shard_begin(bs[0], s0.exchange_buffer(), True, 3)
            assert ei.value.code == -5
        finally:
            for s in systems:
                s.destroy()
