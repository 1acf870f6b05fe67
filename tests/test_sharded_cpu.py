"""Host logic of the row-sharded solve (paper_2503_22863_b200/sharded.py) without a GPU: the row
partition, the lock-step phase loop and the exchanges, with tests/shard_standin.py in the place of the library's
phase calls -- in one process (LocalComm, 3 shards) and under torch.distributed with gloo (world size 2).  The
sharded solution must equal the CPU oracle's LSQR on the WHOLE system: literally for the first iterations, and at
convergence (reading R16).  The same driver with the real kernels: tests/test_gpu_zz_sharded.py."""
import json
import os
import subprocess
import sys

import numpy as np
import pytest
import torch

import oracle
from gaia_synth import host
from gaia_synth.configs import C3, C5
from helpers import rhs, tiny_shape
from paper_2503_22863_b200.sharded import LocalComm, RowRange, ShardedLsqr, partition_stars
from shard_standin import OracleShard

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


# ------------------------------------------------------------------------------------------ the partition
def check_partition(parts, counts, world):
    ptr = np.concatenate([[0], np.cumsum(counts)])
    assert len(parts) == world
    assert parts[0].star_lo == 0 and parts[0].row_lo == 0
    assert parts[-1].star_hi == len(counts) and parts[-1].row_hi == ptr[-1]
    for p, q in zip(parts, parts[1:]):
        assert p.star_hi == q.star_lo and p.row_hi == q.row_lo            # contiguous, nothing lost or doubled
    for p in parts:
        assert p.star_lo <= p.star_hi
        assert p.row_lo == ptr[p.star_lo] and p.row_hi == ptr[p.star_hi]  # cut at star boundaries only


def test_partition_equal_stars():
    parts = partition_stars((1000, 20), 8)
    check_partition(parts, np.full(1000, 20), 8)
    assert all(p.row_hi - p.row_lo == 2500 for p in parts)
    assert partition_stars((7, 3), 1) == [RowRange(0, 7, 0, 21)]
    # a pair and an explicit array mean the same
    assert partition_stars((10, 4), 3) == partition_stars(np.full(10, 4), 3)


def test_partition_skewed_stars_is_balanced_to_one_star():
    shape = C3.scaled(5000)                                   # power-law observations per star (reading R11)
    counts = host.obs_counts(shape)
    m = int(counts.sum())
    for world in (2, 3, 8):
        parts = partition_stars(counts, world)
        check_partition(parts, counts, world)
        # every cut is the boundary nearest to its target: no range is off by more than one star's rows per end
        for p in parts:
            assert abs((p.row_hi - p.row_lo) - m / world) <= 2 * counts.max()


def test_partition_degenerate():
    parts = partition_stars(np.array([5, 0, 0, 7]), 3)        # stars without rows
    check_partition(parts, np.array([5, 0, 0, 7]), 3)
    parts = partition_stars((2, 10), 5)                       # more ranks than stars: some ranges are empty
    check_partition(parts, np.full(2, 10), 5)
    assert sum(p.row_hi > p.row_lo for p in parts) == 2
    parts = partition_stars(np.zeros(0, dtype=np.int64), 2)   # no stars at all
    assert all(p.row_lo == p.row_hi == 0 for p in parts)
    with pytest.raises(ValueError):
        partition_stars((4, 4), 0)
    with pytest.raises(ValueError):
        partition_stars(np.array([3, -1]), 2)


# ------------------------------------------------------------------------------------------ the solve
def shard_rows(shape, a, idx, b, parts, n_con):
    """Rows of every rank: its range of observation rows; rank 0 also holds the constraint rows (they come last in
    the whole system and carry star = S-1, so rank 0's rows stay sorted only if it also ends at S-1 -- the oracle
    stand-in does not care, the library takes them as a section of their own)."""
    m_obs = a.shape[0] - n_con
    out = []
    for k, p in enumerate(parts):
        sel = np.arange(p.row_lo, p.row_hi)
        if k == 0 and n_con:
            sel = np.concatenate([sel, np.arange(m_obs, m_obs + n_con)])
        out.append((a[sel], idx[sel], b[sel]))
    return out


def run_local(shape, a, idx, b, world, n_con, itnlim, atol=0.0, btol=0.0, conlim=0.0, check_every=16):
    parts = partition_stars(host.obs_counts(shape), world)
    rows = shard_rows(shape, a, idx, b, parts, n_con)
    shards = [OracleShard(shape, ak, ik) for ak, ik, _ in rows]
    drv = ShardedLsqr(shards, LocalComm(world), check_every=check_every)
    res = drv.solve([torch.from_numpy(bk.copy()) for _, _, bk in rows], itnlim, atol, btol, conlim)
    xs = drv.solution([torch.zeros(shape.n_unknowns, dtype=torch.float64) for _ in shards])
    for x in xs[1:]:
        assert torch.equal(x, xs[0])                          # every rank ends with the same whole x
    return res, xs[0].numpy(), drv, shards


@pytest.mark.parametrize("world", [1, 2, 3])
def test_sharded_solve_matches_oracle_on_whole_system(world):
    shape = C5.scaled(30, n_knots=24, n_instr=30, n_constraint_rows=10, name="C5-tiny")    # 30 x 80 rows + 10 constraints
    a, idx = host.make_rows(shape)
    b = rhs(shape, a, idx, host.x_true(shape))
    L = oracle.layout_of(shape)
    for k in (0, 1, 2, 3, 5):                                 # literal equality while the trajectory is well-posed
        xr, rr = oracle.lsqr(L, a, idx, b, itnlim=k)
        res, x, drv, _ = run_local(shape, a, idx, b, world, 10, itnlim=k)
        assert res.itn == k == rr["itn"] and res.istop == rr["istop"] == 7
        assert np.linalg.norm(x - xr) <= 1e-9 * max(np.linalg.norm(xr), 1e-300)
        for key in ("anorm", "acond", "xnorm", "bnorm", "r1norm", "arnorm"):      # the scalars at an equal iteration count
            assert abs(getattr(res, key) - rr[key]) <= 1e-9 * abs(rr[key]), key
        ns = shape.n_unknowns - shape.off_att
        # per iteration ONE vector exchange (the replicated tail + 2 scalars) and one scalar; the init: 2 scalars + the tail
        assert drv.exchanges == 3 + 2 * k
        assert drv.exchanged_doubles == (1 + ns + 1) + k * (ns + 2 + 1)
    xr, rr = oracle.lsqr(L, a, idx, b, itnlim=4000, atol=1e-12, btol=1e-12, conlim=1e8)
    res, x, drv, shards = run_local(shape, a, idx, b, world, 10, itnlim=4000, atol=1e-12, btol=1e-12, conlim=1e8,
                                    check_every=7)
    assert res.istop == rr["istop"] and res.istop in (1, 2)
    assert abs(res.itn - rr["itn"]) <= max(3, 0.05 * rr["itn"])
    assert np.linalg.norm(x - xr) <= 1e-9 * np.linalg.norm(xr)
    # the astrometric block is distributed: a rank's own x is zero outside its stars
    parts = partition_stars(host.obs_counts(shape), world)
    for sh, p in zip(shards, parts):
        own = np.zeros(shape.off_att, dtype=bool)
        own[5 * p.star_lo:5 * p.star_hi] = True
        assert not sh.x[:shape.off_att][~own].any()


def test_sharded_trivial_right_hand_sides():
    shape = tiny_shape(n_stars=6, obs=9, n_knots=8, n_instr=7)
    a, idx = host.make_rows(shape)
    res, x, _, _ = run_local(shape, a, idx, np.zeros(a.shape[0]), 2, 0, itnlim=50, atol=1e-12, btol=1e-12)
    assert res.istop == 0 and res.itn == 0 and not x.any()    # b = 0: x = 0 is exact
    b = rhs(shape, a, idx, host.x_true(shape), noisy=False)
    res, x, _, _ = run_local(shape, a, idx, b, 4, 0, itnlim=0)
    assert res.istop == 7 and res.itn == 0 and not x.any()    # no iteration allowed
    # more ranks than stars: empty shards take part in every exchange
    xr, rr = oracle.lsqr(oracle.layout_of(shape), a, idx, b, itnlim=3)
    res, x, _, _ = run_local(shape, a, idx, b, 8, 0, itnlim=3)
    assert res.itn == 3 and np.linalg.norm(x - xr) <= 1e-9 * np.linalg.norm(xr)


WORKER = r'''
import json, os, sys
sys.path.insert(0, {root!r}); sys.path.insert(0, os.path.join({root!r}, "tests"))
import numpy as np, torch, torch.distributed as dist
from gaia_synth import host
from gaia_synth.configs import C5
from helpers import rhs
from paper_2503_22863_b200.sharded import DistComm, ShardedLsqr, partition_stars
from shard_standin import OracleShard
dist.init_process_group("gloo")
comm = DistComm()
assert comm.world == 2 and comm.n_local == 1
shape = C5.scaled(24, n_knots=20, n_instr=25, n_constraint_rows=8, name="C5-tiny")
a, idx = host.make_rows(shape)                      # (every rank could generate its own range; the whole thing is tiny)
b = rhs(shape, a, idx, host.x_true(shape))
m_obs = a.shape[0] - 8
p = partition_stars(host.obs_counts(shape), comm.world)[comm.rank]
sel = np.arange(p.row_lo, p.row_hi)
if comm.rank == 0:
    sel = np.concatenate([sel, np.arange(m_obs, m_obs + 8)])       # the constraint section lives on one rank
drv = ShardedLsqr([OracleShard(shape, a[sel], idx[sel])], comm, check_every=5)
out = {{}}
for itnlim, tol in ((3, 0.0), (4000, 1e-12)):
    res = drv.solve([torch.from_numpy(b[sel].copy())], itnlim, tol, tol, 1e8 if tol else 0.0)
    (x,) = drv.solution([torch.zeros(shape.n_unknowns, dtype=torch.float64)])
    xs = [torch.zeros_like(x) for _ in range(2)]
    dist.all_gather(xs, x)
    assert torch.equal(xs[0], xs[1])                # both ranks hold the same whole solution
    out[str(itnlim)] = {{"istop": int(res.istop), "itn": int(res.itn), "x": x.tolist(), "exchanges": drv.exchanges}}
if comm.rank == 0:
    print("RESULT " + json.dumps(out))
dist.destroy_process_group()
'''


def test_sharded_solve_gloo_world_size_2(tmp_path):
    script = tmp_path / "shard_worker.py"
    script.write_text(WORKER.format(root=ROOT))
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29541", OMP_NUM_THREADS="1")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                          "--master-addr", "127.0.0.1", "--master-port", "29541", str(script)],
                         capture_output=True, text=True, env=env, timeout=600)
    assert out.returncode == 0, out.stderr[-3000:]
    lines = [ln for ln in out.stdout.splitlines() if ln.startswith("RESULT ")]
    assert len(lines) == 1                                    # rank 0 alone reports
    got = json.loads(lines[0][len("RESULT "):])
    shape = C5.scaled(24, n_knots=20, n_instr=25, n_constraint_rows=8, name="C5-tiny")
    a, idx = host.make_rows(shape)
    b = rhs(shape, a, idx, host.x_true(shape))
    L = oracle.layout_of(shape)
    xr, rr = oracle.lsqr(L, a, idx, b, itnlim=3)
    g = got["3"]
    assert g["itn"] == 3 and g["istop"] == 7 and g["exchanges"] == 3 + 2 * 3
    assert np.linalg.norm(np.array(g["x"]) - xr) <= 1e-9 * np.linalg.norm(xr)
    xr, rr = oracle.lsqr(L, a, idx, b, itnlim=4000, atol=1e-12, btol=1e-12, conlim=1e8)
    g = got["4000"]
    assert g["istop"] == rr["istop"] and abs(g["itn"] - rr["itn"]) <= max(3, 0.05 * rr["itn"])
    assert np.linalg.norm(np.array(g["x"]) - xr) <= 1e-9 * np.linalg.norm(xr)
