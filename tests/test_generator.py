"""Seeded generator: structure of the synthetic Gaia-shaped systems (CPU only)."""
import numpy as np

from gaia_synth import host
from gaia_synth.configs import C1, C3, C5


def test_c1_structure():
    a, idx = host.make_rows(C1)
    assert a.shape == (20000, 24) and idx.shape == (20000, 8) and idx.dtype == np.int32
    assert np.all(np.diff(idx[:, 0]) >= 0) and idx[0, 0] == 0 and idx[-1, 0] == 999   # sorted by star
    assert np.all(np.bincount(idx[:, 0]) == 20)
    assert idx[:, 1].min() >= 0 and idx[:, 1].max() <= C1.n_knots - 5                 # start in [0, K-4)
    s = np.sort(idx[:, 2:], axis=1)
    assert s.min() >= 0 and s.max() < 60 and np.all(np.diff(s, axis=1) > 0)           # 6 distinct columns
    assert abs(a.mean()) < 0.01 and abs(a.std() - 1) < 0.01
    assert C1.n_unknowns == 8061


def test_chunks_reproduce_whole():
    a, idx = host.make_rows(C1)
    a2, idx2 = host.make_rows(C1, 5000, 5100)
    assert np.array_equal(a2, a[5000:5100]) and np.array_equal(idx2, idx[5000:5100])
    a3, _ = host.make_rows(C1)
    assert np.array_equal(a, a3)


def test_c3_power_law_and_hot_knots():
    c3 = C3.scaled(20000)
    cnt = host.obs_counts(c3)
    assert cnt.min() >= 10 and cnt.max() <= 2000 and 45 < cnt.mean() < 57   # literal alpha=2 -> mean ~51 (R11)
    sp = host.star_ptr(c3)
    a, idx = host.make_rows(c3, 0, 200000, sp)
    assert np.all(np.diff(idx[:, 0]) >= 0)
    assert np.array_equal(np.bincount(idx[:, 0])[:100], cnt[:100])
    h = np.sort(np.bincount(idx[:, 1], minlength=c3.n_knots))[::-1]
    assert 0.45 < h[: c3.n_knots // 20].sum() / h.sum() < 0.62              # ~5 % of knots get ~50 % of rows (R12)


def test_c5_constraint_rows():
    c5 = C5.scaled(50, n_knots=100, n_instr=30, n_constraint_rows=10)
    a, idx = host.make_rows(c5)
    assert a.shape[0] == 50 * 80 + 10
    att, ins = a[-10:-5], a[-5:]
    assert np.all(att[:, 5:17] == 1.0) and np.all(att[:, :5] == 0) and np.all(att[:, 17:] == 0)
    assert np.all(ins[:, 17:23] == 1.0) and np.all(ins[:, :17] == 0) and np.all(ins[:, 23] == 0)
    assert np.all(idx[-10:, 0] == 49)
