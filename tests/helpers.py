"""Test-side helpers: a third, trivial code path for the slot -> column map (used to pin
the oracle), and small system builders.  No oracle or library code is reused here."""
import numpy as np

from gaia_synth import host
from gaia_synth.configs import SystemShape


def columns_of(shape: SystemShape, idx: np.ndarray) -> np.ndarray:
    """cols[M,24] written straight from the layout statement in BASELINE.json configs[0]:
    5 astro (cols 5*star..+4), 12 attitude (3 axes x 4 consecutive knots, axis offset K),
    6 instr, 1 global; x = [astro | att | instr | glob].  -1 where n_glob == 0."""
    S, K, I, G = shape.n_stars, shape.n_knots, shape.n_instr, shape.n_glob
    m = idx.shape[0]
    cols = np.empty((m, 24), dtype=np.int64)
    star = idx[:, 0].astype(np.int64)
    t = idx[:, 1].astype(np.int64)
    for k in range(5):
        cols[:, k] = 5 * star + k
    for ax in range(3):
        for j in range(4):
            cols[:, 5 + 4 * ax + j] = 5 * S + ax * K + t + j
    for s in range(6):
        cols[:, 17 + s] = 5 * S + 3 * K + idx[:, 2 + s]
    cols[:, 23] = 5 * S + 3 * K + I if G else -1
    return cols


def dense_matrix(shape: SystemShape, a: np.ndarray, idx: np.ndarray) -> np.ndarray:
    """Dense M x n matrix, D[r, col(r,k)] += a[r,k]  (tiny systems only)."""
    cols = columns_of(shape, idx)
    m = a.shape[0]
    D = np.zeros((m, shape.n_unknowns))
    for r in range(m):
        for k in range(24):
            if cols[r, k] >= 0:
                D[r, cols[r, k]] += a[r, k]
    return D


def csr_matrix(shape: SystemShape, a: np.ndarray, idx: np.ndarray):
    import scipy.sparse as sp
    cols = columns_of(shape, idx)
    m = a.shape[0]
    rows = np.repeat(np.arange(m), 24)
    c = cols.ravel()
    v = a.ravel()
    keep = c >= 0
    return sp.coo_matrix((v[keep], (rows[keep], c[keep])), shape=(m, shape.n_unknowns)).tocsr()


def tiny_shape(n_stars=8, obs=12, n_knots=8, n_instr=8, n_glob=1, seed=1234, **kw) -> SystemShape:
    return SystemShape("tiny", n_stars=n_stars, obs_per_star=obs, n_knots=n_knots,
                       n_instr=n_instr, n_glob=n_glob, seed=seed, **kw)


def nonempty_columns(shape: SystemShape, idx: np.ndarray) -> np.ndarray:
    cols = columns_of(shape, idx)
    mask = np.zeros(shape.n_unknowns, dtype=bool)
    mask[cols[cols >= 0]] = True
    return mask


def rhs(shape: SystemShape, a, idx, xt, noisy=True):
    """b = A x_true (+ sigma N(0,1)), A x_true through the test-side column map (float64 dot)."""
    cols = columns_of(shape, idx)
    xg = np.where(cols >= 0, xt[np.clip(cols, 0, None)], 0.0)
    b = np.einsum("rk,rk->r", a, xg)
    if noisy:
        b = b + host.noise(shape, 0, a.shape[0])
    return b
