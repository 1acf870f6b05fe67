"""Host (numpy) side of the seeded generator.  Inputs only - no aprod / LSQR arithmetic here.

Counter-based: every quantity is a pure function of (seed, stream, counter), so any
row range can be produced independently.  `device.cu` implements the same integer
hash; all *integer* outputs (index records) are bit-identical between the two, the
N(0,1) values agree to a few ulp (libm vs CUDA log/sin/cos).

Row layout:
  values [M,24] fp64 : slots 0-4 astro, 5-16 attitude (axis-major, 4 knots each),
                       17-22 instrumental, 23 global
  indices[M,8] int32 : {star, att_start, instr_col[0..5]}
"""
import numpy as np

from . import configs as C

_GOLD = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)
_TWO_M32 = 2.0 ** -32


def _mix64(z):
    z = np.asarray(z, dtype=np.uint64)
    z = (z ^ (z >> np.uint64(30))) * _M1
    z = (z ^ (z >> np.uint64(27))) * _M2
    return z ^ (z >> np.uint64(31))


def _key(seed, stream):
    with np.errstate(over="ignore"):
        return _mix64(np.uint64(seed) + np.uint64(stream) * _GOLD)


def rnd64(seed, stream, ctr):
    """uint64 hash of (seed, stream, ctr); ctr is an integer array."""
    with np.errstate(over="ignore"):
        return _mix64(_key(seed, stream) + np.asarray(ctr, dtype=np.uint64) * _GOLD)


def _hi(h):
    return (h >> np.uint64(32)).astype(np.uint64)


def _lo(h):
    return (h & np.uint64(0xFFFFFFFF)).astype(np.uint64)


def _bounded(u32, n):
    """uniform integer in [0, n) from a 32-bit uniform (multiply-shift)."""
    return ((u32 * np.uint64(n)) >> np.uint64(32)).astype(np.int64)


def normal_pairs(seed, stream, ctr):
    """Two N(0,1) per counter (Box-Muller on the two 32-bit halves of one hash)."""
    h = rnd64(seed, stream, ctr)
    u1 = (_hi(h).astype(np.float64) + 1.0) * _TWO_M32      # (0,1]
    u2 = _lo(h).astype(np.float64) * _TWO_M32              # [0,1)
    rad = np.sqrt(-2.0 * np.log(u1))
    ang = (2.0 * np.pi) * u2
    return rad * np.cos(ang), rad * np.sin(ang)


def normal(seed, stream, i0, i1):
    """N(0,1) for element counters i0..i1-1 (element e uses pair e//2, component e%2)."""
    e = np.arange(i0, i1, dtype=np.int64)
    z0, z1 = normal_pairs(seed, stream, e >> 1)
    return np.where((e & 1) == 0, z0, z1)


# ---------------------------------------------------------------- star / row structure
def obs_counts(shape: C.SystemShape) -> np.ndarray:
    """Observations per star (int64[S])."""
    S = shape.n_stars
    if shape.obs_per_star:
        return np.full(S, shape.obs_per_star, dtype=np.int64)
    alpha, kmin, kmax = shape.obs_powerlaw
    k = np.arange(kmin, kmax + 1, dtype=np.float64)
    cdf = np.cumsum(k ** (-alpha))
    cdf /= cdf[-1]
    u = (_hi(rnd64(shape.seed, C.STREAM_OBS, np.arange(S))).astype(np.float64) + 0.5) * _TWO_M32
    return (kmin + np.searchsorted(cdf, u, side="left")).astype(np.int64)


def star_ptr(shape: C.SystemShape) -> np.ndarray:
    """Row pointer per star (int64[S+1]); observation rows only."""
    p = np.zeros(shape.n_stars + 1, dtype=np.int64)
    np.cumsum(obs_counts(shape), out=p[1:])
    return p


def n_obs_rows(shape: C.SystemShape) -> int:
    if shape.obs_per_star:
        return shape.n_stars * shape.obs_per_star
    return int(star_ptr(shape)[-1])


def n_rows(shape: C.SystemShape) -> int:
    return n_obs_rows(shape) + shape.n_constraint_rows


def hot_windows(shape: C.SystemShape):
    """(window starts int64[N_HOT_WINDOWS], window length) in knot units, for the C3 mixture."""
    span = shape.n_knots - 4
    wlen = max(1, int(span * C.HOT_FRACTION / C.N_HOT_WINDOWS))
    h = rnd64(shape.seed, C.STREAM_HOTSET, np.arange(C.N_HOT_WINDOWS))
    return _bounded(_hi(h), span - wlen + 1), wlen


def _att_start(shape, rows):
    span = shape.n_knots - 4                      # start in [0, K-4)  ->  0 .. K-5
    h1 = rnd64(shape.seed, C.STREAM_ATT, 2 * rows)
    uni = _bounded(_hi(h1), span)
    if not shape.hot_knots:
        return uni
    ws, wlen = hot_windows(shape)
    h2 = rnd64(shape.seed, C.STREAM_ATT, 2 * rows + 1)
    is_hot = _lo(h1) < np.uint64(int(C.HOT_PROB * 2 ** 32))
    w = _bounded(_hi(h2), C.N_HOT_WINDOWS)
    hot = ws[w] + _bounded(_lo(h2), wlen)
    return np.where(is_hot, hot, uni)


def _instr_cols(shape, rows):
    """6 distinct columns per row, uniform without replacement (rank-skipping draw)."""
    I = shape.n_instr
    out = np.empty((rows.size, 6), dtype=np.int64)
    srt = np.empty((rows.size, 6), dtype=np.int64)   # previous picks, ascending
    for s in range(6):
        h = rnd64(shape.seed, C.STREAM_INSTR, 8 * rows + s)
        d = _bounded(_hi(h), I - s)
        for j in range(s):                           # skip over earlier picks in ascending order
            d = d + (d >= srt[:, j])
        out[:, s] = d
        # insert d into the sorted prefix
        if s == 0:
            srt[:, 0] = d
        else:
            pos = (srt[:, :s] < d[:, None]).sum(axis=1)
            new = np.empty((rows.size, s + 1), dtype=np.int64)
            ar = np.arange(s + 1)[None, :]
            src = np.where(ar < pos[:, None], ar, ar - 1)
            new[:] = np.take_along_axis(srt[:, :s], np.clip(src, 0, s - 1), axis=1)
            new[np.arange(rows.size), pos] = d
            srt[:, : s + 1] = new
    return out


def make_rows(shape: C.SystemShape, r0: int = 0, r1: int = None, sptr: np.ndarray = None):
    """values[r1-r0,24] fp64 and indices[r1-r0,8] int32 for rows r0..r1-1."""
    M_obs = n_obs_rows(shape) if sptr is None else int(sptr[-1])
    M = M_obs + shape.n_constraint_rows
    r1 = M if r1 is None else r1
    rows = np.arange(r0, r1, dtype=np.int64)
    nr = rows.size
    z0, z1 = normal_pairs(shape.seed, C.STREAM_VALUES, (rows[:, None] * 12 + np.arange(12)[None, :]).ravel())
    vals = np.empty((nr, 24), dtype=np.float64)
    vals[:, 0::2] = z0.reshape(nr, 12)
    vals[:, 1::2] = z1.reshape(nr, 12)
    idx = np.empty((nr, 8), dtype=np.int32)
    if shape.obs_per_star:
        star = rows // shape.obs_per_star
    else:
        sptr = star_ptr(shape) if sptr is None else sptr
        star = np.searchsorted(sptr, rows, side="right") - 1
    star = np.minimum(star, shape.n_stars - 1)
    idx[:, 0] = star
    idx[:, 1] = _att_start(shape, rows)
    idx[:, 2:8] = _instr_cols(shape, rows)
    if shape.n_glob == 0:
        vals[:, 23] = 0.0
    # constraint rows (reading R9): unit coefficients on attitude / instrumental
    c = rows >= M_obs
    if c.any():
        half = shape.n_constraint_rows // 2
        is_att = c & (rows < M_obs + half)
        is_ins = c & ~is_att
        vals[c, :] = 0.0
        vals[np.ix_(is_att, range(5, 17))] = 1.0
        vals[np.ix_(is_ins, range(17, 23))] = 1.0
        idx[c, 0] = shape.n_stars - 1
    return vals, idx


def x_true(shape: C.SystemShape) -> np.ndarray:
    return normal(shape.seed, C.STREAM_XTRUE, 0, shape.n_unknowns)


def noise(shape: C.SystemShape, r0: int, r1: int) -> np.ndarray:
    """sigma * N(0,1) for rows r0..r1-1 (sigma is a standard deviation, reading R5)."""
    return shape.sigma * normal(shape.seed, C.STREAM_NOISE, r0, r1)


def test_vector(seed: int, tag: int, n: int) -> np.ndarray:
    """Generic N(0,1) vector for tests (tag separates independent vectors)."""
    return normal(seed ^ (tag * 0x100000001B3 & 0xFFFFFFFFFFFF), C.STREAM_VEC, 0, n)
