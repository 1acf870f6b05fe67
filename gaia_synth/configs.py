"""Shapes of the synthetic Gaia-shaped systems (BASELINE.json `configs`, C1..C5).

Nothing here is arithmetic of the method: only sizes and the seeds.  The
readings of the under-specified points (K and I of C5, the C3 power law, the
constraint rows) are listed in DESIGN.md section 3.

Notation: S stars, M rows, K attitude knots per axis,
I instrumental parameters, G in {0,1} global parameters.
x = [astro 5S | attitude 3K | instrumental I | global G].
"""
from dataclasses import dataclass, replace

SEED_BASE = 0x5EED0000


@dataclass(frozen=True)
class SystemShape:
    name: str
    n_stars: int
    n_knots: int          # per axis
    n_instr: int
    n_glob: int = 1
    obs_per_star: int = 0  # uniform case; 0 -> power law (C3)
    obs_powerlaw: tuple = ()  # (alpha, kmin, kmax)
    hot_knots: bool = False   # C3 attitude hot-spot mixture
    n_constraint_rows: int = 0  # C5
    seed: int = SEED_BASE
    sigma: float = 1e-6

    @property
    def n_unknowns(self) -> int:
        return 5 * self.n_stars + 3 * self.n_knots + self.n_instr + self.n_glob

    @property
    def off_att(self) -> int:
        return 5 * self.n_stars

    @property
    def off_instr(self) -> int:
        return 5 * self.n_stars + 3 * self.n_knots

    @property
    def off_glob(self) -> int:
        return 5 * self.n_stars + 3 * self.n_knots + self.n_instr

    def scaled(self, n_stars: int, **kw) -> "SystemShape":
        """Same family, fewer stars (for tests that need a cheaper system)."""
        return replace(self, n_stars=n_stars, **kw)


C1 = SystemShape("C1", n_stars=1_000, obs_per_star=20, n_knots=1_000, n_instr=60, seed=SEED_BASE + 1)
C2 = SystemShape("C2", n_stars=100_000, obs_per_star=100, n_knots=20_000, n_instr=600, seed=SEED_BASE + 2)
C3 = SystemShape("C3", n_stars=1_000_000, obs_powerlaw=(2.0, 10, 2000), n_knots=200_000,
                 n_instr=6_000, hot_knots=True, seed=SEED_BASE + 3)
# C3 as BASELINE.json states its size ("mean ~70 ... ~7e7 rows"): the exponent that gives that mean on 10..2000 is 1.83
# (reading R11; the literal alpha = 2 above gives mean 51.1, ~5.1e7 rows).  Same hot-knot mixture.
C3B = SystemShape("C3b", n_stars=1_000_000, obs_powerlaw=(1.83, 10, 2000), n_knots=200_000,
                  n_instr=6_000, hot_knots=True, seed=SEED_BASE + 3)
C4 = SystemShape("C4", n_stars=5_000_000, obs_per_star=100, n_knots=1_000_000, n_instr=60_000,
                 seed=SEED_BASE + 4)
C5 = SystemShape("C5", n_stars=2_000_000, obs_per_star=80, n_knots=400_000, n_instr=12_000,
                 n_constraint_rows=10_000, seed=SEED_BASE + 5)

CONFIGS = {c.name: c for c in (C1, C2, C3, C3B, C4, C5)}

# stream ids of the counter-based generator (shared by host.py and device.cu)
STREAM_VALUES = 1
STREAM_ATT = 2
STREAM_INSTR = 3
STREAM_OBS = 4
STREAM_XTRUE = 5
STREAM_NOISE = 6
STREAM_HOTSET = 7
STREAM_VEC = 8       # generic test vectors
N_HOT_WINDOWS = 100
HOT_FRACTION = 0.05  # hot windows cover 5 % of the time range
HOT_PROB = 0.5       # and receive 50 % of the rows
