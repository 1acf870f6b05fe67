"""Seeded synthetic Gaia-shaped systems (inputs only; none of the method's arithmetic).

`host`   : numpy generator (CPU tests, small systems).
`device` : the same counter-based generator as a CUDA kernel (C2..C5 sized systems
           are generated directly in HBM; the oracle is then fed bytes copied back).
Both are used by tests/ and bench.py; neither imports the oracle or the library.
"""
from .configs import CONFIGS, C1, C2, C3, C4, C5, SystemShape  # noqa: F401
