"""Host-side checks that need no GPU: the C-ABI library builds, loads and exports every symbol
include/gsr.h declares; argument validation that happens before any CUDA call."""
import ctypes as ct
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libgsr():
    from paper_2503_22863_b200 import build
    build.build()
    from paper_2503_22863_b200 import binding
    return binding.lib()


def declared_symbols():
    hdr = open(os.path.join(ROOT, "include", "gsr.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    return sorted(set(re.findall(r"\b(gsr_[a-z0-9_]+)\s*\(", hdr)))


def test_every_declared_symbol_is_exported(libgsr):
    from paper_2503_22863_b200.binding import SYMBOLS
    decl = declared_symbols()
    assert len(decl) >= 18
    for name in decl:
        assert hasattr(libgsr, name), f"{name} declared in include/gsr.h but not exported"
    assert sorted(SYMBOLS) == decl          # the binding covers exactly the header


def test_strerror_and_version(libgsr):
    assert libgsr.gsr_strerror(0) == b"ok"
    assert b"layout" in libgsr.gsr_strerror(-2)
    assert b"sm_100a" in libgsr.gsr_version()


def test_argument_validation_without_gpu(libgsr):
    from paper_2503_22863_b200.binding import _Layout
    h = ct.c_void_p()
    assert libgsr.gsr_create(None, None, None, None, None) == -1
    assert libgsr.gsr_create(ct.byref(h), None, None, None, None) == -1
    bad = _Layout(10, 1, 8, 6, 2, 0)                                   # n_glob = 2
    assert libgsr.gsr_create(ct.byref(h), ct.byref(bad), None, None, None) == -1
    bad = _Layout(10, 1, 3, 6, 1, 0)                                   # K < 4
    assert libgsr.gsr_create(ct.byref(h), ct.byref(bad), None, None, None) == -1
    bad = _Layout(10, 1, 8, 6, 1, 0)                                   # null arrays with M > 0
    assert libgsr.gsr_create(ct.byref(h), ct.byref(bad), None, None, None) == -1
    bad = _Layout(10, 1, 8, 6, 1, 2)                                   # unknown flag bit
    assert libgsr.gsr_create(ct.byref(h), ct.byref(bad), None, None, None) == -1
    assert libgsr.gsr_aprod1(None, None, None, None) == -1
    assert libgsr.gsr_lsqr_iterate(None, 1, 1, 0.0, 0.0, 0.0, None) == -1
    libgsr.gsr_destroy(None)                                           # no-op


def test_host_entry_validates_before_it_sizes_anything(libgsr):
    """gsr_lsqr_host computes allocation sizes from the layout: a bad layout must be GSR_EINVAL, not GSR_ENOMEM,
    and a host buffer of the wrong dtype must be refused by the binding (it would be read past its end)."""
    import numpy as np
    import torch
    from paper_2503_22863_b200 import binding
    from paper_2503_22863_b200.binding import _Layout, _Result
    r = _Result()
    x = np.zeros(64)
    for bad in (_Layout(4, -3, 8, 6, 1, 0), _Layout(4, 1, 2, 6, 1, 0), _Layout(4, 1, 8, 0, 1, 0), _Layout(4, 1, 8, 6, 5, 0),
                _Layout(-1, 1, 8, 6, 1, 0), _Layout(4, 1, 8, 6, 1, 4)):
        rc = libgsr.gsr_lsqr_host(ct.byref(bad), x.ctypes.data, x.ctypes.data, x.ctypes.data, x.ctypes.data, 1, 0.0, 0.0,
                                  0.0, ct.byref(r))
        assert rc == -1
    with pytest.raises(ValueError):      # float32 values of the right element count
        binding._host_ptr(torch.zeros(4 * 24, dtype=torch.float32), np.float64, 4 * 24, "values")
    with pytest.raises(ValueError):      # int64 indices
        binding._host_ptr(torch.zeros(4 * 8, dtype=torch.int64), np.int32, 4 * 8, "indices")
    with pytest.raises(ValueError):
        binding._host_ptr(np.zeros(4 * 8, dtype=np.int64), np.int32, 4 * 8, "indices")
    assert binding._host_ptr(torch.zeros(4 * 8, dtype=torch.int32), np.int32, 4 * 8, "indices") != 0


def test_no_cpu_fallback():
    """Without a CUDA device the product path must fail loudly, never route through the oracle."""
    import torch
    import paper_2503_22863_b200 as gsr
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(TypeError):
        gsr.gsr_create(1, 8, 6, 1, torch.zeros((4, 24), dtype=torch.float64), torch.zeros((4, 8), dtype=torch.int32))
    src = "".join(open(os.path.join(ROOT, "paper_2503_22863_b200", f)).read()
                  for f in ("__init__.py", "binding.py", "build.py", "sharded.py"))
    assert "import oracle" not in src and "from oracle" not in src
    for f in os.listdir(os.path.join(ROOT, "paper_2503_22863_b200", "csrc")):
        assert "oracle" not in open(os.path.join(ROOT, "paper_2503_22863_b200", "csrc", f)).read().lower()
