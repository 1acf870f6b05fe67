"""Device (CUDA) side of the seeded generator: fills torch CUDA tensors in HBM.

Inputs only.  Mirrors gaia_synth/host.py (same hash, same streams); used for the C2..C5
sized systems, which are generated directly on the GPU -- the oracle is then fed the very
same bytes copied back, never a second generation.
"""
import ctypes as ct
import os
import subprocess

import numpy as np

from . import configs as C
from . import host

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libgaia_synth.so")
_SRC = os.path.join(_HERE, "device.cu")
_lib = None


def build(force: bool = False) -> str:
    if not force and os.path.exists(_SO) and os.path.getmtime(_SO) >= os.path.getmtime(_SRC):
        return _SO
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    tmp = _SO + ".tmp%d" % os.getpid()
    subprocess.check_call([nvcc, "-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
                           "-Xcompiler", "-fPIC", "-shared", "-cudart", "static", "-o", tmp, _SRC])
    os.replace(tmp, _SO)
    return _SO


def lib():
    global _lib
    if _lib is None:
        L = ct.CDLL(build())
        vp = ct.c_void_p
        L.gs_fill_rows.restype = ct.c_int
        L.gs_fill_rows.argtypes = [vp, vp, ct.c_uint64, ct.c_int64, ct.c_int64, ct.c_int64, ct.c_int64, ct.c_int64,
                                   ct.c_int64, ct.c_int64, ct.c_int32, ct.c_int32, vp, ct.c_int32, vp, ct.c_int32,
                                   ct.c_int32, ct.c_double, vp]
        L.gs_fill_normal.restype = ct.c_int
        L.gs_fill_normal.argtypes = [vp, ct.c_int64, ct.c_int64, ct.c_uint64, ct.c_int32, ct.c_double, vp]
        _lib = L
    return _lib


def _stream():
    import torch
    return torch.cuda.current_stream().cuda_stream


def make_system(shape: C.SystemShape, device="cuda", r0: int = 0, r1: int = None):
    """(values [M,24] float64, indices [M,8] int32) as CUDA tensors, generated in place in HBM.
    r0/r1 select a row range (default: the whole system)."""
    import torch
    sptr_dev = None
    if shape.obs_per_star:
        m_obs = shape.n_stars * shape.obs_per_star
    else:
        sptr = host.star_ptr(shape)
        m_obs = int(sptr[-1])
        sptr_dev = torch.from_numpy(sptr).to(device)
    m = m_obs + shape.n_constraint_rows
    hot_dev, wlen = None, 0
    if shape.hot_knots:
        ws, wlen = host.hot_windows(shape)
        hot_dev = torch.from_numpy(ws.astype(np.int64)).to(device)
    r1 = m if r1 is None else min(r1, m)
    nr = max(r1 - r0, 0)
    vals = torch.empty((nr, 24), dtype=torch.float64, device=device)
    idx = torch.empty((nr, 8), dtype=torch.int32, device=device)
    rc = lib().gs_fill_rows(vals.data_ptr(), idx.data_ptr(), shape.seed, r0, nr, m_obs, shape.n_constraint_rows,
                            shape.n_stars, shape.n_knots, shape.n_instr, shape.n_glob, shape.obs_per_star,
                            sptr_dev.data_ptr() if sptr_dev is not None else None, int(shape.hot_knots),
                            hot_dev.data_ptr() if hot_dev is not None else None, C.N_HOT_WINDOWS, wlen,
                            C.HOT_PROB, _stream())
    if rc != 0:
        raise RuntimeError(f"gs_fill_rows: CUDA error {rc}")
    torch.cuda.current_stream().synchronize()   # sptr_dev / hot_dev may be freed after return
    return vals, idx


def normal(seed: int, stream_id: int, i0: int, i1: int, scale: float = 1.0, device="cuda"):
    import torch
    out = torch.empty(i1 - i0, dtype=torch.float64, device=device)
    rc = lib().gs_fill_normal(out.data_ptr(), i0, i1 - i0, seed, stream_id, scale, _stream())
    if rc != 0:
        raise RuntimeError(f"gs_fill_normal: CUDA error {rc}")
    return out


def x_true(shape: C.SystemShape, device="cuda"):
    return normal(shape.seed, C.STREAM_XTRUE, 0, shape.n_unknowns, device=device)


def noise(shape: C.SystemShape, m: int, device="cuda"):
    return normal(shape.seed, C.STREAM_NOISE, 0, m, scale=shape.sigma, device=device)


def test_vector(seed: int, tag: int, n: int, device="cuda"):
    return normal(seed ^ (tag * 0x100000001B3 & 0xFFFFFFFFFFFF), C.STREAM_VEC, 0, n, device=device)
