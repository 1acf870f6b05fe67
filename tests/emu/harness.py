"""Load tests/emu/libgsr_emu.so in the place of libgsr.so FOR THE DURATION OF A TEST and let the binding take host
tensors, so that the bodies of the GPU parity tests can run on the host emulation of the kernels.  Test-side only."""
import contextlib
import ctypes as ct
import os
import sys

import numpy as np
import torch

HERE = os.path.dirname(os.path.abspath(__file__))
if HERE not in sys.path:
    sys.path.insert(0, HERE)

import build_emu  # noqa: E402
from paper_2503_22863_b200 import binding  # noqa: E402

_emu = None


def emu_lib():
    global _emu
    if _emu is None:
        L = ct.CDLL(build_emu.build())
        for name, (res, args) in binding.SYMBOLS.items():
            f = getattr(L, name)
            f.restype, f.argtypes = res, args
        _emu = L
    return _emu


def host_tensor(a):
    """A torch-owned (64-byte aligned) host copy: the ABI wants 32-byte aligned records."""
    return torch.from_numpy(np.ascontiguousarray(a)).clone()


def _host_dev_ptr(t, dtype, numel, name):
    if t is None:
        return None
    if not isinstance(t, torch.Tensor) or t.is_cuda:
        raise TypeError(f"{name}: the emulated library takes host tensors")
    if t.dtype != dtype or not t.is_contiguous() or t.numel() != numel:
        raise ValueError(f"{name}: need contiguous {dtype} with {numel} elements, got {t.dtype} {tuple(t.shape)}")
    return t.data_ptr()


class HostGen:
    """gaia_synth.device's interface on the host generator (the two produce identical index records and values equal
    to a few ulp: tests/test_gpu_parity.py::test_device_generator_matches_host), returning host tensors."""

    @staticmethod
    def make_system(shape, device="cpu", r0=0, r1=None):
        from gaia_synth import host
        a, idx = host.make_rows(shape, r0, r1)
        return host_tensor(a), host_tensor(idx)

    @staticmethod
    def normal(seed, stream_id, i0, i1, scale=1.0, device="cpu"):
        from gaia_synth import host
        return host_tensor(host.normal(seed, stream_id, i0, i1) * scale)

    @staticmethod
    def x_true(shape, device="cpu"):
        from gaia_synth import host
        return host_tensor(host.x_true(shape))

    @staticmethod
    def noise(shape, m, device="cpu"):
        from gaia_synth import host
        return host_tensor(host.noise(shape, 0, m))

    @staticmethod
    def test_vector(seed, tag, n, device="cpu"):
        from gaia_synth import host
        return host_tensor(host.test_vector(seed, tag, n))


@contextlib.contextmanager
def fake_cuda_queries():
    """torch.cuda's capacity queries answered for the dry runs of the full-size test bodies on small stand-in shapes."""
    saved = (torch.cuda.mem_get_info, torch.cuda.empty_cache, torch.cuda.is_available)
    torch.cuda.mem_get_info = lambda *a, **k: (1 << 42, 1 << 42)
    torch.cuda.empty_cache = lambda: None
    torch.cuda.is_available = lambda: True
    try:
        yield
    finally:
        torch.cuda.mem_get_info, torch.cuda.empty_cache, torch.cuda.is_available = saved


@contextlib.contextmanager
def emulated(*modules):
    """Inside the block paper_2503_22863_b200.binding talks to the emulated library; `modules` (GPU test modules) get
    DEV = "cpu" and a dev() that makes aligned host copies.  Everything is put back afterwards."""
    # helpers are shared between the GPU test modules (test_gpu_zzzz_coeff23 calls into test_gpu_z_f3): patch them all
    modules = list(modules) + [m for name, m in list(sys.modules.items())
                               if (name.startswith("test_gpu_") or name == "gpu_helpers") and m not in modules]
    saved = (binding._lib, binding._dev_ptr, binding._stream, binding.GsrSystem.exchange_buffer)
    saved_mod = [(m, getattr(m, "DEV", None), getattr(m, "dev", None), getattr(m, "gdev", None)) for m in modules]
    binding._lib = emu_lib()
    binding._dev_ptr = _host_dev_ptr
    binding._stream = lambda: None
    binding.GsrSystem.exchange_buffer = lambda self: torch.zeros(self.shard_exchange_len(), dtype=torch.float64)
    for m in modules:
        if hasattr(m, "DEV"):
            m.DEV = "cpu"
        if hasattr(m, "dev"):
            m.dev = host_tensor
        if hasattr(m, "gdev"):
            m.gdev = HostGen
    try:
        yield
    finally:
        binding._lib, binding._dev_ptr, binding._stream, binding.GsrSystem.exchange_buffer = saved
        for m, d, f, g in saved_mod:
            if d is not None:
                m.DEV = d
            if f is not None:
                m.dev = f
            if g is not None:
                m.gdev = g
