"""ctypes binding of libgsr.so -- argument marshalling only (same names as include/gsr.h)."""
import ctypes as ct
import os
from dataclasses import dataclass

_PKG = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_PKG, "libgsr.so")

GSR_OK = 0
_vp = ct.c_void_p


class GsrError(RuntimeError):
    def __init__(self, code, where):
        msg = lib().gsr_strerror(code).decode()
        cuda = lib().gsr_last_cuda_error().decode()
        super().__init__(f"{where}: {msg} ({code})" + (f" [{cuda}]" if code == -4 and cuda else ""))
        self.code = code


class _Layout(ct.Structure):
    _fields_ = [("n_rows", ct.c_int64), ("n_stars", ct.c_int64), ("n_knots", ct.c_int64),
                ("n_instr", ct.c_int64), ("n_glob", ct.c_int32), ("flags", ct.c_int32)]


class _Result(ct.Structure):
    _fields_ = [("istop", ct.c_int32), ("itn", ct.c_int64), ("r1norm", ct.c_double),
                ("r2norm", ct.c_double), ("anorm", ct.c_double), ("acond", ct.c_double),
                ("arnorm", ct.c_double), ("xnorm", ct.c_double), ("bnorm", ct.c_double)]


_SCALARS = ("alpha", "beta", "rhobar", "phibar", "bnorm", "rnorm", "arnorm", "anorm", "acond",
            "ddnorm", "xnorm", "xxnorm", "z", "cs2", "sn2")


class _Scalars(ct.Structure):
    _fields_ = [("itn", ct.c_int64), ("istop", ct.c_int32)] + [(k, ct.c_double) for k in _SCALARS]


@dataclass
class LsqrResult:
    istop: int
    itn: int
    r1norm: float
    r2norm: float
    anorm: float
    acond: float
    arnorm: float
    xnorm: float
    bnorm: float


GSR_PRECOND_COLNORM = 1
GSR_SHARD_MORE, GSR_SHARD_INIT_DONE, GSR_SHARD_ITER_DONE = 0, 1, 2
GSR_LAYOUT_TRUSTED = 1
GSR_LAYOUT_COEFF23 = 2

_lib = None

# name -> (restype, argtypes); every symbol include/gsr.h declares
SYMBOLS = {
    "gsr_create": (ct.c_int, [ct.POINTER(_vp), ct.POINTER(_Layout), _vp, _vp, _vp]),
    "gsr_destroy": (None, [_vp]),
    "gsr_attach_constraints": (ct.c_int, [_vp, ct.c_int64, _vp, _vp, _vp]),
    "gsr_dims": (ct.c_int, [_vp, ct.POINTER(ct.c_int64), ct.POINTER(ct.c_int64)]),
    "gsr_aprod1": (ct.c_int, [_vp, _vp, _vp, _vp]),
    "gsr_aprod2": (ct.c_int, [_vp, _vp, _vp, _vp]),
    "gsr_lsqr": (ct.c_int, [_vp, _vp, _vp, ct.c_int64, ct.c_double, ct.c_double, ct.c_double,
                            ct.POINTER(_Result), _vp]),
    "gsr_lsqr_ex": (ct.c_int, [_vp, _vp, _vp, _vp, ct.c_int32, ct.c_int64, ct.c_double, ct.c_double, ct.c_double,
                               ct.POINTER(_Result), _vp]),
    "gsr_colnorms": (ct.c_int, [_vp, _vp, _vp]),
    "gsr_set_cov_pairs": (ct.c_int, [_vp, _vp, _vp, ct.c_int64, _vp, _vp]),
    "gsr_lsqr_init": (ct.c_int, [_vp, _vp, _vp]),
    "gsr_lsqr_iterate": (ct.c_int, [_vp, ct.c_int64, ct.c_int64, ct.c_double, ct.c_double, ct.c_double, _vp]),
    "gsr_lsqr_result_get": (ct.c_int, [_vp, _vp, ct.POINTER(_Result), _vp]),
    "gsr_lsqr_get_state": (ct.c_int, [_vp, _vp, _vp, _vp, _vp, ct.POINTER(_Scalars), _vp]),
    "gsr_lsqr_host": (ct.c_int, [ct.POINTER(_Layout), _vp, _vp, _vp, _vp, ct.c_int64, ct.c_double,
                                 ct.c_double, ct.c_double, ct.POINTER(_Result)]),
    "gsr_shard_exchange_len": (ct.c_int, [_vp, ct.POINTER(ct.c_int64)]),
    "gsr_shard_begin": (ct.c_int, [_vp, _vp, _vp, ct.c_int32, ct.c_int64, ct.c_double, ct.c_double, ct.c_double,
                                   ct.POINTER(ct.c_int64), _vp]),
    "gsr_shard_phase": (ct.c_int, [_vp, ct.POINTER(ct.c_int64), ct.POINTER(ct.c_int32), _vp]),
    "gsr_shard_poll": (ct.c_int, [_vp, ct.POINTER(ct.c_int32), ct.POINTER(_Result), _vp]),
    "gsr_launch_count": (ct.c_int, [_vp, ct.POINTER(ct.c_int64)]),
    "gsr_profile": (ct.c_int, [_vp, ct.c_int]),
    "gsr_profile_get": (ct.c_int, [_vp, ct.c_int, ct.POINTER(ct.c_double), ct.POINTER(ct.c_int64)]),
    "gsr_set_option": (ct.c_int, [_vp, ct.c_char_p, ct.c_int64]),
    "gsr_instr_acc_info": (ct.c_int, [_vp, ct.POINTER(ct.c_int32)]),
    "gsr_strerror": (ct.c_char_p, [ct.c_int]),
    "gsr_last_cuda_error": (ct.c_char_p, []),
    "gsr_version": (ct.c_char_p, []),
}


def lib_path() -> str:
    return _SO


def lib():
    """Load libgsr.so (built in-tree by paper_2503_22863_b200/build.py).  Fails loudly if absent."""
    global _lib
    if _lib is None:
        if not os.path.exists(_SO):
            raise ImportError(f"{_SO} is not built: run `python -m paper_2503_22863_b200.build` "
                              "(or __graft_entry__.build()); there is no CPU fallback")
        L = ct.CDLL(_SO)
        for name, (res, args) in SYMBOLS.items():
            f = getattr(L, name)
            f.restype, f.argtypes = res, args
        _lib = L
    return _lib


def _check(rc, where):
    if rc != GSR_OK:
        raise GsrError(rc, where)


def _dev_ptr(t, dtype, numel, name):
    import torch
    if t is None:
        return None
    if not isinstance(t, torch.Tensor) or not t.is_cuda:
        raise TypeError(f"{name}: expected a CUDA tensor (no CPU fallback)")
    if t.dtype != dtype or not t.is_contiguous() or t.numel() != numel:
        raise ValueError(f"{name}: need contiguous {dtype} with {numel} elements, got {t.dtype} {tuple(t.shape)}")
    return t.data_ptr()


def _stream():
    import torch
    return torch.cuda.current_stream().cuda_stream


def _result(r: _Result) -> LsqrResult:
    return LsqrResult(*(getattr(r, k) for k, _ in _Result._fields_))


def gsr_version() -> str:
    return lib().gsr_version().decode()


class GsrSystem:
    """Handle of a system bound to its device-resident matrix (gsr_create ... gsr_destroy).

    values: CUDA float64 [M,24]; indices: CUDA int32 [M,8] -- borrowed, kept alive by this object."""

    def __init__(self, n_stars, n_knots, n_instr, n_glob, values, indices, trusted=False, coeffs_per_row=24):
        import torch
        m = int(values.shape[0]) if values is not None else 0
        if coeffs_per_row not in (23, 24):
            raise ValueError("coeffs_per_row must be 24 or 23")
        self.coeffs_per_row = int(coeffs_per_row)
        self.layout = _Layout(m, int(n_stars), int(n_knots), int(n_instr), int(n_glob),
                              (GSR_LAYOUT_TRUSTED if trusted else 0) | (GSR_LAYOUT_COEFF23 if coeffs_per_row == 23 else 0))
        self._values, self._indices = values, indices
        self._h = _vp()
        vp = _dev_ptr(values, torch.float64, m * self.coeffs_per_row, "values")
        ip = _dev_ptr(indices, torch.int32, m * 8, "indices")
        _check(lib().gsr_create(ct.byref(self._h), ct.byref(self.layout), vp, ip, _stream()), "gsr_create")
        mm, nn = ct.c_int64(), ct.c_int64()
        _check(lib().gsr_dims(self._h, ct.byref(mm), ct.byref(nn)), "gsr_dims")
        self.n_rows, self.n_unknowns = mm.value, nn.value

    # -- lifetime
    def destroy(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            lib().gsr_destroy(self._h)
            self._h = _vp()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.destroy()

    def attach_constraints(self, values, indices):
        """The constraint equations as a section of their own (rows after the observation rows); None detaches."""
        import torch
        m = int(values.shape[0]) if values is not None else 0
        _check(lib().gsr_attach_constraints(self._h, m, _dev_ptr(values, torch.float64, m * self.coeffs_per_row, "values"),
                                            _dev_ptr(indices, torch.int32, m * 8, "indices"), _stream()),
               "gsr_attach_constraints")
        self._con_refs = (values, indices)      # borrowed: keep alive
        mm, nn = ct.c_int64(), ct.c_int64()
        _check(lib().gsr_dims(self._h, ct.byref(mm), ct.byref(nn)), "gsr_dims")
        self.n_rows = mm.value

    # -- products
    def aprod1(self, x, y):
        """y += A x   (Eq. 2)"""
        import torch
        _check(lib().gsr_aprod1(self._h, _dev_ptr(x, torch.float64, self.n_unknowns, "x"),
                                _dev_ptr(y, torch.float64, self.n_rows, "y"), _stream()), "gsr_aprod1")
        return y

    def aprod2(self, y, x):
        """x += A^T y   (Eq. 3)"""
        import torch
        _check(lib().gsr_aprod2(self._h, _dev_ptr(y, torch.float64, self.n_rows, "y"),
                                _dev_ptr(x, torch.float64, self.n_unknowns, "x"), _stream()), "gsr_aprod2")
        return x

    # -- LSQR
    def lsqr(self, b, x, itnlim, atol=0.0, btol=0.0, conlim=0.0) -> LsqrResult:
        import torch
        r = _Result()
        _check(lib().gsr_lsqr(self._h, _dev_ptr(b, torch.float64, self.n_rows, "b"),
                              _dev_ptr(x, torch.float64, self.n_unknowns, "x"), int(itnlim), float(atol),
                              float(btol), float(conlim), ct.byref(r), _stream()), "gsr_lsqr")
        return _result(r)

    def lsqr_ex(self, b, x, var=None, precond=False, itnlim=0, atol=0.0, btol=0.0, conlim=0.0) -> LsqrResult:
        import torch
        r = _Result()
        _check(lib().gsr_lsqr_ex(self._h, _dev_ptr(b, torch.float64, self.n_rows, "b"),
                                 _dev_ptr(x, torch.float64, self.n_unknowns, "x"),
                                 _dev_ptr(var, torch.float64, self.n_unknowns, "var") if var is not None else None,
                                 GSR_PRECOND_COLNORM if precond else 0, int(itnlim), float(atol), float(btol),
                                 float(conlim), ct.byref(r), _stream()), "gsr_lsqr_ex")
        return _result(r)

    def set_cov_pairs(self, j1, j2, cov):
        """Register (or, with j1 = None, unregister) the covariance pairs; the three tensors are borrowed."""
        import torch
        if j1 is None:
            _check(lib().gsr_set_cov_pairs(self._h, None, None, 0, None, _stream()), "gsr_set_cov_pairs")
            self._cov_refs = None
            return
        n = int(j1.numel())
        _check(lib().gsr_set_cov_pairs(self._h, _dev_ptr(j1, torch.int64, n, "j1"), _dev_ptr(j2, torch.int64, n, "j2"),
                                       n, _dev_ptr(cov, torch.float64, n, "cov"), _stream()), "gsr_set_cov_pairs")
        self._cov_refs = (j1, j2, cov)      # keep the borrowed tensors alive

    def colnorms(self, out):
        import torch
        _check(lib().gsr_colnorms(self._h, _dev_ptr(out, torch.float64, self.n_unknowns, "out"), _stream()),
               "gsr_colnorms")
        return out

    def lsqr_init(self, b):
        import torch
        _check(lib().gsr_lsqr_init(self._h, _dev_ptr(b, torch.float64, self.n_rows, "b"), _stream()),
               "gsr_lsqr_init")

    def lsqr_iterate(self, n_iters, itnlim=2 ** 62, atol=0.0, btol=0.0, conlim=0.0):
        _check(lib().gsr_lsqr_iterate(self._h, int(n_iters), int(itnlim), float(atol), float(btol),
                                      float(conlim), _stream()), "gsr_lsqr_iterate")

    def lsqr_result(self, x=None) -> LsqrResult:
        import torch
        r = _Result()
        _check(lib().gsr_lsqr_result_get(self._h, _dev_ptr(x, torch.float64, self.n_unknowns, "x"),
                                         ct.byref(r), _stream()), "gsr_lsqr_result_get")
        return _result(r)

    def lsqr_state(self, u=None, v=None, w=None, x=None) -> dict:
        import torch
        sc = _Scalars()
        _check(lib().gsr_lsqr_get_state(self._h, _dev_ptr(u, torch.float64, self.n_rows, "u"),
                                        _dev_ptr(v, torch.float64, self.n_unknowns, "v"),
                                        _dev_ptr(w, torch.float64, self.n_unknowns, "w"),
                                        _dev_ptr(x, torch.float64, self.n_unknowns, "x"),
                                        ct.byref(sc), _stream()), "gsr_lsqr_get_state")
        return {k: getattr(sc, k) for k, _ in _Scalars._fields_}

    # -- row-sharded solve in phases (gsr_shard_*; driven by sharded.ShardedLsqr)
    def shard_exchange_len(self) -> int:
        n = ct.c_int64()
        _check(lib().gsr_shard_exchange_len(self._h, ct.byref(n)), "gsr_shard_exchange_len")
        return n.value

    def exchange_buffer(self):
        """A device buffer of the size gsr_shard_begin wants (device memory: PyTorch's part of the job)."""
        import torch
        return torch.zeros(self.shard_exchange_len(), dtype=torch.float64, device="cuda")

    def shard_begin(self, b, xbuf, counts_shared, itnlim, atol=0.0, btol=0.0, conlim=0.0) -> int:
        import torch
        cnt = ct.c_int64()
        _check(lib().gsr_shard_begin(self._h, _dev_ptr(b, torch.float64, self.n_rows, "b"),
                                     _dev_ptr(xbuf, torch.float64, self.shard_exchange_len(), "xbuf"),
                                     int(bool(counts_shared)), int(itnlim), float(atol), float(btol), float(conlim),
                                     ct.byref(cnt), _stream()), "gsr_shard_begin")
        self._shard_refs = (b, xbuf)        # borrowed: keep alive
        return cnt.value

    def shard_phase(self):
        cnt, status = ct.c_int64(), ct.c_int32()
        _check(lib().gsr_shard_phase(self._h, ct.byref(cnt), ct.byref(status), _stream()), "gsr_shard_phase")
        return cnt.value, status.value

    def shard_poll(self):
        stopped, r = ct.c_int32(), _Result()
        _check(lib().gsr_shard_poll(self._h, ct.byref(stopped), ct.byref(r), _stream()), "gsr_shard_poll")
        return bool(stopped.value), _result(r)

    # -- diagnostics
    def launch_count(self) -> int:
        n = ct.c_int64()
        _check(lib().gsr_launch_count(self._h, ct.byref(n)), "gsr_launch_count")
        return n.value

    def profile(self, enable: bool):
        _check(lib().gsr_profile(self._h, int(bool(enable))), "gsr_profile")

    def profile_get(self, which: int):
        ms, cnt = ct.c_double(), ct.c_int64()
        _check(lib().gsr_profile_get(self._h, int(which), ct.byref(ms), ct.byref(cnt)), "gsr_profile_get")
        return ms.value, cnt.value

    def instr_acc_info(self) -> dict:
        a = (ct.c_int32 * 5)()
        _check(lib().gsr_instr_acc_info(self._h, a), "gsr_instr_acc_info")
        return {"two_dies": bool(a[0]), "copies_per_die": a[1], "chunks_per_copy": a[2], "sms_die0": a[3], "sms_die1": a[4]}

    def set_option(self, name: str, value: int):
        _check(lib().gsr_set_option(self._h, name.encode(), int(value)), "gsr_set_option")


# ---- free functions with the C names ----------------------------------------------------------
def gsr_create(n_stars, n_knots, n_instr, n_glob, values, indices, trusted=False, coeffs_per_row=24) -> GsrSystem:
    """trusted=True sets GSR_LAYOUT_TRUSTED (the caller vouches for the index records; no validation pass);
    coeffs_per_row=23 sets GSR_LAYOUT_COEFF23 (values is [M, 23], n_glob must be 0)."""
    return GsrSystem(n_stars, n_knots, n_instr, n_glob, values, indices, trusted, coeffs_per_row)


def gsr_attach_constraints(sys: GsrSystem, values, indices):
    sys.attach_constraints(values, indices)


def gsr_destroy(sys: GsrSystem):
    sys.destroy()


def gsr_aprod1(sys: GsrSystem, x, y):
    return sys.aprod1(x, y)


def gsr_aprod2(sys: GsrSystem, y, x):
    return sys.aprod2(y, x)


def gsr_lsqr(sys: GsrSystem, b, x, itnlim, atol=0.0, btol=0.0, conlim=0.0) -> LsqrResult:
    return sys.lsqr(b, x, itnlim, atol, btol, conlim)


def _host_ptr(a, np_dtype, numel, name):
    """Host buffer: numpy array or CPU torch tensor (pinned or pageable)."""
    import numpy as np
    try:
        import torch
        if isinstance(a, torch.Tensor):
            if a.is_cuda:
                raise TypeError(f"{name}: gsr_lsqr_host takes HOST buffers")
            want = {np.dtype(np.float64): torch.float64, np.dtype(np.int32): torch.int32}[np.dtype(np_dtype)]
            if a.dtype != want or not a.is_contiguous() or a.numel() != numel:
                raise ValueError(f"{name}: need a contiguous {want} host buffer of {numel} elements, "
                                 f"got {a.dtype} {tuple(a.shape)}")
            return a.data_ptr()
    except ImportError:
        pass
    if not isinstance(a, np.ndarray) or a.dtype != np_dtype or not a.flags.c_contiguous or a.size != numel:
        raise ValueError(f"{name}: need a C-contiguous {np_dtype} host array of {numel} elements")
    return a.ctypes.data


def gsr_lsqr_host(n_stars, n_knots, n_instr, n_glob, values, indices, b, x, itnlim, atol=0.0, btol=0.0,
                  conlim=0.0, coeffs_per_row=24) -> LsqrResult:
    """Whole solve from HOST buffers (H2D copies, create, LSQR, D2H of x inside the call)."""
    import numpy as np
    m = int(values.shape[0])
    L = _Layout(m, int(n_stars), int(n_knots), int(n_instr), int(n_glob),
                GSR_LAYOUT_COEFF23 if coeffs_per_row == 23 else 0)
    n = 5 * L.n_stars + 3 * L.n_knots + L.n_instr + L.n_glob
    r = _Result()
    _check(lib().gsr_lsqr_host(ct.byref(L), _host_ptr(values, np.float64, m * int(coeffs_per_row), "values"),
                               _host_ptr(indices, np.int32, m * 8, "indices"),
                               _host_ptr(b, np.float64, m, "b"), _host_ptr(x, np.float64, n, "x"),
                               int(itnlim), float(atol), float(btol), float(conlim), ct.byref(r)),
           "gsr_lsqr_host")
    return _result(r)
