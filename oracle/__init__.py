"""ctypes binding of the CPU oracle (oracle/gsr_oracle.c).  TEST INFRASTRUCTURE ONLY.

Importable only from tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs.  The product package never imports this module.
"""
import ctypes as ct
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libgsr_oracle.so")
_SRC = os.path.join(_HERE, "gsr_oracle.c")
_HDR = os.path.join(_HERE, "gsr_oracle.h")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain C, no FMA contraction).  GSR_ORACLE_SANITIZE=1 builds and loads an
    AddressSanitizer + UBSan variant instead (run the tests with LD_PRELOAD=$(gcc -print-file-name=libasan.so))."""
    global _SO
    flags = ["-O2"]
    if os.environ.get("GSR_ORACLE_SANITIZE", "0") == "1":
        _SO = os.path.join(_HERE, "libgsr_oracle_asan.so")
        flags = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"]
    if not force and os.path.exists(_SO) and os.path.getmtime(_SO) >= max(
            os.path.getmtime(_SRC), os.path.getmtime(_HDR)):
        return _SO
    tmp = _SO + ".tmp%d" % os.getpid()
    subprocess.check_call(["gcc"] + flags + ["-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
                           "-Wall", "-o", tmp, _SRC, "-lm"])
    os.replace(tmp, _SO)
    return _SO


class Layout(ct.Structure):
    _fields_ = [("n_stars", ct.c_int64), ("n_knots", ct.c_int64), ("n_instr", ct.c_int64),
                ("n_glob", ct.c_int32), ("coeffs_per_row", ct.c_int32)]


class LsqrResult(ct.Structure):
    _fields_ = [("istop", ct.c_int32), ("itn", ct.c_int64), ("r1norm", ct.c_double),
                ("r2norm", ct.c_double), ("anorm", ct.c_double), ("acond", ct.c_double),
                ("arnorm", ct.c_double), ("xnorm", ct.c_double), ("bnorm", ct.c_double)]

    def asdict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


_lib = None
_dp = ct.POINTER(ct.c_double)
_ip = ct.POINTER(ct.c_int32)

_STATE_SCALARS = ("alpha", "beta", "rhobar", "phibar", "bnorm", "rnorm", "arnorm", "anorm",
                  "acond", "ddnorm", "xnorm", "xxnorm", "z", "cs2", "sn2")


class _CState(ct.Structure):
    _fields_ = ([("itn", ct.c_int64), ("istop", ct.c_int32)] +
                [(k, ct.c_double) for k in _STATE_SCALARS] +
                [("u", _dp), ("v", _dp), ("w", _dp), ("x", _dp)])


class LsqrState:
    """LSQR state: normalised u (m), v, w, x (n) and the scalar recurrences."""

    def __init__(self, m, n):
        self.u = np.zeros(m)
        self.v = np.zeros(n)
        self.w = np.zeros(n)
        self.x = np.zeros(n)
        self.itn = 0
        self.istop = 0
        for k in _STATE_SCALARS:
            setattr(self, k, 0.0)

    def _to_c(self):
        c = _CState()
        c.itn, c.istop = int(self.itn), int(self.istop)
        for k in _STATE_SCALARS:
            setattr(c, k, float(getattr(self, k)))
        c.u, c.v, c.w, c.x = _d(self.u), _d(self.v), _d(self.w), _d(self.x)
        return c

    def _from_c(self, c):
        self.itn, self.istop = int(c.itn), int(c.istop)
        for k in _STATE_SCALARS:
            setattr(self, k, float(getattr(c, k)))

    def scalars(self):
        d = {k: getattr(self, k) for k in _STATE_SCALARS}
        d.update(itn=self.itn, istop=self.istop)
        return d


def lib():
    global _lib
    if _lib is None:
        L = ct.CDLL(build())
        LP = ct.POINTER(Layout)
        L.orc_n_unknowns.restype = ct.c_int64
        L.orc_n_unknowns.argtypes = [LP]
        L.orc_col.restype = ct.c_int64
        L.orc_col.argtypes = [LP, _ip, ct.c_int]
        L.orc_aprod1.restype = None
        L.orc_aprod1.argtypes = [LP, ct.c_int64, _dp, _ip, _dp, _dp]
        L.orc_aprod2.restype = None
        L.orc_aprod2.argtypes = [LP, ct.c_int64, _dp, _ip, _dp, _dp]
        L.orc_aprod2_comp.restype = None
        L.orc_aprod2_comp.argtypes = [LP, ct.c_int64, _dp, _ip, _dp, _dp, _dp]
        L.orc_aprod1_abs.restype = None
        L.orc_aprod1_abs.argtypes = [LP, ct.c_int64, _dp, _ip, _dp, _dp, _dp]
        L.orc_aprod1_omp.restype = None
        L.orc_aprod1_omp.argtypes = [LP, ct.c_int64, _dp, _ip, _dp, _dp, ct.c_int]
        L.orc_aprod2_omp.restype = None
        L.orc_aprod2_omp.argtypes = [LP, ct.c_int64, _dp, _ip, _dp, _dp, ct.c_int]
        L.orc_lsqr.restype = ct.c_int
        L.orc_lsqr.argtypes = [LP, ct.c_int64, _dp, _ip, _dp, _dp, ct.c_int64, ct.c_double,
                               ct.c_double, ct.c_double, ct.c_int, ct.POINTER(LsqrResult), _dp, _dp]
        L.orc_colnorm2.restype = None
        L.orc_colnorm2.argtypes = [LP, ct.c_int64, _dp, _ip, _dp]
        L.orc_scale_columns.restype = None
        L.orc_scale_columns.argtypes = [LP, ct.c_int64, _dp, _ip, _dp, _dp]
        L.orc_max_threads.restype = ct.c_int
        SP = ct.POINTER(_CState)
        L.orc_lsqr_init.restype = None
        L.orc_lsqr_init.argtypes = [LP, ct.c_int64, _dp, _ip, _dp, ct.c_int, SP]
        L.orc_lsqr_step.restype = None
        L.orc_lsqr_step.argtypes = [LP, ct.c_int64, _dp, _ip, ct.c_int64, ct.c_double, ct.c_double,
                                    ct.c_double, ct.c_int, SP]
        _lib = L
    return _lib


def max_threads() -> int:
    return int(lib().orc_max_threads())


def _d(a):
    assert a.dtype == np.float64 and a.flags.c_contiguous
    return a.ctypes.data_as(_dp)


def _i(a):
    assert a.dtype == np.int32 and a.flags.c_contiguous
    return a.ctypes.data_as(_ip)


def layout(n_stars, n_knots, n_instr, n_glob=1, coeffs_per_row=24) -> Layout:
    """coeffs_per_row = 23: the production record without the global slot (needs n_glob = 0)."""
    assert coeffs_per_row in (23, 24) and (coeffs_per_row == 24 or n_glob == 0)
    return Layout(int(n_stars), int(n_knots), int(n_instr), int(n_glob), int(coeffs_per_row))


def layout_of(shape) -> Layout:
    """Layout from a gaia_synth SystemShape."""
    return layout(shape.n_stars, shape.n_knots, shape.n_instr, shape.n_glob)


def n_unknowns(L: Layout) -> int:
    return int(lib().orc_n_unknowns(ct.byref(L)))


def col(L: Layout, rec: np.ndarray, k: int) -> int:
    rec = np.ascontiguousarray(rec, dtype=np.int32)
    return int(lib().orc_col(ct.byref(L), _i(rec), k))


def _check(L, a, idx):
    m = a.shape[0]
    assert a.shape == (m, 23 if L.coeffs_per_row == 23 else 24) and idx.shape == (m, 8)
    return m


def aprod1(L, a, idx, x, y, threads=1):
    """y += A x  (in place on y).  PAPER.md:45 Eq. 2."""
    m = _check(L, a, idx)
    assert x.shape == (n_unknowns(L),) and y.shape == (m,)
    if threads <= 1:
        lib().orc_aprod1(ct.byref(L), m, _d(a), _i(idx), _d(x), _d(y))
    else:
        lib().orc_aprod1_omp(ct.byref(L), m, _d(a), _i(idx), _d(x), _d(y), threads)
    return y


def aprod2(L, a, idx, y, x, threads=1):
    """x += A^T y  (in place on x).  PAPER.md:49 Eq. 3."""
    m = _check(L, a, idx)
    assert x.shape == (n_unknowns(L),) and y.shape == (m,)
    if threads <= 1:
        lib().orc_aprod2(ct.byref(L), m, _d(a), _i(idx), _d(y), _d(x))
    else:
        lib().orc_aprod2_omp(ct.byref(L), m, _d(a), _i(idx), _d(y), _d(x), threads)
    return x


def aprod2_comp(L, a, idx, y, x, comp):
    m = _check(L, a, idx)
    lib().orc_aprod2_comp(ct.byref(L), m, _d(a), _i(idx), _d(y), _d(x), _d(comp))
    return x


def aprod1_abs(L, a, idx, x, y_in=None):
    m = _check(L, a, idx)
    s = np.empty(m, dtype=np.float64)
    lib().orc_aprod1_abs(ct.byref(L), m, _d(a), _i(idx), _d(x),
                         _d(y_in) if y_in is not None else None, _d(s))
    return s


def lsqr(L, a, idx, b, itnlim, atol=0.0, btol=0.0, conlim=0.0, threads=1, history=False):
    """Paige-Saunders LSQR (damp=0).  Returns (x, result dict[, rnorm_hist, arnorm_hist])."""
    m = _check(L, a, idx)
    n = n_unknowns(L)
    x = np.zeros(n, dtype=np.float64)
    res = LsqrResult()
    rh = np.zeros(itnlim + 1) if history else None
    ah = np.zeros(itnlim + 1) if history else None
    rc = lib().orc_lsqr(ct.byref(L), m, _d(a), _i(idx), _d(b), _d(x), int(itnlim), float(atol),
                        float(btol), float(conlim), int(threads), ct.byref(res),
                        _d(rh) if history else None, _d(ah) if history else None)
    if rc != 0:
        raise MemoryError("orc_lsqr allocation failed")
    out = res.asdict()
    if history:
        k = out["itn"] + 1
        return x, out, rh[:k], ah[:k]
    return x, out


def colnorms(L, a, idx):
    """2-norm of every column of A; 0 for a column no row touches."""
    m = _check(L, a, idx)
    sq = np.zeros(n_unknowns(L), dtype=np.float64)
    lib().orc_colnorm2(ct.byref(L), m, _d(a), _i(idx), _d(sq))
    return np.sqrt(sq)


def scale_columns(L, a, idx, s):
    """The coefficient records of A diag(s)."""
    m = _check(L, a, idx)
    out = np.empty_like(a)
    lib().orc_scale_columns(ct.byref(L), m, _d(a), _i(idx), _d(np.ascontiguousarray(s, dtype=np.float64)), _d(out))
    return out


def lsqr_var(L, a, idx, b, itnlim, atol=0.0, btol=0.0, conlim=0.0, threads=1):
    """LSQR that also returns Paige-Saunders' `var` (the diagonal of (A^T A)^-1 as estimated by the run):
    var += (w / rho)^2 at every iteration, with the w BEFORE its update and rho of that iteration's plane
    rotation, rho = sqrt(rhobar_old^2 + beta_new^2).  Written over lsqr_init / lsqr_step, so the LSQR
    arithmetic itself is the pinned one.  Returns (x, var, result dict)."""
    st = lsqr_init(L, a, idx, b, threads=threads)
    var = np.zeros_like(st.x)
    if st.arnorm == 0.0:
        st.istop = 0
    elif itnlim <= 0:
        st.istop = 7
    else:
        while st.istop == 0:
            w_old, rhobar_old = st.w.copy(), st.rhobar
            lsqr_step(L, a, idx, st, itnlim=itnlim, atol=atol, btol=btol, conlim=conlim, threads=threads)
            rho = np.sqrt(rhobar_old * rhobar_old + st.beta * st.beta)
            var += (w_old / rho) ** 2
    res = st.scalars()
    res.update(r1norm=st.rnorm, r2norm=st.rnorm)
    return st.x.copy(), var, res


def lsqr_cov(L, a, idx, b, j1, j2, itnlim, atol=0.0, btol=0.0, conlim=0.0, threads=1):
    """Covariances of chosen pairs of unknowns, Eq. (4): Cov[p] += factor^itn * x^itn[j1[p]] *
    x^itn[j2[p]] at every LSQR iteration.  Reading (R21): this is the off-diagonal companion of
    Paige-Saunders' var, i.e. x^itn is the direction w of that iteration (before its update) and factor^itn =
    1 / rho^2, so that a pair (j, j) reproduces var[j] and the sum estimates ((A^T A)^-1)[j1, j2].
    Returns (x, cov, result dict)."""
    j1 = np.asarray(j1, dtype=np.int64)
    j2 = np.asarray(j2, dtype=np.int64)
    st = lsqr_init(L, a, idx, b, threads=threads)
    cov = np.zeros(j1.shape[0], dtype=np.float64)
    if st.arnorm == 0.0:
        st.istop = 0
    elif itnlim <= 0:
        st.istop = 7
    else:
        while st.istop == 0:
            w_old, rhobar_old = st.w.copy(), st.rhobar
            lsqr_step(L, a, idx, st, itnlim=itnlim, atol=atol, btol=btol, conlim=conlim, threads=threads)
            rho = np.sqrt(rhobar_old * rhobar_old + st.beta * st.beta)
            for p in range(j1.shape[0]):
                cov[p] += (1.0 / (rho * rho)) * w_old[j1[p]] * w_old[j2[p]]
    res = st.scalars()
    res.update(r1norm=st.rnorm, r2norm=st.rnorm)
    return st.x.copy(), cov, res


def lsqr_precond(L, a, idx, b, itnlim, atol=0.0, btol=0.0, conlim=0.0, threads=1):
    """Column-norm preconditioned solve (R7): d = column 2-norms (1 where a column is empty),
    LSQR on (A D^-1) z = b, x = D^-1 z, var_x = D^-2 var_z.  Returns (x, var, result dict, d)."""
    d = colnorms(L, a, idx)
    d[d == 0.0] = 1.0
    dinv = 1.0 / d
    z, var_z, res = lsqr_var(L, scale_columns(L, a, idx, dinv), idx, b, itnlim, atol, btol, conlim, threads)
    return z * dinv, var_z * dinv * dinv, res, d


def lsqr_init(L, a, idx, b, threads=1) -> LsqrState:
    """x = 0; beta u = b; alpha v = A^T u; w = v  ("initial conditions are set with aprod 2")."""
    m = _check(L, a, idx)
    st = LsqrState(m, n_unknowns(L))
    c = st._to_c()
    lib().orc_lsqr_init(ct.byref(L), m, _d(a), _i(idx), _d(b), int(threads), ct.byref(c))
    st._from_c(c)
    return st


def lsqr_step(L, a, idx, st: LsqrState, itnlim=2 ** 62, atol=0.0, btol=0.0, conlim=0.0, threads=1):
    """One LSQR iteration in place on `st`."""
    m = _check(L, a, idx)
    c = st._to_c()
    lib().orc_lsqr_step(ct.byref(L), m, _d(a), _i(idx), int(itnlim), float(atol), float(btol),
                        float(conlim), int(threads), ct.byref(c))
    st._from_c(c)
    return st
