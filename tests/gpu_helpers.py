"""Helpers shared by the GPU parity tests: LSQR state transfer between the library and the oracle, and the
one-iteration replay (reading R16 (iii)).  Test-side only; no library or oracle arithmetic here."""
import numpy as np
import torch

import oracle

DEV = "cuda"


def gpu_state(s, m, n):
    """(vectors as numpy, scalars as dict) of the library's LSQR state, in the API layout."""
    u = torch.empty(m, dtype=torch.float64, device=DEV)
    v, w, x = (torch.empty(n, dtype=torch.float64, device=DEV) for _ in range(3))
    sc = s.lsqr_state(u, v, w, x)
    out = {}
    for k, t in (("u", u), ("v", v), ("w", w), ("x", x)):
        out[k] = t.cpu().numpy()
    del u, v, w, x
    return out, sc


def oracle_state_from(vecs, sc, m, n, copy=True):
    """An oracle LsqrState holding the given vectors (copied unless copy=False) and scalars."""
    st = oracle.LsqrState(m, n)
    for k in ("u", "v", "w", "x"):
        if copy:
            getattr(st, k)[:] = vecs[k]
        else:
            setattr(st, k, np.ascontiguousarray(vecs[k], dtype=np.float64))
    for k, val in sc.items():
        setattr(st, k, val)
    return st


SCALARS = ("alpha", "beta", "rhobar", "phibar", "rnorm", "arnorm", "anorm", "acond", "ddnorm", "xnorm",
           "xxnorm", "z", "cs2", "sn2", "bnorm")


def replay_one_step(shape, a, idx, s, tol_vec=1e-11, tol_sc=1e-10, threads=1, lean=False):
    """GPU state at k -> one ORACLE iteration -> must equal the GPU state at k+1.
    lean=True hands the copied-back vectors to the oracle without a second host copy and compares
    vector by vector (for systems whose M-vectors are gigabytes).  Returns the worst relative errors."""
    L = oracle.layout_of(shape)
    m, n = a.shape[0], shape.n_unknowns
    vecs, sc = gpu_state(s, m, n)
    st = oracle_state_from(vecs, sc, m, n, copy=not lean)
    del vecs
    oracle.lsqr_step(L, a, idx, st, threads=threads)
    s.lsqr_iterate(1)
    vecs1, sc1 = gpu_state(s, m, n)
    assert sc1["itn"] == st.itn
    worst = {}
    for k in ("u", "v", "w", "x"):
        ref = getattr(st, k)
        got = vecs1.pop(k)
        num = np.linalg.norm(np.subtract(got, ref, out=got))     # in place on the GPU copy: no third M-vector
        e = num / np.linalg.norm(ref)
        assert e <= tol_vec, f"one-step replay at itn {st.itn}: vector {k} off by {e:.3e}"
        worst[k] = float(e)
        del got
    for k in SCALARS:
        ref = getattr(st, k)
        assert abs(sc1[k] - ref) <= tol_sc * abs(ref) + 1e-300, f"one-step replay at itn {st.itn}: {k} {sc1[k]} vs {ref}"
        worst[k] = abs(sc1[k] - ref) / (abs(ref) + 1e-300)
    return worst
