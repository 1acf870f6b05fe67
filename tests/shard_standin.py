"""CPU stand-in for one rank of a row-sharded solve: the phase contract of include/gsr.h (gsr_shard_begin /
gsr_shard_phase / gsr_shard_poll) with the products done by the CPU oracle on the rank's rows and the n-length steps
in numpy.  TEST-SIDE ONLY: it exists so that the host logic of paper_2503_22863_b200/sharded.py (row partition,
lock-step phase loop, what is summed over the ranks and when, one rank counting the replicated tail) runs under
gloo on a box without a GPU.  The sharded result is then compared with oracle.lsqr on the WHOLE system, so a mistake
in here fails the test like a mistake in the driver would.

The recurrences are Paige-Saunders' (paper refs [29,30]) in the lazily normalised form the phases
imply: u_hat = beta * u is kept un-normalised, g = A^T u_hat is exchanged, beta = sqrt(sum u_hat^2) afterwards.
"""
import math
from types import SimpleNamespace

import numpy as np
import torch

import oracle

MORE, INIT_DONE, ITER_DONE = 0, 1, 2


class OracleShard:
    def __init__(self, shape, a, idx):
        self.L = oracle.layout_of(shape)
        self.a, self.idx = np.ascontiguousarray(a), np.ascontiguousarray(idx)
        self.n_rows, self.n_unknowns = self.a.shape[0], shape.n_unknowns
        self.oA = shape.off_att
        self.ns = self.n_unknowns - self.oA
        self.next = -1

    # -- the ABI's shard calls
    def shard_exchange_len(self):
        return self.ns + 2

    def exchange_buffer(self):
        return torch.zeros(self.ns + 2, dtype=torch.float64)

    def shard_begin(self, b, xbuf, counts_shared, itnlim, atol=0.0, btol=0.0, conlim=0.0):
        n = self.n_unknowns
        self.xb = xbuf.numpy()                           # shares memory with the tensor the driver reduces
        self.n_sq = n if counts_shared else self.oA
        self.itnlim, self.atol, self.btol, self.conlim = itnlim, atol, btol, conlim
        self.uh = np.array(b.numpy() if isinstance(b, torch.Tensor) else b, dtype=np.float64)
        self.v, self.w, self.x, self.g = (np.zeros(n) for _ in range(4))
        self.sc = SimpleNamespace(itn=0, istop=0, done=0, usq=float(self.uh @ self.uh), vsq=0.0, wsq=0.0)
        self.xb[0] = self.sc.usq
        self.next = 1
        return 1

    def shard_phase(self):
        sc, xb, ns, oA, n_sq = self.sc, self.xb, self.ns, self.oA, self.n_sq
        st, cnt = MORE, 0
        if self.next == 1:                               # beta ; v = A^T u on this rank's rows
            sc.beta = math.sqrt(xb[0])
            sc.bnorm = sc.beta
            sc.s_y = 1.0 / sc.beta if sc.beta > 0 else 0.0
            sc.usq = 0.0
            oracle.aprod2(self.L, self.a, self.idx, self.uh * sc.s_y, self.v)
            xb[:ns] = self.v[oA:]
            cnt, self.next = ns, 2
        elif self.next == 2:                             # partial ||v||^2
            self.v[oA:] = xb[:ns]
            xb[0] = float(self.v[:n_sq] @ self.v[:n_sq])
            cnt, self.next = 1, 3
        elif self.next == 3:                             # alpha ; v /= alpha ; w = v
            alpha = math.sqrt(xb[0]) if sc.beta > 0 else 0.0
            sc.alpha = alpha
            sc.rhobar, sc.phibar, sc.rnorm, sc.arnorm = alpha, sc.beta, sc.beta, alpha * sc.beta
            sc.anorm = sc.acond = sc.ddnorm = sc.xnorm = sc.xxnorm = sc.z = sc.sn2 = 0.0
            sc.cs2 = -1.0
            sc.c0 = -alpha / sc.beta if sc.beta > 0 else 0.0
            if alpha * sc.beta == 0.0:
                sc.done = 1
            else:
                self.v /= alpha
                self.w[:] = self.v
                sc.wsq = float(self.w[:n_sq] @ self.w[:n_sq])
            st, self.next = INIT_DONE, 4
        elif self.next == 4:                             # u_hat <- A v + c0 u_hat ; g = A^T u_hat
            if not sc.done:
                self.uh *= sc.c0
                oracle.aprod1(self.L, self.a, self.idx, self.v, self.uh)
                self.g[:] = 0.0
                oracle.aprod2(self.L, self.a, self.idx, self.uh, self.g)
                xb[:ns] = self.g[oA:]
                xb[ns] = float(self.uh @ self.uh)
                xb[ns + 1] = sc.wsq
            cnt, self.next = ns + 2, 5
        elif self.next == 5:                             # beta ; v <- g / beta - beta v ; partial ||v||^2
            if not sc.done:
                self.g[oA:] = xb[:ns]
                sc.wsq_all = xb[ns + 1]
                sc.beta = math.sqrt(xb[ns])
                if sc.beta > 0:
                    sc.anorm = math.sqrt(sc.anorm ** 2 + sc.alpha ** 2 + sc.beta ** 2)
                    self.v = self.g / sc.beta - sc.beta * self.v
                    xb[0] = float(self.v[:n_sq] @ self.v[:n_sq])
                else:
                    xb[0] = 0.0
            cnt, self.next = 1, 6
        elif self.next == 6:                             # scalars, stopping rule, x / w / v update
            if not sc.done:
                self._scalars_and_update(xb[0])
            elif sc.done == 2:
                sc.done = 1
            st, self.next = ITER_DONE, 4
        else:
            raise RuntimeError("shard_phase out of order")
        return cnt, st

    def _scalars_and_update(self, vsq):
        sc, n_sq = self.sc, self.n_sq
        beta, alpha = sc.beta, sc.alpha
        if beta > 0:
            alpha = math.sqrt(vsq)
        inv_alpha = 1.0 / alpha if (beta > 0 and alpha > 0) else 1.0
        rho = math.hypot(sc.rhobar, beta)
        cs, sn = sc.rhobar / rho, beta / rho
        theta = sn * alpha
        sc.rhobar = -cs * alpha
        phi = cs * sc.phibar
        sc.phibar = sn * sc.phibar
        tau = sn * phi
        t1, t2 = phi / rho, -theta / rho
        sc.ddnorm += sc.wsq_all / (rho * rho)
        delta, gambar = sc.sn2 * rho, -sc.cs2 * rho
        rhs = phi - delta * sc.z
        zbar = rhs / gambar
        sc.xnorm = math.sqrt(sc.xxnorm + zbar * zbar)
        gamma = math.hypot(gambar, theta)
        sc.cs2, sc.sn2, sc.z = gambar / gamma, theta / gamma, rhs / gamma
        sc.xxnorm += sc.z * sc.z
        sc.acond = sc.anorm * math.sqrt(sc.ddnorm)
        sc.rnorm = abs(sc.phibar)
        sc.arnorm = alpha * abs(tau)
        sc.alpha = alpha
        sc.c0 = -alpha / beta if beta > 0 else 0.0
        sc.itn += 1
        ctol = 1.0 / self.conlim if self.conlim > 0 else 0.0
        test1 = sc.rnorm / sc.bnorm
        den2 = sc.anorm * sc.rnorm
        test2 = sc.arnorm / den2 if den2 > 0 else 0.0
        test3 = 1.0 / sc.acond
        t1p = test1 / (1.0 + sc.anorm * sc.xnorm / sc.bnorm)
        rtol = self.btol + self.atol * sc.anorm * sc.xnorm / sc.bnorm
        istop = 0
        if sc.itn >= self.itnlim: istop = 7
        if 1.0 + test3 <= 1.0: istop = 6
        if 1.0 + test2 <= 1.0: istop = 5
        if 1.0 + t1p <= 1.0: istop = 4
        if test3 <= ctol: istop = 3
        if test2 <= self.atol: istop = 2
        if test1 <= rtol: istop = 1
        sc.istop = istop
        if istop:
            sc.done = 2                                   # this iteration's update still runs
        self.v *= inv_alpha
        self.x += t1 * self.w
        self.w = self.v + t2 * self.w
        sc.wsq = float(self.w[:n_sq] @ self.w[:n_sq])

    def shard_poll(self):
        sc = self.sc
        done, istop = bool(sc.done), sc.istop
        if not done and self.itnlim == 0:
            done, istop = True, 7
        res = SimpleNamespace(istop=istop, itn=sc.itn, r1norm=sc.rnorm, r2norm=sc.rnorm, anorm=sc.anorm,
                              acond=sc.acond, arnorm=sc.arnorm, xnorm=sc.xnorm, bnorm=sc.bnorm)
        return done, res

    def lsqr_result(self, x=None):
        if x is not None:
            x.numpy()[:] = self.x
        return self.shard_poll()[1]
