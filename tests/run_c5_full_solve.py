#!/usr/bin/env python
"""C5 at full size (BASELINE.json configs[4]): 2e6 stars x 80 obs = 1.6e8 rows + 10,000 constraint rows,
LSQR run to convergence (atol = btol = 1e-12, conlim = 1e8) on the GPU and by the CPU oracle (OpenMP,
deterministic for a fixed thread count), solutions compared (reading R16
of DESIGN.md: x at convergence <= 1e-9, istop equal, itn within +-max(3, 5 %)).

Too long for pytest (the oracle needs ~20 min on 16 cores and ~45 GB of host memory), so it is a script:

    python tests/run_c5_full_solve.py [--stars N] [--out report.md]

`--stars` scales the system down (K, I and the constraint rows scale with it) for a quick run.
The system is generated once, on the device; the oracle is fed the same bytes copied back.
"""
import argparse
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--stars", type=int, default=0)
    ap.add_argument("--out", default="")
    ap.add_argument("--itnlim", type=int, default=5000)
    args = ap.parse_args()

    import torch

    import oracle
    import paper_2503_22863_b200 as gsr
    from gaia_synth import device as gdev
    from gaia_synth.configs import C5

    shape = C5
    if args.stars:
        f = args.stars / C5.n_stars
        shape = C5.scaled(args.stars, n_knots=max(int(C5.n_knots * f), 8), n_instr=max(int(C5.n_instr * f), 8),
                          n_constraint_rows=max(int(C5.n_constraint_rows * f), 2))
    lines = []

    def say(s):
        print(s, flush=True)
        lines.append(s)

    vals, idx = gdev.make_system(shape)
    s = gsr.gsr_create(shape.n_stars, shape.n_knots, shape.n_instr, shape.n_glob, vals, idx)
    m, n = s.n_rows, s.n_unknowns
    say(f"system: {shape.name} S={shape.n_stars} K={shape.n_knots}/axis I={shape.n_instr} G={shape.n_glob} "
        f"constraint rows={shape.n_constraint_rows}: M={m} n={n}")
    xt = gdev.x_true(shape)
    b = gdev.noise(shape, m)
    s.aprod1(xt, b)                     # b = A x_true + N(0, 1e-6); aprod 1 parity at this size: tests/test_gpu_fullsize.py
    x = torch.empty(n, dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    res = s.lsqr(b, x, args.itnlim, 1e-12, 1e-12, 1e8)
    torch.cuda.synchronize()
    t_gpu = time.perf_counter() - t0
    say(f"GPU   : istop={res.istop} itn={res.itn} r1norm={res.r1norm:.9e} anorm={res.anorm:.6e} acond={res.acond:.6e} "
        f"arnorm={res.arnorm:.3e} xnorm={res.xnorm:.9e}  ({t_gpu:.2f} s, {1e3 * t_gpu / max(res.itn, 1):.2f} ms/iteration)")
    xg = x.cpu().numpy()
    # residual identity on the device: ||b - A x|| against the recurrence's r1norm
    r = b.clone()
    s.aprod1(-x, r)
    rn = float(torch.linalg.norm(r))
    say(f"GPU   : ||b - A x|| = {rn:.9e}  (recurrence {res.r1norm:.9e}, rel. diff {abs(rn - res.r1norm) / rn:.2e})")
    xth = xt.cpu().numpy()
    a_h, idx_h, b_h = vals.cpu().numpy(), idx.cpu().numpy(), b.cpu().numpy()
    s.destroy()
    del vals, idx, b, x, r, xt
    torch.cuda.empty_cache()

    L = oracle.layout_of(shape)
    th = oracle.max_threads()
    t0 = time.perf_counter()
    xo, ro = oracle.lsqr(L, a_h, idx_h, b_h, itnlim=args.itnlim, atol=1e-12, btol=1e-12, conlim=1e8, threads=th)
    t_cpu = time.perf_counter() - t0
    say(f"oracle: istop={ro['istop']} itn={ro['itn']} r1norm={ro['r1norm']:.9e} anorm={ro['anorm']:.6e} acond={ro['acond']:.6e} "
        f"arnorm={ro['arnorm']:.3e} xnorm={ro['xnorm']:.9e}  ({t_cpu:.1f} s on {th} threads, "
        f"{1e3 * t_cpu / max(ro['itn'], 1):.0f} ms/iteration)")
    err = float(np.linalg.norm(xg - xo) / np.linalg.norm(xo))
    say(f"||x_gpu - x_oracle|| / ||x_oracle|| = {err:.3e}   (bar 1e-9)")
    # columns no row touches (reading R3: knot K-1 of each axis) stay exactly 0 on both sides
    empty = [shape.off_att + ax * shape.n_knots + shape.n_knots - 1 for ax in range(3)]
    say(f"empty attitude columns: gpu {[float(xg[c]) for c in empty]} oracle {[float(xo[c]) for c in empty]}")
    mask = np.ones(n, dtype=bool)
    mask[empty] = False
    e_true = float(np.linalg.norm((xg - xth)[mask]) / np.linalg.norm(xth[mask]))
    say(f"||x_gpu - x_true|| / ||x_true|| on the other columns = {e_true:.3e}")
    ok = (err <= 1e-9 and res.istop == ro["istop"] and abs(res.itn - ro["itn"]) <= max(3, 0.05 * ro["itn"])
          and abs(rn - res.r1norm) <= 1e-8 * rn)
    say("PASS" if ok else "FAIL")
    if args.out:
        with open(args.out, "w") as f:
            f.write("\n".join(lines) + "\n")
    return 0 if ok else 1


if __name__ == "__main__":
    sys.exit(main())
