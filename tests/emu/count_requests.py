"""Static request count of the matrix kernels, from their own source on the host emulation (tests/emu).

For one launch of a kernel on a small system of a given SHAPE (K, I as at C4 by default), every global-memory access
the kernel source makes through a hooked path -- read-only gathers (`__ldg`), fp64 reductions (`red.global.add.f64`,
emulated by atomicAdd), TMA / bulk copies -- is logged per thread and grouped per warp instruction; for each
instruction the distinct 128-byte lines (what one warp-wide request to L2 covers at most) and 32-byte sectors are
counted and charged to the class of memory it addresses.  Plain loads / stores (u of the next tile, the u store)
are not hooked: they are one coalesced 8-byte-per-row stream each and are added analytically (2 lines per tile).

This is an instruction-level count from the source, not a measurement: it says nothing about L1 hits, the order of
requests or time.  Its use is to say WHERE the requests of a row come from, next to the ncu totals of
profiles/r01_fused_full_v5.md.

    python tests/emu/count_requests.py [--stars 400] [--obs 100] [--knots 1000000] [--instr 60000] [--kernel fused|aprod1|aprod2]
"""
import argparse
import ctypes as ct
import os
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(os.path.dirname(HERE))
for p in (ROOT, os.path.join(ROOT, "tests"), HERE):
    if p not in sys.path:
        sys.path.insert(0, p)

import numpy as np  # noqa: E402
import torch  # noqa: E402

import harness  # noqa: E402
from gaia_synth import host  # noqa: E402
from gaia_synth.configs import C4  # noqa: E402
from paper_2503_22863_b200 import binding  # noqa: E402

KIND = {0: "gather (LDG)", 1: "reduction (RED)", 2: "TMA / bulk copy"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--stars", type=int, default=400)
    ap.add_argument("--obs", type=int, default=100)
    ap.add_argument("--knots", type=int, default=1_000_000)
    ap.add_argument("--instr", type=int, default=60_000)
    ap.add_argument("--kernel", default="fused", choices=["fused", "aprod1", "aprod2"])
    ap.add_argument("--option", action="append", default=[])
    args = ap.parse_args()
    shape = C4.scaled(args.stars, n_knots=args.knots, n_instr=args.instr, obs_per_star=args.obs, name="C4-shaped")
    a, idx = host.make_rows(shape)
    m, n = a.shape[0], shape.n_unknowns
    with harness.emulated():
        L = binding.lib()
        L.emu_count_report.restype = ct.c_int
        L.emu_count_report.argtypes = [ct.c_char_p, ct.c_int]
        L.emu_count_region.argtypes = [ct.c_char_p, ct.c_void_p, ct.c_ulonglong]
        L.emu_count_layout.argtypes = [ct.c_ulonglong] * 5
        av, iv = harness.host_tensor(a), harness.host_tensor(idx)
        s = binding.gsr_create(shape.n_stars, shape.n_knots, shape.n_instr, shape.n_glob, av, iv)
        s.set_option("graph", 0)
        for o in args.option:
            k, v = o.split("=")
            s.set_option(k, int(v))
        x = harness.host_tensor(host.test_vector(1, 1, n))
        y = harness.host_tensor(host.test_vector(1, 2, m))
        if args.kernel == "fused":
            s.lsqr_init(y)
            s.lsqr_iterate(1)                               # warm: workspace allocated
        L.emu_count_reset()
        L.emu_count_layout(n * 8, shape.off_att * 8, shape.off_instr * 8, shape.off_glob * 8, m * 8)
        L.emu_count_region(b"A: coefficient records", av.data_ptr(), av.numel() * 8)
        L.emu_count_region(b"A: index records", iv.data_ptr(), iv.numel() * 4)
        L.emu_count_region(b"caller's x", x.data_ptr(), n * 8)
        L.emu_count_region(b"caller's y", y.data_ptr(), m * 8)
        L.emu_count_enable(1)
        if args.kernel == "fused":
            s.lsqr_iterate(1)
        elif args.kernel == "aprod1":
            s.aprod1(x, y)
        else:
            s.aprod2(y, x)
        L.emu_count_enable(0)
        buf = ct.create_string_buffer(1 << 16)
        assert L.emu_count_report(buf, len(buf)) >= 0
        s.destroy()
    rows = []
    for line in buf.value.decode().splitlines():
        kind, rest = line.split(" ", 1)
        cls, instr, lanes, lines, sectors = rest.rsplit(" ", 4)
        rows.append((int(kind), cls, int(instr), int(lanes), int(lines), int(sectors)))
    print(f"{args.kernel}: {m} rows ({m // 32} tiles), K = {shape.n_knots}/axis, I = {shape.n_instr}, options {args.option}")
    print("| access | memory | warp instructions / row | lanes / row | 128-byte lines (requests) / row | 32-byte sectors / row |")
    print("|---|---|---|---|---|---|")
    tot = {}
    outside = []
    for kind, cls, instr, lanes, lines, sectors in sorted(rows):
        if cls.startswith("[outside the row loop]"):      # kernel prologues / epilogues and the n-length kernels of the call
            outside.append(f"{KIND[kind]} of {cls[23:]}: {lines} lines in all")
            continue
        print(f"| {KIND[kind]} | {cls} | {instr / m:.3f} | {lanes / m:.2f} | {lines / m:.3f} | {sectors / m:.3f} |")
        t = tot.setdefault(kind, [0, 0, 0, 0])
        for i, v in enumerate((instr, lanes, lines, sectors)):
            t[i] += v
    for kind, t in sorted(tot.items()):
        print(f"| **{KIND[kind]}, all** | | {t[0] / m:.3f} | {t[1] / m:.2f} | **{t[2] / m:.3f}** | {t[3] / m:.3f} |")
    print("| plain loads + stores of the M-vector (not hooked; coalesced, 2 lines per tile each) | M-vector | 0.062 | 2.00 | 0.125 | 0.500 |")
    if outside:
        print("not per row (prologues, epilogues, the n-length kernels of the same call; n = %d): " % n + "; ".join(outside))


if __name__ == "__main__":
    main()
