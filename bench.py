#!/usr/bin/env python
"""Benchmark of the AVU-GSR hot path on B200: ms per LSQR iteration (aprod1 + aprod2 + the fused
vector work) and achieved HBM GB/s, on a synthetic Gaia-shaped system (BASELINE.json).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C4] [--impl reference]

One "step" = one LSQR iteration = one pass of the whole hot path over the system.  The system is
generated in HBM by the seeded generator before the timed region; the matrix (>= 2 GB) is far
larger than L2, so no L2 flush is needed between iterations.  Prints ONE JSON line.

Multi-GPU: the path is single-GPU by BASELINE.json:north_star ("replicas only", DESIGN.md
section 8): under torchrun every rank times its own replica of the workload; the reported time is
the max over ranks.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

NOMINAL_HBM_GBS = 8000.0          # BASELINE.json metric: "vs 8 TB/s peak"
FALLBACK_HBM_GBS = 6650.0         # B200_PROFILING.md fallback if MEASURED_PEAKS.json is absent


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default=os.environ.get("GSR_BENCH_WORKLOAD", "auto"),
                    help="C1..C5 or auto (C4, the config the 70%%-of-HBM target is quoted on, if it fits)")
    ap.add_argument("--impl", default="gsr", choices=["gsr", "reference"])
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--oracle-rows", type=int, default=0, help="rows of the oracle sample (0 = auto)")
    ap.add_argument("--option", action="append", default=[], help="name=value passed to gsr_set_option")
    ap.add_argument("--stars", type=int, default=0,
                    help="profiling aid: same workload family with this many stars (K, I unchanged); 0 = the config's")
    return ap.parse_args()


# ------------------------------------------------------------------------------------ helpers
def dist_env():
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


def max_over_ranks(value: float, device=None) -> float:
    """Max of a scalar over all ranks (identity when not distributed)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return value
    t = torch.tensor([value], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.barrier()


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.lines.append(ln.strip())

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, pw = [], None, set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx = float(f[1]); pw.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def algorithmic_bytes(m, n):
    """SURVEY.md section 8(d) / DESIGN.md section 7: fixed formulas."""
    return {"aprod1": 240 * m + 8 * n, "aprod2": 232 * m + 16 * n, "iteration": 472 * m + 96 * n,
            # fused LSQR pass: coefficients + indices once, u read + write, v gathered, g read-modify-written
            "lsqr_fused": 240 * m + 24 * n}


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def ncu_traffic(kernel, m):
    """dram bytes per launch from the committed ncu --set full summary (profiles/r01_traffic.csv:
    bytes per row of one captured launch), scaled by the rows of this workload; else None."""
    import csv
    p = os.path.join(ROOT, "profiles", "r01_traffic.csv")
    try:
        with open(p) as f:
            for row in csv.DictReader(f):
                if row["kernel"] == kernel:
                    return float(row["dram_bytes_per_row"]) * m
    except Exception:
        pass
    return None


def pick_workload(name, free_bytes):
    from gaia_synth.configs import CONFIGS
    if name != "auto":
        return CONFIGS[name]
    c4 = CONFIGS["C4"]
    need = 5e8 * (192 + 32 + 8 + 8) + 5 * c4.n_unknowns * 8 + (4 << 30)
    return c4 if free_bytes >= need else CONFIGS["C2"]


def shape_rows(shape):
    from gaia_synth import host
    return host.n_rows(shape)


# ------------------------------------------------------------------------------------ oracle timing
def time_oracle(shape, m_full, a, idx, steps, warmup):
    """ms per LSQR iteration of the CPU oracle (OpenMP, all cores) on a row sample [a, idx] of the
    workload, extrapolated to m_full rows: t = t_rows * (m_full / sample) + t_vectors."""
    import numpy as np
    import oracle
    from gaia_synth import host
    L = oracle.layout_of(shape)
    th = oracle.max_threads()
    ms, n = a.shape[0], shape.n_unknowns
    b = oracle.aprod1(L, a, idx, host.x_true(shape), host.noise(shape, 0, ms), threads=th)
    st = oracle.lsqr_init(L, a, idx, b, threads=th)
    x = host.test_vector(1, 1, n)
    y = np.zeros(ms)
    t_step, t_rows = [], []
    for it in range(warmup + steps):
        t0 = time.perf_counter()
        oracle.lsqr_step(L, a, idx, st, threads=th)
        t1 = time.perf_counter()
        oracle.aprod1(L, a, idx, x, y, threads=th)
        oracle.aprod2(L, a, idx, y, x, threads=th)
        t2 = time.perf_counter()
        if it >= warmup:
            t_step.append(t1 - t0)
            t_rows.append(t2 - t1)
    step = sum(t_step) / len(t_step)
    rows = min(sum(t_rows) / len(t_rows), step)
    full = rows * (m_full / ms) + (step - rows)
    return {"value": full * 1e3, "unit": "ms", "cores": th, "kind": "oracle",
            "sample": f"first {ms} of {m_full} rows of {shape.name} (OpenMP oracle, {steps} LSQR iterations; "
                      f"measured {step * 1e3:.1f} ms/iteration on the sample, row part scaled by {m_full / ms:.1f})"}


def oracle_sample_rows(m_full, requested):
    if requested > 0:
        return min(requested, m_full)
    return min(m_full, 4_000_000)


# ------------------------------------------------------------------------------------ reference arm
def run_reference(args):
    """--impl reference: the CPU oracle, as it stands, on a bounded sample of the same workload."""
    rank, local_rank, world = dist_env()
    if rank != 0:
        return 0
    import oracle  # noqa: F401  (the one other place bench.py may execute oracle/)
    from gaia_synth import host
    from gaia_synth.configs import CONFIGS
    try:
        import torch
        free = torch.cuda.mem_get_info()[0] if torch.cuda.is_available() else 0
    except Exception:
        free = 0
    shape = pick_workload(args.workload, free) if (args.workload != "auto" or free) else CONFIGS["C4"]
    m_full = shape_rows(shape)
    ms = oracle_sample_rows(m_full, args.oracle_rows)
    a, idx = host.make_rows(shape, 0, ms)
    steps, warmup = max(1, min(args.steps, 5)), max(1, min(args.warmup, 2))
    r = time_oracle(shape, m_full, a, idx, steps, warmup)
    line = {"impl": "reference", "metric": "ms_per_lsqr_iteration", "value": r["value"], "unit": "ms",
            "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": r["value"],
            "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{shape.name}: {m_full} rows x {shape.n_unknowns} unknowns",
                       "timed_steps_on_sample": steps},
            "cpu_baseline": r,
            "e2e": {"value": r["value"], "unit": "ms", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------ gsr arm
def run_gsr(args):
    import numpy as np
    import torch
    import torch.distributed as dist

    import paper_2503_22863_b200 as gsr
    from gaia_synth import device as gdev

    rank, local_rank, world = dist_env()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    free, total = torch.cuda.mem_get_info()
    shape = pick_workload(args.workload, free)
    if args.stars > 0:
        shape = shape.scaled(args.stars, name=f"{shape.name}[{args.stars} stars]")
    K, W = args.steps, max(args.warmup, 3)

    vals, idx = gdev.make_system(shape, device=dev)
    m, n = int(vals.shape[0]), shape.n_unknowns
    sysm = gsr.gsr_create(shape.n_stars, shape.n_knots, shape.n_instr, shape.n_glob, vals, idx)
    for opt in args.option:
        k, v = opt.split("=")
        sysm.set_option(k, int(v))
    # b = A x_true + sigma N(0,1), built with the library's own aprod1 (parity-tested; input construction)
    b = gdev.noise(shape, m, device=dev)
    sysm.aprod1(gdev.x_true(shape, device=dev), b)
    torch.cuda.synchronize()

    # ---- warm-up, then EXACTLY K timed iterations
    sysm.lsqr_init(b)
    sysm.lsqr_iterate(W)
    torch.cuda.synchronize()
    sysm.profile(True)
    sysm.profile_get(1); sysm.profile_get(2)
    l0 = sysm.launch_count()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    torch.cuda.synchronize()
    e0.record()
    sysm.lsqr_iterate(K)
    e1.record()
    torch.cuda.synchronize()
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    ms_total = max_over_ranks(e0.elapsed_time(e1), dev)
    launches = sysm.launch_count() - l0
    ap1_ms, ap1_n = sysm.profile_get(1)
    ap2_ms, ap2_n = sysm.profile_get(2)
    fu_ms, fu_n = sysm.profile_get(3)
    sysm.profile(False)
    res = sysm.lsqr_result()
    assert res.itn == W + K, f"expected {W + K} iterations, ran {res.itn} (istop {res.istop})"
    ms_iter = ms_total / K

    # ---- single aprod launches (median of 10 after 3 warm-ups, CUDA events)
    xv = gdev.test_vector(7, 1, n, device=dev)
    yv = torch.zeros(m, dtype=torch.float64, device=dev)

    def median_ms(fn, reps=10, wu=3):
        ts = []
        for i in range(wu + reps):
            a_, b_ = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a_.record(); fn(); b_.record(); b_.synchronize()
            if i >= wu:
                ts.append(a_.elapsed_time(b_))
        ts.sort()
        return ts[len(ts) // 2]
    ap1_alone = median_ms(lambda: sysm.aprod1(xv, yv))
    ap2_alone = median_ms(lambda: sysm.aprod2(yv, xv))
    del xv, yv

    ab = algorithmic_bytes(m, n)
    peak, peak_src = measured_peak()
    cands = [("aprod1", ap1_ms, ap1_n), ("aprod2", ap2_ms, ap2_n), ("lsqr_fused", fu_ms, fu_n)]
    dom, dom_ms, dom_n = max(cands, key=lambda c: c[1] * c[2])
    achieved = ab[dom] / (dom_ms * 1e-3) / 1e9
    roofline = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": ncu_traffic(dom, m), "peak_source": peak_src,
                "algorithmic_bytes": ab[dom], "kernel_ms": dom_ms, "launches_timed": dom_n, "share_of_step": dom_ms * dom_n / ms_total,
                "frac_of_8TBs": achieved / NOMINAL_HBM_GBS}
    iter_gbs = ab["iteration"] / (ms_iter * 1e-3) / 1e9

    line = {"metric": "ms_per_lsqr_iteration", "value": ms_iter, "unit": "ms", "n_gpus": world, "steps": K,
            "warmup": W, "ms_per_step": ms_iter, "higher_is_better": False, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{shape.name}: {m} rows x {n} unknowns (S={shape.n_stars}, K={shape.n_knots}/axis, "
                                   f"I={shape.n_instr}, G={shape.n_glob})",
                       "matrix_bytes": m * 224, "l2_policy": "inputs (matrix) far larger than L2; no flush",
                       "parallelism": "single GPU" if world == 1 else f"{world} independent replicas"},
            "iteration_gbs": iter_gbs, "iteration_frac_of_8TBs": iter_gbs / NOMINAL_HBM_GBS,
            "iteration_frac_of_measured": iter_gbs / peak,
            "aprod1_ms_in_lsqr": ap1_ms, "aprod2_ms_in_lsqr": ap2_ms, "fused_pass_ms_in_lsqr": fu_ms,
            "aprod1_ms_alone": ap1_alone, "aprod2_ms_alone": ap2_alone,
            "aprod1_gbs_alone": ab["aprod1"] / (ap1_alone * 1e-3) / 1e9,
            "aprod2_gbs_alone": ab["aprod2"] / (ap2_alone * 1e-3) / 1e9,
            "gpu_launches": launches, "roofline": roofline, "clocks": clocks,
            "lsqr": {"itn": res.itn, "istop": res.istop, "r1norm": res.r1norm, "anorm": res.anorm}}

    # ---- CPU baseline: the oracle, as it stands, on a bounded sample (rank 0, N = 1 only)
    if rank == 0 and world == 1 and not args.no_cpu:
        ms_rows = oracle_sample_rows(m, args.oracle_rows)
        a_h = vals[:ms_rows].cpu().numpy()
        i_h = idx[:ms_rows].cpu().numpy()
        line["cpu_baseline"] = time_oracle(shape, m, a_h, i_h, steps=3, warmup=1)
        del a_h, i_h

    # ---- end to end: the C-ABI call with HOST buffers (H2D of the system + K iterations + D2H of x)
    if not args.no_e2e:
        line["e2e"] = run_e2e(args, shape, sysm, vals, idx, b, m, n, K, dev, rank)
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def run_e2e(args, shape, sysm, vals, idx, b, m, n, K, dev, rank):
    """gsr_lsqr_host: all inputs in (pinned) HOST memory; the timed call copies them to the device,
    runs K LSQR iterations and copies x back.  Falls back to a row prefix if host RAM is short."""
    import numpy as np
    import torch
    import paper_2503_22863_b200 as gsr
    try:
        import psutil
        avail = psutil.virtual_memory().available
    except Exception:
        avail = 32 << 30
    need = m * 232
    rows = m
    note = "whole workload"
    if need * 1.25 > avail:
        rows = int(avail * 0.5 / 232)
        note = f"first {rows} rows only (host RAM {avail >> 30} GiB available)"
    hv = torch.empty((rows, 24), dtype=torch.float64, pin_memory=True)
    hi = torch.empty((rows, 8), dtype=torch.int32, pin_memory=True)
    hb = torch.empty(rows, dtype=torch.float64, pin_memory=True)
    hx = torch.empty(n, dtype=torch.float64, pin_memory=True)
    hv.copy_(vals[:rows]); hi.copy_(idx[:rows]); hb.copy_(b[:rows])
    torch.cuda.synchronize()
    # the device copy of the system must go: the host-buffer call allocates its own
    sysm.destroy()
    vals.untyped_storage().resize_(0); idx.untyped_storage().resize_(0); b.untyped_storage().resize_(0)
    torch.cuda.empty_cache()

    def call():
        t0 = time.perf_counter()
        r = gsr.gsr_lsqr_host(shape.n_stars, shape.n_knots, shape.n_instr, shape.n_glob, hv, hi, hb, hx, K)
        return (time.perf_counter() - t0) * 1e3, r
    call()                                   # warm-up (allocator, page tables)
    barrier()
    ms, r = call()
    barrier()
    ms = max_over_ranks(ms, dev)
    assert r.itn == K
    return {"value": ms / K, "unit": "ms", "h2d_bytes_per_step": rows * 232 / K, "d2h_bytes_per_step": n * 8 / K,
            "total_ms": ms, "steps": K, "note": f"gsr_lsqr_host, {note}; per-step = whole call / {K} iterations, "
            "host<->device copies (pinned memory) inside the timed call; wall clock around the blocking call"}


def main():
    args = parse()
    if args.impl == "reference":
        return run_reference(args)
    return run_gsr(args)


if __name__ == "__main__":
    sys.exit(main())
