#!/usr/bin/env python
"""Benchmark of the AVU-GSR hot path on B200: ms per LSQR iteration (aprod1 + aprod2 + the fused
vector work) and achieved HBM GB/s, on a synthetic Gaia-shaped system (BASELINE.json).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C4] [--impl reference]
                    [--control uniform-starts] [--mode extras] [--option name=value ...]

`--control uniform-starts` runs the same workload with uniform attitude starts (the control of C3's hot knots: same
rows per star, same M); `--mode extras` times what sits either side of the loop (gsr_colnorms, gsr_lsqr_ex with
preconditioning and variances, covariance pairs) instead of the iteration; `--option` passes gsr_set_option knobs.

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
    ap.add_argument("--control", default="none", choices=["none", "uniform-starts"],
                    help="uniform-starts: the workload with uniform attitude starts instead of its hot-knot mixture")
    ap.add_argument("--mode", default="iterate", choices=["iterate", "extras"],
                    help="extras: time gsr_colnorms / gsr_lsqr_ex (preconditioned, variances) / covariance pairs")
    ap.add_argument("--coeff23", action="store_true",
                    help="control: the same workload with N_Glob = 0 in the 23-coefficient production record (184-byte rows, "
                         "GSR_LAYOUT_COEFF23) instead of the padded 24-slot record")
    ap.add_argument("--sharded", action="store_true",
                    help="SURVEY.md 8(f2): ONE system row-sharded over the ranks (strong scaling) instead of one replica per "
                         "rank; the default for --gpus N stays replicas (BASELINE.json north_star: one GPU)")
    ap.add_argument("--n-glob", type=int, default=-1, choices=[-1, 0, 1],
                    help="control: override the workload's N_Glob (0 = the padded 24-slot record of the system --coeff23 stores in 23)")
    ap.add_argument("--reps", type=int, default=20, help="repetitions of the single aprod 1 / aprod 2 timings")
    ap.add_argument("--cov-pairs", type=int, action="append", default=[], help="--mode extras: pair counts to time")
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


def algorithmic_bytes(m, n, cpr=24):
    """SURVEY.md section 8(d) / DESIGN.md section 7: fixed formulas (192-byte records; with --coeff23 the record is
    8 * 23 = 184 bytes and the formulas shrink by 8 bytes per row and pass)."""
    rec = 8 * cpr + 32
    return {"aprod1": (rec + 16) * m + 8 * n, "aprod2": (rec + 8) * m + 16 * n, "iteration": (2 * rec + 24) * m + 96 * n,
            # fused LSQR pass: coefficients + indices once, u read + write, v gathered, g read-modify-written
            "lsqr_fused": (rec + 16) * m + 24 * n}


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def ncu_traffic(kernel, m):
    """(dram bytes per launch, where the figure comes from).  profiles/r02_traffic.csv, when present, holds
    dram__bytes_read.sum + dram__bytes_write.sum of one `ncu --set full` capture of a launch together with the
    rows of that launch; else profiles/r01_traffic.csv (C4 layout at 2e7 rows).  A capture of another size is
    scaled by rows and says so.  (None, reason) when there is no capture for this kernel."""
    import csv
    for name in ("r02_traffic.csv", "r01_traffic.csv"):
        p = os.path.join(ROOT, "profiles", name)
        try:
            with open(p) as f:
                for row in csv.DictReader(f):
                    if row["kernel"] != kernel:
                        continue
                    per_row = float(row["dram_bytes_per_row"])
                    rows = int(float(row.get("rows") or 20_000_000))
                    src = f"profiles/{name}: ncu --set full capture of one launch at {rows} rows"
                    if rows != m:
                        src += f", {per_row:.1f} B/row scaled to {m} rows"
                    return per_row * m, src
        except Exception:
            continue
    return None, "no ncu capture committed for this kernel"


def pick_workload(name, free_bytes, control="none"):
    from dataclasses import replace
    from gaia_synth.configs import CONFIGS
    if name != "auto":
        shape = CONFIGS[name]
    else:
        c4 = CONFIGS["C4"]
        need = 5e8 * (192 + 32 + 8 + 8) + 5 * c4.n_unknowns * 8 + (4 << 30)
        shape = c4 if free_bytes >= need else CONFIGS["C2"]
    if control == "uniform-starts":
        shape = replace(shape, hot_knots=False, name=shape.name + "[uniform attitude starts]")
    return shape


def shape_rows(shape):
    from gaia_synth import host
    return host.n_rows(shape)


# ------------------------------------------------------------------------------------ oracle timing
def time_oracle(shape, m_full, a, idx, steps, warmup, budget_s=1e9):
    """ms per LSQR iteration of the CPU oracle (OpenMP, all cores) on a row sample [a, idx] of the
    workload, extrapolated to m_full rows: t = t_rows * (m_full / sample) + t_vectors.
    Stops early (after at least one timed step) once budget_s seconds have gone into the loop."""
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
    t_begin = time.perf_counter()
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
            if t2 - t_begin > budget_s:
                break
    step = sum(t_step) / len(t_step)
    rows = min(sum(t_rows) / len(t_rows), step)
    full = rows * (m_full / ms) + (step - rows)
    return {"value": full * 1e3, "unit": "ms", "cores": th, "kind": "oracle", "steps_timed": len(t_step),
            "sample": f"first {ms} of {m_full} rows of {shape.name} (OpenMP oracle, {len(t_step)} LSQR iterations timed; "
                      f"measured {step * 1e3:.1f} ms/iteration on the sample, row part scaled by {m_full / ms:.1f})"}


def oracle_sample_rows(m_full, requested):
    """Rows of the oracle's sample: the whole workload up to 1e8 rows ("time the first 1e8 rows (22 GB)"
    when the host cannot hold C4), less if host memory is short."""
    if requested > 0:
        return min(requested, m_full)
    from gaia_synth.hostmem import available_host_memory
    avail = available_host_memory(default=16 << 30)
    cap = int(max(avail * 0.4, 1 << 30) // 260)        # rows + the M-vectors of the oracle's LSQR state
    return max(1, min(m_full, 100_000_000, cap))


# ------------------------------------------------------------------------------------ reference arm
def run_reference(args):
    """--impl reference: the CPU oracle, as it stands, on a bounded sample of the same workload.  The sample rows come
    from the device generator when a GPU is there (the numpy generator needs minutes for 1e8 rows), copied to the host."""
    rank, local_rank, world = dist_env()
    if rank != 0:
        return 0
    import oracle  # noqa: F401  (the one other place bench.py may execute oracle/)
    from gaia_synth import host
    from gaia_synth.configs import CONFIGS
    cuda = False
    try:
        import torch
        cuda = torch.cuda.is_available()
        free = torch.cuda.mem_get_info()[0] if cuda else 0
    except Exception:
        free = 0
    shape = (pick_workload(args.workload, free, args.control) if (args.workload != "auto" or free)
             else pick_workload("C4", 0, args.control))
    if args.stars > 0:
        shape = shape.scaled(args.stars, name=f"{shape.name}[{args.stars} stars]")
    m_full = shape_rows(shape)
    ms = oracle_sample_rows(m_full, args.oracle_rows)
    if cuda:
        from gaia_synth import device as gdev
        v, i = gdev.make_system(shape, r0=0, r1=ms)
        a, idx = v.cpu().numpy(), i.cpu().numpy()
        del v, i
        torch.cuda.empty_cache()
    else:
        if args.oracle_rows <= 0:
            ms = min(ms, 4_000_000)
        a, idx = host.make_rows(shape, 0, ms)
    steps, warmup = max(1, args.steps), max(1, args.warmup)
    r = time_oracle(shape, m_full, a, idx, steps, warmup, budget_s=150.0)
    line = {"impl": "reference", "metric": "ms_per_lsqr_iteration", "value": r["value"], "unit": "ms",
            "n_gpus": args.gpus, "steps": r["steps_timed"], "warmup": warmup, "ms_per_step": r["value"],
            "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{shape.name}: {m_full} rows x {shape.n_unknowns} unknowns",
                       "steps_requested": args.steps, "steps_timed_on_sample": r["steps_timed"],
                       "note": "every step is one oracle LSQR iteration on the row sample; the row part is scaled to the "
                               "workload's rows (cpu_baseline.sample); the loop stops after 150 s"},
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
    shape = pick_workload(args.workload, free, args.control)
    if args.stars > 0:
        shape = shape.scaled(args.stars, name=f"{shape.name}[{args.stars} stars]")
    K, W = args.steps, max(args.warmup, 3)
    if args.mode == "extras":
        return run_extras(args, shape, dev, rank, world)
    if args.sharded:
        return run_sharded(args, shape, dev, rank, world, K, W)

    cpr = 24
    if args.n_glob >= 0 and not args.coeff23:
        from dataclasses import replace
        shape = replace(shape, n_glob=args.n_glob, name=shape.name + f"[N_Glob = {args.n_glob}]")
    if args.coeff23:
        # the production record: N_Glob = 0, 23 doubles per row.  Generated block by block (the 24-slot rows of a block,
        # slots 0..22 packed) so that C4 never holds both storages.
        from dataclasses import replace
        shape = replace(shape, n_glob=0, name=shape.name + "[N_Glob = 0, 23-coefficient record]")
        cpr = 23
        m_all = shape_rows(shape)
        vals = torch.empty((m_all, 23), dtype=torch.float64, device=dev)
        idx = torch.empty((m_all, 8), dtype=torch.int32, device=dev)
        blk = 8_000_000
        for r0 in range(0, m_all, blk):
            v24, i24 = gdev.make_system(shape, device=dev, r0=r0, r1=min(r0 + blk, m_all))
            vals[r0:r0 + v24.shape[0]].copy_(v24[:, :23])
            idx[r0:r0 + v24.shape[0]].copy_(i24)
            del v24, i24
    else:
        vals, idx = gdev.make_system(shape, device=dev)
    m, n = int(vals.shape[0]), shape.n_unknowns
    sysm = gsr.gsr_create(shape.n_stars, shape.n_knots, shape.n_instr, shape.n_glob, vals, idx, coeffs_per_row=cpr)
    for opt in args.option:
        k, v = opt.split("=")
        sysm.set_option(k, int(v))
    # b = A x_true + sigma N(0,1), built with the library's own aprod1 (parity-tested; input construction)
    b = gdev.noise(shape, m, device=dev)
    sysm.aprod1(gdev.x_true(shape, device=dev), b)
    torch.cuda.synchronize()

    # ---- warm-up, then EXACTLY K timed iterations.  Large systems: the per-kernel CUDA events of gsr_profile are on
    # (two event records per iteration, nothing else changes).  Small, launch-bound systems (matrix <= 256 MB) replay
    # a CUDA graph, which the per-kernel events would switch off: there the K iterations are timed with profiling
    # OFF -- the default product path -- and the kernel durations come from a separate, profiled run afterwards.
    graph_path = m * 224.0 <= 256.0 * 1024 * 1024 and K >= 2
    sysm.lsqr_init(b)
    sysm.lsqr_iterate(W)
    if graph_path:
        sysm.lsqr_iterate(K)      # instantiates the K-iteration graph outside the timed region
        W += K
    torch.cuda.synchronize()
    if not graph_path:
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
    kernel_ms_source = "CUDA events around every launch inside the timed region (gsr_profile)"
    extra = 0
    if graph_path:
        extra = min(K, 8)
        sysm.profile(True)
        sysm.profile_get(1); sysm.profile_get(2); sysm.profile_get(3)
        sysm.lsqr_iterate(extra)
        torch.cuda.synchronize()
        kernel_ms_source = (f"separate profiled run of {extra} iterations after the timed region (the timed region replays "
                            "a CUDA graph, which per-kernel events would disable)")
    ap1_ms, ap1_n = sysm.profile_get(1)
    ap2_ms, ap2_n = sysm.profile_get(2)
    fu_ms, fu_n = sysm.profile_get(3)
    sysm.profile(False)
    res = sysm.lsqr_result()
    assert res.itn == W + K + extra, f"expected {W + K + extra} iterations, ran {res.itn} (istop {res.istop})"
    ms_iter = ms_total / K

    # ---- single aprod launches (median of --reps (20) after 3 warm-ups, CUDA events)
    xv = gdev.test_vector(7, 1, n, device=dev)
    yv = torch.zeros(m, dtype=torch.float64, device=dev)

    def median_ms(fn, reps=max(args.reps, 1), wu=3):
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

    ab = algorithmic_bytes(m, n, cpr)
    peak, peak_src = measured_peak()
    cands = [("aprod1", ap1_ms, ap1_n), ("aprod2", ap2_ms, ap2_n), ("lsqr_fused", fu_ms, fu_n)]
    dom, dom_ms, dom_n = max(cands, key=lambda c: c[1] * c[2])
    achieved = ab[dom] / (dom_ms * 1e-3) / 1e9
    traffic, traffic_src = ncu_traffic(dom, m)
    try:
        l2_dies = sysm.instr_acc_info()
    except Exception:                                              # noqa: BLE001
        l2_dies = None
    # share of the step: durations of the dominant kernel relative to the step, both per iteration
    per_iter_launches = dom_n / (extra if graph_path else K)
    roofline = {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src,
                "algorithmic_bytes": ab[dom], "kernel_ms": dom_ms, "kernel_ms_source": kernel_ms_source,
                "launches_timed": dom_n, "share_of_step": dom_ms * per_iter_launches / ms_iter,
                "frac_of_8TBs": achieved / NOMINAL_HBM_GBS}
    # BASELINE.json's metric: the two-pass formula 472 M + 96 n over the time of one iteration.  With the fused pass
    # (A streamed once) this is an EFFECTIVE figure, not bytes moved; what the fused schedule itself must move is
    # 240 M + 24 n (matrix pass) + 72 n (the n-length kernels).
    eff_gbs = ab["iteration"] / (ms_iter * 1e-3) / 1e9
    fused = fu_n > 0
    moved = (ab["lsqr_fused"] + 72 * n) if fused else ab["iteration"]
    moved_gbs = moved / (ms_iter * 1e-3) / 1e9

    line = {"metric": "ms_per_lsqr_iteration", "value": ms_iter, "unit": "ms", "n_gpus": world, "steps": K,
            "warmup": W, "ms_per_step": ms_iter, "higher_is_better": False, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{shape.name}: {m} rows x {n} unknowns (S={shape.n_stars}, K={shape.n_knots}/axis, "
                                   f"I={shape.n_instr}, G={shape.n_glob})",
                       "matrix_bytes": m * (8 * cpr + 32), "coeffs_per_row": cpr, "l2_policy": "inputs (matrix) far larger than L2; no flush",
                       "parallelism": "single GPU" if world == 1 else f"{world} independent replicas",
                       "timed_path": "CUDA-graph replay, profiling off" if graph_path else "eager launches, per-kernel events on",
                       "options": args.option},
            "iteration_effective_gbs_two_pass_formula": eff_gbs,
            "iteration_effective_frac_of_8TBs": eff_gbs / NOMINAL_HBM_GBS,
            "iteration_effective_frac_of_measured": eff_gbs / peak,
            "iteration_moved_gbs": moved_gbs, "iteration_moved_frac_of_measured": moved_gbs / peak,
            "iteration_formula_note": "effective = (472 M + 96 n) / time, BASELINE.json's two-pass formula (target >= 0.70 of "
                                      "8 TB/s); moved = bytes the schedule that ran must move / time (fused: 240 M + 96 n)",
            "aprod1_ms_in_lsqr": ap1_ms, "aprod2_ms_in_lsqr": ap2_ms, "fused_pass_ms_in_lsqr": fu_ms,
            "aprod1_ms_alone": ap1_alone, "aprod2_ms_alone": ap2_alone,
            "aprod1_gbs_alone": ab["aprod1"] / (ap1_alone * 1e-3) / 1e9,
            "aprod2_gbs_alone": ab["aprod2"] / (ap2_alone * 1e-3) / 1e9,
            "aprod1_frac_of_8TBs_alone": ab["aprod1"] / (ap1_alone * 1e-3) / 1e9 / NOMINAL_HBM_GBS,
            "aprod2_frac_of_8TBs_alone": ab["aprod2"] / (ap2_alone * 1e-3) / 1e9 / NOMINAL_HBM_GBS,
            "single_aprod_reps": max(args.reps, 1),
            "gpu_launches": launches, "roofline": roofline, "clocks": clocks,
            "l2_dies": l2_dies,
            "lsqr": {"itn": res.itn, "istop": res.istop, "r1norm": res.r1norm, "anorm": res.anorm}}

    # ---- CPU baseline: the oracle, as it stands, on a bounded sample (rank 0, N = 1 only).  A failure of this leg or
    # of the end-to-end leg (host memory, say) is reported in the line instead of losing the device-timed result.
    if rank == 0 and world == 1 and not args.no_cpu and cpr == 24:
        try:
            ms_rows = oracle_sample_rows(m, args.oracle_rows)
            a_h = vals[:ms_rows].cpu().numpy()
            i_h = idx[:ms_rows].cpu().numpy()
            line["cpu_baseline"] = time_oracle(shape, m, a_h, i_h, steps=3, warmup=1)
            del a_h, i_h
        except Exception as ex:                                    # noqa: BLE001
            line["cpu_baseline"] = {"value": None, "unit": "ms", "cores": None, "kind": "oracle",
                                    "sample": f"failed: {type(ex).__name__}: {ex}"}

    # ---- end to end: the C-ABI call with HOST buffers (H2D of the system + K iterations + D2H of x)
    if not args.no_e2e and cpr == 24:
        try:
            line["e2e"] = run_e2e(args, shape, sysm, vals, idx, b, m, n, K, dev, rank)
        except Exception as ex:                                    # noqa: BLE001
            line["e2e"] = {"value": None, "unit": "ms", "h2d_bytes_per_step": None, "d2h_bytes_per_step": None,
                           "note": f"failed: {type(ex).__name__}: {ex}"}
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def run_sharded(args, shape, dev, rank, world, K, W):
    """--sharded: the workload's rows cut at star boundaries into one range per rank (paper_2503_22863_b200/sharded.py),
    every rank generating only its own rows; the constraint rows, if any, are rank 0's second section.  K iterations of
    the sharded solve are timed (phases + one NCCL allreduce per exchange), max over ranks.  Strong scaling: the job is
    the same system whatever N."""
    import torch
    import torch.distributed as dist
    import paper_2503_22863_b200 as gsr
    from gaia_synth import configs as C
    from gaia_synth import device as gdev
    from gaia_synth import host
    from paper_2503_22863_b200.sharded import DistComm, LocalComm, ShardedLsqr, partition_stars
    counts = (shape.n_stars, shape.obs_per_star) if shape.obs_per_star else host.obs_counts(shape)
    part = partition_stars(counts, world)[rank]
    m_obs = host.n_obs_rows(shape)
    vals, idx = gdev.make_system(shape, device=dev, r0=part.row_lo, r1=part.row_hi)
    sysm = gsr.gsr_create(shape.n_stars, shape.n_knots, shape.n_instr, shape.n_glob, vals, idx)
    for opt in args.option:
        k, v = opt.split("=")
        sysm.set_option(k, int(v))
    noise = [gdev.normal(shape.seed, C.STREAM_NOISE, part.row_lo, part.row_hi, scale=shape.sigma, device=dev)]
    con = None
    if rank == 0 and shape.n_constraint_rows:
        con = gdev.make_system(shape, device=dev, r0=m_obs, r1=m_obs + shape.n_constraint_rows)
        sysm.attach_constraints(*con)
        noise.append(gdev.normal(shape.seed, C.STREAM_NOISE, m_obs, m_obs + shape.n_constraint_rows, scale=shape.sigma, device=dev))
    b = torch.cat(noise)
    sysm.aprod1(gdev.x_true(shape, device=dev), b)          # this rank's rows of b = A x_true + noise
    m_local, n = sysm.n_rows, shape.n_unknowns
    m_total = host.n_rows(shape)
    drv = ShardedLsqr([sysm], DistComm() if world > 1 else LocalComm(1), check_every=1 << 30)
    stopped, _ = drv.begin([b], 1 << 40)
    assert not stopped
    drv.iterate(W)
    torch.cuda.synchronize()
    l0 = sysm.launch_count()
    sampler = ClockSampler(dev.index or 0)
    if rank == 0:
        sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    torch.cuda.synchronize()
    e0.record()
    drv.iterate(K)
    e1.record()
    torch.cuda.synchronize()
    barrier()
    clocks = sampler.stop() if rank == 0 else None
    ms_iter = max_over_ranks(e0.elapsed_time(e1), dev) / K
    stopped, res = drv.poll()
    assert res.itn == W + K and not stopped
    ab = algorithmic_bytes(m_total, n)
    peak, _ = measured_peak()
    ns = n - 5 * shape.n_stars
    line = {"metric": "ms_per_lsqr_iteration", "value": ms_iter, "unit": "ms", "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms_iter, "higher_is_better": False, "scaling": "strong", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": f"{shape.name}: {m_total} rows x {n} unknowns, row-sharded over {world} rank(s) at star "
                                   f"boundaries (rank 0: {m_local} rows)",
                       "parallelism": f"row-sharded x{world} (gsr_shard_* phases; one allreduce of {ns + 2} doubles and one of 1 "
                                      "double per iteration)",
                       "l2_policy": "inputs (matrix) far larger than L2; no flush", "options": args.option},
            "iteration_effective_gbs_two_pass_formula": ab["iteration"] / (ms_iter * 1e-3) / 1e9,
            "iteration_effective_frac_of_8TBs_per_gpu": ab["iteration"] / (ms_iter * 1e-3) / 1e9 / NOMINAL_HBM_GBS / world,
            "gpu_launches": sysm.launch_count() - l0, "exchanges_per_iteration": 2,
            "exchanged_bytes_per_iteration_per_rank": 8 * (ns + 3), "clocks": clocks,
            "lsqr": {"itn": res.itn, "istop": res.istop, "r1norm": res.r1norm, "anorm": res.anorm}}
    if rank == 0:
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def run_extras(args, shape, dev, rank, world):
    """--mode extras: what sits either side of the LSQR loop, timed through the binding:
    gsr_colnorms, K iterations of gsr_lsqr and of gsr_lsqr_ex (column-norm preconditioned, with variances), K
    iterations with covariance pairs registered, and -- for systems up to 2e7 rows -- both solves to convergence.
    Wall clock around the blocking calls (each synchronises its stream); median of 3 after one warm-up."""
    import torch
    import paper_2503_22863_b200 as gsr
    from gaia_synth import device as gdev
    K = max(args.steps, 1)
    vals, idx = gdev.make_system(shape, device=dev)
    m, n = int(vals.shape[0]), shape.n_unknowns
    sysm = gsr.gsr_create(shape.n_stars, shape.n_knots, shape.n_instr, shape.n_glob, vals, idx)
    for opt in args.option:
        k, v = opt.split("=")
        sysm.set_option(k, int(v))
    b = gdev.noise(shape, m, device=dev)
    sysm.aprod1(gdev.x_true(shape, device=dev), b)
    x = torch.empty(n, dtype=torch.float64, device=dev)
    var = torch.empty(n, dtype=torch.float64, device=dev)
    cn = torch.empty(n, dtype=torch.float64, device=dev)
    torch.cuda.synchronize()

    def wall_ms(fn, reps=3, wu=1):
        ts = []
        for i in range(wu + reps):
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            fn()
            torch.cuda.synchronize()
            if i >= wu:
                ts.append((time.perf_counter() - t0) * 1e3)
        ts.sort()
        return ts[len(ts) // 2]

    out = {"mode": "extras", "workload": f"{shape.name}: {m} rows x {n} unknowns", "iterations": K,
           "options": args.option, "timing": "wall clock around the blocking call, median of 3 after 1 warm-up"}
    out["colnorms_ms"] = wall_ms(lambda: sysm.colnorms(cn))
    out["colnorms_stream_gbs"] = m * 224 / (out["colnorms_ms"] * 1e-3) / 1e9
    out["lsqr_plain_ms_per_iteration"] = wall_ms(lambda: sysm.lsqr(b, x, K)) / K
    t_pre = wall_ms(lambda: sysm.lsqr_ex(b, x, var=var, precond=True, itnlim=K))
    out["lsqr_precond_var_ms_per_iteration"] = (t_pre - out["colnorms_ms"]) / K
    out["lsqr_precond_var_note"] = "column-norm pass (colnorms_ms) subtracted; init included, as for the plain run"
    pairs = args.cov_pairs or [1_000_000, 10_000_000]
    g = torch.Generator(device=dev)
    g.manual_seed(shape.seed)
    cov_rows = []
    for npairs in pairs:
        j1 = torch.randint(0, n, (npairs,), generator=g, device=dev, dtype=torch.int64)
        j2 = torch.randint(0, n, (npairs,), generator=g, device=dev, dtype=torch.int64)
        cov = torch.zeros(npairs, dtype=torch.float64, device=dev)
        sysm.set_cov_pairs(j1, j2, cov)
        t = wall_ms(lambda: sysm.lsqr_ex(b, x, itnlim=K)) / K
        sysm.set_cov_pairs(None, None, None)
        cov_rows.append({"pairs": npairs, "ms_per_iteration": t,
                         "pairs_alone_ms": t - out["lsqr_plain_ms_per_iteration"],
                         "list_and_accumulator_gbs": 32.0 * npairs / max((t - out["lsqr_plain_ms_per_iteration"]) * 1e-3, 1e-9) / 1e9})
        del j1, j2, cov
    out["cov_pairs"] = cov_rows
    if m <= 20_000_000:
        t0 = time.perf_counter()
        r0 = sysm.lsqr(b, x, 5000, 1e-12, 1e-12, 1e8)
        torch.cuda.synchronize()
        t1 = time.perf_counter()
        x0 = x.clone()
        r1 = sysm.lsqr_ex(b, x, var=var, precond=True, itnlim=5000, atol=1e-12, btol=1e-12, conlim=1e8)
        torch.cuda.synchronize()
        t2 = time.perf_counter()
        out["to_convergence"] = {"plain": {"istop": r0.istop, "itn": r0.itn, "wall_ms": (t1 - t0) * 1e3},
                                 "precond_var": {"istop": r1.istop, "itn": r1.itn, "wall_ms": (t2 - t1) * 1e3},
                                 "rel_diff_of_x": float(torch.linalg.norm(x - x0) / torch.linalg.norm(x0))}
    if rank == 0:
        print(json.dumps(out))
    return 0


def run_e2e(args, shape, sysm, vals, idx, b, m, n, K, dev, rank):
    """gsr_lsqr_host: all inputs in (pinned) HOST memory; the timed call copies them to the device,
    runs K LSQR iterations and copies x back.  Falls back to a row prefix if host RAM is short."""
    import numpy as np
    import torch
    import paper_2503_22863_b200 as gsr
    from gaia_synth.hostmem import available_host_memory
    avail = available_host_memory(default=32 << 30)       # MemAvailable capped by the memory cgroup's headroom
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
