#!/usr/bin/env python
"""bench.py -- the hot path of FIESTA 4's integration stage on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]

A "step" is one pass of the whole hot path (point generation, periodising transform, program
walk, accumulation, two-level reduction, estimator: SURVEY 8(a) A1, A2, A5-A7, A9) over the
workload of BASELINE.json config 3 ("large-sampling workload": 2000 sectors, dim 8, 5 epsilon
orders, ~1000 FP64 ops per program, 2^24 points per sector = 8 random shifts x a 2^21-point
Korobov lattice).  Inputs are synthetic and seeded (workloads/).

metric = integrand evaluations per second, an evaluation being one (point, sector, order).
Prints ONE JSON line (rank 0).  With N > 1 (torchrun) every rank integrates its own 2000
sectors (weak scaling, sectors are independent integrals: no data-path collective), results
are gathered once at the end, time is the max over ranks.

--impl reference times the CPU oracle (oracle/, numpy long double) as it stands on the host
cores, on a bounded sample of the same workload.
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "integrand evals/sec (points x sectors x orders), FP64"
UNIT = "evals/s"
WORKLOAD = "C3"
# FP64 ALU roofline: 148 SMs x 64 FP64 FMA lanes x 2 flops x 1.965 GHz (guide's unit counts and
# max clock).  The live DFMA micro-benchmark is reported beside it.
FP64_PEAK_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--sectors", type=int, default=None, help="reduce the sector count (profiling runs only)")
    ap.add_argument("--no-cpu-baseline", action="store_true", help="skip the oracle timing (profiling runs only)")
    ap.add_argument("--no-extras", action="store_true", help="skip the first-result and C4/C5 measurements (profiling runs only)")
    ap.add_argument("--c4-sectors", type=int, default=None, help="reduce C4's sector count in the extras (profiling runs only)")
    ap.add_argument("--c5-sectors", type=int, default=None, help="reduce C5's sector count in the extras (profiling runs only)")
    ap.add_argument("--workload", default="C3", choices=["C1", "C2", "C3", "C4", "C5"],
                    help="profiling runs only: time another BASELINE configuration (the bench line is C3)")
    return ap.parse_args()


# ------------------------------------------------------------------------------ CPU oracle leg

def _oracle_task(args):
    """One sector's partial sums with the oracle, one shift of a reduced lattice (runs in a worker)."""
    sys.path.insert(0, ROOT)
    from oracle import integrate as OI
    from oracle import points as OP
    from oracle.integrate import SectorSpec
    texts, sector_id, dim, n_lattice, a, r, seed, dtype = args
    import numpy as _np
    sec = SectorSpec(texts, sector_id)
    gv = OP.korobov_genvec(a, n_lattice, dim)
    s1, s2, _ = OI.lattice_partial_sums(sec, n_lattice, 1, gv, r, seed, rdtype=_np.longdouble if dtype == "f80" else _np.float64)
    return float(s1[0, 0, 0])


def _warm(_):
    sys.path.insert(0, ROOT)
    import oracle.integrate  # noqa: F401
    return os.getpid()


class OraclePool:
    """The oracle, unmodified, on the host cores: one process per core, sectors dealt out."""

    def __init__(self):
        import multiprocessing as mp
        self.cores = max(1, min(os.cpu_count() or 1, 32))
        self.pool = mp.get_context("spawn").Pool(self.cores)
        self.pool.map(_warm, range(self.cores * 2))

    def close(self):
        self.pool.close()
        self.pool.join()

    def run(self, wl, nsec, n_lattice, dtype="f80"):
        """Time the oracle on nsec sectors x n_lattice points (one shift).  -> (evals, seconds).
        dtype "f80": numpy long double, the parity oracle as it stands; "f64": the same tree walk in double
        (the oracle's rdtype argument), reported beside it."""
        from workloads import korobov_a
        a = korobov_a(n_lattice, wl.dim)
        tasks = [(s.texts, s.sector_id, wl.dim, n_lattice, a, wl.periodize_r, wl.seed, dtype) for s in wl.sectors[:nsec]]
        t0 = time.perf_counter()
        self.pool.map(_oracle_task, tasks, chunksize=1)
        dt = time.perf_counter() - t0
        return nsec * n_lattice * wl.K, dt


def cpu_baseline(wl, pool, nsec, n_lattice):
    evals, dt = pool.run(wl, nsec, n_lattice)
    evals64, dt64 = pool.run(wl, nsec, n_lattice, dtype="f64")
    return {"value": evals / dt, "unit": UNIT, "cores": pool.cores, "kind": "oracle",
            "sample": f"{nsec} sectors x {n_lattice} lattice points x {wl.K} orders of {WORKLOAD} "
                      f"(oracle/ as it stands: numpy long double, one process per core), {dt:.1f} s",
            "sample_s": dt, "value_same_walk_in_double": evals64 / dt64, "double_sample_s": dt64}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from workloads import make_workload
    pool = OraclePool()
    nsec = pool.cores
    wl = make_workload(WORKLOAD, nsectors=nsec)
    n_lattice = 1 << 12
    for _ in range(args.warmup):
        pool.run(wl, nsec, n_lattice)
    tot_e, tot_t = 0, 0.0
    for _ in range(args.steps):
        e, t = pool.run(wl, nsec, n_lattice)
        tot_e += e
        tot_t += t
    pool.close()
    v = tot_e / tot_t
    sample = (f"each step = {nsec} sectors x {n_lattice} lattice points x {wl.K} orders of {WORKLOAD} "
              f"(bounded sample; the full step is 2000 x 2^24 x 5)")
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / max(args.steps, 1), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f80 (x87 long double)", "data": "synthetic",
            "config": {"workload": f"BASELINE config 3 ({WORKLOAD}), bounded sample", "sample": sample},
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": pool.cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)
    return 0


# ------------------------------------------------------------------------------ clocks

class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.lines, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        self.thread.join(timeout=5)
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0]))
                mx.append(float(f[1]))
                pw.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------ the B200 arm

def path_overhead_flops(wl):
    """Algorithmic FP64 flops per point of the steps of the path AROUND the program walk (SURVEY 8(a) A2/A3,
    A4, A6), counted like the program's own (fma 2, mul/add 1, div/sqrt 15): DESIGN.md "Algorithmic work".
      A2 lattice, r = 3, per coordinate: v (1), Horner of phi_3 (3 fma), v^4 (2), p (1), 1-p (1), u(1-u) (fma),
         W *= . (1) = 14;  per point: W = cw^n S^3 (3)
      A3 Vegas, per coordinate: fraction (3), width (1), x (fma), weight (2) = 8
      A4 deformation, dimension n: per k: ls (2), Im z (1), sqrt (8), diagonal (mul, mul, fma = 4); per pair
         l < k: 2;  elimination of I - iS: per column the pivot (cmul 6, reciprocal 3 + 10 + 2), per row below a
         complex multiply (6) and one complex fma (8) per entry of the lower triangle.  (sqrt and the
         reciprocal at what the routines execute, so that the count stays below ncu's executed flops.)
      A6 per order: real g = W o (1), S1 (1), S2 (fma) = 4 [+ h2 (fma) for Vegas];
         complex g = (W det) o (6), S1, S2 of Re and Im (6) = 12, and W det (2) per point
    Point generation itself (A1) is integer work and is not counted."""
    n, K = wl.dim, wl.K
    cplx = bool(wl.sectors[0].is_complex or wl.sectors[0].deform_f_index)
    f = 0.0
    if wl.rule == 0:
        f += 14 * n + 3
    elif wl.rule == 2:
        f += 8 * n
    if cplx and wl.sectors[0].deform_f_index:
        f += n * 15 + n * (n - 1)
        for c in range(n):
            f += 6 + (15 if c + 1 < n else 0)
            for r in range(c + 1, n):
                f += 6 + 8 * (r - c)
    f += (12 * K + 2) if cplx else 4 * K
    if wl.rule == 2:
        f += 2 * K * (2 if cplx else 1)
    return f


def describe(wl, S):
    if wl.rule == 2:
        return (f"{S} sectors, dim {wl.dim}, {wl.K} order(s), Vegas {wl.vegas_bins} bins, {wl.vegas_iters} iterations x "
                f"{wl.npoints} Philox points/sector")
    return (f"{S} sectors, dim {wl.dim}, {wl.K} orders, {wl.npoints} points/sector = {wl.n_shifts} shift(s) x "
            f"2^{wl.n_lattice.bit_length() - 1} Korobov lattice (a={wl.korobov_a}), periodising r={wl.periodize_r}")


class Timer:
    """One workload on one context: steps of fiesta_integrate_async bracketed by CUDA events on the ctx stream."""

    def __init__(self, torch, dev, stream, ctx, flush):
        self.torch, self.dev, self.stream, self.ctx, self.flush = torch, dev, stream, ctx, flush

    def step(self, prog, wl, rule, i):
        torch = self.torch
        with torch.cuda.stream(self.stream):
            self.flush.fill_(i & 0xff)                           # L2 flush between iterations (untimed)
            e0 = torch.cuda.Event(enable_timing=True)
            e1 = torch.cuda.Event(enable_timing=True)
            e0.record(self.stream)
            self.ctx.integrate_async(prog, wl.npoints, rule, wl.seed + i)
            e1.record(self.stream)
        return e0, e1

    def run(self, prog, wl, rule, warmup, steps, first=0):
        for i in range(warmup):
            self.step(prog, wl, rule, first + i)
        self.torch.cuda.synchronize(self.dev)
        step_ms, kern_ms, launches, tiers = [], [], 0, [0, 0]
        for i in range(steps):
            e0, e1 = self.step(prog, wl, rule, first + warmup + i)
            e1.synchronize()
            step_ms.append(e0.elapsed_time(e1))
            km, nl = self.ctx.last_timing()
            kern_ms.append(km)
            launches += nl
            a, b = self.ctx.last_tiers()
            tiers[0] += a
            tiers[1] += b
        return step_ms, kern_ms, launches, tiers


# dram__bytes_read.sum + dram__bytes_write.sum of one native-kernel launch, from the committed ncu --set full
# captures (profiles/r02_ncu_fxj_integrate_c3.md, _c4.md, _c5.md): the points are made on the device and a block
# writes one 256-byte record, so the traffic of the ALU-bound kernels is the program text and the parameters
NCU_DRAM_BYTES = {"C3": 56832, "C4": 54784, "C5": 37888}


def roofline_of(wl, prog, S, kern_ms, peak_live, tiers):
    """bound 'alu': algorithmic FP64 flops of one pass / the evaluation kernels' time (CUDA events inside the
    library, fiesta_last_timing) against the FP64 peak derived in DESIGN.md section 6."""
    iters = wl.vegas_iters if wl.rule == 2 else 1
    prog_flops = float(np.mean(prog.info["flops"]))
    over = path_overhead_flops(wl)
    kms = sum(kern_ms) / len(kern_ms)
    pts = float(wl.npoints) * iters * S
    ach = (prog_flops + over) * pts / (kms * 1e-3) / 1e12
    ach_prog = prog_flops * pts / (kms * 1e-3) / 1e12
    native = tiers[1] == 0
    return {"bound": "alu", "achieved": ach, "peak": FP64_PEAK_TFLOPS, "unit": "TFLOP/s", "frac": ach / FP64_PEAK_TFLOPS,
            "traffic": NCU_DRAM_BYTES.get(wl.name) if native else None, "traffic_unit": "bytes per launch (dram read + write)",
            "achieved_program_only": ach_prog, "frac_program_only": ach_prog / FP64_PEAK_TFLOPS,
            "flops_per_point": prog_flops + over, "flops_per_point_program": prog_flops,
            "flops_per_point_path_overhead": over,
            "kernel": ("fxj_integrate (native kernels, one launch per sector and pass)" if native else
                       "fx_integrate_* (interpreter)" if tiers[0] == 0 else "mixed tiers"),
            "kernel_ms": kms, "kernel_launches_per_step": S * iters,
            "kernel_ms_per_launch": kms / (S * iters),
            "peak_source": "derived: 148 SM x 64 FP64 lanes x 2 x 1.965 GHz (MEASURED_PEAKS.json has no FP64 entry)",
            "peak_dfma_microbench_live": peak_live,
            "evals_per_s_kernel": pts * wl.K / (kms * 1e-3)}


def run_b200(args):
    import torch
    import torch.distributed as dist
    import paper_1511_03614_b200 as fb
    from paper_1511_03614_b200.sharding import gather_results, max_over_ranks, partition_sectors
    from workloads import make_workload

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (sm_100a); there is no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    K, W = args.steps, max(args.warmup, 0)
    D = dist if world > 1 else None

    # CPU oracle baseline first (rank 0, N=1 only), before this process touches CUDA heavily
    cpu = None
    global WORKLOAD
    WORKLOAD = args.workload
    nsec_full = args.sectors if args.sectors is not None else len(make_workload(WORKLOAD).sectors)
    extras = rank == 0 and world == 1 and WORKLOAD == "C3" and not args.no_extras
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        pool = OraclePool()
        wl_s = make_workload(WORKLOAD, nsectors=2 * pool.cores)
        _, t_cal = pool.run(wl_s, 2 * pool.cores, 1 << 12)       # warm + calibrate: aim at ~12 s of CPU work
        n_cpu = 1 << 12
        while n_cpu < (1 << 21) and t_cal * (2 * n_cpu / (1 << 12)) < 14.0:
            n_cpu *= 2
        cpu = cpu_baseline(wl_s, pool, 2 * pool.cores, n_cpu)
        if cpu["sample_s"] < 8.0 and n_cpu < (1 << 21):          # the calibration run carries the pool's start-up
            cpu = cpu_baseline(wl_s, pool, 2 * pool.cores, 2 * n_cpu)
        pool.close()

    # Sectors are independent integrals: ONE program of nsec_full * world sectors is sharded over the ranks
    # by longest-processing-time on the generator's operation counts (sharding.partition_sectors, SURVEY
    # 8(e)); every rank compiles and integrates its share, results are gathered once at the end.  Per-GPU
    # work is fixed as N grows: weak scaling.
    t0 = time.perf_counter()
    wl_all = make_workload(WORKLOAD, nsectors=nsec_full * world)
    if world > 1:
        mine = partition_sectors([s.naive_ops for s in wl_all.sectors], world)[rank]
    else:
        mine = list(range(nsec_full))
    wl = wl_all
    wl.sectors = [wl_all.sectors[i] for i in mine]
    t_gen = time.perf_counter() - t0
    stream = torch.cuda.Stream(dev)
    ctx = fb.Context(local, stream.cuda_stream)
    rule = fb.Rule.from_workload(wl)
    S = len(wl.sectors)
    sel = np.arange(S, dtype=np.int32)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)  # > 126 MB L2
    timer = Timer(torch, dev, stream, ctx, flush)
    torch.cuda.synchronize(dev)

    # ---- first result: fiesta_compile + the first fiesta_integrate, wall clock, nothing warmed up.
    # The program's threads assemble the native kernels while the call runs; sectors whose kernel is
    # not ready yet are served by the interpreter (same bits).
    t0 = time.perf_counter()
    prog = ctx.compile(wl.sectors, wl.dim)
    t_compile = time.perf_counter() - t0
    first = ctx.integrate(prog, wl.npoints, rule, wl.seed, sectors=sel)
    t_first = time.perf_counter() - t0
    first_tiers = ctx.last_tiers()
    n_native = prog.wait_native(wl.rule)
    t_all_native = time.perf_counter() - t0
    jit_stats = prog.native_stats()
    evals_per_step = wl.evals                                    # points x sectors x orders, this rank
    program_bytes = int(np.sum(prog.info["n_ir_ops"] + prog.info["n_deform_ops"] + 2)) * 16

    # ---- steady state: W warm-up + K timed steps, every sector on its native kernel
    peak_live = ctx.fp64_peak(100.0)                             # DFMA micro-benchmark, also a clock warm-up
    for i in range(W):
        timer.step(prog, wl, rule, i)
    torch.cuda.synchronize(dev)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize(dev)
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    step_ms, kern_ms, launches, tiers = timer.run(prog, wl, rule, 0, K, first=W)
    torch.cuda.synchronize(dev)
    clocks = sampler.stop() if rank == 0 else None
    if world > 1:
        dist.barrier()
    res = ctx.fetch_results(S, wl.K)
    total_ms = max_over_ranks(sum(step_ms), D, dev)
    if world > 1:
        t = torch.tensor([float(evals_per_step)], dtype=torch.float64, device=dev)
        dist.all_reduce(t)
        total_evals = float(t.item())
    else:
        total_evals = float(evals_per_step)

    # ---- end to end through the synchronous C-ABI call with HOST buffers: sector list + rule in,
    # results out, both copies inside the timed region
    e2e_t = []
    for i in range(max(1, min(K, 3))):
        with torch.cuda.stream(stream):
            flush.fill_(i)
        torch.cuda.synchronize(dev)
        t0 = time.perf_counter()
        out = ctx.integrate(prog, wl.npoints, rule, wl.seed + 100 + i, sectors=sel)
        e2e_t.append(time.perf_counter() - t0)
    e2e_s = max_over_ranks(sum(e2e_t) / len(e2e_t), D, dev)
    full = gather_results(res, mine, nsec_full * world, D, dev)
    ok = bool(np.all(np.isfinite(full["re"])) and np.all(full["n_nonfinite"] == 0) and np.all(full["re_err"] >= 0))
    # the first (hybrid) result is the same integral as a native-only pass with the same seed
    chk = ctx.integrate(prog, wl.npoints, rule, wl.seed, sectors=sel)
    ok = ok and first.tobytes() == chk.tobytes()
    roof = roofline_of(wl, prog, S, kern_ms, peak_live, tiers)
    info_line = prog.native(0, wl.rule)[1].replace("\n", " ")
    prog.close()

    # ---- extras (rank 0, N = 1, the bench workload only): first result on the interpreter alone, and the
    # complex (C4) and Vegas (C5) configurations at full size with their own roofline
    extra = {}
    if extras:
        os.environ["FIESTA_JIT"] = "0"
        t0 = time.perf_counter()
        prog_i = ctx.compile(wl.sectors, wl.dim)
        tci = time.perf_counter() - t0
        ctx.integrate(prog_i, wl.npoints, rule, wl.seed, sectors=sel)
        t_first_interp = time.perf_counter() - t0
        km_i, _ = ctx.last_timing()
        del os.environ["FIESTA_JIT"]
        prog_i.close()
        extra["e2e_first_result"] = {
            "unit": "s", "workload": f"{WORKLOAD}, {S} sectors, full size: fiesta_compile + first fiesta_integrate, wall clock",
            "default (interpreter at once, native kernels as the background threads finish them)": t_first,
            "default_compile_returns_after": t_compile,
            "default_sector_passes_native_vs_interpreter": list(first_tiers),
            "interpreter_only (FIESTA_JIT=0)": t_first_interp, "interpreter_only_compile": tci,
            "interpreter_only_pass_kernel_ms": km_i,
            "native_only (wait for all kernels, then one pass)": t_all_native + sum(e2e_t) / len(e2e_t),
            "all_native_kernels_ready_after": t_all_native,
            "assembly": {**jit_stats, "note": "cpu_seconds summed over the program's threads"}}
        for name, nsec_x in (("C4", args.c4_sectors), ("C5", args.c5_sectors)):
            wx = make_workload(name, nsectors=nsec_x) if nsec_x else make_workload(name)
            rx = fb.Rule.from_workload(wx)
            t0 = time.perf_counter()
            px = ctx.compile(wx.sectors, wx.dim)
            nn = px.wait_native(wx.rule)
            tcx = time.perf_counter() - t0
            sm, km, ln, tr = timer.run(px, wx, rx, 2, 2)
            rr = ctx.fetch_results(len(wx.sectors), wx.K)
            okx = bool(np.all(np.isfinite(rr["re"])) and np.all(rr["n_nonfinite"] == 0))
            rf = roofline_of(wx, px, len(wx.sectors), km, peak_live, tr)
            extra[name] = {"workload": f"BASELINE config {name[1]} ({name}), full size: " + describe(wx, len(wx.sectors)),
                           "value": wx.evals / (sum(sm) / len(sm) * 1e-3), "unit": UNIT, "ms_per_step": sum(sm) / len(sm),
                           "steps": 2, "warmup": 2, "native_sectors": nn, "compile_and_assemble_s": tcx,
                           "results_ok": okx, "gpu_launches": ln, "roofline": rf,
                           "assembler_report": px.native(0, wx.rule)[1].replace("\n", " ")[:400]}
            px.close()

    if rank == 0:
        line = {
            "metric": METRIC, "value": total_evals * K / (total_ms * 1e-3), "unit": UNIT, "n_gpus": world,
            "steps": K, "warmup": W, "ms_per_step": total_ms / K, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": (f"BASELINE config 3 ({WORKLOAD}): " + describe(wl, S) + " per GPU") if WORKLOAD == "C3" else
                                   (f"PROFILING RUN, not the bench line: BASELINE config {WORKLOAD[1]}, " + describe(wl, S)),
                       "sectors_per_gpu": S, "points_per_sector": wl.npoints, "orders": wl.K,
                       "naive_ops_per_point": wl.naive_ops_per_point, "ir_ops_per_point": float(np.mean(prog.info["n_ir_ops"])),
                       "l2": "flushed between iterations (256 MiB write); programs 16-32 MB, points made on device",
                       "parallelism": (f"{nsec_full * world} sectors sharded over {world} GPU(s) by longest-processing-time "
                                       "(sharding.partition_sectors), no data-path collective, one gather of the results"),
                       "tier": "native sm_100a kernel per sector" if tiers[1] == 0 else f"native/interpreter sector passes {tiers}",
                       "native_sectors": n_native, "assembler_report_sector0": info_line[:400],
                       "results_ok": ok, "generate_s": t_gen, "compile_returns_after_s": t_compile,
                       "all_native_kernels_ready_after_s": t_all_native},
            "gpu_launches": launches,
            "e2e": {"value": total_evals / e2e_s, "unit": UNIT, "h2d_bytes_per_step": int(sel.nbytes + 48),
                    "d2h_bytes_per_step": int(out.nbytes), "call": "fiesta_integrate (host sector list, host results)",
                    "first_result_s": t_first, "program_bytes_uploaded_once": program_bytes},
            "roofline": roof,
            "clocks": clocks,
        }
        line.update(extra)
        if cpu is not None:
            line["cpu_baseline"] = cpu
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    a = parse_args()
    sys.exit(run_reference(a) if a.impl == "reference" else run_b200(a))
