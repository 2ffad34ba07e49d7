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
    texts, sector_id, dim, n_lattice, a, r, seed = args
    sec = SectorSpec(texts, sector_id)
    gv = OP.korobov_genvec(a, n_lattice, dim)
    s1, s2, _ = OI.lattice_partial_sums(sec, n_lattice, 1, gv, r, seed)
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

    def run(self, wl, nsec, n_lattice):
        """Time the oracle on nsec sectors x n_lattice points (one shift).  -> (evals, seconds)."""
        from workloads import korobov_a
        a = korobov_a(n_lattice, wl.dim)
        tasks = [(s.texts, s.sector_id, wl.dim, n_lattice, a, wl.periodize_r, wl.seed) for s in wl.sectors[:nsec]]
        t0 = time.perf_counter()
        self.pool.map(_oracle_task, tasks, chunksize=1)
        dt = time.perf_counter() - t0
        return nsec * n_lattice * wl.K, dt


def cpu_baseline(wl, pool, nsec, n_lattice):
    evals, dt = pool.run(wl, nsec, n_lattice)
    return {"value": evals / dt, "unit": UNIT, "cores": pool.cores, "kind": "oracle",
            "sample": f"{nsec} sectors x {n_lattice} lattice points x {wl.K} orders of {WORKLOAD} "
                      f"(oracle/ as it stands: numpy long double, one process per core), {dt:.1f} s"}


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

def run_b200(args):
    import torch
    import torch.distributed as dist
    import paper_1511_03614_b200 as fb
    from paper_1511_03614_b200.sharding import gather_results, max_over_ranks
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

    # CPU oracle baseline first (rank 0, N=1 only), before this process touches CUDA heavily
    cpu = None
    global WORKLOAD
    WORKLOAD = args.workload
    nsec_full = args.sectors if args.sectors is not None else len(make_workload(WORKLOAD).sectors)
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        pool = OraclePool()
        wl_s = make_workload(WORKLOAD, nsectors=2 * pool.cores)
        _, t_cal = pool.run(wl_s, 2 * pool.cores, 1 << 12)       # warm + calibrate: aim at ~15 s of CPU work
        n_cpu = 1 << 12
        while n_cpu < (1 << 21) and t_cal * (2 * n_cpu / (1 << 12)) < 20.0:
            n_cpu *= 2
        cpu = cpu_baseline(wl_s, pool, 2 * pool.cores, n_cpu)
        pool.close()

    # weak scaling: every rank integrates its own nsec_full sectors (distinct sector ids => distinct streams)
    t0 = time.perf_counter()
    wl = make_workload(WORKLOAD, nsectors=nsec_full, first_sector=rank * nsec_full)
    t_gen = time.perf_counter() - t0
    stream = torch.cuda.Stream(dev)
    ctx = fb.Context(local, stream.cuda_stream)
    t0 = time.perf_counter()
    prog = ctx.compile(wl.sectors, wl.dim)
    t_compile = time.perf_counter() - t0
    rule = fb.Rule.from_workload(wl)
    S = len(wl.sectors)
    n_native = sum(1 for i in range(S) if prog.native(i)[0])     # sectors with an assembled native kernel
    evals_per_step = wl.evals                                    # points x sectors x orders, this rank
    flops_per_point = float(np.mean(prog.info["flops"]))         # nominal weights, DESIGN.md "Roofline"
    program_bytes = int(np.sum(prog.info["n_ir_ops"] + prog.info["n_deform_ops"] + 2)) * 16

    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)  # > 126 MB L2

    def one_step(i):
        with torch.cuda.stream(stream):
            flush.fill_(i & 0xff)                                # L2 flush between iterations (untimed)
            e0 = torch.cuda.Event(enable_timing=True)
            e1 = torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            ctx.integrate_async(prog, wl.npoints, rule, wl.seed + i)
            e1.record(stream)
        return e0, e1

    for i in range(W):
        one_step(i)
    torch.cuda.synchronize(dev)
    peak_live = ctx.fp64_peak(100.0)                             # DFMA micro-benchmark, also a clock warm-up
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize(dev)
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    step_ms, kern_ms, launches = [], [], 0
    for i in range(K):
        e0, e1 = one_step(W + i)
        e1.synchronize()
        step_ms.append(e0.elapsed_time(e1))
        km, nl = ctx.last_timing()
        kern_ms.append(km)
        launches += nl
    torch.cuda.synchronize(dev)
    clocks = sampler.stop() if rank == 0 else None
    if world > 1:
        dist.barrier()
    res = ctx.fetch_results(S, wl.K)
    total_ms = max_over_ranks(sum(step_ms), dist if world > 1 else None, dev)

    # end to end through the synchronous C-ABI call with HOST buffers: sector list + rule in,
    # results out, both copies inside the timed region
    sel = np.arange(S, dtype=np.int32)
    e2e_t = []
    for i in range(max(1, min(K, 3))):
        with torch.cuda.stream(stream):
            flush.fill_(i)
        torch.cuda.synchronize(dev)
        t0 = time.perf_counter()
        out = ctx.integrate(prog, wl.npoints, rule, wl.seed + 100 + i, sectors=sel)
        e2e_t.append(time.perf_counter() - t0)
    e2e_s = max_over_ranks(sum(e2e_t) / len(e2e_t), dist if world > 1 else None, dev)
    full = gather_results(res, list(range(rank * S, (rank + 1) * S)), world * S, dist if world > 1 else None, dev)
    ok = bool(np.all(np.isfinite(full["re"])) and np.all(full["n_nonfinite"] == 0) and np.all(full["re_err"] >= 0))

    if rank == 0:
        kms = sum(kern_ms) / len(kern_ms)
        ach = flops_per_point * wl.npoints * S / (kms * 1e-3) / 1e12
        line = {
            "metric": METRIC, "value": world * evals_per_step * K / (total_ms * 1e-3), "unit": UNIT, "n_gpus": world,
            "steps": K, "warmup": W, "ms_per_step": total_ms / K, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": (f"BASELINE config 3 ({WORKLOAD}): {S} sectors/GPU, dim {wl.dim}, {wl.K} orders, "
                                    f"{wl.npoints} points/sector = {wl.n_shifts} shifts x 2^{wl.n_lattice.bit_length() - 1} "
                                    f"Korobov lattice (a={wl.korobov_a}), periodising r={wl.periodize_r}") if WORKLOAD == "C3" else
                                   (f"PROFILING RUN, not the bench line: BASELINE config {WORKLOAD[1]}, {S} sectors/GPU, dim {wl.dim}, "
                                    f"{wl.K} orders, {wl.npoints} points/sector, rule {wl.rule}"),
                       "sectors_per_gpu": S, "points_per_sector": wl.npoints, "orders": wl.K,
                       "naive_ops_per_point": wl.naive_ops_per_point, "ir_ops_per_point": float(np.mean(prog.info["n_ir_ops"])),
                       "l2": "flushed between iterations (256 MiB write); programs 16-32 MB, points made on device",
                       "parallelism": f"sectors sharded over {world} GPU(s), no data-path collective",
                       "tier": ("native sm_100a kernel per sector (program lowered to PTX and assembled in fiesta_compile)"
                                if n_native == S else "interpreter (fx_ins walk)"),
                       "native_sectors": n_native,
                       "results_ok": ok, "generate_s": t_gen, "compile_s": t_compile},
            "gpu_launches": launches,
            "e2e": {"value": world * evals_per_step / e2e_s, "unit": UNIT, "h2d_bytes_per_step": int(sel.nbytes + 48),
                    "d2h_bytes_per_step": int(out.nbytes), "call": "fiesta_integrate (host sector list, host results)",
                    "compile_and_upload_s": t_compile, "program_bytes_uploaded_once": program_bytes},
            "roofline": {"bound": "alu", "achieved": ach, "peak": FP64_PEAK_TFLOPS, "unit": "TFLOP/s",
                         "frac": ach / FP64_PEAK_TFLOPS,
                         # dram__bytes_read+write of one native kernel launch (one sector, 2^24 points), ncu --set full,
                         # profiles/r01_ncu_fxj_integrate.md; the algorithmic traffic is the 256-byte partial records
                         "traffic": 55296 if n_native == S else None,
                         "kernel": "fxj_integrate (one launch per sector)" if n_native == S else "fx_integrate_real<8>",
                         "kernel_ms": kms, "kernel_launches_per_step": S if n_native == S else 1,
                         "kernel_ms_per_launch": kms / (S if n_native == S else 1),
                         "flops_per_point": flops_per_point,
                         "peak_source": "derived: 148 SM x 64 FP64 lanes x 2 x 1.965 GHz (MEASURED_PEAKS.json has no FP64 entry)",
                         "peak_dfma_microbench_live": peak_live},
            "clocks": clocks,
        }
        if cpu is not None:
            line["cpu_baseline"] = cpu
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    a = parse_args()
    sys.exit(run_reference(a) if a.impl == "reference" else run_b200(a))
