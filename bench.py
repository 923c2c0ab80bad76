#!/usr/bin/env python
"""bench.py — throughput of the M1 radiative-transfer hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--grid 4096] [--no-sweep]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

Workload (BASELINE.json configs[3]): the seeded random medium of m1_workloads.random_medium at 4096 x 4096
(16.8 M cells, 3 fp64 unknowns per cell).  One STEP = one pass of the whole hot path from the same initial state:
    reset state (device-to-device) -> 1 explicit step at CFL 0.4 (rows a1-a4)
                                   -> 1 implicit step at dt = 10 x explicit (rows a5-a7: assembly, GMRES(30)+block-Jacobi to 1e-10)
`value` = cells updated per second by the whole step = 2 N K / T (N cells, K steps, T = timed region, CUDA events).
The JSON line also carries, each measured in the same run with CUDA events:
    explicit  : cell-updates/s of the explicit kernel alone (>= 20 back-to-back steps), fraction of the HBM roofline (64 B/cell)
    implicit  : per dt ratio 10/50/100/200: iterations, ms, cell-updates/s, cell-iterations/s, bytes/iteration, HBM fraction
    break_even: T_implicit(K)/T_explicit vs K (implicit pays off where the ratio < K), beside the paper's 50-100x
    roofline  : the dominant kernel class of the step (by device time), from per-launch CUDA events inside the timed region
    kernels   : the same for every kernel class
    e2e       : the same step through the C ABI with HOST (pinned) buffers: H2D of the 5 input planes and D2H of the 3
                state planes of EVERY step inside the timed region, with the library's overlapped transfers (the next step's
                upload and the last step's download run on the handle's copy stream beside the solve); `e2e.blocking` = the same
                with ark_m1_set_state / ark_m1_get_state, copies and solve in series
    cpu_baseline : the oracle (oracle/oracle_m1.c, as it stands) on a bounded sample of the same workload
Multi-GPU (torchrun): the path does not exchange data between GPUs (one-GPU north star): every rank runs an independent
replica with its own seed, value = sum of units / max-over-ranks time ("scaling": "weak", no collective on the data path).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import m1_workloads as wl  # noqa: E402

METRIC = "M1 cell-updates/s (explicit step + implicit step per pass)"
UNIT = "cell-updates/s"
TOL, RESTART, MAXIT = 1e-10, 30, 4000
BENCH_DT_RATIO = 10.0
SWEEP = (10.0, 50.0, 100.0, 200.0)
PAPER_BREAK_EVEN = "50-100x (relaxation preconditioner; CPU 50, K80 GPU 100; PAPER.md:369)"
FP64_INSTR_PER_CELL = 156       # fp64-pipe instructions (DFMA/DMUL/DADD/DSETP) per cell in the row loop of explicit_march3_kernel (SASS count)


def load_ncu_traffic():
    """profiles/ncu_traffic.csv: measured DRAM bytes over algorithmic bytes per kernel class (copied from the ncu captures)."""
    import csv
    path = os.path.join(ROOT, "profiles", "ncu_traffic.csv")
    out = {}
    if os.path.exists(path):
        with open(path, newline="") as f:
            for row in csv.DictReader(f):
                d = {"captured": row["captured"], "dram_bytes": float(row["dram_bytes"]), "alg_bytes": float(row["alg_bytes"]),
                     "ratio": float(row["ratio"]), "note": row["note"], "alu_note": row["note"]}
                if row["fp64_pipe_busy_frac"]:
                    d["fp64_pipe_busy_frac"] = float(row["fp64_pipe_busy_frac"])
                    d["issue_slots_busy_frac"] = float(row["issue_slots_busy_frac"])
                out[row["class"]] = d
    return out


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return float(p["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


# --------------------------------------------------------------------------------------------------------------
# clocks
# --------------------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.path = index, None, None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        try:
            for line in open(self.path):
                p = [x.strip() for x in line.split(",")]
                if len(p) < 7:
                    continue
                try:
                    sm.append(float(p[0])); mx.append(float(p[1]))
                except ValueError:
                    continue
                for k, nm in enumerate(names):
                    if p[3 + k].lower().startswith("active"):
                        reasons.add(nm)
            os.unlink(self.path)
        except Exception:
            pass
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), reasons=sorted(reasons), samples=len(sm))
        return out


# --------------------------------------------------------------------------------------------------------------
# reference arm / cpu baseline: the oracle on a bounded sample
# --------------------------------------------------------------------------------------------------------------
def oracle_set_threads(nthreads):
    """Set the OpenMP team size of the oracle's next parallel regions (libgomp runtime call; None = leave as is)."""
    if nthreads is None:
        return
    import ctypes
    ctypes.CDLL("libgomp.so.1").omp_set_num_threads(int(nthreads))


def oracle_step_time(n_sample, seed, steps, warmup, threads=None):
    """Times `steps` passes (explicit step + implicit 10x step from the same state) of the oracle at n_sample^2; the explicit and
    the implicit part are also timed separately."""
    from oracle.oracle_m1 import OracleM1, num_threads
    all_cores = num_threads()
    oracle_set_threads(threads)
    w = wl.random_medium(n_sample, seed=seed)
    dt = wl.explicit_dt(w["dx"], w["dy"], w["c"])
    o = OracleM1(w["nx"], w["ny"], w["dx"], w["dy"], w["c"], bc=w["bc"])
    times, t_exp, t_imp, its = [], [], [], 0
    for k in range(warmup + steps):
        o.set_state(w["E"], w["F"], w["sigma_a"], w["sigma_s"])
        t0 = time.perf_counter()
        o.step_explicit(dt)
        t1 = time.perf_counter()
        its, _ = o.step_implicit(BENCH_DT_RATIO * dt, TOL, RESTART, MAXIT)
        t2 = time.perf_counter()
        if k >= warmup:
            times.append(t2 - t0); t_exp.append(t1 - t0); t_imp.append(t2 - t1)
    total = float(sum(times))
    out = dict(seconds=total, per_step=total / max(steps, 1), cells=n_sample * n_sample, iterations=its,
               cores=(threads if threads is not None else all_cores), explicit_s=float(sum(t_exp)) / max(steps, 1),
               implicit_s=float(sum(t_imp)) / max(steps, 1))
    oracle_set_threads(all_cores if threads is not None else None)
    return out


def oracle_protocol(n, seed):
    """The oracle timings SURVEY.md 8(d) lists, at the bench size: explicit alone (3 steps) and one capped GMRES cycle
    (maxit = restart = 30 -> seconds per iteration), with all cores and with 1 thread; full solves at 1024^2, dt = 50x
    (config 3).  Takes minutes; opt-in (--oracle-protocol)."""
    from oracle.oracle_m1 import OracleM1, num_threads
    all_cores = num_threads()
    out = {"grid": n, "all_cores": all_cores}
    w = wl.random_medium(n, seed=seed)
    dt = wl.explicit_dt(w["dx"], w["dy"], w["c"])
    N = n * n
    for label, th in (("all_cores", all_cores), ("one_thread", 1)):
        oracle_set_threads(th)
        o = OracleM1(w["nx"], w["ny"], w["dx"], w["dy"], w["c"], bc=w["bc"])
        o.set_state(w["E"], w["F"], w["sigma_a"], w["sigma_s"])
        nst = 3 if th > 1 else 1
        t0 = time.perf_counter()
        for _ in range(nst):
            o.step_explicit(dt)
        te = (time.perf_counter() - t0) / nst
        o.set_state(w["E"], w["F"], w["sigma_a"], w["sigma_s"])
        t0 = time.perf_counter()
        its, res = o.step_implicit(BENCH_DT_RATIO * dt, TOL, RESTART, RESTART)       # one capped cycle
        ti = time.perf_counter() - t0
        out[label] = {"threads": th, "explicit_steps_timed": nst, "explicit_s_per_step": te, "explicit_cell_updates_per_s": N / te,
                      "implicit_capped_cycle_s": ti, "implicit_iterations": its, "implicit_s_per_iteration": ti / max(its, 1),
                      "implicit_extrapolated_s_per_solve_85_iterations": 85 * ti / max(its, 1)}
        del o
    oracle_set_threads(all_cores)
    w3 = wl.random_medium(1024, seed=seed)
    dt3 = wl.explicit_dt(w3["dx"], w3["dy"], w3["c"])
    o = OracleM1(w3["nx"], w3["ny"], w3["dx"], w3["dy"], w3["c"], bc=w3["bc"])
    o.set_state(w3["E"], w3["F"], w3["sigma_a"], w3["sigma_s"])
    t0 = time.perf_counter()
    its, res = o.step_implicit(50.0 * dt3, TOL, RESTART, MAXIT)
    out["config3_1024_dt50"] = {"threads": all_cores, "iterations": its, "final_residual": res, "s_per_solve": time.perf_counter() - t0}
    return out


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    n_s = args.ref_n
    r = oracle_step_time(n_s, args.seed, args.steps, args.warmup)
    value = 2.0 * r["cells"] * args.steps / r["seconds"]
    sample = (f"{n_s}x{n_s} grid of the same seeded random-medium generator ({r['cells'] / (args.n * args.n):.4f} of the "
              f"{args.n}x{args.n} workload's cells) per step, {r['iterations']} GMRES iterations per implicit step")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * r["per_step"], "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": f"M1 random medium (BASELINE.json configs[3]) {args.n}x{args.n}, fp64, periodic; reference arm = "
                               f"CPU oracle on a bounded sample", "step": "1 explicit step (CFL 0.4) + 1 implicit step (dt = 10x, "
                               "GMRES(30) + block-Jacobi, tol 1e-10)", "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": r["cores"], "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# --------------------------------------------------------------------------------------------------------------
# our arm
# --------------------------------------------------------------------------------------------------------------
def aggregate_over_ranks(elapsed_s, units, dist=None):
    """(max elapsed over ranks, total units over ranks).  `dist` = torch.distributed or None for one process."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return elapsed_s, units
    import torch
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([elapsed_s], dtype=torch.float64, device=dev)
    u = torch.tensor([float(units)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


ARNOLDI_BLOCK = 5      # the library's default (option arnoldi_block): columns per pass over the basis


def iteration_bytes_per_cell(iters, m=RESTART, operator=0, block=None, pair=None):
    """Algorithmic HBM bytes per cell of `iters` GMRES iterations with the kernels as built:
    operator 336 (block stencil) or 136 (matrix-free with the diagonal block and J rebuilt in the kernel, the default; 264 when it
    loads M^-1 and J).  Matrix-free default = s-step Arnoldi blocks of `block` = 5 columns per pass over the basis: per block at inner
    index j five operator applications, one dot pass 24 (j+1 + 5) (per 32 vectors; the block's own slots are dotted like basis vectors
    from L1 / L2 and predict the in-block solve), one update pass 24 (j+1) + 48*5 that applies the predicted solve; a block whose
    prediction is not used adds a pass of 24 (2*5 - 1) (none on the bench medium: `block_stats` in the line; not in this model);
    columns left over go through the two-column step (two operator applications, dots 24 (j+1) + 48 per
    chunk of 8 vectors, update 24 (j+1) + 96, the W2 - gamma W1 pass 72) or the one-column step (dots 24 (j+2), update+norm 24 (j+3), one
    extra read of w per 16-vector pass), which the block-stencil path uses throughout.  Per cycle: combine 8 (3 jj + 15) + true residual
    (block stencil: diag_mul 120 + spmv 360; matrix-free: 216) + norm 24.  A block is enqueued whole: its operator applications, dot
    and update passes are paid even when the cycle stops after its first column.  `pair` (default: with the matrix-free operator; the
    bench medium is periodic): inside a block two operator applications go through one pass (160 B per pair instead of 2 x 136:
    coefficient planes read once, the intermediate vector written but not read back)."""
    if block is None:
        block = ARNOLDI_BLOCK if operator == 1 else 1
    if pair is None:
        pair = operator == 1
    op = 336.0 if operator == 0 else 136.0
    res = 480.0 if operator == 0 else 216.0
    total, done = 0.0, 0
    while done < iters:
        jj = min(m, iters - done)
        j = 0
        while j < jj:
            if block >= 3 and j + block <= m:
                total += ((block // 2) * 160.0 + (block % 2) * op) if pair else block * op
                total += 24.0 * (j + 1) + 24.0 * block * ((j + block) // 32 + 1) + 24.0 * (j + 1) + 48.0 * block
                j += block
            elif block >= 2 and j + 1 < m:
                chunks = j // 8 + 1
                total += (160.0 if pair else 2.0 * op) + 24.0 * (j + 1) + 48.0 * chunks + 24.0 * (j + 1) + 96.0 + (72.0 if j + 1 < jj else 0.0)
                j += 2
            else:
                passes = j // 16 + 1
                total += op + 24.0 * (j + 1 + passes) + 24.0 * (j + 1 + 2 * passes)
                j += 1
        total += 8.0 * (3 * jj + 15) + res + 24.0
        done += jj
    return total


def bicgstab_bytes_per_cell(iters, operator=1):
    """Algorithmic bytes per cell of `iters` BiCGStab iterations as built.  Matrix-free operator (reductions fused into the
    operator kernel): p update 96 + [A M^-1 p with <r^,v>] 160 + s update 72 + [A M^-1 s with <t,s>,<t,t>] 136 + y/r update with
    rho, ||r|| 168 = 632.  Block stencil: 2 x 336 + 96 + 48 + 72 + 72 + 168 = 1128.  One cycle end: x += M^-1 y (168), true
    residual, norm (24), cycle start (96)."""
    per_it = 632.0 if operator == 1 else 1128.0
    res = 480.0 if operator == 0 else 216.0
    return iters * per_it + 168.0 + res + 24.0 + 96.0


def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_2011_13926_b200 as ark

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device — the CUDA library is the only implementation (no CPU fallback)")
    # ARK_BENCH_SHARE_GPU=1 (test only): all ranks use cuda:0 and rendezvous over gloo, to exercise the N > 1 code path on a
    # one-GPU box; the replicas never wait on one another on the device (no data-path collective)
    share = os.environ.get("ARK_BENCH_SHARE_GPU") == "1"
    if share:
        local = 0
    torch.cuda.set_device(local)
    if world > 1:
        if share:
            dist.init_process_group("gloo")
        else:
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)
    peak_gbs, peak_src = peaks()

    n = args.n
    N = n * n
    w = wl.random_medium(n, seed=args.seed + rank)
    dt_e = wl.explicit_dt(w["dx"], w["dy"], w["c"])
    host = {k: torch.from_numpy(np.ascontiguousarray(w[k])).pin_memory() for k in ("E", "F", "sigma_a", "sigma_s")}
    devt = {k: v.to(dev) for k, v in host.items()}
    out_E = torch.empty((n, n), dtype=torch.float64).pin_memory()
    out_F = torch.empty((2, n, n), dtype=torch.float64).pin_memory()
    stream = torch.cuda.current_stream()
    g = ark.ArkM1(n, n, w["dx"], w["dy"], w["c"], bc=w["bc"], stream=stream)
    g.set_option("operator", args.operator)
    if args.preconditioner == 1:
        g.set_option("preconditioner", 1); g.set_option("mg_precision", args.mg_precision)

    def reset_device():
        g.set_state(devt["E"], devt["F"], devt["sigma_a"], devt["sigma_s"])

    def one_step(ratio=BENCH_DT_RATIO):
        g.step_explicit(dt_e)
        return g.step_implicit(ratio * dt_e, TOL, RESTART, MAXIT)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- explicit kernel alone, first: BURST (best of 5 x >= 40 back-to-back steps, ~10 ms each, boost clock) and SUSTAINED
    #      (one back-to-back run of >= 2 s, the regime of the paper's explicit route: 73 823 consecutive steps),
    #      each with its own clock record.  The kernel is fp64-issue bound, so its time follows the SM clock.
    rates = ark.fp64_issue_rate()      # measured fp64 issue rate of this GPU (the "alu" roofline below)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    reset_device()
    g.steps_explicit(dt_e, 10)
    torch.cuda.synchronize()
    n_exp = max(40, 4 * args.steps)
    smp = ClockSampler(local)
    smp.start()
    time.sleep(0.3)
    best, all_ms = None, []
    for _ in range(5):
        e0.record(stream)
        g.steps_explicit(dt_e, n_exp)
        e1.record(stream)
        torch.cuda.synchronize()
        t_ms = e0.elapsed_time(e1) / n_exp
        all_ms.append(t_ms)
        best = t_ms if best is None else min(best, t_ms)
    exp_clocks = smp.stop()
    n_sus = int(max(200, args.sustain_s * 1e3 / best))
    smp = ClockSampler(local)
    smp.start()
    e0.record(stream)
    g.steps_explicit(dt_e, n_sus)
    e1.record(stream)
    torch.cuda.synchronize()
    sus_ms = e0.elapsed_time(e1) / n_sus
    sus_clocks = smp.stop()
    exp_gbs = 64.0 * N / (best * 1e-3) / 1e9
    sus_gbs = 64.0 * N / (sus_ms * 1e-3) / 1e9
    alu_peak = rates["dfma_lanes_per_clk_sm"] * rates["sm_count"] * rates["sm_mhz"] * 1e6       # fp64 lane-instructions per second
    alu_work = FP64_INSTR_PER_CELL * (32.0 / 30.0) * N                                           # halo lanes compute too
    explicit_info = {"cell_updates_per_s": N / (sus_ms * 1e-3), "ms_per_step": sus_ms, "bytes_per_cell": 64,
                     "achieved_gbs": sus_gbs, "hbm_frac": sus_gbs / peak_gbs,
                     "sustained": {"ms_per_step": sus_ms, "steps_timed": n_sus, "hbm_frac": sus_gbs / peak_gbs, "clocks": sus_clocks},
                     "burst": {"ms_per_step": best, "median_ms_per_step": float(np.median(all_ms)), "steps_timed": n_exp, "repeats": 5,
                               "cell_updates_per_s": N / (best * 1e-3), "hbm_frac": exp_gbs / peak_gbs, "clocks": exp_clocks},
                     "alu": {"bound": "alu", "pipe": "fp64", "unit": "fp64 lane-instructions/s",
                             "fp64_instr_per_cell": FP64_INSTR_PER_CELL, "lanes_factor": 32.0 / 30.0,
                             "peak": alu_peak, "achieved_sustained": alu_work / (sus_ms * 1e-3), "achieved_burst": alu_work / (best * 1e-3),
                             "frac_sustained": alu_work / (sus_ms * 1e-3) / alu_peak, "frac_burst": alu_work / (best * 1e-3) / alu_peak,
                             "peak_source": "ark_m1_fp64_issue_rate on this GPU in this run: DFMA lanes/clk/SM x SMs x SM clock measured during the test",
                             "issue_rates": rates},
                     "bound": "fp64 issue (DESIGN.md section 6): 156 fp64 + 106 other instructions per cell"}

    # ---- main timed region: W warm-up + exactly K steps, inputs resident in HBM ----------------------------------
    for _ in range(args.warmup):
        reset_device(); one_step()
    g.set_option("kernel_timing", 1)
    sampler = ClockSampler(local)
    launches0 = g.kernel_launches()
    barrier()
    sampler.start()
    e0.record(stream)
    its_main = 0
    for _ in range(args.steps):
        reset_device()
        its_main, res_main = one_step()
    e1.record(stream)
    barrier()
    clocks = sampler.stop()
    elapsed = e0.elapsed_time(e1) * 1e-3
    launches = g.kernel_launches() - launches0
    stats = g.kernel_stats()
    g.set_option("kernel_timing", 0)
    t_max, units = aggregate_over_ranks(elapsed, 2.0 * N * args.steps, dist if world > 1 else None)
    value = units / t_max

    # ---- e2e: same step through the C ABI with pinned HOST buffers -------------------------------------------------
    # (a) blocking calls: upload, step, download in series (ark_m1_set_state / ark_m1_get_state)
    def e2e_step():
        g.set_state(host["E"], host["F"], host["sigma_a"], host["sigma_s"])
        one_step()
        g.get_state(out=(out_E, out_F))
    e2e_step()
    barrier()
    k_e2e = max(1, min(args.steps, 3))
    e0.record(stream)
    for _ in range(k_e2e):
        e2e_step()
    e1.record(stream)
    barrier()
    t_ser, u_ser = aggregate_over_ranks(e0.elapsed_time(e1) * 1e-3, 2.0 * N * k_e2e, dist if world > 1 else None)
    # (b) the same loop with the library's overlapped transfers (csrc/pipeline.cu): every step's 5 input planes still come from the
    # pinned host buffers and its 3 result planes still go back to them inside the timed region, but step k+1's upload and step k's
    # download run on the handle's copy stream beside the solve.  The first upload and the last download are exposed and timed.
    def e2e_pipelined(k):
        g.prefetch_state(host["E"], host["F"], host["sigma_a"], host["sigma_s"])
        for s_ in range(k):
            g.commit_state()
            if s_ + 1 < k:
                g.prefetch_state(host["E"], host["F"], host["sigma_a"], host["sigma_s"])
            one_step()
            g.get_state_async((out_E, out_F))
        g.wait_transfers()
    e2e_pipelined(1)
    barrier()
    k_pipe = max(1, args.steps)
    e0.record(stream)
    e2e_pipelined(k_pipe)
    e1.record(stream)
    barrier()
    t_e2e, u_e2e = aggregate_over_ranks(e0.elapsed_time(e1) * 1e-3, 2.0 * N * k_pipe, dist if world > 1 else None)
    e2e = {"value": u_e2e / t_e2e, "unit": UNIT, "h2d_bytes_per_step": 5 * N * 8, "d2h_bytes_per_step": 3 * N * 8, "steps": k_pipe,
           "api": "ark_m1_prefetch_state / commit_state / step_explicit / step_implicit / get_state_async / wait_transfers: the next step's upload and "
                  "the last step's download overlap the solve; first upload and last download exposed",
           "blocking": {"value": u_ser / t_ser, "steps": k_e2e, "api": "ark_m1_set_state / step_explicit / step_implicit / ark_m1_get_state, in series"}}

    line_extra = {}
    if rank == 0:
        line_extra["explicit"] = explicit_info
        ms_exp = explicit_info["ms_per_step"]          # SUSTAINED explicit step: the denominator of every break-even statement
        traffic = load_ncu_traffic()
        if n == 4096 and "explicit" in traffic:
            explicit_info["traffic"] = traffic["explicit"]["dram_bytes"]
            explicit_info["alu"]["ncu_fp64_pipe_busy_frac"] = traffic["explicit"].get("fp64_pipe_busy_frac")
        # ---- implicit sweep ----------------------------------------------------------------------------------------
        imp, brk = {}, {}
        ratios = SWEEP if not args.no_sweep else (BENCH_DT_RATIO,)
        for ratio in ratios:
            reset_device()
            torch.cuda.synchronize()
            e0.record(stream)
            its, res = g.step_implicit(ratio * dt_e, TOL, RESTART, MAXIT)
            e1.record(stream)
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1)
            tm = g.timings()
            nE, nf = g.count_unrealizable()
            bpc = iteration_bytes_per_cell(its, operator=args.operator)
            kry_gbs = bpc * N / (tm["krylov_ms"] * 1e-3) / 1e9 if its > 0 else None
            imp[f"{ratio:g}x"] = {"iterations": its, "final_residual": res, "ms": ms, "assembly_ms": tm["assembly_ms"], "krylov_ms": tm["krylov_ms"],
                                  "ms_per_iteration": tm["krylov_ms"] / max(its, 1), "cell_updates_per_s": N / (ms * 1e-3),
                                  "cell_iterations_per_s": N * its / (ms * 1e-3), "bytes_per_cell_per_iteration": bpc / max(its, 1),
                                  "krylov_achieved_gbs": kry_gbs, "krylov_hbm_frac": (kry_gbs / peak_gbs) if kry_gbs else None,
                                  "cells_E_nonpositive": nE, "cells_f_above_one": nf, "block_stats": g.block_stats()}
            brk[f"{ratio:g}x"] = {"T_implicit_over_T_explicit": ms / ms_exp, "implicit_wins": bool(ms / ms_exp < ratio)}
        line_extra["implicit"] = imp
        wins = [k for k, v in brk.items() if v["implicit_wins"]]
        line_extra["break_even"] = {"per_ratio": brk, "reached_in_sweep": bool(wins), "first_winning_ratio": wins[0] if wins else None,
                                    "paper": PAPER_BREAK_EVEN}
        # ---- restart length (the one free parameter north_star leaves the solver; SURVEY 8(f) row 4 "longer restart") ------------
        if args.restart_sweep:
            rsw = {}
            for ngrid in (1024, n):
                wr = w if ngrid == n else wl.random_medium(ngrid, seed=args.seed)
                dtr = wl.explicit_dt(wr["dx"], wr["dy"], wr["c"])
                tr_ = devt if ngrid == n else {k: torch.from_numpy(np.ascontiguousarray(wr[k])).to(dev) for k in ("E", "F", "sigma_a", "sigma_s")}
                gr = g if ngrid == n else ark.ArkM1(ngrid, ngrid, wr["dx"], wr["dy"], wr["c"], bc=wr["bc"], stream=stream)
                tab = {}
                for m_ in (30, 60, 100):
                    for ratio in (50.0, 100.0, 200.0):
                        gr.set_state(tr_["E"], tr_["F"], tr_["sigma_a"], tr_["sigma_s"])
                        torch.cuda.synchronize()
                        e0.record(stream)
                        its, res = gr.step_implicit(ratio * dtr, TOL, m_, MAXIT)
                        e1.record(stream)
                        torch.cuda.synchronize()
                        tab[f"m{m_}_{ratio:g}x"] = {"restart": m_, "dt_ratio": ratio, "iterations": its, "final_residual": res, "converged": bool(res <= TOL),
                                                    "ms": e0.elapsed_time(e1), "device_bytes": gr.device_bytes()}
                rsw[f"{ngrid}x{ngrid}"] = tab
                if ngrid != n:
                    gr.close()
                else:
                    g.set_option("release_workspace", 1)      # give the 100-vector basis back before the remaining sections
            line_extra["restart_sweep"] = rsw
        # ---- smooth problem (config-1 type: Gaussian, sigma_s = 1e3, at the bench resolution): where implicit comes closest --
        if not args.no_sweep:
            ws = wl.gaussian_diffusion(n)
            devs = {k: torch.from_numpy(np.ascontiguousarray(ws[k])).to(dev) for k in ("E", "F", "sigma_a", "sigma_s")}
            sm_out = {}
            for ratio in (50.0, 100.0, 200.0, 1000.0):
                g.set_state(devs["E"], devs["F"], devs["sigma_a"], devs["sigma_s"])
                torch.cuda.synchronize()
                e0.record(stream)
                its, res = g.step_implicit(ratio * dt_e, TOL, RESTART, MAXIT)
                e1.record(stream)
                torch.cuda.synchronize()
                ms = e0.elapsed_time(e1)
                sm_out[f"{ratio:g}x"] = {"iterations": its, "final_residual": res, "ms": ms, "T_implicit_over_T_explicit": ms / ms_exp,
                                         "over_K": ms / ms_exp / ratio, "implicit_wins": bool(ms / ms_exp < ratio)}
            best_k = min(sm_out, key=lambda k: sm_out[k]["over_K"])
            line_extra["break_even"]["smooth_problem"] = {"workload": f"Gaussian pulse, sigma_s = 1e3, {n}x{n} (config-1 type at bench resolution)",
                                                          "per_ratio": sm_out, "closest": best_k, "closest_T_implicit_over_K_T_explicit": sm_out[best_k]["over_K"],
                                                          "reached": bool(any(v["implicit_wins"] for v in sm_out.values()))}
            del devs
        # ---- BiCGStab (the paper's Krylov method): same sweeps, option krylov = 1 -------------------------
        if not args.no_sweep:
            g.set_option("krylov", 1)
            bi = {"rough_medium": {}, "smooth_problem": {}}
            for label, tensors, ratios in (("rough_medium", devt, (10.0, 50.0, 100.0, 200.0)),
                                           ("smooth_problem", None, (50.0, 100.0, 200.0, 300.0, 500.0, 1000.0, 2000.0))):
                if tensors is None:
                    ws = wl.gaussian_diffusion(n)
                    tensors = {k: torch.from_numpy(np.ascontiguousarray(ws[k])).to(dev) for k in ("E", "F", "sigma_a", "sigma_s")}
                for ratio in ratios:
                    g.set_state(tensors["E"], tensors["F"], tensors["sigma_a"], tensors["sigma_s"])
                    torch.cuda.synchronize()
                    e0.record(stream)
                    its, res = g.step_implicit(ratio * dt_e, TOL, RESTART, MAXIT)
                    e1.record(stream)
                    torch.cuda.synchronize()
                    ms = e0.elapsed_time(e1)
                    tm = g.timings()
                    gbs = bicgstab_bytes_per_cell(its, args.operator) * N / (tm["krylov_ms"] * 1e-3) / 1e9 if its > 0 else None
                    bi[label][f"{ratio:g}x"] = {"iterations": its, "operator_applications": 2 * its, "final_residual": res, "ms": ms,
                                                "ms_per_iteration": tm["krylov_ms"] / max(its, 1), "krylov_hbm_frac": (gbs / peak_gbs) if gbs else None,
                                                "T_implicit_over_T_explicit": ms / ms_exp, "over_K": ms / ms_exp / ratio,
                                                "implicit_wins": bool(ms / ms_exp < ratio)}
            wins = [f"{lab}:{k}" for lab, d in bi.items() for k, v in d.items() if v["implicit_wins"]]
            bi["break_even_reached_at"] = wins
            line_extra["bicgstab"] = bi
            g.set_option("krylov", 0)
        # ---- compressed-basis GMRES (option basis_precision = 32: Arnoldi vectors stored in fp32, fp64 arithmetic and fp64 exit test) ----
        if not args.no_sweep:
            g.set_option("basis_precision", 32)
            cbo = {"rough_medium": {}, "smooth_problem": {}}
            for label, tensors, ratios in (("rough_medium", devt, (10.0, 50.0)), ("smooth_problem", None, (100.0,))):
                if tensors is None:
                    ws = wl.gaussian_diffusion(n)
                    tensors = {k: torch.from_numpy(np.ascontiguousarray(ws[k])).to(dev) for k in ("E", "F", "sigma_a", "sigma_s")}
                for ratio in ratios:
                    for rep in range(2 if (label == "rough_medium" and ratio == 10.0) else 1):      # first call allocates the fp32 basis
                        g.set_state(tensors["E"], tensors["F"], tensors["sigma_a"], tensors["sigma_s"])
                        torch.cuda.synchronize()
                        e0.record(stream)
                        its, res = g.step_implicit(ratio * dt_e, TOL, RESTART, MAXIT)
                        e1.record(stream)
                        torch.cuda.synchronize()
                    ms = e0.elapsed_time(e1)
                    tm = g.timings()
                    cbo[label][f"{ratio:g}x"] = {"iterations": its, "final_residual": res, "converged": bool(res <= TOL), "ms": ms,
                                                 "ms_per_iteration": tm["krylov_ms"] / max(its, 1),
                                                 "bytes_per_cell_per_iteration_mean_m30": 556, "T_implicit_over_T_explicit": ms / ms_exp}
            reset_device(); one_step()
            torch.cuda.synchronize()
            e0.record(stream)
            for _ in range(3):
                reset_device()
                its_v, res_v = one_step()
            e1.record(stream)
            torch.cuda.synchronize()
            ms_v = e0.elapsed_time(e1) / 3
            cbo["bench_step_variant"] = {"step": "state reset + 1 explicit + 1 implicit (10x, GMRES(30) + block-Jacobi, fp32-stored basis)", "ms_per_step": ms_v,
                                         "cell_updates_per_s": 2.0 * N / (ms_v * 1e-3), "iterations": its_v, "final_residual": res_v}
            line_extra["compressed_basis"] = cbo
            g.set_option("basis_precision", 64)
        # ---- multigrid preconditioner (SURVEY 8(f) row 4 "stronger preconditioner"): option preconditioner = 1,
        #      blocks stored in fp32 (mg_precision = 32); BiCGStab on the rough medium, GMRES(30) on the smooth problem ----------------
        if not args.no_sweep:
            g.set_option("preconditioner", 1); g.set_option("mg_precision", 32)
            mgo = {"rough_medium": {}, "smooth_problem": {}, "options": {"preconditioner": 1, "mg_precision": 32, "mg_omega": 0.8,
                                                                         "rough_medium_krylov": "bicgstab", "smooth_problem_krylov": "gmres(30)"}}
            reset_device()
            g.step_implicit(BENCH_DT_RATIO * dt_e, TOL, RESTART, 2)        # untimed: allocates the hierarchy
            for label, tensors, ratios, kry in (("rough_medium", devt, (10.0, 50.0, 100.0, 200.0), 1),
                                                ("smooth_problem", None, (50.0, 100.0, 200.0, 300.0, 500.0, 1000.0, 2000.0), 0)):
                g.set_option("krylov", kry)
                if tensors is None:
                    ws = wl.gaussian_diffusion(n)
                    tensors = {k: torch.from_numpy(np.ascontiguousarray(ws[k])).to(dev) for k in ("E", "F", "sigma_a", "sigma_s")}
                for ratio in ratios:
                    g.set_state(tensors["E"], tensors["F"], tensors["sigma_a"], tensors["sigma_s"])
                    torch.cuda.synchronize()
                    e0.record(stream)
                    its, res = g.step_implicit(ratio * dt_e, TOL, RESTART, 400)
                    e1.record(stream)
                    torch.cuda.synchronize()
                    ms = e0.elapsed_time(e1)
                    tm = g.timings()
                    mgo[label][f"{ratio:g}x"] = {"iterations": its, "preconditioner_applications": (2 if kry else 1) * its, "final_residual": res,
                                                 "converged": bool(res <= TOL), "ms": ms, "setup_ms": tm["assembly_ms"],
                                                 "ms_per_iteration": tm["krylov_ms"] / max(its, 1),
                                                 "T_implicit_over_T_explicit": ms / ms_exp, "over_K": ms / ms_exp / ratio,
                                                 "implicit_wins": bool(res <= TOL and ms / ms_exp < ratio)}
            # the bench step itself (reset + explicit + implicit 10x) with the multigrid preconditioner: a variant, not the headline
            g.set_option("krylov", 0)
            reset_device(); one_step()
            torch.cuda.synchronize()
            e0.record(stream)
            for _ in range(3):
                reset_device()
                its_v, res_v = one_step()
            e1.record(stream)
            torch.cuda.synchronize()
            ms_v = e0.elapsed_time(e1) / 3
            mgo["bench_step_variant"] = {"step": "state reset + 1 explicit + 1 implicit (10x, GMRES(30) + multigrid V-cycle)", "ms_per_step": ms_v,
                                         "cell_updates_per_s": 2.0 * N / (ms_v * 1e-3), "iterations": its_v, "final_residual": res_v}
            mgo["break_even_reached_at"] = [f"{lab}:{k}" for lab in ("rough_medium", "smooth_problem") for k, v in mgo[lab].items() if v["implicit_wins"]]
            line_extra["multigrid"] = mgo
            g.set_option("preconditioner", 0); g.set_option("krylov", 0)
        # ---- stage 2 (row a8, BASELINE.json configs[4]): matter coupling + point source + velocity sources at 2048^2 ----------
        if not args.no_sweep and not args.no_stage2:
            w5 = wl.stratified_coupled(2048, seed=4321)
            N5 = w5["nx"] * w5["ny"]
            dt5 = 100.0 * wl.explicit_dt(w5["dx"], w5["dy"], w5["c"])
            g5 = ark.ArkM1(w5["nx"], w5["ny"], w5["dx"], w5["dy"], w5["c"], bc=w5["bc"], stream=stream)
            g5.set_option("operator", args.operator)
            d5 = {k: torch.from_numpy(np.ascontiguousarray(w5[k])).to(dev) for k in ("E", "F", "sigma_a", "sigma_s", "T", "rho_cv", "ux", "uy", "source_E")}
            for name in ("rho_cv", "ux", "uy", "source_E"):
                g5.set_field(name, d5[name])
            g5.set_state(d5["E"], d5["F"], d5["sigma_a"], d5["sigma_s"], d5["T"])
            g5.step_implicit(dt5, TOL, RESTART, 30)          # warm-up (allocations), then the timed step from the same state
            g5.set_state(d5["E"], d5["F"], d5["sigma_a"], d5["sigma_s"], d5["T"])
            torch.cuda.synchronize()
            e0.record(stream)
            its5, res5 = g5.step_implicit(dt5, TOL, RESTART, MAXIT)
            g5.add_velocity_sources(dt5)
            e1.record(stream)
            torch.cuda.synchronize()
            ms5 = e0.elapsed_time(e1)
            tm5 = g5.timings()
            bpc5 = iteration_bytes_per_cell(its5, operator=args.operator)
            line_extra["stage2"] = {"workload": "BASELINE.json configs[4]: 2048x2048 grey radiation-matter coupling, implicit step at 100x explicit dt + velocity sources",
                                    "iterations": its5, "final_residual": res5, "ms": ms5, "cell_updates_per_s": N5 / (ms5 * 1e-3),
                                    "ms_per_iteration": tm5["krylov_ms"] / max(its5, 1),
                                    "krylov_hbm_frac": (bpc5 * N5 / (tm5["krylov_ms"] * 1e-3) / 1e9 / peak_gbs) if its5 > 0 else None}
            # explicit step of the coupled system (marching kernel with emission, source and the Eq. 4 update)
            g5.set_state(d5["E"], d5["F"], d5["sigma_a"], d5["sigma_s"], d5["T"])
            dte5 = wl.explicit_dt(w5["dx"], w5["dy"], w5["c"])
            g5.steps_explicit(dte5, 5)
            torch.cuda.synchronize()
            e0.record(stream)
            g5.steps_explicit(dte5, 40)
            e1.record(stream)
            torch.cuda.synchronize()
            ms5e = e0.elapsed_time(e1) / 40
            line_extra["stage2"]["explicit"] = {"ms_per_step": ms5e, "cell_updates_per_s": N5 / (ms5e * 1e-3), "bytes_per_cell": 96,
                                                "hbm_frac": 96.0 * N5 / (ms5e * 1e-3) / 1e9 / peak_gbs}
            # the same coupled step with BiCGStab + the multigrid V-cycle (fp32 blocks), at 100x and 1000x
            g5.set_option("preconditioner", 1); g5.set_option("mg_precision", 32); g5.set_option("krylov", 1)
            s2mg = {}
            for ratio in (100.0, 1000.0):
                for rep in range(2):                          # first pass allocates the hierarchy
                    g5.set_state(d5["E"], d5["F"], d5["sigma_a"], d5["sigma_s"], d5["T"])
                    torch.cuda.synchronize()
                    e0.record(stream)
                    its5m, res5m = g5.step_implicit(ratio * dte5, TOL, RESTART, 400)
                    g5.add_velocity_sources(ratio * dte5)
                    e1.record(stream)
                    torch.cuda.synchronize()
                ms5m = e0.elapsed_time(e1)
                s2mg[f"{ratio:g}x"] = {"iterations": its5m, "final_residual": res5m, "converged": bool(res5m <= TOL), "ms": ms5m,
                                       "cell_updates_per_s": N5 / (ms5m * 1e-3), "T_implicit_over_T_explicit": ms5m / ms5e,
                                       "over_K": ms5m / ms5e / ratio, "implicit_wins": bool(res5m <= TOL and ms5m / ms5e < ratio)}
            line_extra["stage2"]["bicgstab_multigrid"] = s2mg
            g5.close()
            del d5
        # ---- 3-D (SURVEY 8(f) row 4 tail; generic kernels, csrc/m1_3d.cu): the same number of cells as the 2-D workload ---------------
        if not args.no_sweep and not args.no_3d:
            n3 = int(round(N ** (1.0 / 3.0)))
            w3 = wl.random_medium_3d(n3, seed=args.seed)
            d3 = {k: torch.from_numpy(np.ascontiguousarray(a)).to(dev) for k, a in (("E", w3["E"]), ("F", w3["F"]), ("sa", w3["sigma_a"]), ("ss", w3["sigma_s"]))}
            g3 = ark.ArkM1_3D(n3, n3, n3, 1.0 / n3, 1.0 / n3, 1.0 / n3, 1.0, stream=stream)
            N3 = n3 ** 3
            dt3 = 0.4 / n3 / 1.5
            g3.set_state(d3["E"], d3["F"], d3["sa"], d3["ss"])
            for _ in range(3):
                g3.step_explicit(dt3)
            torch.cuda.synchronize()
            e0.record(stream)
            for _ in range(20):
                g3.step_explicit(dt3)
            e1.record(stream)
            torch.cuda.synchronize()
            ms3e = e0.elapsed_time(e1) / 20
            g3.set_state(d3["E"], d3["F"], d3["sa"], d3["ss"])
            g3.step_implicit(10 * dt3, TOL, RESTART, 30)          # warm-up (allocations)
            g3.set_state(d3["E"], d3["F"], d3["sa"], d3["ss"])
            torch.cuda.synchronize()
            e0.record(stream)
            its3, res3 = g3.step_implicit(10 * dt3, TOL, RESTART, MAXIT)
            e1.record(stream)
            torch.cuda.synchronize()
            ms3i = e0.elapsed_time(e1)
            line_extra["three_d"] = {"workload": f"m1_workloads.random_medium_3d: {n3}^3 cells ({N3 / 1e6:.1f} M), periodic, the config-3 recipe in three dimensions (E lognormal, |F| = u c E with u ~ U[0, 0.9] in a "
                                                 "random direction, log10 sigma ~ U[-3, 3] box-smoothed over 5 cells per direction)",
                                     "explicit": {"ms_per_step": ms3e, "cell_updates_per_s": N3 / (ms3e * 1e-3), "bytes_per_cell": 80, "hbm_frac": 80.0 * N3 / (ms3e * 1e-3) / 1e9 / peak_gbs,
                                                  "note": "two streaming passes (closure once per cell into 13 planes, then the flux-form stencil; ~320 B/cell of DRAM traffic against the algorithmic 80): not the marching organisation of the 2-D kernel"},
                                     "implicit_10x": {"iterations": its3, "final_residual": res3, "ms": ms3i, "ms_per_iteration": ms3i / max(its3, 1), "cell_updates_per_s": N3 / (ms3i * 1e-3)}}
            g3.close()
            del d3
        # ---- roofline of the dominant kernel class ---------------------------------------------------------------
        tot_ms = sum(v["ms"] for v in stats.values()) or 1.0
        kern = {}
        for name, v in stats.items():
            if v["launches"] == 0:
                continue
            gbs = v["bytes"] / (v["ms"] * 1e-3) / 1e9 if v["ms"] > 0 else 0.0
            kern[name] = {"launches": v["launches"], "ms_total": v["ms"], "share": v["ms"] / tot_ms, "achieved_gbs": gbs, "hbm_frac": gbs / peak_gbs,
                          "alg_bytes_per_launch": v["bytes"] / v["launches"]}
        dom = max((k for k in kern if k != "small"), key=lambda k: kern[k]["ms_total"])
        tr = traffic.get(dom, {}) if (n == 4096) else {}
        tr_bytes = tr["ratio"] * kern[dom]["alg_bytes_per_launch"] if "ratio" in tr else None
        line_extra["roofline"] = {"kernel": dom, "bound": "hbm", "achieved": kern[dom]["achieved_gbs"], "peak": peak_gbs, "unit": "GB/s",
                                  "frac": kern[dom]["hbm_frac"], "traffic": tr_bytes, "peak_source": peak_src,
                                  "share_of_step": kern[dom]["share"], "alg_bytes_per_launch": kern[dom]["alg_bytes_per_launch"],
                                  "traffic_note": tr.get("note"),
                                  "pipes_note": (f"ncu of the kernel named in traffic_note: fp64 pipe {float(tr['fp64_pipe_busy_frac']):.2f}, issue slots "
                                                 f"{float(tr['issue_slots_busy_frac']):.2f} busy: the operator rebuilds J and the 3x3 diagonal block in registers instead of "
                                                 "loading them (136 instead of 264 B per cell; 160 B per PAIR of applications inside an s-step block) and sits between "
                                                 "the HBM roof and the issue roof (DESIGN.md section 5)") if tr.get("fp64_pipe_busy_frac") and dom == "spmv_hat" else None,
                                  "frac_of_nominal": kern[dom]["achieved_gbs"] / 7700.0,
                                  "nominal_note": "the measured peak is a torch copy (6544 GB/s here); these kernels are read-dominated and exceed it, "
                                                  "so the fraction of the 7.7 TB/s HGX figure (B200_PROFILING.md) is given as well"}
        line_extra["kernels"] = kern
        # ---- cpu baseline ------------------------------------------------------------------------------------------
        if world == 1 and not args.no_cpu_baseline:
            n_s = args.cpu_n
            r = oracle_step_time(n_s, args.seed, 1, 0)
            r1 = oracle_step_time(512, args.seed, 1, 0, threads=1)
            line_extra["cpu_baseline"] = {"value": 2.0 * r["cells"] / r["seconds"], "unit": UNIT, "cores": r["cores"], "kind": "oracle",
                                          "sample": f"1 step (explicit + implicit 10x, {r['iterations']} GMRES iterations) on a {n_s}x{n_s} grid of "
                                                    f"the same generator = {r['cells'] / N:.4f} of the workload's cells; {r['seconds']:.1f} s",
                                          "explicit_cell_updates_per_s": r["cells"] / r["explicit_s"],
                                          "implicit_cell_updates_per_s": r["cells"] / r["implicit_s"],
                                          "implicit_s_per_iteration_per_Mcell": r["implicit_s"] / max(r["iterations"], 1) / (r["cells"] / 1e6),
                                          "one_thread": {"sample": "the same step on a 512x512 grid, 1 thread", "value": 2.0 * r1["cells"] / r1["seconds"],
                                                         "explicit_cell_updates_per_s": r1["cells"] / r1["explicit_s"],
                                                         "implicit_cell_updates_per_s": r1["cells"] / r1["implicit_s"]},
                                          "protocol": "bounded sample; the full SURVEY 8(d) protocol (bench size, explicit alone, capped cycle, 1 thread) runs with --oracle-protocol"}
            if args.oracle_protocol:
                line_extra["cpu_baseline"]["full_protocol"] = oracle_protocol(n, args.seed)
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1e3 * t_max / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"M1 random medium (BASELINE.json configs[3]) {n}x{n}, fp64, periodic, c=1, seed {args.seed}(+rank)",
                       "step": "state reset (D2D) + 1 explicit step (CFL 0.4) + 1 implicit step (dt = 10x explicit, GMRES(30) + "
                               + ("block-Jacobi" if args.preconditioner == 0 else f"multigrid V-cycle (fp{args.mg_precision} blocks)") + ", tol 1e-10)",
                       "iterations_per_implicit_step": its_main,
                       "operator": "matrix-free coefficient planes" if args.operator == 1 else "pre-multiplied block stencil (BSR 3x3)", "parallelism": "replicas only (one independent problem per GPU)" if world > 1 else "1 GPU",
                       "l2": f"inputs larger than L2 (state+opacity {5 * N * 8 / 1e6:.0f} MB, Krylov basis {31 * 3 * N * 8 / 1e9:.1f} GB vs 126 MB L2)",
                       "device_bytes": g.device_bytes()},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches),
        }
        line.update(line_extra)
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def run_decomposed(args):
    """Strong-scaling form of the same step: ONE global grid cut into y-slabs (include/ark_m1.h "Domain-decomposed step").
    Under torchrun: one slab per rank and GPU, halos and Gram-Schmidt sums over NCCL.  With --decomposed-local R on one GPU: R slabs
    in this process (the emulated form the tests use): measures what the decomposition itself costs (extra launches, halo packing)."""
    import torch
    import torch.distributed as dist
    import paper_2011_13926_b200 as ark

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device — the CUDA library is the only implementation (no CPU fallback)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    n = args.n
    N = n * n
    w = wl.random_medium(n, seed=args.seed)           # the SAME global problem on every rank; each keeps its rows
    dt_e = wl.explicit_dt(w["dx"], w["dy"], w["c"])
    stream = torch.cuda.current_stream()
    if world > 1 or args.decomposed_local < 2:          # --decomposed: one slab per rank over NCCL (a single rank still goes through NCCL)
        box = [ark.nccl_unique_id() if rank == 0 else None]
        if world > 1:
            dist.init_process_group("nccl", device_id=dev)
            dist.broadcast_object_list(box, src=0)
        grp = ark.ArkM1Group(n, n, w["dx"], w["dy"], w["c"], bc=w["bc"], nranks=world, kind="nccl", rank=rank, unique_id=box[0], stream=stream)
        nslab_total, kind = world, "nccl"
    else:
        grp = ark.ArkM1Group(n, n, w["dx"], w["dy"], w["c"], bc=w["bc"], nranks=args.decomposed_local, kind="local", stream=stream)
        nslab_total, kind = args.decomposed_local, "local"
    peak_gbs, peak_src = peaks()
    devs = []
    for s_ in grp.slabs:
        rows = slice(s_.y0, s_.y1)
        devs.append({k: torch.from_numpy(np.ascontiguousarray(np.asarray(w[k])[..., rows, :])).to(dev) for k in ("E", "F", "sigma_a", "sigma_s")})

    def reset():
        for s_, d_ in zip(grp.slabs, devs):
            s_.set_state(d_["E"], d_["F"], d_["sigma_a"], d_["sigma_s"])

    def one_step():
        grp.step_explicit(dt_e)
        return grp.step_implicit(BENCH_DT_RATIO * dt_e, TOL, RESTART, MAXIT)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        reset(); one_step()
    st0 = grp.comm_stats()
    l0 = sum(s_.kernel_launches() for s_ in grp.slabs)
    sampler = ClockSampler(local)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    sampler.start()
    e0.record(stream)
    its = 0
    for _ in range(args.steps):
        reset()
        its, res = one_step()
    e1.record(stream)
    barrier()
    clocks = sampler.stop()
    elapsed = e0.elapsed_time(e1) * 1e-3
    st1 = grp.comm_stats()
    launches = sum(s_.kernel_launches() for s_ in grp.slabs) - l0
    # explicit alone, sustained for ~1 s
    reset()
    grp.step_explicit(dt_e)
    barrier()
    n_e = 400
    e0.record(stream)
    for _ in range(n_e):
        grp.step_explicit(dt_e)
    e1.record(stream)
    barrier()
    t_exp = e0.elapsed_time(e1) / n_e
    t_max, _ = aggregate_over_ranks(elapsed, 0.0, dist if world > 1 else None)
    t_exp_max, _ = aggregate_over_ranks(t_exp, 0.0, dist if world > 1 else None)
    if rank == 0:
        halo_per_step = (st1["halo_bytes"] - st0["halo_bytes"]) / args.steps
        interior = iteration_bytes_per_cell(its, operator=1, pair=False) * N / nslab_total + (64.0 + 288.0) * N / nslab_total
        line = {
            "metric": METRIC, "value": 2.0 * N * args.steps / t_max, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1e3 * t_max / args.steps, "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": f"M1 random medium (BASELINE.json configs[3]) {n}x{n}, fp64, periodic, c=1, seed {args.seed}: ONE global grid "
                                   f"in {nslab_total} y-slabs ({kind} transport)",
                       "step": "state reset (D2D) + 1 explicit step (CFL 0.4) + 1 implicit step (dt = 10x explicit, GMRES(30) + block-Jacobi, tol 1e-10)",
                       "iterations_per_implicit_step": its, "final_residual": res,
                       "parallelism": f"domain decomposition, {nslab_total} slabs of {n // nslab_total} rows, 1-cell halos, all-reduced Gram-Schmidt sums",
                       "l2": "inputs larger than L2"},
            "clocks": clocks, "gpu_launches": int(launches),
            "explicit": {"ms_per_step": t_exp_max, "cell_updates_per_s": N / (t_exp_max * 1e-3), "hbm_frac_per_gpu": 64.0 * N / max(world, 1) / (t_exp_max * 1e-3) / 1e9 / peak_gbs},
            "communication": {"halo_bytes_sent_per_step_this_rank": halo_per_step, "exchanges_per_step": (st1["exchanges"] - st0["exchanges"]) / args.steps,
                              "allreduces_per_step": (st1["allreduces"] - st0["allreduces"]) / args.steps,
                              "interior_algorithmic_bytes_per_step_per_slab": interior, "halo_over_interior": halo_per_step / interior},
            "e2e": None,
        }
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    grp.close()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--grid", "--n", dest="n", type=int, default=4096, help="grid size (BASELINE.json configs[3]: 4096); use --grid under torchrun (--n is ambiguous there)")
    ap.add_argument("--seed", type=int, default=1234)
    ap.add_argument("--operator", type=int, default=1, choices=[0, 1],
                    help="implicit operator: 0 = pre-multiplied block stencil, 1 = matrix-free coefficient planes (default, DESIGN.md)")
    ap.add_argument("--preconditioner", type=int, default=0, choices=[0, 1],
                    help="0: 3x3 block-Jacobi (north_star; the default line)  1: multigrid V-cycle (variant run; uses the block-stencil operator)")
    ap.add_argument("--mg-precision", type=int, default=32, choices=[32, 64], help="storage precision of the multigrid blocks")
    ap.add_argument("--no-sweep", action="store_true", help="skip the dt = 50/100/200x implicit solves")
    ap.add_argument("--sustain-s", type=float, default=2.0, help="length of the sustained back-to-back explicit run, seconds")
    ap.add_argument("--decomposed", action="store_true", help="under torchrun: ONE global grid cut into y-slabs, one per rank, halos and sums over NCCL (strong scaling) instead of independent replicas")
    ap.add_argument("--decomposed-local", type=int, default=0, metavar="R", help="one GPU: the same global grid in R slabs inside this process (what the decomposition itself costs)")
    ap.add_argument("--restart-sweep", action="store_true", help="also sweep the GMRES restart length (30/60/100) at 50/100/200x on the bench medium and at 1024^2 (takes ~3 min)")
    ap.add_argument("--oracle-protocol", action="store_true", help="also time the oracle as SURVEY 8(d) lists it: explicit alone and one capped GMRES cycle at the bench size, all cores and 1 thread (takes several minutes)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-3d", dest="no_3d", action="store_true", help="skip the 3-D section")
    ap.add_argument("--no-stage2", action="store_true", help="skip the config-5 (2048^2, matter coupling) implicit step")
    ap.add_argument("--cpu-n", type=int, default=2048, help="grid size of the oracle's bounded sample (cpu_baseline)")
    ap.add_argument("--ref-n", type=int, default=1024, help="grid size of the oracle's bounded sample per step (--impl reference)")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        print(f"bench.py: note: warmup {args.warmup} < 3 (timing rule wants >= 3)", file=sys.stderr)
    if args.impl == "reference":
        return run_reference(args)
    if args.decomposed or args.decomposed_local > 1:
        return run_decomposed(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
