#!/usr/bin/env python
"""bench.py -- history-integral throughput of libdmfe.so on B200 (driver contract, tier ④).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--L 4096]

Workload (BASELINE.json configs[1]): one evaluation of the
DMFE history integrals (steps a2-a8 of DESIGN.md: A factors, type-1 and type-2 lookups, f', f'',
the eight nu-weighted sums, mu, E, the four derivative vectors) on the seeded synthetic history
L = N = 4096, log-spaced rows on [1e-2, 1e4], s = 4, f = q^3/2, T = 0.5, fp64.  One "step" = one
such evaluation (one dmfe_history_integrals call = 2 kernel launches).  metric = stencil
evaluations per second, 8 per (i,j) pair (C1,R1,C2,R2,B1C,B1R,B2C,B2R).

The JSON line carries, besides the contract keys:
  roofline      the pair kernel against the larger of its two bounds (HBM: unique history cells
                touched x 32 B over the measured copy bandwidth; ALU: algorithmic fp64 flops over
                the DFMA rate measured on this GPU by dmfe_probe_fp64_tflops)
  cpu_baseline  the CPU oracle (oracle/, as it stands, OpenMP over targets) on a bounded sample of
                targets of the same workload, on this box's host cores
  e2e           the same metric through dmfe_history_integrals_host (pinned HOST buffers in,
                HOST results out, copies inside the timed region)
`--impl reference` times the oracle alone (rank 0 only).
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

METRIC = "history-integral stencil-evals/s"
UNIT = "stencil-evals/s"
EVALS_PER_PAIR = 8
L2_BYTES = 126 << 20       # B200 L2; inputs at or below this size get an L2 flush before every timed step
FLUSH_BYTES = 256 << 20

WORKLOADS = {
    # name: (lo, hi, t_max, lambda, T)
    "config2": (-2.0, 4.0, 1e4, [0.0, 0.0, 0.0, 1.0], 0.5),
    "config5": (-2.0, 7.0, 1e7, [0.0, 0.0, 1.0, 0.8, 0.5], 0.5),
}


def flops_per_pair(s: int, lam) -> int:
    """Algorithmic fp64 flops of one (i,j) pair (FMA = 2), counted on the oracle's inner loop
    (oracle/dmfe_oracle.c orc_history_integrals):
      3 sets of s Lagrange weights from the fractional coordinate   3 * (s + 2(s-2) + 2s) ~ 3(5s-4)
      A factors (4 s-point dot products)                            8 s
      type-1 Hermite (2 fields x 4 terms)                           14
      type-2 stencil (8 row quantities) + Hermite                   16 s + 14
      t-weights of the type-2 row pair (cubic, one division)        20
      f''(C1), f'(C1), f''(C2), f''(B1C), f'(B1C), f''(B2C), f'(B2C) Horner
      eight terms and accumulations                                 ~ 30
    """
    pmax = len(lam) - 1
    horner = 4 * 2 * max(pmax - 2, 0) + 3 * 2 * max(pmax - 1, 0)
    return 3 * (5 * s - 4) + 8 * s + 14 + 16 * s + 14 + 20 + horner + 30


def unique_cells(theta, omega, t, s, L, N, sample=None, window=2):
    """Algorithmic bytes: number of distinct history cells (32 B each) that the type-1 and type-2
    lookups of one evaluation touch (computed from integer row / column indices only).  Exact over
    all targets when `sample` is None.  With a strided target sample the type-2 part is the per-row
    hull [min column, max column] of the sampled targets' cells: in every row the columns touched
    by all targets form one run (neighbouring targets overlap), so the hull of a strided sample
    that contains the first and the last target is that run up to the stride's resolution."""
    M = N - 1
    tM = t[M]
    # rows read around the interval [t_n, t_n+1): Hermite (window = 2): n, n+1; values-only history
    # (window = 4, 4-point Lagrange in t): k .. k+3 with k = clamp(n-1, 0, M-3)
    def first_row(n):
        return n if window == 2 else np.clip(n - 1, 0, max(M - 3, 0))
    nwin = 2 if window == 2 else min(4, M + 1)
    # type-1: all columns, all targets (cheap)
    n1 = first_row(np.clip(np.searchsorted(t[:M], theta * tM, side="right") - 1, 0, M - 1))
    full = np.zeros(N, dtype=bool)
    for q in range(nwin):
        full[n1 + q] = True
    idx = np.arange(L) if sample is None else sample
    touched = np.zeros((N, L), dtype=bool) if sample is None else None
    lo = np.full(N, L, dtype=np.int64)
    hi = np.full(N, -1, dtype=np.int64)
    for i in idx:
        phi2 = theta[i] + omega[i] * theta
        n2 = first_row(np.clip(np.searchsorted(t[:M], phi2 * tM, side="right") - 1, 0, M - 1))
        with np.errstate(invalid="ignore", divide="ignore"):
            psi = np.where(phi2 > 0, theta[i] / phi2, 0.0)
        lstar = np.searchsorted(theta, psi, side="right") - 1
        a3 = np.clip(lstar - (s // 2 - 1), 0, L - s)
        if touched is not None:
            for l in range(s):
                for q in range(nwin):
                    touched[n2 + q, a3 + l] = True
        else:
            for rows in [n2 + q for q in range(nwin)]:
                np.minimum.at(lo, rows, a3)
                np.maximum.at(hi, rows, a3 + s - 1)
    if touched is not None:
        touched[full, :] = True
        return int(touched.sum())
    width = np.where(hi >= lo, hi - lo + 1, 0)
    width[full] = L
    return int(width.sum())


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.path = tempfile.mktemp(suffix=".csv")
        self.proc = None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        try:
            for line in open(self.path):
                f = [x.strip() for x in line.split(",")]
                if len(f) < 7:
                    continue
                try:
                    sm.append(float(f[0])); mx.append(float(f[1]))
                except ValueError:
                    continue
                for k, nm in enumerate(names):
                    if f[3 + k].lower().startswith("active"):
                        reasons.add(nm)
            os.unlink(self.path)
        except Exception:
            pass
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), reasons=sorted(reasons),
                       samples=len(sm))
        return out


# ------------------------------------------------------------------------------------------------
def oracle_sample(L, s, t_max, lam, T, theta, omega, nu, t, mu, hist, n_targets, seed=12345, min_seconds=0.0,
                  max_reps=64, values_only=False):
    """Time the CPU oracle (as it stands) on `n_targets` seeded targets x all L nodes; the same
    evaluation is repeated until `min_seconds` of CPU work have been timed.  Returns (targets per
    repetition, repetitions, seconds)."""
    from oracle import dmfe_oracle as O
    rng = np.random.Generator(np.random.PCG64(seed))
    targets = np.sort(rng.choice(L, size=min(n_targets, L), replace=False)).astype(np.int32)
    grid = O.Grid(L=L, s=s, t_max=t_max, theta=theta, omega=omega, nu=nu)
    tables = grid.tables(targets)          # table construction is start-up work, not timed
    model = O.Model(np.array(lam, dtype=np.float64), T, 0.0)
    reps, dt = 0, 0.0
    while reps < max_reps and (reps == 0 or dt < min_seconds):
        t0 = time.perf_counter()
        (O.history_integrals_values if values_only else O.history_integrals)(
            grid, model, t, mu, hist, len(t) - 1, targets=targets, tables=tables)
        dt += time.perf_counter() - t0
        reps += 1
    return len(targets), reps, dt


# ---- multi-rank host logic (replicas only); covered by a gloo test on CPU ----
def replica_seed(rank: int) -> int:
    """Every rank evaluates its own replica: the seed is offset so that the replicas are distinct problems."""
    from paper_2604_06309_b200 import inputs
    return inputs.DEFAULT_SEED + 16 * rank


def max_over_ranks(ms: float, world: int, device=None) -> float:
    """Timing of a multi-rank run = the slowest rank (all_reduce MAX; identity for one rank)."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_value(units_per_rank_step: int, steps: int, world: int, ms_total: float) -> float:
    """Whole-job throughput: the units all ranks processed over the max-over-ranks time."""
    return units_per_rank_step * steps * world / (ms_total * 1e-3)


def host_cores():
    try:
        n = len(os.sched_getaffinity(0))
    except Exception:
        n = os.cpu_count() or 1
    env = os.environ.get("OMP_NUM_THREADS")
    return min(n, int(env)) if env and env.isdigit() else n


def run_reference(args):
    """--impl reference: the oracle alone, on host cores, rank 0 only (tier ④)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from oracle import dmfe_oracle as O
    from paper_2604_06309_b200 import inputs
    lo, hi, t_max, lam, T = WORKLOADS[args.workload]
    L, s = args.L, args.stencil
    grid = O.Grid(L=L, s=s, t_max=t_max)      # the oracle's own tables: no CUDA library on this arm
    t, mu, hist = inputs.synthetic_history(grid.theta, grid.omega, L, lo, hi)
    nt = args.ref_targets
    times = []
    for k in range(args.warmup + args.steps):
        n, reps, dt = oracle_sample(L, s, t_max, lam, T, grid.theta, grid.omega, grid.nu, t, mu, hist, nt, seed=100 + k)
        if k >= args.warmup:
            times.append(dt)
    tot = float(np.sum(times))
    nt = n
    value = EVALS_PER_PAIR * nt * L * args.steps / tot
    cores = host_cores()
    sample = "%d seeded targets x %d nodes per step of the L=N=%d evaluation" % (nt, L, L)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "%s: single history-integral evaluation, L=N=%d, s=%d" % (args.workload, L, s),
                   "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    import torch.distributed as dist

    from paper_2604_06309_b200 import dmfe as D
    from paper_2604_06309_b200 import inputs

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py: no CUDA device; this package has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    lo, hi, t_max, lam, T = WORKLOADS[args.workload]
    L, s = args.L, args.stencil
    N = L
    vo = bool(getattr(args, "values_only", False))
    ctx = D.dmfe_create(L, s, t_max, lam, T=T, values_only=vo)
    tab = D.dmfe_get_tables(ctx, L, want_pairs=False)
    theta, omega, nu = tab["theta"], tab["omega"], tab["nu"]
    # every rank evaluates its own replica of the workload (weak scaling, no data-path collective:
    # DESIGN.md "Multi-GPU"); the seed is offset per rank so that the replicas are distinct problems
    t, mu, hist = inputs.synthetic_history(theta, omega, N, lo, hi, seed=replica_seed(rank))
    if vo:   # the same fields without their slopes, 16-byte cells
        hist = np.ascontiguousarray(hist[:, :, [0, 2]])
    tt, tm, th = (torch.from_numpy(a).to(dev) for a in (t, mu, hist))
    out = dict(d1C=torch.zeros(L, dtype=torch.float64, device=dev), d1R=torch.zeros(L, dtype=torch.float64, device=dev),
               mu_out=torch.zeros(1, dtype=torch.float64, device=dev),
               d2C=torch.zeros(L, dtype=torch.float64, device=dev), d2R=torch.zeros(L, dtype=torch.float64, device=dev),
               energy=torch.zeros(1, dtype=torch.float64, device=dev))

    def step():
        D.dmfe_history_integrals(ctx, N, tt, tm, th, **out)

    # timing rule: inputs larger than L2, or an L2 flush between timed steps
    input_bytes = hist.nbytes + 24 * L * L
    need_flush = input_bytes <= L2_BYTES

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing: W warm-ups, then exactly K steps between barriers -------------
    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    sampler = ClockSampler(local_rank) if rank == 0 else None
    D.dmfe_enable_timing(ctx, True)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    if need_flush:   # inputs fit in L2: overwrite L2 before every step, time each step on its own
        flush = torch.empty(FLUSH_BYTES // 8, dtype=torch.float64, device=dev)
        ms_total = 0.0
        for _ in range(args.steps):
            flush.fill_(1.0)
            e0.record()
            step()
            e1.record()
            e1.synchronize()
            ms_total += e0.elapsed_time(e1)
        del flush
        barrier()
    else:
        e0.record()
        for _ in range(args.steps):
            step()
        e1.record()
        barrier()
        ms_total = e0.elapsed_time(e1)
    n_k, k_ms, k_min = D.dmfe_kernel_time_stats(ctx)
    D.dmfe_enable_timing(ctx, False)
    clocks = sampler.stop() if sampler else None
    ms_total = max_over_ranks(ms_total, world, dev)

    # ---- end-to-end: host buffers through dmfe_history_integrals_host --------------------------
    e2e = None
    if args.e2e_steps > 0:   # 0 skips the leg (scaling sweep at sizes where pinning the history is impractical)
        ht = torch.from_numpy(t).pin_memory()
        hm = torch.from_numpy(mu).pin_memory()
        hh = torch.from_numpy(hist).pin_memory()
        o1, o2 = torch.zeros(L, dtype=torch.float64).pin_memory(), torch.zeros(L, dtype=torch.float64).pin_memory()
        o3, o4 = torch.zeros(1, dtype=torch.float64).pin_memory(), torch.zeros(1, dtype=torch.float64).pin_memory()
        e2e_steps = max(1, min(args.steps, args.e2e_steps))
        pairs_e2e = L * L

        def e2e_step():
            D.dmfe_history_integrals_host(ctx, N, ht.numpy(), hm.numpy(), hh.numpy(), o1.numpy(), o2.numpy(), o3.numpy(),
                                          o4.numpy())

        e2e_step()
        barrier()
        w0 = time.perf_counter()
        e0.record()
        for _ in range(e2e_steps):
            e2e_step()
        e1.record()
        barrier()
        e2e_ms = max(e0.elapsed_time(e1), 0.0)
        e2e_wall = 1e3 * (time.perf_counter() - w0)
        e2e_ms = max(e2e_ms, e2e_wall if world == 1 else e2e_ms)  # host-synchronous call: wall >= device span
        e2e_ms = max_over_ranks(e2e_ms, world, dev)
        h2d = int(t.nbytes + mu.nbytes + hist.nbytes)
        d2h = int(2 * L * 8 + 16)
        e2e = {"value": EVALS_PER_PAIR * pairs_e2e * e2e_steps * world / (e2e_ms * 1e-3), "unit": UNIT,
               "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": e2e_steps,
               "ms_per_step": e2e_ms / e2e_steps}

    if rank != 0:
        D.dmfe_destroy(ctx)
        if world > 1:
            dist.destroy_process_group()
        return 0

    # ---- roofline of the pair kernel ------------------------------------------------------------
    pairs = L * L
    fpp = flops_per_pair(s, lam)
    if vo:   # 4-point Lagrange in t: no Hermite t-weights / slope terms, four rows instead of two
        pmax_ = len(lam) - 1
        fpp = (3 * (5 * s - 4) + 8 * s + 16 + 28 + 16 * s + 16 + 4 * 2 * max(pmax_ - 2, 0) + 3 * 2 * max(pmax_ - 1, 0) + 30)
    if L <= 8192:
        cells, sampled = unique_cells(theta, omega, t, s, L, N, window=4 if vo else 2), False
    else:
        samp = np.unique(np.append(np.arange(0, L, max(1, L // 1024)), L - 1))
        cells, sampled = unique_cells(theta, omega, t, s, L, N, sample=samp, window=4 if vo else 2), True
    alg_bytes = (16 if vo else 32) * cells + 8 * 8 * L
    table_bytes = 24 * pairs
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    hbm_peak, hbm_src = (peaks["hbm_gbs"], "measured") if "hbm_gbs" in peaks else (6650.0, "fallback")
    fp64_tf, sms = D.dmfe_probe_fp64_tflops(ctx, 1 << 16)
    k_avg_ms = k_ms / max(n_k, 1)
    t_hbm = alg_bytes / (hbm_peak * 1e9)
    t_alu = pairs * fpp / (fp64_tf * 1e12)
    if t_hbm >= t_alu:
        roof = {"bound": "hbm", "achieved": alg_bytes / (k_avg_ms * 1e-3) / 1e9, "peak": hbm_peak, "unit": "GB/s"}
    else:
        roof = {"bound": "alu", "achieved": pairs * fpp / (k_avg_ms * 1e-3) / 1e12, "peak": fp64_tf, "unit": "TFLOP/s"}
    roof["frac"] = roof["achieved"] / roof["peak"]
    # the same fraction with SURVEY.md 8(d)'s count of the method's own work, 24 s + 106 flop per pair
    # (interpolation weights given, as the paper tabulates them); `flops_per_pair` above adds the
    # recomputation of the weights from the packed coordinate, a design choice of this library
    fpp_survey = 24 * s + 106
    t_alu_survey = pairs * fpp_survey / (fp64_tf * 1e12)
    traffic, traffic_src = args.traffic_bytes, "--traffic-bytes"
    if traffic is None:
        try:   # dram bytes per launch of this kernel on this workload from the committed ncu capture
            import csv
            key = "%s_L%d_s%d%s" % (args.workload, L, s, "_values" if vo else "")
            rows = {r["workload_key"]: r for r in csv.DictReader(open(os.path.join(ROOT, "profiles", "traffic.csv")))}
            traffic, traffic_src = float(rows[key]["dram_bytes_per_launch"]), rows[key]["source"]
        except Exception:
            traffic, traffic_src = None, None
    roof.update({
        "traffic": traffic, "traffic_source": traffic_src, "peak_source": "hbm: %s copy bandwidth; alu: DFMA chain measured in this run "
        "on %d SMs" % (hbm_src, sms), "kernel": ("history_integrals_values_kernel<%d>" % s if vo else
                   ("history_integrals_s4_kernel" if s == 4 else "history_integrals_kernel<%d>" % s)),
        "kernel_ms_avg": k_avg_ms,
        "kernel_ms_min": k_min, "launches_timed": n_k, "algorithmic_bytes": alg_bytes,
        "algorithmic_bytes_sampled": sampled, "table_bytes": table_bytes, "flops_per_pair": fpp,
        "hbm": {"achieved_GBps": alg_bytes / (k_avg_ms * 1e-3) / 1e9, "peak_GBps": hbm_peak,
                "with_tables_GBps": (alg_bytes + table_bytes) / (k_avg_ms * 1e-3) / 1e9},
        "alu": {"achieved_TFLOPs": pairs * fpp / (k_avg_ms * 1e-3) / 1e12, "peak_TFLOPs": fp64_tf},
        "roofline_time_ms": 1e3 * max(t_hbm, t_alu),
        "survey_count": {"flops_per_pair": fpp_survey, "roofline_time_ms": 1e3 * max(t_hbm, t_alu_survey),
                         "frac": max(t_hbm, t_alu_survey) / (k_avg_ms * 1e-3)},
        # what this design must move through HBM per launch (history cells once per loop that touches
        # them + the 24 B/pair tables) against the measured copy bandwidth
        "design_bytes_hbm_frac": ((traffic if traffic else alg_bytes + table_bytes) / (hbm_peak * 1e9)) / (k_avg_ms * 1e-3),
    })

    # ---- the oracle on this box's host cores, bounded sample -----------------------------------
    nt = args.ref_targets
    n_s, reps, dt = oracle_sample(L, s, t_max, lam, T, theta, omega, nu, t, mu, hist, nt, min_seconds=args.ref_seconds,
                                  values_only=vo)
    cpu = {"value": EVALS_PER_PAIR * n_s * L * reps / dt, "unit": UNIT, "cores": host_cores(), "kind": "oracle",
           "sample": "%d seeded targets x %d nodes of the same L=N=%d evaluation, repeated %d times (%.1f s of "
                     "CPU work)" % (n_s, L, L, reps, dt)}
    D.dmfe_destroy(ctx)

    # ---- adaptive trajectory (BASELINE.json configs[3]): bounded segment, wall time per decade ----
    traj = None
    if args.traj_seconds > 0:
        from paper_2604_06309_b200 import trajectory
        cfg = dict(trajectory.CONFIGS[4])
        out = trajectory.run(t_end=1e7, max_seconds=args.traj_seconds, step_mode=args.step_mode, **cfg)
        stt = out["stats"]
        traj = {"workload": "config4: pure 3-spin aging run, T=0.5, tol=1e-8, L=%d, s=%d, n_cap=%d, first %.0f s of "
                            "wall time" % (cfg["L"], cfg["s"], cfg["n_cap"], args.traj_seconds),
                "steps_per_s": stt["steps"] / stt["wall_s"], "rhs_per_s": stt["n_rhs"] / stt["wall_s"],
                "t_reached": stt["t_reached"], "wall_s_to_t": out["wall_to_t"], "reverted": stt["reverted"],
                "n_rows": stt["n_rows"], "n_rows_max": stt["n_rows_max"], "status": stt["status"],
                "sparsify_passes": stt["sparsify_passes"], "rows_dropped": stt["rows_dropped"],
                "eps_sparse_over_tol": stt["eps_sparse_over_tol"],
                "us_per_stage": 1e5 * stt["wall_s"] / max(stt["steps"], 1),
                "step_kernel": ("one persistent cooperative kernel per batch of 50 steps (csrc/advance_s4.cu)"
                                if args.step_mode == 0 else "one CUDA graph of 21 kernel nodes per step (csrc/rk_step.cu)"),
                "full_runs": "profiles/r2_trajectories.md holds the wall times of the runs to t=1e5 (config 3) and t=1e7 (config 4)"}

    value = job_value(EVALS_PER_PAIR * pairs, args.steps, world, ms_total)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": "%s: single history-integral evaluation, L=N=%d log-spaced rows, s=%d, lambda=%s, T=%g%s"
                   % (args.workload, L, s, lam, T, ", values-only history (4-point Lagrange in t)" if vo else ""), "pairs_per_step": pairs, "replicas": world,
                   "l2": ("inputs fit in L2 (%.0f MB history + %.0f MB pair tables): %d MB written to a scratch "
                          "buffer before every timed step, each step timed on its own"
                          % (hist.nbytes / 1e6, table_bytes / 1e6, FLUSH_BYTES >> 20)) if need_flush else
                         ("inputs larger than L2: %.0f MB history + %.0f MB pair tables streamed per step, no flush"
                          % (hist.nbytes / 1e6, table_bytes / 1e6))},
        "pairs_per_s": pairs * args.steps * world / (ms_total * 1e-3),
        "clocks": clocks, "roofline": roof, "cpu_baseline": cpu,
        "e2e": e2e,
        "gpu_launches": 2 * args.steps,
        "trajectory": traj,
    }
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="config2", choices=sorted(WORKLOADS))
    ap.add_argument("--L", type=int, default=4096)
    ap.add_argument("--stencil", type=int, default=4)
    ap.add_argument("--ref-targets", type=int, default=4096, help="targets per oracle sample")
    ap.add_argument("--ref-seconds", type=float, default=10.0, help="CPU time of the oracle sample in the ours arm")
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--step-mode", type=int, default=0, choices=[0, 1],
                    help="trajectory segment: 0 = persistent kernel per batch (S = 4, L <= 512), 1 = graph of launches")
    ap.add_argument("--traj-seconds", type=float, default=8.0,
                    help="wall-time budget of the adaptive trajectory segment (0 = skip)")
    ap.add_argument("--values-only", action="store_true",
                    help="values-only history with 4-point Lagrange in t (SURVEY.md 8(f)-2) instead of Hermite")
    ap.add_argument("--traffic-bytes", type=float, default=None,
                    help="dram bytes per launch of the pair kernel from the committed ncu capture (profiles/)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
