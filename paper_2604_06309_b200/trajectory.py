"""Adaptive DMFE trajectories on the device: the driver loop around dmfe_rk_step / dmfe_sparsify.

Every step of the path and the step loop itself (thinning schedule, start-up switch: dmfe_integrate) run
inside libdmfe.so; this module reads a few rows back at requested observation times and keeps the clock.  Used by bench.py's
trajectory workloads (BASELINE.json configs 3 and 4) and by the trajectory tests.

    python -m paper_2604_06309_b200.trajectory --config 4 --t-end 1e3
"""
from __future__ import annotations

import argparse
import json
import time

import numpy as np

from . import dmfe as D

CONFIGS = {
    # BASELINE.json configs[2], [3] (sizes: DESIGN.md section 4)
    3: dict(lam=[0.0, 0.0, 1.0, 0.0, 0.5], T=0.5, tol=1e-8, n_cap=2048, t_max=1e5, L=512, s=4),
    4: dict(lam=[0.0, 0.0, 0.0, 1.0], T=0.5, tol=1e-8, n_cap=8192, t_max=1e7, L=512, s=4),
    # SURVEY.md 8(f)-4, second workload: the 3+9 model at lambda = 1/2 quenched to T = 0 (Fig. 3,
    # :410 Fig. 8), f = (q^3 + q^9)/4 in the convention f = 1/2 sum lam_p q^p; run-time degree of f (p_max > 4)
    39: dict(lam=[0.0, 0.0, 0.0, 0.5, 0.0, 0.0, 0.0, 0.0, 0.0, 0.5], T=0.0, tol=1e-8, n_cap=32768, t_max=1e5, L=512, s=4),
}


def observe(theta, t, row, t_w):
    """C(t, t_w), R(t, t_w) from the stored row at time t (values at theta_l t): linear interpolation
    in theta at theta = t_w / t.  Reporting only -- not part of the integrator."""
    out = {}
    for tw in t_w:
        if tw <= t:
            th = tw / t
            out[tw] = (float(np.interp(th, theta, row[:, 0])), float(np.interp(th, theta, row[:, 2])))
    return out


def run(L, s, t_max, lam, T, tol, n_cap, t_end, h0=1e-3, sp_every=200, protect_last=24, beta0=0.0,
        t_w=(1e2, 1e3, 1e4, 1e5), n_obs=64, max_steps=None, max_seconds=None, progress=None, startup="ssprk",
        step_mode=0, batch=50, sp_max_passes=8):
    """Integrate from t = 0 to t_end with the library's step loop (dmfe_integrate: thinning schedule at the
    paper's threshold tol/10, start-up switch, device-resident batches of steps), stopping at log-spaced
    observation times to read one row back.  Returns the observation records, the wall-clock time at which
    each decade of t was first passed, and the loop's statistics.  This module takes no decision of the
    method: it observes and keeps the clock."""
    import torch

    ctx = D.dmfe_create(L, s, t_max, lam, T=T, beta0=beta0, tol=tol)
    D.dmfe_set_step_mode(ctx, step_mode)
    rec = dict(t=[], E=[], mu=[], h=[], n_rows=[], corr=[], wall=[])
    out_stats = dict(status="ok")
    milestones = {}
    try:
        theta = D.dmfe_get_tables(ctx, L, want_pairs=False)["theta"]
        st, ten = D.make_state(L, n_cap)
        D.dmfe_init_state(ctx, st, h0)
        pol = D.dmfe_policy(batch=batch, sp_every=sp_every, sp_max_passes=sp_max_passes, sp_min_gain=0.0,
                            protect_last=protect_last, startup_dp=1 if startup == "dp" else 0)
        stats = D.dmfe_run_stats()
        obs_times = list(np.geomspace(max(10 * h0, 1e-2), t_end, n_obs))
        next_decade = 1.0
        torch.cuda.synchronize()
        w0 = time.perf_counter()
        rc = D.DMFE_OK
        while stats.t < t_end:
            left_s = 0.0
            if max_seconds is not None:
                left_s = max_seconds - (time.perf_counter() - w0)
                if left_s <= 0:
                    out_stats["status"] = "max_seconds"
                    break
            left_n = 0
            if max_steps is not None:
                left_n = max_steps - stats.steps
                if left_n <= 0:
                    out_stats["status"] = "max_steps"
                    break
            target = min(t_end, obs_times[0] if obs_times else t_end, next_decade)
            stats, rc = D.dmfe_integrate(ctx, st, pol, target, max_steps=left_n, max_seconds=left_s, stats=stats,
                                         check=False)
            if rc != D.DMFE_OK:
                out_stats["status"] = {D.DMFE_ECAPACITY: "capacity", D.DMFE_ESTEPMIN: "stepmin"}.get(rc, "error %d" % rc)
                break
            t_now = stats.t
            wall = time.perf_counter() - w0
            while t_now >= next_decade:
                milestones[next_decade] = wall
                next_decade *= 10.0
            if obs_times and t_now >= obs_times[0]:
                while obs_times and t_now >= obs_times[0]:
                    obs_times.pop(0)
                n = st.n_rows - 1
                row = ten["hist"][n].cpu().numpy()
                rec["t"].append(t_now)
                rec["E"].append(float(ten["energy"][n].item()))
                rec["mu"].append(float(ten["mu"][n].item()))
                rec["h"].append(st.h)
                rec["n_rows"].append(st.n_rows)
                rec["corr"].append(observe(theta, t_now, row, t_w))
                rec["wall"].append(wall)
                if progress:
                    progress(rec, stats)
        torch.cuda.synchronize()
        for k in ("steps", "accepted", "reverted", "dp_steps", "sparsify_calls", "sparsify_passes", "rows_dropped",
                  "n_rows", "n_rows_max"):
            out_stats[k] = int(getattr(stats, k))
        out_stats["wall_s"] = time.perf_counter() - w0
        out_stats["t_reached"] = float(ten["t"][st.n_rows - 1].item())
        out_stats["n_rhs"] = int(st.n_rhs)
        out_stats["h_last"] = st.h
        out_stats["eps_sparse_over_tol"] = 0.1      # PAPER.md:334, not a parameter of the library
        n = st.n_rows - 1
        last = ten["hist"][n].cpu().numpy()
        out_stats["C_diag_drift"] = abs(float(last[-1, 0]) - 1.0)
        out_stats["R_diag_drift"] = abs(float(last[-1, 2]) - 1.0)
    finally:
        D.dmfe_destroy(ctx)
    return dict(records=rec, stats=out_stats, wall_to_t={("%g" % k): v for k, v in milestones.items()})


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=4, choices=sorted(CONFIGS))
    ap.add_argument("--beta0", type=float, default=0.0, help="inverse temperature of the initial condition (Eq.(12))")
    ap.add_argument("--tol", type=float, default=None)
    ap.add_argument("--stencil", type=int, default=None)
    ap.add_argument("--t-end", type=float, default=1e3)
    ap.add_argument("--L", type=int, default=None)
    ap.add_argument("--n-cap", type=int, default=None, help="row capacity (default: the config's hard cap)")
    ap.add_argument("--max-seconds", type=float, default=None)
    ap.add_argument("--log", default=None, help="append one JSON line per observation record to this file")
    ap.add_argument("--startup", default="ssprk", choices=["ssprk", "dp"],
                    help="dp: Dormand-Prince steps until the stability boundary, then SSPRK(10,4) (PAPER.md:316)")
    ap.add_argument("--step-mode", type=int, default=0, choices=[0, 1],
                    help="0: persistent kernel per batch where it applies (S = 4, L <= 512); 1: graph of launches per step")
    args = ap.parse_args()
    cfg = dict(CONFIGS[args.config])
    if args.L:
        cfg["L"] = args.L
    if args.n_cap:
        cfg["n_cap"] = args.n_cap
    if args.tol:
        cfg["tol"] = args.tol
    if args.stencil:
        cfg["s"] = args.stencil
    cfg["beta0"] = args.beta0
    progress = None
    if args.log:
        def progress(rec, stats):
            with open(args.log, "a") as f:
                f.write(json.dumps(dict(t=rec["t"][-1], E=rec["E"][-1], mu=rec["mu"][-1], h=rec["h"][-1],
                                        n_rows=rec["n_rows"][-1], corr=rec["corr"][-1], wall=rec["wall"][-1],
                                        steps=int(stats.steps), reverted=int(stats.reverted),
                                        passes=int(stats.sparsify_passes))) + "\n")
    out = run(t_end=args.t_end, max_seconds=args.max_seconds, progress=progress, startup=args.startup,
              step_mode=args.step_mode, **cfg)
    r = out["records"]
    line = dict(config=args.config, **cfg, t_end=args.t_end, stats=out["stats"], wall_to_t=out["wall_to_t"],
                E_last=r["E"][-1] if r["E"] else None, corr_last=r["corr"][-1] if r["corr"] else None)
    print(json.dumps(line))


if __name__ == "__main__":
    main()
