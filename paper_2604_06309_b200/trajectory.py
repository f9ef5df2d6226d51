"""Adaptive DMFE trajectories on the device: the driver loop around dmfe_rk_step / dmfe_sparsify.

Every step of the path runs inside libdmfe.so; this module only decides WHEN to sparsify (reading
G25 in DESIGN.md: one pass every `sp_every` accepted steps and whenever the history is nearly full),
reads a few rows back at requested observation times and keeps the clock.  Used by bench.py's
trajectory workloads (BASELINE.json configs 3 and 4) and by the trajectory tests.

    python -m paper_2604_06309_b200.trajectory --config 4 --t-end 1e3
"""
from __future__ import annotations

import argparse
import json
import time

import numpy as np

from . import dmfe as D

DP_SWITCH = 3.3      # real-axis stability boundary of Dormand-Prince 5(4) is 3.3066 (reading G21)
SSPRK_STAB = 13.9    # step cap of Eq.(24) as the library applies it (include/dmfe.h)
CONFIGS = {
    # BASELINE.json configs[2], [3] (sizes: DESIGN.md section 4)
    3: dict(lam=[0.0, 0.0, 1.0, 0.0, 0.5], T=0.5, tol=1e-8, n_cap=2048, t_max=1e5, L=512, s=4),
    4: dict(lam=[0.0, 0.0, 0.0, 1.0], T=0.5, tol=1e-8, n_cap=8192, t_max=1e7, L=512, s=4),
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


def run(L, s, t_max, lam, T, tol, n_cap, t_end, h0=1e-3, sp_every=200, protect_last=12, beta0=0.0,
        t_w=(1e2, 1e3, 1e4, 1e5), n_obs=64, max_steps=None, max_seconds=None, progress=None, startup="ssprk"):
    """Integrate from t = 0 to t_end.  Returns a dict with the observation records, the wall-clock
    time at which each decade of t was first passed, and step statistics.  startup = "dp": the
    run starts with Dormand-Prince steps and switches to SSPRK(10,4) with half the step when
    h 4 sqrt(f''(1)) reaches 3.3 (reading G21)."""
    import torch

    ctx = D.dmfe_create(L, s, t_max, lam, T=T, beta0=beta0, tol=tol)
    rec = dict(t=[], E=[], mu=[], h=[], n_rows=[], corr=[], wall=[])
    stats = dict(steps=0, accepted=0, reverted=0, sparsify_calls=0, rows_dropped=0, threshold_doublings=0, status="ok")
    eps_sparse = tol / 10.0                      # Eq.(27) threshold
    milestones = {}
    try:
        theta = D.dmfe_get_tables(ctx, L, want_pairs=False)["theta"]
        st, ten = D.make_state(L, n_cap)
        D.dmfe_init_state(ctx, st, h0)
        lam_a = np.asarray(lam, dtype=np.float64)
        f2_1 = 0.5 * sum(p * (p - 1) * lam_a[p] for p in range(2, len(lam_a)))       # f''(1)
        h_switch = DP_SWITCH / (4.0 * np.sqrt(f2_1)) if f2_1 > 0 else np.inf
        h_cap = SSPRK_STAB / (4.0 * np.sqrt(f2_1)) if f2_1 > 0 else np.inf        # Eq.(24), as dmfe_rk_step caps
        use_dp = startup == "dp"
        stats["dp_steps"] = 0
        # observation times: log-spaced, a record is taken at the first accepted step beyond each
        obs_times = list(np.geomspace(max(10 * h0, 1e-2), t_end, n_obs))
        next_decade = 1.0
        t_now, since_sp = 0.0, 0
        torch.cuda.synchronize()
        w0 = time.perf_counter()
        while t_now < t_end:
            if max_steps is not None and stats["steps"] >= max_steps:
                stats["status"] = "max_steps"
                break
            if max_seconds is not None and time.perf_counter() - w0 > max_seconds:
                stats["status"] = "max_seconds"
                break
            if since_sp >= sp_every or st.n_rows + 2 > n_cap:
                forced = st.n_rows + 2 > n_cap
                before = st.n_rows
                n_after, _ = D.dmfe_sparsify(ctx, st, protect_last)
                stats["sparsify_calls"] += 1
                # hard row cap (BASELINE configs 3, 4): a forced pass that leaves the history more
                # than 90 % full doubles the threshold of Eq.(27) and repeats (G25); reported
                while forced and n_after > 0.9 * n_cap and stats["threshold_doublings"] < 60:
                    eps_sparse *= 2.0
                    stats["threshold_doublings"] += 1
                    D.dmfe_set_sparsify_threshold(ctx, eps_sparse)
                    n_after, _ = D.dmfe_sparsify(ctx, st, protect_last)
                    stats["sparsify_calls"] += 1
                stats["rows_dropped"] += before - n_after
                since_sp = 0
                if forced and n_after + 2 > n_cap:
                    stats["status"] = "capacity"      # DMFE_ECAPACITY: forced passes freed nothing
                    break
            if use_dp and st.h >= h_switch:
                use_dp = False
                D.dmfe_set_step_size(ctx, st, min(st.h / 2.0, h_cap))
            h_used = st.h
            try:
                if use_dp:
                    ok = D.dmfe_dp_step(ctx, st)
                    stats["dp_steps"] += 1
                else:
                    ok = D.dmfe_rk_step(ctx, st)
            except D.DmfeError as e:
                stats["status"] = "error %d" % e.code
                break
            stats["steps"] += 1
            if not ok:
                stats["reverted"] += 1
                t_now = float(ten["t"][st.n_rows - 1].item())
                continue
            stats["accepted"] += 1
            since_sp += 1
            # t is tracked on the host (t + h, as the device does) and read back only when a record is due
            t_est = t_now + h_used
            if obs_times and t_est >= obs_times[0] or t_est >= next_decade or t_est >= t_end:
                t_now = float(ten["t"][st.n_rows - 1].item())
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
            else:
                t_now = t_est
        torch.cuda.synchronize()
        stats["wall_s"] = time.perf_counter() - w0
        stats["t_reached"] = float(ten["t"][st.n_rows - 1].item())
        stats["n_rows"] = st.n_rows
        stats["n_rhs"] = int(st.n_rhs)
        stats["h_last"] = st.h
        stats["eps_sparse_over_tol"] = eps_sparse / tol
        n = st.n_rows - 1
        last = ten["hist"][n].cpu().numpy()
        stats["C_diag_drift"] = abs(float(last[-1, 0]) - 1.0)
        stats["R_diag_drift"] = abs(float(last[-1, 2]) - 1.0)
    finally:
        D.dmfe_destroy(ctx)
    return dict(records=rec, stats=stats, wall_to_t={("%g" % k): v for k, v in milestones.items()})


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--config", type=int, default=4, choices=sorted(CONFIGS))
    ap.add_argument("--t-end", type=float, default=1e3)
    ap.add_argument("--L", type=int, default=None)
    ap.add_argument("--n-cap", type=int, default=None, help="row capacity (default: the config's hard cap)")
    ap.add_argument("--max-seconds", type=float, default=None)
    ap.add_argument("--log", default=None, help="append one JSON line per observation record to this file")
    ap.add_argument("--startup", default="ssprk", choices=["ssprk", "dp"],
                    help="dp: Dormand-Prince steps until the stability boundary, then SSPRK(10,4) (PAPER.md:316)")
    args = ap.parse_args()
    cfg = dict(CONFIGS[args.config])
    if args.L:
        cfg["L"] = args.L
    if args.n_cap:
        cfg["n_cap"] = args.n_cap
    progress = None
    if args.log:
        def progress(rec, stats):
            with open(args.log, "a") as f:
                f.write(json.dumps(dict(t=rec["t"][-1], E=rec["E"][-1], mu=rec["mu"][-1], h=rec["h"][-1],
                                        n_rows=rec["n_rows"][-1], corr=rec["corr"][-1], wall=rec["wall"][-1],
                                        steps=stats["steps"], reverted=stats["reverted"],
                                        doublings=stats["threshold_doublings"])) + "\n")
    out = run(t_end=args.t_end, max_seconds=args.max_seconds, progress=progress, startup=args.startup, **cfg)
    r = out["records"]
    line = dict(config=args.config, **cfg, t_end=args.t_end, stats=out["stats"], wall_to_t=out["wall_to_t"],
                E_last=r["E"][-1] if r["E"] else None, corr_last=r["corr"][-1] if r["corr"] else None)
    print(json.dumps(line))


if __name__ == "__main__":
    main()
