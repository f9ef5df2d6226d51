"""GPU parity, Stage C: device-resident SSPRK(10,4) steps, controller and sparsification against
the oracle's step-by-step implementation.

Fixed-step trajectories: observables (E, mu, rows of C and R) within 1e-9 relative (north_star).
Adaptive runs: accept/revert decisions and sparsification keep-masks bit-exact over the compared
window; the oracle runs on the library's tables (theta, omega, nu, start, frac).
"""
import numpy as np
import pytest

from oracle import dmfe_oracle as O

pytestmark = pytest.mark.gpu


class _WithStepMode:
    """The binding with every context switched to one implementation of dmfe_advance (dmfe_set_step_mode):
    0 = the persistent cooperative kernel where it applies (S = 4, L <= 512), 1 = the graph of launches."""

    def __init__(self, dmfe, mode):
        self._dmfe, self._mode = dmfe, mode

    def __getattr__(self, name):
        return getattr(self._dmfe, name)

    def dmfe_create(self, *args, **kw):
        ctx = self._dmfe.dmfe_create(*args, **kw)
        self._dmfe.dmfe_set_step_mode(ctx, self._mode)
        return ctx


@pytest.fixture(scope="module", params=[0, 1], ids=["persistent", "graph"])
def D(request):
    from paper_2604_06309_b200 import dmfe
    dmfe.load_library()
    return _WithStepMode(dmfe, request.param)


def _oracle_grid(D, ctx, L, s, t_max):
    tab = D.dmfe_get_tables(ctx, L)
    g = O.Grid(L=L, s=s, t_max=t_max, theta=tab["theta"], omega=tab["omega"], nu=tab["nu"])
    g._tables = (tab["start"], tab["frac"])
    return g


def _pull(st, ten):
    n = st.n_rows
    return (ten["t"][:n].cpu().numpy(), ten["mu"][:n].cpu().numpy(), ten["energy"][:n].cpu().numpy(),
            ten["hist"][:n].cpu().numpy())


def _assert_traj_close(got, H, rtol):
    """north_star: observables of a trajectory (energy, C(t,t_w), R(t,t_w)) within 1e-9 RELATIVE.  Every
    stored value of C and R is compared relative to itself (no absolute slack: R falls to 1e-6 in these
    runs); mu, E likewise; the stored ray derivatives change sign, so they are compared relative to the
    largest derivative of their row (the scale that enters the next Hermite interpolation)."""
    t, mu, E, hist = got
    n = H.n_rows
    assert len(t) == n
    np.testing.assert_allclose(t, H.t[:n], rtol=1e-14, atol=0)
    np.testing.assert_allclose(mu, H.mu[:n], rtol=rtol, atol=0)
    np.testing.assert_allclose(E[1:], H.E[1:n], rtol=rtol, atol=0)
    assert abs(E[0] - H.E[0]) <= rtol * max(abs(H.E[0]), 1e-300) + 1e-300
    np.testing.assert_allclose(hist[:, :, 0], H.hist[:n, :, 0], rtol=rtol, atol=0)
    np.testing.assert_allclose(hist[:, :, 2], H.hist[:n, :, 2], rtol=rtol, atol=0)
    for k in (1, 3):
        scale = np.max(np.abs(H.hist[:n, :, k]), axis=1, keepdims=True)
        assert np.all(np.abs(hist[:, :, k] - H.hist[:n, :, k]) <= rtol * scale + 1e-300)


@pytest.mark.parametrize("L,s,lam,T,beta0,h,steps", [
    (64, 4, [0, 0, 0, 1.0], 1.0, 0.0, 0.05, 40),          # config 1 shape, shortened
    (48, 6, [0, 0, 1.0, 0, 0.5], 0.5, 0.0, 0.02, 25),     # mixed 2+4
    (40, 4, [0, 0, 0, 1.0], 0.8, 1.2, 0.03, 20),          # beta0 > 0 start
])
def test_fixed_step_trajectory(D, L, s, lam, T, beta0, h, steps):
    t_max = 20.0
    ctx = D.dmfe_create(L, s, t_max, lam, T=T, beta0=beta0)
    try:
        grid = _oracle_grid(D, ctx, L, s, t_max)
        st, ten = D.make_state(L, steps + 3)
        D.dmfe_init_state(ctx, st, h)
        for _ in range(steps):
            assert D.dmfe_rk_step(ctx, st, fixed_step=True)
        got = _pull(st, ten)
        assert st.n_rows == steps + 1 and st.n_rhs == 10 * steps
    finally:
        D.dmfe_destroy(ctx)
    model = O.Model(np.array(lam, dtype=np.float64), T, beta0)
    H = O.run_fixed(grid, model, h, steps)
    _assert_traj_close(got, H, 1e-9)
    # P6 on the GPU result itself: C(t,t) = 1 and R(t,t-) = 1 are preserved by the scheme
    assert np.max(np.abs(got[3][:, -1, 0] - 1.0)) < 1e-13
    assert np.max(np.abs(got[3][:, -1, 2] - 1.0)) < 1e-13


def test_config1_paramagnet_full(D):
    """BASELINE.json config 1: p=3, T=1, h=0.05 to t=20 (400 steps), L=128, s=4; oracle ~10 s."""
    L, s, t_max, h, steps = 128, 4, 20.0, 0.05, 400
    lam = [0, 0, 0, 1.0]
    ctx = D.dmfe_create(L, s, t_max, lam, T=1.0)
    try:
        grid = _oracle_grid(D, ctx, L, s, t_max)
        st, ten = D.make_state(L, steps + 3)
        D.dmfe_init_state(ctx, st, h)
        for _ in range(steps):
            D.dmfe_rk_step(ctx, st, fixed_step=True)
        got = _pull(st, ten)
    finally:
        D.dmfe_destroy(ctx)
    H = O.run_fixed(grid, O.Model(np.array(lam, dtype=np.float64), 1.0, 0.0), h, steps)
    _assert_traj_close(got, H, 1e-9)
    t, mu, E, hist = got
    # P7: paramagnet equilibrium mu -> T + f'(1)/T = 2.5, E -> -f(1)/T = -0.5
    assert abs(mu[-1] - 2.5) < 2e-4 and abs(E[-1] + 0.5) < 1e-4


def _run_both(D, L, s, t_max, lam, T, tol, n_cap, pol_kw, chunks, h0=1e-3, beta0=0.0, between=None):
    """The library's step loop (dmfe_integrate) and the oracle's (O.integrate) on the same tables, in the same
    chunks of attempted steps; after every chunk the loops' states must be EQUAL (integers and step size bit
    for bit: every accept / revert decision, every thinning mask and the start-up switch feed into them)."""
    ctx = D.dmfe_create(L, s, t_max, lam, T=T, beta0=beta0, tol=tol)
    try:
        grid = _oracle_grid(D, ctx, L, s, t_max)
        st, ten = D.make_state(L, n_cap)
        D.dmfe_init_state(ctx, st, h0)
        model = O.Model(np.array(lam, dtype=np.float64), T, beta0)
        H = O.History(grid, model, n_cap)
        pol_o = O.Policy(**pol_kw)
        pol_g = D.dmfe_policy(batch=pol_o.batch, sp_every=pol_o.sp_every, sp_max_passes=pol_o.sp_max_passes,
                              sp_min_gain=pol_o.sp_min_gain, protect_last=pol_o.protect_last,
                              startup_dp=1 if pol_o.startup_dp else 0)
        rs = O.RunState(h=min(h0, O.h_stab(model)))
        stats = D.dmfe_run_stats()
        for c, nsteps in enumerate(chunks):
            if between is not None:
                between(c, D, ctx, st, rs)
            O.integrate(H, pol_o, rs, 1e300, tol, max_steps=nsteps)
            stats, rc = D.dmfe_integrate(ctx, st, pol_g, 1e300, max_steps=nsteps, stats=stats)
            assert st.n_rows == H.n_rows, "row counts differ after chunk %d" % c
            assert st.h == rs.h, "step sizes differ after chunk %d" % c
            assert st.acc_since == rs.acc_since and bool(st.startup) == rs.startup
            # eps_RK = sum |h sum_k (b_k - bhat_k) F_k| is a sum of DIFFERENCES of stage derivatives that agree
            # to 1e-12 of their own scale between the two sides (different summation orders in the eight
            # sums): it is compared against that scale, h sum_k |b_k - bhat_k| sum_i |F_i| (sum_k = 1.2)
            n_last = H.n_rows - 1
            f_scale = np.abs(H.hist[n_last, :, 1]).sum() + np.abs(H.hist[n_last, :, 3]).sum()
            assert abs(st.eps_rk - rs.log[-1][1]) <= 1e-12 * 1.2 * rs.h * f_scale
            assert stats.t == H.t[H.n_rows - 1]
        got = _pull(st, ten)
    finally:
        D.dmfe_destroy(ctx)
    log = rs.log
    assert stats.steps == len(log)
    assert stats.accepted == sum(1 for r in log if r[0]) and stats.reverted == sum(1 for r in log if not r[0])
    assert stats.sparsify_passes == len(rs.masks)
    assert stats.rows_dropped == sum(int((~m).sum()) for m in rs.masks)
    return got, H, rs, stats


def test_step_loop_2000_steps_decisions_and_thinning(D):
    """SURVEY 8(c) Stage C: accept / revert decisions and thinning keep-masks over the first 2000 steps of an
    adaptive run (p = 3, T = 0.5 aging, Dormand-Prince start-up, thinning every 50 accepted steps in up to
    4 passes)."""
    got, H, rs, stats = _run_both(D, 64, 4, 1e3, [0, 0, 0, 1.0], 0.5, 1e-6, 800,
                                  dict(batch=16, sp_every=50, sp_max_passes=4, protect_last=24, startup_dp=True),
                                  chunks=[137, 263, 400, 400, 400, 400])
    assert stats.steps == 2000 and stats.dp_steps > 100 and stats.sparsify_passes > 40
    assert sum(int((~m).sum()) for m in rs.masks) > 500            # the thinning is really exercised
    _assert_traj_close(got, H, 1e-9)


def test_step_loop_with_ten_row_reverts(D):
    """PAPER.md:320 "the previous ten time steps are reverted and the time step is halved": after chunks of
    accepted steps the step size is set far too large on both sides (dmfe_set_step_size / rs.h), so the next
    steps are rejected and ten rows of a populated history are dropped, twice in a row the second time."""
    def between(c, D, ctx, st, rs):
        if c in (1, 3):
            big = 64.0 * st.h
            D.dmfe_set_step_size(ctx, st, big)
            rs.h = big
    got, H, rs, stats = _run_both(D, 48, 4, 100.0, [0, 0, 1.0, 0, 0.5], 0.5, 1e-7, 400,
                                  dict(batch=8, sp_every=10 ** 6, protect_last=24), chunks=[45, 20, 30, 25, 40],
                                  between=between)
    rows = [r[3] for r in rs.log]
    drops = [a - b for a, b in zip(rows[:-1], rows[1:]) if b < a]
    assert stats.reverted >= 3 and drops.count(10) >= 3, "no ten-row revert inside the compared window"
    consecutive = any((not rs.log[k][0]) and (not rs.log[k + 1][0]) for k in range(len(rs.log) - 1))
    assert consecutive, "two consecutive reverts (20 rows) were meant to be covered"
    _assert_traj_close(got, H, 1e-9)


def test_step_loop_config3_shape(D):
    """300 steps at the shape of BASELINE.json config 3 (L = 512, f = (q^2 + 0.5 q^4)/2, T = 0.5, tol = 1e-8,
    s = 4, t_max = 1e5): decisions, thinning and rows against the oracle."""
    got, H, rs, stats = _run_both(D, 512, 4, 1e5, [0, 0, 1.0, 0, 0.5], 0.5, 1e-8, 2048,
                                  dict(batch=50, sp_every=100, protect_last=24), chunks=[120, 180])
    assert stats.steps == 300 and stats.sparsify_passes >= 2
    _assert_traj_close(got, H, 1e-9)


def test_advance_log_matches_single_steps(D):
    """dmfe_advance(n) = n x dmfe_rk_step: same rows bit for bit, and its per-step log holds the decisions."""
    L, s = 48, 4
    lam, T, tol = [0, 0, 0, 1.0], 0.5, 1e-6
    outs = []
    for mode in ("batch", "single"):
        ctx = D.dmfe_create(L, s, 50.0, lam, T=T, tol=tol)
        try:
            st, ten = D.make_state(L, 128)
            D.dmfe_init_state(ctx, st, 1e-3)
            if mode == "batch":
                res, log, rc = D.dmfe_advance(ctx, st, 60, want_log=True)
                assert res.steps == 60 and log.shape == (60, 4)
                assert res.accepted == int(log[:, 0].sum()) and res.n_rows == int(log[-1, 3]) == st.n_rows
                assert res.h_next == log[-1, 2] == st.h
            else:
                for _ in range(60):
                    D.dmfe_rk_step(ctx, st)
            outs.append(_pull(st, ten))
        finally:
            D.dmfe_destroy(ctx)
    for a, b in zip(outs[0], outs[1]):
        assert np.array_equal(a, b)


def test_advance_stops_at_minimal_step(D):
    """the run terminates when the step falls below h_min; the rest of the batch is a no-op."""
    L = 32
    ctx = D.dmfe_create(L, 4, 50.0, [0, 0, 0, 1.0], T=0.5, tol=1e-14, h_min=1e-4)
    try:
        st, ten = D.make_state(L, 64)
        D.dmfe_init_state(ctx, st, 0.4)          # far too large for tol = 1e-14: halved until h < h_min
        res, log, rc = D.dmfe_advance(ctx, st, 40, want_log=True, check=False)
        assert rc == D.DMFE_ESTEPMIN and res.steps < 40 and st.h < 1e-4
        assert res.reverted >= 10 and res.accepted + res.reverted == res.steps == len(log)
        assert log[-1, 2] < 1e-4 and np.all(log[:-1, 2] >= 1e-4)      # the batch stopped at the first h < h_min
    finally:
        D.dmfe_destroy(ctx)


def test_revert_path(D):
    """A step that is far too large must be rejected: rows dropped (at most 10), h halved."""
    L, s = 48, 4
    ctx = D.dmfe_create(L, s, 50.0, [0, 0, 0, 1.0], T=0.5, tol=1e-10)
    try:
        st2, ten2 = D.make_state(L, 64)
        D.dmfe_init_state(ctx, st2, 1.5)      # h0 = 1.5 from t = 0: eps_RK >> tol
        ok = D.dmfe_rk_step(ctx, st2)
        assert not ok and st2.n_rows == 1 and abs(st2.h - 0.75) < 1e-15
    finally:
        D.dmfe_destroy(ctx)


def test_capacity_error(D):
    L = 32
    ctx = D.dmfe_create(L, 4, 50.0, [0, 0, 0, 1.0], T=0.5)
    try:
        st, ten = D.make_state(L, 4)
        D.dmfe_init_state(ctx, st, 1e-3)
        for _ in range(3):
            D.dmfe_rk_step(ctx, st, fixed_step=True)
        with pytest.raises(D.DmfeError) as ei:
            D.dmfe_rk_step(ctx, st, fixed_step=True)
        assert ei.value.code == D.DMFE_ECAPACITY
    finally:
        D.dmfe_destroy(ctx)


def test_sparsify_on_synthetic_rows(D):
    """Sparsify alone on a seeded smooth history: keep mask, compacted t/mu/rows bit-exact."""
    import torch
    from paper_2604_06309_b200 import inputs
    L, N, s, tol = 72, 90, 4, 0.015
    ctx = D.dmfe_create(L, s, 100.0, [0, 0, 0, 1.0], T=0.5, tol=tol)
    try:
        tab = D.dmfe_get_tables(ctx, L, want_pairs=False)
        t, mu, hist = inputs.random_smooth_history(tab["theta"], tab["omega"], N, 3.0, seed=11)
        st, ten = D.make_state(L, N + 5)
        ten["t"][:N] = torch.from_numpy(t).cuda()
        ten["mu"][:N] = torch.from_numpy(mu).cuda()
        ten["hist"][:N] = torch.from_numpy(hist).cuda()
        st.n_rows = N
        n_after, keep = D.dmfe_sparsify(ctx, st, 12, want_mask=True)
        got = _pull(st, ten)
    finally:
        D.dmfe_destroy(ctx)
    eps = O.sparsify_residuals(L, N, t, hist)
    keep_ref = O.sparsify_mask(eps, N, tol, 12)
    assert 0 < (~keep_ref).sum() < N - 13, "test must drop some but not all rows"
    assert np.array_equal(keep, keep_ref)
    assert n_after == keep_ref.sum()
    assert np.array_equal(got[0], t[keep_ref]) and np.array_equal(got[1], mu[keep_ref])
    assert np.array_equal(got[3], hist[keep_ref])


def test_trajectory_driver_with_row_cap(D):
    """The run driver (paper_2604_06309_b200/trajectory.py around dmfe_integrate) under a row cap that the
    paper's thinning rule can hold (threshold tol/10, several greedy passes): constraints kept, energy in the
    aging band; under a cap it cannot hold, the run ends with the capacity status instead of bending the rule."""
    from paper_2604_06309_b200 import trajectory
    kw = dict(L=64, s=4, t_max=200.0, lam=[0, 0, 0, 1.0], T=0.5, tol=1e-6, sp_every=50, n_obs=8, t_w=(1.0, 10.0))
    out = trajectory.run(n_cap=400, t_end=60.0, **kw)
    st = out["stats"]
    assert st["status"] == "ok" and st["t_reached"] >= 60.0
    assert st["n_rows_max"] <= 400 and st["rows_dropped"] > 0 and st["sparsify_passes"] >= st["sparsify_calls"]
    assert st["C_diag_drift"] < 1e-12 and st["R_diag_drift"] < 1e-12
    rec = out["records"]
    assert len(rec["t"]) >= 4 and all(np.isfinite(rec["E"]))
    assert -0.95 < rec["E"][-1] < -0.6
    assert 1.0 in rec["corr"][-1] and 0.0 < rec["corr"][-1][1.0][0] < 1.0
    assert set(out["wall_to_t"]) >= {"1", "10"}
    tight = trajectory.run(n_cap=60, t_end=60.0, **kw)
    assert tight["stats"]["status"] == "capacity" and tight["stats"]["t_reached"] < 60.0


# ------------------------------------------------------------------ Dormand-Prince start-up (8(f)-1)
@pytest.mark.parametrize("L,s,lam,T,beta0,h,steps", [
    (64, 4, [0, 0, 0, 1.0], 1.0, 0.0, 0.05, 30),
    (48, 6, [0, 0, 1.0, 0, 0.5], 0.5, 0.7, 0.02, 20),
])
def test_dormand_prince_fixed_step_trajectory(D, L, s, lam, T, beta0, h, steps):
    """dmfe_dp_step against the oracle's Dormand-Prince steps (pins P11-P14) on identical inputs:
    t, mu, E and all stored rows (values and FSAL derivatives) within 1e-9."""
    t_max = 20.0
    ctx = D.dmfe_create(L, s, t_max, lam, T=T, beta0=beta0)
    try:
        grid = _oracle_grid(D, ctx, L, s, t_max)
        st, ten = D.make_state(L, steps + 3)
        D.dmfe_init_state(ctx, st, h)
        for _ in range(steps):
            assert D.dmfe_dp_step(ctx, st, fixed_step=True)
        got = _pull(st, ten)
        assert st.n_rows == steps + 1 and st.n_rhs == 6 * steps
    finally:
        D.dmfe_destroy(ctx)
    H = O.History(grid, O.Model(np.array(lam, dtype=np.float64), T, beta0), steps + 3)
    for _ in range(steps):
        O.dp_step(H, h)
        H.n_rows += 1
    _assert_traj_close(got, H, 1e-9)
    assert np.max(np.abs(got[3][:, -1, 0] - 1.0)) < 1e-13 and np.max(np.abs(got[3][:, -1, 2] - 1.0)) < 1e-13


def test_dormand_prince_startup_decisions_and_switch(D):
    """Adaptive start-up: Dormand-Prince until h 4 sqrt(f''(1)) >= 3.3, then h/2 and SSPRK(10,4)
    (reading G21): accept / revert sequence, step sizes and the switch step equal the
    oracle's; the trajectory agrees to 1e-9.  Loose tolerance so that the step reaches the boundary."""
    L, s, t_max, tol = 48, 4, 50.0, 1.0
    lam, T = [0, 0, 0, 1.0], 1.0
    ctx = D.dmfe_create(L, s, t_max, lam, T=T, tol=tol)
    try:
        grid = _oracle_grid(D, ctx, L, s, t_max)
        st, ten = D.make_state(L, 200)
        D.dmfe_init_state(ctx, st, 0.42)
        model = O.Model(np.array(lam, dtype=np.float64), T, 0.0)
        H = O.History(grid, model, 200)
        h, use_dp, switched_at = 0.42, True, None
        for step in range(40):
            if use_dp and O.dp_must_switch(model, h):
                use_dp, switched_at = False, step
                h = min(h / 2.0, O.h_stab(model))
                D.dmfe_set_step_size(ctx, st, h)
            if use_dp:
                ok_ref, h, eps_ref = O.dp_controller_step(H, h, tol)
                ok = D.dmfe_dp_step(ctx, st)
            else:
                ok_ref, h, eps_ref = O.controller_step(H, h, tol)
                ok = D.dmfe_rk_step(ctx, st)
            assert ok == ok_ref and st.n_rows == H.n_rows, "decision differs at step %d" % step
            assert abs(st.h - h) <= 1e-15 * h
            assert abs(st.eps_rk - eps_ref) <= 1e-9 * eps_ref   # a sum of differences: see _run_both
        assert switched_at is not None and 3 <= switched_at < 39
        got = _pull(st, ten)
    finally:
        D.dmfe_destroy(ctx)
    _assert_traj_close(got, H, 1e-9)


def test_trajectory_driver_with_dormand_prince_startup(D):
    from paper_2604_06309_b200 import trajectory
    kw = dict(L=64, s=4, t_max=200.0, lam=[0, 0, 0, 1.0], T=0.5, tol=1e-6, n_cap=400, t_end=8.0, sp_every=100,
              n_obs=80, t_w=(1.0,), batch=4)
    a = trajectory.run(startup="dp", h0=1e-3, **kw)
    b = trajectory.run(startup="ssprk", h0=1e-3, **kw)
    assert a["stats"]["status"] == "ok" and a["stats"]["dp_steps"] > 0 and b["stats"]["dp_steps"] == 0
    assert a["stats"]["C_diag_drift"] < 1e-12
    # both integrators resolve the same solution within the tolerance of the run
    ta, Ea = np.array(a["records"]["t"]), np.array(a["records"]["E"])
    tb, Eb = np.array(b["records"]["t"]), np.array(b["records"]["E"])
    assert abs(ta[-1] - tb[-1]) < 0.5 and len(ta) >= 4
    # the records are taken at slightly different times: compare through the local slope of E(t)
    slope = (Eb[-1] - Eb[-2]) / (tb[-1] - tb[-2])
    assert abs(Ea[-1] - (Eb[-1] + slope * (ta[-1] - tb[-1]))) < 5e-5


def test_step_modes_agree():
    """The two implementations of dmfe_advance (persistent kernel / graph of launches) on the same run: the same
    decisions, step sizes bit for bit, rows to rounding (their sums over the nodes run in different orders)."""
    from paper_2604_06309_b200 import dmfe as D0
    L, s, lam, T, tol = 512, 4, [0, 0, 0, 1.0], 0.5, 1e-8
    outs = []
    for mode in (0, 1):
        ctx = D0.dmfe_create(L, s, 1e4, lam, T=T, tol=tol)
        try:
            D0.dmfe_set_step_mode(ctx, mode)
            st, ten = D0.make_state(L, 400)
            D0.dmfe_init_state(ctx, st, 1e-3)
            logs = []
            for n in (1, 7, 50, 120, 33):
                res, log, rc = D0.dmfe_advance(ctx, st, n, want_log=True)
                assert res.steps == n
                logs.append(log)
            outs.append((np.concatenate(logs), st.n_rows, st.h) + _pull(st, ten))
        finally:
            D0.dmfe_destroy(ctx)
    a, b = outs
    assert a[1] == b[1] and a[2] == b[2]
    assert np.array_equal(a[0][:, 0], b[0][:, 0]) and np.array_equal(a[0][:, 2:], b[0][:, 2:])   # accept, h_next, rows
    assert np.array_equal(a[3], b[3])                                                              # t
    for x, y in zip(a[4:], b[4:]):
        scale = np.max(np.abs(y), axis=tuple(range(1, y.ndim)), keepdims=True) if y.ndim > 1 else np.abs(y)
        assert np.all(np.abs(x - y) <= 1e-11 * scale + 1e-300)


def test_step_modes_agree_on_a_long_history():
    """Both implementations of dmfe_advance from the same synthetic state with many more rows than grid nodes
    (6000 rows, L = 512: a grid cell of phi2 spans ~ 12 rows, so the row searches of the general pairs really
    bisect): four fixed steps, new rows compared at the rounding level."""
    import torch
    from paper_2604_06309_b200 import dmfe as D0, inputs
    L, s, N, n_steps, h = 512, 4, 6000, 4, 0.05
    outs = []
    for mode in (0, 1):
        ctx = D0.dmfe_create(L, s, 1e4, [0, 0, 0, 1.0], T=0.5, tol=1e-8)
        try:
            D0.dmfe_set_step_mode(ctx, mode)
            tab = D0.dmfe_get_tables(ctx, L)
            t, mu, hist = inputs.random_smooth_history(tab["theta"], tab["omega"], N, 600.0, seed=11)
            st, ten = D0.make_state(L, N + n_steps + 2)
            ten["t"][:N] = torch.from_numpy(t).cuda()
            ten["mu"][:N] = torch.from_numpy(mu).cuda()
            ten["hist"][:N] = torch.from_numpy(hist).cuda()
            st.n_rows = N
            D0.dmfe_set_step_size(ctx, st, h)
            res, log, rc = D0.dmfe_advance(ctx, st, n_steps, fixed_step=True, want_log=True)
            assert res.steps == n_steps and st.n_rows == N + n_steps
            torch.cuda.synchronize()
            outs.append((ten["t"][N:N + n_steps].cpu().numpy(), ten["mu"][N:N + n_steps].cpu().numpy(),
                         ten["hist"][N:N + n_steps].cpu().numpy(), log))
        finally:
            D0.dmfe_destroy(ctx)
    a, b = outs
    assert np.array_equal(a[0], b[0])
    assert np.all(np.isfinite(a[2])) and np.all(np.isfinite(b[2]))
    assert np.max(np.abs(a[1] - b[1]) / np.abs(b[1])) < 1e-12
    for k in range(4):
        scale = np.max(np.abs(b[2][:, :, k]), axis=1, keepdims=True)
        assert np.max(np.abs(a[2][:, :, k] - b[2][:, :, k]) / scale) < 1e-10, "history component %d" % k
    assert np.max(np.abs(a[3][:, 1] - b[3][:, 1]) / np.abs(b[3][:, 1])) < 1e-4          # eps_RK: a difference of derivatives
