"""Pins for the oracle's time stepping (SSPRK(10,4) on the ray ODE of Eq.(22)).

P5  pure 2-spin, quench T=inf -> T=0 (the exact case the paper uses for Fig.4):
    textbook closed form (Cugliandolo-Dean), written here with scipy Bessel functions:
      Gamma(t) = I1(4t)/(2t),  mu(t) = 2 I0(4t)/I1(4t) - 1/t,  E = -mu/2,
      C(t,t') = [I1(2(t+t'))/(t+t')] / sqrt(Gamma(t)Gamma(t')),
      R(t,t') = [I1(2 tau)/tau] sqrt(Gamma(t')/Gamma(t)),  tau = t-t'.
P6  spherical constraint C(t,t)=1 and R(t,t^-)=1 along the run; causality is
    structural (theta <= 1).
P7  high-T paramagnet (BASELINE.json config 1): mu -> T + f'(1)/T, E -> -f(1)/T and the
    equilibrium FDT  R = (1/T) dC/dt'  at late times.
P8  brute force: uniform tensor grid C[i][j], R[i][j], trapezoid memory sums, Heun, Richardson
    in dt -- a different discretisation of Eq.(1)/(13) written here from scratch.
P9  SSPRK(10,4): order conditions of the Butcher tableau, embedded weights are order 3 and not 4,
    the low-storage form equals the tableau form, 4th-order convergence.
"""
import numpy as np
import pytest
from scipy.special import ive

from oracle import dmfe_oracle as O


# ------------------------------------------------------------------------------------ P9
def _order_conditions(A, b, c):
    """Residuals of the 8 rooted-tree order conditions up to order 4."""
    e = np.ones(len(b))
    Ac = A @ c
    return {
        1: [b @ e - 1.0],
        2: [b @ c - 0.5],
        3: [b @ c ** 2 - 1 / 3, b @ Ac - 1 / 6],
        4: [b @ c ** 3 - 0.25, b @ (c * Ac) - 1 / 8, b @ (A @ c ** 2) - 1 / 12, b @ (A @ Ac) - 1 / 24],
    }


def test_P9_ssprk104_order_conditions():
    A = O.ssprk104_butcher()
    c = A.sum(1)
    assert np.allclose(c, O.SSPRK_C, atol=1e-15)
    r = _order_conditions(A, O.SSPRK_B, c)
    assert max(abs(x) for k in r for x in r[k]) < 1e-15
    rh = _order_conditions(A, O.SSPRK_BHAT, c)
    assert max(abs(x) for k in (1, 2, 3) for x in rh[k]) < 1e-15
    assert max(abs(x) for x in rh[4]) > 1e-3          # embedded pair is genuinely third order


def test_P9_low_storage_form_equals_tableau_and_converges():
    A = O.ssprk104_butcher()
    lam = np.array([-1.0, -0.3, 0.2])

    def F(t, y):
        return lam * y + np.sin(t)

    def tableau_step(y, t0, h):
        K = []
        for i in range(10):
            yi = y + h * sum(A[i, j] * K[j] for j in range(i)) if i else y
            K.append(F(t0 + O.SSPRK_C[i] * h, yi))
        return y + h * sum(O.SSPRK_B[i] * K[i] for i in range(10)), \
            h * sum((O.SSPRK_B[i] - O.SSPRK_BHAT[i]) * K[i] for i in range(10))

    y0 = np.array([1.0, -2.0, 0.5])
    y1, d1 = O.ssprk104(F, y0, 0.3, 0.7)
    y2, d2 = tableau_step(y0, 0.3, 0.7)
    assert np.abs(y1 - y2).max() < 1e-14 and np.abs(d1 - d2).max() < 1e-14

    def integrate(n):
        y, t, h = np.array([1.0]), 0.0, 2.0 / n
        for _ in range(n):
            y, _d = O.ssprk104(lambda tt, yy: -yy + np.cos(tt), y, t, h)
            t += h
        return y[0]
    exact = 0.5 * np.exp(-2.0) + 0.5 * (np.cos(2.0) + np.sin(2.0))
    e1, e2 = abs(integrate(8) - exact), abs(integrate(16) - exact)
    assert 12.0 < e1 / e2 < 20.0


# ------------------------------------------------------------------------------------ P5
def _Gamma(t):
    # I1(4t)/(2t) with the exponential factored out: returns (log-free) scaled value & exponent 4t
    return ive(1, 4 * t) / (2 * t)


@pytest.mark.slow
def test_P5_pure_2spin_closed_form():
    L, s, h, nsteps = 128, 6, 0.025, 320        # t <= 8
    grid = O.Grid(L=L, s=s, t_max=20.0)
    model = O.Model(lam=[0.0, 0.0, 1.0], T=0.0)
    H = O.run_fixed(grid, model, h, nsteps)
    n = np.arange(1, H.n_rows)
    t = H.t[n]
    mu_ex = 2 * ive(0, 4 * t) / ive(1, 4 * t) - 1 / t
    assert np.abs(H.mu[n] - mu_ex).max() < 5e-7
    assert np.abs(H.E[n] + mu_ex / 2).max() < 5e-7
    # fields on the rays of the last row and of one in the middle
    for k in (H.n_rows - 1, H.n_rows // 2):
        tk = H.t[k]
        tp = grid.theta * tk
        tau = grid.omega * tk
        # Gamma(t) = e^{4t} _Gamma(t): C = [ive(1,2(t+t'))e^{2(t+t')}/(t+t')]/(e^{2(t+t')} sqrt(g g'))
        tp_safe = np.maximum(tp, 1e-300)
        g_t = _Gamma(tk)
        g_tp = np.where(tp > 0, ive(1, 4 * tp_safe) / (2 * tp_safe), 1.0)
        C_ex = ive(1, 2 * (tk + tp)) / (tk + tp) / np.sqrt(g_t * g_tp)
        tau_safe = np.maximum(tau, 1e-300)
        R_ex = np.where(tau > 0, ive(1, 2 * tau_safe) / tau_safe, 1.0) * np.sqrt(g_tp / g_t)
        # exponentials: e^{2 tau} * e^{(4t' - 4t)/2} = 1  (they cancel exactly)
        assert np.abs(H.hist[k, :, 0] - C_ex).max() < 2e-7
        assert np.abs(H.hist[k, :, 2] - R_ex).max() < 1e-6
    # 4th-order convergence in h of mu(t=2)
    errs = []
    for hh, ns in ((0.1, 20), (0.05, 40)):
        Hh = O.run_fixed(grid, model, hh, ns)
        tt = Hh.t[ns]
        errs.append(abs(Hh.mu[ns] - (2 * ive(0, 4 * tt) / ive(1, 4 * tt) - 1 / tt)))
    assert errs[0] / errs[1] > 6.0 or errs[1] < 5e-8


# ------------------------------------------------------------------------------------ P6, P7
@pytest.fixture(scope="module")
def paramagnet_run():
    grid = O.Grid(L=128, s=4, t_max=20.0)
    model = O.Model(lam=[0.0, 0.0, 0.0, 1.0], T=1.0)
    return grid, model, O.run_fixed(grid, model, 0.05, 400)


@pytest.mark.slow
def test_P6_constraints_hold_along_the_run(paramagnet_run):
    grid, model, H = paramagnet_run
    N = H.n_rows
    assert np.abs(H.hist[:N, -1, 0] - 1.0).max() < 5e-14      # C(t,t) = 1
    assert np.abs(H.hist[:N, -1, 2] - 1.0).max() < 5e-14      # R(t,t^-) = 1
    assert np.abs(H.hist[:N, -1, 1]).max() < 1e-13            # ray derivative on the diagonal = 0
    assert np.abs(H.hist[:N, -1, 3]).max() < 1e-13
    assert np.all(H.hist[:N, :, 0] <= 1.0 + 1e-12) and np.all(H.hist[:N, :, 0] > -1e-9)
    assert np.all(H.hist[:N, :, 2] > -1e-9)


@pytest.mark.slow
def test_P7_paramagnet_equilibrium_and_FDT(paramagnet_run):
    grid, model, H = paramagnet_run
    M = H.n_rows - 1
    T = model.T
    assert H.t[M] == pytest.approx(20.0, abs=1e-12)
    assert H.mu[M] == pytest.approx(T + model.f(1.0, 1) / T, abs=2e-4)      # 2.5
    assert H.E[M] == pytest.approx(-model.f(1.0, 0) / T, abs=1e-4)          # -0.5
    # FDT: R(t,t') = (1/T) dC(t,t')/dt' for tau = t-t' well inside the equilibrated regime.
    # (a) with dC/dt' from the second-argument equation evaluated by the oracle
    out = O.history_integrals(grid, model, H.t, H.mu, H.hist, M)
    tau = grid.omega * H.t[M]
    sel = (tau < 8.0)
    R = H.hist[M, :, 2]
    assert np.abs(T * R[sel] - out["deriv"][sel, 2]).max() < 2e-3
    # (b) with dC/dt' = (dC/di)/(t dtheta/di) by central differences in the index
    C = H.hist[M, :, 0]
    dCdtp = np.gradient(C) / (np.gradient(grid.theta) * H.t[M])
    mid = sel & (tau > 0.2) & (np.arange(grid.L) < grid.L - 3)
    assert np.abs(T * R[mid] / dCdtp[mid] - 1.0).max() < 2e-2
    # time-translation invariance at late times: C(t, t-tau) equals C(t2, t2-tau)
    M2 = M - 100                                   # t2 = 15
    tau2 = grid.omega * H.t[M2]
    Cb = np.interp(1.0, np.sort(tau2), H.hist[M2, :, 0][np.argsort(tau2)])
    Ca = np.interp(1.0, np.sort(tau), C[np.argsort(tau)])
    assert Ca == pytest.approx(Cb, abs=2e-3)


# ------------------------------------------------------------------------------------ P8
def _brute_force(lam, T, t_end, n):
    """Uniform grid t_k = k dt; C[k][j], R[k][j] (j <= k); trapezoid memory sums; Heun in t.
    Eq.(1) with the -mu terms of Eq.(6), Eq.(10),(11),(13), beta0 = 0."""
    lam = np.asarray(lam, dtype=float)
    p = np.arange(len(lam))

    def f1(q):
        return 0.5 * sum(lam[k] * k * q ** (k - 1) for k in p if k >= 1)

    def f2(q):
        return 0.5 * sum(lam[k] * k * (k - 1) * q ** (k - 2) for k in p if k >= 2)

    dt = t_end / n
    C = np.zeros((n + 1, n + 1)); R = np.zeros((n + 1, n + 1))
    C[0, 0] = 1.0; R[0, 0] = 1.0
    mu = np.zeros(n + 1)

    def trap(y):
        return 0.0 if len(y) < 2 else dt * (y.sum() - 0.5 * (y[0] + y[-1]))

    def rhs(k, Ck, Rk):
        """Ck, Rk = row k (entries 0..k; diagonal entries C=1, R=1).  Rows < k are in C, R."""
        K = f2(Ck) * Rk; D = f1(Ck)
        m = T + trap(K * Ck + D * Rk)
        dC = np.zeros(k + 1); dR = np.zeros(k + 1)
        for j in range(k + 1):
            # C(s,t_j) for s = 0..k: symmetric; rows below k are stored, row k is Ck
            Csj = np.concatenate([C[j, :j], C[j:k, j], [Ck[j]]]) if j < k else Ck.copy()
            I1 = trap(K * Csj)
            I2 = trap(D[:j + 1] * (R[j, :j + 1] if j < k else Rk))
            dC[j] = -m * Ck[j] + I1 + I2
            Rsj = np.concatenate([R[j:k, j], [Rk[j]]]) if j < k else np.array([1.0])
            dR[j] = -m * Rk[j] + trap(K[j:] * Rsj)
        return dC, dR, m

    for k in range(n):
        Ck, Rk = C[k, :k + 1].copy(), R[k, :k + 1].copy()
        dC0, dR0, mu[k] = rhs(k, Ck, Rk)
        # predictor for row k+1 (entries 0..k), diagonal appended
        Cp = np.concatenate([Ck + dt * dC0, [1.0]]); Rp = np.concatenate([Rk + dt * dR0, [1.0]])
        C[k + 1, :k + 2], R[k + 1, :k + 2] = Cp, Rp
        dC1, dR1, _ = rhs(k + 1, Cp, Rp)
        C[k + 1, :k + 1] = Ck + 0.5 * dt * (dC0 + dC1[:k + 1])
        R[k + 1, :k + 1] = Rk + 0.5 * dt * (dR0 + dR1[:k + 1])
        C[k + 1, k + 1] = 1.0; R[k + 1, k + 1] = 1.0
    _, _, mu[n] = rhs(n, C[n, :n + 1].copy(), R[n, :n + 1].copy())
    return C, R, mu


@pytest.mark.slow
def test_P8_uniform_grid_brute_force():
    lam, T, t_end = [0.0, 0.0, 0.0, 1.0], 1.0, 3.0
    Ca, Ra, mua = _brute_force(lam, T, t_end, 150)
    Cb, Rb, mub = _brute_force(lam, T, t_end, 300)
    # Heun + trapezoid are second order: Richardson-extrapolate the last row and mu
    mu_x = (4 * mub[-1] - mua[-1]) / 3
    C_x = (4 * Cb[-1, ::2] - Ca[-1]) / 3
    R_x = (4 * Rb[-1, ::2] - Ra[-1]) / 3
    assert abs(mub[-1] - mua[-1]) < 2e-3           # the brute force is itself converged
    grid = O.Grid(L=192, s=4, t_max=20.0)
    model = O.Model(lam=lam, T=T)
    H = O.run_fixed(grid, model, 0.025, 120)
    M = H.n_rows - 1
    assert H.t[M] == pytest.approx(t_end, abs=1e-12)
    assert H.mu[M] == pytest.approx(mu_x, abs=5e-5)
    tp = np.linspace(0.0, t_end, 151)
    # compare at the theta-grid points by interpolating the (smooth) brute-force row
    from scipy.interpolate import CubicSpline
    Cs = CubicSpline(tp, C_x)(grid.theta * t_end)
    Rs = CubicSpline(tp, R_x)(grid.theta * t_end)
    assert np.abs(H.hist[M, :, 0] - Cs).max() < 5e-5
    assert np.abs(H.hist[M, :, 2] - Rs).max() < 5e-5
    # and the mixed model with beta0 = 0 at lower T (different f', f'' paths)
    lam2, T2 = [0.0, 0.0, 1.0, 0.0, 0.5], 0.5
    C2a, R2a, mu2a = _brute_force(lam2, T2, 2.0, 100)
    C2b, R2b, mu2b = _brute_force(lam2, T2, 2.0, 200)
    H2 = O.run_fixed(O.Grid(L=192, s=4, t_max=20.0), O.Model(lam=lam2, T=T2), 0.025, 80)
    assert H2.mu[H2.n_rows - 1] == pytest.approx((4 * mu2b[-1] - mu2a[-1]) / 3, abs=1e-4)


# ------------------------------------------------------------------------------------ controller
@pytest.mark.slow
def test_adaptive_run_with_sparsification_is_sane():
    """PAPER.md:320, :334 (readings G20, G25; tie-breaks are 'parity unpinned'): an adaptive
    p=3, T=1/2 run with periodic sparsification keeps the constraints, loses rows, and heads to
    the aging band E_inf < E(t) < E(0) with E_inf = -0.886693."""
    grid = O.Grid(L=64, s=4, t_max=1e3)
    model = O.Model(lam=[0.0, 0.0, 0.0, 1.0], T=0.5)
    log = []
    H = O.run_adaptive(grid, model, t_end=30.0, tol=1e-6, h0=1e-3, n_cap=400, sp_every=100, log=log)
    N = H.n_rows
    assert H.t[N - 1] >= 30.0
    assert np.abs(H.hist[:N, -1, 0] - 1.0).max() < 1e-12
    assert np.abs(H.hist[:N, -1, 2] - 1.0).max() < 1e-12
    assert np.all(np.diff(H.t[:N]) > 0)
    accepted = sum(1 for r in log if r[3])
    assert N < accepted + 1                          # sparsification removed rows
    assert -0.8867 < H.E[N - 1] < -0.80
    assert all(r[2] <= 2e-6 for r in log if r[3])


# ------------------------------------------------------------------------------------ P15
def _equilibrium_start_run(T=1.0, L=96, s=6, h=0.025, steps=120):
    grid = O.Grid(L=L, s=s, t_max=20.0)
    model = O.Model(lam=[0.0, 0.0, 0.0, 1.0], T=T, beta0=1.0 / T)
    return grid, model, O.run_fixed(grid, model, h, steps)


def test_P15_equilibrium_start_is_stationary_from_the_first_step():
    """The beta0 forcing path (Eq.(12)-(14)): F_C = beta0 f'(C(t,0)) C(t',0) in
    the C equation, beta0 f'(C(t,0)) C(t,0) in mu, -beta0 f(C(t,0)) in E, and row 0 with
    mu0 = T + beta0 f'(1) (reading G13).  For beta0 = 1/T in the paramagnet (p = 3, T = 1 > T_d) the
    system STARTS in equilibrium, so what P7 only reaches as t -> infinity must hold from t = 0:
      mu(t) = T + f'(1)/T = 2.5,  E(t) = -f(1)/T = -0.5  for every stored row,
      C(t,t') = C(t-t'), R(t,t') = R(t-t')  (time-translation invariance),
      T R(tau) = -dC/dtau                     (FDT), from the first rows on.
    A swapped fc/fc2, a missing beta0 f(C(t,0)) in E, a missing beta0 term in mu or a wrong mu0
    each move these by O(0.1) (checked by mutating dmfe_oracle.c / History.__init__)."""
    from scipy.interpolate import CubicSpline
    T = 1.0
    grid, model, H = _equilibrium_start_run(T=T)
    n = H.n_rows
    assert np.abs(H.mu[:n] - (T + 1.5 / T)).max() < 5e-6
    assert np.abs(H.E[:n] + 0.5 / T).max() < 2e-6
    # read C(t, t - tau), R(t, t - tau) off the stored rows with a cubic spline in theta
    for tau in (0.25, 1.0):
        vals = []
        for k in range(1, n):
            t = H.t[k]
            if t < tau + 0.25:
                continue
            th = 1.0 - tau / t
            sC, sR = CubicSpline(grid.theta, H.hist[k, :, 0]), CubicSpline(grid.theta, H.hist[k, :, 2])
            # dC/dtau at fixed t = -(1/t) dC/dtheta
            vals.append((float(sC(th)), float(sR(th)), float(-sC(th, 1) / t)))
        vals = np.array(vals)
        assert len(vals) > 40
        assert np.ptp(vals[:, 0]) < 2e-5, "C(t, t - tau) depends on t: not stationary"
        assert np.ptp(vals[:, 1]) < 6e-5, "R(t, t - tau) depends on t: not stationary"
        assert np.abs(T * vals[:, 1] + vals[:, 2]).max() < 2e-4, "FDT violated"
        assert 0.2 < vals[0, 0] < 0.95          # not vacuous: the correlation has decayed


def test_P15_beta0_zero_is_not_stationary():
    """Sharpness of P15: the same run from the random start (beta0 = 0) is far from stationary."""
    grid = O.Grid(L=64, s=4, t_max=20.0)
    H = O.run_fixed(grid, O.Model(lam=[0.0, 0.0, 0.0, 1.0], T=1.0, beta0=0.0), 0.05, 20)
    assert abs(H.mu[1] - 2.5) > 0.5 and abs(H.E[1] + 0.5) > 0.2


# ------------------------------------------------------------------------------------ controller constants
def test_controller_constants_from_a_stubbed_error_sequence(monkeypatch):
    """"the previous ten time steps are reverted and the time step is halved" when
    eps_RK > 2 eps; otherwise the step is accepted and the next step is reduced to 0.9 h if
    eps_RK > eps, enlarged to 1.01 h if eps_RK < eps/2 (reading G20); the Eq.(24) cap
    13.9/(4 sqrt(f''(1))) applies throughout.  The error estimate is stubbed, so only the
    controller's constants and its bookkeeping are exercised."""
    grid = O.Grid(L=16, s=4, t_max=20.0)
    model = O.Model(lam=[0.0, 0.0, 0.0, 1.0], T=1.0)
    H = O.History(grid, model, 64)
    eps_list = iter([0.2, 0.4, 0.6, 1.5, 0.5, 1.0, 2.0, 2.0000001] + [0.1] * 14 + [3.0, np.nan, 0.1])
    monkeypatch.setattr(O, "rk_step", lambda H_, h_: next(eps_list))

    def fake_complete(H_):
        H_.n_rows += 1
    monkeypatch.setattr(O, "complete_row", fake_complete)
    tol, h = 1.0, 0.1
    cap = 13.9 / (4.0 * np.sqrt(3.0))            # f''(1) = 3 for f = q^3/2
    assert O.h_stab(model) == pytest.approx(cap, rel=1e-15)
    got = []
    for _ in range(25):
        ok, h, eps = O.controller_step(H, h, tol)
        got.append((ok, h, H.n_rows))
    exp, hh, rows = [], 0.1, 1
    for e in [0.2, 0.4, 0.6, 1.5, 0.5, 1.0, 2.0]:            # all accepted (eps <= 2 tol)
        rows += 1
        hh = hh * 0.9 if e > 1.0 else (hh * 1.01 if e < 0.5 else hh)
        exp.append((True, hh, rows))
    rows = max(1, rows - 10); hh /= 2.0                        # 2.0000001 > 2 tol: ten rows, h/2
    exp.append((False, hh, rows))
    for _ in range(14):
        rows += 1; hh *= 1.01
        exp.append((True, hh, rows))
    rows -= 10; hh /= 2.0                                      # 15 rows -> 5
    exp.append((False, hh, rows))
    rows = max(1, rows - 10); hh /= 2.0                        # NaN: reverted too; never below row 0
    exp.append((False, hh, rows))
    rows += 1; hh *= 1.01
    exp.append((True, hh, rows))
    assert [g[0] for g in got] == [e[0] for e in exp]
    assert [g[2] for g in got] == [e[2] for e in exp]
    np.testing.assert_allclose([g[1] for g in got], [e[1] for e in exp], rtol=1e-15)
    # the cap of Eq.(24)
    ok, h2, _ = (lambda: (monkeypatch.setattr(O, "rk_step", lambda H_, h_: 0.0), O.controller_step(H, cap, tol))[1])()
    assert ok and h2 == cap


# ------------------------------------------------------------------------------------ step loop
def test_greedy_walk_equals_odd_positions_of_flagged_runs():
    """PAPER.md:334 "drop n, then skip to n+2": a candidate's neighbours are never removed before it is
    tested, so the sequential walk equals "in every maximal run of flagged candidates drop the 1st, 3rd,
    5th ..." (the form a parallel implementation can use).  Random flag patterns, brute force."""
    rng = np.random.default_rng(7)
    for trial in range(200):
        N = int(rng.integers(3, 60))
        protect = int(rng.integers(0, 8))
        eps = np.where(rng.random(N) < rng.uniform(0.2, 0.9), 0.0, 1.0)
        eps[0] = eps[-1] = np.inf
        keep = O.sparsify_mask(eps, N, tol=1.0, protect_last=protect)
        exp = np.ones(N, dtype=bool)
        last = min(N - 1 - protect, N - 2)
        run = 0
        for n in range(1, N):
            flagged = n <= last and eps[n] < 0.1
            run = run + 1 if flagged else 0
            if flagged and run % 2 == 1:
                exp[n] = False
        assert np.array_equal(keep, exp)


@pytest.mark.slow
def test_step_loop_thinning_passes_and_startup():
    """The oracle's step loop (integrate): Dormand-Prince start-up switches once, periodic thinning with
    several greedy passes drops more rows than one pass, constraints are kept, the state is resumable
    (two calls = one call), and a cap the rule cannot hold ends the run with the capacity status."""
    grid = O.Grid(L=32, s=4, t_max=100.0)
    model = O.Model(lam=[0.0, 0.0, 0.0, 1.0], T=0.5)
    tol = 1e-3          # loose: the step keeps growing by 1.01 and reaches the start-up switch after ~620 steps

    def run(passes, chunks, n_cap=300):
        H = O.History(grid, model, n_cap)
        rs = O.RunState(h=1e-3)
        pol = O.Policy(batch=8, sp_every=40, sp_max_passes=passes, protect_last=24, startup_dp=True)
        for n in chunks:
            O.integrate(H, pol, rs, 1e300, tol, max_steps=n)
        return H, rs

    H1, r1 = run(1, [700])
    H4, r4 = run(4, [700])
    assert r1.status == r4.status == "ok" and not r4.startup
    assert H4.n_rows < H1.n_rows and len(r4.masks) > len(r1.masks)
    n = H4.n_rows
    assert np.abs(H4.hist[:n, -1, 0] - 1.0).max() < 1e-12 and np.abs(H4.hist[:n, -1, 2] - 1.0).max() < 1e-12
    # resumable: the same 700 steps in three calls whose boundaries coincide with batch boundaries
    Hc, rc_ = run(4, [8 * 11, 8 * 30, 700 - 8 * 41])
    assert Hc.n_rows == H4.n_rows and rc_.h == r4.h and np.array_equal(Hc.t[:n], H4.t[:n])
    Ht, rt = run(4, [700], n_cap=40)
    assert rt.status == "capacity" and Ht.n_rows + 2 > 40
