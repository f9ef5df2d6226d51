"""Pins for the oracle's single right-hand-side evaluation (no time stepping).

P1  interpolation exact on polynomials up to the stencil order (north_star): a history field
    P(t) * Q(index) with deg P <= 3, deg Q <= s-1 is reproduced exactly by the theta-stencil
    (Eq.(18)), the type-1 Hermite lookup (Eq.(19), :256-260) and the type-2
    2-D lookup (Eq.(20), :262-266).  The expected sums are assembled here from *exact* polynomial
    evaluation at the tabulated coordinates, never from the oracle's interpolation code.
P4  constant history closed form: C = R = 1, f = q^2/2 -> mu = T + 2t,
    dC/dt = -T - t(1-theta), dR/dt = -(T+2t) + t(1-theta)  (Eq.(1), Eq.(13) with the -mu terms).
Also: row search against brute force, f', f'' against finite differences, Lagrange weights
against numpy's polynomial fit, sparsification residual Eq.(26) against numerical quadrature of
the two Hermite interpolants.
"""
import numpy as np
import pytest

from oracle import dmfe_oracle as O


def _poly(c, x):
    return np.polyval(c[::-1], x)


def _dpoly(c, x):
    return np.polyval(np.polyder(np.poly1d(c[::-1])).coeffs, x)


def _field_history(grid, t, Pc, Qc, Pr, Qr):
    """hist[n,l] = {P(t_n) Q(l), P'(t_n) Q(l)} for C (Pc,Qc) and R (Pr,Qr); l = 0-based index."""
    L = grid.L
    l = np.arange(L, dtype=np.float64) / L        # scaled index keeps numbers O(1)
    hist = np.zeros((len(t), L, 4))
    hist[:, :, 0] = _poly(Pc, t)[:, None] * _poly(Qc, l)[None, :]
    hist[:, :, 1] = _dpoly(Pc, t)[:, None] * _poly(Qc, l)[None, :]
    hist[:, :, 2] = _poly(Pr, t)[:, None] * _poly(Qr, l)[None, :]
    hist[:, :, 3] = _dpoly(Pr, t)[:, None] * _poly(Qr, l)[None, :]
    return hist


@pytest.mark.parametrize("s,degP", [(4, 2), (6, 2), (4, 3), (10, 3)])
def test_P1_polynomial_fields_are_reproduced(s, degP):
    L, N = 48, 23
    rng = np.random.default_rng(10 + s + degP)
    grid = O.Grid(L=L, s=s, t_max=50.0)
    t = np.concatenate([[0.0], np.cumsum(rng.uniform(0.3, 1.4, N - 1))])
    M = N - 1
    if degP == 3:
        # the top interval uses the quadratic of reading G12 (exact only for deg P <= 2): make
        # that interval so short (1e-7) that its O(D^3) defect is far below rounding, so that
        # the cubic pin tests the Hermite weights of all other intervals alone
        t[M] = t[M - 1] + 1e-7
    Pc = rng.uniform(-1, 1, degP + 1) / (1.0 + t[-1]) ** np.arange(degP + 1)
    Pr = rng.uniform(-1, 1, degP + 1) / (1.0 + t[-1]) ** np.arange(degP + 1)
    Qc = rng.uniform(-1, 1, s)
    Qr = rng.uniform(-1, 1, s)
    hist = _field_history(grid, t, Pc, Qc, Pr, Qr)
    hist[M, :, 1] = hist[M, :, 3] = 777.0        # derivative slots of row M must be ignored
    mu_hist = np.ones(N)
    start, frac = grid.tables()
    X = (start + frac) / L                         # exact (scaled) index coordinates
    model = O.Model(lam=[0.0, 0.0, 1.0], T=0.3)   # f = q^2/2: f'(q) = q, f'' = 1
    out = O.history_integrals(grid, model, t, mu_hist, hist, M, want_rows=True)
    assert (out["rows2"] < M - 1).any() and (out["rows1"] < M - 1).any()
    nu = grid.nu
    targets = np.arange(L)
    th_i = grid.theta[targets][:, None]
    om_i = grid.omega[targets][:, None]
    tM = t[M]
    tau1 = th_i * tM
    tau2 = (th_i + om_i * grid.theta[None, :]) * tM
    lj = (np.arange(L) / L)[None, :]
    C1 = _poly(Pc, tM) * _poly(Qc, X[0]); R1 = _poly(Pr, tM) * _poly(Qr, X[0])
    C2 = _poly(Pc, tM) * _poly(Qc, X[1]); R2 = _poly(Pr, tM) * _poly(Qr, X[1])
    B1C = _poly(Pc, tau1) * _poly(Qc, lj); B1R = _poly(Pr, tau1) * _poly(Qr, lj)
    B2C = _poly(Pc, tau2) * _poly(Qc, X[2]); B2R = _poly(Pr, tau2) * _poly(Qr, X[2])
    exp = np.stack([
        (nu * (R1 * B1C)).sum(1), (nu * (R2 * B2C)).sum(1), (nu * (C1 * B1R)).sum(1),
        (nu * (R2 * B2R)).sum(1), (nu * (B1R * C1)).sum(1), (nu * (B1C * R1)).sum(1),
        (nu * (B2C * R2)).sum(1), (nu * (R2 * B2R)).sum(1)], axis=1)
    scale = np.abs(out["abssums"]).max() + 1e-300
    assert np.abs(out["sums"] - exp).max() < 2e-13 * max(1.0, scale)
    assert np.abs(exp).max() > 1e-3                 # the pin is not vacuous


def test_P1_breaks_one_degree_above_the_stencil():
    # sharpness: degree s in the index is NOT reproduced
    L, N, s = 48, 12, 4
    grid = O.Grid(L=L, s=s, t_max=50.0)
    t = np.linspace(0.0, 6.0, N)
    Qc = np.zeros(s + 1); Qc[-1] = 50.0
    hist = _field_history(grid, t, [1.0], Qc, [1.0], [1.0])
    start, frac = grid.tables()
    X = (start + frac) / L
    model = O.Model(lam=[0.0, 0.0, 1.0], T=0.3)
    out = O.history_integrals(grid, model, t, np.ones(N), hist, N - 1)
    exp_S3 = (grid.nu * _poly(Qc, X[0])).sum(1)      # sum nu f'(C1) B1R with B1R = 1
    assert np.abs(out["sums"][:, 2] - exp_S3).max() > 1e-9


@pytest.mark.parametrize("T,tM", [(0.7, 3.0), (0.0, 11.0)])
def test_P4_constant_history_closed_form(T, tM):
    L, N = 64, 17
    grid = O.Grid(L=L, s=4, t_max=1e3)
    t = np.linspace(0.0, tM, N)
    hist = np.zeros((N, L, 4)); hist[:, :, 0] = 1.0; hist[:, :, 2] = 1.0
    model = O.Model(lam=[0.0, 0.0, 1.0], T=T)
    mu_hist = T + 2.0 * t
    out = O.history_integrals(grid, model, t, mu_hist, hist, N - 1)
    om = grid.omega
    assert out["mu"] == pytest.approx(T + 2 * tM, abs=1e-13 * (1 + tM))
    assert out["E"] == pytest.approx(-tM, abs=1e-13 * (1 + tM))
    d = out["deriv"]
    assert np.abs(d[:, 0] - (-T - tM * om)).max() < 1e-12 * (1 + tM)
    assert np.abs(d[:, 1] - (-(T + 2 * tM) + tM * om)).max() < 1e-12 * (1 + tM)
    # second-argument equations (readings G9-G11): mu(theta_i t) = T + 2 theta_i t is linear in t, so
    # the 4-point Lagrange of orc_mu_at reproduces it; d2C = T + t w_i, d2R = T + 2 theta_i t - t w_i,
    # and the ray derivatives F = d1 + theta_i d2 (Eq.(22))
    th = grid.theta
    assert np.abs(d[:, 2] - (T + tM * om)).max() < 1e-12 * (1 + tM)
    assert np.abs(d[:, 3] - (T + 2 * th * tM - tM * om)).max() < 1e-12 * (1 + tM)
    assert np.abs(d[:, 4] - (d[:, 0] + th * d[:, 2])).max() < 1e-13 * (1 + tM)
    assert np.abs(d[:, 5] - (d[:, 1] + th * d[:, 3])).max() < 1e-13 * (1 + tM)
    assert abs(d[-1, 4]) < 1e-12 * (1 + tM) and abs(d[-1, 5]) < 1e-12 * (1 + tM)   # C(t,t), R(t,t-) stay 1


@pytest.mark.parametrize("M", [1, 2, 3, 4, 9, 33])
def test_mu_at_reproduces_cubics_and_uses_the_new_mu(M):
    """orc_mu_at (reading G11): local 4-point Lagrange in t over rows k..k+3 with
    k = clamp(n(tau) - 1, 0, M - 3) and mu_M = the value just computed.  Any cubic in t is
    reproduced to rounding for every tau in [0, t_M] (fewer rows: degree M); the interpolant goes
    through the nodes; a lower-order or mis-centred window does not pass."""
    rng = np.random.default_rng(M)
    t = np.concatenate([[0.0], np.cumsum(rng.uniform(0.05, 1.5, M))])
    deg = min(3, M)
    coef = rng.uniform(-1.0, 1.0, deg + 1)
    mu_all = np.polyval(coef, t)
    lib = O._load()
    taus = np.concatenate([rng.uniform(0.0, t[M], 40), t, [0.5 * (t[M - 1] + t[M])]])
    for tau in taus:
        got = lib.orc_mu_at(O._p(t), O._p(mu_all), M, float(tau))
        assert got == pytest.approx(np.polyval(coef, tau), abs=2e-12 * (1 + t[M]) ** 3)
    if M >= 4:
        # not exact one degree above (the window is 4 points) ...
        quartic = t ** 4
        tau = 0.5 * (t[M - 1] + t[M])
        assert abs(lib.orc_mu_at(O._p(t), O._p(quartic), M, float(tau)) - tau ** 4) > 1e-6
        # ... and the window is rows n-1 .. n+2 around the interval of tau (clamped at both ends):
        # a spike on a row outside that window leaves the value untouched
        n = 2 if M >= 6 else 1
        tau = 0.5 * (t[n] + t[n + 1])
        base = lib.orc_mu_at(O._p(t), O._p(mu_all), M, float(tau))
        for far in range(M + 1):
            spiked = mu_all.copy(); spiked[far] += 1.0
            moved = lib.orc_mu_at(O._p(t), O._p(spiked), M, float(tau)) != base
            k = min(max(n - 1, 0), M - 3)
            assert moved == (k <= far <= k + 3)


def test_row_search_brute_force():
    rng = np.random.default_rng(0)
    t = np.concatenate([[0.0], np.cumsum(rng.uniform(0.01, 2.0, 40))])
    lib = O._load()
    for M in (1, 2, 7, 40):
        for tau in np.concatenate([t[:M + 1], rng.uniform(0, t[M], 50), [t[M]]]):
            n = lib.orc_row_search(O._p(t), M, float(tau))
            exp = max(k for k in range(M) if t[k] <= tau)
            assert n == exp


def test_f_derivatives_finite_difference():
    m = O.Model(lam=[0.0, 0.0, 1.0, 0.8, 0.5, 0.0, 0.3], T=1.0)
    for q in (-0.4, 0.0, 0.37, 1.0):
        e = 1e-5
        assert m.f(q, 1) == pytest.approx((m.f(q + e) - m.f(q - e)) / (2 * e), abs=1e-9)
        assert m.f(q, 2) == pytest.approx((m.f(q + e, 1) - m.f(q - e, 1)) / (2 * e), abs=1e-9)
    assert m.f(1.0) == pytest.approx(0.5 * (1.0 + 0.8 + 0.5 + 0.3))


@pytest.mark.parametrize("s", [2, 4, 6, 10])
def test_lagrange_weights_vs_polyfit(s):
    import ctypes
    lib = O._load()
    rng = np.random.default_rng(s)
    w = np.zeros(s)
    for u in np.concatenate([rng.uniform(0, s - 1, 5), [0.0, s - 1.0, 1.0]]):
        lib.orc_lagrange_weights(ctypes.c_int(s), ctypes.c_double(u), O._p(w))
        vals = rng.uniform(-1, 1, s)
        p = np.polyfit(np.arange(s), vals, s - 1)
        assert np.dot(w, vals) == pytest.approx(np.polyval(p, u), abs=1e-9)
        assert w.sum() == pytest.approx(1.0, abs=1e-12)


def _hermite(ta, tb, ya, da, yb, db, x):
    D = tb - ta
    u = (x - ta) / D
    return ((2 * u ** 3 - 3 * u ** 2 + 1) * ya + (u ** 3 - 2 * u ** 2 + u) * D * da
            + (-2 * u ** 3 + 3 * u ** 2) * yb + (u ** 3 - u ** 2) * D * db)


def test_sparsify_residual_vs_numerical_quadrature():
    """Eq.(26): integral over [t_{n-1}, t_{n+1}] of (with slice n) - (without)."""
    rng = np.random.default_rng(4)
    L, N = 5, 6
    t = np.concatenate([[0.0], np.cumsum(rng.uniform(0.2, 1.0, N - 1))])
    hist = rng.uniform(-1, 1, (N, L, 4))
    eps = O.sparsify_residuals(L, N, t, hist)
    xg, wg = np.polynomial.legendre.leggauss(8)
    for n in range(1, N - 1):
        acc = 0.0
        for i in range(L):
            for v in (0, 2):
                ya, da = hist[n - 1, i, v], hist[n - 1, i, v + 1]
                yn, dn = hist[n, i, v], hist[n, i, v + 1]
                yb, db = hist[n + 1, i, v], hist[n + 1, i, v + 1]
                tot = 0.0
                for (a, b, yl, dl, yr, dr) in ((t[n - 1], t[n], ya, da, yn, dn), (t[n], t[n + 1], yn, dn, yb, db)):
                    x = 0.5 * (b - a) * xg + 0.5 * (a + b)
                    with_n = _hermite(a, b, yl, dl, yr, dr, x)
                    without = _hermite(t[n - 1], t[n + 1], ya, da, yb, db, x)
                    tot += 0.5 * (b - a) * np.dot(wg, with_n - without)
                acc += abs(tot)
        assert eps[n] == pytest.approx(acc, rel=1e-11, abs=1e-14)
    assert np.isinf(eps[0]) and np.isinf(eps[-1])


def test_sparsify_mask_greedy_rule():
    # drop n if below tol/10 and continue with n+2
    eps = np.array([np.inf, 0.0, 0.0, 0.0, 5.0, 0.0, 0.0, 0.0, 0.0, np.inf])
    keep = O.sparsify_mask(eps, len(eps), tol=1.0, protect_last=0)
    assert keep.tolist() == [True, False, True, False, True, False, True, False, True, True]
    keep = O.sparsify_mask(eps, len(eps), tol=1.0, protect_last=4)
    assert keep.tolist() == [True, False, True, False, True, False, True, True, True, True]
