"""Pins for the oracle's values-only right-hand side (BASELINE.json config 2's
"4-point-per-axis Lagrange stencils"): oracle/dmfe_oracle.c orc_history_integrals_values, orc_t_lagrange.

V1  a history field P(t) Q(index) with deg P <= 3 (cubic in t, including the window that contains the current row)
    and deg Q <= s-1 is reproduced exactly by the 4-point-in-t x s-point-in-index lookup; the expected sums are
    assembled here from exact polynomial evaluation, never from the oracle's interpolation code.  One degree above
    (quartic in t) is NOT reproduced.
V2  the t-weights sum to 1, the window is rows n-1 .. n+2 clamped to [0, M], fewer rows than four use all of them.
V3  constant history closed form (same as P4: needs only sum(nu) = 1).
V4  on a smooth field the values-only lookup and the Hermite lookup (which also uses the exact slopes) agree to
    O(Delta^4): the difference falls by ~16 when the row spacing is halved.
"""
import ctypes

import numpy as np
import pytest

from oracle import dmfe_oracle as O
from paper_2604_06309_b200 import inputs


def _poly(c, x):
    return np.polyval(c[::-1], x)


@pytest.mark.parametrize("s,degP,N", [(4, 3, 23), (6, 3, 9), (4, 2, 3), (10, 1, 2)])
def test_V1_polynomial_fields_are_reproduced(s, degP, N):
    L = 48
    rng = np.random.default_rng(100 + s + degP + N)
    grid = O.Grid(L=L, s=s, t_max=50.0)
    t = np.concatenate([[0.0], np.cumsum(rng.uniform(0.3, 1.4, N - 1))])
    M = N - 1
    Pc = rng.uniform(-1, 1, degP + 1) / (1.0 + t[-1]) ** np.arange(degP + 1)
    Pr = rng.uniform(-1, 1, degP + 1) / (1.0 + t[-1]) ** np.arange(degP + 1)
    Qc, Qr = rng.uniform(-1, 1, s), rng.uniform(-1, 1, s)
    l = np.arange(L, dtype=np.float64) / L
    histv = np.zeros((N, L, 2))
    histv[:, :, 0] = _poly(Pc, t)[:, None] * _poly(Qc, l)[None, :]
    histv[:, :, 1] = _poly(Pr, t)[:, None] * _poly(Qr, l)[None, :]
    start, frac = grid.tables()
    X = (start + frac) / L
    model = O.Model(lam=[0.0, 0.0, 1.0], T=0.3)   # f = q^2/2: f'(q) = q, f'' = 1
    out = O.history_integrals_values(grid, model, t, np.ones(N), histv, M, want_rows=True)
    nu, tM = grid.nu, t[M]
    th_i, om_i = grid.theta[:, None], grid.omega[:, None]
    tau1 = th_i * tM
    tau2 = (th_i + om_i * grid.theta[None, :]) * tM
    lj = l[None, :]
    C1 = _poly(Pc, tM) * _poly(Qc, X[0]); R1 = _poly(Pr, tM) * _poly(Qr, X[0])
    C2 = _poly(Pc, tM) * _poly(Qc, X[1]); R2 = _poly(Pr, tM) * _poly(Qr, X[1])
    B1C = _poly(Pc, tau1) * _poly(Qc, lj); B1R = _poly(Pr, tau1) * _poly(Qr, lj)
    B2C = _poly(Pc, tau2) * _poly(Qc, X[2]); B2R = _poly(Pr, tau2) * _poly(Qr, X[2])
    exp = np.stack([
        (nu * (R1 * B1C)).sum(1), (nu * (R2 * B2C)).sum(1), (nu * (C1 * B1R)).sum(1),
        (nu * (R2 * B2R)).sum(1), (nu * (B1R * C1)).sum(1), (nu * (B1C * R1)).sum(1),
        (nu * (B2C * R2)).sum(1), (nu * (R2 * B2R)).sum(1)], axis=1)
    scale = np.abs(out["abssums"]).max() + 1e-300
    assert np.abs(out["sums"] - exp).max() < 5e-13 * max(1.0, scale)
    assert np.abs(exp).max() > 1e-3
    # windows: k = clamp(n - 1, 0, M + 1 - npts)
    npts = min(4, M + 1)
    n2 = np.searchsorted(t[:M], tau2, side="right") - 1
    assert np.array_equal(out["rows2"], np.clip(n2 - 1, 0, M + 1 - npts))


def test_V1_breaks_one_degree_above_in_t():
    L, N, s = 40, 14, 4
    grid = O.Grid(L=L, s=s, t_max=50.0)
    t = np.linspace(0.0, 6.5, N)
    histv = np.ones((N, L, 2))
    histv[:, :, 1] = (t ** 4 / 100.0)[:, None]             # R = t^4/100, C = 1
    model = O.Model(lam=[0.0, 0.0, 1.0], T=0.3)
    out = O.history_integrals_values(grid, model, t, np.ones(N), histv, N - 1)
    tau1 = grid.theta * t[-1]
    exp_S3 = tau1 ** 4 / 100.0                              # sum nu f'(C1) B1R with C1 = 1, sum(nu) = 1
    assert np.abs(out["sums"][:, 2] - exp_S3).max() > 1e-6


@pytest.mark.parametrize("M", [1, 2, 3, 4, 11])
def test_V2_t_lagrange_window_and_partition_of_unity(M):
    rng = np.random.default_rng(M)
    t = np.concatenate([[0.0], np.cumsum(rng.uniform(0.05, 1.5, M))])
    lib = O._load()
    lib.orc_t_lagrange.restype = ctypes.c_int
    w = np.zeros(4)
    npts = ctypes.c_int(0)
    for tau in np.concatenate([rng.uniform(0.0, t[M], 30), t]):
        k = lib.orc_t_lagrange(O._p(t), ctypes.c_int(M), ctypes.c_double(float(tau)), O._p(w), ctypes.byref(npts))
        n = max(j for j in range(M) if t[j] <= tau)
        assert npts.value == min(4, M + 1)
        assert k == min(max(n - 1, 0), M + 1 - npts.value)
        assert abs(w[:npts.value].sum() - 1.0) < 1e-12
        assert abs(np.dot(w[:npts.value], t[k:k + npts.value]) - tau) < 1e-12 * (1 + t[M]) or npts.value < 2


def test_V3_constant_history_closed_form():
    T, tM, L, N = 0.7, 3.0, 64, 17
    grid = O.Grid(L=L, s=4, t_max=1e3)
    t = np.linspace(0.0, tM, N)
    histv = np.ones((N, L, 2))
    model = O.Model(lam=[0.0, 0.0, 1.0], T=T)
    out = O.history_integrals_values(grid, model, t, T + 2.0 * t, histv, N - 1)
    om, th = grid.omega, grid.theta
    assert out["mu"] == pytest.approx(T + 2 * tM, abs=1e-13 * (1 + tM))
    d = out["deriv"]
    assert np.abs(d[:, 0] - (-T - tM * om)).max() < 1e-12 * (1 + tM)
    assert np.abs(d[:, 1] - (-(T + 2 * tM) + tM * om)).max() < 1e-12 * (1 + tM)
    assert np.abs(d[:, 2] - (T + tM * om)).max() < 1e-12 * (1 + tM)
    assert np.abs(d[:, 3] - (T + 2 * th * tM - tM * om)).max() < 1e-12 * (1 + tM)


def test_V4_agrees_with_the_hermite_lookup_to_fourth_order():
    """Smooth analytic field exp(-a t (1 - theta)) on uniform rows: values-only (4-point Lagrange in t) against
    Hermite (values + exact slopes): same theta-stencil, so the difference is the t-interpolation error alone."""
    L, s = 48, 4
    grid = O.Grid(L=L, s=s, t_max=50.0)
    model = O.Model(lam=[0.0, 0.0, 0.0, 1.0], T=0.5)
    diffs = []
    for N in (17, 33, 65):
        t = np.linspace(0.0, 8.0, N)
        tn, om = t[:, None], grid.omega[None, :]
        hist = np.zeros((N, L, 4))
        for a_, w_ in ((0.3, 0.6), (1.1, 0.4)):
            e = np.exp(-a_ * tn * om)
            hist[:, :, 0] += w_ * e
            hist[:, :, 1] += w_ * (-a_ * om) * e
            hist[:, :, 2] += 0.5 * w_ * e
            hist[:, :, 3] += 0.5 * w_ * (-a_ * om) * e
        mu = 1.0 + 0.1 * t
        ref = O.history_integrals(grid, model, t, mu, hist, N - 1)
        val = O.history_integrals_values(grid, model, t, mu, np.ascontiguousarray(hist[:, :, [0, 2]]), N - 1)
        diffs.append(np.abs(val["sums"] - ref["sums"]).max())
        assert np.abs(val["sums"]).max() > 0.05
    assert diffs[0] < 2e-4 and diffs[2] < 2e-6
    assert 8.0 < diffs[0] / diffs[1] < 32.0 and 8.0 < diffs[1] / diffs[2] < 32.0
