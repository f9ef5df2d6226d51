"""Pins for the oracle's precomputed tables (theta-grid, nu, index coordinates, stencil starts).

P2  quadrature exact on low-degree polynomials (north_star)
P3  grid identities of Eq.(16) and a 50-digit mpmath cross-check of theta_i
    against Eq.(16) AS PRINTED, and of the index coordinate X(c) against the inverse of that map.
"""
import numpy as np
import pytest

from oracle import dmfe_oracle as O

mp = pytest.importorskip("mpmath")


def _theta_printed_mp(x, L, t_max):
    """Eq.(16) exactly as printed (alpha=0), at real 1-based index x, in 50-digit arithmetic."""
    mp.mp.dps = 50
    g = -mp.lambertw(-mp.mpf(1) / mp.mpf(t_max), -1).real
    y = (2 * mp.mpf(float(x) if not isinstance(x, mp.mpf) else x) - 1 - L) / (L - 1)
    num = mp.atan(mp.e ** g) - mp.atan(mp.e ** (-g * y))
    den = mp.atan(mp.e ** g) - mp.atan(mp.e ** (-g))
    return num / den


@pytest.mark.parametrize("t_max", [20.0, 1e4, 1e7])
def test_gamma_solves_its_defining_equation(t_max):
    # gamma = -W_{-1}(-1/t_max)  <=>  gamma * exp(-gamma) = 1/t_max on the branch gamma > 1
    g = O.gamma_of_tmax(t_max)
    assert g > 1.0
    assert abs(g * np.exp(-g) * t_max - 1.0) < 1e-13


@pytest.mark.parametrize("L,t_max", [(64, 20.0), (512, 1e4), (4096, 1e4), (1024, 1e7), (257, 1e7)])
def test_grid_identities(L, t_max):
    th, om = O.theta_grid(L, t_max)
    assert th[0] == 0.0 and th[-1] == 1.0
    assert np.all(np.diff(th) > 0)
    assert np.max(np.abs(th + th[::-1] - 1.0)) <= 2.3e-16
    assert np.array_equal(om, th[::-1])
    # condition (15): the finest spacing (at both ends) resolves tau_micro ~ 1 at t = t_max:
    # min spacing * t_max ~ 4/(pi (L-1)) * (1 + O(1/gamma)) << 1
    dmin = np.min(np.diff(th)) * t_max
    assert dmin < 1.0
    g = O.gamma_of_tmax(t_max)
    assert dmin == pytest.approx(2 * g / (L - 1) / (np.pi / 2), rel=0.15) or dmin < 0.05


@pytest.mark.parametrize("L,t_max", [(128, 20.0), (1024, 1e4), (512, 1e7)])
def test_grid_matches_eq16_as_printed_mpmath(L, t_max):
    th, om = O.theta_grid(L, t_max)
    idx = np.unique(np.concatenate([np.arange(0, 6), np.arange(L - 6, L),
                                    np.linspace(0, L - 1, 25).astype(int)]))
    for i in idx:
        i = int(i)
        ref = _theta_printed_mp(i + 1, L, t_max)
        if i in (0, L - 1):
            assert abs(float(ref) - th[i]) < 1e-15
            continue
        assert abs((mp.mpf(th[i]) - ref) / ref) < 2e-14, i
        # omega is the accurate complement: relative accuracy also where theta -> 1
        assert abs((mp.mpf(om[i]) - (1 - ref)) / (1 - ref)) < 2e-14, i


@pytest.mark.parametrize("L,degree", [(64, 5), (256, 5), (1024, 5), (128, 3)])
def test_quadrature_exact_on_polynomials(L, degree):
    th, _ = O.theta_grid(L, 1e4)
    nu = O.quad_weights(th, degree)
    assert abs(nu.sum() - 1.0) < 1e-14
    for k in range(1, degree + 1):
        assert abs(np.dot(nu, th ** k) - 1.0 / (k + 1)) < 1e-13, k
    # a smooth non-polynomial integrand: int_0^1 exp(-3x) dx
    assert abs(np.dot(nu, np.exp(-3 * th)) - (1 - np.exp(-3.0)) / 3.0) < (1e-7 if degree >= 5 else 1e-6)


def test_quadrature_is_not_trivially_exact_beyond_degree():
    # degree-5 spline weights are NOT exact for theta^12 on a coarse grid: the pin above is sharp
    th, _ = O.theta_grid(16, 20.0)
    nu = O.quad_weights(th, 5)
    assert abs(np.dot(nu, th ** 12) - 1.0 / 13) > 1e-9


@pytest.mark.parametrize("L,t_max", [(128, 20.0), (4096, 1e4), (1024, 1e7)])
def test_index_coordinate_inverts_eq16_mpmath(L, t_max):
    """theta_printed(X(c)+1) == c to ~1e-11 index units, for c spread over [0,1] incl. both ends,
    using the complement branch for c > 1/2."""
    rng = np.random.default_rng(5)
    th, om = O.theta_grid(L, t_max)
    i = rng.integers(0, L, size=40)
    j = rng.integers(0, L, size=40)
    (phi1, phi2, psi), (b1, b2, b3) = O.pair_coordinates(th, om, i)
    for c_arr, cb_arr in ((phi1, b1), (phi2, b2), (psi, b3)):
        c = c_arr[np.arange(40), j]
        cb = cb_arr[np.arange(40), j]
        X = O.index_coordinate(c, cb, L, t_max)
        for ck, cbk, Xk in zip(c, cb, X):
            if ck == 0.0 or cbk == 0.0:
                continue
            mp.mp.dps = 50
            # Newton-free check: residual of theta(X) - c divided by dtheta/dx (finite difference)
            f0 = _theta_printed_mp(Xk + 1, L, t_max)
            f1 = _theta_printed_mp(Xk + 1 + mp.mpf("1e-6"), L, t_max)
            slope = (f1 - f0) / mp.mpf("1e-6")
            target = mp.mpf(ck) if ck <= 0.5 else 1 - mp.mpf(cbk)
            assert abs((f0 - target) / slope) < 2e-11, (ck, Xk)


def test_complements_are_cancellation_free():
    L, t_max = 512, 1e7
    th, om = O.theta_grid(L, t_max)
    tg = np.array([L - 1, L - 2, L - 5, 3])
    (phi1, phi2, psi), (b1, b2, b3) = O.pair_coordinates(th, om, tg)
    mp.mp.dps = 40
    for a, i in enumerate(tg):
        for j in (1, 7, L // 2, L - 3):
            ti, oi, tj, oj = (mp.mpf(float(v)) for v in (th[i], om[i], th[j], om[j]))
            # exact complements from (theta, omega) taken as exact inputs with theta+omega == 1
            assert abs(mp.mpf(float(b1[a, j])) - (oi + ti * oj)) <= 4e-16 * (oi + ti * oj)
            assert abs(mp.mpf(float(b2[a, j])) - (oi * oj)) <= 4e-16 * (oi * oj)
            p2 = ti + oi * tj
            assert abs(mp.mpf(float(b3[a, j])) - (oi * tj / p2)) <= 6e-16 * (oi * tj / p2)


@pytest.mark.parametrize("s", [4, 6, 10])
def test_stencil_start_brute_force(s):
    L = 97
    th, om = O.theta_grid(L, 1e4)
    rng = np.random.default_rng(3)
    c = np.concatenate([rng.uniform(0, 1, 200), th[::7], [0.0, 1.0]])
    got = O.stencil_start(th, c, s)
    for ck, gk in zip(c, got):
        lstar = max(l for l in range(L) if th[l] <= ck)
        assert gk == min(max(lstar - (s // 2 - 1), 0), L - s)


def test_tables_shapes_and_ranges():
    g = O.Grid(L=64, s=4, t_max=20.0)
    start, frac = g.tables()
    assert start.shape == (3, 64, 64) and frac.shape == (3, 64, 64)
    assert start.min() >= 0 and start.max() <= 64 - 4
    X = start + frac
    assert X.min() > -1e-9 and X.max() < 63 + 1e-9
    # phi1 is symmetric in (i, j); X(phi1_ij) increases with j; X(psi_ij) decreases with j
    assert np.allclose(X[0], X[0].T, atol=1e-9)
    assert np.all(np.diff(X[0][5:], axis=1) > -1e-9)
    assert np.all(np.diff(X[2][1:], axis=1) < 1e-9)
    # on-grid special cases: j = L-1 (theta_j = 1): phi1 = theta_i, phi2 = 1; psi_{i,0} = 1 (phi2 = theta_i)
    assert np.allclose(X[0][:, -1], np.arange(64), atol=1e-9)
    assert np.allclose(X[1][:, -1], 63.0, atol=1e-9)
    assert np.allclose(X[2][1:, 0], 63.0, atol=1e-9)
    assert np.allclose(X[2][1:, -1], np.arange(1, 64), atol=1e-9)
