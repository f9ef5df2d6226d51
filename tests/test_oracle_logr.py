"""Pins for the oracle's logarithmic interpolation of the response history (reading G32):
orc_history_integrals_logr.

LR1  a response history R(t, index) = exp(a(t) + b(index)) with a cubic in t and b of degree s-1 is reproduced
     EXACTLY by the type-1 and type-2 lookups (the interpolant acts on log R = a + b and on dR/R = a'); the ordinary
     interpolation is not exact on it.  Expected sums are assembled from the exact field.
LR2  automatic fallback: as soon as one value read by a lookup is non-positive, that lookup equals the ordinary
     interpolation bit for bit; lookups that read only positive values still differ from it.
LR3  positivity: on a steep positive response the log path stays positive where the ordinary 4-point stencil
     overshoots below zero.
LR4  the C channel and the A factors are untouched by the option.
"""
import numpy as np
import pytest

from oracle import dmfe_oracle as O


def _poly(c, x):
    return np.polyval(c[::-1], x)


def _dpoly(c, x):
    return np.polyval(np.polyder(np.poly1d(c[::-1])).coeffs, x)


def _setup(s, seed, N=19, L=48, top_short=True):
    rng = np.random.default_rng(seed)
    grid = O.Grid(L=L, s=s, t_max=50.0)
    t = np.concatenate([[0.0], np.cumsum(rng.uniform(0.3, 1.2, N - 1))])
    if top_short:
        t[-1] = t[-2] + 1e-7        # the top interval is the quadratic of G12: make its defect invisible (as in P1)
    return rng, grid, t


@pytest.mark.parametrize("s", [4, 6])
def test_LR1_exponential_fields_are_reproduced(s):
    rng, grid, t = _setup(s, 40 + s)
    L, N = grid.L, len(t)
    M = N - 1
    a = rng.uniform(-1, 1, 4) / (1.0 + t[-1]) ** np.arange(4)
    b = rng.uniform(-1, 1, s)
    l = np.arange(L) / L
    logR = _poly(a, t)[:, None] + _poly(b, l)[None, :]
    hist = np.zeros((N, L, 4))
    hist[:, :, 0] = 1.0                                   # C = 1
    hist[:, :, 2] = np.exp(logR)
    hist[:, :, 3] = _dpoly(a, t)[:, None] * hist[:, :, 2]   # dR/dt along the ray
    start, frac = grid.tables()
    X = (start + frac) / L
    model = O.Model(lam=[0.0, 0.0, 1.0], T=0.3)           # f' = q, f'' = 1
    out = O.history_integrals(grid, model, t, np.ones(N), hist, M, log_r=True)
    ordinary = O.history_integrals(grid, model, t, np.ones(N), hist, M)
    tM = t[M]
    th_i, om_i = grid.theta[:, None], grid.omega[:, None]
    tau1 = th_i * tM
    B1R = np.exp(_poly(a, tau1) + _poly(b, l[None, :]))
    nu = grid.nu
    # type-1 lookup: S3 = sum_j nu_j f'(C1) B1R with C1 = 1 (the type-2 lookup is pinned pair by pair below)
    assert np.abs(out["sums"][:, 2] - (nu * B1R).sum(1)).max() < 1e-12
    # the ordinary interpolation is NOT exact on this field (sharpness)
    assert np.abs(ordinary["sums"][:, 2] - (nu * B1R).sum(1)).max() > 1e-7


def test_LR1_type2_exact_on_every_clean_pair():
    """Type-2 lookup alone, pair by pair: with f = q^2/2, C = 1 and R_M = 1 the term of S8 = nu R2 f''(B2C) B2R is
    nu_j B2R_ij; one node at a time (nu = unit vector through a one-hot replacement of the grid's weights)."""
    s = 4
    rng, grid, t = _setup(s, 77)
    L, N = grid.L, len(t)
    M = N - 1
    a = rng.uniform(-1, 1, 4) / (1.0 + t[-1]) ** np.arange(4)
    b = rng.uniform(-1, 1, s)
    l = np.arange(L) / L
    hist = np.zeros((N, L, 4))
    hist[:, :, 0] = 1.0
    hist[:, :, 2] = np.exp(_poly(a, t)[:, None] + _poly(b, l)[None, :])
    hist[:, :, 3] = _dpoly(a, t)[:, None] * hist[:, :, 2]
    hist[M, :, 2] = 1.0
    start, frac = grid.tables()
    X = (start + frac) / L
    model = O.Model(lam=[0.0, 0.0, 1.0], T=0.3)
    rows = O.history_integrals(grid, model, t, np.ones(N), hist, M, want_rows=True)["rows2"]
    tau2 = (grid.theta[:, None] + grid.omega[:, None] * grid.theta[None, :]) * t[M]
    B2R = np.exp(_poly(a, tau2) + _poly(b, X[2]))
    checked = 0
    for j in (0, 3, L // 3, L // 2, L - 5):
        g1 = O.Grid(L=L, s=s, t_max=50.0, theta=grid.theta, omega=grid.omega, nu=np.eye(L)[j])
        g1._tables = (start, frac)
        out = O.history_integrals(g1, model, t, np.ones(N), hist, M, log_r=True)
        clean = rows[:, j] + 1 < M
        assert np.abs(out["sums"][clean, 7] - B2R[clean, j]).max() < 1e-12 * max(1.0, B2R[clean, j].max())
        checked += int(clean.sum())
    assert checked > 50


def test_LR2_fallback_is_the_ordinary_interpolation_bit_for_bit():
    s = 4
    rng, grid, t = _setup(s, 5, top_short=False)
    L, N = grid.L, len(t)
    M = N - 1
    hist = np.zeros((N, L, 4))
    hist[:, :, 0] = 1.0
    hist[:, :, 2] = np.exp(-0.3 * t[:, None] * grid.omega[None, :])
    hist[:, :, 3] = -0.3 * grid.omega[None, :] * hist[:, :, 2]
    bad_n, bad_l = 7, 20
    hist[bad_n, bad_l, 2] = -1e-3                         # one non-positive response value
    start, frac = grid.tables()
    model = O.Model(lam=[0.0, 0.0, 1.0], T=0.3)
    rows = O.history_integrals(grid, model, t, np.ones(N), hist, M, want_rows=True)
    touched = 0
    for j in (bad_l - 3, bad_l, bad_l + 2, 5, L - 4):
        g1 = O.Grid(L=L, s=s, t_max=50.0, theta=grid.theta, omega=grid.omega, nu=np.eye(L)[j])
        g1._tables = (start, frac)
        a_ = O.history_integrals(g1, model, t, np.ones(N), hist, M, log_r=True)
        b_ = O.history_integrals(g1, model, t, np.ones(N), hist, M)
        n2, a3 = rows["rows2"][:, j], start[2][:, j]
        reads_bad2 = ((n2 == bad_n) | (n2 + 1 == bad_n)) & (a3 <= bad_l) & (bad_l < a3 + s)
        reads_bad1 = (j == bad_l) & ((rows["rows1"] == bad_n) | (rows["rows1"] + 1 == bad_n))
        # type-2 terms: S4 (index 3), S8 (7); type-1: S3 (2), S5 (4)
        assert np.array_equal(a_["sums"][reads_bad2, 3], b_["sums"][reads_bad2, 3])
        assert np.array_equal(a_["sums"][reads_bad1, 2], b_["sums"][reads_bad1, 2])
        assert np.mean(a_["sums"][~reads_bad2, 3] != b_["sums"][~reads_bad2, 3]) > 0.9   # the option is live elsewhere
        touched += int(reads_bad2.sum()) + int(np.sum(reads_bad1))
    assert touched >= 3


def test_LR3_positivity_on_a_steep_response_and_LR4_C_channel_untouched():
    s = 4
    rng, grid, t = _setup(s, 9, top_short=False)
    L, N = grid.L, len(t)
    M = N - 1
    hist = np.zeros((N, L, 4))
    hist[:, :, 0] = np.exp(-0.2 * t[:, None] * grid.omega[None, :])
    hist[:, :, 1] = -0.2 * grid.omega[None, :] * hist[:, :, 0]
    # response: a step of 12 decades across two grid cells (the ordinary cubic stencil overshoots below zero)
    step = np.where(np.arange(L)[None, :] < L // 2, 1e-12, 1.0)
    hist[:, :, 2] = step * np.exp(-0.1 * t[:, None])
    hist[:, :, 3] = -0.1 * hist[:, :, 2]
    start, frac = grid.tables()
    model = O.Model(lam=[0.0, 0.0, 1.0], T=0.3)
    neg_seen = False
    for j in range(L // 2 - 6, L // 2 + 6):
        g1 = O.Grid(L=L, s=s, t_max=50.0, theta=grid.theta, omega=grid.omega, nu=np.eye(L)[j])
        g1._tables = (start, frac)
        lg = O.history_integrals(g1, model, t, np.ones(N), hist, M, log_r=True)
        od = O.history_integrals(g1, model, t, np.ones(N), hist, M)
        # S8 = nu R2 f''(B2C) B2R: sign(B2R) = sign(S8 / R2); use S4/S8 ratio free check: B2R_log > 0 always
        # R2 > 0 is not guaranteed by the ordinary A factor, so test through S3 = f'(C1) B1R (type-1, C1 > 0) ...
        assert np.all(lg["sums"][:, 2] > 0.0)
        # ... and the C-only sums are identical in both runs (LR4): S1 = f''(C1) R1 B1C, S7 = f'(B2C) R2 share R1, R2 (A factors)
        assert np.array_equal(lg["sums"][:, 0], od["sums"][:, 0]) and np.array_equal(lg["sums"][:, 6], od["sums"][:, 6])
        neg_seen = neg_seen or bool(np.any(od["sums"][:, 7] * lg["sums"][:, 7] < 0.0))
    assert neg_seen, "the ordinary stencil was expected to overshoot below zero somewhere on this field"
