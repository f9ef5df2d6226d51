"""Pins of the oracle's Dormand-Prince 5(4) start-up:
P11 the tableau satisfies the 17 order conditions up to order 5 (b) and the 8 up to order 4 (bhat),
    bhat is not fifth order, row sums equal c, row 7 equals b (FSAL);
P12 real-axis stability limit of the fifth-order method from its stability function (3.3066...),
    above the switch threshold of reading G21;
P13 fifth-order convergence on a scalar ODE with a closed form, the embedded estimate tracks the
    local error;
P14 on the DMFE itself the Dormand-Prince trajectory converges to the pure 2-spin closed form
    (textbook Cugliandolo-Dean, same as pin P5) and agrees with the SSPRK(10,4) trajectory."""
import numpy as np
from scipy.special import ive

from oracle import dmfe_oracle as O


def _trees(A, b, c):
    e = np.ones(len(b))
    Ac, Ac2, AAc = A @ c, A @ c ** 2, A @ (A @ c)
    return {
        1: [b @ e - 1.0],
        2: [b @ c - 1 / 2],
        3: [b @ c ** 2 - 1 / 3, b @ Ac - 1 / 6],
        4: [b @ c ** 3 - 1 / 4, b @ (c * Ac) - 1 / 8, b @ Ac2 - 1 / 12, b @ AAc - 1 / 24],
        5: [b @ c ** 4 - 1 / 5, b @ (c ** 2 * Ac) - 1 / 10, b @ (c * Ac2) - 1 / 15, b @ (c * AAc) - 1 / 30,
            b @ (Ac * Ac) - 1 / 20, b @ (A @ c ** 3) - 1 / 20, b @ (A @ (c * Ac)) - 1 / 40,
            b @ (A @ Ac2) - 1 / 60, b @ (A @ AAc) - 1 / 120],
    }


def test_P11_dormand_prince_order_conditions():
    A, b, bh, c = O.DP_A, O.DP_B, O.DP_BHAT, O.DP_C
    assert np.abs(A.sum(1) - c).max() < 1e-15 and np.array_equal(A[6], b) and np.all(np.triu(A) == 0.0)
    r = _trees(A, b, c)
    assert max(abs(x) for k in r for x in r[k]) < 5e-16
    rh = _trees(A, bh, c)
    assert max(abs(x) for k in (1, 2, 3, 4) for x in rh[k]) < 5e-16
    assert max(abs(x) for x in rh[5]) > 1e-4            # the embedded solution is genuinely fourth order


def test_P12_real_axis_stability_limit():
    A, b = O.DP_A, O.DP_B
    R = lambda z: 1.0 + z * (b @ np.linalg.solve(np.eye(7) - z * A, np.ones(7)))
    # polynomial form of the same function: 1 + z + ... + z^5/120 + z^6/600
    for z in (-0.3, -1.7, -3.0):
        p = sum(z ** k / np.prod(np.arange(1, k + 1)) for k in range(6)) + z ** 6 / 600.0
        assert abs(R(z) - p) < 1e-13
    xs = np.linspace(0.0, 4.0, 40001)
    stable = np.array([abs(R(-x)) <= 1.0 + 1e-14 for x in xs])
    limit = xs[np.argmin(stable) - 1]                   # last stable point before the first unstable one
    assert abs(limit - 3.3066) < 2e-4
    assert O.DP_SWITCH < limit


def test_P13_fifth_order_and_error_estimate():
    F = lambda t, y: -y + np.sin(t)
    exact = lambda t: 1.5 * np.exp(-t) + 0.5 * (np.sin(t) - np.cos(t))

    def run(n):
        y, t, h = np.array([1.0]), 0.0, 1.0 / n
        for _ in range(n):
            y, k7, d = O.dopri54(F, y, t, h, F(t, y))
            t += h
            assert abs(k7[0] - F(t, y)[0]) < 1e-15        # FSAL: k7 is the derivative of the new point
        return abs(y[0] - exact(1.0))
    e1, e2 = run(10), run(20)
    assert 4.6 < np.log2(e1 / e2) < 5.6
    # one step: delta = y5 - y4 is an O(h^5) estimate of the fourth-order solution's local error
    y0, h = np.array([exact(0.4)]), 0.2
    y5, _, d = O.dopri54(F, y0, 0.4, h, F(0.4, y0))
    y4 = y5 - d
    assert abs((y4[0] - exact(0.6)) + d[0]) < 0.15 * abs(d[0])       # up to the O(h^6) error of y5 itself


def test_P14_dormand_prince_on_the_dmfe_matches_2spin_closed_form_and_ssprk():
    L, s, h, n = 64, 6, 0.05, 40
    grid = O.Grid(L=L, s=s, t_max=20.0)
    model = O.Model(np.array([0.0, 0.0, 1.0]), 0.0, 0.0)     # f = q^2/2, T = 0: the case of pin P5
    Hd = O.History(grid, model, n + 2)
    for _ in range(n):
        O.dp_step(Hd, h)
        Hd.n_rows += 1
    Hs = O.run_fixed(grid, model, h, n)
    t = Hd.t[1:n + 1]
    mu_ex = 2.0 * ive(0, 4 * t) / ive(1, 4 * t) - 1.0 / t
    assert np.abs(Hd.mu[1:n + 1] - mu_ex).max() < 5e-6
    assert np.abs(Hd.mu[1:n + 1] - Hs.mu[1:n + 1]).max() < 2e-6
    assert np.abs(Hd.hist[n, :, 0] - Hs.hist[n, :, 0]).max() < 2e-6
    assert abs(Hd.hist[n, -1, 0] - 1.0) < 1e-13 and abs(Hd.hist[n, -1, 2] - 1.0) < 1e-13   # C(t,t) = R(t,t-) = 1


def test_startup_switches_to_ssprk_at_the_stability_boundary():
    grid = O.Grid(L=48, s=4, t_max=50.0)
    model = O.Model(np.array([0.0, 0.0, 0.0, 1.0]), 1.0, 0.0)
    lim = O.DP_SWITCH / (4.0 * np.sqrt(model.f(1.0, 2)))
    log = []
    H = O.run_adaptive(grid, model, t_end=12.0, tol=1.0, h0=0.42, n_cap=400, log=log, startup="dp")
    hs = np.array([x[1] for x in log])                  # step size proposed after each step
    k = int(np.argmax(hs >= lim))                       # first proposal at the boundary: the next step switches
    assert hs[k] >= lim and np.all(hs[:k] < lim) and k >= 3
    # the step after the switch ran with h/2 (then the controller's factor), and nothing later
    # exceeds the SSPRK cap
    assert hs[k + 1] in (0.9 * hs[k] / 2.0, hs[k] / 2.0, 1.01 * hs[k] / 2.0)
    assert np.all(hs[k + 1:] <= O.h_stab(model) + 1e-15)
    assert H.t[H.n_rows - 1] >= 12.0 and abs(H.hist[H.n_rows - 1, -1, 0] - 1.0) < 1e-12
