"""GPU parity: libdmfe.so (through its C ABI, via the ctypes binding) against the CPU oracle on
identical seeded inputs.  Stage A tables, Stage B single right-hand side, edge cases.

Tolerances: integer results (stencil starts, row indices) bit-exact; each of
the eight sums within 1e-12 * sum_j |term| (north_star: 1e-12 relative, different summation
order); mu, E 1e-12 relative; combined derivatives within 1e-12 of their magnitude scale.
"""
import numpy as np
import pytest

from oracle import dmfe_oracle as O
from paper_2604_06309_b200 import inputs

pytestmark = pytest.mark.gpu

RTOL = 1e-12


@pytest.fixture(scope="module")
def D():
    from paper_2604_06309_b200 import dmfe
    dmfe.load_library()  # fails loudly if the CUDA library is missing
    return dmfe


def _oracle_grid_from_library(tab, L, s, t_max):
    return O.Grid(L=L, s=s, t_max=t_max, theta=tab["theta"], omega=tab["omega"], nu=tab["nu"])


def gpu_rhs(D, ctx, L, t, mu, hist, n_rows, want_rows=True):
    import torch
    dev = "cuda"
    tt = torch.from_numpy(np.ascontiguousarray(t)).to(dev)
    tm = torch.from_numpy(np.ascontiguousarray(mu)).to(dev)
    th = torch.from_numpy(np.ascontiguousarray(hist)).to(dev)
    z = lambda *shape: torch.full(shape, float("nan"), dtype=torch.float64, device=dev)
    out = dict(d1C=z(L), d1R=z(L), mu_out=z(1), d2C=z(L), d2R=z(L), F=z(L, 2), energy=z(1), sums=z(8, L))
    if want_rows:
        out["rows1"] = torch.full((L,), -1, dtype=torch.int32, device=dev)
        out["rows2"] = torch.full((L, L), -1, dtype=torch.int32, device=dev)
    D.dmfe_history_integrals(ctx, n_rows, tt, tm, th, **out)
    torch.cuda.synchronize()
    return {k: v.cpu().numpy() for k, v in out.items()}


def compare_rhs(g, ref, tol=RTOL):
    """g: GPU outputs, ref: oracle outputs (dict of history_integrals)."""
    if "rows1" in g:
        assert np.array_equal(g["rows1"], ref["rows1"]), "type-1 row indices differ"
        assert np.array_equal(g["rows2"], ref["rows2"]), "type-2 row indices differ"
    sums = g["sums"].T  # [L,8]
    err = np.abs(sums - ref["sums"])
    bound = tol * ref["abssums"] + 1e-300
    worst = np.max(err / bound)
    assert worst <= 1.0, "sums off by %.3g x tolerance" % worst
    assert abs(g["mu_out"][0] - ref["mu"]) <= tol * abs(ref["mu"])
    assert abs(g["energy"][0] - ref["E"]) <= tol * max(abs(ref["E"]), 1e-300)
    d = ref["deriv"]
    sc = ref["scale"]
    for k, name in enumerate(["d1C", "d1R", "d2C", "d2R"]):
        e = np.abs(g[name] - d[:, k])
        w = np.max(e / (tol * sc[:, k] + 1e-300))
        assert w <= 1.0, "%s off by %.3g x tolerance" % (name, w)
    th = ref["theta"]
    scF = np.stack([sc[:, 0] + th * sc[:, 2], sc[:, 1] + th * sc[:, 3]], axis=1)
    e = np.abs(g["F"] - d[:, 4:6])
    assert np.max(e / (tol * scF + 1e-300)) <= 1.0


# ------------------------------------------------------------------------------------ Stage A
@pytest.mark.parametrize("L,s,t_max", [(128, 4, 20.0), (257, 6, 1e7), (512, 4, 1e4), (96, 10, 1e5)])
def test_tables_match_oracle(D, L, s, t_max):
    ctx = D.dmfe_create(L, s, t_max, [0, 0, 0, 1.0], T=1.0)
    try:
        tab = D.dmfe_get_tables(ctx, L)
    finally:
        D.dmfe_destroy(ctx)
    ref = O.Grid(L=L, s=s, t_max=t_max)
    # grid: endpoints exact, symmetric complement, relative 1e-13 against the oracle's own grid
    assert tab["theta"][0] == 0.0 and tab["theta"][-1] == 1.0
    assert np.array_equal(tab["omega"], tab["theta"][::-1])
    assert np.all(np.diff(tab["theta"]) > 0)
    np.testing.assert_allclose(tab["theta"][1:], ref.theta[1:], rtol=1e-13, atol=0)
    # quadrature weights: relative 1e-10 (spline solve) and the pin P2 on the library's own weights
    np.testing.assert_allclose(tab["nu"], ref.nu, rtol=1e-10, atol=1e-10 * np.max(np.abs(ref.nu)))
    for k in range(6):
        assert abs(np.sum(tab["nu"] * tab["theta"] ** k) - 1.0 / (k + 1)) < 5e-14
    # pair tables: the oracle recomputes them from the library's theta/omega
    g2 = _oracle_grid_from_library(tab, L, s, t_max)
    start, frac = g2.tables()
    assert np.array_equal(tab["start"], start), "stencil starts are not bit-exact"
    assert np.max(np.abs(tab["frac"] - frac)) <= 1e-11


def test_tables_row_range_hook(D):
    L, s = 128, 4
    ctx = D.dmfe_create(L, s, 1e4, [0, 0, 1.0, 0, 0.5], T=0.5)
    try:
        full = D.dmfe_get_tables(ctx, L)
        part = D.dmfe_get_tables(ctx, L, i0=17, n_targets=9)
    finally:
        D.dmfe_destroy(ctx)
    assert np.array_equal(part["start"], full["start"][:, 17:26])
    assert np.array_equal(part["frac"], full["frac"][:, 17:26])


# ------------------------------------------------------------------------------------ Stage B
CASES = [
    # L, N, s, lam, T, beta0, t_max, t_end
    (96, 37, 4, [0, 0, 0, 1.0], 1.0, 0.0, 50.0, 30.0),
    (100, 23, 6, [0, 0, 1.0, 0, 0.5], 0.5, 0.0, 1e3, 200.0),
    (130, 41, 10, [0, 0, 1.0, 0.8, 0.5], 0.7, 0.0, 1e2, 60.0),
    (64, 9, 4, [0, 0, 0, 0.5, 0, 0, 0, 0, 0, 0.5], 0.3, 1.5, 40.0, 7.0),   # 3+9 model, beta0 > 0
    (333, 301, 4, [0, 0, 2.0], 0.0, 0.0, 1e4, 900.0),                      # ragged L, pure 2-spin, T = 0
    (48, 2, 2, [0, 0, 0, 1.0], 1.0, 0.0, 10.0, 0.01),                      # n_rows = 2: only row 0 + current row
    (48, 3, 8, [0, 0, 0, 1.0], 1.0, 0.0, 10.0, 0.02),
]


@pytest.mark.parametrize("L,N,s,lam,T,beta0,t_max,t_end", CASES)
def test_rhs_matches_oracle_small(D, L, N, s, lam, T, beta0, t_max, t_end):
    ctx = D.dmfe_create(L, s, t_max, lam, T=T, beta0=beta0)
    try:
        tab = D.dmfe_get_tables(ctx, L)
        grid = _oracle_grid_from_library(tab, L, s, t_max)
        t, mu, hist = inputs.random_smooth_history(tab["theta"], tab["omega"], N, t_end, seed=L + N)
        hist[N - 1, :, 1] = np.nan  # derivative slots of the current row must be ignored
        hist[N - 1, :, 3] = np.inf
        mu[N - 1] = np.nan
        g = gpu_rhs(D, ctx, L, t, mu, hist, N)
    finally:
        D.dmfe_destroy(ctx)
    model = O.Model(np.array(lam, dtype=np.float64), T, beta0)
    ref = O.history_integrals(grid, model, t, mu, hist, N - 1, tables=(tab["start"], tab["frac"]), want_rows=True)
    ref["theta"] = tab["theta"]
    compare_rhs(g, ref)


@pytest.mark.parametrize("L,lo,hi,t_max,lam", [
    (512, -2.0, 4.0, 1e4, [0, 0, 0, 1.0]),                 # config-2 recipe at reduced L
    (1024, -2.0, 7.0, 1e7, [0, 0, 1.0, 0.8, 0.5]),         # config-5 recipe, smallest L
])
def test_rhs_matches_oracle_synthetic(D, L, lo, hi, t_max, lam):
    s = 4
    ctx = D.dmfe_create(L, s, t_max, lam, T=0.5)
    try:
        tab = D.dmfe_get_tables(ctx, L)
        grid = _oracle_grid_from_library(tab, L, s, t_max)
        t, mu, hist = inputs.synthetic_history(tab["theta"], tab["omega"], L, lo, hi)
        g = gpu_rhs(D, ctx, L, t, mu, hist, L)
    finally:
        D.dmfe_destroy(ctx)
    model = O.Model(np.array(lam, dtype=np.float64), 0.5, 0.0)
    ref = O.history_integrals(grid, model, t, mu, hist, L - 1, tables=(tab["start"], tab["frac"]), want_rows=True)
    ref["theta"] = tab["theta"]
    compare_rhs(g, ref)


def _sampled_blocks_parity(D, L, s, t_max, lam, lo, hi, n_blocks):
    """Every output of seeded blocks of 32 targets (first and last block included) of one full-size
    evaluation against the oracle run on those targets with the library's tables."""
    ctx = D.dmfe_create(L, s, t_max, lam, T=0.5)
    try:
        tab = D.dmfe_get_tables(ctx, L, want_pairs=False)
        t, mu, hist = inputs.synthetic_history(tab["theta"], tab["omega"], L, lo, hi)
        g = gpu_rhs(D, ctx, L, t, mu, hist, L, want_rows=False)
        rng = np.random.Generator(np.random.PCG64(L))
        blocks = np.sort(rng.choice(L // 32, size=n_blocks, replace=False)) * 32
        blocks = np.unique(np.concatenate([[0], blocks, [L - 32]]))
        grid = _oracle_grid_from_library(tab, L, s, t_max)
        model = O.Model(np.array(lam, dtype=np.float64), 0.5, 0.0)
        for i0 in blocks:
            part = D.dmfe_get_tables(ctx, L, i0=int(i0), n_targets=32)
            targets = np.arange(i0, i0 + 32, dtype=np.int32)
            ref = O.history_integrals(grid, model, t, mu, hist, L - 1, targets=targets,
                                      tables=(part["start"], part["frac"]))
            err = np.abs(g["sums"].T[targets] - ref["sums"])
            worst = np.max(err / (RTOL * ref["abssums"] + 1e-300))
            assert worst <= 1.0, "block %d: sums off by %.3g x tolerance" % (i0, worst)
            for k, name in enumerate(["d1C", "d1R", "d2C", "d2R"]):
                e = np.abs(g[name][targets] - ref["deriv"][:, k])
                assert np.max(e / (RTOL * ref["scale"][:, k] + 1e-300)) <= 1.0, name
        assert abs(g["mu_out"][0] - ref["mu"]) <= RTOL * abs(ref["mu"])
        assert abs(g["energy"][0] - ref["E"]) <= RTOL * max(abs(ref["E"]), 1e-300)
    finally:
        D.dmfe_destroy(ctx)


def test_rhs_full_bench_size_sampled_targets(D):
    """BASELINE.json config 2 at its full size (L = N = 4096, the launch configuration bench.py
    times)."""
    _sampled_blocks_parity(D, 4096, 4, 1e4, [0, 0, 0, 1.0], -2.0, 4.0, n_blocks=8)


def test_rhs_large_grid_global_table_path_sampled_targets(D):
    """Config-5 recipe (mixed f, rows on [1e-2, 1e7]) at L = N = 10240: above L = 9685 the per-call
    tables (24 L bytes) no longer fit in shared memory and the kernel reads them from global
    memory -- the launch configuration of the L = 16384 and 32768 points of the scaling sweep."""
    _sampled_blocks_parity(D, 10240, 4, 1e7, [0, 0, 1.0, 0.8, 0.5], -2.0, 7.0, n_blocks=6)


def test_rhs_mode1_row_table_in_global_memory_sampled_targets(D):
    """Config-5 recipe at L = N = 8192: the current row and the brackets fit in shared memory, the
    row table does not (third launch configuration of the pair kernel, the one of the L = 8192
    point of the scaling sweep)."""
    _sampled_blocks_parity(D, 8192, 4, 1e7, [0, 0, 1.0, 0.8, 0.5], -2.0, 7.0, n_blocks=4)


def test_rhs_one_warp_per_target_launch_shape_all_targets(D):
    """L = 2304 = just below 16 x 148 warps: the launcher gives every target ONE warp (G = 1: no cross-warp
    reduction, no group barrier) -- the launch shape of the L = 16384 and 32768 sweep points.  All targets,
    row indices bit-exact."""
    L, s, t_max, lam = 2304, 4, 1e4, [0, 0, 1.0, 0.8, 0.5]
    ctx = D.dmfe_create(L, s, t_max, lam, T=0.5)
    try:
        tab = D.dmfe_get_tables(ctx, L)
        grid = _oracle_grid_from_library(tab, L, s, t_max)
        N = 700
        t, mu, hist = inputs.synthetic_history(tab["theta"], tab["omega"], N, -2.0, 4.0)
        g = gpu_rhs(D, ctx, L, t, mu, hist, N)
    finally:
        D.dmfe_destroy(ctx)
    model = O.Model(np.array(lam, dtype=np.float64), 0.5, 0.0)
    ref = O.history_integrals(grid, model, t, mu, hist, N - 1, tables=(tab["start"], tab["frac"]), want_rows=True)
    ref["theta"] = tab["theta"]
    compare_rhs(g, ref)


def test_rhs_config5_L16384_sampled_targets(D):
    """BASELINE.json configs[4] at L = N = 16384 (8.6 GB of history, 6.4 GB of pair tables, one warp per
    target, per-call tables in global memory): 512 seeded targets (16 blocks of 32, first and last included)
    against the oracle, as SURVEY.md 8(d) asks for L >= 16384."""
    _sampled_blocks_parity(D, 16384, 4, 1e7, [0, 0, 1.0, 0.8, 0.5], -2.0, 7.0, n_blocks=14)


def test_rhs_closed_form_constant_history_full_size_all_targets(D):
    """A property that holds at any size, checked on every target of the bench-size evaluation
    (L = N = 4096, log-spaced rows of config 2) without the oracle: for the constant history
    C = R = 1 (slopes 0), f = q^2/2 and mu_n = T + 2 t_n every interpolation is exact and the sums
    need only sum(nu) = 1 (oracle pin P4, Eq.(1), (13), (14)):
      mu = T + 2t, E = -t, d1C_i = -T - t w_i, d1R_i = -(T + 2t) + t w_i,
      d2C_i = T + t w_i, d2R_i = T + 2 theta_i t - t w_i, F = d1 + theta_i d2      (w_i = 1 - theta_i)."""
    L, s, t_max, T = 4096, 4, 1e4, 0.7
    ctx = D.dmfe_create(L, s, t_max, [0.0, 0.0, 1.0], T=T)
    try:
        tab = D.dmfe_get_tables(ctx, L, want_pairs=False)
        th, om = tab["theta"], tab["omega"]
        t = inputs.log_times(L, -2.0, 4.0)
        mu = T + 2.0 * t
        hist = np.zeros((L, L, 4))
        hist[:, :, 0] = 1.0
        hist[:, :, 2] = 1.0
        g = gpu_rhs(D, ctx, L, t, mu, hist, L, want_rows=False)
    finally:
        D.dmfe_destroy(ctx)
    tM = t[-1]
    tol = 1e-12 * (1.0 + tM)
    assert abs(g["mu_out"][0] - (T + 2 * tM)) < tol and abs(g["energy"][0] + tM) < tol
    assert np.abs(g["sums"] - 1.0).max() < 1e-12                      # all eight sums are sum(nu) = 1
    assert np.abs(g["d1C"] - (-T - tM * om)).max() < tol
    assert np.abs(g["d1R"] - (-(T + 2 * tM) + tM * om)).max() < tol
    assert np.abs(g["d2C"] - (T + tM * om)).max() < tol
    assert np.abs(g["d2R"] - (T + 2 * th * tM - tM * om)).max() < tol
    FC = (-T - tM * om) + th * (T + tM * om)
    FR = (-(T + 2 * tM) + tM * om) + th * (T + 2 * th * tM - tM * om)
    assert np.abs(g["F"][:, 0] - FC).max() < tol and np.abs(g["F"][:, 1] - FR).max() < tol


@pytest.mark.parametrize("L,N,s,lam,T,t_max,t_end,poison", [
    (96, 37, 4, [0, 0, 0, 1.0], 1.0, 50.0, 30.0, False),
    (100, 23, 6, [0, 0, 1.0, 0, 0.5], 0.5, 1e3, 200.0, True),
    (130, 41, 10, [0, 0, 1.0, 0.8, 0.5], 0.7, 1e2, 60.0, True),
    (64, 3, 2, [0, 0, 0, 1.0], 1.0, 10.0, 0.02, False),
])
def test_rhs_log_response_interpolation(D, L, N, s, lam, T, t_max, t_end, poison):
    """dmfe_params.log_r (reading G32): logarithmic interpolation of the response history with
    automatic fallback, against the oracle's orc_history_integrals_logr; `poison` plants non-positive response
    values so that both branches run inside one evaluation."""
    ctx = D.dmfe_create(L, s, t_max, lam, T=T, log_r=True)
    try:
        tab = D.dmfe_get_tables(ctx, L)
        grid = _oracle_grid_from_library(tab, L, s, t_max)
        t, mu, hist = inputs.random_smooth_history(tab["theta"], tab["omega"], N, t_end, seed=L + N)
        if poison:
            rng = np.random.Generator(np.random.PCG64(N))
            for _ in range(40):
                hist[rng.integers(0, N - 1), rng.integers(0, L), 2] *= -1.0
            hist[N // 2, L // 3, 2] = 0.0
        g = gpu_rhs(D, ctx, L, t, mu, hist, N)
    finally:
        D.dmfe_destroy(ctx)
    model = O.Model(np.array(lam, dtype=np.float64), T, 0.0)
    ref = O.history_integrals(grid, model, t, mu, hist, N - 1, tables=(tab["start"], tab["frac"]), want_rows=True,
                              log_r=True)
    ref["theta"] = tab["theta"]
    compare_rhs(g, ref)
    plain = O.history_integrals(grid, model, t, mu, hist, N - 1, tables=(tab["start"], tab["frac"]))
    assert np.abs(plain["sums"] - ref["sums"]).max() > 1e-9 * np.abs(ref["abssums"]).max()   # the option is live


def test_rhs_rows_in_a_larger_buffer(D):
    """n_rows < n_cap: rows beyond the current one are never touched (filled with NaN here)."""
    L, N, s = 80, 20, 4
    ctx = D.dmfe_create(L, s, 100.0, [0, 0, 0, 1.0], T=0.8)
    try:
        tab = D.dmfe_get_tables(ctx, L)
        grid = _oracle_grid_from_library(tab, L, s, 100.0)
        t, mu, hist = inputs.random_smooth_history(tab["theta"], tab["omega"], N, 12.0, seed=5)
        cap = N + 7
        t2 = np.full(cap, np.nan); t2[:N] = t
        mu2 = np.full(cap, np.nan); mu2[:N] = mu
        h2 = np.full((cap, L, 4), np.nan); h2[:N] = hist
        g = gpu_rhs(D, ctx, L, t2, mu2, h2, N)
    finally:
        D.dmfe_destroy(ctx)
    model = O.Model(np.array([0, 0, 0, 1.0]), 0.8, 0.0)
    ref = O.history_integrals(grid, model, t, mu, hist, N - 1, tables=(tab["start"], tab["frac"]), want_rows=True)
    ref["theta"] = tab["theta"]
    compare_rhs(g, ref)


def test_host_buffer_call_equals_device_call(D):
    L, N, s = 96, 30, 4
    ctx = D.dmfe_create(L, s, 100.0, [0, 0, 0, 1.0], T=0.8)
    try:
        tab = D.dmfe_get_tables(ctx, L, want_pairs=False)
        t, mu, hist = inputs.random_smooth_history(tab["theta"], tab["omega"], N, 12.0, seed=6)
        g = gpu_rhs(D, ctx, L, t, mu, hist, N, want_rows=False)
        d1C, d1R, m, e = np.zeros(L), np.zeros(L), np.zeros(1), np.zeros(1)
        D.dmfe_history_integrals_host(ctx, N, t, mu, hist, d1C, d1R, m, e)
    finally:
        D.dmfe_destroy(ctx)
    assert np.array_equal(d1C, g["d1C"]) and np.array_equal(d1R, g["d1R"])
    assert m[0] == g["mu_out"][0] and e[0] == g["energy"][0]


def test_bad_arguments_are_rejected(D):
    with pytest.raises(D.DmfeError):
        D.dmfe_create(6, 4, 100.0, [0, 0, 0, 1.0], T=1.0)        # L < 2s
    with pytest.raises(D.DmfeError):
        D.dmfe_create(64, 5, 100.0, [0, 0, 0, 1.0], T=1.0)       # odd stencil
    with pytest.raises(D.DmfeError):
        D.dmfe_create(64, 4, 2.0, [0, 0, 0, 1.0], T=1.0)         # t_max <= e
    import torch
    ctx = D.dmfe_create(64, 4, 100.0, [0, 0, 0, 1.0], T=1.0)
    try:
        z = torch.zeros(4, dtype=torch.float64, device="cuda")
        h = torch.zeros((4, 64, 4), dtype=torch.float64, device="cuda")
        with pytest.raises(D.DmfeError):
            D.dmfe_history_integrals(ctx, 1, z, z, h)              # n_rows < 2
    finally:
        D.dmfe_destroy(ctx)


@pytest.mark.parametrize("s,values_only", [(4, False), (10, False), (4, True)])
def test_every_target_is_computed_when_rounds_are_handed_out_dynamically(D, s, values_only):
    """L = 4096 is past the point (four rounds of targets per CTA) from which the pair kernels take their rounds from a
    global counter instead of a static round-robin.  Outputs start as NaN: every target must have been written, by
    whoever took it, and two evaluations must agree bit for bit (the result of a target does not depend on which CTA
    computed it, nor on the order).  Parity against the oracle at this size: the sampled-target tests."""
    import torch
    L, N = 4096, 96
    ctx = D.dmfe_create(L, s, 1e4, [0, 0, 0.6, 1.0], T=0.5, values_only=values_only)
    try:
        tab = D.dmfe_get_tables(ctx, L)
        t, mu, hist = inputs.random_smooth_history(tab["theta"], tab["omega"], N, 300.0, seed=5)
        if values_only:
            hist = np.ascontiguousarray(hist[:, :, [0, 2]])
        runs = []
        for _ in range(2):
            g = gpu_rhs(D, ctx, L, t, mu, hist, N, want_rows=False)
            runs.append(g)
        for k, v in runs[0].items():
            assert np.all(np.isfinite(v)), "%s: a target was not computed" % k
            assert np.array_equal(v, runs[1][k]), "%s differs between two evaluations" % k
    finally:
        D.dmfe_destroy(ctx)
