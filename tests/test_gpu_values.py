"""GPU parity of the values-only history mode (dmfe_params.values_only): libdmfe.so through its
C ABI against the oracle's orc_history_integrals_values on identical seeded inputs and the library's tables.
Window starts (integers) bit-exact; sums within 1e-12 * sum |term|; combined derivatives within 1e-12 of their scale."""
import numpy as np
import pytest

from oracle import dmfe_oracle as O
from paper_2604_06309_b200 import inputs

pytestmark = pytest.mark.gpu
RTOL = 1e-12


@pytest.fixture(scope="module")
def D():
    from paper_2604_06309_b200 import dmfe
    dmfe.load_library()
    return dmfe


def _gpu(D, ctx, L, t, mu, histv, n_rows, want_rows=True):
    import torch
    dev = "cuda"
    tt, tm, th = (torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in (t, mu, histv))
    z = lambda *shape: torch.full(shape, float("nan"), dtype=torch.float64, device=dev)
    out = dict(d1C=z(L), d1R=z(L), mu_out=z(1), d2C=z(L), d2R=z(L), F=z(L, 2), energy=z(1), sums=z(8, L))
    if want_rows:
        out["rows1"] = torch.full((L,), -1, dtype=torch.int32, device=dev)
        out["rows2"] = torch.full((L, L), -1, dtype=torch.int32, device=dev)
    D.dmfe_history_integrals(ctx, n_rows, tt, tm, th, **out)
    torch.cuda.synchronize()
    return {k: v.cpu().numpy() for k, v in out.items()}


def _compare(g, ref, targets=None):
    sel = slice(None) if targets is None else targets
    if "rows1" in g and "rows1" in ref:
        assert np.array_equal(g["rows1"][sel], ref["rows1"]) and np.array_equal(g["rows2"][sel], ref["rows2"])
    err = np.abs(g["sums"].T[sel] - ref["sums"])
    worst = np.max(err / (RTOL * ref["abssums"] + 1e-300))
    assert worst <= 1.0, "sums off by %.3g x tolerance" % worst
    assert abs(g["mu_out"][0] - ref["mu"]) <= RTOL * abs(ref["mu"])
    assert abs(g["energy"][0] - ref["E"]) <= RTOL * max(abs(ref["E"]), 1e-300)
    for k, name in enumerate(["d1C", "d1R", "d2C", "d2R"]):
        e = np.abs(g[name][sel] - ref["deriv"][:, k])
        assert np.max(e / (RTOL * ref["scale"][:, k] + 1e-300)) <= 1.0, name


CASES = [
    # L, N, s, lam, T, beta0, t_max, t_end
    (96, 37, 4, [0, 0, 0, 1.0], 1.0, 0.0, 50.0, 30.0),
    (100, 23, 6, [0, 0, 1.0, 0, 0.5], 0.5, 0.0, 1e3, 200.0),
    (130, 41, 10, [0, 0, 1.0, 0.8, 0.5], 0.7, 0.0, 1e2, 60.0),
    (64, 9, 4, [0, 0, 0, 0.5, 0, 0, 0, 0, 0, 0.5], 0.3, 1.5, 40.0, 7.0),   # 3+9 model, beta0 > 0
    (333, 120, 2, [0, 0, 2.0], 0.0, 0.0, 1e4, 90.0),                       # ragged L, s = 2
    (48, 2, 4, [0, 0, 0, 1.0], 1.0, 0.0, 10.0, 0.01),                      # two rows: linear in t
    (48, 3, 8, [0, 0, 0, 1.0], 1.0, 0.0, 10.0, 0.02),                      # three rows: quadratic in t
    (48, 4, 4, [0, 0, 0, 1.0], 1.0, 0.0, 10.0, 0.05),                      # exactly one window
]


@pytest.mark.parametrize("L,N,s,lam,T,beta0,t_max,t_end", CASES)
def test_values_rhs_matches_oracle_small(D, L, N, s, lam, T, beta0, t_max, t_end):
    ctx = D.dmfe_create(L, s, t_max, lam, T=T, beta0=beta0, values_only=True)
    try:
        tab = D.dmfe_get_tables(ctx, L)
        grid = O.Grid(L=L, s=s, t_max=t_max, theta=tab["theta"], omega=tab["omega"], nu=tab["nu"])
        t, mu, hist = inputs.random_smooth_history(tab["theta"], tab["omega"], N, t_end, seed=L + N)
        histv = np.ascontiguousarray(hist[:, :, [0, 2]])
        mu[N - 1] = np.nan                                  # mu of the current row must be ignored
        g = _gpu(D, ctx, L, t, mu, histv, N)
    finally:
        D.dmfe_destroy(ctx)
    model = O.Model(np.array(lam, dtype=np.float64), T, beta0)
    ref = O.history_integrals_values(grid, model, t, mu, histv, N - 1, tables=(tab["start"], tab["frac"]),
                                     want_rows=True)
    _compare(g, ref)


def test_values_rhs_synthetic_all_targets(D):
    """Config-2 recipe at L = N = 512, all targets."""
    L, s, t_max, lam = 512, 4, 1e4, [0, 0, 0, 1.0]
    ctx = D.dmfe_create(L, s, t_max, lam, T=0.5, values_only=True)
    try:
        tab = D.dmfe_get_tables(ctx, L)
        grid = O.Grid(L=L, s=s, t_max=t_max, theta=tab["theta"], omega=tab["omega"], nu=tab["nu"])
        t, mu, hist = inputs.synthetic_history(tab["theta"], tab["omega"], L, -2.0, 4.0)
        histv = np.ascontiguousarray(hist[:, :, [0, 2]])
        g = _gpu(D, ctx, L, t, mu, histv, L)
    finally:
        D.dmfe_destroy(ctx)
    ref = O.history_integrals_values(grid, O.Model(np.array(lam, dtype=np.float64), 0.5, 0.0), t, mu, histv, L - 1,
                                     tables=(tab["start"], tab["frac"]), want_rows=True)
    _compare(g, ref)


@pytest.mark.parametrize("L,lo,hi,t_max,lam,nblocks", [
    (4096, -2.0, 4.0, 1e4, [0, 0, 0, 1.0], 6),                      # config 2 at full size (bench shape)
    (10240, -2.0, 7.0, 1e7, [0, 0, 1.0, 0.8, 0.5], 4),              # per-call tables in global memory
])
def test_values_rhs_full_size_sampled_targets(D, L, lo, hi, t_max, lam, nblocks):
    s = 4
    ctx = D.dmfe_create(L, s, t_max, lam, T=0.5, values_only=True)
    try:
        tab = D.dmfe_get_tables(ctx, L, want_pairs=False)
        t, mu, hist = inputs.synthetic_history(tab["theta"], tab["omega"], L, lo, hi)
        histv = np.ascontiguousarray(hist[:, :, [0, 2]])
        del hist
        g = _gpu(D, ctx, L, t, mu, histv, L, want_rows=False)
        rng = np.random.Generator(np.random.PCG64(L))
        blocks = np.unique(np.concatenate([[0], np.sort(rng.choice(L // 32, size=nblocks, replace=False)) * 32, [L - 32]]))
        grid = O.Grid(L=L, s=s, t_max=t_max, theta=tab["theta"], omega=tab["omega"], nu=tab["nu"])
        model = O.Model(np.array(lam, dtype=np.float64), 0.5, 0.0)
        for i0 in blocks:
            part = D.dmfe_get_tables(ctx, L, i0=int(i0), n_targets=32)
            targets = np.arange(i0, i0 + 32, dtype=np.int32)
            ref = O.history_integrals_values(grid, model, t, mu, histv, L - 1, targets=targets,
                                             tables=(part["start"], part["frac"]))
            _compare(g, ref, targets)
    finally:
        D.dmfe_destroy(ctx)


def test_values_mode_has_no_integrator(D):
    ctx = D.dmfe_create(64, 4, 100.0, [0, 0, 0, 1.0], T=1.0, values_only=True)
    try:
        st, ten = D.make_state(64, 16)
        with pytest.raises(D.DmfeError) as ei:
            D.dmfe_init_state(ctx, st, 1e-3)
        assert ei.value.code == D.DMFE_EINVAL
    finally:
        D.dmfe_destroy(ctx)
