"""dmfe_history_integrals_static (include/dmfe.h): the north-star call with its per-call tables in the library's
file-scope device array, for callers that may not allocate.  Checked against the existing path
dmfe_history_integrals on the same inputs, on calls in a row that share the array (different histories, different
contexts, different pair kernels), at the tolerance of tests/test_gpu_parity.py (integer results bit-exact, floating
point within 1e-12 of its scale; the two paths run the same kernels, so in practice they agree bit for bit).

Named test_zz_* so that pytest collects it last: the suite runs with `pytest -x`.
"""
import numpy as np
import pytest

from paper_2604_06309_b200 import inputs

pytestmark = pytest.mark.gpu

RTOL = 1e-12


@pytest.fixture(scope="module")
def D():
    from paper_2604_06309_b200 import dmfe
    dmfe.load_library()  # fails loudly if the CUDA library is missing
    return dmfe


def _run(D, call, ctx, L, t, mu, hist, n_rows):
    import torch
    dev = "cuda"
    tt = torch.from_numpy(np.ascontiguousarray(t)).to(dev)
    tm = torch.from_numpy(np.ascontiguousarray(mu)).to(dev)
    th = torch.from_numpy(np.ascontiguousarray(hist)).to(dev)
    z = lambda *shape: torch.full(shape, float("nan"), dtype=torch.float64, device=dev)
    out = dict(d1C=z(L), d1R=z(L), mu_out=z(1), d2C=z(L), d2R=z(L), F=z(L, 2), energy=z(1), sums=z(8, L),
               rows1=torch.full((L,), -1, dtype=torch.int32, device=dev),
               rows2=torch.full((L, L), -1, dtype=torch.int32, device=dev))
    call(ctx, n_rows, tt, tm, th, **out)
    torch.cuda.synchronize()
    return {k: v.cpu().numpy() for k, v in out.items()}


def _same(a, b):
    for k in ("rows1", "rows2"):
        assert np.array_equal(a[k], b[k]), k
    for k in ("sums", "d1C", "d1R", "d2C", "d2R", "F", "mu_out", "energy"):
        assert np.all(np.isfinite(a[k])) and np.all(np.isfinite(b[k])), k
        scale = np.max(np.abs(b[k]))
        assert np.max(np.abs(a[k] - b[k])) <= RTOL * scale, "%s differs by %.3g of its scale" % (
            k, np.max(np.abs(a[k] - b[k])) / scale)


def test_static_limits(D):
    max_L, max_rows, nbytes = D.dmfe_static_limits()
    assert (max_L, max_rows) == (D.DMFE_STATIC_MAX_L, D.DMFE_STATIC_MAX_ROWS) == (4096, 16384)
    assert 0 < nbytes <= 2 * 1024 * 1024 and nbytes % 256 == 0
    assert D.load_library().dmfe_strerror(D.DMFE_ETOOLARGE).startswith(b"size beyond the static scratch")


def test_static_entry_point_matches_the_existing_path_on_calls_in_a_row(D):
    # (L, stencil, lam, T, t_max, [(N, t_end, seed), ...]): the 4-point kernel, the generic kernel, a run-time degree
    # of f; every call below shares the one static array, so each call sees the previous call's contents in it
    cases = [
        (160, 4, [0, 0, 0, 1.0], 1.0, 50.0, [(37, 30.0, 3), (61, 45.0, 4), (5, 0.3, 5)]),
        (130, 6, [0, 0, 1.0, 0, 0.5], 0.5, 1e3, [(23, 200.0, 6), (41, 700.0, 7)]),
        (333, 4, [0, 0, 0, 0.5, 0, 0, 0, 0, 0, 0.5], 0.3, 1e4, [(97, 5e3, 8), (97, 5e3, 8)]),
    ]
    ctxs = []
    try:
        for (L, s, lam, T, t_max, _) in cases:
            ctxs.append(D.dmfe_create(L, s, t_max, lam, T=T))
        D.dmfe_static_init(ctxs[0])
        # interleave the contexts: A1 B1 C1 A2 B2 C2 A3
        order = [(ci, hi) for hi in range(3) for ci in range(len(cases)) if hi < len(cases[ci][5])]
        assert len(order) >= 2
        for ci, hi in order:
            L, s, lam, T, t_max, hs = cases[ci]
            N, t_end, seed = hs[hi]
            tab = D.dmfe_get_tables(ctxs[ci], L)
            t, mu, hist = inputs.random_smooth_history(tab["theta"], tab["omega"], N, t_end, seed=seed)
            new = _run(D, D.dmfe_history_integrals_static, ctxs[ci], L, t, mu, hist, N)
            old = _run(D, D.dmfe_history_integrals, ctxs[ci], L, t, mu, hist, N)
            _same(new, old)
            again = _run(D, D.dmfe_history_integrals_static, ctxs[ci], L, t, mu, hist, N)  # after the ordinary path
            _same(again, old)
    finally:
        for c in ctxs:
            D.dmfe_destroy(c)


def test_static_entry_point_rejects_what_does_not_fit(D):
    import torch
    L = 24
    ctx = D.dmfe_create(L, 4, 100.0, [0, 0, 0, 1.0], T=1.0)
    ctx_v = D.dmfe_create(L, 4, 100.0, [0, 0, 0, 1.0], T=1.0, values_only=True)
    try:
        n = D.DMFE_STATIC_MAX_ROWS + 2  # M = n - 1 = max + 1
        t = torch.linspace(0.0, 50.0, n, dtype=torch.float64, device="cuda")
        mu = torch.ones(n, dtype=torch.float64, device="cuda")
        hist = torch.zeros((n, L, 4), dtype=torch.float64, device="cuda")
        hist[:, :, 0] = 1.0
        d1C = torch.full((L,), float("nan"), dtype=torch.float64, device="cuda")
        with pytest.raises(D.DmfeError) as ei:
            D.dmfe_history_integrals_static(ctx, n, t, mu, hist, d1C=d1C)
        assert ei.value.code == D.DMFE_ETOOLARGE
        torch.cuda.synchronize()
        assert torch.isnan(d1C).all()  # nothing was launched
        # the largest history that fits is accepted and equals the ordinary path
        d1C_old = torch.empty_like(d1C)
        D.dmfe_history_integrals_static(ctx, n - 1, t, mu, hist, d1C=d1C)
        D.dmfe_history_integrals(ctx, n - 1, t, mu, hist, d1C=d1C_old)
        torch.cuda.synchronize()
        a, b = d1C.cpu().numpy(), d1C_old.cpu().numpy()
        assert np.all(np.isfinite(a)) and np.max(np.abs(a - b)) <= RTOL * np.max(np.abs(b))
        hv = torch.ones((8, L, 2), dtype=torch.float64, device="cuda")
        with pytest.raises(D.DmfeError) as ei:
            D.dmfe_history_integrals_static(ctx_v, 8, t[:8].contiguous(), mu[:8].contiguous(), hv, d1C=d1C)
        assert ei.value.code == D.DMFE_EINVAL
    finally:
        D.dmfe_destroy(ctx)
        D.dmfe_destroy(ctx_v)
