"""Host-side pieces of the trajectory driver that need no GPU."""
import numpy as np

from paper_2604_06309_b200 import trajectory


def test_observe_interpolates_in_theta():
    theta = np.linspace(0.0, 1.0, 11)
    row = np.zeros((11, 4))
    row[:, 0] = 2.0 * theta          # C(t, theta t) = 2 theta
    row[:, 2] = 1.0 - theta          # R
    obs = trajectory.observe(theta, 10.0, row, (1.0, 2.5, 20.0))
    assert set(obs) == {1.0, 2.5}                      # t_w > t is skipped
    assert abs(obs[2.5][0] - 0.5) < 1e-15 and abs(obs[2.5][1] - 0.75) < 1e-15


def test_configs_follow_baseline():
    c3, c4 = trajectory.CONFIGS[3], trajectory.CONFIGS[4]
    assert c3["lam"] == [0.0, 0.0, 1.0, 0.0, 0.5] and c3["T"] == 0.5 and c3["n_cap"] == 2048 and c3["tol"] == 1e-8
    assert c4["lam"] == [0.0, 0.0, 0.0, 1.0] and c4["T"] == 0.5 and c4["n_cap"] == 8192 and c4["t_max"] == 1e7


def test_bench_algorithmic_bytes_hull_estimate_matches_exact_count():
    """bench.py counts the distinct history cells one evaluation touches (the roofline's algorithmic
    bytes) exactly up to L = 8192 and from the per-row hull of a strided target sample above; on a
    size where both run the two agree to a fraction of a percent and the estimate never exceeds
    the full array."""
    import bench
    from oracle import dmfe_oracle as O
    from paper_2604_06309_b200 import inputs
    L = N = 384
    g = O.Grid(L=L, s=4, t_max=1e7)
    t = inputs.log_times(N, -2.0, 7.0)
    exact = bench.unique_cells(g.theta, g.omega, t, 4, L, N)
    samp = np.unique(np.append(np.arange(0, L, 8), L - 1))
    est = bench.unique_cells(g.theta, g.omega, t, 4, L, N, sample=samp)
    assert 0 < exact <= N * L and 0 < est <= N * L
    assert abs(est - exact) <= 0.01 * exact
    # brute force on a tiny case: every (i, j) pair, cell by cell
    L = N = 24
    g = O.Grid(L=L, s=4, t_max=1e3)
    t = inputs.log_times(N, -2.0, 3.0)
    M = N - 1
    cells = set()
    for i in range(L):
        n1 = max(0, min(M - 1, int(np.searchsorted(t[:M], g.theta[i] * t[M], side="right")) - 1))
        for j in range(L):
            cells.add((n1, j)), cells.add((n1 + 1, j))
            phi2 = g.theta[i] + g.omega[i] * g.theta[j]
            n2 = max(0, min(M - 1, int(np.searchsorted(t[:M], phi2 * t[M], side="right")) - 1))
            psi = g.theta[i] / phi2 if phi2 > 0 else 0.0
            a3 = max(0, min(L - 4, int(np.searchsorted(g.theta, psi, side="right")) - 1 - 1))
            for l in range(4):
                cells.add((n2, a3 + l)), cells.add((n2 + 1, a3 + l))
    assert bench.unique_cells(g.theta, g.omega, t, 4, L, N) == len(cells)
