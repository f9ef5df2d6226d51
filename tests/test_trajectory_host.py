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
