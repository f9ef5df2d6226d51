"""Seeded synthetic inputs shared by the CUDA path's tests/bench and the CPU oracle.

This module holds none of the method's arithmetic: it only fills history arrays with the
synthetic two-time fields that BASELINE.json's configs 2 and 5 prescribe, on a theta-grid that
the caller supplies (from the library or from the oracle).  Recipe:

  rows      t_0 = 0, t_n = 10^(lo + (hi-lo)(n-1)/(N-2)), n = 1..N-1   (log-spaced on [10^lo,10^hi])
  C(t,t')   = exp(-(t-t')/tau(t')), tau(t') = 1 + t'^0.8
  R(t,t')   = C(t,t') / (1 + t'^0.1)
  stored    C[n][l] = C(t_n, theta_l t_n), R likewise, and the analytic derivatives along the
            ray (d/dt at fixed theta); row 0: C = R = 1, slopes -(1-theta)
  mu_n      = 1 + 1/(1+t_n)
  jitter    every entry of the four arrays times (1 + 1e-6 xi), xi ~ U(-1,1) from
            numpy PCG64(seed + k), k = 0..3 for (C, dC, R, dR), drawn row-major
"""
from __future__ import annotations

import numpy as np

DEFAULT_SEED = 20260406


def log_times(N: int, lo: float, hi: float) -> np.ndarray:
    t = np.zeros(N, dtype=np.float64)
    n = np.arange(1, N, dtype=np.float64)
    t[1:] = 10.0 ** (lo + (hi - lo) * (n - 1.0) / (N - 2.0))
    return t


def synthetic_history(theta: np.ndarray, omega: np.ndarray, N: int, lo: float, hi: float,
                      seed: int = DEFAULT_SEED, jitter: float = 1e-6):
    """Returns (t[N], mu[N], hist[N, L, 4]) with hist[..., :] = {C, dC, R, dR}."""
    L = len(theta)
    t = log_times(N, lo, hi)
    mu = 1.0 + 1.0 / (1.0 + t)
    hist = np.empty((N, L, 4), dtype=np.float64)
    rngs = [np.random.Generator(np.random.PCG64(seed + k)) for k in range(4)]
    # row blocks bound the temporaries (nine N x L arrays otherwise: 77 GB at L = N = 32768); the
    # jitter streams are consumed row-major, so the blocking does not change which number goes where
    blk = N if N * L <= (1 << 27) else max(1, (1 << 27) // L)
    for r0 in range(0, N, blk):
        r1 = min(N, r0 + blk)
        tn = t[r0:r1, None]
        th = theta[None, :]
        om = omega[None, :]
        x = th * tn                       # t' = theta t
        tau = 1.0 + x ** 0.8
        g = tn * om / tau                 # (t - t')/tau(t')
        C = np.exp(-g)
        x01 = x ** 0.1
        R = C / (1.0 + x01)
        gp = (om / tau) * (1.0 - 0.8 * x ** 0.8 / tau)
        dC = -gp * C
        with np.errstate(divide="ignore", invalid="ignore"):
            dR = -gp * R - C * 0.1 * x01 / (tn * (1.0 + x01) ** 2)
        if r0 == 0:
            C[0], R[0] = 1.0, 1.0
            dC[0], dR[0] = -omega, -omega
        for k, arr in enumerate((C, dC, R, dR)):
            xi = rngs[k].uniform(-1.0, 1.0, size=(r1 - r0, L))
            hist[r0:r1, :, k] = arr * (1.0 + jitter * xi)
    return t, mu, hist


def random_smooth_history(theta, omega, N: int, t_end: float, seed: int = 1):
    """Small generic case for parity tests: uneven (seeded) time steps, smooth positive fields
    built from a few seeded exponentials; same packed layout as synthetic_history."""
    rng = np.random.Generator(np.random.PCG64(seed))
    L = len(theta)
    steps = rng.uniform(0.5, 1.5, size=N - 1)
    t = np.concatenate([[0.0], np.cumsum(steps)])
    t *= t_end / t[-1]
    a = rng.uniform(0.2, 2.0, size=3)
    w = rng.uniform(0.1, 1.0, size=3)
    w /= w.sum()
    tn, th, om = t[:, None], theta[None, :], omega[None, :]
    hist = np.zeros((N, L, 4))
    for ak, wk in zip(a, w):
        e = np.exp(-ak * tn * om)
        hist[:, :, 0] += wk * e
        hist[:, :, 1] += wk * (-ak * om) * e
        hist[:, :, 2] += wk * e * (0.5 + 0.5 * th)
        hist[:, :, 3] += wk * (-ak * om) * e * (0.5 + 0.5 * th)
    hist *= 1.0 + 1e-3 * rng.uniform(-1, 1, size=hist.shape)
    mu = 1.0 + 0.5 * np.exp(-t) + 1e-3 * rng.uniform(-1, 1, size=N)
    return t, mu, hist
