"""CPU oracle for the DMFE history-integral path -- TEST INFRASTRUCTURE ONLY.

Plain numpy / C (dmfe_oracle.c) restatement of the method of arxiv/paper_2604_06309
(section 3), independent of the CUDA library: nothing here imports the
product package and nothing in the product imports this.  Only tests/,
__graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs use it.

Pins (tests/test_oracle_*.py, all `-m "not gpu"`): P1 polynomial reproduction,
P2 quadrature exactness, P3 grid identities + mpmath cross-check, P4 constant-history
closed form, P5 pure 2-spin closed form, P6 C(t,t)=1 / R(t,t-)=1, P7 paramagnet + FDT,
P8 uniform-grid brute force, P9 RK order conditions, P10 the numbers printed in Fig. 7
(tests/test_oracle_golden.py), P11-P14 Dormand-Prince start-up (tests/test_oracle_dp.py), P15 the beta0 forcing
path (equilibrium start beta0 = 1/T is stationary from the first step: mu, E, time-translation invariance, FDT),
orc_mu_at (cubic reproduction, window placement), the controller constants of PAPER.md:320 on a stubbed error
sequence, the greedy thinning walk (brute force over flag patterns) and the step loop `integrate` (tests/test_oracle_traj.py),
V1-V4 the values-only history (tests/test_oracle_values.py), LR1-LR4 the log-R option (tests/test_oracle_logr.py).
"parity unpinned": controller tie-breaks and the sparsification schedule (paper silent; readings G20,
G25, G31 in DESIGN.md).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liboracle_dmfe.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile dmfe_oracle.c (gcc, no FMA contraction, OpenMP over targets)."""
    src = os.path.join(_HERE, "dmfe_oracle.c")
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(src):
        subprocess.check_call(
            ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-std=c11",
             "-o", _SO, src, "-lm"])
    return _SO


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_SO)
        _lib.orc_f.restype = ctypes.c_double
        _lib.orc_f.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_int]
        _lib.orc_row_search.restype = ctypes.c_int
        _lib.orc_row_search.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_double]
        _lib.orc_mu_at.restype = ctypes.c_double
        _lib.orc_mu_at.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int, ctypes.c_double]
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


# --------------------------------------------------------------------------- model
@dataclass
class Model:
    """f(q) = 1/2 sum_p lam[p] q^p (Eq.(4), reading G2), bath temperature T,
    beta0 = inverse temperature of the initial condition (Eq.(12))."""
    lam: np.ndarray
    T: float
    beta0: float = 0.0

    def __post_init__(self):
        self.lam = np.ascontiguousarray(self.lam, dtype=np.float64)

    @property
    def pmax(self):
        return len(self.lam) - 1

    def f(self, q, order=0):
        return _load().orc_f(_p(self.lam), self.pmax, float(q), order)


# --------------------------------------------------------------------------- tables
def gamma_of_tmax(t_max: float) -> float:
    """gamma = -W_{-1}(-1/t_max)."""
    from scipy.special import lambertw
    return float(-lambertw(-1.0 / t_max, k=-1).real)


def theta_grid(L: int, t_max: float):
    """theta-grid of Eq.(16) for alpha=0, in the cancellation-free form
    theta_i = [atan(e^{gamma y_i}) - atan(e^{-gamma})] / (A - B)  (reading G7), lower half by
    atan a - atan b = atan((a-b)/(1+ab)), upper half by the symmetry theta_{L+1-i} = 1-theta_i.
    Returns (theta, omega) with omega_i = theta_{L+1-i} the accurate complement 1-theta_i."""
    g = gamma_of_tmax(t_max)
    A, B = np.arctan(np.exp(g)), np.arctan(np.exp(-g))
    i = np.arange(1, L + 1, dtype=np.float64)
    y = (2.0 * i - 1.0 - L) / (L - 1.0)
    theta = np.empty(L)
    half = (L + 1) // 2
    yl = y[:half]
    theta[:half] = np.arctan(np.exp(-g) * np.expm1(g * (1.0 + yl)) / (1.0 + np.exp(g * yl - g))) / (A - B)
    upper = np.arange(half, L)
    theta[upper] = 1.0 - theta[L - 1 - upper]
    theta[0], theta[-1] = 0.0, 1.0
    omega = theta[::-1].copy()
    return theta, omega


def quad_weights(theta: np.ndarray, degree: int = 5) -> np.ndarray:
    """nu_j = integral over [0,1] of the j-th cardinal function of the global interpolating
    spline (not-a-knot, degree 5 by default) with knots on the theta-grid (G18)."""
    from scipy.interpolate import make_interp_spline
    L = len(theta)
    spl = make_interp_spline(theta, np.eye(L), k=degree)
    return np.asarray(spl.integrate(0.0, 1.0), dtype=np.float64)


def index_coordinate(c, cbar, L: int, t_max: float):
    """0-based real index coordinate X(c) of a point c in [0,1] from the analytic inverse of the
    grid ("theta(i) is known analytically"); cbar = 1-c supplied without
    cancellation and used for c > 1/2 (reading G17)."""
    g = gamma_of_tmax(t_max)
    A, B = np.arctan(np.exp(g)), np.arctan(np.exp(-g))
    c = np.asarray(c, dtype=np.float64)
    cbar = np.asarray(cbar, dtype=np.float64)
    lower = c <= 0.5
    arg = np.where(lower, c, cbar)
    with np.errstate(divide="ignore"):
        y = np.log(np.tan(B + arg * (A - B))) / g
    y = np.where(lower, y, -y)
    return (L - 1.0) * (1.0 + y) / 2.0


def pair_coordinates(theta, omega, targets):
    """(phi1, phi2, psi) and their complements for pairs (i in targets, all j)  (PAPER.md:245,
    :264): phi1 = theta_i theta_j; phi2 = theta_i + omega_i theta_j; psi = theta_i / phi2."""
    th_i = theta[targets][:, None]
    om_i = omega[targets][:, None]
    th_j, om_j = theta[None, :], omega[None, :]
    phi1 = th_i * th_j
    phi2 = th_i + om_i * th_j
    with np.errstate(invalid="ignore", divide="ignore"):
        psi = np.where(phi2 > 0.0, th_i / phi2, 0.0)
        psibar = np.where(phi2 > 0.0, om_i * th_j / phi2, 1.0)
    phi1bar = om_i + th_i * om_j
    phi2bar = om_i * om_j
    return (phi1, phi2, psi), (phi1bar, phi2bar, psibar)


def stencil_start(theta, c, s: int):
    """l* = max{l : theta_l <= c} by comparison on the stored grid; start = clamp(l* - (s/2-1),
    0, L-s)  (0-based; reading G16)."""
    L = len(theta)
    lstar = np.searchsorted(theta, c, side="right") - 1
    return np.clip(lstar - (s // 2 - 1), 0, L - s).astype(np.int32)


def pair_tables(theta, omega, t_max: float, s: int, targets):
    """start[3][nt][L] (int32) and frac[3][nt][L] (u = X - start) for phi1, phi2, psi."""
    L = len(theta)
    targets = np.asarray(targets, dtype=np.int64)
    cs, cbars = pair_coordinates(theta, omega, targets)
    start = np.empty((3, len(targets), L), dtype=np.int32)
    frac = np.empty((3, len(targets), L), dtype=np.float64)
    for k in range(3):
        start[k] = stencil_start(theta, cs[k], s)
        frac[k] = index_coordinate(cs[k], cbars[k], L, t_max) - start[k]
    return start, frac


@dataclass
class Grid:
    L: int
    s: int
    t_max: float
    quad_degree: int = 5
    theta: np.ndarray = field(default=None, repr=False)
    omega: np.ndarray = field(default=None, repr=False)
    nu: np.ndarray = field(default=None, repr=False)

    def __post_init__(self):
        if self.theta is None:
            self.theta, self.omega = theta_grid(self.L, self.t_max)
        if self.nu is None:
            self.nu = quad_weights(self.theta, self.quad_degree)
        self._tables = None

    def tables(self, targets=None):
        if targets is None:
            if self._tables is None:
                self._tables = pair_tables(self.theta, self.omega, self.t_max, self.s, np.arange(self.L))
            return self._tables
        return pair_tables(self.theta, self.omega, self.t_max, self.s, targets)


# --------------------------------------------------------------------------- history integrals
def history_integrals(grid: Grid, model: Model, t, mu_hist, hist, M: int, targets=None,
                      tables=None, want_rows=False, log_r=False):
    """The per-stage right-hand side: Eq.(17)-(21), Eq.(13), Eq.(14), Eq.(1).

    t[0..M], mu_hist[0..M-1], hist[(M+1), L, 4] = {C, dC, R, dR}; row M values only.
    Returns dict with sums[nt,8], abssums[nt,8], deriv[nt,6] (d1C,d1R,d2C,d2R,FC,FR),
    scale[nt,4], mu, E and (optionally) rows1[nt], rows2[nt,L]."""
    lib = _load()
    L, s = grid.L, grid.s
    if targets is None:
        targets = np.arange(L)
    targets = np.ascontiguousarray(targets, dtype=np.int32)
    nt = len(targets)
    if tables is None:
        tables = grid.tables(None if nt == L and np.array_equal(targets, np.arange(L)) else targets)
    start = np.ascontiguousarray(tables[0], dtype=np.int32)
    frac = np.ascontiguousarray(tables[1], dtype=np.float64)
    assert start.shape == (3, nt, L) and frac.shape == (3, nt, L)
    t = np.ascontiguousarray(t, dtype=np.float64)
    mu_hist = np.ascontiguousarray(mu_hist, dtype=np.float64)
    hist = np.ascontiguousarray(hist, dtype=np.float64)
    assert hist.ndim == 3 and hist.shape[1] == L and hist.shape[2] == 4 and hist.shape[0] >= M + 1
    assert M >= 1 and len(t) >= M + 1 and len(mu_hist) >= M
    sums = np.zeros((nt, 8)); abssums = np.zeros((nt, 8))
    deriv = np.zeros((nt, 6)); scale = np.zeros((nt, 4))
    rows1 = np.zeros(nt, dtype=np.int32) if want_rows else None
    rows2 = np.zeros((nt, L), dtype=np.int32) if want_rows else None
    mu = ctypes.c_double(0.0); E = ctypes.c_double(0.0)
    # log_r: logarithmic interpolation of the response history (reading G32)
    (lib.orc_history_integrals_logr if log_r else lib.orc_history_integrals)(
        ctypes.c_int(L), ctypes.c_int(s), ctypes.c_int(M), _p(model.lam), ctypes.c_int(model.pmax),
        ctypes.c_double(model.T), ctypes.c_double(model.beta0), _p(grid.theta), _p(grid.omega),
        _p(grid.nu), _p(t), _p(mu_hist), _p(hist), ctypes.c_int(nt), _p(targets), _p(start),
        _p(frac), _p(sums), _p(abssums), _p(deriv), _p(scale), _p(rows1), _p(rows2),
        ctypes.byref(mu), ctypes.byref(E))
    out = dict(sums=sums, abssums=abssums, deriv=deriv, scale=scale, mu=mu.value, E=E.value)
    if want_rows:
        out["rows1"], out["rows2"] = rows1, rows2
    return out


def history_integrals_values(grid: Grid, model: Model, t, mu_hist, histv, M: int, targets=None, tables=None,
                             want_rows=False):
    """The same right-hand side on a VALUES-ONLY history: histv[(M+1), L, 2] =
    {C, R}; interpolation in t = local 4-point Lagrange through rows k..k+3, k = clamp(n(tau)-1, 0, M-3).
    rows1 / rows2 are the window starts k.  Same return dict as history_integrals."""
    lib = _load()
    L, s = grid.L, grid.s
    if targets is None:
        targets = np.arange(L)
    targets = np.ascontiguousarray(targets, dtype=np.int32)
    nt = len(targets)
    if tables is None:
        tables = grid.tables(None if nt == L and np.array_equal(targets, np.arange(L)) else targets)
    start = np.ascontiguousarray(tables[0], dtype=np.int32)
    frac = np.ascontiguousarray(tables[1], dtype=np.float64)
    t = np.ascontiguousarray(t, dtype=np.float64)
    mu_hist = np.ascontiguousarray(mu_hist, dtype=np.float64)
    histv = np.ascontiguousarray(histv, dtype=np.float64)
    assert histv.ndim == 3 and histv.shape[1] == L and histv.shape[2] == 2 and histv.shape[0] >= M + 1
    assert M >= 1 and len(t) >= M + 1 and len(mu_hist) >= M
    sums = np.zeros((nt, 8)); abssums = np.zeros((nt, 8))
    deriv = np.zeros((nt, 6)); scale = np.zeros((nt, 4))
    rows1 = np.zeros(nt, dtype=np.int32) if want_rows else None
    rows2 = np.zeros((nt, L), dtype=np.int32) if want_rows else None
    mu = ctypes.c_double(0.0); E = ctypes.c_double(0.0)
    lib.orc_history_integrals_values(
        ctypes.c_int(L), ctypes.c_int(s), ctypes.c_int(M), _p(model.lam), ctypes.c_int(model.pmax),
        ctypes.c_double(model.T), ctypes.c_double(model.beta0), _p(grid.theta), _p(grid.omega),
        _p(grid.nu), _p(t), _p(mu_hist), _p(histv), ctypes.c_int(nt), _p(targets), _p(start),
        _p(frac), _p(sums), _p(abssums), _p(deriv), _p(scale), _p(rows1), _p(rows2),
        ctypes.byref(mu), ctypes.byref(E))
    out = dict(sums=sums, abssums=abssums, deriv=deriv, scale=scale, mu=mu.value, E=E.value)
    if want_rows:
        out["rows1"], out["rows2"] = rows1, rows2
    return out


def sparsify_residuals(L: int, N: int, t, hist):
    """eps_sparse[n] of Eq.(27) for every interior row."""
    lib = _load()
    t = np.ascontiguousarray(t, dtype=np.float64)
    hist = np.ascontiguousarray(hist, dtype=np.float64)
    eps = np.zeros(N)
    lib.orc_sparsify_residuals(ctypes.c_int(L), ctypes.c_int(N), _p(t), _p(hist), _p(eps))
    return eps


# --------------------------------------------------------------------------- time stepping
# SSPRK(10,4) (refs [64,65] PAPER.md:540-542) in Ketcheson's low-storage form.
SSPRK_C = np.array([0, 1, 2, 3, 4, 2, 3, 4, 5, 6], dtype=np.float64) / 6.0
SSPRK_B = np.full(10, 0.1)
SSPRK_BHAT = np.array([0, 2 / 9, 0, 0, 5 / 18, 1 / 3, 0, 0, 0, 1 / 6], dtype=np.float64)  # G22
STAB_REAL_AXIS = 13.9  # real-axis stability limit used for the step cap (Eq.24, reading G20)


def ssprk104_butcher():
    """Butcher matrix A of SSPRK(10,4) (used only by the order-condition pin P9)."""
    A = np.zeros((10, 10))
    for i in range(10):
        for j in range(i):
            if i <= 4:
                A[i, j] = 1 / 6
            else:
                A[i, j] = 1 / 15 if j <= 4 else 1 / 6
    return A


class History:
    """t[], mu[], E[], packed rows {C,dC,R,dR}; rows 0..n_rows-1 valid and complete."""

    def __init__(self, grid: Grid, model: Model, n_cap: int):
        L = grid.L
        self.grid, self.model, self.n_cap = grid, model, n_cap
        self.t = np.zeros(n_cap)
        self.mu = np.zeros(n_cap)
        self.E = np.zeros(n_cap)
        self.hist = np.zeros((n_cap, L, 4))
        # row 0 at t=0 (reading G13): C=R=1, ray slopes -T(1-theta), -mu0(1-theta)
        mu0 = model.T + model.beta0 * model.f(1.0, 1)
        self.hist[0, :, 0] = 1.0
        self.hist[0, :, 2] = 1.0
        self.hist[0, :, 1] = -model.T * grid.omega
        self.hist[0, :, 3] = -mu0 * grid.omega
        self.mu[0] = mu0
        self.E[0] = -model.beta0 * model.f(1.0, 0)
        self.n_rows = 1
        self.n_rhs = 0

    def rhs_current(self, M: int):
        """F = (F^C, F^R) for the current row M (values in hist[M], time in t[M])."""
        out = history_integrals(self.grid, self.model, self.t, self.mu, self.hist, M)
        self.n_rhs += 1
        return out["deriv"][:, 4].copy(), out["deriv"][:, 5].copy(), out["mu"], out["E"]


def ssprk104(F, y, t0: float, h: float, F1=None):
    """One step of SSPRK(10,4) in low-storage form for y' = F(t, y) (y any numpy array).
    F1 = F(t0, y) if already known (the derivative stored with the history).
    Returns (y_next, delta) with delta = h sum_k (b_k - bhat_k) F_k the embedded error estimate."""
    q1 = y.copy()
    q2 = y.copy()
    delta = np.zeros_like(y)
    for k in range(10):
        Fk = F1 if (k == 0 and F1 is not None) else F(t0 + SSPRK_C[k] * h, q1)
        delta = delta + (h * (SSPRK_B[k] - SSPRK_BHAT[k])) * Fk
        if k < 9:
            q1 = q1 + (h / 6.0) * Fk
            if k == 4:
                q2 = q2 / 25.0 + (9.0 / 25.0) * q1
                q1 = 15.0 * q2 - 5.0 * q1
        else:
            q1 = q2 + 0.6 * q1 + (0.1 * h) * Fk
    return q1, delta


def rk_step(H: History, h: float):
    """One SSPRK(10,4) step from the last (complete) row N.  Writes the new row N+1 (values) at
    t_N + h and returns eps_RK of Eq.(25).  Does not complete or accept the row.
    During stages 2..10 the stage state is the value-only current row M = N+1 (Eq.22)."""
    N = H.n_rows - 1
    M = N + 1
    assert M < H.n_cap
    L = H.grid.L
    y = np.concatenate([H.hist[N, :, 0], H.hist[N, :, 2]])
    F1 = np.concatenate([H.hist[N, :, 1], H.hist[N, :, 3]])

    def F(ts, q):
        H.t[M] = ts
        H.hist[M, :, 0], H.hist[M, :, 2] = q[:L], q[L:]
        H.hist[M, :, 1], H.hist[M, :, 3] = 0.0, 0.0
        FC, FR, _, _ = H.rhs_current(M)
        return np.concatenate([FC, FR])

    ynew, delta = ssprk104(F, y, H.t[N], h, F1)
    H.t[M] = H.t[N] + h
    H.hist[M, :, 0], H.hist[M, :, 2] = ynew[:L], ynew[L:]
    H.hist[M, :, 1], H.hist[M, :, 3] = 0.0, 0.0
    return float(np.sum(np.abs(delta)))


def complete_row(H: History):
    """Evaluate the right-hand side on the freshly appended row (= stage 1 of the next step) and
    store its ray derivative, mu and E with the history."""
    M = H.n_rows
    FC, FR, mu, E = H.rhs_current(M)
    H.hist[M, :, 1], H.hist[M, :, 3] = FC, FR
    H.mu[M], H.E[M] = mu, E
    H.n_rows = M + 1


# ---- Dormand-Prince 5(4) ("uses the Dormand-Prince method [63] at short times"),
# the textbook tableau of ref. [63]; row 7 of A equals the fifth-order weights b (FSAL)
DP_C = np.array([0.0, 1.0 / 5.0, 3.0 / 10.0, 4.0 / 5.0, 8.0 / 9.0, 1.0, 1.0])
DP_A = np.zeros((7, 7))
DP_A[1, :1] = [1.0 / 5.0]
DP_A[2, :2] = [3.0 / 40.0, 9.0 / 40.0]
DP_A[3, :3] = [44.0 / 45.0, -56.0 / 15.0, 32.0 / 9.0]
DP_A[4, :4] = [19372.0 / 6561.0, -25360.0 / 2187.0, 64448.0 / 6561.0, -212.0 / 729.0]
DP_A[5, :5] = [9017.0 / 3168.0, -355.0 / 33.0, 46732.0 / 5247.0, 49.0 / 176.0, -5103.0 / 18656.0]
DP_A[6, :6] = [35.0 / 384.0, 0.0, 500.0 / 1113.0, 125.0 / 192.0, -2187.0 / 6784.0, 11.0 / 84.0]
DP_B = DP_A[6].copy()
DP_BHAT = np.array([5179.0 / 57600.0, 0.0, 7571.0 / 16695.0, 393.0 / 640.0, -92097.0 / 339200.0,
                    187.0 / 2100.0, 1.0 / 40.0])
DP_SWITCH = 3.3  # switch to SSPRK(10,4) when h 4 sqrt(f''(1)) reaches the real-axis limit of DP5 (3.3066; G21)


def dopri54(F, y, t0: float, h: float, F1):
    """One Dormand-Prince 5(4) step for y' = F(t, y).  F1 = F(t0, y) (stored with the history).
    Stage i: y_i = y + h sum_{j<i} a_ij k_j (terms in the order j = 1, 2, ...; zero coefficients
    skipped), k_i = F(t0 + c_i h, y_i); y_next = y_7; k_7 = F(t0 + h, y_next) is the derivative of
    the new point (FSAL) and enters the error estimate delta = h sum_j (b_j - bhat_j) k_j.
    Returns (y_next, k_7, delta)."""
    k = [F1]
    yi = y
    for i in range(1, 7):
        acc = None
        for j in range(i):
            if DP_A[i, j] == 0.0:
                continue
            term = DP_A[i, j] * k[j]
            acc = term if acc is None else acc + term
        yi = y + h * acc
        k.append(F(t0 + DP_C[i] * h, yi))
    acc = None
    for j in range(7):
        e = DP_B[j] - DP_BHAT[j]
        if e == 0.0:
            continue
        term = e * k[j]
        acc = term if acc is None else acc + term
    return yi, k[6], h * acc


def dp_step(H: "History", h: float):
    """One Dormand-Prince step from the last complete row N: writes row N+1 (values, then its
    derivative, mu and E from the FSAL evaluation) and returns eps_RK of Eq.(25).  Does not accept
    the row (n_rows unchanged)."""
    N = H.n_rows - 1
    M = N + 1
    assert M < H.n_cap
    L = H.grid.L
    y = np.concatenate([H.hist[N, :, 0], H.hist[N, :, 2]])
    F1 = np.concatenate([H.hist[N, :, 1], H.hist[N, :, 3]])
    last = {}

    def F(ts, q):
        H.t[M] = ts
        H.hist[M, :, 0], H.hist[M, :, 2] = q[:L], q[L:]
        H.hist[M, :, 1], H.hist[M, :, 3] = 0.0, 0.0
        FC, FR, mu, E = H.rhs_current(M)
        last["mu"], last["E"] = mu, E
        return np.concatenate([FC, FR])

    ynew, k7, delta = dopri54(F, y, H.t[N], h, F1)
    H.hist[M, :, 1], H.hist[M, :, 3] = k7[:L], k7[L:]
    H.mu[M], H.E[M] = last["mu"], last["E"]
    return float(np.sum(np.abs(delta)))


def dp_controller_step(H: "History", h: float, tol: float):
    """One adaptive Dormand-Prince step with the controller of PAPER.md:320 (reading G20); no step
    cap here: the caller switches to SSPRK(10,4) when h reaches the stability boundary (G21).
    Returns (accepted, h_next, eps_RK)."""
    eps = dp_step(H, h)
    if not np.isfinite(eps) or eps > 2.0 * tol:
        H.n_rows = max(1, H.n_rows - 10)
        return False, h / 2.0, eps
    H.n_rows += 1
    if eps > tol:
        h = 0.9 * h
    elif eps < tol / 2.0:
        h = 1.01 * h
    return True, h, eps


def dp_must_switch(model: "Model", h: float) -> bool:
    """Dormand-Prince "until the time step grows sufficiently to reach the boundary of
    its stability domain"; with the spectral bound 4 sqrt(f''(1)) of Eq.(24) (reading G21)."""
    return h * 4.0 * np.sqrt(model.f(1.0, 2)) >= DP_SWITCH


def h_stab(model: Model) -> float:
    """Step cap from Eq.(24) and the real-axis stability limit of SSPRK(10,4)."""
    return STAB_REAL_AXIS / (4.0 * np.sqrt(model.f(1.0, 2)))


def run_fixed(grid: Grid, model: Model, h: float, n_steps: int, n_cap=None):
    """Fixed-step trajectory (BASELINE.json config 1): no controller, no sparsification."""
    H = History(grid, model, n_cap or n_steps + 2)
    for _ in range(n_steps):
        rk_step(H, h)
        complete_row(H)
    return H


def controller_step(H: History, h: float, tol: float):
    """One adaptive step (reading G20).  Returns (accepted, h_next, eps_RK)."""
    eps = rk_step(H, h)
    cap = h_stab(H.model)
    if not np.isfinite(eps) or eps > 2.0 * tol:
        H.n_rows = max(1, H.n_rows - 10)
        return False, min(h / 2.0, cap), eps
    complete_row(H)
    if eps > tol:
        h = 0.9 * h
    elif eps < tol / 2.0:
        h = 1.01 * h
    return True, min(h, cap), eps


def sparsify_mask(eps_sparse, N: int, tol: float, protect_last: int):
    """Greedy rule of PAPER.md:334: walking n upward, drop slice n if eps_sparse < tol/10 and
    continue with n+2, else continue with n+1.  Row 0 and the last `protect_last` rows are kept
    (reading G25).  Returns keep[N] (bool)."""
    keep = np.ones(N, dtype=bool)
    n = 1
    last = N - 1 - protect_last
    while n <= last and n <= N - 2:
        if eps_sparse[n] < tol / 10.0:
            keep[n] = False
            n += 2
        else:
            n += 1
    return keep


def sparsify(H: History, tol: float, protect_last: int = 12):
    """Selective history reduction: compaction of t, mu, E and packed rows."""
    N = H.n_rows
    eps = sparsify_residuals(H.grid.L, N, H.t[:N], H.hist[:N])
    keep = sparsify_mask(eps, N, tol, protect_last)
    idx = np.nonzero(keep)[0]
    m = len(idx)
    H.t[:m], H.mu[:m], H.E[:m] = H.t[idx], H.mu[idx], H.E[idx]
    H.hist[:m] = H.hist[idx]
    H.n_rows = m
    return keep, eps


def run_adaptive(grid: Grid, model: Model, t_end: float, tol: float, h0=1e-3, n_cap=2048,
                 sp_every=200, protect_last=12, h_min=1e-12, max_steps=10 ** 9, log=None, startup="ssprk"):
    """Adaptive trajectory with periodic sparsification.
    startup = "dp": Dormand-Prince steps until dp_must_switch, then h/2 and SSPRK(10,4)."""
    H = History(grid, model, n_cap)
    h = min(h0, h_stab(model))
    use_dp = startup == "dp"
    acc = 0
    steps = 0
    while H.t[H.n_rows - 1] < t_end and steps < max_steps:
        if H.n_rows + 1 >= n_cap or (acc > 0 and acc % sp_every == 0):
            before = H.n_rows
            sparsify(H, tol, protect_last)
            if H.n_rows + 1 >= n_cap:
                raise RuntimeError("capacity: sparsify freed nothing (%d rows)" % before)
            acc += 1 if acc % sp_every == 0 else 0
        if use_dp and dp_must_switch(model, h):
            use_dp = False
            h = min(h / 2.0, h_stab(model))
        ok, h, eps = dp_controller_step(H, h, tol) if use_dp else controller_step(H, h, tol)
        steps += 1
        if ok:
            acc += 1
        if log is not None:
            log.append((H.t[H.n_rows - 1], h, eps, ok, H.n_rows))
        if h < h_min:
            raise RuntimeError("step below h_min")
    return H


# --------------------------------------------------------------------------- the step loop of a run
@dataclass
class Policy:
    """The loop's free parameters (PAPER.md:334-336 leaves the thinning schedule and the number of passes to
    the user, PAPER.md:316 the start-up switch; reading G25/G21).  The Eq.(27) threshold tol/10 is not one."""
    batch: int = 50            # SSPRK steps between two looks at the state
    sp_every: int = 200        # thin the history once this many steps were accepted since the last time
    sp_max_passes: int = 8     # greedy passes per thinning at most ...
    sp_min_gain: float = 0.01  # ... repeated while a pass still drops this fraction of the rows
    protect_last: int = 24     # two consecutive reverts take back 20 rows
    startup_dp: bool = False


@dataclass
class RunState:
    h: float
    acc_since: int = 0
    startup: bool = False
    status: str = "ok"
    log: list = field(default_factory=list)   # (accepted, eps_RK, h_next, n_rows) per attempted step
    masks: list = field(default_factory=list)  # keep mask of every thinning pass


def integrate(H: History, policy: Policy, rs: RunState, t_end: float, tol: float, max_steps: int = 0,
              h_min: float = 1e-12):
    """The step loop of a run, as the library's dmfe_integrate holds it:
      loop until t >= t_end (or max_steps more steps):
        thin the history if due (acc_since >= sp_every, or fewer than two free rows): greedy passes
           until one drops less than sp_min_gain of the rows or sp_max_passes is reached;
          still fewer than two free rows: capacity error;
        start-up: h 4 sqrt(f''(1)) >= 3.3 -> h = min(h/2, cap), SSPRK(10,4) from then on;
          else one Dormand-Prince step;
        otherwise min(batch, steps left, free rows) SSPRK(10,4) steps with the controller of PAPER.md:320;
          a step that leaves h < h_min ends the run.
    Returns the number of steps attempted in this call."""
    model = H.model
    if H.n_rows == 1 and policy.startup_dp:
        rs.startup = True
    done = 0
    while H.t[H.n_rows - 1] < t_end:
        if max_steps > 0 and done >= max_steps:
            break
        if rs.acc_since >= policy.sp_every or H.n_rows + 2 > H.n_cap:
            for _ in range(policy.sp_max_passes):
                before = H.n_rows
                keep, _eps = sparsify(H, tol, policy.protect_last)
                rs.masks.append(keep)
                freed = before - H.n_rows
                if freed < policy.sp_min_gain * before or freed < 1:
                    break
            rs.acc_since = 0
            if H.n_rows + 2 > H.n_cap:
                rs.status = "capacity"
                break
        if rs.startup:
            if dp_must_switch(model, rs.h):
                rs.startup = False
                rs.h = min(rs.h / 2.0, h_stab(model))
                continue
            ok, rs.h, eps = dp_controller_step(H, rs.h, tol)
            rs.log.append((ok, eps, rs.h, H.n_rows))
            done += 1
            if ok:
                rs.acc_since += 1
            if rs.h < h_min:
                rs.status = "stepmin"
                break
        else:
            nb = policy.batch
            if max_steps > 0:
                nb = min(nb, max_steps - done)
            nb = min(nb, H.n_cap - H.n_rows)
            stop = False
            for _ in range(nb):
                ok, rs.h, eps = controller_step(H, rs.h, tol)
                rs.log.append((ok, eps, rs.h, H.n_rows))
                done += 1
                if ok:
                    rs.acc_since += 1
                if rs.h < h_min:
                    rs.status = "stepmin"
                    stop = True
                    break
            if stop:
                break
    return done
