"""Thin ctypes binding of libdmfe.so (include/dmfe.h): same names, argument marshalling only.

Device memory and the stream come from torch (plumbing); every step of the path runs inside the
CUDA library.  There is no fallback: importing works without the library (so that CPU-only tests
can check its symbols), but every call raises if libdmfe.so is missing or a call fails.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import POINTER, Structure, byref, c_char_p, c_double, c_int, c_int32, c_int64, c_uint8, c_void_p

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libdmfe.so")

DMFE_OK, DMFE_EINVAL, DMFE_ECUDA, DMFE_ECAPACITY, DMFE_ESTEPMIN, DMFE_ENONFINITE, DMFE_ENOMEM = 0, -1, -2, -3, -4, -5, -6
DMFE_ETOOLARGE = -7
DMFE_STATIC_MAX_L, DMFE_STATIC_MAX_ROWS = 4096, 16384

EXPORTS = ["dmfe_create", "dmfe_destroy", "dmfe_last_cuda_error", "dmfe_strerror", "dmfe_get_tables",
           "dmfe_history_integrals", "dmfe_history_integrals_host", "dmfe_static_limits", "dmfe_static_init",
           "dmfe_history_integrals_static", "dmfe_init_state", "dmfe_rk_step",
           "dmfe_advance", "dmfe_set_step_mode", "dmfe_dp_step", "dmfe_set_step_size",
           "dmfe_sparsify", "dmfe_integrate", "dmfe_enable_timing", "dmfe_last_kernel_ms", "dmfe_kernel_time_stats",
           "dmfe_probe_fp64_tflops"]


class dmfe_params(Structure):
    _fields_ = [("L", c_int32), ("stencil", c_int32), ("quad_degree", c_int32), ("p_max", c_int32),
                ("t_max", c_double), ("beta0", c_double), ("tol", c_double), ("h_min", c_double),
                ("values_only", c_int32), ("log_r", c_int32), ("stream", c_void_p)]


class dmfe_grid(Structure):
    _fields_ = [("n_rows", c_int32), ("n_cap", c_int32), ("t", c_void_p), ("mu", c_void_p), ("hist", c_void_p)]


class dmfe_rhs_out(Structure):
    _fields_ = [("d1C", c_void_p), ("d1R", c_void_p), ("mu", c_void_p), ("d2C", c_void_p), ("d2R", c_void_p),
                ("F", c_void_p), ("energy", c_void_p), ("sums", c_void_p), ("rows1", c_void_p), ("rows2", c_void_p)]


class dmfe_state(Structure):
    _fields_ = [("n_rows", c_int32), ("n_cap", c_int32), ("t", c_void_p), ("mu", c_void_p), ("energy", c_void_p),
                ("hist", c_void_p), ("h", c_double), ("eps_rk", c_double), ("n_rhs", c_int64),
                ("acc_since", c_int32), ("startup", c_int32)]


class dmfe_policy(Structure):
    _fields_ = [("batch", c_int32), ("sp_every", c_int32), ("sp_max_passes", c_int32), ("sp_min_gain", c_double),
                ("protect_last", c_int32), ("startup_dp", c_int32)]


class dmfe_run_stats(Structure):
    _fields_ = [("steps", c_int64), ("accepted", c_int64), ("reverted", c_int64), ("dp_steps", c_int64),
                ("sparsify_calls", c_int64), ("sparsify_passes", c_int64), ("rows_dropped", c_int64),
                ("n_rows", c_int32), ("n_rows_max", c_int32), ("status", c_int32), ("pad", c_int32),
                ("t", c_double), ("h", c_double), ("eps_rk", c_double)]


class dmfe_advance_result(Structure):
    _fields_ = [("steps", c_int32), ("accepted", c_int32), ("reverted", c_int32), ("n_rows", c_int32),
                ("last_accepted", c_int32), ("t_last", c_double), ("h_next", c_double), ("eps_rk", c_double)]


class DmfeError(RuntimeError):
    def __init__(self, code, what, cuda=0):
        self.code = code
        super().__init__("%s failed: %s (code %d, cuda error %d)" % (what, _strerror(code), code, cuda))


_lib = None


def load_library():
    """dlopen libdmfe.so and declare the prototypes of include/dmfe.h.  Raises if it is missing."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError("libdmfe.so not built (run `python -m paper_2604_06309_b200.build`); "
                           "this package has no CPU fallback")
    lib = ctypes.CDLL(LIB_PATH)
    lib.dmfe_create.restype = c_int
    lib.dmfe_create.argtypes = [POINTER(dmfe_params), POINTER(c_double), c_double, POINTER(c_void_p)]
    lib.dmfe_destroy.restype = c_int
    lib.dmfe_destroy.argtypes = [c_void_p]
    lib.dmfe_last_cuda_error.restype = c_int
    lib.dmfe_last_cuda_error.argtypes = [c_void_p]
    lib.dmfe_strerror.restype = c_char_p
    lib.dmfe_strerror.argtypes = [c_int]
    lib.dmfe_get_tables.restype = c_int
    lib.dmfe_get_tables.argtypes = [c_void_p, c_void_p, c_void_p, c_void_p, c_int32, c_int32, c_void_p, c_void_p]
    lib.dmfe_history_integrals.restype = c_int
    lib.dmfe_history_integrals.argtypes = [c_void_p, POINTER(dmfe_grid), POINTER(dmfe_rhs_out)]
    lib.dmfe_static_limits.restype = c_int
    lib.dmfe_static_limits.argtypes = [POINTER(c_int32), POINTER(c_int32), POINTER(c_int64)]
    lib.dmfe_static_init.restype = c_int
    lib.dmfe_static_init.argtypes = [c_void_p]
    lib.dmfe_history_integrals_static.restype = c_int
    lib.dmfe_history_integrals_static.argtypes = [c_void_p, POINTER(dmfe_grid), POINTER(dmfe_rhs_out)]
    lib.dmfe_history_integrals_host.restype = c_int
    lib.dmfe_history_integrals_host.argtypes = [c_void_p, c_int32] + [c_void_p] * 7
    lib.dmfe_init_state.restype = c_int
    lib.dmfe_init_state.argtypes = [c_void_p, POINTER(dmfe_state), c_double]
    lib.dmfe_rk_step.restype = c_int
    lib.dmfe_rk_step.argtypes = [c_void_p, POINTER(dmfe_state), c_int32, POINTER(c_int32)]
    lib.dmfe_advance.restype = c_int
    lib.dmfe_advance.argtypes = [c_void_p, POINTER(dmfe_state), c_int32, c_int32, POINTER(dmfe_advance_result),
                                 c_void_p]
    lib.dmfe_set_step_mode.restype = c_int
    lib.dmfe_set_step_mode.argtypes = [c_void_p, c_int32]
    lib.dmfe_dp_step.restype = c_int
    lib.dmfe_dp_step.argtypes = [c_void_p, POINTER(dmfe_state), c_int32, POINTER(c_int32)]
    lib.dmfe_set_step_size.restype = c_int
    lib.dmfe_set_step_size.argtypes = [c_void_p, POINTER(dmfe_state), c_double]
    lib.dmfe_sparsify.restype = c_int
    lib.dmfe_sparsify.argtypes = [c_void_p, POINTER(dmfe_state), c_int32, POINTER(c_int32), c_void_p]
    lib.dmfe_integrate.restype = c_int
    lib.dmfe_integrate.argtypes = [c_void_p, POINTER(dmfe_state), POINTER(dmfe_policy), c_double, c_int64, c_double,
                                   POINTER(dmfe_run_stats)]
    lib.dmfe_enable_timing.restype = c_int
    lib.dmfe_enable_timing.argtypes = [c_void_p, c_int32]
    lib.dmfe_last_kernel_ms.restype = c_int
    lib.dmfe_last_kernel_ms.argtypes = [c_void_p, POINTER(ctypes.c_float)]
    lib.dmfe_kernel_time_stats.restype = c_int
    lib.dmfe_kernel_time_stats.argtypes = [c_void_p, POINTER(c_int32), POINTER(c_double), POINTER(c_double)]
    lib.dmfe_probe_fp64_tflops.restype = c_int
    lib.dmfe_probe_fp64_tflops.argtypes = [c_void_p, c_int32, POINTER(c_double), POINTER(c_int32)]
    _lib = lib
    return lib


def _strerror(code):
    try:
        return load_library().dmfe_strerror(code).decode()
    except Exception:
        return "?"


def _check(rc, what, ctx=None):
    if rc != DMFE_OK:
        cuda = load_library().dmfe_last_cuda_error(ctx) if ctx else 0
        raise DmfeError(rc, what, cuda)


def _dev(t):
    """device pointer of a torch CUDA tensor (None -> NULL)"""
    if t is None:
        return None
    assert t.is_cuda and t.is_contiguous(), "device, contiguous tensors only"
    return c_void_p(t.data_ptr())


def _host(a):
    if a is None:
        return None
    assert isinstance(a, np.ndarray) and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(c_void_p)


# ------------------------------------------------------------------------------------------------
def dmfe_create(L, stencil, t_max, lam, T, beta0=0.0, tol=0.0, h_min=0.0, quad_degree=5, stream=None,
                values_only=False, log_r=False):
    """-> opaque context handle.  lam[p] are the lambda_p of f(q) = 1/2 sum_p lam[p] q^p."""
    import torch
    lib = load_library()
    if not torch.cuda.is_available():
        raise RuntimeError("dmfe_create: no CUDA device (this package has no CPU fallback)")
    lam = np.ascontiguousarray(lam, dtype=np.float64)
    if stream is None:
        stream = torch.cuda.current_stream().cuda_stream
    p = dmfe_params(L=L, stencil=stencil, quad_degree=quad_degree, p_max=len(lam) - 1, t_max=t_max, beta0=beta0,
                    tol=tol, h_min=h_min, values_only=1 if values_only else 0, log_r=1 if log_r else 0, stream=c_void_p(stream))
    ctx = c_void_p()
    _check(lib.dmfe_create(byref(p), lam.ctypes.data_as(POINTER(c_double)), float(T), byref(ctx)), "dmfe_create")
    return ctx


def dmfe_destroy(ctx):
    _check(load_library().dmfe_destroy(ctx), "dmfe_destroy")


def dmfe_get_tables(ctx, L, i0=0, n_targets=None, want_pairs=True):
    """-> dict(theta, omega, nu, start[3,nt,L], frac[3,nt,L]) as numpy arrays (host)."""
    lib = load_library()
    theta, omega, nu = np.empty(L), np.empty(L), np.empty(L)
    start = frac = None
    nt = L if n_targets is None else n_targets
    if want_pairs:
        start = np.empty((3, nt, L), dtype=np.int32)
        frac = np.empty((3, nt, L), dtype=np.float64)
    _check(lib.dmfe_get_tables(ctx, _host(theta), _host(omega), _host(nu), i0, nt, _host(start), _host(frac)),
           "dmfe_get_tables", ctx)
    return dict(theta=theta, omega=omega, nu=nu, start=start, frac=frac)


def dmfe_history_integrals(ctx, n_rows, t, mu, hist, d1C=None, d1R=None, mu_out=None, d2C=None, d2R=None, F=None,
                           energy=None, sums=None, rows1=None, rows2=None):
    """(grid, C, R, t_n) -> (dC, dR, mu): all arguments are torch CUDA tensors; asynchronous."""
    lib = load_library()
    g = dmfe_grid(n_rows=n_rows, n_cap=t.shape[0], t=_dev(t), mu=_dev(mu), hist=_dev(hist))
    o = dmfe_rhs_out(d1C=_dev(d1C), d1R=_dev(d1R), mu=_dev(mu_out), d2C=_dev(d2C), d2R=_dev(d2R), F=_dev(F),
                     energy=_dev(energy), sums=_dev(sums), rows1=_dev(rows1), rows2=_dev(rows2))
    _check(lib.dmfe_history_integrals(ctx, byref(g), byref(o)), "dmfe_history_integrals", ctx)


def dmfe_static_limits():
    """(max L, max history rows, bytes of the static scratch array) of dmfe_history_integrals_static."""
    a, b, c = c_int32(0), c_int32(0), c_int64(0)
    load_library().dmfe_static_limits(byref(a), byref(b), byref(c))
    return a.value, b.value, c.value


def dmfe_static_init(ctx):
    _check(load_library().dmfe_static_init(ctx), "dmfe_static_init", ctx)


def dmfe_history_integrals_static(ctx, n_rows, t, mu, hist, d1C=None, d1R=None, mu_out=None, d2C=None, d2R=None,
                                  F=None, energy=None, sums=None, rows1=None, rows2=None):
    """dmfe_history_integrals without any allocation: per-call tables in the library's static device array
    (L <= DMFE_STATIC_MAX_L, n_rows - 1 <= DMFE_STATIC_MAX_ROWS, else DMFE_ETOOLARGE); asynchronous."""
    lib = load_library()
    g = dmfe_grid(n_rows=n_rows, n_cap=t.shape[0], t=_dev(t), mu=_dev(mu), hist=_dev(hist))
    o = dmfe_rhs_out(d1C=_dev(d1C), d1R=_dev(d1R), mu=_dev(mu_out), d2C=_dev(d2C), d2R=_dev(d2R), F=_dev(F),
                     energy=_dev(energy), sums=_dev(sums), rows1=_dev(rows1), rows2=_dev(rows2))
    _check(lib.dmfe_history_integrals_static(ctx, byref(g), byref(o)), "dmfe_history_integrals_static", ctx)


def dmfe_history_integrals_host(ctx, n_rows, t, mu, hist, d1C, d1R, mu_out, energy):
    """Same call with HOST numpy buffers (copies inside); synchronous."""
    lib = load_library()
    _check(lib.dmfe_history_integrals_host(ctx, n_rows, _host(t), _host(mu), _host(hist), _host(d1C), _host(d1R),
                                           _host(mu_out), _host(energy)), "dmfe_history_integrals_host", ctx)


def make_state(L, n_cap, device="cuda"):
    """Allocate the caller-owned device arrays of a dmfe_state with torch; returns (state, tensors)."""
    import torch
    ten = dict(t=torch.zeros(n_cap, dtype=torch.float64, device=device),
               mu=torch.zeros(n_cap, dtype=torch.float64, device=device),
               energy=torch.zeros(n_cap, dtype=torch.float64, device=device),
               hist=torch.zeros((n_cap, L, 4), dtype=torch.float64, device=device))
    st = dmfe_state(n_rows=0, n_cap=n_cap, t=_dev(ten["t"]), mu=_dev(ten["mu"]), energy=_dev(ten["energy"]),
                    hist=_dev(ten["hist"]), h=0.0, eps_rk=0.0, n_rhs=0, acc_since=0, startup=0)
    return st, ten


def dmfe_set_step_mode(ctx, mode):
    """0: automatic (persistent kernel for S = 4, L <= 512); 1: always the graph of launches."""
    _check(load_library().dmfe_set_step_mode(ctx, int(mode)), "dmfe_set_step_mode", ctx)


def dmfe_init_state(ctx, st, h0):
    _check(load_library().dmfe_init_state(ctx, byref(st), float(h0)), "dmfe_init_state", ctx)


def dmfe_rk_step(ctx, st, fixed_step=False):
    """-> accepted (bool).  Raises DmfeError on capacity / minimal step / CUDA errors."""
    acc = c_int32(0)
    _check(load_library().dmfe_rk_step(ctx, byref(st), 1 if fixed_step else 0, byref(acc)), "dmfe_rk_step", ctx)
    return bool(acc.value)


def dmfe_advance(ctx, st, n_steps, fixed_step=False, want_log=False, check=True):
    """n_steps device-resident SSPRK(10,4) steps (one CUDA graph launch per step, one record back per
    batch).  -> (dmfe_advance_result, log[steps, 4] or None, return code).  With check=True a stop code
    (minimal step, non-finite error) raises DmfeError; capacity always does."""
    res = dmfe_advance_result()
    log = np.zeros((n_steps, 4)) if want_log else None
    rc = load_library().dmfe_advance(ctx, byref(st), int(n_steps), 1 if fixed_step else 0, byref(res), _host(log))
    if rc != DMFE_OK and (check or rc in (DMFE_EINVAL, DMFE_ECUDA, DMFE_ECAPACITY)):
        _check(rc, "dmfe_advance", ctx)
    return res, (log[:res.steps] if want_log else None), rc


def dmfe_dp_step(ctx, st, fixed_step=False):
    """Dormand-Prince 5(4) start-up step -> accepted (bool)."""
    acc = c_int32(0)
    _check(load_library().dmfe_dp_step(ctx, byref(st), 1 if fixed_step else 0, byref(acc)), "dmfe_dp_step", ctx)
    return bool(acc.value)


def dmfe_set_step_size(ctx, st, h):
    _check(load_library().dmfe_set_step_size(ctx, byref(st), float(h)), "dmfe_set_step_size", ctx)


def dmfe_sparsify(ctx, st, protect_last=12, want_mask=False):
    """-> (n_rows_after, keep_mask or None)"""
    n_out = c_int32(0)
    mask = np.zeros(st.n_rows, dtype=np.uint8) if want_mask else None
    _check(load_library().dmfe_sparsify(ctx, byref(st), protect_last, byref(n_out), _host(mask)), "dmfe_sparsify", ctx)
    return n_out.value, (mask.astype(bool) if want_mask else None)


def dmfe_integrate(ctx, st, policy, t_end, max_steps=0, max_seconds=0.0, stats=None, check=True):
    """The step loop of a run inside the library (thinning schedule, start-up switch, batches of steps).
    -> (stats, return code); stats accumulates over calls when passed back in."""
    if stats is None:
        stats = dmfe_run_stats()
    rc = load_library().dmfe_integrate(ctx, byref(st), byref(policy) if policy is not None else None, float(t_end),
                                       int(max_steps), float(max_seconds), byref(stats))
    if rc != DMFE_OK and check:
        _check(rc, "dmfe_integrate", ctx)
    return stats, rc


def dmfe_enable_timing(ctx, on=True):
    _check(load_library().dmfe_enable_timing(ctx, 1 if on else 0), "dmfe_enable_timing", ctx)


def dmfe_last_kernel_ms(ctx):
    ms = ctypes.c_float(0.0)
    _check(load_library().dmfe_last_kernel_ms(ctx, byref(ms)), "dmfe_last_kernel_ms", ctx)
    return float(ms.value)


def dmfe_kernel_time_stats(ctx):
    """-> (launches timed, total ms, min ms) of the pair kernel since dmfe_enable_timing(True)"""
    n, tot, mn = c_int32(0), c_double(0.0), c_double(0.0)
    _check(load_library().dmfe_kernel_time_stats(ctx, byref(n), byref(tot), byref(mn)), "dmfe_kernel_time_stats", ctx)
    return n.value, tot.value, mn.value


def dmfe_probe_fp64_tflops(ctx, n_iter=1 << 16):
    """-> (achieved DFMA TFLOP/s, SM count)"""
    tf, sms = c_double(0.0), c_int32(0)
    _check(load_library().dmfe_probe_fp64_tflops(ctx, n_iter, byref(tf), byref(sms)), "dmfe_probe_fp64_tflops", ctx)
    return tf.value, sms.value
