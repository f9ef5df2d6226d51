/*
 * dmfe.h -- C ABI of libdmfe.so: the B200 (sm_100a, fp64) hot path of the DMFE solver of
 * arxiv/paper_2604_06309 ("DYNAMITE"): per-RK-stage evaluation of the history (memory)
 * integrals, the device-resident SSPRK(10,4) step with its error controller, and the
 * selective history reduction ("sparsification").
 *
 * Citations are PAPER.md:<line> (+ equation); readings Gnn are listed in DESIGN.md.
 *
 * Conventions
 *   L        length of the fixed theta-grid, theta = t'/t in [0,1]       (Eq.(16))
 *   rows     stored time slices t_0 = 0 < t_1 < ...; row n holds, for every theta_l,
 *            one 32-byte cell {C, dC, R, dR}:  C(t_n, theta_l t_n), R(t_n, theta_l t_n) and their
 *            derivatives along the ray (d/dt at fixed theta)
 *   f(q)     = 1/2 sum_{p=0..p_max} lambda[p] q^p                        (Eq.(4); G2)
 *   i, j, l  target node, quadrature node, stencil column (0-based)
 *
 * Every entry point returns 0 on success or a negative DMFE_E* code; nothing throws, nothing
 * calls exit().  "device" pointers are CUDA device pointers owned by the caller (the Python
 * binding takes them from torch tensors); "host" pointers are ordinary host memory.  All work is
 * enqueued on the stream given at creation; calls that return a host scalar synchronise that
 * stream, the others are asynchronous.  There is no CPU fallback anywhere in this library.
 */
#ifndef DMFE_H
#define DMFE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define DMFE_API __attribute__((visibility("default")))
#else
#define DMFE_API
#endif

#define DMFE_OK 0
#define DMFE_EINVAL (-1)      /* bad parameter (L < 2s, t_max <= e, n_rows < 2, NULL pointer ...) */
#define DMFE_ECUDA (-2)       /* a CUDA call failed; dmfe_last_cuda_error() has the code (0 when the
                                 persistent step kernel gave up on its grid barrier after 2 s)     */
#define DMFE_ECAPACITY (-3)   /* a step needs a free row: n_rows + 1 > n_cap                      */
#define DMFE_ESTEPMIN (-4)    /* controller drove h below h_min                    */
#define DMFE_ENONFINITE (-5)  /* eps_RK not finite and nothing left to revert                     */
#define DMFE_ENOMEM (-6)      /* host or device allocation failed                                 */
#define DMFE_ETOOLARGE (-7)   /* dmfe_history_integrals_static: L or n_rows beyond the static scratch */

typedef struct dmfe_ctx dmfe_ctx; /* opaque: tables + O(L) scratch on the device */

typedef struct {
  int32_t L;           /* theta-grid length, >= 2*stencil                                        */
  int32_t stencil;     /* s = points of the index-Lagrange stencil, even, 2..10   */
  int32_t quad_degree; /* odd degree of the global spline that defines nu_j; 5 = paper default
                          (PAPER.md:278); 1 and 3 are accepted                                   */
  int32_t p_max;       /* lambda has p_max+1 entries, 2 <= p_max <= 15                           */
  double t_max;        /* sets gamma = -W_{-1}(-1/t_max); must be > e.  The grid is
                          Eq.(16) with alpha = delta = 0 (the closed-form invertible grid): the
                          (alpha, delta) warp of PAPER.md:217-228 is NOT offered by this library
                          (reading G6 in DESIGN.md)                            */
  double beta0;        /* inverse temperature of the initial condition, 0 = random start (Eq.(12)) */
  double tol;          /* epsilon of Eq.(25); used by rk_step / sparsify only      */
  double h_min;        /* terminate below this step; 0 -> 1e-12                    */
  int32_t values_only; /* != 0: the history holds {C, R} only (16-byte cells, [n_cap][L][2]) and the
                          interpolation in t is the local 4-point Lagrange polynomial through rows
                          n-1 .. n+2 instead of cubic Hermite.
                          dmfe_history_integrals(_host) only: the integrator calls return DMFE_EINVAL */
  int32_t log_r;       /* != 0: logarithmic interpolation of the response history: the type-1
                          and type-2 lookups of R act on log R and dR/R whenever every value read is
                          positive, with automatic fallback to the ordinary interpolation (reading G32);
                          not with values_only                                                        */
  void *stream;        /* cudaStream_t borrowed from the caller (0 = default stream)             */
} dmfe_params;

/* Build the t-independent tables ("precomputed once"): theta_i and the complement
 * omega_i = 1-theta_i (Eq.(16)), quadrature weights nu_j, and for every pair
 * (i,j) and each coordinate phi1 = theta_i theta_j, phi2 = theta_i + omega_i theta_j,
 * psi = theta_i/phi2 the stencil start and the fractional index coordinate
 * (Eq.(18), (20)).  lambda: host, [p_max+1].  T: bath temperature.  *out receives the context. */
DMFE_API int dmfe_create(const dmfe_params *params, const double *lambda, double T, dmfe_ctx **out);
DMFE_API int dmfe_destroy(dmfe_ctx *ctx);

/* Last CUDA error code seen by this context (cudaError_t as int), 0 if none. */
DMFE_API int dmfe_last_cuda_error(const dmfe_ctx *ctx);
DMFE_API const char *dmfe_strerror(int code);

/* Test hook (table parity): copy tables to HOST buffers.  theta, omega, nu: [L] (any may be NULL).
 * start: [3][n_targets][L] int32, frac: [3][n_targets][L] fp64 for the coordinates
 * (phi1, phi2, psi) of targets i0 .. i0+n_targets-1 (NULL to skip).  Synchronises. */
DMFE_API int dmfe_get_tables(dmfe_ctx *ctx, double *theta, double *omega, double *nu, int32_t i0,
                    int32_t n_targets, int32_t *start, double *frac);

/* The history as the caller holds it (all DEVICE pointers, caller-owned). */
typedef struct {
  int32_t n_rows;     /* rows 0..n_rows-1 are valid; row M = n_rows-1 is the CURRENT row: its
                         derivative slots and mu[M] are ignored on input (G12)                  */
  int32_t n_cap;      /* row capacity of the three arrays                                       */
  const double *t;    /* [n_cap] ascending, t[0] = 0                                            */
  const double *mu;   /* [n_cap] Lagrange multiplier of rows 0..M-1 (Eq.(13))                   */
  const double *hist; /* [n_cap][L][4] packed cells {C, dC, R, dR}; values_only: [n_cap][L][2] {C, R} */
} dmfe_grid;

/* Outputs of one right-hand-side evaluation; DEVICE pointers, any may be NULL. */
typedef struct {
  double *d1C;    /* [L] dC/dt  of Eq.(1) (with the -mu C term, G1)              */
  double *d1R;    /* [L] dR/dt  of Eq.(1)                                                        */
  double *mu;     /* [1] mu(t), Eq.(13)                                           */
  double *d2C;    /* [L] dC/dt' (second-argument equation, G9/G10)                               */
  double *d2R;    /* [L] dR/dt'                                                                  */
  double *F;      /* [L][2] ray derivatives {d1C + theta d2C, d1R + theta d2R} = ODE rhs, Eq.(22) */
  double *energy; /* [1] E(t), Eq.(14)                                            */
  double *sums;   /* [8][L] the eight nu-weighted sums S1..S8 of Eq.(21) (DESIGN.md step 6)      */
  int32_t *rows1; /* [L]    test hook: type-1 row index n(theta_i t)                             */
  int32_t *rows2; /* [L][L] test hook: type-2 row index n(phi2_ij t)                             */
} dmfe_rhs_out;

/* north-star call (grid, C, R, t_n) -> (dC, dR, mu): C, R are row M of grid->hist, t_n = t[M].
 * Eq.(17)-(21) with K = f''(C)R, D = f'(C) (Eq.(10)-(11)).  Asynchronous. */
DMFE_API int dmfe_history_integrals(dmfe_ctx *ctx, const dmfe_grid *grid, const dmfe_rhs_out *out);

/* Same call with HOST buffers (the end-to-end leg of bench.py): copies t, mu, hist rows
 * 0..n_rows-1 to library-owned device staging (grown on demand), evaluates, copies
 * d1C, d1R [L] and mu, energy [1] back (any may be NULL).  Synchronises. */
DMFE_API int dmfe_history_integrals_host(dmfe_ctx *ctx, int32_t n_rows, const double *t, const double *mu_hist,
                                const double *hist, double *d1C, double *d1R, double *mu,
                                double *energy);

/* The north-star call for callers that may not allocate (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid cudaMalloc): same kernels and same results as dmfe_history_integrals
 * (Eq.(17)-(21); Hermite history, any stencil, log_r honoured; values_only: DMFE_EINVAL), but the per-call
 * tables of the pre-pass live in one file-scope device array of fixed size instead of context memory that
 * the ordinary path grows with cudaMalloc on demand.  Limits: L <= DMFE_STATIC_MAX_L grid nodes and
 * n_rows - 1 <= DMFE_STATIC_MAX_ROWS history rows, beyond which the call returns DMFE_ETOOLARGE and
 * launches nothing; the array is 1 245 440 bytes and every GPU that loads the library holds it until the
 * process exits.  The call issues two cudaMemsetAsync (the slices that must start at zero) and the two
 * kernels on the context's stream and calls no cudaMalloc, cudaFree or allocating library routine.  All
 * pointers are DEVICE pointers owned by the caller, as for dmfe_history_integrals.  Asynchronous.
 * The array is shared by every call on a device, whatever the context, and keeps the last call's contents:
 * calls ordered on one stream are safe; calls that overlap on the GPU (two streams without an event between
 * them, two host threads) race on it and give wrong results.
 * dmfe_static_init resolves the array's device address for the CURRENT device (which must be the
 * context's) and clears the array on the context's stream; call it once per device before the first
 * capture (the first dmfe_history_integrals_static on a device does the same resolution otherwise, which
 * may load a module).  dmfe_static_limits reports the limits and the array size; any pointer may be NULL. */
#define DMFE_STATIC_MAX_L 4096
#define DMFE_STATIC_MAX_ROWS 16384
DMFE_API int dmfe_static_limits(int32_t *max_L, int32_t *max_rows, int64_t *bytes);
DMFE_API int dmfe_static_init(dmfe_ctx *ctx);
DMFE_API int dmfe_history_integrals_static(dmfe_ctx *ctx, const dmfe_grid *grid, const dmfe_rhs_out *out);

/* Device-resident integrator state.  The arrays are caller-owned DEVICE memory.  The device copies of the
 * step size, the row count and the decisions live in the context: a context drives ONE state at a time
 * (dmfe_init_state or any call with another state's arrays re-synchronises from the host fields below). */
typedef struct {
  int32_t n_rows;  /* complete rows (value + derivative + mu); updated by the library            */
  int32_t n_cap;   /* capacity; a step needs n_rows + 1 <= n_cap                                  */
  double *t;       /* [n_cap]                                                                     */
  double *mu;      /* [n_cap]                                                                     */
  double *energy;  /* [n_cap] E(t_n) of every stored row                                          */
  double *hist;    /* [n_cap][L][4]                                                               */
  double h;        /* current step size (host copy; the device copy lives in the context)        */
  double eps_rk;   /* Eq.(25) of the last attempted step (host copy)                              */
  int64_t n_rhs;   /* history-integral evaluations so far                                         */
  int32_t acc_since; /* dmfe_integrate: steps accepted since the history was last thinned          */
  int32_t startup;   /* dmfe_integrate: 1 while the run is in its Dormand-Prince start-up          */
} dmfe_state;

/* Row 0 at t = 0 (G13): C = R = 1, ray slopes -T(1-theta), -mu0(1-theta), mu0 = T + beta0 f'(1);
 * sets n_rows = 1 and h = h0 (capped by the stability bound of Eq.(24)). */
DMFE_API int dmfe_init_state(dmfe_ctx *ctx, dmfe_state *st, double h0);

/* What comes back from a batch of steps (one device-to-host copy per batch). */
typedef struct {
  int32_t steps;         /* steps attempted (fewer than asked if the batch stopped or would outgrow n_cap) */
  int32_t accepted;      /* of which accepted ...                                                        */
  int32_t reverted;      /* ... and reverted (each drops the last ten rows)                */
  int32_t n_rows;        /* complete rows after the batch                                                 */
  int32_t last_accepted; /* decision of the last step                                                     */
  double t_last;         /* time of the last complete row                                                 */
  double h_next;         /* step size the controller proposes for the next step                           */
  double eps_rk;         /* Eq.(25) of the last attempted step                                            */
} dmfe_advance_result;

/* n_steps SSPRK(10,4) steps from the last row without returning to the host: the
 * row count, the step size and every decision live in device memory, and one step (ten stage updates
 * + evaluations and the commit of the decision) is one CUDA graph that is re-launched n_steps times.
 * fixed_step != 0: no controller, every row is appended.  Otherwise the controller of PAPER.md:320
 * (G20) runs on the device after every step: eps_RK > 2 tol or non-finite -> drop the last 10 rows,
 * h/2; else append, h *= 0.9 if eps_RK > tol, h *= 1.01 if eps_RK < tol/2; always h <= the cap of
 * Eq.(24).  The batch is cut to n_cap - n_rows steps so that it cannot outgrow the arrays (nothing
 * to do: DMFE_ECAPACITY).  A step that ends with h < h_min (DMFE_ESTEPMIN) or with a non-finite
 * error and nothing left to revert (DMFE_ENONFINITE) turns the rest of the batch into no-ops and is
 * returned as the call's code; st and *res describe the state at that point.
 * step_log: optional HOST [n_steps][4] doubles {accepted, eps_RK, h_next, n_rows after} per step.
 * Synchronises on the context's stream.
 * Two implementations of the same arithmetic and decisions (dmfe_set_step_mode): for the 4-point stencil
 * and L <= 512 the whole batch runs as ONE persistent cooperative kernel (every CTA carries the stage state
 * in shared memory, a stage costs one grid-wide barrier; csrc/advance_s4.cu); otherwise, or when the device
 * cannot launch it, as the graph of 21 kernel nodes per step described above.  Sums over the L nodes
 * (mu, E, eps_RK) are formed in a different order by the two, so their rows agree to rounding, not bit for bit. */
DMFE_API int dmfe_advance(dmfe_ctx *ctx, dmfe_state *st, int32_t n_steps, int32_t fixed_step,
                          dmfe_advance_result *res, double *step_log);

/* mode 0 (default): dmfe_advance picks the persistent kernel where it applies; mode 1: always the graph of
 * launches (the path every stencil order and every L takes).  Other values: DMFE_EINVAL. */
DMFE_API int dmfe_set_step_mode(dmfe_ctx *ctx, int32_t mode);

/* One step: dmfe_advance(ctx, st, 1, fixed_step, ...) with *accepted = the decision. */
DMFE_API int dmfe_rk_step(dmfe_ctx *ctx, dmfe_state *st, int32_t fixed_step, int32_t *accepted);

/* One Dormand-Prince 5(4) step (the start-up integrator "at short times", textbook
 * tableau of ref. [63]) from the last row, all stages on the device; same state, same record and
 * same controller as dmfe_rk_step except that no step cap is applied: the caller switches to
 * dmfe_rk_step when h 4 sqrt(f''(1)) reaches the stability boundary of the method (3.3; reading
 * G21 in DESIGN.md) with dmfe_set_step_size(h/2).  Six evaluations per step; the
 * last one (FSAL) stores the derivative, mu and E of the appended row and enters the error
 * estimate, so the record is read after it.  Synchronises on the context's stream. */
DMFE_API int dmfe_dp_step(dmfe_ctx *ctx, dmfe_state *st, int32_t fixed_step, int32_t *accepted);

/* Sets the step size the next dmfe_rk_step / dmfe_dp_step starts from (device copy and st->h).
 * h <= 0: DMFE_EINVAL.  Asynchronous. */
DMFE_API int dmfe_set_step_size(dmfe_ctx *ctx, dmfe_state *st, double h);

/* Selective history reduction, Eq.(26)-(27): drop row n if eps_sparse < tol/10,
 * then skip to n+2; row 0 and the last protect_last rows are kept; t, mu, energy and the packed
 * rows are compacted on the device.  keep_mask: optional HOST [n_rows before] bytes (test hook). */
DMFE_API int dmfe_sparsify(dmfe_ctx *ctx, dmfe_state *st, int32_t protect_last, int32_t *n_rows_out,
                  uint8_t *keep_mask);

/* The step loop of a run: when to thin the history, how many greedy passes a
 * thinning takes (PAPER.md:336 makes "the number of sparsification passes" a user control), the
 * Dormand-Prince start-up and its switch to SSPRK(10,4).  The paper fixes none of the
 * numbers below except the Eq.(27) threshold tol/10, which is NOT a parameter here (reading G25).
 * A zero field selects the default in brackets. */
typedef struct {
  int32_t batch;         /* SSPRK(10,4) steps per device batch; the loop below looks at the state only
                            between batches [50]                                                      */
  int32_t sp_every;      /* thin the history once this many steps were accepted since the last time
                            [200]                                                                     */
  int32_t sp_max_passes; /* greedy passes per thinning at most [8] ...                                */
  double sp_min_gain;    /* ... repeated while a pass still drops this fraction of the rows [0.01]    */
  int32_t protect_last;  /* newest rows that are never dropped: two consecutive reverts take back 20
                            rows [24]                                                  */
  int32_t startup_dp;    /* != 0: start with Dormand-Prince steps and switch to SSPRK(10,4) with
                            min(h/2, Eq.(24) cap) when h 4 sqrt(f''(1)) >= 3.3 (reading G21) [0]      */
} dmfe_policy;

typedef struct {
  int64_t steps;           /* attempted steps ...                                                     */
  int64_t accepted;        /* ... of which accepted ...                                               */
  int64_t reverted;        /* ... and reverted                                                        */
  int64_t dp_steps;        /* Dormand-Prince steps among them                                         */
  int64_t sparsify_calls;  /* thinnings ...                                                           */
  int64_t sparsify_passes; /* ... greedy passes they took ...                                         */
  int64_t rows_dropped;    /* ... rows they dropped                                                   */
  int32_t n_rows;          /* complete rows now                                                       */
  int32_t n_rows_max;      /* most rows held at any time                                              */
  int32_t status;          /* DMFE_OK or the code that ended the loop                                 */
  int32_t pad;
  double t;                /* time of the last complete row                                           */
  double h;                /* next step size                                                          */
  double eps_rk;           /* Eq.(25) of the last step                                                */
} dmfe_run_stats;

/* Runs the step loop until t >= t_end, max_steps more steps were attempted (<= 0: no limit) or
 * max_seconds of wall time have passed (<= 0: no limit); stats (in/out) accumulates over calls:
 *   loop:  thin the history if due (acc_since >= sp_every, or fewer than two free rows): passes of
 *          dmfe_sparsify until one drops less than sp_min_gain of the rows or sp_max_passes is reached;
 *          still fewer than two free rows: DMFE_ECAPACITY;
 *          start-up: h 4 sqrt(f''(1)) >= 3.3 -> h = min(h/2, cap) and SSPRK(10,4) from then on, else one
 *          dmfe_dp_step; otherwise dmfe_advance(min(batch, steps left)).
 * The test oracle holds the same loop; the tests compare the two decision for decision.
 * st->acc_since and st->startup carry the loop's state between calls. */
DMFE_API int dmfe_integrate(dmfe_ctx *ctx, dmfe_state *st, const dmfe_policy *policy, double t_end,
                            int64_t max_steps, double max_seconds, dmfe_run_stats *stats);

/* Measurement hooks (bench.py).  dmfe_enable_timing: when on, every dmfe_history_integrals launch
 * records CUDA events on the context's stream immediately before and after the pair kernel (the
 * dominant kernel); dmfe_last_kernel_ms synchronises on the closing event and returns the elapsed
 * time of the most recent one.  dmfe_probe_fp64_tflops runs a register-resident DFMA chain on all
 * SMs (n_iter fused multiply-adds per thread, 8 independent chains) and reports the achieved
 * 2*DFMA/s: the denominator of the FP64 roofline, measured rather than assumed. */
DMFE_API int dmfe_enable_timing(dmfe_ctx *ctx, int32_t on);
DMFE_API int dmfe_last_kernel_ms(dmfe_ctx *ctx, float *ms);
/* Sum (and minimum) of the pair-kernel durations of all launches since timing was switched on
 * (at most 512 are kept); synchronises on the last one.  No synchronisation happens between the
 * launches themselves, so this can bracket every launch of a timed region. */
DMFE_API int dmfe_kernel_time_stats(dmfe_ctx *ctx, int32_t *n_launches, double *total_ms, double *min_ms);
DMFE_API int dmfe_probe_fp64_tflops(dmfe_ctx *ctx, int32_t n_iter, double *tflops, int32_t *sm_count);
#ifdef __cplusplus
}
#endif
#endif /* DMFE_H */
