// Internal declarations of libdmfe.so (not part of the C ABI; see include/dmfe.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <string.h>

#include "dmfe.h"

#define DMFE_PMAX_MAX 15
#define DMFE_EV_RING 512

// f(q) = 1/2 sum_p lambda_p q^p (Eq.(4)).  Horner coefficients, lowest power first:
//   f (q) = sum_k c0[k] q^k        c0[k] = lambda_k / 2
//   f'(q) = sum_k c1[k] q^k        c1[k] = (k+1) lambda_{k+1} / 2
//   f''(q)= sum_k c2[k] q^k        c2[k] = (k+2)(k+1) lambda_{k+2} / 2
struct ModelCoef {
  double c0[DMFE_PMAX_MAX + 1];
  double c1[DMFE_PMAX_MAX + 1];
  double c2[DMFE_PMAX_MAX + 1];
  double T;
  double beta0;
  int32_t pmax;
};

// device scalar block (ctx->scal), indices
enum {
  SC_MU = 0,     // mu(t) of the row being evaluated (Eq.(13))
  SC_E = 1,      // E(t) (Eq.(14))
  SC_H = 2,      // current step size
  SC_EPS = 3,    // eps_RK of the last attempted step (Eq.(25))
  SC_T0 = 4,     // t_N at the start of the step
  SC_HNEXT = 5,  // step size proposed by the controller (latched into SC_H by stage 0 of the next step)
  SC_ACCEPT = 6, // accept flag of the last step as a double (so that one copy returns the whole record)
  SC_TLAST = 7,  // time of the last complete row after the last committed step
  SC_COUNT = 16
};
// device int block (ctx->iscal)
enum {
  IS_ACCEPT = 0,  // 1 accepted, 0 reverted
  IS_NROWS = 1,   // complete rows after the step / after sparsify
  IS_FIRST = 2,   // sparsify: first row that moves
  IS_STATUS = 3,  // 0, or the DMFE_E* code that stopped a batch of steps (later steps of the batch are no-ops)
  IS_NACC = 4,    // accepted / reverted / attempted steps of the running dmfe_advance call
  IS_NREV = 5,
  IS_STEP = 6,
  IS_RTVALID = 7, // leading entries of the per-call row table that are final (device-resident steps)
  IS_COUNT = 8
};

struct dmfe_ctx {
  dmfe_params p;
  ModelCoef model;
  cudaStream_t stream;
  int cuda_err;
  int sm_count;  // SMs of the device the context was created on
  int smem_max;  // opt-in dynamic shared memory per CTA, minus the kernels' static use
  double gamma, A, B;  // gamma = -W_{-1}(-1/t_max); A = atan(e^gamma), B = atan(e^-gamma)
  double h_stab;       // 13.9 / (4 sqrt(f''(1)))  (Eq.(24))
  // ---- tables (device) ----
  double *theta, *omega, *nu;  // [L]
  double2 *thnu;               // [L] {theta_j, nu_j}
  uint64_t *tab;               // [3][L][L] packed {stencil start : 16 | fractional coordinate : 48}
  // ---- O(L) scratch (device) ----
  double2 *cur;     // [L] {C, R} of the current row, packed for 16-byte gathers
  int32_t *blo;     // [L] per-call row bracket table: blo[c] = n(theta_c t_M)
  double *win;      // values-only mode: [win_cap][8] per-call t-windows {t_k..t_k+3, inverse denominators}
  int32_t win_cap;
  double2 *muw;     // [L] per call: mu(theta_c t_M) = muw.x + muw.y * mu(t_M)  (reading G11)
  double2 *rowtab;  // [rowtab_cap] per-call {t_n, 1 / (t_{n+1} - t_n)}
  // S = 4 only (pairs_s4.cuh), rebuilt per call by the pre-pass
  int2 *br;         // [L] row bracket of the grid cell of phi2, indexed by the phi2 stencil start
  int32_t *jtop;    // [L] first node of every target whose type-2 interval is the top one
  double *coefM;    // [L][8]  centred cubics of {C, R} of the current row, per stencil start
  double *coefT;    // [L][16] centred cubics of {C, dC, R, dR} of row M-1
  int32_t *tgt_next;  // [1] work counter of the S = 4 pair kernel (reset by the pre-pass of every evaluation)
  int32_t rowtab_cap;
  int rowtab_dirty;  // the row table was (or may have been) rebuilt for another history: rebuild it in full
  double *scal;     // [SC_COUNT]
  int32_t *iscal;   // [IS_COUNT]
  double *rk;       // [4][L][2]: q1, q2, delta, F
  double *dpk;      // [7][L][2]: Dormand-Prince k_1..k_6 and F (allocated by the first dmfe_dp_step)
  double *eps_sp;   // [n] sparsify residuals (grown on demand)
  int32_t *keep;    // [n] keep flags / scan
  int32_t *newidx;  // [n] compacted source index
  int32_t sp_cap;
  double *row_tmp;  // staging for compaction
  size_t row_tmp_bytes;
  // ---- host-buffer leg ----
  double *stage_t, *stage_mu, *stage_hist, *stage_out;
  int32_t stage_rows;
  // measurement hooks
  int timing_on;
  cudaEvent_t ev[2 * DMFE_EV_RING];  // (before, after) pairs around the pair kernel, lazily created
  int ev_made;                       // pairs created so far
  int ev_n;                          // pairs recorded since timing was switched on
  // pinned host scalars for the one-record-per-step readback
  double *h_scal;
  int32_t *h_iscal;
  // one SSPRK(10,4) step as a CUDA graph (21 kernel nodes), re-launched for every step of
  // dmfe_advance; all of its arguments live in device memory, so it is captured once per state
  cudaGraph_t step_graph;
  cudaGraphExec_t step_exec;
  const void *graph_key[5];  // t, mu, energy, hist pointers of the state it was captured for + flags
  int graph_off;             // capture failed once: plain launches from then on
  double *steplog;           // [steplog_cap][4] device: {accepted, eps_RK, h_next, n_rows} per step
  double *h_steplog;         // pinned host copy
  int32_t steplog_cap;
  // a batch of steps as one persistent cooperative kernel (advance_s4.cu)
  unsigned *adv_bar;  // arrival counter of its grid barrier
  int adv_off;        // that path is not available on this device / for this size: use the graph of launches
  int step_mode;      // dmfe_set_step_mode: 0 = automatic, 1 = always the graph of launches
};

#define CUDA_TRY(ctx, call)                              \
  do {                                                   \
    cudaError_t e__ = (call);                            \
    if (e__ != cudaSuccess) {                            \
      (ctx)->cuda_err = (int)e__;                        \
      return DMFE_ECUDA;                                 \
    }                                                    \
  } while (0)

// Packed pair-table entry: bits 63..48 = stencil start (L <= 65535), bits 47..0 = the fractional
// index coordinate u = X - start in fixed point, q = rint((u + 1) 2^44).  q is exactly the mantissa
// field of the double x = 16 + (u + 1)/16 in [16, 17) (ulp 2^-48, top 16 bits 0x4030), so decoding
// is one mask/or on the high word and one exact DFMA: u = 16 x - 257.  Resolution 2^-44 = 5.7e-14
// index units (far below the ~4e-12 accuracy of X itself in fp64); -1 <= u < 15 covers every
// stencil (s <= 10).  The decoded value is THE coordinate of the library: dmfe_get_tables returns it.
#if defined(__CUDACC__)
#define DMFE_HD __host__ __device__ __forceinline__
#else
#define DMFE_HD inline
#endif
DMFE_HD uint64_t dmfe_tab_encode(int32_t start, double frac) {
  const double x = (frac + 1.0) * 17592186044416.0;  // 2^44: exact scaling
  long long q = (long long)rint(x);
  if (q < 0) q = 0;
  if (q > (1LL << 48) - 1) q = (1LL << 48) - 1;
  return ((uint64_t)(uint32_t)start << 48) | (uint64_t)q;
}
DMFE_HD void dmfe_tab_decode(uint64_t e, int32_t *start, double *frac) {
  *start = (int32_t)(e >> 48);
  const uint64_t bits = 0x4030000000000000ULL | (e & 0xFFFFFFFFFFFFULL);
  double x;
#if defined(__CUDA_ARCH__)
  x = __longlong_as_double((long long)bits);
#else
  memcpy(&x, &bits, sizeof(x));
#endif
  *frac = x * 16.0 - 257.0;  // exact: x has at most 48 significant fraction bits below 2^4
}

// One SSPRK(10,4) stage update fused into the O(L + M) pre-pass of the right-hand side that follows
// it (rk_step.cu fills this in; k < 0 = no stage update, plain evaluation of row M).
struct dmfe_stage {
  int32_t k;           // stage 0..9 of PAPER.md:314-316; the update writes the value slots of row N+1
  int32_t N;           // last complete row (host value; ignored when dev_rows is set)
  int32_t fixed_step;  // k == 9: 1 = no controller
  int32_t complete;    // the evaluation completes the appended row M: mu[M], energy[M], derivative slots
  double tol, cap;     // k == 9: epsilon of Eq.(25), step cap of Eq.(24)
  double *hist, *t;    // writable views of the caller's history
  double *mu, *energy; // complete != 0: writable per-row arrays
  double *rk;          // [4][2L]: q1, q2, delta, F
  double *scal;
  int32_t *iscal;
  const int32_t *dev_rows;  // device-resident step: number of complete rows (= M) is read from here and
                            // a non-zero iscal[IS_STATUS] turns the launch into a no-op
};

// tables.cu
int dmfe_build_tables(dmfe_ctx *ctx);
// pairs_values.cu: the right-hand side on a values-only history (dmfe_params.values_only)
int dmfe_launch_rhs_values(dmfe_ctx *ctx, int32_t M, int32_t n_cap, const double *t, const double *mu_hist,
                           const double *hist, const dmfe_rhs_out *out);
// advance_s4.cu: one batch of SSPRK(10,4) steps as a persistent kernel; 1 = not applicable (take the graph path)
int dmfe_launch_advance_s4(dmfe_ctx *ctx, dmfe_state *st, int n_steps, int fixed_step, double *log, int log_cap);
// history_integrals.cu
// stage: optional stage update run by the pre-pass; deriv_row: optional row of the history whose
// derivative slots receive F (the derivative is stored with the appended row)
int dmfe_launch_rhs(dmfe_ctx *ctx, int32_t M, int32_t n_cap, const double *t, const double *mu_hist,
                    const double *hist, const dmfe_rhs_out *out, const dmfe_stage *stage = nullptr,
                    double *deriv_row = nullptr);
