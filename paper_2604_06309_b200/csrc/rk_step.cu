// Device-resident SSPRK(10,4) steps and error controller (Eq.(22), Eq.(25)).
// The stage arithmetic itself lives in the pre-pass of the right-hand side that consumes the
// stage state (history_integrals.cu: prepare_kernel), so a step is 10 x (pre-pass + pair kernel)
// + one commit kernel = 21 kernel nodes.  Everything a step needs to know about the state -- the
// number of complete rows, the step size, the accept flag, the stop status -- lives in device
// memory, so the 21 nodes have constant arguments: they are captured once into a CUDA graph and
// dmfe_advance re-launches that graph for every step of a batch without returning to the host
// ("launch overhead"); one record and the optional per-step log come back per batch.
//   stage k (k = 0..9) writes the value-only current row M = N+1 (Eq.(22)); stage 0 uses the
//   derivative stored with row N; stage 9 forms y+, eps_RK and the controller
//   decision, and the evaluation that follows it completes the appended row (its derivative, mu
//   and E are stored with the history) -- it is stage 1 of the next step.  If the step is
//   rejected that evaluation is discarded with the row.
#include <math.h>
#include <string.h>

#include "dmfe_internal.cuh"

namespace {

__global__ void init_row0_kernel(int L, ModelCoef mc, const double *__restrict__ omega, double *__restrict__ hist,
                                 double *__restrict__ t, double *__restrict__ mu, double *__restrict__ energy,
                                 double *__restrict__ scal, double h0) {
  double f1 = 0.0, f0 = 0.0;
  for (int k = mc.pmax; k >= 0; --k) {
    f1 += mc.c1[k];
    f0 += mc.c0[k];
  }
  const double mu0 = mc.T + mc.beta0 * f1;
  for (int l = blockIdx.x * blockDim.x + threadIdx.x; l < L; l += gridDim.x * blockDim.x) {
    double *c = hist + (size_t)l * 4;
    c[0] = 1.0;
    c[1] = -mc.T * omega[l];
    c[2] = 1.0;
    c[3] = -mu0 * omega[l];
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    t[0] = 0.0;
    mu[0] = mu0;
    if (energy) energy[0] = -mc.beta0 * f0;
    scal[SC_H] = h0;
    scal[SC_HNEXT] = h0;
  }
}

// Applies the decision of the step that has just run: accepted -> the appended row
// becomes the last complete row; rejected -> the previous ten rows are dropped.  One thread.
__global__ void commit_step_kernel(int32_t *__restrict__ iscal, double *__restrict__ scal, const double *__restrict__ t,
                                   int fixed_step, double h_min, double *__restrict__ log, int log_cap) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  if (iscal[IS_STATUS] != 0) return;
  int n = iscal[IS_NROWS];
  const int acc = iscal[IS_ACCEPT];
  const double eps = scal[SC_EPS], hn = scal[SC_HNEXT];
  int status = 0;
  if (acc) {
    n += 1;
    iscal[IS_NACC] += 1;
  } else {
    if (!isfinite(eps) && n == 1) status = DMFE_ENONFINITE;
    n = (n - 10 > 1) ? n - 10 : 1;  // revert the previous ten steps
    iscal[IS_NREV] += 1;
  }
  // row-table entries below the last complete row of the step that has just run are final; after a
  // revert only those below the new last row
  {
    const int n_before = acc ? n - 1 : iscal[IS_NROWS];
    const int v = (n < n_before ? n : n_before) - 1;
    iscal[IS_RTVALID] = v > 0 ? v : 0;
  }
  iscal[IS_NROWS] = n;
  scal[SC_TLAST] = t[n - 1];
  const int step = iscal[IS_STEP];
  iscal[IS_STEP] = step + 1;
  if (log && step < log_cap) {
    double *r = log + 4 * (size_t)step;
    r[0] = (double)acc, r[1] = eps, r[2] = hn, r[3] = (double)n;
  }
  if (!fixed_step && hn < h_min && status == 0) status = DMFE_ESTEPMIN;
  iscal[IS_STATUS] = status;
}

__global__ void begin_batch_kernel(int32_t *__restrict__ iscal, int n_rows, int rowtab_dirty) {
  if (rowtab_dirty) iscal[IS_RTVALID] = 0;
  iscal[IS_NROWS] = n_rows;
  iscal[IS_STATUS] = 0;
  iscal[IS_NACC] = 0;
  iscal[IS_NREV] = 0;
  iscal[IS_STEP] = 0;
}

// the 21 launches of one step; all state-dependent values are read on the device
int enqueue_step(dmfe_ctx *ctx, dmfe_state *st, int fixed_step, double *log, int log_cap) {
  const int L = ctx->p.L;
  double *F = ctx->rk + 6 * (size_t)L;
  dmfe_stage sg;
  memset(&sg, 0, sizeof(sg));
  sg.fixed_step = fixed_step;
  sg.tol = ctx->p.tol;
  sg.cap = ctx->h_stab;
  sg.hist = st->hist;
  sg.t = st->t;
  sg.mu = st->mu;
  sg.energy = st->energy;
  sg.rk = ctx->rk;
  sg.scal = ctx->scal;
  sg.iscal = ctx->iscal;
  sg.dev_rows = ctx->iscal + IS_NROWS;
  for (int k = 0; k < 10; ++k) {
    dmfe_rhs_out o;
    memset(&o, 0, sizeof(o));
    o.F = F;
    sg.k = k;
    sg.complete = (k == 9) ? 1 : 0;  // the evaluation after the last stage completes the appended row
    const int rc = dmfe_launch_rhs(ctx, st->n_cap, st->n_cap, st->t, st->mu, st->hist, &o, &sg, nullptr);
    if (rc != DMFE_OK) return rc;
  }
  commit_step_kernel<<<1, 32, 0, ctx->stream>>>(ctx->iscal, ctx->scal, st->t, fixed_step, ctx->p.h_min, log, log_cap);
  return DMFE_OK;
}

}  // namespace

extern "C" {

int dmfe_init_state(dmfe_ctx *ctx, dmfe_state *st, double h0) {
  if (ctx && ctx->p.values_only) return DMFE_EINVAL;  // the integrator keeps the Hermite history
  if (!ctx || !st || !st->t || !st->mu || !st->hist || st->n_cap < 3 || !(h0 > 0.0)) return DMFE_EINVAL;
  const int L = ctx->p.L;
  const double h = fmin(h0, ctx->h_stab);
  init_row0_kernel<<<(L + 255) / 256, 256, 0, ctx->stream>>>(L, ctx->model, ctx->omega, st->hist, st->t, st->mu,
                                                           st->energy, ctx->scal, h);
  CUDA_TRY(ctx, cudaGetLastError());
  ctx->rowtab_dirty = 1;
  st->n_rows = 1;
  st->h = h;
  st->eps_rk = 0.0;
  st->n_rhs = 0;
  st->acc_since = 0;
  st->startup = 0;
  return DMFE_OK;
}

int dmfe_advance(dmfe_ctx *ctx, dmfe_state *st, int32_t n_steps, int32_t fixed_step, dmfe_advance_result *res,
                 double *step_log) {
  if (ctx && ctx->p.values_only) return DMFE_EINVAL;  // the integrator keeps the Hermite history
  if (!ctx || !st || !st->t || !st->mu || !st->hist || n_steps < 1) return DMFE_EINVAL;
  if (st->n_rows < 1) return DMFE_EINVAL;
  if (st->n_rows + 1 > st->n_cap) return DMFE_ECAPACITY;
  // every accepted step appends one row: a batch never outgrows the caller's arrays
  if (n_steps > st->n_cap - st->n_rows) n_steps = st->n_cap - st->n_rows;
  cudaStream_t s = ctx->stream;
  double *dlog = nullptr;
  if (step_log) {
    if (n_steps > ctx->steplog_cap) {
      CUDA_TRY(ctx, cudaStreamSynchronize(s));
      cudaFree(ctx->steplog);
      if (ctx->h_steplog) cudaFreeHost(ctx->h_steplog);
      ctx->steplog = ctx->h_steplog = nullptr;
      ctx->steplog_cap = 0;
      const int cap = n_steps < 256 ? 256 : n_steps;
      CUDA_TRY(ctx, cudaMalloc(&ctx->steplog, sizeof(double) * 4 * (size_t)cap));
      CUDA_TRY(ctx, cudaMallocHost(&ctx->h_steplog, sizeof(double) * 4 * (size_t)cap));
      ctx->steplog_cap = cap;
      ctx->graph_key[0] = nullptr;  // the log pointer is an argument of the captured commit kernel
    }
    dlog = ctx->steplog;
  }
  if (st->n_cap > ctx->rowtab_cap) {  // no allocation may happen inside a capture
    CUDA_TRY(ctx, cudaStreamSynchronize(s));
    cudaFree(ctx->rowtab);
    ctx->rowtab = nullptr;
    ctx->rowtab_cap = 0;
    CUDA_TRY(ctx, cudaMalloc(&ctx->rowtab, sizeof(double2) * (size_t)st->n_cap));
    ctx->rowtab_cap = st->n_cap;
  }
  begin_batch_kernel<<<1, 1, 0, s>>>(ctx->iscal, st->n_rows, ctx->rowtab_dirty);
  ctx->rowtab_dirty = 0;
  CUDA_TRY(ctx, cudaGetLastError());
  // L <= 512, S = 4: the whole batch as one persistent cooperative kernel (advance_s4.cu)
  bool persistent = false;
  {
    const int rc = dmfe_launch_advance_s4(ctx, st, n_steps, fixed_step, dlog, ctx->steplog_cap);
    if (rc < 0) return rc;
    persistent = (rc == DMFE_OK);
    if (persistent) ctx->rowtab_dirty = 1;  // that kernel keeps the row table its own way
  }
  // one step as a graph, captured once per (state arrays, mode); plain launches if capture is unavailable
  const void *key[5] = {st->t, st->mu, st->energy, st->hist,
                        (const void *)(uintptr_t)(((uintptr_t)st->n_cap << 2) | (fixed_step ? 1u : 0u) | (dlog ? 2u : 0u))};
  if (!persistent && !ctx->graph_off && (ctx->step_exec == nullptr || memcmp(key, ctx->graph_key, sizeof(key)) != 0)) {
    if (ctx->step_exec) cudaGraphExecDestroy(ctx->step_exec);
    if (ctx->step_graph) cudaGraphDestroy(ctx->step_graph);
    ctx->step_exec = nullptr;
    ctx->step_graph = nullptr;
    cudaError_t e = cudaStreamBeginCapture(s, cudaStreamCaptureModeThreadLocal);
    int rc = DMFE_OK;
    if (e == cudaSuccess) {
      rc = enqueue_step(ctx, st, fixed_step, dlog, ctx->steplog_cap);
      e = cudaStreamEndCapture(s, &ctx->step_graph);
    }
    if (e == cudaSuccess && rc == DMFE_OK) e = cudaGraphInstantiate(&ctx->step_exec, ctx->step_graph, 0);
    if (e != cudaSuccess || rc != DMFE_OK) {
      cudaGetLastError();  // clear the sticky-free capture error
      if (ctx->step_graph) cudaGraphDestroy(ctx->step_graph);
      ctx->step_graph = nullptr;
      ctx->step_exec = nullptr;
      ctx->graph_off = 1;
    } else {
      memcpy(ctx->graph_key, key, sizeof(key));
    }
  }
  for (int k = 0; k < n_steps && !persistent; ++k) {
    if (ctx->step_exec) {
      CUDA_TRY(ctx, cudaGraphLaunch(ctx->step_exec, s));
    } else {
      const int rc = enqueue_step(ctx, st, fixed_step, dlog, ctx->steplog_cap);
      if (rc != DMFE_OK) return rc;
      CUDA_TRY(ctx, cudaGetLastError());
    }
  }
  // the one record that returns to the host per batch
  CUDA_TRY(ctx, cudaMemcpyAsync(ctx->h_scal, ctx->scal, sizeof(double) * SC_COUNT, cudaMemcpyDeviceToHost, s));
  CUDA_TRY(ctx, cudaMemcpyAsync(ctx->h_iscal, ctx->iscal, sizeof(int32_t) * IS_COUNT, cudaMemcpyDeviceToHost, s));
  if (dlog)
    CUDA_TRY(ctx, cudaMemcpyAsync(ctx->h_steplog, dlog, sizeof(double) * 4 * (size_t)n_steps, cudaMemcpyDeviceToHost, s));
  CUDA_TRY(ctx, cudaStreamSynchronize(s));
  const int done = ctx->h_iscal[IS_STEP];
  st->n_rows = ctx->h_iscal[IS_NROWS];
  st->eps_rk = ctx->h_scal[SC_EPS];
  st->h = ctx->h_scal[SC_HNEXT];
  st->n_rhs += 10LL * done;
  if (step_log) memcpy(step_log, ctx->h_steplog, sizeof(double) * 4 * (size_t)done);
  if (res) {
    res->steps = done;
    res->accepted = ctx->h_iscal[IS_NACC];
    res->reverted = ctx->h_iscal[IS_NREV];
    res->n_rows = st->n_rows;
    res->last_accepted = ctx->h_iscal[IS_ACCEPT];
    res->t_last = ctx->h_scal[SC_TLAST];
    res->h_next = st->h;
    res->eps_rk = st->eps_rk;
  }
  return ctx->h_iscal[IS_STATUS];
}

int dmfe_set_step_mode(dmfe_ctx *ctx, int32_t mode) {
  if (!ctx || mode < 0 || mode > 1) return DMFE_EINVAL;
  ctx->step_mode = mode;
  return DMFE_OK;
}

int dmfe_rk_step(dmfe_ctx *ctx, dmfe_state *st, int32_t fixed_step, int32_t *accepted) {
  dmfe_advance_result r;
  memset(&r, 0, sizeof(r));
  const int rc = dmfe_advance(ctx, st, 1, fixed_step, &r, nullptr);
  if (accepted) *accepted = r.last_accepted;
  return rc;
}

}  // extern "C"
