// Device-resident SSPRK(10,4) step and error controller (Eq.(22), Eq.(25)).
// The stage arithmetic itself lives in the pre-pass of the right-hand side that consumes the
// stage state (history_integrals.cu: prepare_kernel), so a step is 10 x (pre-pass + pair kernel)
// = 20 launches and one 128-byte record back to the host:
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

}  // namespace

extern "C" {

int dmfe_init_state(dmfe_ctx *ctx, dmfe_state *st, double h0) {
  if (!ctx || !st || !st->t || !st->mu || !st->hist || st->n_cap < 3 || !(h0 > 0.0)) return DMFE_EINVAL;
  const int L = ctx->p.L;
  const double h = fmin(h0, ctx->h_stab);
  init_row0_kernel<<<(L + 255) / 256, 256, 0, ctx->stream>>>(L, ctx->model, ctx->omega, st->hist, st->t, st->mu,
                                                           st->energy, ctx->scal, h);
  CUDA_TRY(ctx, cudaGetLastError());
  st->n_rows = 1;
  st->h = h;
  st->eps_rk = 0.0;
  st->n_rhs = 0;
  return DMFE_OK;
}

int dmfe_rk_step(dmfe_ctx *ctx, dmfe_state *st, int32_t fixed_step, int32_t *accepted) {
  if (!ctx || !st || !st->t || !st->mu || !st->hist) return DMFE_EINVAL;
  if (st->n_rows < 1) return DMFE_EINVAL;
  if (st->n_rows + 1 > st->n_cap) return DMFE_ECAPACITY;
  const int L = ctx->p.L;
  const int N = st->n_rows - 1, M = N + 1;
  double *F = ctx->rk + 6 * (size_t)L;
  dmfe_stage sg;
  sg.N = N;
  sg.fixed_step = fixed_step;
  sg.tol = ctx->p.tol;
  sg.cap = ctx->h_stab;
  sg.hist = st->hist;
  sg.t = st->t;
  sg.rk = ctx->rk;
  sg.scal = ctx->scal;
  sg.iscal = ctx->iscal;
  for (int k = 0; k < 10; ++k) {
    dmfe_rhs_out o;
    memset(&o, 0, sizeof(o));
    o.F = F;
    double *deriv_row = nullptr;
    if (k == 9) {  // the evaluation after the last stage completes the appended row
      o.mu = st->mu + M;
      o.energy = st->energy ? st->energy + M : nullptr;
      deriv_row = st->hist + (size_t)M * (size_t)L * 4;
    }
    sg.k = k;
    sg.after_prepass = (k == 9) ? ctx->ev_decided : nullptr;
    const int rc = dmfe_launch_rhs(ctx, M, st->n_cap, st->t, st->mu, st->hist, &o, &sg, deriv_row);
    if (rc != DMFE_OK) return rc;
    st->n_rhs++;
  }
  // the one record that returns to the host: {accept flag, eps_RK, next h}
  // It is final once the pre-pass of the last stage has run, so it is copied on the side stream
  // behind that point: the host learns the decision and queues the next step while the evaluation
  // that completes the appended row is still running.
  CUDA_TRY(ctx, cudaStreamWaitEvent(ctx->side, ctx->ev_decided, 0));
  CUDA_TRY(ctx, cudaMemcpyAsync(ctx->h_scal, ctx->scal, sizeof(double) * SC_COUNT, cudaMemcpyDeviceToHost,
                                ctx->side));
  CUDA_TRY(ctx, cudaStreamSynchronize(ctx->side));
  const int acc = ctx->h_scal[SC_ACCEPT] != 0.0;
  st->eps_rk = ctx->h_scal[SC_EPS];
  st->h = ctx->h_scal[SC_HNEXT];
  if (accepted) *accepted = acc;
  if (acc) {
    st->n_rows = M + 1;
  } else {
    if (!isfinite(st->eps_rk) && st->n_rows == 1) return DMFE_ENONFINITE;
    st->n_rows = (st->n_rows - 10 > 1) ? st->n_rows - 10 : 1;  // revert the previous ten steps
  }
  if (!fixed_step && st->h < ctx->p.h_min) return DMFE_ESTEPMIN;
  return DMFE_OK;
}

}  // extern "C"
