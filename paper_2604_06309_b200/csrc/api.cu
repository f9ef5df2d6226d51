// C ABI of libdmfe.so (include/dmfe.h): context life cycle, table hook, the north-star call
// dmfe_history_integrals and its host-buffer variant.  rk_step.cu / sparsify.cu hold the rest.
#include <math.h>
#include <stdlib.h>
#include <string.h>

#include <new>

#include "dmfe_internal.cuh"

extern "C" {

const char *dmfe_strerror(int code) {
  switch (code) {
    case DMFE_OK: return "ok";
    case DMFE_EINVAL: return "invalid argument";
    case DMFE_ECUDA: return "CUDA error (see dmfe_last_cuda_error)";
    case DMFE_ECAPACITY: return "history capacity exhausted";
    case DMFE_ESTEPMIN: return "step size below h_min";
    case DMFE_ENONFINITE: return "non-finite error estimate";
    case DMFE_ENOMEM: return "out of memory";
    case DMFE_ETOOLARGE: return "size beyond the static scratch (DMFE_STATIC_MAX_L, DMFE_STATIC_MAX_ROWS)";
    default: return "unknown error";
  }
}

int dmfe_last_cuda_error(const dmfe_ctx *ctx) { return ctx ? ctx->cuda_err : 0; }

static void free_all(dmfe_ctx *c) {
  cudaFree(c->theta);
  cudaFree(c->omega);
  cudaFree(c->nu);
  cudaFree(c->thnu);
  cudaFree(c->tab);
  cudaFree(c->blo);
  cudaFree(c->muw);
  cudaFree(c->win);
  cudaFree(c->rowtab);
  cudaFree(c->br);
  cudaFree(c->jtop);
  cudaFree(c->coefM);
  cudaFree(c->coefT);
  cudaFree(c->cur);
  cudaFree(c->scal);
  cudaFree(c->iscal);
  cudaFree(c->tgt_next);
  cudaFree(c->rk);
  cudaFree(c->dpk);
  cudaFree(c->eps_sp);
  cudaFree(c->keep);
  cudaFree(c->newidx);
  cudaFree(c->row_tmp);
  cudaFree(c->stage_t);
  cudaFree(c->stage_mu);
  cudaFree(c->stage_hist);
  cudaFree(c->stage_out);
  for (int k = 0; k < 2 * c->ev_made; ++k) cudaEventDestroy(c->ev[k]);
  if (c->h_scal) cudaFreeHost(c->h_scal);
  if (c->h_iscal) cudaFreeHost(c->h_iscal);
  if (c->step_exec) cudaGraphExecDestroy(c->step_exec);
  if (c->step_graph) cudaGraphDestroy(c->step_graph);
  cudaFree(c->steplog);
  cudaFree(c->adv_bar);
  if (c->h_steplog) cudaFreeHost(c->h_steplog);
}

int dmfe_create(const dmfe_params *params, const double *lambda, double T, dmfe_ctx **out) {
  if (!params || !lambda || !out) return DMFE_EINVAL;
  const dmfe_params &p = *params;
  if (p.stencil < 2 || p.stencil > 10 || (p.stencil & 1)) return DMFE_EINVAL;
  if (p.L < 2 * p.stencil || p.L > 65535) return DMFE_EINVAL;
  if (!(p.t_max > 2.718281828459045)) return DMFE_EINVAL;
  if (p.p_max < 2 || p.p_max > DMFE_PMAX_MAX) return DMFE_EINVAL;
  if (!(T >= 0.0) || !(p.beta0 >= 0.0) || !(p.tol >= 0.0)) return DMFE_EINVAL;
  if (p.values_only && p.log_r) return DMFE_EINVAL;
  dmfe_ctx *c = new (std::nothrow) dmfe_ctx;
  if (!c) return DMFE_ENOMEM;
  memset(c, 0, sizeof(*c));
  c->p = p;
  c->rowtab_dirty = 1;
  if (c->p.h_min <= 0.0) c->p.h_min = 1e-12;
  c->stream = (cudaStream_t)p.stream;
  ModelCoef &m = c->model;
  m.T = T;
  m.beta0 = p.beta0;
  m.pmax = p.p_max;
  for (int k = 0; k <= p.p_max; ++k) {
    m.c0[k] = 0.5 * lambda[k];
    m.c1[k] = (k + 1 <= p.p_max) ? 0.5 * (double)(k + 1) * lambda[k + 1] : 0.0;
    m.c2[k] = (k + 2 <= p.p_max) ? 0.5 * (double)((k + 2) * (k + 1)) * lambda[k + 2] : 0.0;
  }
  double f2_1 = 0.0;  // f''(1) for the step cap of Eq.(24)
  for (int k = 0; k <= p.p_max; ++k) f2_1 += m.c2[k];
  c->h_stab = (f2_1 > 0.0) ? 13.9 / (4.0 * sqrt(f2_1)) : INFINITY;
  {
    int dev = 0, v = 0;
    cudaGetDevice(&dev);
    c->sm_count = (cudaDeviceGetAttribute(&v, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && v > 0) ? v : 148;
    c->smem_max = (cudaDeviceGetAttribute(&v, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev) == cudaSuccess && v > 0)
                      ? v - 2048 : 46 * 1024;
  }
  int rc = dmfe_build_tables(c);
  const int L = p.L;
  if (rc == DMFE_OK) {
    cudaError_t e = cudaSuccess;
    if (e == cudaSuccess) e = cudaMalloc(&c->cur, sizeof(double2) * (size_t)L);
    if (e == cudaSuccess) e = cudaMalloc(&c->blo, sizeof(int32_t) * (size_t)L);
    if (e == cudaSuccess) e = cudaMalloc(&c->muw, sizeof(double2) * (size_t)L);
    if (e == cudaSuccess) e = cudaMalloc(&c->br, sizeof(int2) * (size_t)L);
    if (e == cudaSuccess) e = cudaMalloc(&c->jtop, sizeof(int32_t) * (size_t)L);
    if (e == cudaSuccess) e = cudaMalloc(&c->coefM, sizeof(double) * 8 * (size_t)L);
    if (e == cudaSuccess) e = cudaMalloc(&c->coefT, sizeof(double) * 16 * (size_t)L);
    if (e == cudaSuccess) e = cudaMalloc(&c->scal, sizeof(double) * SC_COUNT);
    if (e == cudaSuccess) e = cudaMalloc(&c->iscal, sizeof(int32_t) * IS_COUNT);
    if (e == cudaSuccess) e = cudaMalloc(&c->tgt_next, sizeof(int32_t) * 32);
    if (e == cudaSuccess) e = cudaMalloc(&c->rk, sizeof(double) * 8 * (size_t)L);
    if (e == cudaSuccess) e = cudaMallocHost(&c->h_scal, sizeof(double) * SC_COUNT);
    if (e == cudaSuccess) e = cudaMallocHost(&c->h_iscal, sizeof(int32_t) * IS_COUNT);
    if (e == cudaSuccess) e = cudaMemsetAsync(c->scal, 0, sizeof(double) * SC_COUNT, c->stream);
    if (e == cudaSuccess) e = cudaMemsetAsync(c->iscal, 0, sizeof(int32_t) * IS_COUNT, c->stream);
    if (e != cudaSuccess) {
      c->cuda_err = (int)e;
      rc = DMFE_ECUDA;
    }
  }
  if (rc != DMFE_OK) {
    free_all(c);
    delete c;
    return rc;
  }
  *out = c;
  return DMFE_OK;
}

int dmfe_destroy(dmfe_ctx *ctx) {
  if (!ctx) return DMFE_EINVAL;
  cudaStreamSynchronize(ctx->stream);
  free_all(ctx);
  delete ctx;
  return DMFE_OK;
}

int dmfe_get_tables(dmfe_ctx *ctx, double *theta, double *omega, double *nu, int32_t i0, int32_t n_targets,
                    int32_t *start, double *frac) {
  if (!ctx) return DMFE_EINVAL;
  const int L = ctx->p.L;
  const size_t vb = sizeof(double) * (size_t)L;
  if (theta) CUDA_TRY(ctx, cudaMemcpyAsync(theta, ctx->theta, vb, cudaMemcpyDeviceToHost, ctx->stream));
  if (omega) CUDA_TRY(ctx, cudaMemcpyAsync(omega, ctx->omega, vb, cudaMemcpyDeviceToHost, ctx->stream));
  if (nu) CUDA_TRY(ctx, cudaMemcpyAsync(nu, ctx->nu, vb, cudaMemcpyDeviceToHost, ctx->stream));
  if (start || frac) {
    if (i0 < 0 || n_targets < 1 || i0 + n_targets > L) return DMFE_EINVAL;
    const size_t plane = (size_t)L * (size_t)L, blk = (size_t)n_targets * (size_t)L;
    uint64_t *tmp = (uint64_t *)malloc(blk * sizeof(uint64_t));
    if (!tmp) return DMFE_ENOMEM;
    for (int k = 0; k < 3; ++k) {
      cudaError_t e = cudaMemcpyAsync(tmp, ctx->tab + k * plane + (size_t)i0 * L, blk * sizeof(uint64_t),
                                      cudaMemcpyDeviceToHost, ctx->stream);
      if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
      if (e != cudaSuccess) {
        free(tmp);
        ctx->cuda_err = (int)e;
        return DMFE_ECUDA;
      }
      for (size_t q = 0; q < blk; ++q) {  // decode: exactly the values the pair kernel uses
        int32_t st;
        double fr;
        dmfe_tab_decode(tmp[q], &st, &fr);
        if (start) start[k * blk + q] = st;
        if (frac) frac[k * blk + q] = fr;
      }
    }
    free(tmp);
  }
  CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
  return DMFE_OK;
}

int dmfe_history_integrals(dmfe_ctx *ctx, const dmfe_grid *g, const dmfe_rhs_out *out) {
  if (!ctx || !g || !out) return DMFE_EINVAL;
  if (g->n_rows < 2 || g->n_rows > g->n_cap || !g->t || !g->mu || !g->hist) return DMFE_EINVAL;
  if (ctx->p.values_only) return dmfe_launch_rhs_values(ctx, g->n_rows - 1, g->n_cap, g->t, g->mu, g->hist, out);
  return dmfe_launch_rhs(ctx, g->n_rows - 1, g->n_cap, g->t, g->mu, g->hist, out);
}

int dmfe_history_integrals_host(dmfe_ctx *ctx, int32_t n_rows, const double *t, const double *mu_hist,
                                const double *hist, double *d1C, double *d1R, double *mu, double *energy) {
  if (!ctx || n_rows < 2 || !t || !mu_hist || !hist) return DMFE_EINVAL;
  const int L = ctx->p.L;
  const size_t cell = ctx->p.values_only ? 2 : 4;  // doubles per history cell
  if (n_rows > ctx->stage_rows) {
    cudaFree(ctx->stage_t);
    cudaFree(ctx->stage_mu);
    cudaFree(ctx->stage_hist);
    cudaFree(ctx->stage_out);
    ctx->stage_t = ctx->stage_mu = ctx->stage_hist = ctx->stage_out = nullptr;
    ctx->stage_rows = 0;
    CUDA_TRY(ctx, cudaMalloc(&ctx->stage_t, sizeof(double) * (size_t)n_rows));
    CUDA_TRY(ctx, cudaMalloc(&ctx->stage_mu, sizeof(double) * (size_t)n_rows));
    CUDA_TRY(ctx, cudaMalloc(&ctx->stage_hist, sizeof(double) * cell * (size_t)L * (size_t)n_rows));
    CUDA_TRY(ctx, cudaMalloc(&ctx->stage_out, sizeof(double) * (2 * (size_t)L + 2)));
    ctx->stage_rows = n_rows;
  }
  cudaStream_t s = ctx->stream;
  CUDA_TRY(ctx, cudaMemcpyAsync(ctx->stage_t, t, sizeof(double) * (size_t)n_rows, cudaMemcpyHostToDevice, s));
  CUDA_TRY(ctx, cudaMemcpyAsync(ctx->stage_mu, mu_hist, sizeof(double) * (size_t)n_rows, cudaMemcpyHostToDevice, s));
  CUDA_TRY(ctx, cudaMemcpyAsync(ctx->stage_hist, hist, sizeof(double) * cell * (size_t)L * (size_t)n_rows,
                                cudaMemcpyHostToDevice, s));
  dmfe_rhs_out o;
  memset(&o, 0, sizeof(o));
  o.d1C = ctx->stage_out;
  o.d1R = ctx->stage_out + L;
  o.mu = ctx->stage_out + 2 * L;
  o.energy = ctx->stage_out + 2 * L + 1;
  const int rc = ctx->p.values_only
                     ? dmfe_launch_rhs_values(ctx, n_rows - 1, n_rows, ctx->stage_t, ctx->stage_mu, ctx->stage_hist, &o)
                     : dmfe_launch_rhs(ctx, n_rows - 1, n_rows, ctx->stage_t, ctx->stage_mu, ctx->stage_hist, &o);
  if (rc != DMFE_OK) return rc;
  if (d1C) CUDA_TRY(ctx, cudaMemcpyAsync(d1C, o.d1C, sizeof(double) * (size_t)L, cudaMemcpyDeviceToHost, s));
  if (d1R) CUDA_TRY(ctx, cudaMemcpyAsync(d1R, o.d1R, sizeof(double) * (size_t)L, cudaMemcpyDeviceToHost, s));
  if (mu) CUDA_TRY(ctx, cudaMemcpyAsync(mu, o.mu, sizeof(double), cudaMemcpyDeviceToHost, s));
  if (energy) CUDA_TRY(ctx, cudaMemcpyAsync(energy, o.energy, sizeof(double), cudaMemcpyDeviceToHost, s));
  CUDA_TRY(ctx, cudaStreamSynchronize(s));
  return DMFE_OK;
}

}  // extern "C"
