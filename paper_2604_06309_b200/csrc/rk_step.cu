// Device-resident SSPRK(10,4) step and error controller (Eq.(22), Eq.(25)).
// Low-storage form (refs [64,65]):
//   q1 = q2 = y;  5 x { q1 += h/6 F(q1) };  q2 = q2/25 + 9/25 q1;  q1 = 15 q2 - 5 q1;
//   4 x { q1 += h/6 F(q1) };  y+ = q2 + 3/5 q1 + h/10 F(q1)
// stage times t + c_k h, c = (0,1,2,3,4,2,3,4,5,6)/6; embedded 3rd-order weights
// bhat = (0,2/9,0,0,5/18,1/3,0,0,0,1/6) (reading G22); delta = h sum (b_k - bhat_k) F_k.
// The stage state is the value-only current row M = N+1 of the history (Eq.(22)); the first stage
// uses the derivative stored with row N.  One scalar record returns per step.
#include <math.h>
#include <string.h>

#include "dmfe_internal.cuh"

namespace {

__constant__ double c_stage_c[10] = {0.0,       1.0 / 6.0, 2.0 / 6.0, 3.0 / 6.0, 4.0 / 6.0,
                                     2.0 / 6.0, 3.0 / 6.0, 4.0 / 6.0, 5.0 / 6.0, 6.0 / 6.0};
__constant__ double c_b_minus_bhat[10] = {0.1 - 0.0, 0.1 - 2.0 / 9.0, 0.1 - 0.0, 0.1 - 0.0, 0.1 - 5.0 / 18.0,
                                          0.1 - 1.0 / 3.0, 0.1 - 0.0, 0.1 - 0.0, 0.1 - 0.0, 0.1 - 1.0 / 6.0};

// rk = [4][2L]: q1, q2, delta, F
__global__ void rk_stage_kernel(int k, int L, int N, double *__restrict__ hist, double *__restrict__ t,
                                double *__restrict__ rk, const double *__restrict__ scal) {
  const int n2 = 2 * L;
  const double h = scal[SC_H];
  const double t0 = t[N];
  double *q1 = rk, *q2 = rk + n2, *dl = rk + 2 * n2;
  const double *F = rk + 3 * n2;
  const int M = N + 1;
  const double hb = __dmul_rn(h, c_b_minus_bhat[k]);
  const double h6 = h / 6.0;
  for (int e = blockIdx.x * blockDim.x + threadIdx.x; e < n2; e += gridDim.x * blockDim.x) {
    const int l = e >> 1, comp = e & 1;
    const size_t cellN = ((size_t)N * L + l) * 4, cellM = ((size_t)M * L + l) * 4;
    double a, b, d, Fk;
    if (k == 0) {
      a = b = hist[cellN + 2 * comp];
      d = 0.0;
      Fk = hist[cellN + 2 * comp + 1];
    } else {
      a = q1[e];
      b = q2[e];
      d = dl[e];
      Fk = F[e];
    }
    d = __dadd_rn(d, __dmul_rn(hb, Fk));
    if (k < 9) {
      a = __dadd_rn(a, __dmul_rn(h6, Fk));
      if (k == 4) {
        b = __dadd_rn(b / 25.0, __dmul_rn(9.0 / 25.0, a));
        a = __dsub_rn(__dmul_rn(15.0, b), __dmul_rn(5.0, a));
      }
    } else {
      a = __dadd_rn(__dadd_rn(b, __dmul_rn(0.6, a)), __dmul_rn(__dmul_rn(0.1, h), Fk));
    }
    q1[e] = a;
    q2[e] = b;
    dl[e] = d;
    hist[cellM + 2 * comp] = a;  // stage state = value slots of the current row M
  }
  if (blockIdx.x == 0 && threadIdx.x == 0)
    t[M] = (k < 9) ? __dadd_rn(t0, __dmul_rn(c_stage_c[k + 1], h)) : __dadd_rn(t0, h);
}

// eps_RK = sum_i |delta C_i| + |delta R_i| (Eq.(25)) and the controller of PAPER.md:320 (G20).
__global__ void __launch_bounds__(1024) rk_finish_kernel(int L, int fixed_step, double tol, double cap,
                                                         const double *__restrict__ rk, double *__restrict__ scal,
                                                         int32_t *__restrict__ iscal) {
  __shared__ double sm[32];
  const int n2 = 2 * L;
  const double *dl = rk + 2 * n2;
  double acc = 0.0;
  for (int e = threadIdx.x; e < n2; e += blockDim.x) acc += fabs(dl[e]);
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = acc;
  __syncthreads();
  if (threadIdx.x != 0) return;
  double eps = 0.0;
  for (int w = 0; w < (int)(blockDim.x >> 5); ++w) eps += sm[w];
  double h = scal[SC_H];
  int accept = 1;
  if (!fixed_step) {
    if (!isfinite(eps) || eps > 2.0 * tol) {
      accept = 0;
      h = fmin(h / 2.0, cap);
    } else {
      if (eps > tol)
        h = 0.9 * h;
      else if (eps < tol / 2.0)
        h = 1.01 * h;
      h = fmin(h, cap);
    }
  }
  scal[SC_EPS] = eps;
  scal[SC_H] = h;
  iscal[IS_ACCEPT] = accept;
}

// store the ray derivative of the freshly appended row with the history
__global__ void store_derivative_kernel(int L, int M, double *__restrict__ hist, const double *__restrict__ F) {
  for (int l = blockIdx.x * blockDim.x + threadIdx.x; l < L; l += gridDim.x * blockDim.x) {
    const size_t cell = ((size_t)M * L + l) * 4;
    hist[cell + 1] = F[2 * l];
    hist[cell + 3] = F[2 * l + 1];
  }
}

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
  cudaStream_t s = ctx->stream;
  const int nb = (2 * L + 255) / 256;
  double *F = ctx->rk + 6 * (size_t)L;
  dmfe_rhs_out o;
  memset(&o, 0, sizeof(o));
  o.F = F;
  for (int k = 0; k < 10; ++k) {
    if (k > 0) {
      const int rc = dmfe_launch_rhs(ctx, M, st->n_cap, st->t, st->mu, st->hist, &o);
      if (rc != DMFE_OK) return rc;
      st->n_rhs++;
    }
    rk_stage_kernel<<<nb, 256, 0, s>>>(k, L, N, st->hist, st->t, ctx->rk, ctx->scal);
  }
  rk_finish_kernel<<<1, 1024, 0, s>>>(L, fixed_step, ctx->p.tol, ctx->h_stab, ctx->rk, ctx->scal, ctx->iscal);
  CUDA_TRY(ctx, cudaGetLastError());
  // the one record that returns to the host: {accept flag; eps_RK, next h}
  CUDA_TRY(ctx, cudaMemcpyAsync(ctx->h_iscal, ctx->iscal, sizeof(int32_t) * IS_COUNT, cudaMemcpyDeviceToHost, s));
  CUDA_TRY(ctx, cudaMemcpyAsync(ctx->h_scal, ctx->scal, sizeof(double) * SC_COUNT, cudaMemcpyDeviceToHost, s));
  CUDA_TRY(ctx, cudaStreamSynchronize(s));
  const int acc = ctx->h_iscal[IS_ACCEPT];
  st->eps_rk = ctx->h_scal[SC_EPS];
  st->h = ctx->h_scal[SC_H];
  if (accepted) *accepted = acc;
  if (acc) {
    // complete the appended row: its derivative, mu and E are stored with the history
    // (PAPER.md:230); this evaluation is stage 1 of the next step.
    o.mu = st->mu + M;
    o.energy = st->energy ? st->energy + M : nullptr;
    const int rc = dmfe_launch_rhs(ctx, M, st->n_cap, st->t, st->mu, st->hist, &o);
    if (rc != DMFE_OK) return rc;
    st->n_rhs++;
    store_derivative_kernel<<<(L + 255) / 256, 256, 0, s>>>(L, M, st->hist, F);
    CUDA_TRY(ctx, cudaGetLastError());
    st->n_rows = M + 1;
  } else {
    if (!isfinite(st->eps_rk) && st->n_rows == 1) return DMFE_ENONFINITE;
    st->n_rows = (st->n_rows - 10 > 1) ? st->n_rows - 10 : 1;  // revert the previous ten steps
  }
  if (!fixed_step && st->h < ctx->p.h_min) return DMFE_ESTEPMIN;
  return DMFE_OK;
}

}  // extern "C"
