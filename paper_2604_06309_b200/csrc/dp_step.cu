// Device-resident Dormand-Prince 5(4) step ("Dynamite ... uses the Dormand-Prince
// method [63] at short times"; "initialized with the Dormand-Prince method until the time step
// grows sufficiently to reach the boundary of its stability domain"), the start-up integrator
// before SSPRK(10,4).  Textbook tableau of ref. [63]; row 7 of A equals the fifth-order weights
// (FSAL): the evaluation of the new point is both the derivative stored with the appended row
// and the seventh stage of the error estimate delta = h sum_j (b_j - bhat_j) k_j.
// Stage i: y_i = y_N + h sum_{j<i} a_ij k_j (terms in the order j = 1, 2, ..., separate roundings,
// zero coefficients skipped), written to the value slots of the current row M = N+1 (Eq.(22)).
// A step is 6 x (stage kernel + pre-pass + pair kernel) + one decision kernel and one 128-byte
// record back to the host.  Only the first steps of a run use it: clarity over launch count.
#include <math.h>
#include <string.h>

#include "dmfe_internal.cuh"

namespace {

__constant__ double c_dp_c[7] = {0.0, 1.0 / 5.0, 3.0 / 10.0, 4.0 / 5.0, 8.0 / 9.0, 1.0, 1.0};
__constant__ double c_dp_a[7][6] = {
    {0.0, 0.0, 0.0, 0.0, 0.0, 0.0},
    {1.0 / 5.0, 0.0, 0.0, 0.0, 0.0, 0.0},
    {3.0 / 40.0, 9.0 / 40.0, 0.0, 0.0, 0.0, 0.0},
    {44.0 / 45.0, -56.0 / 15.0, 32.0 / 9.0, 0.0, 0.0, 0.0},
    {19372.0 / 6561.0, -25360.0 / 2187.0, 64448.0 / 6561.0, -212.0 / 729.0, 0.0, 0.0},
    {9017.0 / 3168.0, -355.0 / 33.0, 46732.0 / 5247.0, 49.0 / 176.0, -5103.0 / 18656.0, 0.0},
    {35.0 / 384.0, 0.0, 500.0 / 1113.0, 125.0 / 192.0, -2187.0 / 6784.0, 11.0 / 84.0}};
// b_j - bhat_j, j = 1..7 (b_7 = 0)
__constant__ double c_dp_e[7] = {35.0 / 384.0 - 5179.0 / 57600.0,
                                 0.0 - 0.0,
                                 500.0 / 1113.0 - 7571.0 / 16695.0,
                                 125.0 / 192.0 - 393.0 / 640.0,
                                 -2187.0 / 6784.0 - -92097.0 / 339200.0,
                                 11.0 / 84.0 - 187.0 / 2100.0,
                                 0.0 - 1.0 / 40.0};

// dpk = [6][L]{C,R}: k_1 .. k_6; F = [L]{C,R}: output of the evaluation that has just run
// Stage s = 0..5 stores k_{s+1} (s = 0: the derivative kept with row N) and writes y_{s+2}.
__global__ void dp_stage_kernel(int s, int L, int N, double4 *__restrict__ hist, double *__restrict__ t,
                                double2 *__restrict__ dpk, const double2 *__restrict__ F,
                                double *__restrict__ scal) {
  const double h = (s == 0) ? scal[SC_HNEXT] : scal[SC_H];
  const int M = N + 1, i = s + 1;  // row of the tableau that is formed
  for (int l = blockIdx.x * blockDim.x + threadIdx.x; l < L; l += gridDim.x * blockDim.x) {
    const double4 c = hist[(size_t)N * (size_t)L + l];
    const double2 ks = (s == 0) ? make_double2(c.y, c.w) : F[l];
    dpk[(size_t)s * L + l] = ks;
    double ax = 0.0, ay = 0.0;
    bool first = true;
    for (int j = 0; j <= s; ++j) {
      const double a = c_dp_a[i][j];
      if (a == 0.0) continue;
      const double2 kj = (j == s) ? ks : dpk[(size_t)j * L + l];
      const double tx = __dmul_rn(a, kj.x), ty = __dmul_rn(a, kj.y);
      ax = first ? tx : __dadd_rn(ax, tx);
      ay = first ? ty : __dadd_rn(ay, ty);
      first = false;
    }
    double *cell = reinterpret_cast<double *>(hist + (size_t)M * (size_t)L + l);
    cell[0] = __dadd_rn(c.x, __dmul_rn(h, ax));  // stage state = value slots of the current row M
    cell[2] = __dadd_rn(c.z, __dmul_rn(h, ay));
  }
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    t[M] = __dadd_rn(t[N], __dmul_rn(c_dp_c[i], h));
    if (s == 0) scal[SC_H] = h;
  }
}

// eps_RK = sum_i |delta C_i| + |delta R_i| (Eq.(25)) from k_1..k_6 and k_7 = F, and the controller
// of PAPER.md:320 (reading G20).  No step cap: the caller leaves Dormand-Prince when the step
// reaches the stability boundary (reading G21).
__global__ void __launch_bounds__(1024) dp_decide_kernel(int L, int fixed_step, double tol,
                                                         const double2 *__restrict__ dpk,
                                                         const double2 *__restrict__ F, double *__restrict__ scal,
                                                         int32_t *__restrict__ iscal) {
  __shared__ double sm[32];
  const double h = scal[SC_H];
  double eacc = 0.0;
  for (int l = threadIdx.x; l < L; l += blockDim.x) {
    double ax = 0.0, ay = 0.0;
    bool first = true;
    for (int j = 0; j < 7; ++j) {
      const double e = c_dp_e[j];
      if (e == 0.0) continue;
      const double2 kj = (j == 6) ? F[l] : dpk[(size_t)j * L + l];
      const double tx = __dmul_rn(e, kj.x), ty = __dmul_rn(e, kj.y);
      ax = first ? tx : __dadd_rn(ax, tx);
      ay = first ? ty : __dadd_rn(ay, ty);
      first = false;
    }
    eacc += fabs(__dmul_rn(h, ax)) + fabs(__dmul_rn(h, ay));
  }
  for (int o = 16; o > 0; o >>= 1) eacc += __shfl_xor_sync(0xffffffffu, eacc, o);
  if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = eacc;
  __syncthreads();
  if (threadIdx.x != 0) return;
  double eps = 0.0;
  for (int w = 0; w < (int)(blockDim.x >> 5); ++w) eps += sm[w];
  double hn = h;
  int accept = 1;
  if (!fixed_step) {
    if (!isfinite(eps) || eps > 2.0 * tol) {
      accept = 0;
      hn = h / 2.0;
    } else if (eps > tol) {
      hn = 0.9 * h;
    } else if (eps < tol / 2.0) {
      hn = 1.01 * h;
    }
  }
  scal[SC_EPS] = eps;
  scal[SC_HNEXT] = hn;
  scal[SC_ACCEPT] = (double)accept;
  iscal[IS_ACCEPT] = accept;
}

__global__ void set_step_kernel(double *__restrict__ scal, double h) {
  scal[SC_HNEXT] = h;
  scal[SC_H] = h;
}

}  // namespace

extern "C" {

int dmfe_set_step_size(dmfe_ctx *ctx, dmfe_state *st, double h) {
  if (!ctx || !st || !(h > 0.0)) return DMFE_EINVAL;
  set_step_kernel<<<1, 1, 0, ctx->stream>>>(ctx->scal, h);
  CUDA_TRY(ctx, cudaGetLastError());
  st->h = h;
  return DMFE_OK;
}

int dmfe_dp_step(dmfe_ctx *ctx, dmfe_state *st, int32_t fixed_step, int32_t *accepted) {
  if (ctx && ctx->p.values_only) return DMFE_EINVAL;  // the integrator keeps the Hermite history
  if (!ctx || !st || !st->t || !st->mu || !st->hist) return DMFE_EINVAL;
  if (st->n_rows < 1) return DMFE_EINVAL;
  if (st->n_rows + 1 > st->n_cap) return DMFE_ECAPACITY;
  const int L = ctx->p.L;
  const int N = st->n_rows - 1, M = N + 1;
  cudaStream_t s = ctx->stream;
  if (!ctx->dpk) CUDA_TRY(ctx, cudaMalloc(&ctx->dpk, sizeof(double) * 14 * (size_t)L));  // k_1..k_6, F
  double2 *dpk = reinterpret_cast<double2 *>(ctx->dpk);
  double *F = ctx->dpk + 12 * (size_t)L;
  const int nb = (L + 255) / 256;
  for (int k = 0; k < 6; ++k) {
    dp_stage_kernel<<<nb, 256, 0, s>>>(k, L, N, reinterpret_cast<double4 *>(st->hist), st->t, dpk,
                                       reinterpret_cast<const double2 *>(F), ctx->scal);
    CUDA_TRY(ctx, cudaGetLastError());
    dmfe_rhs_out o;
    memset(&o, 0, sizeof(o));
    o.F = F;
    double *deriv_row = nullptr;
    if (k == 5) {  // y_7 = the new point: its evaluation completes the appended row (FSAL)
      o.mu = st->mu + M;
      o.energy = st->energy ? st->energy + M : nullptr;
      deriv_row = st->hist + (size_t)M * (size_t)L * 4;
    }
    const int rc = dmfe_launch_rhs(ctx, M, st->n_cap, st->t, st->mu, st->hist, &o, nullptr, deriv_row);
    if (rc != DMFE_OK) return rc;
    st->n_rhs++;
  }
  dp_decide_kernel<<<1, 1024, 0, s>>>(L, fixed_step, ctx->p.tol, dpk, reinterpret_cast<const double2 *>(F),
                                      ctx->scal, ctx->iscal);
  CUDA_TRY(ctx, cudaGetLastError());
  // the one record that returns to the host: {accept flag, eps_RK, next h}
  CUDA_TRY(ctx, cudaMemcpyAsync(ctx->h_scal, ctx->scal, sizeof(double) * SC_COUNT, cudaMemcpyDeviceToHost, s));
  CUDA_TRY(ctx, cudaStreamSynchronize(s));
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
