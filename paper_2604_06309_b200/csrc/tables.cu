// t-independent tables of the history-integral path ("precomputed once"):
//   theta-grid Eq.(16), quadrature weights nu,
//   per-pair stencil start + fractional index coordinate for phi1, phi2, psi.
// Host part: O(L) work in long double.  Device part: the 3 L^2 pair tables.
#include <math.h>
#include <stdlib.h>

#include <vector>

#include "dmfe_internal.cuh"

// ---------------------------------------------------------------------------------------------
// gamma = -W_{-1}(-1/t_max), i.e. the root > 1 of  gamma - ln(gamma) = ln(t_max)
static long double solve_gamma(long double t_max) {
  const long double lt = logl(t_max);
  long double g = lt + logl(lt > 1.0L ? lt : 1.5L);
  for (int it = 0; it < 100; ++it) {
    const long double F = g - logl(g) - lt;
    const long double dF = 1.0L - 1.0L / g;
    const long double gn = g - F / dF;
    if (fabsl(gn - g) <= 1e-19L * fabsl(gn)) {
      g = gn;
      break;
    }
    g = gn;
  }
  return g;
}

// theta_i = [atan(e^{gamma y_i}) - atan(e^{-gamma})] / (A - B),  y_i = (2i-1-L)/(L-1), i = 1..L
// (Eq.(16) with alpha = 0 in the cancellation-free form, reading G7).  Lower half from
// atan a - atan b = atan((a-b)/(1+ab)); upper half by the symmetry theta_{L+1-i} = 1 - theta_i.
static void build_theta(int L, long double g, std::vector<double> &theta, std::vector<double> &omega) {
  const long double A = atanl(expl(g)), B = atanl(expl(-g));
  theta.assign(L, 0.0);
  omega.assign(L, 0.0);
  const int half = (L + 1) / 2;
  for (int i0 = 0; i0 < half; ++i0) {
    const long double y = (2.0L * (i0 + 1) - 1.0L - L) / (L - 1.0L);
    const long double num = expl(-g) * expm1l(g * (1.0L + y));
    const long double den = 1.0L + expl(g * y - g);
    theta[i0] = (double)(atanl(num / den) / (A - B));
  }
  for (int i0 = half; i0 < L; ++i0) theta[i0] = 1.0 - theta[L - 1 - i0];
  theta[0] = 0.0;
  theta[L - 1] = 1.0;
  for (int i0 = 0; i0 < L; ++i0) omega[i0] = theta[L - 1 - i0];
}

// ---------------------------------------------------------------------------------------------
// nu_j = integral over [0,1] of the j-th cardinal function of the interpolating spline of odd
// degree k with not-a-knot ends and data sites theta (reading G18).
// With B-spline collocation matrix A[i][c] = B_c(theta_i) and b_c = int B_c = (u_{c+k+1}-u_c)/(k+1):
// nu solves A^T nu = b.  Banded elimination with row pivoting, long double.
static void bspline_nonzero(const std::vector<long double> &u, int k, int span, long double x,
                            long double *N /*k+1*/) {
  // Cox-de Boor recursion for the k+1 basis functions that are non-zero on [u_span, u_span+1)
  long double left[16], right[16];
  N[0] = 1.0L;
  for (int d = 1; d <= k; ++d) {
    left[d] = x - u[span + 1 - d];
    right[d] = u[span + d] - x;
    long double saved = 0.0L;
    for (int r = 0; r < d; ++r) {
      const long double tmp = N[r] / (right[r + 1] + left[d - r]);
      N[r] = saved + right[r + 1] * tmp;
      saved = left[d - r] * tmp;
    }
    N[d] = saved;
  }
}

static int build_nu(const std::vector<double> &theta, int k, std::vector<double> &nu) {
  const int L = (int)theta.size();
  if (k < 1 || k > 9 || (k % 2) == 0 || L < k + 1) return DMFE_EINVAL;
  const int m = (k - 1) / 2;
  std::vector<long double> u;  // knot vector, L + k + 1 entries
  for (int a = 0; a <= k; ++a) u.push_back(theta[0]);
  for (int a = m + 1; a < L - m - 1; ++a) u.push_back(theta[a]);
  for (int a = 0; a <= k; ++a) u.push_back(theta[L - 1]);
  const int n = L;
  if ((int)u.size() != n + k + 1) return DMFE_EINVAL;
  // system matrix Mx = A^T stored by rows in windows: row r holds columns [r-kl, r+ku+kl]
  const int kl = k + 1, ku = k + 1, W = 2 * kl + ku + 1;
  std::vector<long double> w((size_t)n * W, 0.0L), rhs(n);
  auto at = [&](int r, int c) -> long double & { return w[(size_t)r * W + (c - (r - kl))]; };
  for (int i = 0; i < L; ++i) {
    const long double x = theta[i];
    int span;
    if (i == L - 1) {
      span = n - 1;  // last non-empty knot interval
    } else {
      span = k;
      while (span < n - 1 && u[span + 1] <= x) ++span;
    }
    long double N[16];
    bspline_nonzero(u, k, span, x, N);
    for (int a = 0; a <= k; ++a) {
      const int c = span - k + a;  // A[i][c] = N[a]  ->  Mx[c][i]
      if (i < c - kl || i > c + ku) return DMFE_EINVAL;  // band assumption violated
      at(c, i) = N[a];
    }
  }
  for (int c = 0; c < n; ++c) rhs[c] = (u[c + k + 1] - u[c]) / (long double)(k + 1);
  // elimination
  for (int c = 0; c < n; ++c) {
    int piv = c;
    long double best = fabsl(at(c, c));
    for (int r = c + 1; r <= c + kl && r < n; ++r) {
      const long double v = fabsl(at(r, c));
      if (v > best) best = v, piv = r;
    }
    if (best == 0.0L) return DMFE_EINVAL;
    const int cmax = (c + ku + kl < n - 1) ? c + ku + kl : n - 1;
    if (piv != c) {
      for (int cc = c; cc <= cmax; ++cc) {
        const long double tmp = at(c, cc);
        at(c, cc) = at(piv, cc);
        at(piv, cc) = tmp;
      }
      const long double tr = rhs[c];
      rhs[c] = rhs[piv];
      rhs[piv] = tr;
    }
    for (int r = c + 1; r <= c + kl && r < n; ++r) {
      const long double f = at(r, c) / at(c, c);
      if (f == 0.0L) continue;
      for (int cc = c; cc <= cmax; ++cc) at(r, cc) -= f * at(c, cc);
      rhs[r] -= f * rhs[c];
    }
  }
  nu.assign(n, 0.0);
  std::vector<long double> sol(n);
  for (int r = n - 1; r >= 0; --r) {
    long double acc = rhs[r];
    const int cmax = (r + ku + kl < n - 1) ? r + ku + kl : n - 1;
    for (int cc = r + 1; cc <= cmax; ++cc) acc -= at(r, cc) * sol[cc];
    sol[r] = acc / at(r, r);
    nu[r] = (double)sol[r];
  }
  return DMFE_OK;
}

// ---------------------------------------------------------------------------------------------
// Pair tables on the device.  For pair (i target, j node) and coordinate c in {phi1, phi2, psi}:
//   l*    = max{ l : theta_l <= c }  by comparison on the stored grid (bit-reproducible, G16)
//   start = clamp(l* - (s/2-1), 0, L-s)
//   X(c)  = (L-1)(1+y)/2,  y = +-ln tan(B + c'(A-B))/gamma with c' = c (c <= 1/2) or the
//           complement 1-c formed without cancellation (c > 1/2)   (G17)
//   frac  = X - start, stored packed with start in one 8-byte entry (dmfe_tab_encode)
__device__ __forceinline__ int cell_of(const double *__restrict__ theta, int L, double c) {
  int lo = 0, hi = L - 1;  // theta[lo] <= c always holds (theta[0] = 0 <= c)
  while (lo < hi) {
    const int mid = lo + ((hi - lo + 1) >> 1);
    if (theta[mid] <= c)
      lo = mid;
    else
      hi = mid - 1;
  }
  return lo;
}

__device__ __forceinline__ double index_coord(double c, double cbar, double A, double B, double g, int L) {
  const bool lower = c <= 0.5;
  const double arg = lower ? c : cbar;
  const double x = __dadd_rn(B, __dmul_rn(arg, __dsub_rn(A, B)));
  double y = log(tan(x)) / g;
  if (!lower) y = -y;
  return (double)(L - 1) * (1.0 + y) / 2.0;
}

__global__ void pair_tables_kernel(int L, int s, double A, double B, double g,
                                   const double *__restrict__ theta, const double *__restrict__ omega,
                                   uint64_t *__restrict__ tab) {
  const size_t plane = (size_t)L * (size_t)L;
  const int i = blockIdx.y;
  const double th_i = theta[i], om_i = omega[i];
  for (int j = blockIdx.x * blockDim.x + threadIdx.x; j < L; j += gridDim.x * blockDim.x) {
    const double th_j = theta[j], om_j = omega[j];
    double c[3], cb[3];
    c[0] = __dmul_rn(th_i, th_j);
    cb[0] = __dadd_rn(om_i, __dmul_rn(th_i, om_j));
    c[1] = __dadd_rn(th_i, __dmul_rn(om_i, th_j));
    cb[1] = __dmul_rn(om_i, om_j);
    if (c[1] > 0.0) {
      c[2] = __ddiv_rn(th_i, c[1]);
      cb[2] = __ddiv_rn(__dmul_rn(om_i, th_j), c[1]);
    } else {
      c[2] = 0.0;
      cb[2] = 1.0;
    }
    const size_t e = (size_t)i * (size_t)L + (size_t)j;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
      const int lstar = cell_of(theta, L, c[k]);
      int st = lstar - (s / 2 - 1);
      st = st < 0 ? 0 : (st > L - s ? L - s : st);
      const double X = index_coord(c[k], cb[k], A, B, g, L);
      tab[k * plane + e] = dmfe_tab_encode(st, X - (double)st);
    }
  }
}

int dmfe_build_tables(dmfe_ctx *ctx) {
  const int L = ctx->p.L, s = ctx->p.stencil;
  const long double g = solve_gamma((long double)ctx->p.t_max);
  ctx->gamma = (double)g;
  ctx->A = atan(exp(ctx->gamma));
  ctx->B = atan(exp(-ctx->gamma));
  std::vector<double> theta, omega, nu;
  build_theta(L, g, theta, omega);
  const int rc = build_nu(theta, ctx->p.quad_degree, nu);
  if (rc != DMFE_OK) return rc;
  const size_t vb = sizeof(double) * (size_t)L;
  const size_t plane = (size_t)L * (size_t)L;
  CUDA_TRY(ctx, cudaMalloc(&ctx->theta, vb));
  CUDA_TRY(ctx, cudaMalloc(&ctx->omega, vb));
  CUDA_TRY(ctx, cudaMalloc(&ctx->nu, vb));
  CUDA_TRY(ctx, cudaMalloc(&ctx->tab, 3 * plane * sizeof(uint64_t)));
  CUDA_TRY(ctx, cudaMemcpyAsync(ctx->theta, theta.data(), vb, cudaMemcpyHostToDevice, ctx->stream));
  CUDA_TRY(ctx, cudaMemcpyAsync(ctx->omega, omega.data(), vb, cudaMemcpyHostToDevice, ctx->stream));
  CUDA_TRY(ctx, cudaMemcpyAsync(ctx->nu, nu.data(), vb, cudaMemcpyHostToDevice, ctx->stream));
  // {theta_j, nu_j} interleaved: the pair kernel reads both with one 16-byte load
  std::vector<double> thnu(2 * (size_t)L);
  for (int j = 0; j < L; ++j) thnu[2 * j] = theta[j], thnu[2 * j + 1] = nu[j];
  CUDA_TRY(ctx, cudaMalloc(&ctx->thnu, 2 * vb));
  CUDA_TRY(ctx, cudaMemcpyAsync(ctx->thnu, thnu.data(), 2 * vb, cudaMemcpyHostToDevice, ctx->stream));
  const int nt = 256;
  int gx = (L + nt - 1) / nt;
  if (gx > 64) gx = 64;
  dim3 grid(gx, L);
  pair_tables_kernel<<<grid, nt, 0, ctx->stream>>>(L, s, ctx->A, ctx->B, ctx->gamma, ctx->theta,
                                                    ctx->omega, ctx->tab);
  CUDA_TRY(ctx, cudaGetLastError());
  CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));  // host vectors go out of scope
  return DMFE_OK;
}
