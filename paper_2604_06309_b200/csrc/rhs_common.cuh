// Device helpers shared by the kernels of one right-hand-side evaluation (history_integrals.cu,
// pairs_generic.cuh, pairs_s4.cuh).  Not part of the C ABI.
#pragma once
#include "dmfe_internal.cuh"

namespace dmfe_rhs {

// Programmatic dependent launch (all kernels of a right-hand side are launched with
// cudaLaunchAttributeProgrammaticStreamSerialization): a kernel lets its successor in the stream
// start launching at once and itself waits, before it touches anything a predecessor wrote, until
// the predecessor grid has completed and its writes are visible.  The launch latency of each of
// the kernels of an RK step is hidden behind the kernel before it.
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }

template <class... KArgs, class... Args>
cudaError_t launch_pdl(void (*kernel)(KArgs...), int grid, int block, size_t smem, cudaStream_t stream,
                       Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(grid);
  cfg.blockDim = dim3(block);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = stream;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

// One history cell {C, dC, R, dR} = one 256-bit load.  Plain ld.global (not .nc): the evaluation
// that completes an appended row writes derivative slots of row M while other CTAs of the same
// grid may still read its value slots, and the per-call tables are written by the predecessor
// grid; both are outside the read-only contract of the non-coherent path.
// Not volatile: the compiler is free to schedule the load (its address always depends on data read
// after griddepcontrol.wait, so it cannot move above that).
__device__ __forceinline__ double4 ld_cell(const double4 *p) {
  double4 v;
  asm("ld.global.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(v.x), "=d"(v.y), "=d"(v.z), "=d"(v.w) : "l"(p));
  return v;
}

// the t-independent pair tables: streamed once per call, never written after dmfe_create: keep them
// out of L1 and first in line for L2 eviction
__device__ __forceinline__ uint64_t ld_stream(const uint64_t *p) {
  unsigned long long v;
  asm volatile("ld.global.nc.L1::no_allocate.b64 %0, [%1];" : "=l"(v) : "l"(p));
  return (uint64_t)v;
}

__device__ __forceinline__ double horner(const double *c, int deg, double q) {
  double acc = c[deg];
  for (int k = deg - 1; k >= 0; --k) acc = fma(acc, q, c[k]);
  return acc;
}

// f'(q) and f''(q) (Eq.(10)-(11)) with the polynomial degree fixed at compile
// time (PD = degree of f; the coefficient arrays are zero beyond p_max, so a model with
// p_max < PD evaluates exactly the same value); PD = 0 selects the run-time loop.
template <int PD>
__device__ __forceinline__ double f1(const ModelCoef &mc, double q) {
  if (PD == 0) return horner(mc.c1, mc.pmax - 1, q);
  double acc = mc.c1[PD - 1];
#pragma unroll
  for (int k = PD - 2; k >= 0; --k) acc = fma(acc, q, mc.c1[k]);
  return acc;
}
template <int PD>
__device__ __forceinline__ double f2(const ModelCoef &mc, double q) {
  if (PD == 0) return horner(mc.c2, mc.pmax - 2, q);
  double acc = mc.c2[PD - 2];
#pragma unroll
  for (int k = PD - 3; k >= 0; --k) acc = fma(acc, q, mc.c2[k]);
  return acc;
}

// Lagrange cardinal weights on the integer nodes 0..S-1 at u (PAPER.md:236 index interpolation):
// w_l = prod_{m<l}(u-m) * prod_{m>l}(u-m) / prod_{m!=l}(l-m)
template <int S>
__device__ __forceinline__ void lagrange_weights(double u, double (&w)[S]) {
  double d[S], pre[S], suf[S];
#pragma unroll
  for (int m = 0; m < S; ++m) d[m] = u - (double)m;
  pre[0] = 1.0;
#pragma unroll
  for (int m = 1; m < S; ++m) pre[m] = pre[m - 1] * d[m - 1];
  suf[S - 1] = 1.0;
#pragma unroll
  for (int m = S - 2; m >= 0; --m) suf[m] = suf[m + 1] * d[m + 1];
#pragma unroll
  for (int l = 0; l < S; ++l) {
    double den = 1.0;
#pragma unroll
    for (int m = 0; m < S; ++m)
      if (m != l) den *= (double)(l - m);
    w[l] = pre[l] * suf[l] * (1.0 / den);  // 1/den folds to a compile-time constant
  }
}

// S = 4: with A = u(u-3) and B = (u-1)(u-2) = A + 2 the four cardinal cubics are
//   w0 = B(3-u)/6, w1 = A(u-2)/2, w2 = A(1-u)/2, w3 = B u/6      (10 FP64 instructions)
template <>
__device__ __forceinline__ void lagrange_weights<4>(double u, double (&w)[4]) {
  const double A = u * (u - 3.0);
  const double B = A + 2.0;
  const double hA = 0.5 * A;
  const double t6 = u * (1.0 / 6.0);
  w[3] = B * t6;
  w[0] = fma(-B, t6, 0.5 * B);
  w[1] = fma(hA, u, -A);
  w[2] = fma(-hA, u, hA);
}

// n = max{ n in [lo, hi] : t[n] <= tau }; requires t[lo] <= tau.
__device__ __forceinline__ int row_search(const double *__restrict__ t, int lo, int hi, double tau) {
  while (lo < hi) {
    const int mid = lo + ((hi - lo + 1) >> 1);
    if (t[mid] <= tau)
      lo = mid;
    else
      hi = mid - 1;
  }
  return lo;
}

// The same n, found from a guess g (any value): bracket by doubling steps away from g, then bisect.
// prepare_kernel passes the value the previous evaluation left in the table: successive stages
// differ by a fraction of a step, so the bracket closes after one or two loads instead of log2 M.
__device__ __forceinline__ int row_search_from(const double *__restrict__ t, int top, int g, double tau) {
  g = min(max(g, 0), top);
  int lo, hi;
  if (t[g] <= tau) {
    lo = g;
    for (int st = 1;; st <<= 1) {
      const int nx = min(lo + st, top);
      if (nx == lo) return lo;  // lo == top
      if (t[nx] <= tau) {
        lo = nx;
      } else {
        hi = nx - 1;
        break;
      }
    }
  } else {  // g >= 1 here because t[0] = 0 <= tau
    hi = g - 1;
    lo = 0;
    for (int st = 1;; st <<= 1) {
      const int nx = g - st;
      if (nx <= 0) break;
      if (t[nx] <= tau) {
        lo = nx;
        break;
      }
      hi = nx - 1;
    }
  }
  return row_search(t, lo, hi, tau);
}

// weights of the local interpolant in t between rows n and n+1 (PAPER.md:260 cubic Hermite);
// quadratic (value, slope, value) when the upper row is the current row M (reading G12).  With
// d = tau - t_n, u = d/D, v = u - 1:
//   h00 = 2u^3-3u^2+1, h10 = u v^2 D = d v^2, h01 = 1-h00, h11 = u^2 v D = d u v;  top: 1-u^2, -d v, u^2, 0
// rD = 1/D comes from the per-call row table, so a pair costs no division.
__device__ __forceinline__ void t_weights(double tn, double rD, double tau, bool top, double (&h)[4]) {
  const double d = tau - tn;
  const double u = d * rD;
  const double v = u - 1.0;
  const double u2 = u * u;
  const double dv = d * v;
  if (top) {
    h[0] = 1.0 - u2;
    h[1] = -dv;
    h[2] = u2;
    h[3] = 0.0;
  } else {
    h[0] = fma(u2, fma(2.0, u, -3.0), 1.0);
    h[1] = dv * v;
    h[2] = 1.0 - h[0];
    h[3] = dv * u;
  }
}

__device__ __forceinline__ void group_barrier(int id, int nthreads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// arguments of the pair kernels
struct RhsArgs {
  int32_t L, M;
  const double *theta, *omega;
  const double2 *thnu;  // {theta_j, nu_j}
  const double *nu;
  const uint64_t *tab;  // [3][L][L] packed pair tables
  const double *t, *mu_hist;
  const double4 *hist;
  // per-call tables written by prepare_kernel
  const double2 *cur;     // [L] {C, R} of row M
  const double2 *rowtab;  // [M] {t_n, 1/(t_{n+1} - t_n)}
  const int32_t *blo;     // [L] blo[c] = n(theta_c t_M)
  const double2 *muw;     // [L] mu(theta_c t_M) = muw.x + muw.y mu(t_M)  (reading G11)
  const int2 *br;         // [L-3] S = 4: row bracket of the grid cell of phi2, indexed by the stencil start
  const int32_t *jtop;    // [L]   S = 4: first node j of target i whose type-2 interval is the top one
  const double4 *coefM;   // [L-3][2] S = 4: centred cubics of {C, R} of row M per stencil start
  const double4 *coefT;   // [L-3][4] S = 4: centred cubics of {C, dC, R, dR} of row M-1
  const double *scal;     // SC_MU, SC_E written by prepare_kernel
  int32_t G;              // warps per target group
  int32_t *tgt_next;      // S = 4: next target to hand out (groups fetch their targets after the first round)
  double4 *deriv_row;     // optional: row of the history whose derivative slots receive F
  // device-resident step (rk_step.cu): M is read from dev_rows[0]; when `complete` is set the
  // evaluation completes the appended row M: mu_w[M], energy_w[M] and the derivative slots of hist_w[M]
  const int32_t *dev_rows;
  const int32_t *dev_status;
  int32_t complete;
  double *mu_w, *energy_w;
  double4 *hist_w;
  dmfe_rhs_out out;
};

// current row of a launch: the host's value or, in a device-resident step, the device's
__device__ __forceinline__ int current_row(const RhsArgs &a) { return a.dev_rows ? a.dev_rows[0] : a.M; }
__device__ __forceinline__ bool batch_stopped(const RhsArgs &a) { return a.dev_status && a.dev_status[0] != 0; }

// Reduction over j of a group's eight sums and the O(1) work per target: Eq.(1), the
// second-argument equations (readings G9, G10) and the ray derivative of
// Eq.(22).  red[warp][k] holds the warp sums; called by the group's first thread after the barrier.
template <int PD, bool SMT>
__device__ __forceinline__ void combine_target(const RhsArgs &a, const ModelCoef &mc, int i, int n1, double th_i,
                                               double om_i, double tM, double tau1, double b1c_first,
                                               const double (*red)[8], int w0, int G, const double2 *cur, int M) {
  const int L = a.L;
  double Sd[8];
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    double s = 0.0;
    for (int w = 0; w < G; ++w) s += red[w0 + w][k];
    Sd[k] = s;
    if (a.out.sums) a.out.sums[(size_t)k * L + i] = s;
  }
  if (a.out.rows1) a.out.rows1[i] = n1;
  const double mu = a.scal[SC_MU];
  // mu(theta_i t): local 4-point Lagrange in t (reading G11); the pre-pass formed the part that comes
  // from the stored rows and the weight of the current row's mu
  const double2 mw = a.muw[i];
  const double mu_p = fma(mw.y, mu, mw.x);
  const double2 ci = SMT ? cur[i] : a.cur[i], c0 = SMT ? cur[0] : a.cur[0];
  const double fc = mc.beta0 * f1<PD>(mc, c0.x) * b1c_first;
  const double fc2 = mc.beta0 * f1<PD>(mc, b1c_first) * c0.x;
  const double d1C = -mu * ci.x + tM * (th_i * Sd[0] + om_i * Sd[1] + th_i * Sd[2]) + fc;
  const double d1R = -mu * ci.y + tM * (om_i * Sd[3]);
  const double d2C = -mu_p * ci.x + tM * (th_i * Sd[4] + th_i * Sd[5] + om_i * Sd[6]) + 2.0 * mc.T * ci.y + fc2;
  const double d2R = mu_p * ci.y - tM * (om_i * Sd[7]);
  if (a.out.d1C) a.out.d1C[i] = d1C;
  if (a.out.d1R) a.out.d1R[i] = d1R;
  if (a.out.d2C) a.out.d2C[i] = d2C;
  if (a.out.d2R) a.out.d2R[i] = d2R;
  const double FC = d1C + th_i * d2C, FR = d1R + th_i * d2R;
  if (a.out.F) {
    a.out.F[2 * i] = FC;
    a.out.F[2 * i + 1] = FR;
  }
  double4 *drow = a.complete ? a.hist_w + (size_t)M * (size_t)L : a.deriv_row;
  if (drow) {  // the ray derivative is stored with the appended row
    double *cell = reinterpret_cast<double *>(drow + i);
    cell[1] = FC;
    cell[3] = FR;
  }
  if (i == 0) {
    if (a.out.mu) a.out.mu[0] = mu;
    if (a.out.energy) a.out.energy[0] = a.scal[SC_E];
    if (a.complete) {
      a.mu_w[M] = mu;
      if (a.energy_w) a.energy_w[M] = a.scal[SC_E];
    }
  }
}

constexpr int RHS_THREADS = 512;  // pairs_generic.cuh
constexpr int S4_THREADS = 512;   // pairs_s4.cuh

}  // namespace dmfe_rhs

// launchers of the pair kernels (pairs_generic.cu, pairs_s4.cu); grid = CTAs, a.G = warps per target
int dmfe_launch_pairs_generic(dmfe_ctx *ctx, const dmfe_rhs::RhsArgs &a, int grid);
int dmfe_launch_pairs_s4(dmfe_ctx *ctx, const dmfe_rhs::RhsArgs &a, int grid);
