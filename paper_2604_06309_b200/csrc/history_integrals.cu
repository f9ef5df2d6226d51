// The per-RK-stage history integrals (section 3.3-3.4): for every target theta_i and
// quadrature node theta_j
//   A factors    C1,R1 = row M at phi1_ij, C2,R2 = row M at phi2_ij     (Eq.(18))
//   type-1       B1C,B1R = history at (theta_i t, theta_j): Hermite in t  (Eq.(19))
//   type-2       B2C,B2R = history at (phi2_ij t, psi_ij): theta-stencil, then Hermite in t after a
//                row search                                             (Eq.(20))
//   kernels      K = f''(C) R, D = f'(C)                                 (Eq.(10)-(11))
//   sums         eight nu-weighted sums over j                           (Eq.(21))
// and the O(L) parts: mu(t) Eq.(13), E(t) Eq.(14), the right-hand sides of Eq.(1) and of the
// second-argument equations (readings G1, G9, G10 in DESIGN.md), the ray derivative of Eq.(22).
//
// Mapping: persistent kernel, one CTA per SM.  The CTA's warps form groups of G warps; a group
// evaluates one target i at a time, lanes <-> adjacent nodes j (type-1 rows and the pair tables
// are read coalesced; the type-2 cells of adjacent lanes are neighbours in the packed history);
// the groups of one CTA take adjacent targets.  Every history cell {C,dC,R,dR} is one 256-bit
// load.  The per-call O(L + M) tables (current row, row table, bracket table) are copied into
// shared memory once per CTA when they fit.  fp64 throughout; no tensor cores: every "matrix"
// here is a gather.
//
// Launch 1 (prepare_kernel, O(L + M)): packs row M into {C,R} pairs, reduces mu and E, builds the
// per-call row table {t_n, 1/(t_{n+1}-t_n)} and the row bracket table blo[c] = n(theta_c t_M).
// Launch 2 (history_integrals_kernel): the L^2 pairs.  The row search of a pair is
// a bisection inside the bracket [blo[l*], blo[l*+1]] of the grid cell theta_l* <= phi2 < theta_l*+1
// that the phi2 stencil start already identifies -- same predicate and same result as a full
// bisection.  The loop over j is software-pipelined: while pair p is evaluated, the table entries
// of pair p+2 are in flight and the index stage of pair p+1 (bracket, bisection) has run.  It runs
// twice per target (DMFE_SPLIT): the type-1 half of Eq.(21) first, then the type-2 half; every sum
// receives its terms in the same order either way.
#include "dmfe_internal.cuh"

namespace {

#ifndef DMFE_THREADS
#define DMFE_THREADS 512
#endif
#ifndef DMFE_SPLIT
#define DMFE_SPLIT 1  // 1: type-1 and type-2 halves of the pair loop in two loops; 0: one fused loop (v6)
#endif
#ifndef DMFE_T1DEPTH
#define DMFE_T1DEPTH 1  // how many pairs ahead the type-1 loop requests its two cells
#endif
#ifndef DMFE_SYNC1
#define DMFE_SYNC1 0  // 1: CTA-wide barrier at the start of every round of targets
#endif
#ifndef DMFE_DIAG
#define DMFE_DIAG 0  // timing diagnostics only (wrong results): 1 = type-1 loop alone, 2 = type-2 loop alone
#endif
#ifndef DMFE_PRELOAD
#define DMFE_PRELOAD 2  // type-2 cell loads issued before the index stage of the next pair: 1 = all 2 S, 2 = the S of the lower row, 0 = none
#endif
constexpr int RHS_THREADS = DMFE_THREADS;
constexpr int PREP_THREADS = 1024;

struct RhsArgs {
  int32_t L, M;
  const double *theta, *omega;
  const double2 *thnu;
  const uint64_t *tab;
  const double *t, *mu_hist;
  const double4 *hist;
  const double2 *cur;
  const double2 *rowtab;
  const int32_t *blo;
  const double *scal;  // SC_MU, SC_E written by prepare_kernel
  int32_t G;           // warps per target group
  double4 *deriv_row;  // optional: row of the history whose derivative slots receive F
  dmfe_rhs_out out;
};

// Programmatic dependent launch (both kernels of a right-hand side are launched with
// cudaLaunchAttributeProgrammaticStreamSerialization): a kernel lets its successor in the stream
// start launching at once and itself waits, before it touches anything a predecessor wrote, until
// the predecessor grid has completed and its writes are visible.  The launch latency of each of
// the 20 kernels of an RK step is hidden behind the kernel before it.
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

__device__ __forceinline__ double4 ld_cell(const double4 *p) {
  double4 v;
  asm volatile("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];"
               : "=d"(v.x), "=d"(v.y), "=d"(v.z), "=d"(v.w)
               : "l"(p));
  return v;
}

// streamed once per call: keep it out of L1 and first in line for L2 eviction
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

// f'(q) and f''(q) with the polynomial degree fixed at compile time (PD = degree of f; the
// coefficient arrays are zero beyond p_max, so a model with p_max < PD evaluates exactly the same
// value); PD = 0 selects the run-time loop.
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
    if (__ldg(t + mid) <= tau)
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
  if (__ldg(t + g) <= tau) {
    lo = g;
    for (int st = 1;; st <<= 1) {
      const int nx = min(lo + st, top);
      if (nx == lo) return lo;  // lo == top
      if (__ldg(t + nx) <= tau) {
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
      if (__ldg(t + nx) <= tau) {
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

// ---------------------------------------------------------------------------------------------
// O(L + M) pre-pass, optionally preceded by one SSPRK(10,4) stage update that
// produces the row to be evaluated.  Low-storage form (refs [64,65]):
//   q1 = q2 = y;  5 x { q1 += h/6 F(q1) };  q2 = q2/25 + 9/25 q1;  q1 = 15 q2 - 5 q1;
//   4 x { q1 += h/6 F(q1) };  y+ = q2 + 3/5 q1 + h/10 F(q1)
// stage times t + c_k h, c = (0,1,2,3,4,2,3,4,5,6)/6; embedded 3rd-order weights
// bhat = (0,2/9,0,0,5/18,1/3,0,0,0,1/6) (reading G22); delta = h sum (b_k - bhat_k) F_k.
// Block 0: stage update of the 2L state entries (stage k = 9 also reduces eps_RK of Eq.(25) and
// runs the controller of PAPER.md:320, reading G20), then packs row M into {C,R} pairs and
// reduces mu(t) (Eq.(13)) and E(t) (Eq.(14)).  Blocks >= 1 (or block 0 too when launched alone):
// the per-call row table rowtab[n] = {t_n, 1/(t_{n+1} - t_n)}, n < M, and the bracket table
// blo[c] = n(fl(theta_c t_M)): for theta_a <= phi < theta_b rounding is monotone, so
// n(fl(phi t_M)) lies in [blo[a], blo[b]].  They compute t_M from the step scalars instead of
// reading t[M], which block 0 is writing.
__constant__ double c_stage_c[10] = {0.0,       1.0 / 6.0, 2.0 / 6.0, 3.0 / 6.0, 4.0 / 6.0,
                                     2.0 / 6.0, 3.0 / 6.0, 4.0 / 6.0, 5.0 / 6.0, 6.0 / 6.0};
__constant__ double c_b_minus_bhat[10] = {0.1 - 0.0, 0.1 - 2.0 / 9.0, 0.1 - 0.0, 0.1 - 0.0, 0.1 - 5.0 / 18.0,
                                          0.1 - 1.0 / 3.0, 0.1 - 0.0, 0.1 - 0.0, 0.1 - 0.0, 0.1 - 1.0 / 6.0};

__global__ void __launch_bounds__(PREP_THREADS) prepare_kernel(int L, int M, ModelCoef mc, dmfe_stage sg,
                                                               const double *__restrict__ theta,
                                                               const double *__restrict__ nu, const double *t,
                                                               const double4 *hist, double2 *__restrict__ cur,
                                                               double2 *__restrict__ rowtab,
                                                               int32_t *__restrict__ blo, double *scal) {
  __shared__ double sm[32], se[32];
  pdl_launch_dependents();
  pdl_wait();
  const int k = sg.k;
  // time of the row being evaluated.  The step size of stage 0 is the controller's proposal
  // (SC_HNEXT); block 0 latches it into SC_H, which stages 1..9 read.
  double tM, h = 0.0;
  if (k >= 0) {
    h = (k == 0) ? scal[SC_HNEXT] : scal[SC_H];
    const double t0 = t[sg.N];
    tM = (k < 9) ? __dadd_rn(t0, __dmul_rn(c_stage_c[k + 1], h)) : __dadd_rn(t0, h);
  } else {
    tM = t[M];
  }
  if (blockIdx.x > 0 || gridDim.x == 1) {
    const int nb = gridDim.x == 1 ? 1 : gridDim.x - 1;
    const int b = gridDim.x == 1 ? 0 : blockIdx.x - 1;
    for (int e = b * PREP_THREADS + threadIdx.x; e < M + L; e += nb * PREP_THREADS) {
      if (e < M) {
        const double tn = t[e];
        const double tn1 = (e + 1 == M) ? tM : t[e + 1];
        rowtab[e] = make_double2(tn, 1.0 / (tn1 - tn));
      } else {
        const int c = e - M;
        blo[c] = row_search_from(t, M - 1, blo[c], __dmul_rn(theta[c], tM));
      }
    }
    if (blockIdx.x > 0) return;
  }
  // ---- block 0: optional stage update, then pack row M and reduce mu, E; a thread owns the two
  // state entries {C, R} of a node l and keeps them in registers from the update to the sums ----
  const int N = sg.N;
  double2 *q1 = reinterpret_cast<double2 *>(sg.rk), *q2 = q1 + L, *dl = q2 + L;
  const double2 *F = dl + L;  // rk = [4][L]{C,R}: q1, q2, delta, F
  const double hb = (k >= 0) ? __dmul_rn(h, c_b_minus_bhat[k]) : 0.0;
  const double h6 = h / 6.0;
  double4 *rowM = const_cast<double4 *>(hist) + (size_t)M * (size_t)L;
  double eacc = 0.0, am = 0.0, ae = 0.0;
  __shared__ double s_c0;
  for (int l = threadIdx.x; l < L; l += blockDim.x) {
    double2 y;  // {C, R} of row M at node l
    if (k >= 0) {
      double2 a, b, d, Fk;
      if (k == 0) {
        const double4 c = hist[(size_t)N * (size_t)L + l];
        a = b = make_double2(c.x, c.z);
        d = make_double2(0.0, 0.0);
        Fk = make_double2(c.y, c.w);
      } else {
        a = q1[l];
        b = q2[l];
        d = dl[l];
        Fk = F[l];
      }
      auto upd = [&](double &av, double &bv, double &dv, double Fv) {
        dv = __dadd_rn(dv, __dmul_rn(hb, Fv));
        if (k < 9) {
          av = __dadd_rn(av, __dmul_rn(h6, Fv));
          if (k == 4) {
            bv = __dadd_rn(bv / 25.0, __dmul_rn(9.0 / 25.0, av));
            av = __dsub_rn(__dmul_rn(15.0, bv), __dmul_rn(5.0, av));
          }
        } else {
          av = __dadd_rn(__dadd_rn(bv, __dmul_rn(0.6, av)), __dmul_rn(__dmul_rn(0.1, h), Fv));
          eacc += fabs(dv);
        }
      };
      upd(a.x, b.x, d.x, Fk.x);
      upd(a.y, b.y, d.y, Fk.y);
      q1[l] = a;
      q2[l] = b;
      dl[l] = d;
      double *cell = reinterpret_cast<double *>(rowM + l);
      cell[0] = a.x;  // stage state = value slots of the current row M
      cell[2] = a.y;
      y = a;
    } else {
      const double4 c = rowM[l];
      y = make_double2(c.x, c.z);
    }
    cur[l] = y;
    if (l == 0) s_c0 = y.x;
    const double fp = horner(mc.c1, mc.pmax - 1, y.x), fpp = horner(mc.c2, mc.pmax - 2, y.x);
    const double nj = nu[l];
    am += nj * (fpp * y.y * y.x + fp * y.y);
    ae += nj * (fp * y.y);
  }
  if (k >= 0 && threadIdx.x == 0) {
    sg.t[M] = tM;
    if (k == 0) scal[SC_H] = h;
  }
  for (int o = 16; o > 0; o >>= 1) {
    am += __shfl_xor_sync(0xffffffffu, am, o);
    ae += __shfl_xor_sync(0xffffffffu, ae, o);
    eacc += __shfl_xor_sync(0xffffffffu, eacc, o);
  }
  const int w = threadIdx.x >> 5, nw = blockDim.x >> 5;
  __shared__ double sx[32];
  if ((threadIdx.x & 31) == 0) sm[w] = am, se[w] = ae, sx[w] = eacc;
  __syncthreads();
  if (threadIdx.x == 0) {
    double tm = 0.0, te = 0.0, eps = 0.0;
    for (int q = 0; q < nw; ++q) tm += sm[q], te += se[q], eps += sx[q];
    const double c0 = s_c0;
    scal[SC_MU] = mc.T + tM * tm + mc.beta0 * horner(mc.c1, mc.pmax - 1, c0) * c0;
    scal[SC_E] = -tM * te - mc.beta0 * horner(mc.c0, mc.pmax, c0);
    if (k == 9) {
      // eps_RK = sum_i |delta C_i| + |delta R_i| (Eq.(25)) and the controller (G20)
      double hn = h;
      int accept = 1;
      if (!sg.fixed_step) {
        if (!isfinite(eps) || eps > 2.0 * sg.tol) {
          accept = 0;
          hn = fmin(h / 2.0, sg.cap);
        } else {
          if (eps > sg.tol)
            hn = 0.9 * h;
          else if (eps < sg.tol / 2.0)
            hn = 1.01 * h;
          hn = fmin(hn, sg.cap);
        }
      }
      scal[SC_EPS] = eps;
      scal[SC_HNEXT] = hn;
      scal[SC_ACCEPT] = (double)accept;
      sg.iscal[IS_ACCEPT] = accept;
    }
  }
}

// Small per-call tables (current row, row table, bracket table) live in shared memory when they
// fit (SM = true): the gathers into them are the head of every pair's dependent load chain, and
// the history cells streaming through L1 (1 KB per warp-wide load) would otherwise evict them
// once per iteration.  SM = false reads the same arrays from global memory.
template <bool SM, class T>
__device__ __forceinline__ T ld_tab(const T *p) {
  if (SM) return *p;
  return __ldg(p);
}

// n = max{ n in [lo, hi] : rowtab[n].x <= tau }; requires t[lo] <= tau.
template <bool SM>
__device__ __forceinline__ int row_search_tab(const double2 *rowtab, int lo, int hi, double tau) {
  while (lo < hi) {
    const int mid = lo + ((hi - lo + 1) >> 1);
    if (ld_tab<SM>(&rowtab[mid].x) <= tau)
      lo = mid;
    else
      hi = mid - 1;
  }
  return lo;
}

// Index stage of one pair (the integer half of Eq.(20)): tau2 = fl(phi2 t_M) and its
// row n2, found by bisection inside the bracket of the grid cell of phi2.  l* = max{l : theta_l <=
// phi2} equals a2 + S/2 - 1 unless the stencil start was clamped, in which case l* lies in
// [0, S/2-1] (a2 = 0) or [L-S/2-1, L-1] (a2 = L-S).  n2 <= M-1, so the search runs on rowtab[0..M-1].
template <int S, bool SMT, bool SMR>
__device__ __forceinline__ int index_stage(const double2 *rowtab, const int32_t *blo, const double4 *hist, int L,
                                           double th_i, double om_i, double tM, double th_j, int a2, int a3,
                                           double *tau2_out) {
  const double phi2 = __dadd_rn(th_i, __dmul_rn(om_i, th_j));
  const double tau2 = __dmul_rn(phi2, tM);
  int clo = a2 + (S / 2 - 1), chi = clo + 1;
  if (a2 == 0) clo = 0, chi = S / 2;
  if (a2 == L - S) clo = (a2 == 0) ? 0 : L - S / 2 - 1, chi = L - 1;
  const int n2 = row_search_tab<SMR>(rowtab, ld_tab<SMT>(blo + clo), ld_tab<SMT>(blo + chi), tau2);
  *tau2_out = tau2;
  return n2;
}

__device__ __forceinline__ void group_barrier(int id, int nthreads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// Persistent kernel: one CTA per SM; the CTA's warps form groups of G warps, a group evaluates one
// target i at a time (lanes <-> adjacent nodes j), groups of one CTA take adjacent targets.
// SM: 0 = per-call tables read from global memory, 1 = cur and blo in shared memory, 2 = rowtab too
template <int S, int PD, int SM>
__global__ void __launch_bounds__(RHS_THREADS, 1) history_integrals_kernel(RhsArgs a, ModelCoef mc) {
  constexpr bool SMT = SM >= 1, SMR = SM == 2;
  extern __shared__ double4 smem_dyn[];
  pdl_launch_dependents();
  pdl_wait();
  const int L = a.L, M = a.M;
  const double2 *cur = a.cur;
  const double2 *rowtab = a.rowtab;
  const int32_t *blo = a.blo;
  if (SMT) {
    double2 *s_cur = reinterpret_cast<double2 *>(smem_dyn);
    double2 *s_row = s_cur + L;
    int32_t *s_blo = reinterpret_cast<int32_t *>(s_row + (SMR ? M : 0));
    for (int k = threadIdx.x; k < L; k += RHS_THREADS) s_cur[k] = a.cur[k], s_blo[k] = a.blo[k];
    if (SMR)
      for (int k = threadIdx.x; k < M; k += RHS_THREADS) s_row[k] = a.rowtab[k];
    __syncthreads();
    cur = s_cur, blo = s_blo;
    if (SMR) rowtab = s_row;
  }
  __shared__ double red[2][RHS_THREADS / 32][8];

  const int G = a.G;                 // warps per group (power of two, <= RHS_THREADS/32)
  const int TG = 32 * G;             // threads per group = stride of j
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int group = warp / G, wg = warp % G;
  const int ngroups = (RHS_THREADS / 32) / G;
  const int tig = wg * 32 + lane;    // thread index inside the group
  const size_t plane = (size_t)L * (size_t)L;
  const double tM = a.t[M];
  int parity = 0;

#if DMFE_SYNC1
  // the groups of a CTA take adjacent targets, whose type-1 rows mostly coincide or overlap (rows n1, n1+1 of
  // target i and n1' in {n1, n1+1} of target i+1): starting their type-1 loops together lets one group's
  // L1 fill serve the others
  for (int base = blockIdx.x * ngroups; base < L; base += gridDim.x * ngroups, parity ^= 1) {
    const int i = base + group;
    __syncthreads();
    if (i >= L) continue;
#else
  for (int i = blockIdx.x * ngroups + group; i < L; i += gridDim.x * ngroups, parity ^= 1) {
#endif
    const uint64_t *tab1 = a.tab + (size_t)i * (size_t)L, *tab2 = tab1 + plane, *tab3 = tab2 + plane;
    const double th_i = a.theta[i], om_i = a.omega[i];
    // type-1: one row search per target, tau = theta_i t  (Eq.(19)); blo[i] is exactly that row
    const double tau1 = __dmul_rn(th_i, tM);
    const int n1 = ld_tab<SMT>(blo + i);
    const bool top1 = (n1 + 1 == M);
    double h1[4];
    {
      const double2 rt = ld_tab<SMR>(rowtab + n1);
      t_weights(rt.x, rt.y, tau1, top1, h1);
    }
    const double4 *row1lo = a.hist + (size_t)n1 * (size_t)L;
    const double4 *row1hi = row1lo + L;

    double acc[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) acc[k] = 0.0;
    double b1c_first = 0.0;

#if DMFE_SPLIT
    // ---- loop fission: the type-1 half of Eq.(21) (S1, S3, S5, S6; coalesced rows n1, n1+1) runs in a
    // loop of its own, then the type-2 half (S2, S4, S7, S8; gathers).  Each sum sees its terms in the
    // same order as in the fused loop, so the results are bit-identical; the type-2 loop no longer
    // carries the type-1 table entries, weights and cells, which leaves registers to request all of
    // its 2 S cells at once. ----
    {
      uint64_t eA1 = 0, eB1 = 0;
      double nuA = 0.0, nuB = 0.0;
      double4 lo = make_double4(0, 0, 0, 0), hi = lo;
      int j = tig;
      if (j < L) {
        eA1 = ld_stream(tab1 + j);
        nuA = __ldg(&a.thnu[j].y);
        lo = ld_cell(row1lo + j);
        hi = ld_cell(row1hi + j);
      }
#if DMFE_T1DEPTH == 2
      double4 lon = make_double4(0, 0, 0, 0), hin = lon;
#endif
      if (j + TG < L) {
        eB1 = ld_stream(tab1 + j + TG);
        nuB = __ldg(&a.thnu[j + TG].y);
#if DMFE_T1DEPTH == 2
        lon = ld_cell(row1lo + j + TG);
        hin = ld_cell(row1hi + j + TG);
#endif
      }
      for (; j < L && DMFE_DIAG != 2; j += TG) {
        uint64_t eC1 = 0;
        double nuC = 0.0;
#if DMFE_T1DEPTH == 2
        double4 lo2 = make_double4(0, 0, 0, 0), hi2 = lo2;
        if (j + 2 * TG < L) {
          eC1 = ld_stream(tab1 + j + 2 * TG);
          nuC = __ldg(&a.thnu[j + 2 * TG].y);
          lo2 = ld_cell(row1lo + j + 2 * TG);
          hi2 = ld_cell(row1hi + j + 2 * TG);
        }
#else
        double4 lon = make_double4(0, 0, 0, 0), hin = lon;
        if (j + 2 * TG < L) {
          eC1 = ld_stream(tab1 + j + 2 * TG);
          nuC = __ldg(&a.thnu[j + 2 * TG].y);
        }
        if (j + TG < L) {
          lon = ld_cell(row1lo + j + TG);
          hin = ld_cell(row1hi + j + TG);
        }
#endif
        int a1;
        double u1;
        dmfe_tab_decode(eA1, &a1, &u1);
        double w[S];
        double C1 = 0.0, R1 = 0.0;
        lagrange_weights<S>(u1, w);
#pragma unroll
        for (int l = 0; l < S; ++l) {
          const double2 v = ld_tab<SMT>(cur + a1 + l);
          C1 = fma(w[l], v.x, C1);
          R1 = fma(w[l], v.y, R1);
        }
        if (top1) hi.y = 0.0, hi.w = 0.0;
        const double B1C = h1[0] * lo.x + h1[1] * lo.y + h1[2] * hi.x + h1[3] * hi.y;
        const double B1R = h1[0] * lo.z + h1[1] * lo.w + h1[2] * hi.z + h1[3] * hi.w;
        if (j == 0) b1c_first = B1C;
        const double nR1 = nuA * R1, nB1R = nuA * B1R;
        acc[0] = fma(f2<PD>(mc, C1) * nR1, B1C, acc[0]);    // S1: K(t,s) C(t',s)
        acc[2] = fma(f1<PD>(mc, C1), nB1R, acc[2]);         // S3: D(t,s) R(t',s)
        acc[4] = fma(f2<PD>(mc, B1C) * nB1R, C1, acc[4]);   // S5: K(t',s) C(t,s)
        acc[5] = fma(f1<PD>(mc, B1C), nR1, acc[5]);         // S6: D(t',s) R(t,s)
        eA1 = eB1, eB1 = eC1, nuA = nuB, nuB = nuC, lo = lon, hi = hin;
#if DMFE_T1DEPTH == 2
        lon = lo2, hin = hi2;
#endif
      }
      // the four type-1 sums leave the registers before the type-2 loop starts
#pragma unroll
      for (int k = 0; k < 8; ++k) {
        if (k == 1 || k == 3 || k >= 6) continue;
        double v = acc[k];
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) red[parity][warp][k] = v;
      }
    }
    {
      uint64_t eA2 = 0, eA3 = 0, eB2 = 0, eB3 = 0;
      double2 tnA = make_double2(0.0, 0.0), tnB = tnA;
      int n2A = 0;
      double tau2A = 0.0;
      int j = tig;
      if (j < L) {
        eA2 = ld_stream(tab2 + j);
        eA3 = ld_stream(tab3 + j);
        tnA = __ldg(a.thnu + j);
      }
      if (j + TG < L) {
        eB2 = ld_stream(tab2 + j + TG);
        eB3 = ld_stream(tab3 + j + TG);
        tnB = __ldg(a.thnu + j + TG);
      }
      if (j < L)
        n2A = index_stage<S, SMT, SMR>(rowtab, blo, a.hist, L, th_i, om_i, tM, tnA.x, (int)(eA2 >> 48),
                                       (int)(eA3 >> 48), &tau2A);
      for (; j < L && DMFE_DIAG != 1; j += TG) {
        uint64_t eC2 = 0, eC3 = 0;
        double2 tnC = make_double2(0.0, 0.0);
        if (j + 2 * TG < L) {
          eC2 = ld_stream(tab2 + j + 2 * TG);
          eC3 = ld_stream(tab3 + j + 2 * TG);
          tnC = __ldg(a.thnu + j + 2 * TG);
        }
        const int n2 = n2A;
        const double4 *p2 = a.hist + (size_t)n2 * (size_t)L + (int)(eA3 >> 48);
#if DMFE_PRELOAD == 1
        double4 x[S], y[S];
#pragma unroll
        for (int l = 0; l < S; ++l) {
          x[l] = ld_cell(p2 + l);
          y[l] = ld_cell(p2 + L + l);
        }
#elif DMFE_PRELOAD == 2  // lower row only
        double4 x[S];
#pragma unroll
        for (int l = 0; l < S; ++l) x[l] = ld_cell(p2 + l);
#endif
        int n2B = 0;
        double tau2B = 0.0;
        if (j + TG < L)
          n2B = index_stage<S, SMT, SMR>(rowtab, blo, a.hist, L, th_i, om_i, tM, tnB.x, (int)(eB2 >> 48),
                                         (int)(eB3 >> 48), &tau2B);
        const double nj = tnA.y;
        int a2, a3d;
        double u2, u3;
        dmfe_tab_decode(eA2, &a2, &u2);
        dmfe_tab_decode(eA3, &a3d, &u3);
        double w[S];
        double C2 = 0.0, R2 = 0.0;
        lagrange_weights<S>(u2, w);
#pragma unroll
        for (int l = 0; l < S; ++l) {
          const double2 v = ld_tab<SMT>(cur + a2 + l);
          C2 = fma(w[l], v.x, C2);
          R2 = fma(w[l], v.y, R2);
        }
        if (a.out.rows2) a.out.rows2[(size_t)i * (size_t)L + (size_t)j] = n2;
        const bool top2 = (n2 + 1 == M);
        double h2[4];
        {
          const double2 rt = ld_tab<SMR>(rowtab + n2);
          t_weights(rt.x, rt.y, tau2A, top2, h2);
        }
        lagrange_weights<S>(u3, w);
        double cl = 0.0, dcl = 0.0, rl = 0.0, drl = 0.0, cu = 0.0, dcu = 0.0, ru = 0.0, dru = 0.0;
#pragma unroll
        for (int l = 0; l < S; ++l) {
#if DMFE_PRELOAD == 1
          const double4 xl = x[l], yl = y[l];
#elif DMFE_PRELOAD == 2
          const double4 xl = x[l], yl = ld_cell(p2 + L + l);
#else
          const double4 xl = ld_cell(p2 + l), yl = ld_cell(p2 + L + l);
#endif
          cl = fma(w[l], xl.x, cl);
          dcl = fma(w[l], xl.y, dcl);
          rl = fma(w[l], xl.z, rl);
          drl = fma(w[l], xl.w, drl);
          cu = fma(w[l], yl.x, cu);
          dcu = fma(w[l], yl.y, dcu);
          ru = fma(w[l], yl.z, ru);
          dru = fma(w[l], yl.w, dru);
        }
        if (top2) dcu = 0.0, dru = 0.0;
        const double B2C = h2[0] * cl + h2[1] * dcl + h2[2] * cu + h2[3] * dcu;
        const double B2R = h2[0] * rl + h2[1] * drl + h2[2] * ru + h2[3] * dru;
        const double nR2 = nj * R2;
        const double K2 = f2<PD>(mc, C2) * nR2;
        acc[1] = fma(K2, B2C, acc[1]);                            // S2: K(t,s) C(s,t')
        acc[3] = fma(K2, B2R, acc[3]);                            // S4: K(t,s) R(s,t')
        acc[6] = fma(f1<PD>(mc, B2C), nR2, acc[6]);               // S7: D(s,t') R(t,s)
        acc[7] = fma(nR2, f2<PD>(mc, B2C) * B2R, acc[7]);         // S8: R(t,s) K(s,t')
        eA2 = eB2, eA3 = eB3, tnA = tnB;
        eB2 = eC2, eB3 = eC3, tnB = tnC;
        n2A = n2B;
        tau2A = tau2B;
      }
    }
#else
    // ---- software pipeline over this thread's pairs p = j, j + TG, j + 2 TG, ... ----
    //   eA*: table entries of the pair being evaluated; n2A / tau2A: its row and time
    //   eB*, thB: table entries and theta_j of the next pair; eC*, thC: in flight for the one after
    uint64_t eA1 = 0, eA2 = 0, eA3 = 0, eB1 = 0, eB2 = 0, eB3 = 0;
    double2 tnA = make_double2(0.0, 0.0), tnB = tnA;
    int n2A = 0;
    double tau2A = 0.0;
    int j = tig;
    if (j < L) {
      eA1 = ld_stream(tab1 + j);
      eA2 = ld_stream(tab2 + j);
      eA3 = ld_stream(tab3 + j);
      tnA = __ldg(a.thnu + j);
    }
    if (j + TG < L) {
      eB1 = ld_stream(tab1 + j + TG);
      eB2 = ld_stream(tab2 + j + TG);
      eB3 = ld_stream(tab3 + j + TG);
      tnB = __ldg(a.thnu + j + TG);
    }
    if (j < L)
      n2A = index_stage<S, SMT, SMR>(rowtab, blo, a.hist, L, th_i, om_i, tM, tnA.x, (int)(eA2 >> 48), (int)(eA3 >> 48),
                               &tau2A);
    for (; j < L; j += TG) {
      uint64_t eC1 = 0, eC2 = 0, eC3 = 0;
      double2 tnC = make_double2(0.0, 0.0);
      if (j + 2 * TG < L) {
        eC1 = ld_stream(tab1 + j + 2 * TG);
        eC2 = ld_stream(tab2 + j + 2 * TG);
        eC3 = ld_stream(tab3 + j + 2 * TG);
        tnC = __ldg(a.thnu + j + 2 * TG);
      }
      // type-1 cells and type-2 cells of this pair: issue all ten 32-byte loads up front
      const double4 lo = ld_cell(row1lo + j);
      double4 hi = ld_cell(row1hi + j);
      const int n2 = n2A;
      const int a3 = (int)(eA3 >> 48);
      const double4 *p2 = a.hist + (size_t)n2 * (size_t)L + a3;
#if DMFE_PRELOAD
      double4 x[S], y[S];
#pragma unroll
      for (int l = 0; l < S; ++l) {
        x[l] = ld_cell(p2 + l);
        y[l] = ld_cell(p2 + L + l);
      }
#endif
      // index stage of the next pair (shared-memory chain) while those loads are in flight
      int n2B = 0;
      double tau2B = 0.0;
      if (j + TG < L)
        n2B = index_stage<S, SMT, SMR>(rowtab, blo, a.hist, L, th_i, om_i, tM, tnB.x, (int)(eB2 >> 48),
                                 (int)(eB3 >> 48), &tau2B);

      const double nj = tnA.y;
      int a1, a2, a3d;
      double u1, u2, u3;
      dmfe_tab_decode(eA1, &a1, &u1);
      dmfe_tab_decode(eA2, &a2, &u2);
      dmfe_tab_decode(eA3, &a3d, &u3);
      double w[S];
      // ---- A factors at phi1 (Eq.(18)) and the type-1 lookup (Eq.(19)): sums S1, S3, S5, S6 ----
      {
        double C1 = 0.0, R1 = 0.0;
        lagrange_weights<S>(u1, w);
#pragma unroll
        for (int l = 0; l < S; ++l) {
          const double2 v = ld_tab<SMT>(cur + a1 + l);
          C1 = fma(w[l], v.x, C1);
          R1 = fma(w[l], v.y, R1);
        }
        if (top1) hi.y = 0.0, hi.w = 0.0;
        const double B1C = h1[0] * lo.x + h1[1] * lo.y + h1[2] * hi.x + h1[3] * hi.y;
        const double B1R = h1[0] * lo.z + h1[1] * lo.w + h1[2] * hi.z + h1[3] * hi.w;
        if (j == 0) b1c_first = B1C;
        // every term carries nu_j and exactly one of R1, B1R: fold nu_j into those two
        const double nR1 = nj * R1, nB1R = nj * B1R;
        acc[0] = fma(f2<PD>(mc, C1) * nR1, B1C, acc[0]);    // S1: K(t,s) C(t',s)
        acc[2] = fma(f1<PD>(mc, C1), nB1R, acc[2]);         // S3: D(t,s) R(t',s)
        acc[4] = fma(f2<PD>(mc, B1C) * nB1R, C1, acc[4]);   // S5: K(t',s) C(t,s)
        acc[5] = fma(f1<PD>(mc, B1C), nR1, acc[5]);         // S6: D(t',s) R(t,s)
      }
      // ---- A factors at phi2 (Eq.(18)) ----
      double C2 = 0.0, R2 = 0.0;
      lagrange_weights<S>(u2, w);
#pragma unroll
      for (int l = 0; l < S; ++l) {
        const double2 v = ld_tab<SMT>(cur + a2 + l);
        C2 = fma(w[l], v.x, C2);
        R2 = fma(w[l], v.y, R2);
      }
      // ---- type-2 lookup (Eq.(20)) in the rows n2, n2+1 found by the index stage ----
      if (a.out.rows2) a.out.rows2[(size_t)i * (size_t)L + (size_t)j] = n2;
      const bool top2 = (n2 + 1 == M);
      double h2[4];
      {
        const double2 rt = ld_tab<SMR>(rowtab + n2);
        t_weights(rt.x, rt.y, tau2A, top2, h2);
      }
      // theta-stencil first, then t
      lagrange_weights<S>(u3, w);
      double cl = 0.0, dcl = 0.0, rl = 0.0, drl = 0.0, cu = 0.0, dcu = 0.0, ru = 0.0, dru = 0.0;
#pragma unroll
      for (int l = 0; l < S; ++l) {
#if DMFE_PRELOAD
        const double4 xl = x[l], yl = y[l];
#else
        const double4 xl = ld_cell(p2 + l), yl = ld_cell(p2 + L + l);
#endif
        cl = fma(w[l], xl.x, cl);
        dcl = fma(w[l], xl.y, dcl);
        rl = fma(w[l], xl.z, rl);
        drl = fma(w[l], xl.w, drl);
        cu = fma(w[l], yl.x, cu);
        dcu = fma(w[l], yl.y, dcu);
        ru = fma(w[l], yl.z, ru);
        dru = fma(w[l], yl.w, dru);
      }
      if (top2) dcu = 0.0, dru = 0.0;
      const double B2C = h2[0] * cl + h2[1] * dcl + h2[2] * cu + h2[3] * dcu;
      const double B2R = h2[0] * rl + h2[1] * drl + h2[2] * ru + h2[3] * dru;
      // ---- kernel functions (Eq.(10)-(11)) and the type-2 terms (Eq.(21)) ----
      const double nR2 = nj * R2;
      const double K2 = f2<PD>(mc, C2) * nR2;
      acc[1] = fma(K2, B2C, acc[1]);                            // S2: K(t,s) C(s,t')
      acc[3] = fma(K2, B2R, acc[3]);                            // S4: K(t,s) R(s,t')
      acc[6] = fma(f1<PD>(mc, B2C), nR2, acc[6]);               // S7: D(s,t') R(t,s)
      acc[7] = fma(nR2, f2<PD>(mc, B2C) * B2R, acc[7]);         // S8: R(t,s) K(s,t')
      // ---- rotate the pipeline ----
      eA1 = eB1, eA2 = eB2, eA3 = eB3, tnA = tnB;
      eB1 = eC1, eB2 = eC2, eB3 = eC3, tnB = tnC;
      n2A = n2B;
      tau2A = tau2B;
    }
#endif
    // ---- reduction over j: shuffle within the warp, fixed order across the warps of the group ----
#if DMFE_SPLIT
    constexpr bool kViaRed = true;  // the type-1 sums are already in red[parity][warp]
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      if (!(k == 1 || k == 3 || k >= 6)) continue;
      for (int o = 16; o > 0; o >>= 1) acc[k] += __shfl_xor_sync(0xffffffffu, acc[k], o);
      if (lane == 0) red[parity][warp][k] = acc[k];
    }
    if (G > 1) group_barrier(1 + group, TG);
#else
    constexpr bool kViaRed = false;
#pragma unroll
    for (int k = 0; k < 8; ++k)
      for (int o = 16; o > 0; o >>= 1) acc[k] += __shfl_xor_sync(0xffffffffu, acc[k], o);
    if (G > 1) {
      if (lane == 0) {
#pragma unroll
        for (int k = 0; k < 8; ++k) red[parity][warp][k] = acc[k];
      }
      group_barrier(1 + group, TG);  // red[parity] is reused two targets later: one barrier suffices
    }
#endif
    if (tig != 0) continue;

    double Sd[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      double s = acc[k];
      if (G > 1 || kViaRed) {
        s = 0.0;
        for (int w = 0; w < G; ++w) s += red[parity][group * G + w][k];
      }
      Sd[k] = s;
      if (a.out.sums) a.out.sums[(size_t)k * L + i] = s;
    }
    if (a.out.rows1) a.out.rows1[i] = n1;

    // ---- combine (Eq.(1), second-argument equations, Eq.(22)) ----
    const double mu = a.scal[SC_MU];
    // mu(theta_i t): local 4-point Lagrange in t over rows k..k+3 (reading G11), mu_M = mu
    const int npts = (M + 1 < 4) ? M + 1 : 4;
    int k0 = n1 - 1;
    if (k0 > M + 1 - npts) k0 = M + 1 - npts;
    if (k0 < 0) k0 = 0;
    double mu_p = 0.0;
    for (int p = 0; p < npts; ++p) {
      double wgt = 1.0;
      for (int q = 0; q < npts; ++q)
        if (q != p) wgt *= (tau1 - a.t[k0 + q]) / (a.t[k0 + p] - a.t[k0 + q]);
      const double mv = (k0 + p == M) ? mu : a.mu_hist[k0 + p];
      mu_p += wgt * mv;
    }
    const double2 ci = ld_tab<SMT>(cur + i), c0 = ld_tab<SMT>(cur);
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
    if (a.deriv_row) {  // the ray derivative is stored with the appended row
      double *cell = reinterpret_cast<double *>(a.deriv_row + i);
      cell[1] = FC;
      cell[3] = FR;
    }
    if (i == 0) {
      if (a.out.mu) a.out.mu[0] = mu;
      if (a.out.energy) a.out.energy[0] = a.scal[SC_E];
    }
  }
}

}  // namespace

// M = index of the current row; its time t[M] is read on the device (the RK step keeps t there).
int dmfe_launch_rhs(dmfe_ctx *ctx, int32_t M, int32_t n_cap, const double *t, const double *mu_hist,
                    const double *hist, const dmfe_rhs_out *out, const dmfe_stage *stage, double *deriv_row) {
  const int L = ctx->p.L;
  if (M > ctx->rowtab_cap) {  // per-call row table: sized by the caller's capacity, grown on demand
    const int cap = n_cap > M ? n_cap : M;
    CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    cudaFree(ctx->rowtab);
    ctx->rowtab = nullptr;
    ctx->rowtab_cap = 0;
    CUDA_TRY(ctx, cudaMalloc(&ctx->rowtab, sizeof(double2) * (size_t)cap));
    ctx->rowtab_cap = cap;
  }
  int pb = 1 + (M + L + PREP_THREADS - 1) / PREP_THREADS;
  if (pb > 17) pb = 17;
  dmfe_stage sg;
  if (stage) {
    sg = *stage;
  } else {
    memset(&sg, 0, sizeof(sg));
    sg.k = -1;
  }
  CUDA_TRY(ctx, launch_pdl(prepare_kernel, pb, PREP_THREADS, 0, ctx->stream, L, M, ctx->model, sg, ctx->theta,
                           ctx->nu, t, (const double4 *)hist, ctx->cur, ctx->rowtab, ctx->blo, ctx->scal));
  if (stage && stage->after_prepass) CUDA_TRY(ctx, cudaEventRecord(stage->after_prepass, ctx->stream));
  RhsArgs a;
  a.L = L;
  a.M = M;
  a.theta = ctx->theta;
  a.omega = ctx->omega;
  a.thnu = ctx->thnu;
  a.tab = ctx->tab;
  a.t = t;
  a.mu_hist = mu_hist;
  a.hist = (const double4 *)hist;
  a.cur = ctx->cur;
  a.rowtab = ctx->rowtab;
  a.blo = ctx->blo;
  a.scal = ctx->scal;
  a.deriv_row = reinterpret_cast<double4 *>(deriv_row);
  a.out = *out;
  const bool timed = ctx->timing_on && ctx->ev_n < DMFE_EV_RING;
  if (timed) {
    if (ctx->ev_n >= ctx->ev_made) {
      CUDA_TRY(ctx, cudaEventCreate(&ctx->ev[2 * ctx->ev_made]));
      CUDA_TRY(ctx, cudaEventCreate(&ctx->ev[2 * ctx->ev_made + 1]));
      ctx->ev_made++;
    }
    CUDA_TRY(ctx, cudaEventRecord(ctx->ev[2 * ctx->ev_n], ctx->stream));
  }
  // the polynomial degree of f is a compile-time constant for p_max <= 4 (the paper's models
  // p = 2, 3, 2+4, 3+4, 2+3+4); larger p_max (3+9) takes the run-time Horner loop
  const int pd = ctx->model.pmax <= 3 ? 3 : (ctx->model.pmax == 4 ? 4 : 0);
  // persistent grid: one CTA per SM.  Warps per target group: as few as keeps every warp slot of
  // the GPU busy (L * G >= resident warps), so that a group's loop over j is as long as possible.
  const int warps_cta = RHS_THREADS / 32;
  // G = warps per target group.  As few as possible (long loops over j), subject to (a) every warp
  // slot of the GPU has work (L * G >= resident warps) and (b) the number of rounds
  // ceil(L / (groups per CTA * SMs)) wastes less than 3 % of the last round (else the best G).
  int G = 1;
  {
    double best = -1.0;
    for (int g = 1; g <= warps_cta && g <= 16; g *= 2) {
      if (warps_cta % g) continue;
      const long long slots = (long long)ctx->sm_count * (warps_cta / g);
      const long long rounds = ((long long)L + slots - 1) / slots;
      const double eff = (double)L / (double)(rounds * slots);
      if (eff > best + 1e-9) best = eff, G = g;
      if (eff >= 0.97) break;
    }
  }
  a.G = G;
  const int ngroups = warps_cta / G;
  int grid = (L + ngroups - 1) / ngroups;
  if (grid > ctx->sm_count) grid = ctx->sm_count;
  // shared-memory copies of cur [L] double2 and blo [L] int32 when they fit, and of rowtab [M]
  // double2 too when that fits and a CTA has enough pairs to amortise copying M entries
  const size_t smem1 = 20 * (size_t)L, smem2 = smem1 + 16 * (size_t)M;
  const long long pairs_cta = (long long)L * L / grid;
  const int mode = (smem2 <= (size_t)ctx->smem_max && 2LL * M <= pairs_cta) ? 2
                   : (smem1 <= (size_t)ctx->smem_max ? 1 : 0);
  const size_t smem = mode == 2 ? smem2 : (mode == 1 ? smem1 : 0);
#define DMFE_LAUNCH_M(S_, PD_, SM_)                                                                     \
  do {                                                                                                  \
    auto kfn = history_integrals_kernel<S_, PD_, SM_>;                                                  \
    if (smem + 4096 > 48 * 1024)                                                                        \
      CUDA_TRY(ctx, cudaFuncSetAttribute(kfn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)); \
    CUDA_TRY(ctx, launch_pdl(kfn, grid, RHS_THREADS, smem, ctx->stream, a, ctx->model));                \
  } while (0)
#define DMFE_LAUNCH(S_, PD_)       \
  do {                             \
    if (mode == 2)                 \
      DMFE_LAUNCH_M(S_, PD_, 2);   \
    else if (mode == 1)            \
      DMFE_LAUNCH_M(S_, PD_, 1);   \
    else                           \
      DMFE_LAUNCH_M(S_, PD_, 0);   \
  } while (0)
#define DMFE_LAUNCH_S(S_)        \
  do {                           \
    if (pd == 3)                 \
      DMFE_LAUNCH(S_, 3);        \
    else if (pd == 4)            \
      DMFE_LAUNCH(S_, 4);        \
    else                         \
      DMFE_LAUNCH(S_, 0);        \
  } while (0)
  switch (ctx->p.stencil) {
    case 2: DMFE_LAUNCH_S(2); break;
    case 4: DMFE_LAUNCH_S(4); break;
    case 6: DMFE_LAUNCH_S(6); break;
    case 8: DMFE_LAUNCH_S(8); break;
    case 10: DMFE_LAUNCH_S(10); break;
    default: return DMFE_EINVAL;
  }
#undef DMFE_LAUNCH_S
#undef DMFE_LAUNCH
#undef DMFE_LAUNCH_M
  if (timed) {
    CUDA_TRY(ctx, cudaEventRecord(ctx->ev[2 * ctx->ev_n + 1], ctx->stream));
    ctx->ev_n++;
  }
  CUDA_TRY(ctx, cudaGetLastError());
  return DMFE_OK;
}
