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
// Launch 1 (prepare_kernel, O(L + M)): optional RK stage update, packs row M into {C,R} pairs,
// reduces mu and E, builds the per-call tables (row table, row brackets and, for S = 4, the
// coefficient forms of rows M and M-1 and the first top-interval node of every target).
// Launch 2: the L^2 pairs -- pairs_s4.cuh for the 4-point stencil, pairs_generic.cuh otherwise.
#include "rhs_common.cuh"

namespace {
using namespace dmfe_rhs;

constexpr int PREP_THREADS = 1024;
constexpr int PREP_SCUR = 2048;  // block 0 keeps the packed current row in shared memory up to this L

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

// S = 4 only (s4 != 0): the tables of pairs_s4.cuh.  A 4-point index-Lagrange interpolant through
// y_0..y_3 on the nodes a..a+3 is the cubic d0 + d1 v + d2 v^2 + d3 v^3 in v = u - 3/2:
//   d0 = (9 (y1+y2) - (y0+y3))/16, d1 = (27 (y2-y1) - (y3-y0))/24, d2 = ((y0+y3) - (y1+y2))/4,
//   d3 = ((y3-y0) - 3 (y2-y1))/6
struct PrepS4 {
  int32_t on;
  int2 *br;          // [L-3] {blo[clo(a)], blo[chi(a)]}: row bracket of the grid cell of phi2 by stencil start
  int32_t *jtop;     // [L]   first j with fl(fl(theta_i + fl(omega_i theta_j)) t_M) >= t_{M-1}
  double4 *coefM;    // [L-3][2] cubics of {C, R} of row M
  double4 *coefT;    // [L-3][4] cubics of {C, dC, R, dR} of row M-1
  const double *omega;
  int32_t *tgt_next;   // work counter of the pair kernel: reset to the first target its groups fetch dynamically
  int32_t tgt_first;
};

__device__ __forceinline__ double4 centred_cubic(double y0, double y1, double y2, double y3) {
  const double a = y1 + y2, b = y0 + y3, c = y2 - y1, e = y3 - y0;
  return make_double4((9.0 * a - b) * (1.0 / 16.0), (27.0 * c - e) * (1.0 / 24.0), (b - a) * 0.25,
                      (e - 3.0 * c) * (1.0 / 6.0));
}

__global__ void __launch_bounds__(PREP_THREADS) prepare_kernel(int L, int M, ModelCoef mc, dmfe_stage sg,
                                                               const double *__restrict__ theta,
                                                               const double *__restrict__ nu, const double *t,
                                                               const double4 *hist, double2 *__restrict__ cur,
                                                               double2 *__restrict__ rowtab,
                                                               int32_t *__restrict__ blo, double *scal,
                                                               const double *__restrict__ mu_hist,
                                                               double2 *__restrict__ muw, PrepS4 s4) {  // M, sg: by value, adjusted below
  __shared__ double sm[32], se[32];
  pdl_launch_dependents();
  pdl_wait();
  if (sg.dev_rows) {  // device-resident step: the row count lives on the device (rk_step.cu)
    if (sg.iscal[IS_STATUS] != 0) return;
    M = sg.dev_rows[0];
    sg.N = M - 1;
  }
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
    // jtop [L] and coefT [L-3]; a host-driven evaluation (no stage update: row M is in the history) also forms
    // coefM [L-3] here, off block 0's path
    const int n_extra = s4.on ? 2 * L - 3 + (k < 0 ? L - 3 : 0) : 0;
    // rows below rt0 already have their final row-table entries (device-resident steps: only the
    // entries at the end of the history change between evaluations; rk_step.cu keeps the count)
    const int rt0 = sg.dev_rows ? min(max(sg.iscal[IS_RTVALID], 0), M - 1) : 0;
    const int n_rt = M - rt0;
    for (int e0 = b * PREP_THREADS + threadIdx.x; e0 < n_rt + L + n_extra; e0 += nb * PREP_THREADS) {
      const int e = e0 + rt0;  // item index as if every row-table entry were rebuilt
      if (e < M) {
        const double tn = t[e];
        const double tn1 = (e + 1 == M) ? tM : t[e + 1];
        rowtab[e] = make_double2(tn, 1.0 / (tn1 - tn));
      } else if (e < M + L) {
        const int c = e - M;
        const double tau1 = __dmul_rn(theta[c], tM);
        const int n = row_search_from(t, M - 1, blo[c], tau1);
        blo[c] = n;
        {
          // mu(theta_c t_M): local 4-point Lagrange in t over rows k0..k0+3 (reading G11); the last point
          // may be the current row M, whose mu is being reduced by block 0: keep its weight apart
          const int npts = (M + 1 < 4) ? M + 1 : 4;
          int k0 = n - 1;
          if (k0 > M + 1 - npts) k0 = M + 1 - npts;
          if (k0 < 0) k0 = 0;
          double tq[4];
          for (int q = 0; q < npts; ++q) tq[q] = (k0 + q == M) ? tM : t[k0 + q];
          double part = 0.0, wM = 0.0;
          for (int p = 0; p < npts; ++p) {
            double wgt = 1.0;
            for (int q = 0; q < npts; ++q)
              if (q != p) wgt *= (tau1 - tq[q]) / (tq[p] - tq[q]);
            if (k0 + p == M)
              wM = wgt;
            else
              part += wgt * mu_hist[k0 + p];
          }
          muw[c] = make_double2(part, wM);
        }
        if (s4.on) {
          // l* = a + 1 for an unclamped start a (S/2 - 1 = 1): clo(a) = a + 1, chi(a) = a + 2; clamped
          // starts: a = 0 -> l* in {0, 1}: [blo[0], blo[2]]; a = L-4 -> l* in {L-3 .. L-1}: [blo[L-3], blo[L-1]]
          if (c >= 2 && c <= L - 3) s4.br[c - 1].x = n;
          if (c >= 2 && c <= L - 3) s4.br[c - 2].y = n;
          if (c == 0) s4.br[0].x = n;
          if (c == L - 1) s4.br[L - 4].y = n;
        }
      } else if (e < M + 2 * L) {
        const int i = e - M - L;
        const double th_i = theta[i], om_i = s4.omega[i], tTop = t[M - 1];
        int lo = 0, hi = L;  // first j in [0, L] with tau2(i, j) >= t_{M-1} (tau2 is monotone in j)
        while (lo < hi) {
          const int mid = (lo + hi) >> 1;
          const double tau2 = __dmul_rn(__dadd_rn(th_i, __dmul_rn(om_i, theta[mid])), tM);
          if (tau2 >= tTop)
            hi = mid;
          else
            lo = mid + 1;
        }
        s4.jtop[i] = lo;
      } else if (e >= M + 3 * L - 3) {
        const int a = e - M - 3 * L + 3;  // 0 .. L-4: cubics of {C, R} of row M (host-driven evaluation only)
        const double4 *r = hist + (size_t)M * (size_t)L + a;
        const double4 y0 = r[0], y1 = r[1], y2 = r[2], y3 = r[3];
        s4.coefM[2 * (size_t)a] = centred_cubic(y0.x, y1.x, y2.x, y3.x);
        s4.coefM[2 * (size_t)a + 1] = centred_cubic(y0.z, y1.z, y2.z, y3.z);
      } else {
        const int a = e - M - 2 * L;  // 0 .. L-4
        const double4 *r = hist + (size_t)(M - 1) * (size_t)L + a;
        const double4 y0 = r[0], y1 = r[1], y2 = r[2], y3 = r[3];
        double4 *o = s4.coefT + 4 * (size_t)a;
        o[0] = centred_cubic(y0.x, y1.x, y2.x, y3.x);
        o[1] = centred_cubic(y0.y, y1.y, y2.y, y3.y);
        o[2] = centred_cubic(y0.z, y1.z, y2.z, y3.z);
        o[3] = centred_cubic(y0.w, y1.w, y2.w, y3.w);
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
  __shared__ double2 s_cur[PREP_SCUR];
  if (k < 0) {  // host-driven evaluation: row M is read, nothing is updated; several nodes' loads in flight
#pragma unroll 4
    for (int l = threadIdx.x; l < L; l += blockDim.x) {
      const double4 c = rowM[l];
      const double2 y = make_double2(c.x, c.z);
      cur[l] = y;
      if (l < PREP_SCUR) s_cur[l] = y;
      if (l == 0) s_c0 = y.x;
      const double fp = horner(mc.c1, mc.pmax - 1, y.x), fpp = horner(mc.c2, mc.pmax - 2, y.x);
      const double nj = nu[l];
      am += nj * (fpp * y.y * y.x + fp * y.y);
      ae += nj * (fp * y.y);
    }
  }
  for (int l = threadIdx.x; l < L && k >= 0; l += blockDim.x) {
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
    if (l < PREP_SCUR) s_cur[l] = y;
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
  if (threadIdx.x == 0) *s4.tgt_next = s4.tgt_first;
  if (s4.on && k >= 0) {  // coefficient form of the row just formed (block-wide: a start needs four neighbours)
    __syncthreads();
    const double2 *src = (L <= PREP_SCUR) ? s_cur : cur;  // small L: no round trip through L2
    for (int a = threadIdx.x; a < L - 3; a += blockDim.x) {
      const double2 y0 = src[a], y1 = src[a + 1], y2 = src[a + 2], y3 = src[a + 3];
      s4.coefM[2 * (size_t)a] = centred_cubic(y0.x, y1.x, y2.x, y3.x);
      s4.coefM[2 * (size_t)a + 1] = centred_cubic(y0.y, y1.y, y2.y, y3.y);
    }
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
  if (threadIdx.x < 32) {  // second level: the first warp adds the warp sums (fixed order)
    double tm = threadIdx.x < nw ? sm[threadIdx.x] : 0.0;
    double te = threadIdx.x < nw ? se[threadIdx.x] : 0.0;
    double eps = threadIdx.x < nw ? sx[threadIdx.x] : 0.0;
    for (int o = 16; o > 0; o >>= 1) {
      tm += __shfl_xor_sync(0xffffffffu, tm, o);
      te += __shfl_xor_sync(0xffffffffu, te, o);
      eps += __shfl_xor_sync(0xffffffffu, eps, o);
    }
    if (threadIdx.x == 0) {
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
}


}  // namespace

// M = index of the current row; its time t[M] is read on the device (the RK step keeps t there).  With
// stage->dev_rows set, M is read on the device too and the host's M only sizes launches (pass n_cap).
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
  if (!(stage && stage->dev_rows)) ctx->rowtab_dirty = 1;  // host-driven evaluation: full rebuild, here and next time
  const bool s4 = ctx->p.stencil == 4 && !ctx->p.log_r;  // the log-R option runs the generic kernel
  const bool host_call = !(stage && stage->k >= 0);
  int pb = 1 + (M + (s4 ? (host_call ? 4 : 3) : 1) * L + PREP_THREADS - 1) / PREP_THREADS;
  if (pb > 33) pb = 33;
  dmfe_stage sg;
  if (stage) {
    sg = *stage;
  } else {
    memset(&sg, 0, sizeof(sg));
    sg.k = -1;
  }
  // persistent grid: one CTA per SM.  G = warps per target group.  As few as possible (long loops
  // over j), subject to (a) every warp slot of the GPU has work (L * G >= resident warps) and (b)
  // the number of rounds ceil(L / (groups per CTA * SMs)) wastes less than 3 % of the last round
  // (else the best G).
  const int warps_cta = (s4 ? S4_THREADS : RHS_THREADS) / 32;
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
  const int ngroups = warps_cta / G;
  int grid = (L + ngroups - 1) / ngroups;
  if (grid > ctx->sm_count) grid = ctx->sm_count;
  PrepS4 ps;
  ps.on = s4 ? 1 : 0;
  ps.br = ctx->br;
  ps.jtop = ctx->jtop;
  ps.coefM = reinterpret_cast<double4 *>(ctx->coefM);
  ps.coefT = reinterpret_cast<double4 *>(ctx->coefT);
  ps.omega = ctx->omega;
  ps.tgt_next = ctx->tgt_next;
  ps.tgt_first = grid * ngroups;  // the first round of targets is static (CTA b, group g: target b * ngroups + g)
  CUDA_TRY(ctx, launch_pdl(prepare_kernel, pb, PREP_THREADS, 0, ctx->stream, L, M, ctx->model, sg, ctx->theta,
                           ctx->nu, t, (const double4 *)hist, ctx->cur, ctx->rowtab, ctx->blo, ctx->scal, mu_hist,
                           ctx->muw, ps));
  RhsArgs a;
  memset(&a, 0, sizeof(a));
  a.L = L;
  a.M = M;
  a.theta = ctx->theta;
  a.omega = ctx->omega;
  a.thnu = ctx->thnu;
  a.nu = ctx->nu;
  a.tab = ctx->tab;
  a.t = t;
  a.mu_hist = mu_hist;
  a.hist = (const double4 *)hist;
  a.cur = ctx->cur;
  a.rowtab = ctx->rowtab;
  a.blo = ctx->blo;
  a.muw = ctx->muw;
  a.br = ctx->br;
  a.jtop = ctx->jtop;
  a.coefM = reinterpret_cast<const double4 *>(ctx->coefM);
  a.coefT = reinterpret_cast<const double4 *>(ctx->coefT);
  a.scal = ctx->scal;
  a.G = G;
  // dynamic hand-out of rounds pays from four rounds per CTA on (a CTA barrier and an atomic per round)
  a.tgt_next = ((L + ngroups - 1) / ngroups >= 4 * grid) ? ctx->tgt_next : nullptr;
  a.deriv_row = reinterpret_cast<double4 *>(deriv_row);
  if (stage && stage->dev_rows) {
    a.dev_rows = stage->dev_rows;
    a.dev_status = ctx->iscal + IS_STATUS;
    a.complete = stage->complete;
    a.mu_w = stage->mu;
    a.energy_w = stage->energy;
    a.hist_w = reinterpret_cast<double4 *>(stage->hist);
  }
  a.out = *out;
  cudaStreamCaptureStatus cap_status = cudaStreamCaptureStatusNone;
  cudaStreamIsCapturing(ctx->stream, &cap_status);
  const bool timed = ctx->timing_on && ctx->ev_n < DMFE_EV_RING && cap_status == cudaStreamCaptureStatusNone;
  if (timed) {
    if (ctx->ev_n >= ctx->ev_made) {
      CUDA_TRY(ctx, cudaEventCreate(&ctx->ev[2 * ctx->ev_made]));
      CUDA_TRY(ctx, cudaEventCreate(&ctx->ev[2 * ctx->ev_made + 1]));
      ctx->ev_made++;
    }
    CUDA_TRY(ctx, cudaEventRecord(ctx->ev[2 * ctx->ev_n], ctx->stream));
  }
  const int rc = s4 ? dmfe_launch_pairs_s4(ctx, a, grid) : dmfe_launch_pairs_generic(ctx, a, grid);
  if (rc != DMFE_OK) return rc;
  if (timed) {
    CUDA_TRY(ctx, cudaEventRecord(ctx->ev[2 * ctx->ev_n + 1], ctx->stream));
    ctx->ev_n++;
  }
  if (cap_status == cudaStreamCaptureStatusNone) CUDA_TRY(ctx, cudaGetLastError());
  return DMFE_OK;
}
