// Right-hand side on a VALUES-ONLY history ("higher-order interpolation
// schemes on the adaptive t grid, which would allow a further reduction of stored history points";
// BASELINE.json config 2's "4-point-per-axis Lagrange stencils"): the rows hold {C, R} only, 16 bytes per
// cell, and the interpolation in t is the local 4-point Lagrange polynomial through rows k..k+3 with
// k = clamp(n(tau) - 1, 0, M - 3) (the window rule of reading G11; the current row M is an ordinary point).
// Everything else is the path of pairs_generic.cuh: theta-stencil first, then t, the same
// eight sums (Eq.(21)) and per-target combination.  Offered for the north-star call
// dmfe_history_integrals only (dmfe_params.values_only); the integrator keeps the Hermite history, whose
// stored derivative is the first stage of every step.
//
// Per-call tables (prepare_values_kernel): packed current row, mu / E, bracket table blo, mu weights and,
// per window start k, win[k] = {t_k .. t_k+3, 1/prod_{b != a}(t_k+a - t_k+b)}: a pair forms its four
// t-weights with 4 subtractions and 10 multiplications, no division.
#include "rhs_common.cuh"

namespace {
using namespace dmfe_rhs;

constexpr int PV_THREADS = 1024;
constexpr int VAL_THREADS = 512;

struct ValArgs {
  int32_t L, M, G;
  const double *theta, *omega;
  const double2 *thnu;
  const uint64_t *tab;
  const double *t;
  const double2 *hist;   // [M+1][L] {C, R}
  const double2 *cur;    // [L] row M
  const int32_t *blo;    // [L] n(theta_c t_M)
  const double2 *muw;    // [L] mu(theta_c t_M) = muw.x + muw.y mu(t_M)
  const double4 *win;    // [max(M-2,1)][2]: {t_k..t_k+3}, {inverse denominators}
  const double *scal;
  int32_t *tgt_next;     // next block of targets to hand out (reset by prepare_values_kernel)
  dmfe_rhs_out out;
};

__global__ void __launch_bounds__(PV_THREADS) prepare_values_kernel(int L, int M, ModelCoef mc,
                                                                    const double *__restrict__ theta,
                                                                    const double *__restrict__ nu,
                                                                    const double *__restrict__ t,
                                                                    const double *__restrict__ mu_hist,
                                                                    const double2 *__restrict__ hist,
                                                                    double2 *__restrict__ cur, int32_t *__restrict__ blo,
                                                                    double2 *__restrict__ muw, double4 *__restrict__ win,
                                                                    double *__restrict__ scal, int32_t *tgt_next, int tgt_first) {
  __shared__ double sm[32], se[32];
  __shared__ double s_c0;
  pdl_launch_dependents();
  pdl_wait();
  const double tM = t[M];
  const int npts = (M + 1 < 4) ? M + 1 : 4;
  const int nwin = M + 2 - npts;  // window starts 0 .. M + 1 - npts
  if (blockIdx.x > 0 || gridDim.x == 1) {
    const int nb = gridDim.x == 1 ? 1 : gridDim.x - 1;
    const int b = gridDim.x == 1 ? 0 : blockIdx.x - 1;
    for (int e = b * PV_THREADS + threadIdx.x; e < nwin + L; e += nb * PV_THREADS) {
      if (e < nwin) {
        double tq[4] = {0.0, 0.0, 0.0, 0.0}, inv[4] = {0.0, 0.0, 0.0, 0.0};
        for (int a = 0; a < npts; ++a) tq[a] = t[e + a];
        for (int a = 0; a < npts; ++a) {
          double den = 1.0;
          for (int q = 0; q < npts; ++q)
            if (q != a) den *= (tq[a] - tq[q]);
          inv[a] = 1.0 / den;
        }
        win[2 * (size_t)e] = make_double4(tq[0], tq[1], tq[2], tq[3]);
        win[2 * (size_t)e + 1] = make_double4(inv[0], inv[1], inv[2], inv[3]);
      } else {
        const int c = e - nwin;
        const double tau1 = __dmul_rn(theta[c], tM);
        const int n = row_search_from(t, M - 1, blo[c], tau1);
        blo[c] = n;
        int k0 = n - 1;  // mu(theta_c t_M): 4-point Lagrange in t (reading G11), weight of mu_M kept apart
        if (k0 > M + 1 - npts) k0 = M + 1 - npts;
        if (k0 < 0) k0 = 0;
        double part = 0.0, wM = 0.0;
        for (int p = 0; p < npts; ++p) {
          double wgt = 1.0;
          for (int q = 0; q < npts; ++q)
            if (q != p) wgt *= (tau1 - t[k0 + q]) / (t[k0 + p] - t[k0 + q]);
          if (k0 + p == M)
            wM = wgt;
          else
            part += wgt * mu_hist[k0 + p];
        }
        muw[c] = make_double2(part, wM);
      }
    }
    if (blockIdx.x > 0) return;
  }
  // block 0: pack row M, reduce mu (Eq.(13)) and E (Eq.(14))
  double am = 0.0, ae = 0.0;
  for (int l = threadIdx.x; l < L; l += blockDim.x) {
    const double2 y = hist[(size_t)M * (size_t)L + l];
    cur[l] = y;
    if (l == 0) s_c0 = y.x;
    const double fp = horner(mc.c1, mc.pmax - 1, y.x), fpp = horner(mc.c2, mc.pmax - 2, y.x);
    const double nj = nu[l];
    am += nj * (fpp * y.y * y.x + fp * y.y);
    ae += nj * (fp * y.y);
  }
  for (int o = 16; o > 0; o >>= 1) {
    am += __shfl_xor_sync(0xffffffffu, am, o);
    ae += __shfl_xor_sync(0xffffffffu, ae, o);
  }
  const int w = threadIdx.x >> 5, nw = blockDim.x >> 5;
  if ((threadIdx.x & 31) == 0) sm[w] = am, se[w] = ae;
  __syncthreads();
  if (threadIdx.x == 0) {
    double tm = 0.0, te = 0.0;
    for (int q = 0; q < nw; ++q) tm += sm[q], te += se[q];
    const double c0 = s_c0;
    scal[SC_MU] = mc.T + tM * tm + mc.beta0 * horner(mc.c1, mc.pmax - 1, c0) * c0;
    scal[SC_E] = -tM * te - mc.beta0 * horner(mc.c0, mc.pmax, c0);
    *tgt_next = tgt_first;
  }
}

// the four Lagrange weights in t at tau from a window entry: w_a = inv_a prod_{b != a} (tau - t_b);
// windows of fewer than four rows carry inv = 0 for the missing points and their factors are skipped
__device__ __forceinline__ void t_lagrange(const double4 tq, const double4 inv, double tau, int npts, double (&g)[4]) {
  const double p0 = tau - tq.x, p1 = tau - tq.y;
  const double p2 = npts > 2 ? tau - tq.z : 1.0, p3 = npts > 3 ? tau - tq.w : 1.0;
  const double p01 = p0 * p1, p23 = p2 * p3;
  g[0] = inv.x * (p1 * p23);
  g[1] = inv.y * (p0 * p23);
  g[2] = inv.z * (p01 * p3);
  g[3] = inv.w * (p01 * p2);
}

__device__ __forceinline__ double2 ld_vcell(const double2 *p) { return *p; }

// SMT: cur and blo in shared memory.  Same mapping as the generic kernel: persistent CTA per SM, groups of
// G warps per target, lanes <-> adjacent nodes j; a plain loop per pair (table entries one pair ahead).
template <int S, int PD, bool SMT>
__global__ void __launch_bounds__(VAL_THREADS, 1) history_integrals_values_kernel(ValArgs a, ModelCoef mc) {
  extern __shared__ double4 smem_dyn[];
  pdl_launch_dependents();
  pdl_wait();
  const int L = a.L, M = a.M;
  const double2 *cur = a.cur;
  const int32_t *blo = a.blo;
  if (SMT) {
    double2 *s_cur = reinterpret_cast<double2 *>(smem_dyn);
    int32_t *s_blo = reinterpret_cast<int32_t *>(s_cur + L);
    for (int k = threadIdx.x; k < L; k += VAL_THREADS) s_cur[k] = a.cur[k], s_blo[k] = a.blo[k];
    __syncthreads();
    cur = s_cur, blo = s_blo;
  }
  __shared__ double red[2][VAL_THREADS / 32][8];
  __shared__ int s_base[2];  // first target of the CTA's next round
  const int G = a.G, TG = 32 * G;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int group = warp / G, wg = warp % G;
  const int ngroups = (VAL_THREADS / 32) / G;
  const int tig = wg * 32 + lane;
  const size_t plane = (size_t)L * (size_t)L;
  const double tM = a.t[M];
  const int npts = (M + 1 < 4) ? M + 1 : 4;
  const int kmax = M + 1 - npts;
  int parity = 0;

  // rounds of ngroups adjacent targets per CTA, handed out dynamically after the first one (pairs_s4.cuh)
  int rnd = 0;
  for (int base = blockIdx.x * ngroups; base < L; parity ^= 1, ++rnd) {
    if (a.tgt_next && threadIdx.x == 0) s_base[rnd & 1] = atomicAdd(a.tgt_next, ngroups);
    const int i = base + group;
    if (i < L) {
    const uint64_t *tab1 = a.tab + (size_t)i * (size_t)L, *tab2 = tab1 + plane, *tab3 = tab2 + plane;
    const double th_i = a.theta[i], om_i = a.omega[i];
    // type-1: one window per target, tau = theta_i t (Eq.(19))
    const double tau1 = __dmul_rn(th_i, tM);
    const int n1 = blo[i];
    const int k1 = min(max(n1 - 1, 0), kmax);
    double g1[4];
    t_lagrange(a.win[2 * (size_t)k1], a.win[2 * (size_t)k1 + 1], tau1, npts, g1);
    const double2 *rows1p = a.hist + (size_t)k1 * (size_t)L;
    double b1c_first = 0.0;
    double acc[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) acc[q] = 0.0;
    uint64_t e1n = 0, e2n = 0, e3n = 0;
    double2 tnn = make_double2(0.0, 0.0);
    if (tig < L) {
      e1n = ld_stream(tab1 + tig);
      e2n = ld_stream(tab2 + tig);
      e3n = ld_stream(tab3 + tig);
      tnn = a.thnu[tig];
    }
    for (int j = tig; j < L; j += TG) {
      const uint64_t e1 = e1n, e2 = e2n, e3 = e3n;
      const double2 tn = tnn;
      if (j + TG < L) {
        e1n = ld_stream(tab1 + j + TG);
        e2n = ld_stream(tab2 + j + TG);
        e3n = ld_stream(tab3 + j + TG);
        tnn = a.thnu[j + TG];
      }
      int a1, a2, a3;
      double u1, u2, u3;
      dmfe_tab_decode(e1, &a1, &u1);
      dmfe_tab_decode(e2, &a2, &u2);
      dmfe_tab_decode(e3, &a3, &u3);
      double w[S];
      // ---- A factors at phi1 and the type-1 lookup: S1, S3, S5, S6 ----
      double C1 = 0.0, R1 = 0.0;
      lagrange_weights<S>(u1, w);
#pragma unroll
      for (int l = 0; l < S; ++l) {
        const double2 v = cur[a1 + l];
        C1 = fma(w[l], v.x, C1);
        R1 = fma(w[l], v.y, R1);
      }
      double B1C = 0.0, B1R = 0.0;
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        if (q < npts) {
          const double2 v = ld_vcell(rows1p + (size_t)q * L + j);
          B1C = fma(g1[q], v.x, B1C);
          B1R = fma(g1[q], v.y, B1R);
        }
      }
      if (j == 0) b1c_first = B1C;
      const double nj = tn.y;
      const double nR1 = nj * R1, nB1R = nj * B1R;
      acc[0] = fma(f2<PD>(mc, C1) * nR1, B1C, acc[0]);   // S1
      acc[2] = fma(f1<PD>(mc, C1), nB1R, acc[2]);        // S3
      acc[4] = fma(f2<PD>(mc, B1C) * nB1R, C1, acc[4]);  // S5
      acc[5] = fma(f1<PD>(mc, B1C), nR1, acc[5]);        // S6
      // ---- A factors at phi2 ----
      double C2 = 0.0, R2 = 0.0;
      lagrange_weights<S>(u2, w);
#pragma unroll
      for (int l = 0; l < S; ++l) {
        const double2 v = cur[a2 + l];
        C2 = fma(w[l], v.x, C2);
        R2 = fma(w[l], v.y, R2);
      }
      // ---- type-2 lookup (Eq.(20)): row search inside the bracket of the grid cell of phi2 (same
      // predicate and result as a full bisection), window k2, theta-stencil on its rows,
      // then Lagrange in t ----
      const double tau2 = __dmul_rn(__dadd_rn(th_i, __dmul_rn(om_i, tn.x)), tM);
      int clo = a2 + (S / 2 - 1), chi = clo + 1;
      if (a2 == 0) clo = 0, chi = S / 2;
      if (a2 == L - S) clo = (a2 == 0) ? 0 : L - S / 2 - 1, chi = L - 1;
      const int n2 = row_search(a.t, blo[clo], blo[chi], tau2);
      const int k2 = min(max(n2 - 1, 0), kmax);
      if (a.out.rows2) a.out.rows2[(size_t)i * (size_t)L + (size_t)j] = k2;
      double g2[4];
      t_lagrange(a.win[2 * (size_t)k2], a.win[2 * (size_t)k2 + 1], tau2, npts, g2);
      lagrange_weights<S>(u3, w);
      const double2 *p2 = a.hist + (size_t)k2 * (size_t)L + a3;
      double B2C = 0.0, B2R = 0.0;
#pragma unroll
      for (int q = 0; q < 4; ++q) {
        if (q < npts) {
          double cr = 0.0, rr = 0.0;
#pragma unroll
          for (int l = 0; l < S; ++l) {
            const double2 v = ld_vcell(p2 + (size_t)q * L + l);
            cr = fma(w[l], v.x, cr);
            rr = fma(w[l], v.y, rr);
          }
          B2C = fma(g2[q], cr, B2C);
          B2R = fma(g2[q], rr, B2R);
        }
      }
      const double nR2 = nj * R2;
      const double K2 = f2<PD>(mc, C2) * nR2;
      acc[1] = fma(K2, B2C, acc[1]);                     // S2
      acc[3] = fma(K2, B2R, acc[3]);                     // S4
      acc[6] = fma(f1<PD>(mc, B2C), nR2, acc[6]);        // S7
      acc[7] = fma(nR2, f2<PD>(mc, B2C) * B2R, acc[7]);  // S8
    }
#pragma unroll
    for (int q = 0; q < 8; ++q) {
      double v = acc[q];
      for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
      if (lane == 0) red[parity][warp][q] = v;
    }
    if (G > 1)
      group_barrier(1 + group, TG);
    else
      __syncwarp();
    if (tig == 0) {
    double Sd[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) {
      double s = 0.0;
      for (int w2 = 0; w2 < G; ++w2) s += red[parity][group * G + w2][q];
      Sd[q] = s;
      if (a.out.sums) a.out.sums[(size_t)q * L + i] = s;
    }
    if (a.out.rows1) a.out.rows1[i] = k1;
    // combine: Eq.(1), the second-argument equations (G9, G10), Eq.(22)
    const double mu = a.scal[SC_MU];
    const double2 mw = a.muw[i];
    const double mu_p = fma(mw.y, mu, mw.x);
    const double2 ci = cur[i], c0 = cur[0];
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
    if (a.out.F) {
      a.out.F[2 * i] = d1C + th_i * d2C;
      a.out.F[2 * i + 1] = d1R + th_i * d2R;
    }
    if (i == 0) {
      if (a.out.mu) a.out.mu[0] = mu;
      if (a.out.energy) a.out.energy[0] = a.scal[SC_E];
    }
    }  // tig == 0
    }  // i < L
    if (a.tgt_next) {
      __syncthreads();
      base = s_base[rnd & 1];
    } else {  // few rounds per CTA: static round-robin
      base += gridDim.x * ngroups;
    }
  }
}

}  // namespace

int dmfe_launch_rhs_values(dmfe_ctx *ctx, int32_t M, int32_t n_cap, const double *t, const double *mu_hist,
                           const double *hist, const dmfe_rhs_out *out) {
  const int L = ctx->p.L;
  if (M + 1 > ctx->win_cap) {  // per-call window table, grown on demand
    const int cap = n_cap > M + 1 ? n_cap : M + 1;
    CUDA_TRY(ctx, cudaStreamSynchronize(ctx->stream));
    cudaFree(ctx->win);
    ctx->win = nullptr;
    ctx->win_cap = 0;
    CUDA_TRY(ctx, cudaMalloc(&ctx->win, sizeof(double) * 8 * (size_t)cap));
    ctx->win_cap = cap;
  }
  const int warps_cta = VAL_THREADS / 32;
  int G = 1;
  {
    double best = -1.0;
    for (int g = 1; g <= warps_cta && g <= 16; g *= 2) {
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
  int pb = 1 + (M + L + PV_THREADS - 1) / PV_THREADS;
  if (pb > 33) pb = 33;
  CUDA_TRY(ctx, launch_pdl(prepare_values_kernel, pb, PV_THREADS, 0, ctx->stream, L, M, ctx->model, ctx->theta, ctx->nu,
                           t, mu_hist, (const double2 *)hist, ctx->cur, ctx->blo, ctx->muw,
                           reinterpret_cast<double4 *>(ctx->win), ctx->scal, ctx->tgt_next, grid * ngroups));
  ValArgs a;
  memset(&a, 0, sizeof(a));
  a.L = L;
  a.M = M;
  a.theta = ctx->theta;
  a.omega = ctx->omega;
  a.thnu = ctx->thnu;
  a.tab = ctx->tab;
  a.t = t;
  a.hist = (const double2 *)hist;
  a.cur = ctx->cur;
  a.blo = ctx->blo;
  a.muw = ctx->muw;
  a.win = reinterpret_cast<const double4 *>(ctx->win);
  a.scal = ctx->scal;
  a.G = G;
  a.tgt_next = ((L + ngroups - 1) / ngroups >= 4 * grid) ? ctx->tgt_next : nullptr;
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
  const size_t smem1 = 20 * (size_t)L;
  const bool smt = smem1 <= (size_t)ctx->smem_max;
  const size_t smem = smt ? smem1 : 0;
  const int pd = ctx->model.pmax <= 3 ? 3 : (ctx->model.pmax == 4 ? 4 : 0);
#define DMFE_LAUNCH_K(KFN)                                                                              \
  do {                                                                                                  \
    auto kfn = KFN;                                                                                     \
    if (smem + 4096 > 48 * 1024)                                                                        \
      CUDA_TRY(ctx, cudaFuncSetAttribute(kfn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)); \
    CUDA_TRY(ctx, launch_pdl(kfn, grid, VAL_THREADS, smem, ctx->stream, a, ctx->model));                \
  } while (0)
#define DMFE_LAUNCH_V(S_, PD_)                                            \
  do {                                                                    \
    if (smt)                                                              \
      DMFE_LAUNCH_K((history_integrals_values_kernel<S_, PD_, true>));    \
    else                                                                  \
      DMFE_LAUNCH_K((history_integrals_values_kernel<S_, PD_, false>));   \
  } while (0)
#define DMFE_LAUNCH_VS(S_)   \
  do {                       \
    if (pd == 3)             \
      DMFE_LAUNCH_V(S_, 3);  \
    else if (pd == 4)        \
      DMFE_LAUNCH_V(S_, 4);  \
    else                     \
      DMFE_LAUNCH_V(S_, 0);  \
  } while (0)
  switch (ctx->p.stencil) {
    case 2: DMFE_LAUNCH_VS(2); break;
    case 4: DMFE_LAUNCH_VS(4); break;
    case 6: DMFE_LAUNCH_VS(6); break;
    case 8: DMFE_LAUNCH_VS(8); break;
    case 10: DMFE_LAUNCH_VS(10); break;
    default: return DMFE_EINVAL;
  }
#undef DMFE_LAUNCH_VS
#undef DMFE_LAUNCH_V
#undef DMFE_LAUNCH_K
  if (timed) {
    CUDA_TRY(ctx, cudaEventRecord(ctx->ev[2 * ctx->ev_n + 1], ctx->stream));
    ctx->ev_n++;
  }
  CUDA_TRY(ctx, cudaGetLastError());
  return DMFE_OK;
}
