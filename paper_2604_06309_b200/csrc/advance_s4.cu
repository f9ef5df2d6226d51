// A batch of SSPRK(10,4) steps as ONE persistent cooperative kernel (S = 4, L <= 512: the shape of BASELINE.json's
// run configurations).  Same arithmetic per stage as rk_step.cu's graph of 21 launches per step (stage update,
// mu / E, per-call tables, the L^2 pairs of pairs_s4.cuh, controller of PAPER.md:320, commit), restructured so
// that a stage costs one grid-wide barrier instead of two dependent kernel launches:
//
//  * Every CTA keeps the whole stage state (q1, q2, delta: 2L entries each) in its shared memory and applies
//    every stage update itself, redundantly: all CTAs run the same instructions on the same data, so they hold
//    bit-identical states, mu, E, eps_RK and controller decisions without exchanging them.  Thread l owns node l.
//  * The only data a stage exchanges is F (2L doubles): each CTA writes the F_i of its targets, the grid barrier
//    follows, every CTA reads all of F.  Two F buffers alternate, so that a CTA that runs ahead cannot overwrite
//    values a slower CTA has not read yet.
//  * The per-call tables of the pre-pass are rebuilt by every CTA in its shared memory: the packed current row and
//    its cubic coefficient forms from the state it carries, the forms of row M-1 once per step, the row brackets of
//    all grid cells, and jtop for its own targets.  Brackets and jtop depend on the stage time and on complete rows
//    only, so those of stage k + 1 are built between the two halves of the barrier that ends stage k, from the
//    values of stage k as guesses (one round of independent loads).  The weights of mu(theta_i t_M) are formed
//    per target in the pair phase.  The row table lives in global memory and only grows: entry
//    N = {t_N, 1 / (t_{N+1} - t_N)} is written at the start of the step that appends row N + 1 (t_{N+1} = t_N + h
//    is known then) and is first read one step later.  The entry of the top interval [t_{M-1}, t_M] of the stage
//    being evaluated is formed locally (t_M changes with the stage).
//  * Targets are dealt out across the CTAs (CTA b: b, b + #CTAs, ...), so that the expensive targets at small
//    theta_i (long general loops) do not sit in the same few CTAs.  A thread has at most four pairs per target
//    here, so every phase of the pair loops of pairs_s4.cuh requests what all of its pairs need before it uses
//    any of it, and the row searches of a thread's pairs run in lock step.
//  * CTA 0 alone writes what leaves the kernel: the value slots of the appended row, t[M], the step scalars, the
//    counters and the optional per-step log.  Nothing it writes is read by another CTA before the next barrier.
//  * Nothing the kernel itself writes (history, t, mu, row table, F) is read through a read-only (.nc) load.
//
// Grid barrier: monotone arrival counter in global memory; thread 0 of every CTA arrives with red.release.gpu after
// a CTA barrier and spins with ld.acquire.gpu before the next CTA barrier; the kernel is launched cooperatively, so
// all CTAs are co-resident.  A barrier that is not completed within two seconds makes every CTA leave the kernel
// with status DMFE_ECUDA instead of hanging the device.
//
// Measured on B200 at the shape of BASELINE.json config 4 (L = 512, 128 CTAs x 512 threads, 139 KB of shared
// memory): ~32 k clk = 16 us per stage (pair phase 20 k, update + reductions 5 k, tables behind the barrier 3.5 k,
// barrier 1.5 - 3 k) against 22 us for the two launches of the graph path; the pair phase is bound by the L1 data
// path like the full-size kernel, growing to 27 k clk at 20 k rows.
#include <math.h>
#include <string.h>

#include "pairs_s4.cuh"

namespace {
using namespace dmfe_rhs;

constexpr int ADV_THREADS = S4_THREADS;
constexpr int ADV_MAX_L = 512;
constexpr int ADV_WARPS = ADV_THREADS / 32;

__constant__ double a_stage_c[10] = {0.0,       1.0 / 6.0, 2.0 / 6.0, 3.0 / 6.0, 4.0 / 6.0,
                                     2.0 / 6.0, 3.0 / 6.0, 4.0 / 6.0, 5.0 / 6.0, 6.0 / 6.0};
__constant__ double a_b_minus_bhat[10] = {0.1 - 0.0, 0.1 - 2.0 / 9.0, 0.1 - 0.0, 0.1 - 0.0, 0.1 - 5.0 / 18.0,
                                          0.1 - 1.0 / 3.0, 0.1 - 0.0, 0.1 - 0.0, 0.1 - 0.0, 0.1 - 1.0 / 6.0};

struct AdvArgs {
  int32_t L, G, n_steps, fixed_step;
  double tol, cap, h_min;
  const double *theta, *omega, *nu;
  const double2 *thnu;
  const uint64_t *tab;
  double *t, *mu, *energy;  // per-row arrays of the state
  double4 *hist;
  double2 *rowtab;  // [n_cap]
  double2 *Fbuf;    // [2][L] {F_C, F_R}
  double *scal;
  int32_t *iscal;
  unsigned *bar;    // arrival counter of the grid barrier (zeroed before the launch)
  double *log;      // optional [log_cap][4]
  int32_t log_cap;
};

__device__ __forceinline__ double4 cubic_form(double y0, double y1, double y2, double y3) {
  // 4-point index-Lagrange interpolant through y0..y3 as a cubic in v = u - 3/2 (history_integrals.cu)
  const double a = y1 + y2, b = y0 + y3, c = y2 - y1, e = y3 - y0;
  return make_double4((9.0 * a - b) * (1.0 / 16.0), (27.0 * c - e) * (1.0 / 24.0), (b - a) * 0.25,
                      (e - 3.0 * c) * (1.0 / 6.0));
}

__device__ __forceinline__ unsigned long long global_ns() {
  unsigned long long v;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(v));
  return v;
}

// The thread that arrives and spins for its CTA sits in the last warp: the release stalls its warp for a round trip
// to L2, and that warp is given no table work between the two halves of the barrier.
constexpr int BAR_THREAD = ADV_THREADS - 32;

// Grid barrier of the (cooperative) grid in two halves, so that work that needs nothing from the other CTAs can
// run between them: grid_arrive publishes this CTA's writes, grid_wait returns once every CTA has arrived (false
// when that did not happen within two seconds).
__device__ __forceinline__ void grid_arrive(unsigned *ctr, unsigned &target, unsigned nb) {
  __syncthreads();
  target += nb;
  if (threadIdx.x == BAR_THREAD) asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(ctr) : "memory");
}
__device__ __forceinline__ bool grid_wait(unsigned *ctr, unsigned target, int *s_fail) {
  if (threadIdx.x == BAR_THREAD) {
    const unsigned long long t0 = global_ns();
    for (;;) {
      unsigned v;
      asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(ctr) : "memory");
      if (v >= target) break;
      if (global_ns() - t0 > 2000000000ull) {
        *s_fail = 1;
        break;
      }
    }
  }
  __syncthreads();
  return *s_fail == 0;
}
__device__ __forceinline__ bool grid_sync(unsigned *ctr, unsigned &target, unsigned nb, int *s_fail) {
  grid_arrive(ctr, target, nb);
  return grid_wait(ctr, target, s_fail);
}

// n = max{ n in [0, top] : t[n] <= tau } from a guess g (rhs_common.cuh: row_search_from; here without the
// read-only qualifier, because t grows inside this kernel)
__device__ __forceinline__ int row_search_hint(const double *t, int top, int g, double tau) {
  g = min(max(g, 0), top);
  int lo, hi;
  if (t[g] <= tau) {
    lo = g;
    for (int st = 1;; st <<= 1) {
      const int nx = min(lo + st, top);
      if (nx == lo) return lo;
      if (t[nx] <= tau) {
        lo = nx;
      } else {
        hi = nx - 1;
        break;
      }
    }
  } else {
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
  while (lo < hi) {
    const int mid = lo + ((hi - lo + 1) >> 1);
    if (t[mid] <= tau)
      lo = mid;
    else
      hi = mid - 1;
  }
  return lo;
}

template <int PD>
__global__ void __launch_bounds__(ADV_THREADS, 1) advance_s4_kernel(AdvArgs a, ModelCoef mc) {
  extern __shared__ double4 smem_dyn[];
  __shared__ double red[2][ADV_WARPS][8];
  __shared__ double s_part[3][ADV_WARPS];
  __shared__ double s_c0;
  __shared__ double s_mu[2];  // mu(t_M), E(t_M) of the stage
  __shared__ int s_fail;
  const int L = a.L;
  double2 *s_q1 = reinterpret_cast<double2 *>(smem_dyn), *s_q2 = s_q1 + L, *s_dl = s_q2 + L;
  double2 *s_cur = s_dl + L;
  double4 *s_coefM = reinterpret_cast<double4 *>(s_cur + L);  // [L][2]
  double4 *s_coefT = s_coefM + 2 * (size_t)L;                 // [L][4]
  int2 *s_br = reinterpret_cast<int2 *>(s_coefT + 4 * (size_t)L);
  int32_t *s_blo = reinterpret_cast<int32_t *>(s_br + L), *s_jtop = s_blo + L;

  const int tid = threadIdx.x;
  const unsigned nb = gridDim.x;
  const int G = a.G, TG = 32 * G;
  const int warp = tid >> 5, lane = tid & 31;
  const int group = warp / G, wg = warp % G;
  const int ngroups = ADV_WARPS / G;
  const int tig = wg * 32 + lane;
  const size_t plane = (size_t)L * (size_t)L;
  const int K = (tig < L) ? (L - tig + TG - 1) / TG : 0;  // pairs j = tig + k TG of this thread
  // no __restrict__ / read-only loads on anything the kernel itself writes (history, t, mu, row table, F)
  const double4 *hist = a.hist;
  const double2 *rowtab = a.rowtab;
  unsigned bar_target = 0;
  int parity = 0;
  if (tid == 0) s_fail = 0;
  for (int c = tid; c < L; c += ADV_THREADS) s_blo[c] = 0, s_jtop[c] = 0;

  int rows = a.iscal[IS_NROWS];  // complete rows = index M of the row a step appends
  double h_next = a.scal[SC_HNEXT];
  int n_acc = 0, n_rev = 0, step = 0, status = 0, last_acc = 0;
  double last_eps = 0.0;

  // row table of the complete rows: entries e <= rows - 2 (t[e + 1] is final)
  for (int e = blockIdx.x * ADV_THREADS + tid; e < rows - 1; e += (int)nb * ADV_THREADS) {
    const double tn = a.t[e];
    a.rowtab[e] = make_double2(tn, 1.0 / (a.t[e + 1] - tn));
  }
  if (!grid_sync(a.bar, bar_target, nb, &s_fail)) status = DMFE_ECUDA;

  for (; step < a.n_steps && status == 0; ++step) {
    const int M = rows, N = rows - 1;
    const double h = h_next;
    const double t0 = a.t[N];
    const double tNext = __dadd_rn(t0, h);
    if (blockIdx.x == 0 && tid == 0) {
      a.scal[SC_H] = h;
      a.rowtab[N] = make_double2(t0, 1.0 / (tNext - t0));  // first read by the step after this one, if accepted
    }
    // cubic coefficient forms of row N = M - 1 (complete: values and slopes), fixed for the whole step
    for (int s0 = tid; s0 < L - 3; s0 += ADV_THREADS) {
      const double4 *r = hist + (size_t)N * (size_t)L + s0;
      const double4 y0 = ld_cell(r), y1 = ld_cell(r + 1), y2 = ld_cell(r + 2), y3 = ld_cell(r + 3);
      double4 *o = s_coefT + 4 * (size_t)s0;
      o[0] = cubic_form(y0.x, y1.x, y2.x, y3.x);
      o[1] = cubic_form(y0.y, y1.y, y2.y, y3.y);
      o[2] = cubic_form(y0.z, y1.z, y2.z, y3.z);
      o[3] = cubic_form(y0.w, y1.w, y2.w, y3.w);
    }
    // ---- per-call tables of a stage time tM, every CTA its own copy in shared memory.  They depend on the stage
    // time and on complete rows only, so the tables of stage k + 1 are built between the two halves of the grid
    // barrier that ends stage k.  (1) All nodes c: blo[c] = n(theta_c t_M) and the row brackets br of the grid cells
    // (every target's general pairs use them); the value of the previous stage is the guess: successive stage
    // times differ by a fraction of a step, so n is the guess or a neighbour, decided by one round of four
    // independent loads.  (2) Only for the targets of this CTA: jtop[i], by the first warp of the target's group
    // (the weights of mu(theta_i t_M) are formed in the pair phase, behind the loads of the type-1 half) ----
    auto build_tables = [&](const double tM) {
      const int top = M - 1;
      for (int c = tid; c < L && tid < BAR_THREAD; c += BAR_THREAD) {  // every warp but the barrier's
        const double tau1 = __dmul_rn(a.theta[c], tM);
        const int g = min(max(s_blo[c], 0), top);
        const double ta = (g >= 1) ? a.t[g - 1] : -INFINITY, tb = a.t[g];
        const double tc = (g + 1 <= top) ? a.t[g + 1] : INFINITY, td = (g + 2 <= top) ? a.t[g + 2] : INFINITY;
        int n;
        if (ta <= tau1 && tau1 < td) {
          n = (tc <= tau1) ? g + 1 : ((tb <= tau1) ? g : g - 1);
        } else {  // far guess (first stage after a thinning or a revert)
          n = row_search_hint(a.t, top, g, tau1);
        }
        s_blo[c] = n;
        // row bracket of the grid cell of phi2 by stencil start (history_integrals.cu: PrepS4::br)
        if (c >= 2 && c <= L - 3) s_br[c - 1].x = n;
        if (c >= 2 && c <= L - 3) s_br[c - 2].y = n;
        if (c == 0) s_br[0].x = n;
        if (c == L - 1) s_br[L - 4].y = n;
      }
      // no CTA barrier here: jtop does not read the brackets, and a CTA barrier follows before the pair phase reads
      // either (the one that ends grid_wait, or the one after the stage update)
      if (wg == 0) {
        for (int i = group * (int)nb + blockIdx.x; i < L; i += (int)nb * ngroups) {
          const double th_i = a.theta[i], om_i = a.omega[i];
          const double tau1 = __dmul_rn(th_i, tM);
          {
            // jtop[i]: first node j whose type-2 lookup falls into the top interval [t_{M-1}, t_M):
            // tau2(i, j) = fl(fl(theta_i + fl(omega_i theta_j)) t_M) is monotone in j.  The lanes test the 32 nodes
            // around the previous stage's value; nodes past the end count as inside
            auto in_top = [&](int j) { return __dmul_rn(__dadd_rn(th_i, __dmul_rn(om_i, a.theta[j])), tM) >= t0; };
            const int gj = min(max(s_jtop[i], 0), L);
            const int j0 = gj - 16, jq = j0 + lane;
            const bool in_l = (jq >= L) || (jq >= 0 && in_top(jq));
            const unsigned mask = __ballot_sync(0xffffffffu, in_l);
            int jt;
            if ((mask >> 31) && (j0 <= 0 || !(mask & 1u))) {
              jt = min(j0 + (__ffs(mask) - 1), L);
            } else {
              int lo = 0, hi = L;
              if (mask >> 31) hi = max(j0, 0); else lo = min(j0 + 32, L);
              while (lo < hi) {
                const int mid = (lo + hi) >> 1;
                if (in_top(mid))
                  hi = mid;
                else
                  lo = mid + 1;
              }
              jt = lo;
            }
            if (lane == 0) s_jtop[i] = jt;
          }
        }
      }
    };
    int accept = 1;
    double hn = h, eps_step = 0.0;
    build_tables(__dadd_rn(t0, __dmul_rn(a_stage_c[1], h)));  // stage 0

    for (int k = 0; k < 10 && status == 0; ++k) {
      const double tM = (k < 9) ? __dadd_rn(t0, __dmul_rn(a_stage_c[k + 1], h)) : tNext;
      // ---- stage update k (low-storage SSPRK(10,4), history_integrals.cu), thread l owns node l ----
      const double hb = __dmul_rn(h, a_b_minus_bhat[k]);
      const double h6 = h / 6.0;
      double am = 0.0, ae = 0.0, eacc = 0.0;
      for (int l = tid; l < L; l += ADV_THREADS) {
        double2 qa, qb, d, Fk;
        if (k == 0) {
          const double4 c = ld_cell(hist + (size_t)N * (size_t)L + l);
          qa = qb = make_double2(c.x, c.z);
          d = make_double2(0.0, 0.0);
          Fk = make_double2(c.y, c.w);
        } else {
          qa = s_q1[l];
          qb = s_q2[l];
          d = s_dl[l];
          Fk = a.Fbuf[(size_t)(k & 1) * L + l];
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
        upd(qa.x, qb.x, d.x, Fk.x);
        upd(qa.y, qb.y, d.y, Fk.y);
        s_q1[l] = qa;
        s_q2[l] = qb;
        s_dl[l] = d;
        s_cur[l] = qa;
        if (blockIdx.x == 0) {  // stage state = value slots of the appended row M
          double *cell = reinterpret_cast<double *>(a.hist + (size_t)M * (size_t)L + l);
          cell[0] = qa.x;
          cell[2] = qa.y;
        }
        if (l == 0) s_c0 = qa.x;
        const double fp = f1<PD>(mc, qa.x), fpp = f2<PD>(mc, qa.x);
        const double nj = a.nu[l];
        am += nj * (fpp * qa.y * qa.x + fp * qa.y);
        ae += nj * (fp * qa.y);
      }
      for (int o = 16; o > 0; o >>= 1) {
        am += __shfl_xor_sync(0xffffffffu, am, o);
        ae += __shfl_xor_sync(0xffffffffu, ae, o);
        eacc += __shfl_xor_sync(0xffffffffu, eacc, o);
      }
      if (lane == 0) s_part[0][warp] = am, s_part[1][warp] = ae, s_part[2][warp] = eacc;
      __syncthreads();  // also: s_cur, s_q* complete
      // mu (Eq.(13)) and E (Eq.(14)) from the 16 warp sums, added in a fixed order; only the threads that combine a
      // target (and the one that writes the scalars) need them, so this is off the path to the pair loops
      auto stage_mu = [&](double &mu, double &E) {
        double tm = 0.0, te = 0.0;
#pragma unroll
        for (int w = 0; w < ADV_WARPS; ++w) tm += s_part[0][w], te += s_part[1][w];
        const double c0 = s_c0;
        mu = mc.T + tM * tm, E = -tM * te;
        if (mc.beta0 != 0.0) {
          mu += mc.beta0 * f1<PD>(mc, c0) * c0;
          E -= mc.beta0 * horner(mc.c0, mc.pmax, c0);
        }
      };
      if (warp == ADV_WARPS - 1 && lane == 0) {  // one thread; the CTA barrier below publishes it
        double mu, E;
        stage_mu(mu, E);
        s_mu[0] = mu, s_mu[1] = E;
      }
      for (int s0 = tid; s0 < L - 3; s0 += ADV_THREADS) {  // cubic forms of the row just formed
        const double2 y0 = s_cur[s0], y1 = s_cur[s0 + 1], y2 = s_cur[s0 + 2], y3 = s_cur[s0 + 3];
        s_coefM[2 * (size_t)s0] = cubic_form(y0.x, y1.x, y2.x, y3.x);
        s_coefM[2 * (size_t)s0 + 1] = cubic_form(y0.y, y1.y, y2.y, y3.y);
      }
      __syncthreads();
      const double2 rtT = make_double2(t0, 1.0 / (tM - t0));  // top interval [t_{M-1}, t_M] of this stage
      double2 *Fout = a.Fbuf + (size_t)((k + 1) & 1) * L;

      // ---- the L^2 pairs (pairs_s4.cuh: same loops, tables in shared memory) ----
      // targets are dealt out across the CTAs (CTA b: b, b + nb, b + 2 nb, ...): the expensive small-theta targets
      // (long general loops) are spread over all SMs instead of sitting in the first few CTAs
      for (int i = group * (int)nb + blockIdx.x; i < L; i += (int)nb * ngroups, parity ^= 1) {
        const double th_i = a.theta[i], om_i = a.omega[i];
        const double tau1 = __dmul_rn(th_i, tM);
        const int n1 = s_blo[i];
        const bool top1 = (n1 + 1 == M);
        double h1[4];
        {
          const double2 rt = top1 ? rtT : rowtab[n1];
          t_weights(rt.x, rt.y, tau1, top1, h1);
        }
        // A thread has K <= KMAX = 4 pairs per target here (L <= 512, at least four warps per target), so the
        // loops of pairs_s4.cuh, which keep one pair in flight, would pay a memory round trip per pair.  Instead
        // every phase requests what all of the thread's pairs need before it uses any of it.
        constexpr int KMAX = 4;
        double2 mw = make_double2(0.0, 0.0);  // weights of mu(theta_i t_M); used by the group's first thread
        const uint64_t *pt1 = a.tab + (size_t)i * (size_t)L + tig;
        const uint64_t *pt2 = pt1 + plane, *pt3 = pt2 + plane;
        // ================= type-1 half of Eq.(21): S1, S3, S5, S6 =================
        {
          uint64_t e1[KMAX];
          double nu1[KMAX];
          double4 lo1[KMAX], hi1[KMAX];
          const double4 *pc = hist + (size_t)n1 * (size_t)L + tig;
#pragma unroll
          for (int q = 0; q < KMAX; ++q) {
            e1[q] = 0, nu1[q] = 0.0;
            lo1[q] = hi1[q] = make_double4(0.0, 0.0, 0.0, 0.0);
            if (q < K) {
              e1[q] = ld_stream(pt1 + q * TG);
              nu1[q] = a.nu[tig + q * TG];
              lo1[q] = ld_cell(pc + q * TG);
              if (top1) {  // upper row = the current row: values only (reading G12)
                const double2 c = s_cur[tig + q * TG];
                hi1[q] = make_double4(c.x, 0.0, c.y, 0.0);
              } else {
                hi1[q] = ld_cell(pc + L + q * TG);
              }
            }
          }
          if (wg == 0) {
            // mu(theta_i t_M) = mw.x + mw.y mu(t_M): local 4-point Lagrange in t over rows k0..k0+3 (reading G11),
            // lane p holds point p, the weight of the current row's mu kept apart; its loads travel with the
            // type-1 loads above.  w_p = prod_{q != p} (tau - t_q) / prod_{q != p} (t_p - t_q)
            const int npts = (M + 1 < 4) ? M + 1 : 4;
            const int k0 = min(max(n1 - 1, 0), M + 1 - npts);
            const bool stored = lane < npts && k0 + lane < M;
            const double tq_l = stored ? a.t[k0 + lane] : tM, mq_l = stored ? a.mu[k0 + lane] : 0.0;
            double num = 1.0, den = 1.0;
            for (int q = 0; q < npts; ++q) {
              const double tq = __shfl_sync(0xffffffffu, tq_l, q);
              if (q != lane) num *= (tau1 - tq), den *= (tq_l - tq);
            }
            const double wgt = num / den;
            const bool is_cur = (k0 + lane == M);
            const double part_l = (lane < npts && !is_cur) ? wgt * mq_l : 0.0, wM_l = (lane < npts && is_cur) ? wgt : 0.0;
            double part = 0.0, wM = 0.0;
            for (int q = 0; q < npts; ++q) {  // points in order, as a sequential sum
              part += __shfl_sync(0xffffffffu, part_l, q);
              wM += __shfl_sync(0xffffffffu, wM_l, q);
            }
            mw = make_double2(part, wM);
          }
          double acc0 = 0.0, acc1 = 0.0, acc2 = 0.0, acc3 = 0.0;
#pragma unroll
          for (int q = 0; q < KMAX; ++q) {
            if (q < K) {
              const double2 A1 = a_factor(s_cur, e1[q]);
              const double C1 = A1.x, R1 = A1.y;
              const double B1C = h1[0] * lo1[q].x + h1[1] * lo1[q].y + h1[2] * hi1[q].x + h1[3] * hi1[q].y;
              const double B1R = h1[0] * lo1[q].z + h1[1] * lo1[q].w + h1[2] * hi1[q].z + h1[3] * hi1[q].w;
              const double nR1 = nu1[q] * R1, nB1R = nu1[q] * B1R;
              acc0 = fma(f2<PD>(mc, C1) * nR1, B1C, acc0);   // S1: K(t,s) C(t',s)
              acc1 = fma(f1<PD>(mc, C1), nB1R, acc1);        // S3: D(t,s) R(t',s)
              acc2 = fma(f2<PD>(mc, B1C) * nB1R, C1, acc2);  // S5: K(t',s) C(t,s)
              acc3 = fma(f1<PD>(mc, B1C), nR1, acc3);        // S6: D(t',s) R(t,s)
            }
          }
          const double acc[4] = {acc0, acc1, acc2, acc3};
          constexpr int slot[4] = {0, 2, 4, 5};
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            double v = acc[q];
            for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            if (lane == 0) red[parity][warp][slot[q]] = v;
          }
        }
        // ================= type-2 half: S2, S4, S7, S8 =================
        {
          const int jt = s_jtop[i];
          int Kg = (jt > tig) ? (jt - tig + TG - 1) / TG : 0;  // this thread's pairs with j < jtop[i]
          if (Kg > K) Kg = K;
          uint64_t e2[KMAX], e3[KMAX];
          double2 tn[KMAX];
          double tau2[KMAX];
#pragma unroll
          for (int q = 0; q < KMAX; ++q) {
            e2[q] = e3[q] = 0;
            tn[q] = make_double2(0.0, 0.0);
            if (q < K) {
              e2[q] = ld_stream(pt2 + q * TG);
              e3[q] = ld_stream(pt3 + q * TG);
              tn[q] = a.thnu[tig + q * TG];
            }
          }
#pragma unroll
          for (int q = 0; q < KMAX; ++q) tau2[q] = __dmul_rn(__dadd_rn(th_i, __dmul_rn(om_i, tn[q].x)), tM);
          // ---- index stage of the general pairs (j < jtop[i]: n2 <= M - 2, both rows complete): n2 =
          // max{n in [lo, hi] : t_n <= tau2} by bisection inside the bracket br[a2], the thread's
          // pairs in lock step so that the row-table loads of one round are independent ----
          int lo2[KMAX], hi2[KMAX];
          double2 rt2[KMAX];
#pragma unroll
          for (int q = 0; q < KMAX; ++q) {
            lo2[q] = hi2[q] = 0;
            rt2[q] = make_double2(0.0, 1.0);
            if (q < Kg) {
              const int2 b = s_br[tab_start(e2[q])];
              lo2[q] = b.x;
              hi2[q] = min(b.y, M - 2);
              rt2[q] = rowtab[b.x];
            }
          }
          for (bool more = true; more;) {
            more = false;
            int mid[KMAX];
            double2 rm[KMAX];
#pragma unroll
            for (int q = 0; q < KMAX; ++q) {
              mid[q] = lo2[q] + ((hi2[q] - lo2[q] + 1) >> 1);
              rm[q] = rt2[q];
              if (lo2[q] < hi2[q]) rm[q] = rowtab[mid[q]];
            }
#pragma unroll
            for (int q = 0; q < KMAX; ++q) {
              if (lo2[q] < hi2[q]) {
                if (rm[q].x <= tau2[q])
                  lo2[q] = mid[q], rt2[q] = rm[q];
                else
                  hi2[q] = mid[q] - 1;
                more |= (lo2[q] < hi2[q]);
              }
            }
          }
          double acc0 = 0.0, acc1 = 0.0, acc2 = 0.0, acc3 = 0.0;
          auto finish = [&](double nj, double C2, double R2, double B2C, double B2R) {
            const double nR2 = nj * R2;
            const double K2 = f2<PD>(mc, C2) * nR2;
            acc0 = fma(K2, B2C, acc0);                     // S2: K(t,s) C(s,t')
            acc1 = fma(K2, B2R, acc1);                     // S4: K(t,s) R(s,t')
            acc2 = fma(f1<PD>(mc, B2C), nR2, acc2);        // S7: D(s,t') R(t,s)
            acc3 = fma(nR2, f2<PD>(mc, B2C) * B2R, acc3);  // S8: R(t,s) K(s,t')
          };
          // ---- general pairs: theta-stencil on the cells of rows n2 and n2 + 1, cubic Hermite in t (Eq.(20)) ----
#pragma unroll
          for (int q = 0; q < KMAX; ++q) {
            if (q < Kg) {
              const int a3 = tab_start(e3[q]);
              const double4 *p2 = hist + ((size_t)lo2[q] * (size_t)L + (size_t)a3);
              double4 x[4], y[4];
#pragma unroll
              for (int l = 0; l < 4; ++l) x[l] = ld_cell(p2 + l);
#pragma unroll
              for (int l = 0; l < 4; ++l) y[l] = ld_cell(p2 + L + l);
              const double v3 = tab_v(e3[q]);
              double h2[4];
              t_weights(rt2[q].x, rt2[q].y, tau2[q], false, h2);
              double w[4];
              lagrange4_centred(v3, w);
              double cl = 0.0, dcl = 0.0, rl = 0.0, drl = 0.0, cu = 0.0, dcu = 0.0, ru = 0.0, dru = 0.0;
#pragma unroll
              for (int l = 0; l < 4; ++l) {
                cl = fma(w[l], x[l].x, cl);
                dcl = fma(w[l], x[l].y, dcl);
                rl = fma(w[l], x[l].z, rl);
                drl = fma(w[l], x[l].w, drl);
              }
#pragma unroll
              for (int l = 0; l < 4; ++l) {
                cu = fma(w[l], y[l].x, cu);
                dcu = fma(w[l], y[l].y, dcu);
                ru = fma(w[l], y[l].z, ru);
                dru = fma(w[l], y[l].w, dru);
              }
              const double2 A2 = a_factor(s_cur, e2[q]);
              const double B2C = h2[0] * cl + h2[1] * dcl + h2[2] * cu + h2[3] * dcu;
              const double B2R = h2[0] * rl + h2[1] * drl + h2[2] * ru + h2[3] * dru;
              finish(tn[q].y, A2.x, A2.y, B2C, B2R);
            }
          }
          // ---- top pairs (j >= jtop[i]: n2 = M - 1): rows M-1 and M through their coefficient forms, quadratic
          // in t (reading G12): B = (1 - u^2) Y_{M-1} + d (1 - u) Y'_{M-1} + u^2 Y_M ----
          // The six cubics of a stencil start stay in registers while the start does not change (psi moves slowly
          // over the top interval): most top pairs read nothing but the A factor's four cells.
          int a3_held = -1;
          double4 qc = make_double4(0, 0, 0, 0), qdc = qc, qr = qc, qdr = qc, uc = qc, ur = qc;
#pragma unroll
          for (int q = 0; q < KMAX; ++q) {
            if (q >= Kg && q < K) {
              const int a3 = tab_start(e3[q]);
              if (a3 != a3_held) {
                qc = s_coefT[4 * a3], qdc = s_coefT[4 * a3 + 1];
                qr = s_coefT[4 * a3 + 2], qdr = s_coefT[4 * a3 + 3];
                uc = s_coefM[2 * a3], ur = s_coefM[2 * a3 + 1];
                a3_held = a3;
              }
              const double v3 = tab_v(e3[q]);
              const double2 A2 = a_factor(s_cur, e2[q]);
              const double d = tau2[q] - rtT.x;
              const double u = d * rtT.y;
              const double q2 = u * u;
              const double q0 = 1.0 - q2;
              const double q1 = d * (1.0 - u);
              const double B2C = fma(q0, cubic(qc, v3), fma(q1, cubic(qdc, v3), q2 * cubic(uc, v3)));
              const double B2R = fma(q0, cubic(qr, v3), fma(q1, cubic(qdr, v3), q2 * cubic(ur, v3)));
              finish(tn[q].y, A2.x, A2.y, B2C, B2R);
            }
          }
          const double acc[4] = {acc0, acc1, acc2, acc3};
          constexpr int slot[4] = {1, 3, 6, 7};
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            double v = acc[q];
            for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
            if (lane == 0) red[parity][warp][slot[q]] = v;
          }
        }
        if (G > 1)
          group_barrier(1 + group, TG);
        else
          __syncwarp();
        if (wg == 0) {
          // per-target combination (rhs_common.cuh: combine_target): Eq.(1), the second-argument equations (readings
          // G9, G10) and the ray derivative of Eq.(22).  Lanes 0..3 of the group's first warp form d1C, d1R, d2C, d2R
          // side by side with the same instructions: value = c X + t_M (k_a S_a + k_b S_b + k_c S_c) + add_1 + add_2
          const int r = lane & 3;
          const int qa = (r == 0) ? 0 : ((r == 1) ? 3 : ((r == 2) ? 4 : 7));
          const bool three = (r == 0) || (r == 2);
          double Sa = 0.0, Sb = 0.0, Sc = 0.0;
          for (int w = 0; w < G; ++w) {
            const double *rw = red[parity][group * G + w];
            Sa += rw[qa];
            Sb += three ? rw[qa + 1] : 0.0;
            Sc += three ? rw[qa + 2] : 0.0;
          }
          const double mu = s_mu[0], E = s_mu[1];
          double b1c_first = 0.0;  // C(theta_i t, 0): the beta0 forcing of Eq.(12)
          if (mc.beta0 != 0.0) {
            const double4 lo = ld_cell(hist + (size_t)n1 * (size_t)L);
            double4 hi = make_double4(s_cur[0].x, 0.0, s_cur[0].y, 0.0);
            if (!top1) hi = ld_cell(hist + (size_t)(n1 + 1) * (size_t)L);
            b1c_first = h1[0] * lo.x + h1[1] * lo.y + h1[2] * hi.x + h1[3] * hi.y;
          }
          const double mu_p = fma(mw.y, mu, mw.x);
          const double2 ci = s_cur[i], cz = s_cur[0];
          const double fc = mc.beta0 * f1<PD>(mc, cz.x) * b1c_first;
          const double fc2 = mc.beta0 * f1<PD>(mc, b1c_first) * cz.x;
          // r = 0: d1C = -mu C_i + t (th S1 + om S2 + th S3) + fc          r = 1: d1R = -mu R_i + t (om S4)
          // r = 2: d2C = -mu' C_i + t (th S5 + th S6 + om S7) + 2 T R_i + fc2    r = 3: d2R = mu' R_i - t (om S8)
          const double cX = (r == 0) ? -mu * ci.x : ((r == 1) ? -mu * ci.y : ((r == 2) ? -mu_p * ci.x : mu_p * ci.y));
          const double ka = (r == 0 || r == 2) ? th_i : ((r == 1) ? om_i : -om_i);
          const double kb = (r == 0) ? om_i : ((r == 2) ? th_i : 0.0);
          const double kc = (r == 0) ? th_i : ((r == 2) ? om_i : 0.0);
          const double add1 = (r == 0) ? fc : ((r == 2) ? 2.0 * mc.T * ci.y : 0.0);
          const double add2 = (r == 2) ? fc2 : 0.0;
          const double val = cX + tM * (ka * Sa + kb * Sb + kc * Sc) + add1 + add2;
          const double other = __shfl_down_sync(0xffffffffu, val, 2);  // lane 0: d2C, lane 1: d2R
          const double Fv = val + th_i * other;                          // lane 0: F_C, lane 1: F_R
          if (lane < 2) {
            reinterpret_cast<double *>(Fout + i)[lane] = Fv;
            if (k == 9) {  // this evaluation completes the appended row
              double *cell = reinterpret_cast<double *>(a.hist + (size_t)M * (size_t)L + i);
              cell[1 + 2 * lane] = Fv;
              if (i == 0 && lane == 0) {
                a.mu[M] = mu;
                if (a.energy) a.energy[M] = E;
              }
            }
          }
        }
      }
      if (k == 9) {  // eps_RK (Eq.(25)) and the controller (reading G20), identical in every thread
        double eps = 0.0;
#pragma unroll
        for (int w = 0; w < ADV_WARPS; ++w) eps += s_part[2][w];
        eps_step = eps;
        if (!a.fixed_step) {
          if (!isfinite(eps) || eps > 2.0 * a.tol) {
            accept = 0;
            hn = fmin(h / 2.0, a.cap);
          } else {
            if (eps > a.tol)
              hn = 0.9 * h;
            else if (eps < a.tol / 2.0)
              hn = 1.01 * h;
            hn = fmin(hn, a.cap);
          }
        }
      }
      if (blockIdx.x == 0 && tid == 0) {
        a.t[M] = tM;
        a.scal[SC_MU] = s_mu[0];
        a.scal[SC_E] = s_mu[1];
        if (k == 9) {
          a.scal[SC_EPS] = eps_step;
          a.scal[SC_HNEXT] = hn;
          a.scal[SC_ACCEPT] = (double)accept;
          a.iscal[IS_ACCEPT] = accept;
        }
      }
      grid_arrive(a.bar, bar_target, nb);
      if (k < 9) build_tables((k + 1 < 9) ? __dadd_rn(t0, __dmul_rn(a_stage_c[k + 2], h)) : tNext);
      if (!grid_wait(a.bar, bar_target, &s_fail)) status = DMFE_ECUDA;
    }  // stages
    if (status != 0) break;
    // ---- commit (rk_step.cu: commit_step_kernel), identical in every CTA ----
    int n = rows;
    if (accept) {
      n += 1;
      n_acc += 1;
    } else {
      if (!isfinite(eps_step) && n == 1) status = DMFE_ENONFINITE;
      n = (n - 10 > 1) ? n - 10 : 1;  // revert the previous ten steps
      n_rev += 1;
    }
    rows = n;
    last_acc = accept;
    last_eps = eps_step;
    h_next = hn;
    if (blockIdx.x == 0 && tid == 0 && a.log && step < a.log_cap) {
      double *r = a.log + 4 * (size_t)step;
      r[0] = (double)accept, r[1] = eps_step, r[2] = hn, r[3] = (double)n;
    }
    if (!a.fixed_step && hn < a.h_min && status == 0) status = DMFE_ESTEPMIN;
    if (status != 0) {
      ++step;
      break;
    }
  }
  if (tid == 0) {
    if (status == DMFE_ECUDA) {
      a.iscal[IS_STATUS] = DMFE_ECUDA;  // barrier time-out: whichever CTA saw it
    } else if (blockIdx.x == 0) {
      a.iscal[IS_NROWS] = rows;
      a.iscal[IS_STATUS] = status;
      a.iscal[IS_NACC] = n_acc;
      a.iscal[IS_NREV] = n_rev;
      a.iscal[IS_STEP] = step;
      a.iscal[IS_ACCEPT] = last_acc;
      a.scal[SC_TLAST] = a.t[rows - 1];
      a.scal[SC_EPS] = last_eps;
      a.scal[SC_HNEXT] = h_next;
    }
  }
}

}  // namespace

// Launches one batch.  Returns DMFE_OK when the batch was enqueued, 1 when this path does not apply (the caller
// then takes the graph path of rk_step.cu), or an error code.
int dmfe_launch_advance_s4(dmfe_ctx *ctx, dmfe_state *st, int n_steps, int fixed_step, double *log, int log_cap) {
  const int L = ctx->p.L;
  if (ctx->step_mode == 1 || ctx->adv_off) return 1;
  if (ctx->p.stencil != 4 || ctx->p.log_r || ctx->p.values_only || L > ADV_MAX_L) return 1;
  if (!ctx->adv_bar) {
    int dev = 0, coop = 0;
    cudaGetDevice(&dev);
    if (cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev) != cudaSuccess || !coop) {
      ctx->adv_off = 1;
      return 1;
    }
    CUDA_TRY(ctx, cudaMalloc(&ctx->adv_bar, 256));
  }
  // warps per target as in dmfe_launch_rhs: as few as fill the machine
  int G = 1;
  {
    double best = -1.0;
    for (int g = 1; g <= ADV_WARPS; g *= 2) {
      const long long slots = (long long)ctx->sm_count * (ADV_WARPS / g);
      const long long rounds = ((long long)L + slots - 1) / slots;
      const double eff = (double)L / (double)(rounds * slots);
      if (eff > best + 1e-9) best = eff, G = g;
      if (eff >= 0.97) break;
    }
  }
  while (G < ADV_WARPS && L > 4 * 32 * G) G *= 2;  // the kernel's pair phase holds at most 4 pairs per thread
  if (L > 4 * 32 * G) return 1;
  const int ngroups = ADV_WARPS / G;
  int grid = (L + ngroups - 1) / ngroups;
  if (grid > ctx->sm_count) grid = ctx->sm_count;
  const size_t smem = 272 * (size_t)L;  // q1, q2, delta, cur: 4 x 16 L; coefM 64 L, coefT 128 L; br 8 L, blo + jtop 8 L
  if (smem > (size_t)ctx->smem_max) return 1;
  AdvArgs a;
  memset(&a, 0, sizeof(a));
  a.L = L;
  a.G = G;
  a.n_steps = n_steps;
  a.fixed_step = fixed_step;
  a.tol = ctx->p.tol;
  a.cap = ctx->h_stab;
  a.h_min = ctx->p.h_min;
  a.theta = ctx->theta;
  a.omega = ctx->omega;
  a.nu = ctx->nu;
  a.thnu = ctx->thnu;
  a.tab = ctx->tab;
  a.t = st->t;
  a.mu = st->mu;
  a.energy = st->energy;
  a.hist = reinterpret_cast<double4 *>(st->hist);
  a.rowtab = ctx->rowtab;
  a.Fbuf = reinterpret_cast<double2 *>(ctx->rk);  // [4][L][2] doubles: the first half holds the two F buffers
  a.scal = ctx->scal;
  a.iscal = ctx->iscal;
  a.bar = ctx->adv_bar;
  a.log = log;
  a.log_cap = log_cap;
  ModelCoef mc = ctx->model;
  const void *fn = nullptr;
  if (mc.pmax <= 3)
    fn = (const void *)advance_s4_kernel<3>;
  else if (mc.pmax == 4)
    fn = (const void *)advance_s4_kernel<4>;
  else
    fn = (const void *)advance_s4_kernel<0>;
  CUDA_TRY(ctx, cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  int per_sm = 0;
  CUDA_TRY(ctx, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, ADV_THREADS, smem));
  if (per_sm < 1 || grid > per_sm * ctx->sm_count) {
    ctx->adv_off = 1;
    return 1;
  }
  CUDA_TRY(ctx, cudaMemsetAsync(ctx->adv_bar, 0, 256, ctx->stream));
  void *args[2] = {&a, &mc};
  const cudaError_t e = cudaLaunchCooperativeKernel(fn, dim3(grid), dim3(ADV_THREADS), args, smem, ctx->stream);
  if (e != cudaSuccess) {  // not launchable here: nothing was enqueued, the graph path takes over
    cudaGetLastError();
    ctx->adv_off = 1;
    return 1;
  }
  return DMFE_OK;
}
