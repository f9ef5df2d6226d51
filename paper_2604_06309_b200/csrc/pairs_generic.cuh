// Pair kernel for any stencil size S in {2, 4, 6, 8, 10}: the L^2 pairs of one right-hand side
// (section 3.3-3.4, steps a2-a6, a8 of DESIGN.md).  Used for S != 4; S = 4 (the
// configurations of BASELINE.json) runs the specialised kernel of pairs_s4.cuh.
//
// Mapping: persistent kernel, one CTA of 512 threads per SM.  The CTA's warps form groups of G
// warps; a group evaluates one target i at a time, lanes <-> adjacent nodes j (type-1 rows and the
// pair tables are read coalesced; the type-2 cells of adjacent lanes are neighbours in the packed
// history); the groups of one CTA take adjacent targets.  Every history cell {C,dC,R,dR} is one
// 256-bit load.  The per-call O(L + M) tables (current row, row table, bracket table) are copied
// into shared memory once per CTA when they fit.
//
// The row search of a pair is a bisection inside the bracket [blo[l*], blo[l*+1]]
// of the grid cell theta_l* <= phi2 < theta_l*+1 that the phi2 stencil start already identifies --
// same predicate and same result as a full bisection.  The loop over a thread's pairs is
// software-pipelined (table entries two pairs ahead, index stage one pair ahead) and runs twice
// per target: the type-1 half of Eq.(21) first (S1, S3, S5, S6; its four sums are parked in shared
// memory), then the type-2 half (S2, S4, S7, S8).
#pragma once
#include "rhs_common.cuh"

namespace dmfe_rhs {


// n = max{ n in [lo, hi] : rowtab[n].x <= tau }; requires t[lo] <= tau.
__device__ __forceinline__ int row_search_tab(const double2 *rowtab, int lo, int hi, double tau) {
  while (lo < hi) {
    const int mid = lo + ((hi - lo + 1) >> 1);
    if (rowtab[mid].x <= tau)
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
template <int S>
__device__ __forceinline__ int index_stage(const double2 *rowtab, const int32_t *blo, int L, double th_i, double om_i,
                                           double tM, double th_j, int a2, double *tau2_out) {
  const double phi2 = __dadd_rn(th_i, __dmul_rn(om_i, th_j));
  const double tau2 = __dmul_rn(phi2, tM);
  int clo = a2 + (S / 2 - 1), chi = clo + 1;
  if (a2 == 0) clo = 0, chi = S / 2;
  if (a2 == L - S) clo = (a2 == 0) ? 0 : L - S / 2 - 1, chi = L - 1;
  const int n2 = row_search_tab(rowtab, blo[clo], blo[chi], tau2);
  *tau2_out = tau2;
  return n2;
}

// SM: 0 = per-call tables read from global memory, 1 = cur and blo in shared memory, 2 = rowtab too
// LOGR: logarithmic interpolation of the response history (reading G32): in the type-1 and
// type-2 lookups the interpolant acts on log R and dR/R whenever every R value it reads is positive and the
// result is exponentiated; otherwise the ordinary interpolation stands.
template <int S, int PD, int SM, bool LOGR = false>
__global__ void __launch_bounds__(RHS_THREADS, 1) history_integrals_kernel(RhsArgs a, ModelCoef mc) {
  constexpr bool SMT = SM >= 1, SMR = SM == 2;
  extern __shared__ double4 smem_dyn[];
  pdl_launch_dependents();
  pdl_wait();
  if (batch_stopped(a)) return;
  const int L = a.L, M = current_row(a);
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
  __shared__ int s_base[2];  // first target of the CTA's next round

  const int G = a.G;      // warps per group (power of two, <= RHS_THREADS/32)
  const int TG = 32 * G;  // threads per group = stride of j
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int group = warp / G, wg = warp % G;
  const int ngroups = (RHS_THREADS / 32) / G;
  const int tig = wg * 32 + lane;  // thread index inside the group
  const size_t plane = (size_t)L * (size_t)L;
  const double tM = a.t[M];
  int parity = 0;

  // rounds of ngroups adjacent targets per CTA, handed out dynamically after the first one (pairs_s4.cuh)
  int rnd = 0;
  for (int base = blockIdx.x * ngroups; base < L; parity ^= 1, ++rnd) {
    if (a.tgt_next && threadIdx.x == 0) s_base[rnd & 1] = atomicAdd(a.tgt_next, ngroups);
    const int i = base + group;
    if (i < L) {
    const uint64_t *tab1 = a.tab + (size_t)i * (size_t)L, *tab2 = tab1 + plane, *tab3 = tab2 + plane;
    const double th_i = a.theta[i], om_i = a.omega[i];
    // type-1: one row search per target, tau = theta_i t  (Eq.(19)); blo[i] is exactly that row
    const double tau1 = __dmul_rn(th_i, tM);
    const int n1 = blo[i];
    const bool top1 = (n1 + 1 == M);
    double h1[4];
    {
      const double2 rt = rowtab[n1];
      t_weights(rt.x, rt.y, tau1, top1, h1);
    }
    const double4 *row1lo = a.hist + (size_t)n1 * (size_t)L;
    const double4 *row1hi = row1lo + L;
    double b1c_first = 0.0;

    // ---- type-1 half of Eq.(21): S1, S3, S5, S6 (coalesced rows n1, n1+1, requested one pair ahead) ----
    {
      double acc[4] = {0.0, 0.0, 0.0, 0.0};
      uint64_t eA1 = 0, eB1 = 0;
      double nuA = 0.0, nuB = 0.0;
      double4 lo = make_double4(0, 0, 0, 0), hi = lo;
      int j = tig;
      if (j < L) {
        eA1 = ld_stream(tab1 + j);
        nuA = a.thnu[j].y;
        lo = ld_cell(row1lo + j);
        hi = ld_cell(row1hi + j);
      }
      if (j + TG < L) {
        eB1 = ld_stream(tab1 + j + TG);
        nuB = a.thnu[j + TG].y;
      }
      for (; j < L; j += TG) {
        uint64_t eC1 = 0;
        double nuC = 0.0;
        double4 lon = make_double4(0, 0, 0, 0), hin = lon;
        if (j + 2 * TG < L) {
          eC1 = ld_stream(tab1 + j + 2 * TG);
          nuC = a.thnu[j + 2 * TG].y;
        }
        if (j + TG < L) {
          lon = ld_cell(row1lo + j + TG);
          hin = ld_cell(row1hi + j + TG);
        }
        int a1;
        double u1;
        dmfe_tab_decode(eA1, &a1, &u1);
        double w[S];
        double C1 = 0.0, R1 = 0.0;
        lagrange_weights<S>(u1, w);
#pragma unroll
        for (int l = 0; l < S; ++l) {
          const double2 v = cur[a1 + l];
          C1 = fma(w[l], v.x, C1);
          R1 = fma(w[l], v.y, R1);
        }
        if (top1) hi.y = 0.0, hi.w = 0.0;
        const double B1C = h1[0] * lo.x + h1[1] * lo.y + h1[2] * hi.x + h1[3] * hi.y;
        double B1R = h1[0] * lo.z + h1[1] * lo.w + h1[2] * hi.z + h1[3] * hi.w;
        if (LOGR && lo.z > 0.0 && hi.z > 0.0)
          B1R = exp(h1[0] * log(lo.z) + h1[1] * (lo.w / lo.z) + h1[2] * log(hi.z) + h1[3] * (hi.w / hi.z));
        if (j == 0) b1c_first = B1C;
        // every term carries nu_j and exactly one of R1, B1R: fold nu_j into those two
        const double nR1 = nuA * R1, nB1R = nuA * B1R;
        acc[0] = fma(f2<PD>(mc, C1) * nR1, B1C, acc[0]);   // S1: K(t,s) C(t',s)
        acc[1] = fma(f1<PD>(mc, C1), nB1R, acc[1]);        // S3: D(t,s) R(t',s)
        acc[2] = fma(f2<PD>(mc, B1C) * nB1R, C1, acc[2]);  // S5: K(t',s) C(t,s)
        acc[3] = fma(f1<PD>(mc, B1C), nR1, acc[3]);        // S6: D(t',s) R(t,s)
        eA1 = eB1, eB1 = eC1, nuA = nuB, nuB = nuC, lo = lon, hi = hin;
      }
      constexpr int slot[4] = {0, 2, 4, 5};
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        double v = acc[k];
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) red[parity][warp][slot[k]] = v;
      }
    }
    // ---- type-2 half: S2, S4, S7, S8 (row search per pair, theta-stencil on two rows, Hermite in t) ----
    {
      double acc[4] = {0.0, 0.0, 0.0, 0.0};
      uint64_t eA2 = 0, eA3 = 0, eB2 = 0, eB3 = 0;
      double2 tnA = make_double2(0.0, 0.0), tnB = tnA;
      int n2A = 0;
      double tau2A = 0.0;
      int j = tig;
      if (j < L) {
        eA2 = ld_stream(tab2 + j);
        eA3 = ld_stream(tab3 + j);
        tnA = a.thnu[j];
      }
      if (j + TG < L) {
        eB2 = ld_stream(tab2 + j + TG);
        eB3 = ld_stream(tab3 + j + TG);
        tnB = a.thnu[j + TG];
      }
      if (j < L) n2A = index_stage<S>(rowtab, blo, L, th_i, om_i, tM, tnA.x, (int)(eA2 >> 48), &tau2A);
      for (; j < L; j += TG) {
        uint64_t eC2 = 0, eC3 = 0;
        double2 tnC = make_double2(0.0, 0.0);
        if (j + 2 * TG < L) {
          eC2 = ld_stream(tab2 + j + 2 * TG);
          eC3 = ld_stream(tab3 + j + 2 * TG);
          tnC = a.thnu[j + 2 * TG];
        }
        const int n2 = n2A;
        const double4 *p2 = a.hist + (size_t)n2 * (size_t)L + (int)(eA3 >> 48);
        double4 x[S];  // the lower row's cells are requested before the next pair's index stage
#pragma unroll
        for (int l = 0; l < S; ++l) x[l] = ld_cell(p2 + l);
        int n2B = 0;
        double tau2B = 0.0;
        if (j + TG < L) n2B = index_stage<S>(rowtab, blo, L, th_i, om_i, tM, tnB.x, (int)(eB2 >> 48), &tau2B);
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
          const double2 v = cur[a2 + l];
          C2 = fma(w[l], v.x, C2);
          R2 = fma(w[l], v.y, R2);
        }
        if (a.out.rows2) a.out.rows2[(size_t)i * (size_t)L + (size_t)j] = n2;
        const bool top2 = (n2 + 1 == M);
        double h2[4];
        {
          const double2 rt = rowtab[n2];
          t_weights(rt.x, rt.y, tau2A, top2, h2);
        }
        // theta-stencil first, then t
        lagrange_weights<S>(u3, w);
        double cl = 0.0, dcl = 0.0, rl = 0.0, drl = 0.0, cu = 0.0, dcu = 0.0, ru = 0.0, dru = 0.0;
        double ll = 0.0, dll = 0.0, lu = 0.0, dlu = 0.0;
        bool positive = true;
#pragma unroll
        for (int l = 0; l < S; ++l) {
          const double4 xl = x[l], yl = ld_cell(p2 + L + l);
          if (LOGR) {
            positive = positive && (xl.z > 0.0) && (yl.z > 0.0);
            ll = fma(w[l], log(xl.z), ll);
            dll = fma(w[l], xl.w / xl.z, dll);
            lu = fma(w[l], log(yl.z), lu);
            dlu = fma(w[l], yl.w / yl.z, dlu);
          }
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
        double B2R = h2[0] * rl + h2[1] * drl + h2[2] * ru + h2[3] * dru;
        if (LOGR && positive) {
          if (top2) dlu = 0.0;
          B2R = exp(h2[0] * ll + h2[1] * dll + h2[2] * lu + h2[3] * dlu);
        }
        const double nR2 = nj * R2;
        const double K2 = f2<PD>(mc, C2) * nR2;
        acc[0] = fma(K2, B2C, acc[0]);                     // S2: K(t,s) C(s,t')
        acc[1] = fma(K2, B2R, acc[1]);                     // S4: K(t,s) R(s,t')
        acc[2] = fma(f1<PD>(mc, B2C), nR2, acc[2]);        // S7: D(s,t') R(t,s)
        acc[3] = fma(nR2, f2<PD>(mc, B2C) * B2R, acc[3]);  // S8: R(t,s) K(s,t')
        eA2 = eB2, eA3 = eB3, tnA = tnB;
        eB2 = eC2, eB3 = eC3, tnB = tnC;
        n2A = n2B;
        tau2A = tau2B;
      }
      constexpr int slot[4] = {1, 3, 6, 7};
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        double v = acc[k];
        for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) red[parity][warp][slot[k]] = v;
      }
    }
    // ---- fixed-order sum over the warps of the group, then the O(1) work per target ----
    // red[parity] is reused two targets later: one barrier per target suffices
    if (G > 1)
      group_barrier(1 + group, TG);
    else
      __syncwarp();
    if (tig == 0)
      combine_target<PD, SMT>(a, mc, i, n1, th_i, om_i, tM, tau1, b1c_first, red[parity], group * G, G, cur, M);
    }  // i < L
    if (a.tgt_next) {
      __syncthreads();
      base = s_base[rnd & 1];
    } else {  // few rounds per CTA: static round-robin
      base += gridDim.x * ngroups;
    }
  }
}

}  // namespace dmfe_rhs
