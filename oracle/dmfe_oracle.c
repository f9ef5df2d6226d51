/*
 * dmfe_oracle.c -- TEST INFRASTRUCTURE ONLY (CPU oracle; never on the product path).
 *
 * Plain, slow, obviously-correct fp64 implementation of the DMFE history
 * integrals of arxiv/paper_2604_06309 ("DYNAMITE"), written from PAPER.md.
 * It shares no code with the CUDA library under paper_2604_06309_b200/csrc.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load it.
 *
 * What it follows, in the paper's order and notation (readings G1..G32 are
 * listed in DESIGN.md):
 *   Eq.(17)  PAPER.md:238-245  integrals I1 on [0,theta], I2 on [theta,1] with
 *            nodes phi1_ij = theta_i*theta_j, phi2_ij = theta_i + (1-theta_i)*theta_j
 *   Eq.(18)  PAPER.md:249-252  s-point theta-stencil of the current slice (A factors)
 *   Eq.(19)  PAPER.md:256-260  type-1 lookup: cubic Hermite in t only
 *   Eq.(20)  PAPER.md:262-266  type-2 lookup: theta-stencil, then cubic Hermite in t
 *   Eq.(21)  PAPER.md:274-276  nu-weighted sums over j
 *   Eq.(10)-(13) PAPER.md:131-143  K=f''(C)R, D=f'(C), F_C, mu(t)
 *   Eq.(14)  PAPER.md:147      E(t)
 *   Eq.(1)   PAPER.md:69-75    dC/dt, dR/dt (with the -mu terms of Eq.(6), reading G1)
 *   Eq.(26)-(27) PAPER.md:326-332 sparsification residual
 *   PAPER.md:435      values-only history, 4-point Lagrange in t (orc_history_integrals_values,
 *                     reading G30; pins V1-V4)
 *   PAPER.md:453      logarithmic interpolation of the response history with fallback
 *                     (orc_history_integrals_logr, reading G32; pins LR1-LR4)
 *
 * Floating point: every product/sum below is a separate IEEE fp64 operation
 * (compile with -ffp-contract=off); the eight sums over j accumulate in
 * long double.  Index decisions (row search) use plain fp64 comparisons.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

/* ---- f'(q), f''(q) for f(q) = 1/2 sum_{p=0..pmax} lambda[p] q^p  (Eq.(4)) ---- */
static double f0(const double *lam, int pmax, double q) {
    double acc = 0.0;
    for (int p = pmax; p >= 0; --p) acc = acc * q + lam[p];
    return 0.5 * acc;
}
static double f1(const double *lam, int pmax, double q) {
    double acc = 0.0;
    for (int p = pmax; p >= 1; --p) acc = acc * q + (double)p * lam[p];
    return 0.5 * acc;
}
static double f2(const double *lam, int pmax, double q) {
    double acc = 0.0;
    for (int p = pmax; p >= 2; --p) acc = acc * q + (double)(p * (p - 1)) * lam[p];
    return 0.5 * acc;
}

double orc_f(const double *lam, int pmax, double q, int order) {
    return order == 0 ? f0(lam, pmax, q) : order == 1 ? f1(lam, pmax, q) : f2(lam, pmax, q);
}

/* Lagrange cardinal weights on the integer nodes 0..s-1 evaluated at u
 * ("index interpolation"). */
void orc_lagrange_weights(int s, double u, double *w) {
    for (int l = 0; l < s; ++l) {
        double num = 1.0, den = 1.0;
        for (int m = 0; m < s; ++m) {
            if (m == l) continue;
            num *= (u - (double)m);
            den *= (double)(l - m);
        }
        w[l] = num / den;
    }
}

/* Row search: n = max{ n <= M-1 : t[n] <= tau }.  t is ascending with
 * t[0] = 0 <= tau, so the set is never empty; textbook bisection on the predicate. */
int orc_row_search(const double *t, int M, double tau) {
    int lo = 0, hi = M - 1; /* invariant: t[lo] <= tau; answer in [lo, hi] */
    while (lo < hi) {
        int mid = lo + (hi - lo + 1) / 2;
        if (t[mid] <= tau) lo = mid; else hi = mid - 1;
    }
    return lo;
}

/* Weights of the local interpolant in t between rows n and n+1 at tau
 * ("local cubic Hermite").  If the upper row is the current row M
 * (no derivative yet) the interpolant is the quadratic through
 * (value, slope) at t_n and the value at t_{n+1}  (reading G12).
 * Returns {h00 (value n), h10 (slope n), h01 (value n+1), h11 (slope n+1)}. */
void orc_t_weights(const double *t, int n, int M, double tau, double *h) {
    double D = t[n + 1] - t[n];
    double u = (tau - t[n]) / D;
    if (n + 1 == M) {
        h[0] = 1.0 - u * u;
        h[1] = (u - u * u) * D;
        h[2] = u * u;
        h[3] = 0.0;
    } else {
        double u2 = u * u, u3 = u2 * u;
        h[0] = 2.0 * u3 - 3.0 * u2 + 1.0;
        h[1] = (u3 - 2.0 * u2 + u) * D;
        h[2] = -2.0 * u3 + 3.0 * u2;
        h[3] = (u3 - u2) * D;
    }
}

/* mu at an earlier time tau: local 4-point Lagrange in t over rows k..k+3
 * (reading G11); mu_all[0..M], with mu_all[M] = the mu just computed. */
double orc_mu_at(const double *t, const double *mu_all, int M, double tau) {
    int npts = M + 1 < 4 ? M + 1 : 4;
    int n = orc_row_search(t, M, tau);
    int k = n - 1;
    if (k > M + 1 - npts) k = M + 1 - npts;
    if (k < 0) k = 0;
    double acc = 0.0;
    for (int a = 0; a < npts; ++a) {
        double w = 1.0;
        for (int b = 0; b < npts; ++b) {
            if (b == a) continue;
            w *= (tau - t[k + b]) / (t[k + a] - t[k + b]);
        }
        acc += w * mu_all[k + a];
    }
    return acc;
}

#define HC(n, l) hist[((size_t)(n) * (size_t)L + (size_t)(l)) * 4 + 0]
#define HDC(n, l) hist[((size_t)(n) * (size_t)L + (size_t)(l)) * 4 + 1]
#define HR(n, l) hist[((size_t)(n) * (size_t)L + (size_t)(l)) * 4 + 2]
#define HDR(n, l) hist[((size_t)(n) * (size_t)L + (size_t)(l)) * 4 + 3]

/* On-grid reductions: mu(t) Eq.(13) and E(t) Eq.(14) on the current row M. */
void orc_mu_energy(int L, int M, const double *lam, int pmax, double T, double beta0,
                   const double *nu, const double *t, const double *hist,
                   double *mu_out, double *E_out) {
    long double sm = 0.0L, se = 0.0L;
    double tM = t[M];
    for (int j = 0; j < L; ++j) {
        double c = HC(M, j), r = HR(M, j);
        double fp = f1(lam, pmax, c), fpp = f2(lam, pmax, c);
        sm += (long double)(nu[j] * (fpp * r * c + fp * r));
        se += (long double)(nu[j] * (fp * r));
    }
    double c0 = HC(M, 0);
    *mu_out = T + tM * (double)sm + beta0 * f1(lam, pmax, c0) * c0;
    *E_out = -tM * (double)se - beta0 * f0(lam, pmax, c0);
}

/*
 * The history integrals for a list of targets.
 *
 *  L, s           theta-grid length, stencil size (points)
 *  M              index of the current row (rows 0..M-1 carry value+ray-derivative,
 *                 row M values only); t[0..M], mu_hist[0..M-1]
 *  hist           [M+1][L][4] packed {C, dC, R, dR}
 *  theta/omega/nu [L]; omega_i is the accurate complement 1-theta_i
 *  nt, targets    which target indices i (0-based) to evaluate
 *  start, frac    [3][nt][L] stencil start (0-based) and fractional index coordinate
 *                 u = X - start for the coordinates phi1, phi2, psi of pair (target, j)
 * outputs (any may be NULL):
 *  sums     [nt][8]  S1..S8 of DESIGN.md / SURVEY 8(c) step 6
 *  abssums  [nt][8]  sum_j |term| of the same (scale for the parity tolerance)
 *  deriv    [nt][6]  d1C, d1R, d2C, d2R, F^C, F^R
 *  scale    [nt][4]  magnitude scale of d1C, d1R, d2C, d2R (sum of |contributions|)
 *  rows1    [nt]     type-1 row index n(theta_i t)
 *  rows2    [nt][L]  type-2 row index n(phi2_ij t)
 *  mu_out, E_out     Eq.(13), Eq.(14)
 */
static void history_integrals_worker(int logR, int L, int s, int M, const double *lam, int pmax, double T,
                           double beta0, const double *theta, const double *omega,
                           const double *nu, const double *t, const double *mu_hist,
                           const double *hist, int nt, const int32_t *targets,
                           const int32_t *start, const double *frac, double *sums,
                           double *abssums, double *deriv, double *scale, int32_t *rows1,
                           int32_t *rows2, double *mu_out, double *E_out) {
    double mu, E;
    orc_mu_energy(L, M, lam, pmax, T, beta0, nu, t, hist, &mu, &E);
    if (mu_out) *mu_out = mu;
    if (E_out) *E_out = E;
    const double tM = t[M];
    double *mu_all = (double *)malloc(sizeof(double) * (size_t)(M + 1));
    for (int n = 0; n < M; ++n) mu_all[n] = mu_hist[n];
    mu_all[M] = mu;
    const size_t plane = (size_t)nt * (size_t)L;

#pragma omp parallel for schedule(dynamic, 1)
    for (int it = 0; it < nt; ++it) {
        const int i = targets[it];
        const double th_i = theta[i], om_i = omega[i];
        long double S[8], A[8];
        for (int k = 0; k < 8; ++k) S[k] = A[k] = 0.0L;
        double w1[16], w2[16], w3[16], h1[4], h2[4];

        /* type-1: one row search per target, tau = theta_i * t   (Eq.19) */
        const double tau1 = th_i * tM;
        const int n1 = orc_row_search(t, M, tau1);
        orc_t_weights(t, n1, M, tau1, h1);
        if (rows1) rows1[it] = n1;
        double B1C_first = 0.0;

        for (int j = 0; j < L; ++j) {
            const size_t e = (size_t)it * (size_t)L + (size_t)j;
            /* ---- A factors on the current row (Eq.18) ---- */
            const int a1 = start[0 * plane + e], a2 = start[1 * plane + e],
                      a3 = start[2 * plane + e];
            orc_lagrange_weights(s, frac[0 * plane + e], w1);
            orc_lagrange_weights(s, frac[1 * plane + e], w2);
            orc_lagrange_weights(s, frac[2 * plane + e], w3);
            double C1 = 0.0, R1 = 0.0, C2 = 0.0, R2 = 0.0;
            for (int l = 0; l < s; ++l) {
                C1 += w1[l] * HC(M, a1 + l);
                R1 += w1[l] * HR(M, a1 + l);
                C2 += w2[l] * HC(M, a2 + l);
                R2 += w2[l] * HR(M, a2 + l);
            }
            /* ---- type-1 lookup: B(theta_i t, theta_j), t-interpolation only (Eq.19) ---- */
            const double B1C = h1[0] * HC(n1, j) + h1[1] * HDC(n1, j) +
                               h1[2] * HC(n1 + 1, j) + h1[3] * (n1 + 1 == M ? 0.0 : HDC(n1 + 1, j));
            double B1R = h1[0] * HR(n1, j) + h1[1] * HDR(n1, j) +
                         h1[2] * HR(n1 + 1, j) + h1[3] * (n1 + 1 == M ? 0.0 : HDR(n1 + 1, j));
            if (logR && HR(n1, j) > 0.0 && HR(n1 + 1, j) > 0.0) {
                /* logarithmic interpolation of the response history: the same
                 * interpolant applied to log R with the scaled slope dR/R; reading G32 */
                const double ell = h1[0] * log(HR(n1, j)) + h1[1] * (HDR(n1, j) / HR(n1, j)) +
                                   h1[2] * log(HR(n1 + 1, j)) +
                                   h1[3] * (n1 + 1 == M ? 0.0 : HDR(n1 + 1, j) / HR(n1 + 1, j));
                B1R = exp(ell);
            }
            if (j == 0) B1C_first = B1C;
            /* ---- type-2 lookup: B(phi2 t, theta_i/phi2): theta-stencil first, then t (Eq.20) ---- */
            const double phi2 = th_i + om_i * theta[j];
            const double tau2 = phi2 * tM;
            const int n2 = orc_row_search(t, M, tau2);
            if (rows2) rows2[e] = n2;
            orc_t_weights(t, n2, M, tau2, h2);
            double cl = 0.0, dcl = 0.0, cu = 0.0, dcu = 0.0, rl = 0.0, drl = 0.0, ru = 0.0,
                   dru = 0.0;
            for (int l = 0; l < s; ++l) {
                cl += w3[l] * HC(n2, a3 + l);
                dcl += w3[l] * HDC(n2, a3 + l);
                rl += w3[l] * HR(n2, a3 + l);
                drl += w3[l] * HDR(n2, a3 + l);
                cu += w3[l] * HC(n2 + 1, a3 + l);
                ru += w3[l] * HR(n2 + 1, a3 + l);
                if (n2 + 1 != M) {
                    dcu += w3[l] * HDC(n2 + 1, a3 + l);
                    dru += w3[l] * HDR(n2 + 1, a3 + l);
                }
            }
            const double B2C = h2[0] * cl + h2[1] * dcl + h2[2] * cu + h2[3] * dcu;
            double B2R = h2[0] * rl + h2[1] * drl + h2[2] * ru + h2[3] * dru;
            if (logR) {
                /* all 2 s stencil values positive: theta-stencil and t-interpolant on log R and dR/R;
                 * otherwise the ordinary interpolation above stands ("automatic fallback") */
                int positive = 1;
                for (int l = 0; l < s; ++l)
                    if (!(HR(n2, a3 + l) > 0.0) || !(HR(n2 + 1, a3 + l) > 0.0)) positive = 0;
                if (positive) {
                    double ll = 0.0, dll = 0.0, lu = 0.0, dlu = 0.0;
                    for (int l = 0; l < s; ++l) {
                        ll += w3[l] * log(HR(n2, a3 + l));
                        dll += w3[l] * (HDR(n2, a3 + l) / HR(n2, a3 + l));
                        lu += w3[l] * log(HR(n2 + 1, a3 + l));
                        if (n2 + 1 != M) dlu += w3[l] * (HDR(n2 + 1, a3 + l) / HR(n2 + 1, a3 + l));
                    }
                    B2R = exp(h2[0] * ll + h2[1] * dll + h2[2] * lu + h2[3] * dlu);
                }
            }
            /* ---- kernel functions (Eq.10, Eq.11) and the eight terms (Eq.21) ---- */
            const double nj = nu[j];
            double term[8];
            term[0] = nj * (f2(lam, pmax, C1) * R1 * B1C);          /* S1: K(t,s) C(t',s)   */
            term[1] = nj * (f2(lam, pmax, C2) * R2 * B2C);          /* S2: K(t,s) C(s,t')   */
            term[2] = nj * (f1(lam, pmax, C1) * B1R);               /* S3: D(t,s) R(t',s)   */
            term[3] = nj * (f2(lam, pmax, C2) * R2 * B2R);          /* S4: K(t,s) R(s,t')   */
            term[4] = nj * (f2(lam, pmax, B1C) * B1R * C1);         /* S5: K(t',s) C(t,s)   */
            term[5] = nj * (f1(lam, pmax, B1C) * R1);               /* S6: D(t',s) R(t,s)   */
            term[6] = nj * (f1(lam, pmax, B2C) * R2);               /* S7: D(s,t') R(t,s)   */
            term[7] = nj * (R2 * (f2(lam, pmax, B2C) * B2R));       /* S8: R(t,s) K(s,t')   */
            for (int k = 0; k < 8; ++k) {
                S[k] += (long double)term[k];
                A[k] += (long double)fabs(term[k]);
            }
        }
        double Sd[8];
        for (int k = 0; k < 8; ++k) {
            Sd[k] = (double)S[k];
            if (sums) sums[(size_t)it * 8 + k] = Sd[k];
            if (abssums) abssums[(size_t)it * 8 + k] = (double)A[k];
        }
        if (deriv || scale) {
            const double Ci = HC(M, i), Ri = HR(M, i), C0 = HC(M, 0);
            const double mu_p = orc_mu_at(t, mu_all, M, tau1);
            const double fc = beta0 * f1(lam, pmax, C0) * B1C_first;
            const double fc2 = beta0 * f1(lam, pmax, B1C_first) * C0;
            const double d1C = -mu * Ci + tM * (th_i * Sd[0] + om_i * Sd[1] + th_i * Sd[2]) + fc;
            const double d1R = -mu * Ri + tM * (om_i * Sd[3]);
            const double d2C = -mu_p * Ci + tM * (th_i * Sd[4] + th_i * Sd[5] + om_i * Sd[6]) +
                               2.0 * T * Ri + fc2;
            const double d2R = mu_p * Ri - tM * (om_i * Sd[7]);
            if (deriv) {
                double *d = deriv + (size_t)it * 6;
                d[0] = d1C; d[1] = d1R; d[2] = d2C; d[3] = d2R;
                d[4] = d1C + th_i * d2C;
                d[5] = d1R + th_i * d2R;
            }
            if (scale) {
                double *q = scale + (size_t)it * 4;
                q[0] = fabs(mu * Ci) + tM * (th_i * (double)A[0] + om_i * (double)A[1] + th_i * (double)A[2]) + fabs(fc);
                q[1] = fabs(mu * Ri) + tM * om_i * (double)A[3];
                q[2] = fabs(mu_p * Ci) + tM * (th_i * (double)A[4] + th_i * (double)A[5] + om_i * (double)A[6]) + fabs(2.0 * T * Ri) + fabs(fc2);
                q[3] = fabs(mu_p * Ri) + tM * om_i * (double)A[7];
            }
        }
    }
    free(mu_all);
}

void orc_history_integrals(int L, int s, int M, const double *lam, int pmax, double T,
                           double beta0, const double *theta, const double *omega,
                           const double *nu, const double *t, const double *mu_hist,
                           const double *hist, int nt, const int32_t *targets,
                           const int32_t *start, const double *frac, double *sums,
                           double *abssums, double *deriv, double *scale, int32_t *rows1,
                           int32_t *rows2, double *mu_out, double *E_out) {
    history_integrals_worker(0, L, s, M, lam, pmax, T, beta0, theta, omega, nu, t, mu_hist, hist, nt,
                             targets, start, frac, sums, abssums, deriv, scale, rows1, rows2, mu_out, E_out);
}

/* The same with logarithmic interpolation of the response history (reading G32 in
 * DESIGN.md): in the type-1 and type-2 lookups the interpolant acts on log R and on the scaled slope
 * dR/R and the result is exponentiated, whenever every R value it reads is positive; otherwise the
 * ordinary interpolation is used.  The A factors (current slice) are interpolated as before. */
void orc_history_integrals_logr(int L, int s, int M, const double *lam, int pmax, double T,
                           double beta0, const double *theta, const double *omega,
                           const double *nu, const double *t, const double *mu_hist,
                           const double *hist, int nt, const int32_t *targets,
                           const int32_t *start, const double *frac, double *sums,
                           double *abssums, double *deriv, double *scale, int32_t *rows1,
                           int32_t *rows2, double *mu_out, double *E_out) {
    history_integrals_worker(1, L, s, M, lam, pmax, T, beta0, theta, omega, nu, t, mu_hist, hist, nt,
                             targets, start, frac, sums, abssums, deriv, scale, rows1, rows2, mu_out, E_out);
}

/* Sparsification residual (Eq.(26)-(27)): for every interior row n
 * (1..N-2) the 1-norm over theta_i of the difference between the integral over
 * [t_{n-1}, t_{n+1}] of the two cubic Hermite pieces through row n and of the single
 * piece that skips it.  eps_sparse[n] for n=1..N-2; entries 0 and N-1 set to +inf. */
void orc_sparsify_residuals(int L, int N, const double *t, const double *hist, double *eps_sparse) {
    eps_sparse[0] = INFINITY;
    if (N > 1) eps_sparse[N - 1] = INFINITY;
    for (int n = 1; n <= N - 2; ++n) {
        const double h1 = t[n] - t[n - 1], h2 = t[n + 1] - t[n], H = h1 + h2;
        long double acc = 0.0L;
        for (int i = 0; i < L; ++i) {
            for (int fld = 0; fld < 2; ++fld) {
                const int v = 2 * fld, d = 2 * fld + 1;
                const double Ya = hist[((size_t)(n - 1) * L + i) * 4 + v], Da = hist[((size_t)(n - 1) * L + i) * 4 + d];
                const double Yn = hist[((size_t)n * L + i) * 4 + v], Dn = hist[((size_t)n * L + i) * 4 + d];
                const double Yb = hist[((size_t)(n + 1) * L + i) * 4 + v], Db = hist[((size_t)(n + 1) * L + i) * 4 + d];
                const double with_n = h1 / 2.0 * (Ya + Yn) + h1 * h1 / 12.0 * (Da - Dn) +
                                      h2 / 2.0 * (Yn + Yb) + h2 * h2 / 12.0 * (Dn - Db);
                const double without = H / 2.0 * (Ya + Yb) + H * H / 12.0 * (Da - Db);
                acc += (long double)fabs(with_n - without);
            }
        }
        eps_sparse[n] = (double)acc;
    }
}

/* ------------------------------------------------------------------------------------------------
 * Values-only history ("higher-order interpolation schemes on the
 * adaptive t grid, which would allow a further reduction of stored history points"; BASELINE.json
 * config 2's "4-point-per-axis Lagrange stencils"): the rows hold C and R only, 16 bytes per cell,
 * and the interpolation in t is the local 4-point Lagrange polynomial through rows k..k+3 with
 *   k = clamp(n(tau) - 1, 0, M - 3)   (the window of orc_mu_at: one row below the interval of tau,
 * two above, clamped at both ends; fewer rows: all of them).  The current row M is an ordinary
 * point of the window.  Everything else is orc_history_integrals: theta-stencil first, then t
 * (PAPER.md:266), the same eight sums, mu, E and combinations.
 *   histv  [M+1][L][2] packed {C, R}
 * ------------------------------------------------------------------------------------------------ */
#define VC(n, l) histv[((size_t)(n) * (size_t)L + (size_t)(l)) * 2 + 0]
#define VR(n, l) histv[((size_t)(n) * (size_t)L + (size_t)(l)) * 2 + 1]

/* window start k, number of points and Lagrange weights in t at tau */
int orc_t_lagrange(const double *t, int M, double tau, double *w, int *npts_out) {
    int npts = M + 1 < 4 ? M + 1 : 4;
    int n = orc_row_search(t, M, tau);
    int k = n - 1;
    if (k > M + 1 - npts) k = M + 1 - npts;
    if (k < 0) k = 0;
    for (int a = 0; a < npts; ++a) {
        double wa = 1.0;
        for (int b = 0; b < npts; ++b) {
            if (b == a) continue;
            wa *= (tau - t[k + b]) / (t[k + a] - t[k + b]);
        }
        w[a] = wa;
    }
    *npts_out = npts;
    return k;
}

void orc_history_integrals_values(int L, int s, int M, const double *lam, int pmax, double T,
                                  double beta0, const double *theta, const double *omega,
                                  const double *nu, const double *t, const double *mu_hist,
                                  const double *histv, int nt, const int32_t *targets,
                                  const int32_t *start, const double *frac, double *sums,
                                  double *abssums, double *deriv, double *scale, int32_t *rows1,
                                  int32_t *rows2, double *mu_out, double *E_out) {
    /* on-grid reductions, Eq.(13), Eq.(14) */
    long double sm = 0.0L, se = 0.0L;
    const double tM = t[M];
    for (int j = 0; j < L; ++j) {
        double c = VC(M, j), r = VR(M, j);
        double fp = f1(lam, pmax, c), fpp = f2(lam, pmax, c);
        sm += (long double)(nu[j] * (fpp * r * c + fp * r));
        se += (long double)(nu[j] * (fp * r));
    }
    const double c00 = VC(M, 0);
    const double mu = T + tM * (double)sm + beta0 * f1(lam, pmax, c00) * c00;
    const double E = -tM * (double)se - beta0 * f0(lam, pmax, c00);
    if (mu_out) *mu_out = mu;
    if (E_out) *E_out = E;
    double *mu_all = (double *)malloc(sizeof(double) * (size_t)(M + 1));
    for (int n = 0; n < M; ++n) mu_all[n] = mu_hist[n];
    mu_all[M] = mu;
    const size_t plane = (size_t)nt * (size_t)L;

#pragma omp parallel for schedule(dynamic, 1)
    for (int it = 0; it < nt; ++it) {
        const int i = targets[it];
        const double th_i = theta[i], om_i = omega[i];
        long double S[8], A[8];
        for (int k = 0; k < 8; ++k) S[k] = A[k] = 0.0L;
        double w1[16], w2[16], w3[16], g1[4], g2[4];
        int np1, np2;
        /* type-1: one window per target, tau = theta_i * t  (Eq.19) */
        const double tau1 = th_i * tM;
        const int k1 = orc_t_lagrange(t, M, tau1, g1, &np1);
        if (rows1) rows1[it] = k1;
        double B1C_first = 0.0;
        for (int j = 0; j < L; ++j) {
            const size_t e = (size_t)it * (size_t)L + (size_t)j;
            const int a1 = start[0 * plane + e], a2 = start[1 * plane + e], a3 = start[2 * plane + e];
            orc_lagrange_weights(s, frac[0 * plane + e], w1);
            orc_lagrange_weights(s, frac[1 * plane + e], w2);
            orc_lagrange_weights(s, frac[2 * plane + e], w3);
            double C1 = 0.0, R1 = 0.0, C2 = 0.0, R2 = 0.0;
            for (int l = 0; l < s; ++l) {
                C1 += w1[l] * VC(M, a1 + l);
                R1 += w1[l] * VR(M, a1 + l);
                C2 += w2[l] * VC(M, a2 + l);
                R2 += w2[l] * VR(M, a2 + l);
            }
            /* type-1 lookup: t-interpolation of column j (Eq.19) */
            double B1C = 0.0, B1R = 0.0;
            for (int a = 0; a < np1; ++a) {
                B1C += g1[a] * VC(k1 + a, j);
                B1R += g1[a] * VR(k1 + a, j);
            }
            if (j == 0) B1C_first = B1C;
            /* type-2 lookup: theta-stencil on every row of the window, then t (Eq.20) */
            const double phi2 = th_i + om_i * theta[j];
            const double tau2 = phi2 * tM;
            const int k2 = orc_t_lagrange(t, M, tau2, g2, &np2);
            if (rows2) rows2[e] = k2;
            double B2C = 0.0, B2R = 0.0;
            for (int a = 0; a < np2; ++a) {
                double cr = 0.0, rr = 0.0;
                for (int l = 0; l < s; ++l) {
                    cr += w3[l] * VC(k2 + a, a3 + l);
                    rr += w3[l] * VR(k2 + a, a3 + l);
                }
                B2C += g2[a] * cr;
                B2R += g2[a] * rr;
            }
            const double nj = nu[j];
            double term[8];
            term[0] = nj * (f2(lam, pmax, C1) * R1 * B1C);
            term[1] = nj * (f2(lam, pmax, C2) * R2 * B2C);
            term[2] = nj * (f1(lam, pmax, C1) * B1R);
            term[3] = nj * (f2(lam, pmax, C2) * R2 * B2R);
            term[4] = nj * (f2(lam, pmax, B1C) * B1R * C1);
            term[5] = nj * (f1(lam, pmax, B1C) * R1);
            term[6] = nj * (f1(lam, pmax, B2C) * R2);
            term[7] = nj * (R2 * (f2(lam, pmax, B2C) * B2R));
            for (int k = 0; k < 8; ++k) {
                S[k] += (long double)term[k];
                A[k] += (long double)fabs(term[k]);
            }
        }
        double Sd[8];
        for (int k = 0; k < 8; ++k) {
            Sd[k] = (double)S[k];
            if (sums) sums[(size_t)it * 8 + k] = Sd[k];
            if (abssums) abssums[(size_t)it * 8 + k] = (double)A[k];
        }
        if (deriv || scale) {
            const double Ci = VC(M, i), Ri = VR(M, i), C0 = VC(M, 0);
            const double mu_p = orc_mu_at(t, mu_all, M, tau1);
            const double fc = beta0 * f1(lam, pmax, C0) * B1C_first;
            const double fc2 = beta0 * f1(lam, pmax, B1C_first) * C0;
            const double d1C = -mu * Ci + tM * (th_i * Sd[0] + om_i * Sd[1] + th_i * Sd[2]) + fc;
            const double d1R = -mu * Ri + tM * (om_i * Sd[3]);
            const double d2C = -mu_p * Ci + tM * (th_i * Sd[4] + th_i * Sd[5] + om_i * Sd[6]) +
                               2.0 * T * Ri + fc2;
            const double d2R = mu_p * Ri - tM * (om_i * Sd[7]);
            if (deriv) {
                double *d = deriv + (size_t)it * 6;
                d[0] = d1C; d[1] = d1R; d[2] = d2C; d[3] = d2R;
                d[4] = d1C + th_i * d2C;
                d[5] = d1R + th_i * d2R;
            }
            if (scale) {
                double *q = scale + (size_t)it * 4;
                q[0] = fabs(mu * Ci) + tM * (th_i * (double)A[0] + om_i * (double)A[1] + th_i * (double)A[2]) + fabs(fc);
                q[1] = fabs(mu * Ri) + tM * om_i * (double)A[3];
                q[2] = fabs(mu_p * Ci) + tM * (th_i * (double)A[4] + th_i * (double)A[5] + om_i * (double)A[6]) + fabs(2.0 * T * Ri) + fabs(fc2);
                q[3] = fabs(mu_p * Ri) + tM * om_i * (double)A[7];
            }
        }
    }
    free(mu_all);
}
