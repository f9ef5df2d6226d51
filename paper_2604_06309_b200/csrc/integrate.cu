// The step loop of a run: thinning schedule, Dormand-Prince
// start-up and switch, batches of device-resident SSPRK(10,4) steps.  Host logic only;
// every step of the path runs in the kernels behind dmfe_advance / dmfe_dp_step / dmfe_sparsify.
// The test oracle holds the same loop on the CPU; the tests compare the two decision for decision.
#include <math.h>
#include <string.h>

#include <chrono>

#include "dmfe_internal.cuh"

extern "C" int dmfe_integrate(dmfe_ctx *ctx, dmfe_state *st, const dmfe_policy *policy, double t_end,
                              int64_t max_steps, double max_seconds, dmfe_run_stats *stats) {
  if (!ctx || !st || !st->t || !st->mu || !st->hist || st->n_rows < 1) return DMFE_EINVAL;
  dmfe_policy p;
  memset(&p, 0, sizeof(p));
  if (policy) p = *policy;
  if (p.batch <= 0) p.batch = 50;
  if (p.sp_every <= 0) p.sp_every = 200;
  if (p.sp_max_passes <= 0) p.sp_max_passes = 8;
  if (!(p.sp_min_gain > 0.0)) p.sp_min_gain = 0.01;
  if (p.protect_last <= 0) p.protect_last = 24;
  dmfe_run_stats loc;
  memset(&loc, 0, sizeof(loc));
  dmfe_run_stats &S = stats ? *stats : loc;
  double f2_1 = 0.0;  // f''(1)
  for (int k = 0; k <= ctx->model.pmax; ++k) f2_1 += ctx->model.c2[k];
  const double rate = 4.0 * sqrt(f2_1);  // spectral bound of Eq.(24)
  if (st->n_rows == 1 && p.startup_dp) st->startup = 1;
  cudaStream_t s = ctx->stream;
  double t_now = 0.0;
  CUDA_TRY(ctx, cudaMemcpyAsync(&t_now, st->t + (st->n_rows - 1), sizeof(double), cudaMemcpyDeviceToHost, s));
  CUDA_TRY(ctx, cudaStreamSynchronize(s));
  const auto w0 = std::chrono::steady_clock::now();
  int64_t done = 0;
  int rc = DMFE_OK;
  while (t_now < t_end) {
    if (max_steps > 0 && done >= max_steps) break;
    if (max_seconds > 0.0 &&
        std::chrono::duration<double>(std::chrono::steady_clock::now() - w0).count() > max_seconds)
      break;
    // ---- thinning: threshold tol/10, greedy passes while they still pay ----
    if (st->acc_since >= p.sp_every || st->n_rows + 2 > st->n_cap) {
      S.sparsify_calls++;
      for (int pass = 0; pass < p.sp_max_passes; ++pass) {
        const int before = st->n_rows;
        int after = before;
        rc = dmfe_sparsify(ctx, st, p.protect_last, &after, nullptr);
        if (rc != DMFE_OK) break;
        S.sparsify_passes++;
        S.rows_dropped += before - after;
        if ((double)(before - after) < p.sp_min_gain * (double)before || before - after < 1) break;
      }
      if (rc != DMFE_OK) break;
      st->acc_since = 0;
      if (st->n_rows + 2 > st->n_cap) {
        rc = DMFE_ECAPACITY;
        break;
      }
    }
    if (st->startup) {
      // ---- Dormand-Prince start-up (reading G21) ----
      if (st->h * rate >= 3.3) {
        st->startup = 0;
        rc = dmfe_set_step_size(ctx, st, fmin(st->h / 2.0, ctx->h_stab));
        if (rc != DMFE_OK) break;
        continue;
      }
      int32_t acc = 0;
      rc = dmfe_dp_step(ctx, st, 0, &acc);
      S.steps++, S.dp_steps++, done++;
      if (acc) {
        S.accepted++;
        st->acc_since++;
      } else {
        S.reverted++;
      }
      cudaError_t e = cudaMemcpyAsync(&t_now, st->t + (st->n_rows - 1), sizeof(double), cudaMemcpyDeviceToHost, s);
      if (e == cudaSuccess) e = cudaStreamSynchronize(s);
      if (e != cudaSuccess) {
        ctx->cuda_err = (int)e;
        rc = DMFE_ECUDA;
      }
      if (rc != DMFE_OK) break;
    } else {
      // ---- a batch of device-resident SSPRK(10,4) steps ----
      int64_t nb = p.batch;
      if (max_steps > 0 && max_steps - done < nb) nb = max_steps - done;
      dmfe_advance_result r;
      memset(&r, 0, sizeof(r));
      rc = dmfe_advance(ctx, st, (int32_t)nb, 0, &r, nullptr);
      S.steps += r.steps, S.accepted += r.accepted, S.reverted += r.reverted, done += r.steps;
      st->acc_since += r.accepted;
      if (r.steps > 0) t_now = r.t_last;
      if (rc != DMFE_OK) break;
    }
    if (st->n_rows > S.n_rows_max) S.n_rows_max = st->n_rows;
  }
  S.n_rows = st->n_rows;
  if (st->n_rows > S.n_rows_max) S.n_rows_max = st->n_rows;
  S.t = t_now;
  S.h = st->h;
  S.eps_rk = st->eps_rk;
  S.status = rc;
  return rc;
}
