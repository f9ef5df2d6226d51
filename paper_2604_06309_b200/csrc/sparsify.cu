// Selective history reduction.  For an interior row n with neighbours n-1, n+1
// the residual of Eq.(26) is the difference between the integral over [t_{n-1}, t_{n+1}] of the
// two cubic Hermite pieces through row n and of the single piece that skips it (closed form),
// eps_sparse[n] = sum_i |Delta^C_i| + |Delta^R_i| (Eq.(27)).  Walking n upward, row n is dropped if
// eps_sparse[n] < tol/10 and the walk continues at n+2, else at n+1.  Because a
// candidate's neighbours are never removed before it is tested, all residuals are computed in
// parallel on the uncompacted history; the walk and the index scan are O(N) integer work; the
// rows, t, mu and E are compacted on the device.
#include <math.h>

#include "dmfe_internal.cuh"

namespace {

__global__ void __launch_bounds__(256) sparsify_residual_kernel(int L, int N, const double *__restrict__ t,
                                                                const double4 *__restrict__ hist,
                                                                double *__restrict__ eps_sp) {
  const int n = blockIdx.x + 1;  // interior rows 1..N-2
  if (n > N - 2) return;
  __shared__ double sm[8];
  const double h1 = t[n] - t[n - 1], h2 = t[n + 1] - t[n], H = h1 + h2;
  const double4 *ra = hist + (size_t)(n - 1) * L, *rn = hist + (size_t)n * L, *rb = hist + (size_t)(n + 1) * L;
  double acc = 0.0;
  for (int i = threadIdx.x; i < L; i += blockDim.x) {
    const double4 a = ra[i], c = rn[i], b = rb[i];
    const double wC = h1 / 2.0 * (a.x + c.x) + h1 * h1 / 12.0 * (a.y - c.y) + h2 / 2.0 * (c.x + b.x) +
                      h2 * h2 / 12.0 * (c.y - b.y);
    const double oC = H / 2.0 * (a.x + b.x) + H * H / 12.0 * (a.y - b.y);
    const double wR = h1 / 2.0 * (a.z + c.z) + h1 * h1 / 12.0 * (a.w - c.w) + h2 / 2.0 * (c.z + b.z) +
                      h2 * h2 / 12.0 * (c.w - b.w);
    const double oR = H / 2.0 * (a.z + b.z) + H * H / 12.0 * (a.w - b.w);
    acc += fabs(wC - oC) + fabs(wR - oR);
  }
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if ((threadIdx.x & 31) == 0) sm[threadIdx.x >> 5] = acc;
  __syncthreads();
  if (threadIdx.x == 0) {
    double s = 0.0;
    for (int w = 0; w < (int)(blockDim.x >> 5); ++w) s += sm[w];
    eps_sp[n] = s;
  }
}

// greedy walk + exclusive scan of the keep flags; newidx[d] = source row of
// compacted row d; iscal[IS_NROWS] = rows kept, iscal[IS_NROWS+1] = first row that moves.
__global__ void sparsify_walk_kernel(int N, int protect_last, double thr, const double *__restrict__ eps_sp,
                                     int32_t *__restrict__ keep, int32_t *__restrict__ newidx,
                                     int32_t *__restrict__ iscal) {
  if (blockIdx.x != 0 || threadIdx.x != 0) return;
  for (int n = 0; n < N; ++n) keep[n] = 1;
  int n = 1;
  const int last = N - 1 - protect_last;
  while (n <= last && n <= N - 2) {
    if (eps_sp[n] < thr) {
      keep[n] = 0;
      n += 2;
    } else {
      n += 1;
    }
  }
  int m = 0, first = N;
  for (int r = 0; r < N; ++r) {
    if (keep[r]) {
      newidx[m++] = r;
    } else if (first == N) {
      first = r;
    }
  }
  iscal[IS_NROWS] = m;
  iscal[IS_FIRST] = first;
}

// gather kept rows d >= first into the staging buffer, then copy back (two launches: an in-place
// parallel move would overwrite sources that other CTAs still have to read)
__global__ void sparsify_gather_kernel(int L, const int32_t *__restrict__ iscal, const int32_t *__restrict__ newidx,
                                       const double4 *__restrict__ hist, const double *__restrict__ t,
                                       const double *__restrict__ mu, const double *__restrict__ energy,
                                       double4 *__restrict__ tmp_rows, double *__restrict__ tmp_sc) {
  const int m = iscal[IS_NROWS], first = iscal[IS_FIRST];
  const int moved = m - first;
  for (int d = blockIdx.x; d < moved; d += gridDim.x) {
    const int src = newidx[first + d];
    const double4 *r = hist + (size_t)src * L;
    double4 *o = tmp_rows + (size_t)d * L;
    for (int i = threadIdx.x; i < L; i += blockDim.x) o[i] = r[i];
    if (threadIdx.x == 0) {
      tmp_sc[3 * d] = t[src];
      tmp_sc[3 * d + 1] = mu[src];
      tmp_sc[3 * d + 2] = energy ? energy[src] : 0.0;
    }
  }
}

__global__ void sparsify_scatter_kernel(int L, const int32_t *__restrict__ iscal, double4 *__restrict__ hist,
                                        double *__restrict__ t, double *__restrict__ mu, double *__restrict__ energy,
                                        const double4 *__restrict__ tmp_rows, const double *__restrict__ tmp_sc) {
  const int m = iscal[IS_NROWS], first = iscal[IS_FIRST];
  const int moved = m - first;
  for (int d = blockIdx.x; d < moved; d += gridDim.x) {
    double4 *r = hist + (size_t)(first + d) * L;
    const double4 *o = tmp_rows + (size_t)d * L;
    for (int i = threadIdx.x; i < L; i += blockDim.x) r[i] = o[i];
    if (threadIdx.x == 0) {
      t[first + d] = tmp_sc[3 * d];
      mu[first + d] = tmp_sc[3 * d + 1];
      if (energy) energy[first + d] = tmp_sc[3 * d + 2];
    }
  }
}

}  // namespace

extern "C" int dmfe_set_sparsify_threshold(dmfe_ctx *ctx, double eps_sparse) {
  if (!ctx || !(eps_sparse >= 0.0)) return DMFE_EINVAL;
  ctx->eps_sparse = eps_sparse;
  return DMFE_OK;
}

extern "C" int dmfe_sparsify(dmfe_ctx *ctx, dmfe_state *st, int32_t protect_last, int32_t *n_rows_out,
                             uint8_t *keep_mask) {
  if (!ctx || !st || !st->t || !st->mu || !st->hist || protect_last < 0) return DMFE_EINVAL;
  const int L = ctx->p.L, N = st->n_rows;
  cudaStream_t s = ctx->stream;
  if (N < 3) {
    if (n_rows_out) *n_rows_out = N;
    if (keep_mask)
      for (int n = 0; n < N; ++n) keep_mask[n] = 1;
    return DMFE_OK;
  }
  if (N > ctx->sp_cap) {
    cudaFree(ctx->eps_sp);
    cudaFree(ctx->keep);
    cudaFree(ctx->newidx);
    ctx->eps_sp = nullptr;
    ctx->keep = ctx->newidx = nullptr;
    ctx->sp_cap = 0;
    const int cap = st->n_cap > N ? st->n_cap : N;
    CUDA_TRY(ctx, cudaMalloc(&ctx->eps_sp, sizeof(double) * (size_t)cap));
    CUDA_TRY(ctx, cudaMalloc(&ctx->keep, sizeof(int32_t) * (size_t)cap));
    CUDA_TRY(ctx, cudaMalloc(&ctx->newidx, sizeof(int32_t) * (size_t)cap));
    ctx->sp_cap = cap;
  }
  // rows 1.. can move; staging = (N-1) rows + 3 scalars per row
  const size_t need = ((size_t)(N - 1) * L * 4 + 3 * (size_t)(N - 1)) * sizeof(double);
  if (need > ctx->row_tmp_bytes) {
    cudaFree(ctx->row_tmp);
    ctx->row_tmp = nullptr;
    ctx->row_tmp_bytes = 0;
    CUDA_TRY(ctx, cudaMalloc(&ctx->row_tmp, need));
    ctx->row_tmp_bytes = need;
  }
  double4 *tmp_rows = (double4 *)ctx->row_tmp;
  double *tmp_sc = ctx->row_tmp + (size_t)(N - 1) * L * 4;
  sparsify_residual_kernel<<<N - 2, 256, 0, s>>>(L, N, st->t, (const double4 *)st->hist, ctx->eps_sp);
  sparsify_walk_kernel<<<1, 32, 0, s>>>(N, protect_last, ctx->eps_sparse > 0.0 ? ctx->eps_sparse : ctx->p.tol / 10.0, ctx->eps_sp, ctx->keep, ctx->newidx,
                                        ctx->iscal);
  const int nb = (N - 1 < 1184) ? N - 1 : 1184;
  sparsify_gather_kernel<<<nb, 128, 0, s>>>(L, ctx->iscal, ctx->newidx, (const double4 *)st->hist, st->t, st->mu,
                                            st->energy, tmp_rows, tmp_sc);
  sparsify_scatter_kernel<<<nb, 128, 0, s>>>(L, ctx->iscal, (double4 *)st->hist, st->t, st->mu, st->energy, tmp_rows,
                                             tmp_sc);
  CUDA_TRY(ctx, cudaGetLastError());
  CUDA_TRY(ctx, cudaMemcpyAsync(ctx->h_iscal, ctx->iscal, sizeof(int32_t) * IS_COUNT, cudaMemcpyDeviceToHost, s));
  if (keep_mask) {
    // test hook: flags back as int32, narrowed on the host
    int32_t *tmp = (int32_t *)malloc(sizeof(int32_t) * (size_t)N);
    if (!tmp) return DMFE_ENOMEM;
    cudaError_t e = cudaMemcpyAsync(tmp, ctx->keep, sizeof(int32_t) * (size_t)N, cudaMemcpyDeviceToHost, s);
    if (e == cudaSuccess) e = cudaStreamSynchronize(s);
    if (e != cudaSuccess) {
      free(tmp);
      ctx->cuda_err = (int)e;
      return DMFE_ECUDA;
    }
    for (int n = 0; n < N; ++n) keep_mask[n] = (uint8_t)tmp[n];
    free(tmp);
  }
  CUDA_TRY(ctx, cudaStreamSynchronize(s));
  st->n_rows = ctx->h_iscal[IS_NROWS];
  if (n_rows_out) *n_rows_out = st->n_rows;
  return DMFE_OK;
}
