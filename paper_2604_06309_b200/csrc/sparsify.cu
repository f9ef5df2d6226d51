// Selective history reduction.  For an interior row n with neighbours n-1, n+1
// the residual of Eq.(26) is the difference between the integral over [t_{n-1}, t_{n+1}] of the
// two cubic Hermite pieces through row n and of the single piece that skips it (closed form),
// eps_sparse[n] = sum_i |Delta^C_i| + |Delta^R_i| (Eq.(27)).  Walking n upward, row n is dropped if
// eps_sparse[n] < tol/10 and the walk continues at n+2, else at n+1.  Because a
// candidate's neighbours are never removed before it is tested, all residuals are computed in
// parallel on the uncompacted history; the walk and the index scan are O(N) integer work; the
// rows, t, mu and E are compacted on the device, in place.
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

// Greedy walk + exclusive scan of the keep flags, one CTA.  Candidates are the rows
// 1 .. last (row 0, the last protect_last rows and row N-1 are kept).  Because a candidate's
// neighbours are never removed before it is tested, "drop n if flagged, then continue at n+2" is
// the same as: in every maximal run of flagged candidates drop the 1st, 3rd, 5th ...  A thread owns
// a contiguous chunk of rows; the position inside a run comes from a max-scan of "last unflagged
// row", the compacted index from a sum-scan of the keep flags.  newidx[d] = source row of
// compacted row d; iscal[IS_NROWS] = rows kept, iscal[IS_FIRST] = first row that moves.
constexpr int WALK_THREADS = 1024;

__global__ void __launch_bounds__(WALK_THREADS) sparsify_walk_kernel(int N, int protect_last, double thr,
                                                                     const double *__restrict__ eps_sp,
                                                                     int32_t *__restrict__ keep,
                                                                     int32_t *__restrict__ newidx,
                                                                     int32_t *__restrict__ iscal) {
  __shared__ int s_last[WALK_THREADS];  // last unflagged row of each chunk (-1: none)
  __shared__ int s_cnt[WALK_THREADS];   // rows kept in each chunk
  const int tid = threadIdx.x;
  const int chunk = (N + WALK_THREADS - 1) / WALK_THREADS;
  const int lo = tid * chunk, hi = min(N, lo + chunk);
  int last_c = N - 1 - protect_last;
  if (last_c > N - 2) last_c = N - 2;
  auto flagged = [&](int n) { return n >= 1 && n <= last_c && eps_sp[n] < thr; };
  int lastun = -1;
  for (int n = lo; n < hi; ++n)
    if (!flagged(n)) lastun = n;
  s_last[tid] = lastun;
  __syncthreads();
  // inclusive max-scan over the chunks (Hillis-Steele)
  for (int o = 1; o < WALK_THREADS; o <<= 1) {
    const int v = (tid >= o) ? s_last[tid - o] : -1;
    __syncthreads();
    if (v > s_last[tid]) s_last[tid] = v;
    __syncthreads();
  }
  int prev = (tid > 0) ? s_last[tid - 1] : -1;  // last unflagged row before this chunk
  int cnt = 0;
  for (int n = lo; n < hi; ++n) {
    int k = 1;
    if (flagged(n)) {
      k = ((n - prev) & 1) ? 0 : 1;  // position in the run = n - prev: odd positions are dropped
    } else {
      prev = n;
    }
    keep[n] = k;
    cnt += k;
  }
  s_cnt[tid] = cnt;
  __syncthreads();
  for (int o = 1; o < WALK_THREADS; o <<= 1) {  // inclusive sum-scan
    const int v = (tid >= o) ? s_cnt[tid - o] : 0;
    __syncthreads();
    s_cnt[tid] += v;
    __syncthreads();
  }
  int m = s_cnt[tid] - cnt;  // compacted index of this chunk's first kept row
  for (int n = lo; n < hi; ++n)
    if (keep[n]) newidx[m++] = n;
  if (tid == WALK_THREADS - 1) iscal[IS_NROWS] = s_cnt[tid];
  // first row that moves = first dropped row
  __shared__ int s_first;
  if (tid == 0) s_first = N;
  __syncthreads();
  for (int n = lo; n < hi; ++n)
    if (!keep[n]) {
      atomicMin(&s_first, n);
      break;
    }
  __syncthreads();
  if (tid == 0) iscal[IS_FIRST] = s_first;
}

// Compaction in place, in chunks of `rows` destination rows through a bounded staging buffer: rows
// only move down (source >= destination), and the sources of a chunk lie at or above its own
// destinations, hence above every destination of the chunks before it -- so chunks run one after
// the other, each as gather (sources -> staging) then scatter (staging -> destinations).
__global__ void sparsify_gather_kernel(int L, int d0, int rows, const int32_t *__restrict__ iscal,
                                       const int32_t *__restrict__ newidx, const double4 *__restrict__ hist,
                                       const double *__restrict__ t, const double *__restrict__ mu,
                                       const double *__restrict__ energy, double4 *__restrict__ tmp_rows,
                                       double *__restrict__ tmp_sc) {
  const int m = iscal[IS_NROWS], first = iscal[IS_FIRST];
  const int moved = m - first;
  for (int r = blockIdx.x; r < rows && d0 + r < moved; r += gridDim.x) {
    const int src = newidx[first + d0 + r];
    const double4 *x = hist + (size_t)src * L;
    double4 *o = tmp_rows + (size_t)r * L;
    for (int i = threadIdx.x; i < L; i += blockDim.x) o[i] = x[i];
    if (threadIdx.x == 0) {
      tmp_sc[3 * r] = t[src];
      tmp_sc[3 * r + 1] = mu[src];
      tmp_sc[3 * r + 2] = energy ? energy[src] : 0.0;
    }
  }
}

__global__ void sparsify_scatter_kernel(int L, int d0, int rows, const int32_t *__restrict__ iscal,
                                        double4 *__restrict__ hist, double *__restrict__ t, double *__restrict__ mu,
                                        double *__restrict__ energy, const double4 *__restrict__ tmp_rows,
                                        const double *__restrict__ tmp_sc) {
  const int m = iscal[IS_NROWS], first = iscal[IS_FIRST];
  const int moved = m - first;
  for (int r = blockIdx.x; r < rows && d0 + r < moved; r += gridDim.x) {
    double4 *x = hist + (size_t)(first + d0 + r) * L;
    const double4 *o = tmp_rows + (size_t)r * L;
    for (int i = threadIdx.x; i < L; i += blockDim.x) x[i] = o[i];
    if (threadIdx.x == 0) {
      t[first + d0 + r] = tmp_sc[3 * r];
      mu[first + d0 + r] = tmp_sc[3 * r + 1];
      if (energy) energy[first + d0 + r] = tmp_sc[3 * r + 2];
    }
  }
}

}  // namespace

extern "C" int dmfe_sparsify(dmfe_ctx *ctx, dmfe_state *st, int32_t protect_last, int32_t *n_rows_out,
                             uint8_t *keep_mask) {
  if (ctx && ctx->p.values_only) return DMFE_EINVAL;  // the integrator keeps the Hermite history
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
  // bounded staging for the compaction: at most 8 MB of rows (at least one) + 3 scalars per row
  int chunk = (int)((size_t)(8u << 20) / ((size_t)L * 32));
  if (chunk < 1) chunk = 1;
  if (chunk > N - 1) chunk = N - 1;
  const size_t need = ((size_t)chunk * L * 4 + 3 * (size_t)chunk) * sizeof(double);
  if (need > ctx->row_tmp_bytes) {
    cudaFree(ctx->row_tmp);
    ctx->row_tmp = nullptr;
    ctx->row_tmp_bytes = 0;
    CUDA_TRY(ctx, cudaMalloc(&ctx->row_tmp, need));
    ctx->row_tmp_bytes = need;
  }
  double4 *tmp_rows = (double4 *)ctx->row_tmp;
  double *tmp_sc = ctx->row_tmp + (size_t)chunk * L * 4;
  sparsify_residual_kernel<<<N - 2, 256, 0, s>>>(L, N, st->t, (const double4 *)st->hist, ctx->eps_sp);
  sparsify_walk_kernel<<<1, WALK_THREADS, 0, s>>>(N, protect_last, ctx->p.tol / 10.0, ctx->eps_sp, ctx->keep,
                                                  ctx->newidx, ctx->iscal);
  // the number of moved rows is known on the device only: the chunk loop covers the worst case
  // (all of rows 1 .. N-1 move) and the kernels of chunks beyond the moved range find nothing to do;
  // the host learns the new row count first, to stop launching once that range is covered
  CUDA_TRY(ctx, cudaMemcpyAsync(ctx->h_iscal, ctx->iscal, sizeof(int32_t) * IS_COUNT, cudaMemcpyDeviceToHost, s));
  CUDA_TRY(ctx, cudaStreamSynchronize(s));
  const int moved = ctx->h_iscal[IS_NROWS] - ctx->h_iscal[IS_FIRST];
  for (int d0 = 0; d0 < moved; d0 += chunk) {
    const int nb = chunk < 1184 ? chunk : 1184;
    sparsify_gather_kernel<<<nb, 128, 0, s>>>(L, d0, chunk, ctx->iscal, ctx->newidx, (const double4 *)st->hist, st->t,
                                              st->mu, st->energy, tmp_rows, tmp_sc);
    sparsify_scatter_kernel<<<nb, 128, 0, s>>>(L, d0, chunk, ctx->iscal, (double4 *)st->hist, st->t, st->mu,
                                               st->energy, tmp_rows, tmp_sc);
  }
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
  ctx->rowtab_dirty = 1;  // the rows moved
  if (n_rows_out) *n_rows_out = st->n_rows;
  return DMFE_OK;
}
