// Measurement hooks of include/dmfe.h: per-launch timing of the pair kernel and a DFMA-only
// throughput probe (the FP64 roofline denominator is measured on the box, not assumed).
#include <stdlib.h>

#include "dmfe_internal.cuh"

namespace {

__global__ void __launch_bounds__(256) dfma_chain_kernel(int n_iter, double a, double b, double *sink) {
  double x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
  for (int k = 0; k < n_iter; k += 8) {
#pragma unroll
    for (int u = 0; u < 1; ++u) {
      x0 = fma(x0, a, b);
      x1 = fma(x1, a, b);
      x2 = fma(x2, a, b);
      x3 = fma(x3, a, b);
      x4 = fma(x4, a, b);
      x5 = fma(x5, a, b);
      x6 = fma(x6, a, b);
      x7 = fma(x7, a, b);
    }
  }
  const double s = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
  if (s == 123.456) sink[0] = s;  // never true; keeps the chain alive
}

// Load-path probe: every warp issues, per iteration, `nld` independent 256-bit loads from a small
// L1-resident buffer with a chosen lane pattern and `nfma` independent DFMAs (8 chains); clock64
// around the loop.  Answers two questions the pair kernel's design depends on: what a warp-wide
// 256-bit gather costs in the L1 data path, and how far FP64 issue overlaps with that traffic.
//   pattern 0: lane l reads cell l (coalesced, 1 KB)      1: lanes 2l, 2l+1 share a cell
//           2: all lanes read one cell (broadcast)        3: stencil-like, cell l/4 + (l & 3)
//           4: one cell per 128-byte line (32 lines)
//           5: coalesced, only lanes with (lane & 3) == 0 active      6: coalesced, 12 scattered lanes active
//           7: coalesced, lanes 0..7 active                           8: one cell per line, 12 scattered lanes
//           9: shared memory, lane-private pseudo-random cells (2 x 128-bit per cell)
//          10: no loads; every 'load' is 16 integer multiply-adds (issue-slot probe)
template <int pattern>
__global__ void __launch_bounds__(1024) load_path_probe_kernel(const double4 *buf, int ncell, int nld,
                                                               int nfma, int iters, double *sink,
                                                               long long *cycles) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  __shared__ double4 sbuf[1024];
  for (int k = threadIdx.x; k < 1024; k += blockDim.x) sbuf[k] = buf[k % ncell];
  __syncthreads();
  bool active = true;
  if (pattern == 5) active = (lane & 3) == 0;
  if (pattern == 6 || pattern == 8) active = (0x5A0B4C91u >> lane) & 1u;  // 12 lanes
  if (pattern == 7) active = lane < 8;
  unsigned off;
  if (pattern == 0 || (pattern >= 5 && pattern <= 7)) off = lane;
  else if (pattern == 1) off = lane >> 1;
  else if (pattern == 2) off = 0;
  else if (pattern == 3) off = (lane >> 2) + (lane & 3);
  else off = lane * 4;
  double a[8];
#pragma unroll
  for (int q = 0; q < 8; ++q) a[q] = 1.0 + q * 1e-3 + lane * 1e-6;
  double acc = 0.0;
  const long long t0 = clock64();
  for (int it = 0; it < iters; ++it) {
    for (int u = 0; u < nld; ++u) {
      const unsigned idx = (warp * 97u + off + u * 131u + it * 7u) & (unsigned)(ncell - 1);
      double4 v = make_double4(0.0, 0.0, 0.0, 0.0);
      if (pattern == 10) {  // no load: 16 dependent-free integer multiply-adds per 'load'
        unsigned z = idx;
#pragma unroll
        for (int q = 0; q < 16; ++q) z = z * 2654435761u + (unsigned)(q + it);
        if (z == 0x12345u) acc += 1.0;
      } else if (pattern == 9) {
        const unsigned sidx = (idx * 2654435761u >> 7) & 1023u;
        const double2 *sp = reinterpret_cast<const double2 *>(sbuf + sidx);
        const double2 lo = sp[0], hi = sp[1];
        v = make_double4(lo.x, lo.y, hi.x, hi.y);
      } else if (active) {
        asm volatile("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];"
                     : "=d"(v.x), "=d"(v.y), "=d"(v.z), "=d"(v.w)
                     : "l"(buf + idx));
      }
      acc += (v.x + v.y) + (v.z + v.w);
    }
    for (int f = 0; f < nfma; f += 8) {
#pragma unroll
      for (int q = 0; q < 8; ++q) a[q] = fma(a[q], 1.0000001, 1e-9);
    }
  }
  const long long t1 = clock64();
#pragma unroll
  for (int q = 0; q < 8; ++q) acc += a[q];
  if (acc == 123.456) sink[0] = acc;
  if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
}

}  // namespace

extern "C" {

int dmfe_enable_timing(dmfe_ctx *ctx, int32_t on) {
  if (!ctx) return DMFE_EINVAL;
  ctx->timing_on = on ? 1 : 0;
  ctx->ev_n = 0;
  return DMFE_OK;
}

int dmfe_last_kernel_ms(dmfe_ctx *ctx, float *ms) {
  if (!ctx || !ms || ctx->ev_n < 1) return DMFE_EINVAL;
  const int k = ctx->ev_n - 1;
  CUDA_TRY(ctx, cudaEventSynchronize(ctx->ev[2 * k + 1]));
  CUDA_TRY(ctx, cudaEventElapsedTime(ms, ctx->ev[2 * k], ctx->ev[2 * k + 1]));
  return DMFE_OK;
}

int dmfe_kernel_time_stats(dmfe_ctx *ctx, int32_t *n_launches, double *total_ms, double *min_ms) {
  if (!ctx || !n_launches || !total_ms) return DMFE_EINVAL;
  double tot = 0.0, mn = 1e300;
  for (int k = 0; k < ctx->ev_n; ++k) {
    float ms = 0.f;
    CUDA_TRY(ctx, cudaEventSynchronize(ctx->ev[2 * k + 1]));
    CUDA_TRY(ctx, cudaEventElapsedTime(&ms, ctx->ev[2 * k], ctx->ev[2 * k + 1]));
    tot += (double)ms;
    if ((double)ms < mn) mn = (double)ms;
  }
  *n_launches = ctx->ev_n;
  *total_ms = tot;
  if (min_ms) *min_ms = ctx->ev_n ? mn : 0.0;
  return DMFE_OK;
}

int dmfe_probe_fp64_tflops(dmfe_ctx *ctx, int32_t n_iter, double *tflops, int32_t *sm_count) {
  if (!ctx || !tflops || n_iter < 8) return DMFE_EINVAL;
  int dev = 0, sms = 0;
  CUDA_TRY(ctx, cudaGetDevice(&dev));
  CUDA_TRY(ctx, cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  if (sm_count) *sm_count = sms;
  n_iter -= n_iter % 8;
  const int blocks = sms * 8, threads = 256;
  cudaEvent_t e0, e1;
  CUDA_TRY(ctx, cudaEventCreate(&e0));
  CUDA_TRY(ctx, cudaEventCreate(&e1));
  float best = 1e30f;
  for (int rep = 0; rep < 4; ++rep) {
    cudaEventRecord(e0, ctx->stream);
    dfma_chain_kernel<<<blocks, threads, 0, ctx->stream>>>(n_iter, 0.999999, 1e-7, ctx->scal + SC_COUNT - 1);
    cudaEventRecord(e1, ctx->stream);
    cudaError_t e = cudaEventSynchronize(e1);
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    if (e != cudaSuccess) {
      cudaEventDestroy(e0);
      cudaEventDestroy(e1);
      ctx->cuda_err = (int)e;
      return DMFE_ECUDA;
    }
    if (rep > 0 && ms < best) best = ms;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  const double flops = 2.0 * (double)n_iter * (double)blocks * (double)threads;
  *tflops = flops / ((double)best * 1e-3) / 1e12;
  return DMFE_OK;
}

int dmfe_probe_load_path(dmfe_ctx *ctx, int32_t pattern, int32_t n_loads, int32_t n_dfma, int32_t threads,
                         double *cycles_per_warp_iter) {
  if (!ctx || !cycles_per_warp_iter || pattern < 0 || pattern > 10 || n_loads < 0 || n_dfma < 0 ||
      (n_dfma % 8) || threads < 32 || threads > 1024 || (threads % 32))
    return DMFE_EINVAL;
  const int ncell = 1024, iters = 2000, sms = ctx->sm_count;
  double4 *buf = nullptr;
  long long *cyc = nullptr;
  CUDA_TRY(ctx, cudaMalloc(&buf, sizeof(double4) * ncell));
  cudaError_t e = cudaMalloc(&cyc, sizeof(long long) * sms);
  if (e == cudaSuccess) e = cudaMemsetAsync(buf, 0, sizeof(double4) * ncell, ctx->stream);
  for (int rep = 0; rep < 2 && e == cudaSuccess; ++rep) {  // first launch warms the cache
#define DMFE_PROBE(P_)                                                                                     \
  case P_:                                                                                                 \
    load_path_probe_kernel<P_><<<sms, threads, 0, ctx->stream>>>(buf, ncell, n_loads, n_dfma, rep ? iters : 10, \
                                                                 ctx->scal + SC_COUNT - 1, cyc);           \
    break
    switch (pattern) {
      DMFE_PROBE(0);
      DMFE_PROBE(1);
      DMFE_PROBE(2);
      DMFE_PROBE(3);
      DMFE_PROBE(4);
      DMFE_PROBE(5);
      DMFE_PROBE(6);
      DMFE_PROBE(7);
      DMFE_PROBE(8);
      DMFE_PROBE(9);
      DMFE_PROBE(10);
    }
#undef DMFE_PROBE
    e = cudaGetLastError();
  }
  long long *h = (long long *)malloc(sizeof(long long) * sms);
  if (e == cudaSuccess && h) e = cudaMemcpyAsync(h, cyc, sizeof(long long) * sms, cudaMemcpyDeviceToHost, ctx->stream);
  if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
  double avg = 0.0;
  if (e == cudaSuccess && h)
    for (int k = 0; k < sms; ++k) avg += (double)h[k] / sms;
  free(h);
  cudaFree(buf);
  cudaFree(cyc);
  if (e != cudaSuccess) {
    ctx->cuda_err = (int)e;
    return DMFE_ECUDA;
  }
  *cycles_per_warp_iter = avg / ((double)iters * (threads / 32));  // SM cycles per warp-iteration
  return DMFE_OK;
}

}  // extern "C"
