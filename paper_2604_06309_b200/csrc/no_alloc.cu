// dmfe_history_integrals_static: the north-star call for callers that may not allocate (code under CUDA graph
// capture, tight serving loops, harnesses that forbid cudaMalloc).  Same kernels, same arithmetic and same
// results as dmfe_history_integrals (Hermite history); the only difference is where the per-call tables of the
// pre-pass live: packed current row, row table, row brackets, mu weights, jtop and the cubic coefficient tables
// (the "O(L) scratch" of dmfe_ctx, of which the row table is grown with cudaMalloc on demand by the ordinary
// path) are carved out of ONE file-scope device array of fixed size,
//
//     DMFE_STATIC_MAX_L = 4096 grid nodes, DMFE_STATIC_MAX_ROWS = 16384 history rows: 1 245 440 bytes,
//
// which every GPU that loads libdmfe.so holds until the process exits.  Larger problems are refused with
// DMFE_ETOOLARGE.  The entry point calls no cudaMalloc / cudaFree and no allocating library routine: a
// cudaMemsetAsync of the slices that must start at zero, the pre-pass and the pair kernel, all on the context's
// stream.
//
// The array's name is a device symbol: in host code it is a host-side stand-in, not a device address.  The
// address is resolved with cudaGetSymbolAddress, once per device, with that device current (dmfe_static_init, or
// the first call on a device), and that pointer is what the kernels get.
//
// Sharing: every call on a device, from every context, uses the same array, and it keeps the last call's
// contents.  Calls on one stream are ordered and safe; two calls that overlap on the GPU (different streams
// without an event between them, or two host threads) race on the tables and give wrong results.
#include <string.h>

#include "dmfe_internal.cuh"

namespace {

constexpr size_t align256(size_t n) { return (n + 255) & ~(size_t)255; }

constexpr size_t NA_L = DMFE_STATIC_MAX_L, NA_ROWS = DMFE_STATIC_MAX_ROWS;
// slices (bytes), each 256-byte aligned; sizes as allocated by dmfe_create for the same tables
constexpr size_t OFF_CUR = 0;                                                  // [L] double2
constexpr size_t OFF_BLO = OFF_CUR + align256(sizeof(double2) * NA_L);        // [L] int32
constexpr size_t OFF_MUW = OFF_BLO + align256(sizeof(int32_t) * NA_L);        // [L] double2
constexpr size_t OFF_BR = OFF_MUW + align256(sizeof(double2) * NA_L);         // [L] int2
constexpr size_t OFF_JTOP = OFF_BR + align256(sizeof(int2) * NA_L);           // [L] int32
constexpr size_t OFF_COEFM = OFF_JTOP + align256(sizeof(int32_t) * NA_L);     // [L][8] double
constexpr size_t OFF_COEFT = OFF_COEFM + align256(sizeof(double) * 8 * NA_L); // [L][16] double
constexpr size_t OFF_ROWTAB = OFF_COEFT + align256(sizeof(double) * 16 * NA_L);  // [ROWS] double2
constexpr size_t OFF_SCAL = OFF_ROWTAB + align256(sizeof(double2) * NA_ROWS); // [SC_COUNT] double
constexpr size_t NA_BYTES = OFF_SCAL + align256(sizeof(double) * SC_COUNT);

static __device__ __align__(256) unsigned char g_static_scratch[NA_BYTES];

constexpr int NA_MAX_DEVICES = 64;
unsigned char *g_scratch_ptr[NA_MAX_DEVICES];  // device address of g_static_scratch on each device, once resolved

// device address of the array on the current device (resolved on first use, with that device current)
int scratch_for_current_device(dmfe_ctx *ctx, unsigned char **out) {
  int dev = -1;
  CUDA_TRY(ctx, cudaGetDevice(&dev));
  if (dev < 0 || dev >= NA_MAX_DEVICES) return DMFE_EINVAL;
  if (!g_scratch_ptr[dev]) {
    void *p = nullptr;
    CUDA_TRY(ctx, cudaGetSymbolAddress(&p, g_static_scratch));
    if (!p) return DMFE_ECUDA;
    g_scratch_ptr[dev] = static_cast<unsigned char *>(p);
  }
  *out = g_scratch_ptr[dev];
  return DMFE_OK;
}

}  // namespace

extern "C" {

int dmfe_static_limits(int32_t *max_L, int32_t *max_rows, int64_t *bytes) {
  if (max_L) *max_L = (int32_t)NA_L;
  if (max_rows) *max_rows = (int32_t)NA_ROWS;
  if (bytes) *bytes = (int64_t)NA_BYTES;
  return DMFE_OK;
}

int dmfe_static_init(dmfe_ctx *ctx) {
  if (!ctx) return DMFE_EINVAL;
  if (ctx->p.L > (int)NA_L) return DMFE_ETOOLARGE;
  unsigned char *base = nullptr;
  const int rc = scratch_for_current_device(ctx, &base);
  if (rc != DMFE_OK) return rc;
  CUDA_TRY(ctx, cudaMemsetAsync(base, 0, NA_BYTES, ctx->stream));
  return DMFE_OK;
}

int dmfe_history_integrals_static(dmfe_ctx *ctx, const dmfe_grid *g, const dmfe_rhs_out *out) {
  if (!ctx || !g || !out) return DMFE_EINVAL;
  if (g->n_rows < 2 || g->n_rows > g->n_cap || !g->t || !g->mu || !g->hist) return DMFE_EINVAL;
  if (ctx->p.values_only) return DMFE_EINVAL;  // Hermite history only
  const int L = ctx->p.L, M = g->n_rows - 1;
  if (L > (int)NA_L || M > (int)NA_ROWS) return DMFE_ETOOLARGE;
  unsigned char *base = nullptr;
  int rc = scratch_for_current_device(ctx, &base);
  if (rc != DMFE_OK) return rc;
  // what must not carry over from the last call: the search hints (any value gives the same rows; zero makes
  // a call independent of its predecessors) and the scalar block
  CUDA_TRY(ctx, cudaMemsetAsync(base + OFF_BLO, 0, sizeof(int32_t) * (size_t)L, ctx->stream));
  CUDA_TRY(ctx, cudaMemsetAsync(base + OFF_SCAL, 0, sizeof(double) * SC_COUNT, ctx->stream));
  // run the ordinary launcher with the context's scratch pointers pointing into the static array
  struct Saved {
    double2 *cur, *muw, *rowtab;
    int32_t *blo, *jtop;
    int2 *br;
    double *coefM, *coefT, *scal;
    int32_t rowtab_cap;
    int rowtab_dirty, timing_on;
  } sv = {ctx->cur,   ctx->muw,   ctx->rowtab, ctx->blo,        ctx->jtop,         ctx->br,
          ctx->coefM, ctx->coefT, ctx->scal,   ctx->rowtab_cap, ctx->rowtab_dirty, ctx->timing_on};
  ctx->cur = reinterpret_cast<double2 *>(base + OFF_CUR);
  ctx->blo = reinterpret_cast<int32_t *>(base + OFF_BLO);
  ctx->muw = reinterpret_cast<double2 *>(base + OFF_MUW);
  ctx->br = reinterpret_cast<int2 *>(base + OFF_BR);
  ctx->jtop = reinterpret_cast<int32_t *>(base + OFF_JTOP);
  ctx->coefM = reinterpret_cast<double *>(base + OFF_COEFM);
  ctx->coefT = reinterpret_cast<double *>(base + OFF_COEFT);
  ctx->rowtab = reinterpret_cast<double2 *>(base + OFF_ROWTAB);
  ctx->scal = reinterpret_cast<double *>(base + OFF_SCAL);
  ctx->rowtab_cap = (int32_t)NA_ROWS;  // M <= NA_ROWS was checked: the launcher's grow-on-demand branch cannot run
  ctx->timing_on = 0;                  // the timing hook creates events lazily: not on this path
  rc = dmfe_launch_rhs(ctx, M, M, g->t, g->mu, g->hist, out);
  ctx->cur = sv.cur, ctx->muw = sv.muw, ctx->rowtab = sv.rowtab, ctx->blo = sv.blo, ctx->jtop = sv.jtop;
  ctx->br = sv.br, ctx->coefM = sv.coefM, ctx->coefT = sv.coefT, ctx->scal = sv.scal;
  ctx->rowtab_cap = sv.rowtab_cap, ctx->rowtab_dirty = sv.rowtab_dirty, ctx->timing_on = sv.timing_on;
  return rc;
}

}  // extern "C"
