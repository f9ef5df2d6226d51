// Instantiations and launcher of the pair kernel for any stencil size (pairs_generic.cuh).
#include "pairs_generic.cuh"

using namespace dmfe_rhs;

int dmfe_launch_pairs_generic(dmfe_ctx *ctx, const RhsArgs &a, int grid) {
  const int L = a.L, M = a.M;
  const long long pairs_cta = (long long)L * L / grid;
  // shared-memory copies of cur [L] double2 and blo [L] int32 when they fit, and of rowtab [M]
  // double2 too when that fits and a CTA has enough pairs to amortise copying M entries
  const size_t smem1 = 20 * (size_t)L, smem2 = smem1 + 16 * (size_t)M;
  const int mode = (smem2 <= (size_t)ctx->smem_max && 2LL * M <= pairs_cta) ? 2
                   : (smem1 <= (size_t)ctx->smem_max ? 1 : 0);
  const size_t smem = mode == 2 ? smem2 : (mode == 1 ? smem1 : 0);
  const int pd = ctx->model.pmax <= 3 ? 3 : (ctx->model.pmax == 4 ? 4 : 0);
#define DMFE_LAUNCH_K(KFN)                                                                              \
  do {                                                                                                  \
    auto kfn = KFN;                                                                                     \
    if (smem + 4096 > 48 * 1024)                                                                        \
      CUDA_TRY(ctx, cudaFuncSetAttribute(kfn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem)); \
    CUDA_TRY(ctx, launch_pdl(kfn, grid, RHS_THREADS, smem, ctx->stream, a, ctx->model));                \
  } while (0)
#define DMFE_LAUNCH_G(S_, PD_)                                \
  do {                                                        \
    if (mode == 2)                                            \
      DMFE_LAUNCH_K((history_integrals_kernel<S_, PD_, 2>));  \
    else if (mode == 1)                                       \
      DMFE_LAUNCH_K((history_integrals_kernel<S_, PD_, 1>));  \
    else                                                      \
      DMFE_LAUNCH_K((history_integrals_kernel<S_, PD_, 0>));  \
  } while (0)
#define DMFE_LAUNCH_GS(S_)   \
  do {                       \
    if (pd == 3)             \
      DMFE_LAUNCH_G(S_, 3);  \
    else if (pd == 4)        \
      DMFE_LAUNCH_G(S_, 4);  \
    else                     \
      DMFE_LAUNCH_G(S_, 0);  \
  } while (0)
#define DMFE_LAUNCH_LOG(S_)                                          \
  do {                                                              \
    if (mode == 2)                                                  \
      DMFE_LAUNCH_K((history_integrals_kernel<S_, 0, 2, true>));    \
    else if (mode == 1)                                             \
      DMFE_LAUNCH_K((history_integrals_kernel<S_, 0, 1, true>));    \
    else                                                            \
      DMFE_LAUNCH_K((history_integrals_kernel<S_, 0, 0, true>));    \
  } while (0)
  if (ctx->p.log_r) {  // logarithmic interpolation of the response history: run-time degree of f only
    switch (ctx->p.stencil) {
      case 2: DMFE_LAUNCH_LOG(2); break;
      case 4: DMFE_LAUNCH_LOG(4); break;
      case 6: DMFE_LAUNCH_LOG(6); break;
      case 8: DMFE_LAUNCH_LOG(8); break;
      case 10: DMFE_LAUNCH_LOG(10); break;
      default: return DMFE_EINVAL;
    }
    return DMFE_OK;
  }
#undef DMFE_LAUNCH_LOG
  switch (ctx->p.stencil) {
    case 2: DMFE_LAUNCH_GS(2); break;
    case 6: DMFE_LAUNCH_GS(6); break;
    case 8: DMFE_LAUNCH_GS(8); break;
    case 10: DMFE_LAUNCH_GS(10); break;
    default: return DMFE_EINVAL;
  }
#undef DMFE_LAUNCH_GS
#undef DMFE_LAUNCH_G
#undef DMFE_LAUNCH_K
  return DMFE_OK;
}
