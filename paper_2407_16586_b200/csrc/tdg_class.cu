// tdg_class.cu — instantiates the gradient kernel of ONE quartet class; compile with
// -DTDG_LA=.. -DTDG_LB=.. -DTDG_LC=.. -DTDG_LD=.. (one kernel per non-redundant angular class).
#include "tdg_grad.cuh"

#if !defined(TDG_LA) || !defined(TDG_LB) || !defined(TDG_LC) || !defined(TDG_LD)
#error "compile with -DTDG_LA=<la> -DTDG_LB=<lb> -DTDG_LC=<lc> -DTDG_LD=<ld>"
#endif

static void launch(const KParams& P, int nblocks, cudaStream_t s) {
  typedef QC<TDG_LA, TDG_LB, TDG_LC, TDG_LD> C;
  constexpr int smem = (C::RYS_SH_DOUBLES + TDG_ACC_DOUBLES) * (int)sizeof(double);
  static bool attr_set = false;
  if (!attr_set) {
    cudaFuncSetAttribute(tdg_grad_kernel<TDG_LA, TDG_LB, TDG_LC, TDG_LD>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    attr_set = true;
  }
  tdg_grad_kernel<TDG_LA, TDG_LB, TDG_LC, TDG_LD><<<dim3(nblocks, C::NROLE), TDG_WARPS * TDG_WARP, smem, s>>>(P);
}
#define TDG_CAT2(a, b, c, d, e) a##b##c##d##e
#define TDG_CAT(a, b, c, d, e) TDG_CAT2(a, b, c, d, e)
tdg_launch_fn TDG_CAT(tdg_class_launcher_, TDG_LA, TDG_LB, TDG_LC, TDG_LD)() { return &launch; }
