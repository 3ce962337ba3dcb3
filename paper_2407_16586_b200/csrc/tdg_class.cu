// tdg_class.cu — instantiates the gradient kernel of ONE quartet class; compile with
// -DTDG_LA=.. -DTDG_LB=.. -DTDG_LC=.. -DTDG_LD=.. (one kernel per non-redundant angular class).
#include "tdg_gradb.cuh"

#if !defined(TDG_LA) || !defined(TDG_LB) || !defined(TDG_LC) || !defined(TDG_LD)
#error "compile with -DTDG_LA=<la> -DTDG_LB=<lb> -DTDG_LC=<lc> -DTDG_LD=<ld>"
#endif

static void launch(const KParams& P, int nblocks, cudaStream_t s) {
  typedef QC<TDG_LA, TDG_LB, TDG_LC, TDG_LD> C;
  // the shared-memory attribute is per device and the call is cheap: set it on every launch (contexts may live on several devices)
  if constexpr (C::SMALL) {   // one thread per quartet, registers only (tdg_grad.cuh)
    constexpr int smem = (C::RYS_SH_DOUBLES + TDG_ACC_DOUBLES) * (int)sizeof(double);
    cudaFuncSetAttribute(tdg_grad_kernel<TDG_LA, TDG_LB, TDG_LC, TDG_LD>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    tdg_grad_kernel<TDG_LA, TDG_LB, TDG_LC, TDG_LD><<<dim3(nblocks, C::NROLE), TDG_WARPS * TDG_WARP, smem, s>>>(P);
  } else {                    // one block per quartet, 2-D integrals in shared memory (tdg_gradb.cuh)
    typedef QB<TDG_LA, TDG_LB, TDG_LC, TDG_LD> B;
    constexpr int smem = B::SMEM_DOUBLES * (int)sizeof(double);
    cudaFuncSetAttribute(tdg_gradb_kernel<TDG_LA, TDG_LB, TDG_LC, TDG_LD>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    tdg_gradb_kernel<TDG_LA, TDG_LB, TDG_LC, TDG_LD><<<nblocks, B::G, smem, s>>>(P);
  }
}
#define TDG_CAT2(a, b, c, d, e) a##b##c##d##e
#define TDG_CAT(a, b, c, d, e) TDG_CAT2(a, b, c, d, e)
tdg_launch_fn TDG_CAT(tdg_class_launcher_, TDG_LA, TDG_LB, TDG_LC, TDG_LD)() { return &launch; }
