// tdg_class.cu — instantiates the gradient kernels of one bra pair class (compile with -DTDG_LA=.. -DTDG_LB=..);
// one kernel per non-redundant angular class: ket pair class <= bra pair class.
#include "tdg_grad.cuh"

#ifndef TDG_LA
#error "compile with -DTDG_LA=<la> -DTDG_LB=<lb>"
#endif
#define PCLS(la, lb) ((la) * ((la) + 1) / 2 + (lb))

template <int LC, int LD>
static void launch(const KParams& P, int nblocks, cudaStream_t s) {
  typedef QC<TDG_LA, TDG_LB, LC, LD> C;
  constexpr int smem = (C::RYS_SH_DOUBLES + TDG_ACC_DOUBLES) * (int)sizeof(double);
  static bool attr_set = false;
  if (!attr_set && smem > 0) {
    cudaFuncSetAttribute(tdg_grad_kernel<TDG_LA, TDG_LB, LC, LD>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    attr_set = true;
  }
  tdg_grad_kernel<TDG_LA, TDG_LB, LC, LD><<<dim3(nblocks, C::NROLE), TDG_WARPS * TDG_WARP, smem, s>>>(P);
}
template <int LC, int LD>
static tdg_launch_fn pick() {
  if constexpr (PCLS(LC, LD) <= PCLS(TDG_LA, TDG_LB) && LC <= TDG_LMAX_BUILD) return &launch<LC, LD>;
  else return nullptr;
}
#define TDG_CAT2(a, b, c) a##b##c
#define TDG_CAT(a, b, c) TDG_CAT2(a, b, c)
tdg_launch_fn TDG_CAT(tdg_class_launcher_, TDG_LA, TDG_LB)(int lc, int ld) {
  switch (PCLS(lc, ld)) {
    case 0: return pick<0, 0>();
    case 1: return pick<1, 0>();
    case 2: return pick<1, 1>();
    case 3: return pick<2, 0>();
    case 4: return pick<2, 1>();
    case 5: return pick<2, 2>();
    case 6: return pick<3, 0>();
    case 7: return pick<3, 1>();
    case 8: return pick<3, 2>();
    case 9: return pick<3, 3>();
  }
  return nullptr;
}
