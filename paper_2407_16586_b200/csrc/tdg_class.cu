// tdg_class.cu — instantiates the gradient kernel of ONE (quartet class, role); compile with
// -DTDG_LA=.. -DTDG_LB=.. -DTDG_LC=.. -DTDG_LD=.. -DTDG_ROLE=.. (one kernel per non-redundant angular class, PAPER.md:309;
// classes with many function quartets are split into roles, tdg_grad.cuh).
#include "tdg_gradb.cuh"
#include "tdg_fock.cuh"

#if !defined(TDG_LA) || !defined(TDG_LB) || !defined(TDG_LC) || !defined(TDG_LD) || !defined(TDG_ROLE)
#error "compile with -DTDG_LA=<la> -DTDG_LB=<lb> -DTDG_LC=<lc> -DTDG_LD=<ld> -DTDG_ROLE=<role>"
#endif

static void launch(const KParams& P, int nblocks, cudaStream_t s) {
  typedef QC<TDG_LA, TDG_LB, TDG_LC, TDG_LD> C;
  // the shared-memory attribute is per device and the call is cheap: set it on every launch (contexts may live on several devices)
  if constexpr (C::SMALL) {   // one thread per quartet, registers only (tdg_grad.cuh)
    constexpr int smem = (C::RYS_SH_DOUBLES + C::IJ_SH_DOUBLES + TDG_ACC_DOUBLES) * (int)sizeof(double);
    cudaFuncSetAttribute(tdg_grad_kernel<TDG_LA, TDG_LB, TDG_LC, TDG_LD, TDG_ROLE>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    tdg_grad_kernel<TDG_LA, TDG_LB, TDG_LC, TDG_LD, TDG_ROLE><<<nblocks, TDG_WARPS * TDG_WARP, smem, s>>>(P);
  } else {                    // one block per quartet, 2-D integrals in shared memory (tdg_gradb.cuh)
    static_assert(C::SMALL || TDG_ROLE == 0, "the block-per-quartet kernel has one role");
    typedef QB<TDG_LA, TDG_LB, TDG_LC, TDG_LD> B;
    constexpr int smem = B::SMEM_DOUBLES * (int)sizeof(double);
    cudaFuncSetAttribute(tdg_gradb_kernel<TDG_LA, TDG_LB, TDG_LC, TDG_LD, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    tdg_gradb_kernel<TDG_LA, TDG_LB, TDG_LC, TDG_LD, 0><<<dim3(nblocks, TDG_GRADB_SLICES), B::G, smem, s>>>(P);
  }
}
// Fock-type build of the same (class, role) (NEXT-1; tdg_fock.cuh / MODE 1 of tdg_gradb.cuh)
static void launch_fock(const KParams& P, int nblocks, cudaStream_t s) {
  typedef QC<TDG_LA, TDG_LB, TDG_LC, TDG_LD> C;
  if constexpr (C::SMALL) {
    constexpr int nr = (TDG_LA + TDG_LB + TDG_LC + TDG_LD) / 2 + 1;
    constexpr int smem = nr <= 4 ? rys_sh_doubles(nr) * (int)sizeof(double) : 0;
    cudaFuncSetAttribute(tdg_fock_kernel<TDG_LA, TDG_LB, TDG_LC, TDG_LD, TDG_ROLE>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    tdg_fock_kernel<TDG_LA, TDG_LB, TDG_LC, TDG_LD, TDG_ROLE><<<nblocks, TDG_WARPS * TDG_WARP, smem, s>>>(P);
  } else {
    typedef QB<TDG_LA, TDG_LB, TDG_LC, TDG_LD> B;
    constexpr int smem = B::SMEM_DOUBLES * (int)sizeof(double);
    cudaFuncSetAttribute(tdg_gradb_kernel<TDG_LA, TDG_LB, TDG_LC, TDG_LD, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    tdg_gradb_kernel<TDG_LA, TDG_LB, TDG_LC, TDG_LD, 1><<<dim3(nblocks, TDG_GRADB_SLICES), B::G, smem, s>>>(P);
  }
}
namespace {
struct Registrar {
  Registrar() {
    tdg_register_launcher(TDG_LA, TDG_LB, TDG_LC, TDG_LD, TDG_ROLE, &launch);
    tdg_register_launcher(TDG_LA, TDG_LB, TDG_LC, TDG_LD, TDG_ROLE + TDG_FOCK_ROLE_BASE, &launch_fock);
  }
};
Registrar registrar;
}
