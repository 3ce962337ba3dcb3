// tdg_internal.h — host-side declarations shared by the translation units of libtdgrad (not part of the ABI).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

struct DevShell { int32_t atom, l, nprim, prim_off, bf_off, pad; };

// tdg_aux.cu
cudaError_t tdg_upload_rys_table(double** d_tab);
// Q[ns*ns] (device) = sqrt(max_{m in i, n in j} (mn|mn)), full operator (reading S9)
cudaError_t tdg_launch_schwarz(const DevShell* sh, int ns, const double* xyz, const double* exps, const double* cn,
                               const double* rys_tab, double* Q, cudaStream_t s);
// out = max |M - M^T|  (device scalar, must be zeroed)
cudaError_t tdg_launch_asym(const double* M, int n, double* out, cudaStream_t s);
// m[i*ns+j] = max over the nmat matrices and the block (i,j) of max(|M_mn|, |M_nm|)   (reading S9: d_ij)
struct MatList { const double* m[16]; int n; };   // passed to the kernel by value: no upload, no host synchronisation
cudaError_t tdg_launch_dmax(const MatList& mats, int n, const DevShell* sh, int ns, double* m, cudaStream_t s);
cudaError_t tdg_launch_rys(int n, int count, const double* T, const double* rho, double omega, const double* tab, double* out, cudaStream_t s);
cudaError_t tdg_run_fp64_peak(double ms, double* tflops);

// Packed density array (a3): shell-blocked, 4 canonical matrices interleaved.  For shells I (rows) and K (columns),
// element (a, c) of canonical matrix m sits at pk[4*(off_I*nbf + n_I*off_K) + (a*n_K + c)*4 + m].  src[m] is an input
// matrix (row-major, device) or nullptr (slot = 0); kind[m] = 0: symmetric part (M+M^T)/2, 1: antisymmetric part (M-M^T)/2.
struct PackSrc { const double* src[4]; int kind[4]; };
cudaError_t tdg_launch_pack(const PackSrc& ps, int n, const int* bf2sh, const DevShell* sh, double* pk, cudaStream_t s);

// Spherical shells (NEXT-2): dir 0: out (Cartesian, nout x nout) = C^T in C with `in` in the input basis (nin_dim x nin_dim);
// dir 1: out (input basis, nout x nout) = C in C^T with `in` Cartesian (nin_dim x nin_dim).  out2sh: shell of each function of
// the OUTPUT basis; inoff: first input-basis function of each shell; sphflag: 1 = shell is spherical (acts for l >= 2).
cudaError_t tdg_launch_sph_transform(const double* in, double* out, int nout, int nin_dim, int dir, const int* out2sh, const DevShell* sh,
                                     const int* inoff, const int* sphflag, cudaStream_t s);
// F += G + sign G^T  (n x n row-major, device)
cudaError_t tdg_launch_fock_finalize(const double* G, int n, double sign, double* F, cudaStream_t s);

// Contracted energy (tdg_energy): runtime-l, untuned; one launch per bucket pair, same work lists and screening as the
// gradient kernels; *E (device) is accumulated with FP64 atomics.
struct KParams;
cudaError_t tdg_launch_energy(const KParams& P, int la, int lb, int lc, int ld, int nblocks, double* E, cudaStream_t s);

// One-electron gradient terms (tdg_onee.cu; NEXT-4): one launch per pair bucket; grad is accumulated with FP64 atomics.
struct PairHdr;
cudaError_t tdg_launch_onee(const PairHdr* hdr, const double* prim, int npair, int npp, int la, int lb, const double* xyz, const double* Z,
                            int natom, const double* Pm, const double* Wm, int nbf, double* grad, const double* rys_tab, cudaStream_t s);
cudaError_t tdg_launch_vnuc_grad(const double* xyz, const double* Z, int natom, double* grad, cudaStream_t s);

// Allocation-free Rys evaluation (tdg_noalloc.cu): all device workspace in a file-scope __device__ array; count <= TDG_RYS_STATIC_MAX.
#define TDG_RYS_STATIC_MAX 16384
int tdg_rys_static_max(void);
cudaError_t tdg_run_rys_static(int device, int n, int count, const double* T, const double* rho, double omega, const double* tab, double* out,
                               unsigned long long* nbad, cudaStream_t s);
