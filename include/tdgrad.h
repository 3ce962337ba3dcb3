/*
 * tdgrad.h — C ABI of libtdgrad.so: integral-direct ERI-derivative gradient on one B200 (sm_100a).
 *
 * What the library computes (PAPER.md = /root/reference/PAPER.md, arXiv 2407.16586):
 *
 *   E(R)    = sum_k [ wJ_k cJ J(A_k,B_k) - wK_k ( cK K(A_k,B_k) + cLR K_w(A_k,B_k) ) ]
 *   J(A,B)  = sum A_mn B_ls (mn|ls)      K(A,B) = sum A_ml B_ns (mn|ls)      K_w: (mn|ls)_lr
 *   grad[E][x] = dE/dR_{E,x}   with all matrices held fixed
 *
 * i.e. the 4th and 5th terms of eq 7 with the density products of eqs 13-14
 * (PAPER.md:110-114); (mn|ls) uses 1/r (eqs 3-4), (mn|ls)_lr uses erf(omega r)/r
 * (eq 5); basis functions are contracted Cartesian Gaussians (eqs 38, 43, PAPER.md:234-241,
 * 268-273); centre derivatives by eq 39/42; one centre by translational
 * invariance (eq 41); algorithm of Fig. 1; pair list sorted by
 * contraction degree and Schwarz bound, one kernel per angular class; Rys quadrature
 * (PAPER.md:311).  With the paper's P0 = 2 C_o C_o^T eqs 13-14 are pairs (P0,P0),(PD,P0),(R,R) with
 * wJ = (1/2,1,2), wK = (1/4,1/2,1), cJ = 1, cK = alpha, cLR = beta.
 *
 * Conventions: bohr / hartree; gradient in E_h/bohr.  Cartesian functions of a shell are ordered
 * lx descending then ly descending (x,y,z; xx,xy,xz,yy,yz,zz; xxx,xxy,...,zzz); every contracted
 * function is normalised to unit self-overlap (readings S7, O1).  Basis functions are
 * numbered in shell order.
 *
 * All functions return 0 on success and a negative TDG_E* code on error; they never throw, abort or
 * print.  Everything runs on the CUDA device given to tdg_create; there is NO CPU fallback
 * (no device => TDG_ECUDA).  The context owns all memory it allocates; the caller owns every buffer it
 * passes and may free it when the call returns.
 */
#ifndef TDGRAD_H
#define TDGRAD_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

#define TDG_OK 0
#define TDG_EINVAL (-1)        /* null pointer, non-positive count, bad shell/atom index, exponent <= 0, ... */
#define TDG_EUNSUPPORTED (-2)  /* shell angular momentum > 3 */
#define TDG_ENOTPLANNED (-3)   /* tdg_gradient before tdg_set_system + tdg_plan */
#define TDG_ENOMEM (-4)        /* host or device allocation failed */
#define TDG_ECUDA (-5)         /* CUDA runtime error; text kept in the context (tdg_last_error) */

#define TDG_MAX_L 3
#define TDG_NPAIRCLASS 10      /* (la>=lb) pair classes for l <= 3 */
#define TDG_NCLASS 55          /* quartet classes (pair class c1 >= c2), PAPER.md:309 has 21 for l <= 2 */

typedef struct tdg_ctx tdg_ctx; /* opaque */

/* One contracted shell (eq 43): nprim primitives exps/coefs[prim_off .. prim_off+nprim). */
typedef struct { int32_t atom, l, nprim, prim_off; } tdg_shell;

/* Screening options (reading S9, S12). */
typedef struct {
  double tau;               /* threshold; <= 0: no screening                                             */
  int32_t density_weighted; /* 0: keep quartet iff Q_ij Q_kl >= tau; 1: also Q_ij Q_kl W_ijkl >= tau      */
  uint32_t sample_mod;      /* 0: all quartets; else keep canonical shell quartet iff hash % mod == 0     */
  uint32_t sample_seed;
} tdg_options;

typedef struct {
  int64_t pairs_total, pairs_kept;     /* shell pairs i>=j; those with Q_ij Q_max >= tau                  */
  int64_t quartets_visited;            /* quartets passing the Schwarz product test                       */
  int64_t quartets_computed;           /* ... and the density-weighted test and the subsample filter      */
  int64_t prim_quartets;               /* primitive quartets of the computed ones                         */
  int64_t quartets_by_class[TDG_NCLASS];
  int64_t prim_quartets_by_class[TDG_NCLASS];
  float ms_by_class[TDG_NCLASS];       /* CUDA-event time of each class (only when stats != NULL)         */
  float ms_prepare;                    /* density preparation (a3)                                        */
  float ms_total;                      /* whole tdg_gradient device time                                  */
  int32_t launches;                    /* kernels launched by this call                                   */
  int32_t groups;                      /* passes over the class kernels (1 unless the pairs need > 4 canonical matrices) */
} tdg_stats;

/* Create a context on CUDA device `cuda_device`.  TDG_ECUDA if there is none. */
int tdg_create(tdg_ctx** out, int cuda_device);
int tdg_destroy(tdg_ctx* ctx);

/* Geometry and basis (HOST pointers, copied).  xyz_bohr[natom][3]; shells[nshell]; exps/coefs[nprim_total];
 * coefs multiply NORMALISED primitives; the library normalises each contracted function (step a0).
 * Invalidates any previous plan. */
int tdg_set_system(tdg_ctx* ctx, int natom, const double* xyz_bohr, int nshell, const tdg_shell* shells,
                   int nprim_total, const double* exps, const double* coefs);
/* Size of the square matrices the caller passes and receives: the number of Cartesian functions, or, after
 * tdg_set_spherical, the number of functions of the mixed Cartesian / spherical input basis. */
int tdg_nbf(const tdg_ctx* ctx, int* nbf);

/* Spherical-harmonic shells (PAPER.md:241 n_sph = 2l+1, "transform Cartesian ERI derivatives
 * into spherical basis", def2-SVP).  spherical[nshell] (HOST; NULL = all Cartesian): a nonzero flag on a d or f
 * shell means its 2l+1 functions are the real solid harmonics m = -l..l, each normalised to unit self-overlap:
 *   d: xy, yz, zz-(xx+yy)/2, xz, (sqrt3/2)(xx-yy);   f: y(3xx-yy), xyz, y(4zz-xx-yy), z(2zz-3xx-3yy), x(4zz-xx-yy), z(xx-yy), x(xx-3yy)
 * (s and p shells are unaffected: a p shell is x, y, z either way).  The input matrices of tdg_gradient / tdg_energy /
 * tdg_fock and the output of tdg_fock are then tdg_nbf x tdg_nbf in that basis.  Exact route, no kernel change: the transformation
 * coefficients do not depend on the geometry, so the library back-transforms every input, D_cart = C^T D C, runs the Cartesian
 * kernels, and forward-transforms Fock-type results, F = C F_cart C^T.  Schwarz bounds and the density-weighted test are those of
 * the Cartesian representation.  Call after tdg_set_system (which resets all shells to Cartesian); the plan stays valid. */
int tdg_set_spherical(tdg_ctx* ctx, const int32_t* spherical);

/* Steps a1-a2: shell pairs, Schwarz bounds Q_ij = sqrt(max (mn|mn)) (full operator) computed
 * ON THE DEVICE, pair screening, sort into (la,lb,contraction degree) buckets by Q descending, work lists.
 * Cached until tdg_set_system / tdg_plan is called again. */
int tdg_plan(tdg_ctx* ctx, const tdg_options* opt);

/* Multi-GPU sharding ("block-cyclic", 280-282, 304): this context computes only the
 * (launch, bra tile) work items whose running index is congruent to `rank` modulo `nranks`; tiles within a bucket
 * pair are ordered by Schwarz bound, so neighbouring items cost about the same and the deal balances.  The system,
 * the pair plan and the densities stay replicated.  tdg_gradient / tdg_energy then return this rank's PARTIAL
 * result and per-rank stats; the caller sums over ranks (one all-reduce of 3*natom doubles).  The union of the
 * nranks shards is exactly the unsharded work list, each quartet on exactly one rank.  Default (0, 1).
 * Invalidates the plan when the shard changes.  TDG_EINVAL unless 0 <= rank < nranks. */
int tdg_set_shard(tdg_ctx* ctx, int rank, int nranks);

/* The kernel launches of one quartet class (one per bucket pair and role) are independent of each other; they are dealt over the
 * caller's stream and nstreams-1 internal streams that fork from it before the class and join it after (events), so tails and
 * under-filled launches overlap while the call stays stream-ordered for the caller and tdg_stats.ms_by_class stays the wall time
 * of each class.  1 <= nstreams <= 8; default 6; 1 = strictly serial launches. */
int tdg_set_streams(tdg_ctx* ctx, int nstreams);

/* Schwarz bounds of the current system: Q[nshell][nshell] to a HOST buffer (for tests/diagnostics). */
int tdg_schwarz(tdg_ctx* ctx, double* Q_host);

/* Steps a3-a9.  A[k], B[k]: npair matrices nbf x nbf row-major FP64, ALL device pointers if
 * `matrices_on_device` != 0, else all host pointers (copied in inside the call); never modified.
 * wJ, wK: [npair] host.  cLR == 0 skips the long-range pass; omega > 0 required otherwise.
 * stream: cudaStream_t (as void*) or NULL for the default stream.
 * grad: [natom][3], device pointer if `grad_on_device` != 0 (completion is then stream-ordered) else host
 * (the call synchronises).  Overwritten, not accumulated.  stats may be NULL (non-NULL adds per-class
 * event timing and synchronises; the quartet counters are only read back then).
 * The call blocks the host ONCE mid-way when exchange is on (cK or cLR != 0 and some wK != 0): it reads back which
 * inputs are nonsymmetric, because that decides how many canonical matrices are packed (reading R1). */
int tdg_gradient(tdg_ctx* ctx, int npair, const double* const* A, const double* const* B, int matrices_on_device,
                 const double* wJ, const double* wK, double cJ, double cK, double cLR, double omega,
                 void* stream, double* grad, int grad_on_device, tdg_stats* stats);

/* Contracted energy E (same arguments, same screening and subsample rule; HOST result; synchronises) for
 * finite-difference checks of the gradient; runtime-l kernel, not tuned. */
int tdg_energy(tdg_ctx* ctx, int npair, const double* const* A, const double* const* B, int matrices_on_device,
               const double* wJ, const double* wK, double cJ, double cK, double cLR, double omega,
               void* stream, double* E_host);

/* One-electron terms of the gradient (terms 1-3 of eq 7; evaluated on the CPU in the paper,
 * PAPER.md:404):
 *
 *   grad[E][x] = sum_mn P_mn d(T + V)_mn/dR_{E,x} + sum_mn W_mn dS_mn/dR_{E,x} + dV_nuc/dR_{E,x}
 *
 * S overlap, T = <m|-1/2 Laplacian|n>, V_mn = -sum_C Z_C <m|1/|r - R_C||n>, V_nuc = sum_{C<D} Z_C Z_D / R_CD; P (the density of
 * eq 8) and W (the energy-weighted density of eq 7) are held fixed, general nbf x nbf row-major matrices in the input basis of
 * tdg_nbf (all device pointers if matrices_on_device != 0, else host; either may be NULL = zero).  Z[natom]: nuclear charges, HOST.
 * Runs over the shell pairs kept by tdg_plan (pairs with Q_ij Q_max < tau are dropped here too; tau = 0 keeps all).
 * grad: [natom][3], device pointer if grad_on_device != 0 else host; overwritten.  The call synchronises the stream (Z is a host
 * array).  ms (may be NULL): device time of the call.  Not concurrent with other calls on the same context. */
int tdg_onee_gradient(tdg_ctx* ctx, const double* Z, const double* P, const double* W, int matrices_on_device, void* stream,
                      double* grad, int grad_on_device, float* ms);

/* Fock-type (J/K) build, integral-direct with the same plan, screening and kernels' machinery as tdg_gradient (SURVEY.md 8(f)
 * NEXT-1).  For each of the nmat input matrices B_k (nbf x nbf row-major, general; all device or all host pointers):
 *
 *   F_k[mn] = sum_ls [ wJ_k B_k[sl] (mn|ls)  -  X_k[sl] ( cK (ml|sn) + cLR (ml|sn)_lr ) ],    X_k = wK_k B_k + wKT_k B_k^T
 *
 * PAPER.md:197-207 (eqs 33-34, the sigma vector of the Z-vector iterations): wJ = 4, wK = wKT = 1, cK = alpha, cLR = beta.
 * PAPER.md:138 (eq 19, F of a symmetric relaxed-difference density): wJ = 2, wK = 1, wKT = 0.  The XC-kernel term of both
 * equations is not part of this library.  Screening: quartet kept iff Q_ij Q_kl >= tau and (density_weighted) Q_ij Q_kl W >= tau,
 * W = max(max_k|wJ_k| max(d_ij,d_kl), (|cK|+|cLR|) max_k(|wK_k|+|wKT_k|) max(d_ik,d_il,d_jk,d_jl)), d = shell-block maxima of
 * |B_k| over all k and both orientations.  F[k]: nbf x nbf row-major, device pointers if F_on_device != 0
 * (completion stream-ordered) else host (the call synchronises); overwritten.  1 <= nmat <= 8.  stats may be NULL. */
int tdg_fock(tdg_ctx* ctx, int nmat, const double* const* B, int matrices_on_device, const double* wJ, const double* wK,
             const double* wKT, double cK, double cLR, double omega, void* stream, double* const* F, int F_on_device,
             tdg_stats* stats);

/* Rys roots/weights evaluator (step a5; reading S8), exposed for parity tests:
 * for each of `count` (T[i], rho[i]) HOST inputs writes n roots x_r and n weights w_r to out[i][2n] (host),
 * for the full operator (omega <= 0) or the attenuated one (x_r <- s^2 x_r(s^2 T), w_r <- s w_r(s^2 T),
 * s^2 = omega^2/(omega^2+rho)).  Runs on the device.  1 <= n <= 7. */
int tdg_rys(tdg_ctx* ctx, int n, int count, const double* T, const double* rho, double omega, double* out);

/* Allocation-free variant of tdg_rys for callers that may not call cudaMalloc (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid allocation).  Same arithmetic and the same arguments and result layout as tdg_rys (n = 1..7 roots;
 * T, rho, out are HOST arrays of count and count*2n doubles; per evaluation x_0..x_{n-1}, w_0..w_{n-1}), but every byte of device
 * workspace is a fixed file-scope device array of the library (csrc/tdg_noalloc.cu): 2 MiB + 256 B, held by every GPU that loads
 * the library until the process exits.  The call makes NO cudaMalloc / cudaFree / allocating library call (tdg_create, which
 * uploads the Rys tables, has to have happened before).  Limit: 1 <= count <= TDG_RYS_STATIC_MAX, larger counts are rejected with
 * TDG_EINVAL and a text in tdg_last_error (split the batch).  Arguments with T < 0, rho <= 0, NaN or infinite are rejected with
 * TDG_EINVAL as well (out is then unspecified).  stream: cudaStream_t as void* or NULL; the call synchronises it.
 * ALL calls on one GPU share the array, which keeps the last call's contents (each call overwrites what it reads and clears its
 * error counter): calls that overlap on the GPU - other streams, other host threads, other contexts on the same device - RACE;
 * serialise them. */
#define TDG_RYS_STATIC_MAX 16384
int tdg_rys_static(tdg_ctx* ctx, int n, int count, const double* T, const double* rho, double omega, void* stream, double* out);

/* FP64 FMA throughput microbenchmark on this device (the roofline denominator; step 8d): runs chains of
 * dependent DFMAs on all SMs for about `ms` milliseconds; writes achieved TFLOP/s (2 flop per FMA). */
int tdg_fp64_peak(tdg_ctx* ctx, double ms, double* tflops);

const char* tdg_strerror(int code);
const char* tdg_last_error(const tdg_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif
