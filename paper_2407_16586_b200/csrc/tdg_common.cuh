// tdg_common.cuh — device data layout and small device helpers shared by the CUDA kernels of libtdgrad.
// (Product code: shares nothing with oracle/.)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#define TDG_WARP 32
#define TDG_KW 32                 // kets per warp per work item
#define TDG_WARPS 4               // warps per block
#define TDG_KB (TDG_KW * TDG_WARPS)  // kets per block work item
#define TDG_MAXP 8                // max canonical density pairs (J or K) per call

// Shell-pair header (80 B).  The pair is oriented so that l(first) >= l(second) ("highest l first").
struct __align__(16) PairHdr {
  double A[3];    // centre of the first shell
  double AB[3];   // A - B
  double Q;       // Schwarz bound sqrt(max (mn|mn))
  int32_t ish, jsh;      // INPUT shell indices of first/second shell
  int32_t atomA, atomB;
  int32_t offA, offB;    // first basis function of each shell
};
// Primitive-pair record: 8 doubles: p, Px, Py, Pz, K_ab/p, a, b, 1/p   (K_ab = c_a c_b exp(-ab/p |AB|^2), coefficients of step a0)
#define TDG_PRIM_STRIDE 8


struct KParams {
  const PairHdr* bra_hdr; const double* bra_prim; int nbra; int nppb;
  const PairHdr* ket_hdr; const double* ket_prim; int nket; int nppk;
  const int* cum;        // [ntiles+1] cumulative number of block work items per bra tile
  int ntiles; int same_bucket;
  double tau; int density_weighted; int wmode; const double* dmax; int nshell;   // wmode 0: gradient weight (S9), 1: Fock-build weight
  double CJ, CK;         // S9 weights of the density-weighted bound
  uint32_t sample_mod, sample_seed;
  // Packed densities (tdg_internal.h): 4 canonical matrices interleaved, shell-blocked.  With u = pk(ik)[a,c][.],
  // v = pk(jl)[b,d][.], s = pk(jk)[b,c][.], t = pk(il)[a,d][.]:  Gt_K = u.MK.v + s.MK.t ;  Gt_J = pk(ij)[a,b].MJ.pk(kl)[c,d]
  // (MJ, MK symmetric 4x4: sum over density pairs of w (e_x e_y^T + e_y e_x^T)).
  const double* pk; double MJ[16], MK[16];
  int nbf;
  double cK, cLR, omega, omega2; int use_lr;
  double* grad;                    // [natom][3]
  unsigned long long* counters;    // [3]: visited, computed, prim quartets
  const double* rys_tab;
};

__host__ __device__ constexpr int ncart(int l) { return (l + 1) * (l + 2) / 2; }

// Cartesian exponent d (0:x 1:y 2:z) of component idx of shell l; order lx desc, then ly desc (reading S7).
__host__ __device__ constexpr int cart_exp(int l, int idx, int d) {
  int c = 0;
  for (int lx = l; lx >= 0; --lx)
    for (int ly = l - lx; ly >= 0; --ly) {
      if (c == idx) return d == 0 ? lx : (d == 1 ? ly : l - lx - ly);
      ++c;
    }
  return 0;
}
// the same, forced to compile time: 4 bits per component packed into one constant (cheap to fold after unrolling)
__host__ __device__ constexpr unsigned long long cart_pack(int l, int d) {
  unsigned long long v = 0;
  for (int i = 0; i < ncart(l); ++i) v |= (unsigned long long)cart_exp(l, i, d) << (4 * i);
  return v;
}
template <int L, int D> struct CartPack { static constexpr unsigned long long v = cart_pack(L, D); };
// packed runtime table: [l][idx] -> lx | ly<<4 | lz<<8
__constant__ static uint16_t c_cart[4][10] = {
  {0x000},
  {0x001, 0x010, 0x100},
  {0x002, 0x011, 0x101, 0x020, 0x110, 0x200},
  {0x003, 0x012, 0x102, 0x021, 0x111, 0x201, 0x030, 0x120, 0x210, 0x300}};
// per-component normalisation 1/sqrt((2lx-1)!!(2ly-1)!!(2lz-1)!!) (eq 38 "N"; O1)
__host__ __device__ constexpr double dfact_odd(int n) { return n <= 0 ? 1.0 : (n == 1 ? 1.0 : (n == 2 ? 3.0 : 15.0)); }
__host__ __device__ constexpr double cnorm_c(int l, int idx) {   // compile-time form (folds to an immediate after unrolling)
  constexpr double r3 = 0.57735026918962576451, r15 = 0.25819888974716112568;
  constexpr double t[4][10] = {{1.0}, {1.0, 1.0, 1.0}, {r3, 1.0, 1.0, r3, 1.0, r3}, {r15, r3, r3, r3, 1.0, r3, r15, r3, r3, r15}};
  return t[l][idx];
}
__constant__ static double c_cnorm[4][10] = {
  {1.0},
  {1.0, 1.0, 1.0},
  {0.57735026918962576451, 1.0, 1.0, 0.57735026918962576451, 1.0, 0.57735026918962576451},
  {0.25819888974716112568, 0.57735026918962576451, 0.57735026918962576451, 0.57735026918962576451, 1.0,
   0.57735026918962576451, 0.25819888974716112568, 0.57735026918962576451, 0.57735026918962576451,
   0.25819888974716112568}};

// S12 subsample filter: fixed 64-bit finaliser on canonical INPUT shell-pair indices.
__host__ __device__ inline uint64_t tdg_mix64(uint64_t z) {
  z ^= z >> 30; z *= 0xbf58476d1ce4e5b9ULL;
  z ^= z >> 27; z *= 0x94d049bb133111ebULL;
  z ^= z >> 31;
  return z;
}
__host__ __device__ inline bool tdg_sample_keep(int i, int j, int k, int l, uint32_t mod, uint32_t seed) {
  if (mod == 0) return true;
  if (i < j) { int t = i; i = j; j = t; }
  if (k < l) { int t = k; k = l; l = t; }
  uint64_t ij = (uint64_t)i * (uint64_t)(i + 1) / 2 + (uint64_t)j;
  uint64_t kl = (uint64_t)k * (uint64_t)(k + 1) / 2 + (uint64_t)l;
  uint64_t hi = ij > kl ? ij : kl, lo = ij > kl ? kl : ij;
  uint64_t key = (hi << 32) ^ lo ^ ((uint64_t)seed * 0x9E3779B97F4A7C15ULL);
  return (tdg_mix64(key) % mod) == 0;
}

// ---- Rys roots and weights (step a5) ----
// Table layout (rys_tables.inc): for n: [interval][power, highest first][2n]; constants in __constant__.
#include "rys_meta.inc"

// `tabN` points at the table of this N (global: tab + rys_off(N); or a copy of it staged in shared memory, where the
// lanes' different intervals cost bank conflicts instead of one L1 wavefront per lane).
#define RYS_TABLE_DOUBLES(N) (rys_tmax(N) * (RYS_DEG + 1) * 2 * (N))
// Shared-memory layout of a staged table (SH = true; rys_sh_index maps the global layout to it).  Lanes evaluate different T, so
// they read different rows; in the global layout the rows of the lanes start at a few bank offsets only (Boys rows: 64 bytes, two
// offsets; polynomial intervals: 672 bytes for n = 3, four offsets; 896 bytes for n = 4, ONE offset) and a 128-bit load of a warp
// costs 8-32 wavefronts instead of 4.  Staged layout: n <= 2: the four 16-byte chunks of Boys row r are stored at chunk ^ ((r >> 1) & 3);
// n >= 3: every interval is padded by 16 bytes.  Either way consecutive rows cycle through all eight 16-byte bank groups.
#ifndef TDG_RYS_SH_LAYOUT
#define TDG_RYS_SH_LAYOUT 1
#endif
#define RYS_SH_PAD (TDG_RYS_SH_LAYOUT ? 2 : 0)   // doubles of padding per polynomial interval
template <int N, bool SH = false>
__device__ __forceinline__ void rys_roots_tab(const double* __restrict__ tabN, double T, double* __restrict__ x, double* __restrict__ w) {
  if (T >= (double)rys_tmax(N)) {
    double rT = 1.0 / T, rs = sqrt(rT);
#pragma unroll
    for (int r = 0; r < N; ++r) { x[r] = rys_inf(N, r) * rT; w[r] = rys_inf(N, N + r) * rs; }
    return;
  }
  int i = (int)T;                       // RYS_H == 1
  double u = (T - ((double)i + 0.5)) * 2.0;
  const double2* c = reinterpret_cast<const double2*>(tabN + i * ((RYS_DEG + 1) * 2 * N + (SH ? RYS_SH_PAD : 0)));   // rows of 2N doubles: 16-byte aligned
  double2 v[N];
#pragma unroll
  for (int f = 0; f < N; ++f) v[f] = c[f];
#pragma unroll
  for (int k = 1; k <= RYS_DEG; ++k) {
#pragma unroll
    for (int f = 0; f < N; ++f) { const double2 ck = c[k * N + f]; v[f].x = fma(v[f].x, u, ck.x); v[f].y = fma(v[f].y, u, ck.y); }
  }
  // row layout: x_0..x_{N-1}, w_0..w_{N-1}
#pragma unroll
  for (int r = 0; r < N; ++r) {
    x[r] = (r & 1) ? v[r >> 1].y : v[r >> 1].x;
    w[r] = ((N + r) & 1) ? v[(N + r) >> 1].y : v[(N + r) >> 1].x;
  }
}
// n <= 2: closed-form rule from the Boys moments F_0..F_{2n-1} (fewer table loads than the polynomial tables: one
// 64-byte Taylor row for F_{2n-1}, downward recursion F_{m-1} = (2T F_m + e^-T)/(2m-1), then x = F1/F0, w = F0 for n = 1
// and the roots of the monic orthogonal quadratic of the 2x2 Hankel system for n = 2).  boys_tables.inc layout.
#define BOYS_PER_UNIT 8
#define BOYS_K 8
template <int N, bool SH = false>
__device__ __forceinline__ void rys_roots_boys(const double* __restrict__ tabN, double T, double* __restrict__ x, double* __restrict__ w) {
  static_assert(N == 1 || N == 2, "closed form only for n <= 2");
  if (T >= (double)rys_tmax(N)) {
    double rT = 1.0 / T, rs = sqrt(rT);
#pragma unroll
    for (int r = 0; r < N; ++r) { x[r] = rys_inf(N, r) * rT; w[r] = rys_inf(N, N + r) * rs; }
    return;
  }
  const int i = (int)(T * BOYS_PER_UNIT);
  const double d = T - ((double)i + 0.5) * (1.0 / BOYS_PER_UNIT);
  const double2* c = reinterpret_cast<const double2*>(tabN + i * BOYS_K);
  const int sw = (SH && TDG_RYS_SH_LAYOUT) ? ((i >> 1) & 3) : 0;
  const double2 c01 = c[sw], c23 = c[1 ^ sw], c45 = c[2 ^ sw], c67 = c[3 ^ sw];
  double F = fma(c67.y, d, c67.x);
  F = fma(F, d, c45.y); F = fma(F, d, c45.x); F = fma(F, d, c23.y); F = fma(F, d, c23.x); F = fma(F, d, c01.y); F = fma(F, d, c01.x);
  const double e = exp(-T), T2 = 2.0 * T;
  if (N == 1) {
    const double F0 = fma(T2, F, e);
    x[0] = F / F0; w[0] = F0;
  } else {
    const double m3 = F, m2 = fma(T2, m3, e) * 0.2, m1 = fma(T2, m2, e) * (1.0 / 3.0), m0 = fma(T2, m1, e);
    // roots of x^2 + c1 x + c0 (the monic orthogonal quadratic): with D = c1^2 - 4 c0 and r = D^(-1/2): x2 - x1 = D r = 1/r, so
    // one division (the Hankel determinant) and one rsqrt replace three divisions and a square root; x1 = -(c1 + sqrt D)/2
    // loses at most one digit (x2/x1 <= ~10 for every T), well inside the 3e-13 moment tolerance of the tests
    const double rdet = 1.0 / (m0 * m2 - m1 * m1);
    const double c1 = (m1 * m2 - m0 * m3) * rdet, c0 = (m1 * m3 - m2 * m2) * rdet;
    const double disc = fma(c1, c1, -4.0 * c0), r = rsqrt(disc), sq = disc * r;
    const double x2 = 0.5 * (sq - c1), x1 = -0.5 * (sq + c1);
    const double w1 = fma(m0, x2, -m1) * r;
    x[0] = x1; x[N - 1] = x2; w[0] = w1; w[N - 1] = m0 - w1;
  }
}
// Device table = [Rys polynomial tables | Boys Taylor tables]; offset/size of the part a class with N roots uses.
__host__ __device__ constexpr int rys_part_off(int n) { return n <= 2 ? rys_off(RYS_NMAX + 1) + (n == 2 ? rys_tmax(1) * BOYS_PER_UNIT * BOYS_K : 0) : rys_off(n); }
__host__ __device__ constexpr int rys_part_doubles(int n) { return n <= 2 ? rys_tmax(n) * BOYS_PER_UNIT * BOYS_K : RYS_TABLE_DOUBLES(n); }
// `part` points at rys_part_off(N) of the device table (or at a shared-memory copy of that part)
template <int N, bool SH = false>
__device__ __forceinline__ void rys_eval(const double* __restrict__ part, double T, double* __restrict__ x, double* __restrict__ w) {
  if constexpr (N <= 2) rys_roots_boys<N, SH>(part, T, x, w);
  else rys_roots_tab<N, SH>(part, T, x, w);
}
// Staged (shared-memory) size of the part, and position of double2 element i of the global part in the staged layout.
__host__ __device__ constexpr int rys_sh_doubles(int n) { return n <= 2 ? rys_part_doubles(n) : rys_part_doubles(n) + rys_tmax(n) * RYS_SH_PAD; }
template <int N>
__device__ __forceinline__ int rys_sh_index(int i) {
  if (!TDG_RYS_SH_LAYOUT) return i;
  if (N <= 2) { const int row = i >> 2, chunk = i & 3; return (row << 2) | (chunk ^ ((row >> 1) & 3)); }
  constexpr int per = (RYS_DEG + 1) * N;     // double2 elements per interval
  const int iv = i / per;
  return i + iv * (RYS_SH_PAD / 2);
}
template <int N>
__device__ __forceinline__ void rys_roots(const double* __restrict__ tab, double T, double* __restrict__ x, double* __restrict__ w) {
  rys_eval<N>(tab + rys_part_off(N), T, x, w);
}

// 256-bit read-only global load (sm_100: LDG.E.256): 4 doubles from a 32-byte-aligned address in ONE load instruction;
// the density gathers and primitive-pair records are lane-divergent, so the L1 cost is per instruction, not per byte.
struct d4 { double x, y, z, w; };
__device__ __forceinline__ d4 ld256(const double* p) {
  d4 v;
  asm("ld.global.nc.v4.f64 {%0,%1,%2,%3}, [%4];" : "=d"(v.x), "=d"(v.y), "=d"(v.z), "=d"(v.w) : "l"(p));
  return v;
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}
