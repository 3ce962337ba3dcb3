// tdg_onee.cu — one-electron terms of the gradient (terms 1-3 of eq 7):
//
//   g_E = sum_mn P_mn dH^core_mn/dR_E + sum_mn W_mn dS_mn/dR_E + dV_nuc/dR_E,   H^core = T + V,
//   T_mn = <m|-1/2 Laplacian|n>,  V_mn = -sum_C Z_C <m|1/|r-R_C||n>,  V_nuc = sum_{C<D} Z_C Z_D/R_CD,   P, W fixed.
//
// The paper evaluates these on the CPU; here they run on the device over the planner's sorted shell-pair
// buckets (steps a1-a2), so a full non-XC gradient needs no host integral code.
//
// One thread per shell pair, blockIdx.y over chunks of ONEE_ATOMS nuclei.  Overlap and kinetic parts: Obara-Saika
// 1-D overlap tables s(i,j), the kinetic 1-D factor k(i,j) = -1/2 [j(j-1) s(i,j-2) - 2b(2j+1) s(i,j) + 4b^2 s(i,j+2)],
// centre derivative 2a (i+1) - i (i-1) (eq 39); two-centre integrals depend on A - B only, so d/dB = -d/dA.  Nuclear
// attraction: Rys quadrature with n = floor((la+lb+1)/2)+1 roots at T = p |P-C|^2 (the q -> infinity limit of the 2-D
// recurrences of the ERI kernels: C00 = (P-A) - x (P-C), B10 = (1-x)/(2p)), derivatives on A and B, and the operator
// centre by translational invariance d/dC = -(d/dA + d/dB) (eq 41 applied to the three-centre integral).  The per-nucleus
// terms are summed over the pairs of a warp by shuffles and kept in per-warp shared slots; one FP64 RED per touched slot.
#include "tdg_common.cuh"
#include "tdg_internal.h"

#define ONEE_NT 128
#define ONEE_ATOMS 256

struct OneeParams {
  const PairHdr* hdr; const double* prim; int npair, npp;
  const double* xyz; const double* Z; int natom;
  const double* Pm; const double* Wm; int nbf;
  double* grad; const double* rys_tab;
};

template <int LA, int LB>
struct OC {
  static constexpr int NA = ncart(LA), NB = ncart(LB);
  static constexpr int NR = (LA + LB + 1) / 2 + 1;
  static constexpr int U = (NA * NB <= 18) ? 64 : 1;   // full unrolling (registers) for the low-l classes that carry the pairs
};

template <int L, int U>
__device__ __forceinline__ void onee_exps(int idx, int& x, int& y, int& z) {
  if (U > 1) {
    x = (int)((CartPack<L, 0>::v >> (4 * idx)) & 15); y = (int)((CartPack<L, 1>::v >> (4 * idx)) & 15); z = (int)((CartPack<L, 2>::v >> (4 * idx)) & 15);
  } else { const unsigned v = c_cart[L][idx]; x = v & 15; y = (v >> 4) & 15; z = (v >> 8) & 15; }
}

// Overlap and kinetic parts of one shell pair: adds sum_ab [W_ab dS_ab + P_ab dT_ab]/dA to gA and the negative to gB.
template <int LA, int LB>
__device__ __forceinline__ void onee_overlap_kinetic(const OneeParams& P, const PairHdr& h, const double* __restrict__ prim, double deg,
                                                     const double* wP, double (&gA)[3], double (&gB)[3]) {
  typedef OC<LA, LB> C;
  constexpr int NA = C::NA, NB = C::NB, U = C::U;
  for (int ip = 0; ip < P.npp; ++ip) {
    const d4 r0 = ld256(prim + ip * TDG_PRIM_STRIDE), r1 = ld256(prim + ip * TDG_PRIM_STRIDE + 4);
    const double p = r0.x, a2 = 2.0 * r1.y, eb = r1.z, rp2 = 0.5 * r1.w;
    const double Kab = r1.x * p * 5.5683279968317078453 /* pi^(3/2) */ * r1.w * sqrt(r1.w);   // K_ab (pi/p)^(3/2)
    const double PA[3] = {r0.y - h.A[0], r0.z - h.A[1], r0.w - h.A[2]};
    // s[d][i][j], i <= LA+1, j <= LB+3:  v(i+1) = PA v(i) + i/(2p) v(i-1) on centre A, then s(i,j+1) = s(i+1,j) + AB s(i,j)
    double s[3][LA + 2][LB + 4], k[3][LA + 2][LB + 2];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      double v[LA + LB + 5];
      v[0] = 1.0; v[1] = PA[d];
#pragma unroll(U)
      for (int i = 1; i < LA + LB + 4; ++i) v[i + 1] = PA[d] * v[i] + i * rp2 * v[i - 1];
#pragma unroll(U)
      for (int j = 0; j <= LB + 3; ++j) {
#pragma unroll(U)
        for (int i = 0; i <= LA + 1; ++i) s[d][i][j] = v[i];
#pragma unroll(U)
        for (int i = 0; i + j < LA + LB + 4; ++i) v[i] = v[i + 1] + h.AB[d] * v[i];
      }
#pragma unroll(U)
      for (int i = 0; i <= LA + 1; ++i)
#pragma unroll(U)
        for (int j = 0; j <= LB + 1; ++j) {
          double kv = 4.0 * eb * eb * s[d][i][j + 2] - 2.0 * eb * (2 * j + 1) * s[d][i][j];
          if (j > 1) kv += j * (j - 1) * s[d][i][j - 2];
          k[d][i][j] = -0.5 * kv;
        }
    }
    const size_t n2 = (size_t)P.nbf;
#pragma unroll(U)
    for (int a = 0; a < NA; ++a) {
      int ax[3]; onee_exps<LA, U>(a, ax[0], ax[1], ax[2]);
#pragma unroll(U)
      for (int b = 0; b < NB; ++b) {
        int bx[3]; onee_exps<LB, U>(b, bx[0], bx[1], bx[2]);
        const double ww = Kab * deg * (U > 1 ? cnorm_c(LA, a) * cnorm_c(LB, b) : c_cnorm[LA][a] * c_cnorm[LB][b]) *
                          (P.Wm ? __ldg(P.Wm + (size_t)(h.offA + a) * n2 + h.offB + b) + __ldg(P.Wm + (size_t)(h.offB + b) * n2 + h.offA + a) : 0.0);
        const double wp = Kab * wP[a * NB + b];
        double s0[3], k0[3], ds[3], dk[3];
#pragma unroll
        for (int d = 0; d < 3; ++d) {
          s0[d] = s[d][ax[d]][bx[d]]; k0[d] = k[d][ax[d]][bx[d]];
          ds[d] = a2 * s[d][ax[d] + 1][bx[d]]; dk[d] = a2 * k[d][ax[d] + 1][bx[d]];
          if (ax[d] > 0) { ds[d] -= ax[d] * s[d][ax[d] - 1][bx[d]]; dk[d] -= ax[d] * k[d][ax[d] - 1][bx[d]]; }
        }
        // d/dA_x of S = ds_x s_y s_z; of T = dk_x s_y s_z + ds_x (k_y s_z + s_y k_z)
        const double gx = ww * ds[0] * s0[1] * s0[2] + wp * (dk[0] * s0[1] * s0[2] + ds[0] * (k0[1] * s0[2] + s0[1] * k0[2]));
        const double gy = ww * ds[1] * s0[0] * s0[2] + wp * (dk[1] * s0[0] * s0[2] + ds[1] * (k0[0] * s0[2] + s0[0] * k0[2]));
        const double gz = ww * ds[2] * s0[0] * s0[1] + wp * (dk[2] * s0[0] * s0[1] + ds[2] * (k0[0] * s0[1] + s0[0] * k0[1]));
        gA[0] += gx; gA[1] += gy; gA[2] += gz;
        gB[0] -= gx; gB[1] -= gy; gB[2] -= gz;
      }
    }
  }
}

// Nuclear attraction of one shell pair with one nucleus (charge Zc at C): adds sum_ab P_ab dV_ab/dA, /dB to vA, vB.
template <int LA, int LB>
__device__ __forceinline__ void onee_attraction(const OneeParams& P, const PairHdr& h, const double* __restrict__ prim, const double* __restrict__ rys,
                                                double Cx, double Cy, double Cz, double Zc, const double* wP, double (&vA)[3], double (&vB)[3]) {
  typedef OC<LA, LB> C;
  constexpr int NA = C::NA, NB = C::NB, NR = C::NR, U = C::U;
  for (int ip = 0; ip < P.npp; ++ip) {
    const d4 r0 = ld256(prim + ip * TDG_PRIM_STRIDE), r1 = ld256(prim + ip * TDG_PRIM_STRIDE + 4);
    const double p = r0.x, a2 = 2.0 * r1.y, b2 = 2.0 * r1.z, rp2 = 0.5 * r1.w;
    const double PA[3] = {r0.y - h.A[0], r0.z - h.A[1], r0.w - h.A[2]};
    const double PC[3] = {r0.y - Cx, r0.z - Cy, r0.w - Cz};
    const double pref = -6.2831853071795864769 * Zc * r1.x;          // -Z 2 pi K_ab / p
    double xr[NR], wr[NR];
    rys_eval<NR>(rys, p * (PC[0] * PC[0] + PC[1] * PC[1] + PC[2] * PC[2]), xr, wr);
    for (int r = 0; r < NR; ++r) {
      const double x = xr[r], b10 = (1.0 - x) * rp2;
      double I[3][LA + 2][LB + 2];
#pragma unroll
      for (int d = 0; d < 3; ++d) {
        const double c00 = PA[d] - x * PC[d];
        double v[LA + LB + 2];
        v[0] = d == 2 ? wr[r] * pref : 1.0;
#pragma unroll(U)
        for (int i = 0; i < LA + LB + 1; ++i) v[i + 1] = c00 * v[i] + (i > 0 ? i * b10 * v[i - 1] : 0.0);
#pragma unroll(U)
        for (int j = 0; j <= LB + 1; ++j) {
#pragma unroll(U)
          for (int i = 0; i <= LA + 1; ++i)
            if (i + j <= LA + LB + 1) I[d][i][j] = v[i];
#pragma unroll(U)
          for (int i = 0; i + j < LA + LB + 1; ++i) v[i] = v[i + 1] + h.AB[d] * v[i];
        }
      }
#pragma unroll(U)
      for (int a = 0; a < NA; ++a) {
        int ax[3]; onee_exps<LA, U>(a, ax[0], ax[1], ax[2]);
#pragma unroll(U)
        for (int b = 0; b < NB; ++b) {
          int bx[3]; onee_exps<LB, U>(b, bx[0], bx[1], bx[2]);
          const double w = wP[a * NB + b];
          const double X0 = I[0][ax[0]][bx[0]], Y0 = I[1][ax[1]][bx[1]], Z0 = I[2][ax[2]][bx[2]];
          const double tx = w * Y0 * Z0, ty = w * X0 * Z0, tz = w * X0 * Y0;
          double dAx = a2 * I[0][ax[0] + 1][bx[0]], dAy = a2 * I[1][ax[1] + 1][bx[1]], dAz = a2 * I[2][ax[2] + 1][bx[2]];
          if (ax[0] > 0) dAx -= ax[0] * I[0][ax[0] - 1][bx[0]];
          if (ax[1] > 0) dAy -= ax[1] * I[1][ax[1] - 1][bx[1]];
          if (ax[2] > 0) dAz -= ax[2] * I[2][ax[2] - 1][bx[2]];
          double dBx = b2 * I[0][ax[0]][bx[0] + 1], dBy = b2 * I[1][ax[1]][bx[1] + 1], dBz = b2 * I[2][ax[2]][bx[2] + 1];
          if (bx[0] > 0) dBx -= bx[0] * I[0][ax[0]][bx[0] - 1];
          if (bx[1] > 0) dBy -= bx[1] * I[1][ax[1]][bx[1] - 1];
          if (bx[2] > 0) dBz -= bx[2] * I[2][ax[2]][bx[2] - 1];
          vA[0] += tx * dAx; vA[1] += ty * dAy; vA[2] += tz * dAz;
          vB[0] += tx * dBx; vB[1] += ty * dBy; vB[2] += tz * dBz;
        }
      }
    }
  }
}

template <int LA, int LB>
__global__ void __launch_bounds__(ONEE_NT) onee_kernel(const OneeParams P) {
  typedef OC<LA, LB> C;
  constexpr int NA = C::NA, NB = C::NB, NR = C::NR, U = C::U;
  __shared__ double s_xyz[ONEE_ATOMS][4];                       // x, y, z, Z of the chunk's nuclei
  __shared__ double s_gc[ONEE_NT / 32][ONEE_ATOMS][3];          // operator-centre terms, one slice per warp
  const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
  const int c0 = blockIdx.y * ONEE_ATOMS, nc = min(ONEE_ATOMS, P.natom - c0);
  for (int i = t; i < nc; i += ONEE_NT) {
    s_xyz[i][0] = P.xyz[3 * (c0 + i)]; s_xyz[i][1] = P.xyz[3 * (c0 + i) + 1]; s_xyz[i][2] = P.xyz[3 * (c0 + i) + 2]; s_xyz[i][3] = P.Z[c0 + i];
  }
  for (int i = t; i < (ONEE_NT / 32) * ONEE_ATOMS * 3; i += ONEE_NT) (&s_gc[0][0][0])[i] = 0.0;
  __syncthreads();
  const int pi = blockIdx.x * ONEE_NT + t;
  const bool act = pi < P.npair;
  PairHdr h;
  double wP[NA * NB], gA[3] = {0.0, 0.0, 0.0}, gB[3] = {0.0, 0.0, 0.0};
  const double* prim = nullptr;
  if (act) {
    h = P.hdr[pi];
    prim = P.prim + (size_t)pi * P.npp * TDG_PRIM_STRIDE;
    const double deg = h.ish == h.jsh ? 0.5 : 1.0;   // every unordered pair once; (m,n) and (n,m) elements are both read
    const size_t n = (size_t)P.nbf;
#pragma unroll(U)
    for (int a = 0; a < NA; ++a)
#pragma unroll(U)
      for (int b = 0; b < NB; ++b)
        wP[a * NB + b] = deg * (U > 1 ? cnorm_c(LA, a) * cnorm_c(LB, b) : c_cnorm[LA][a] * c_cnorm[LB][b]) *
                         (P.Pm ? __ldg(P.Pm + (size_t)(h.offA + a) * n + h.offB + b) + __ldg(P.Pm + (size_t)(h.offB + b) * n + h.offA + a) : 0.0);
    // overlap and kinetic parts: first nucleus chunk only; one-centre pairs do not move with anything else
    if (blockIdx.y == 0 && h.atomA != h.atomB) onee_overlap_kinetic<LA, LB>(P, h, prim, deg, wP, gA, gB);
  }
  const double* rys = P.rys_tab + rys_part_off(NR);
  for (int c = 0; c < nc; ++c) {
    const double Zc = s_xyz[c][3];
    double vA[3] = {0.0, 0.0, 0.0}, vB[3] = {0.0, 0.0, 0.0};
    if (act && Zc != 0.0 && P.Pm) {
      onee_attraction<LA, LB>(P, h, prim, rys, s_xyz[c][0], s_xyz[c][1], s_xyz[c][2], Zc, wP, vA, vB);
#pragma unroll
      for (int d = 0; d < 3; ++d) { gA[d] += vA[d]; gB[d] += vB[d]; }
    }
    // operator centre: -(dA + dB), summed over the warp's pairs
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      const double v = warp_sum(-(vA[d] + vB[d]));
      if (lane == 0 && v != 0.0) s_gc[warp][c][d] += v;
    }
  }
  if (act) {
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      if (gA[d] != 0.0) atomicAdd(P.grad + 3 * h.atomA + d, gA[d]);
      if (gB[d] != 0.0) atomicAdd(P.grad + 3 * h.atomB + d, gB[d]);
    }
  }
  __syncthreads();
  for (int i = t; i < nc * 3; i += ONEE_NT) {
    double v = 0.0;
#pragma unroll
    for (int w = 0; w < ONEE_NT / 32; ++w) v += (&s_gc[w][0][0])[i];
    if (v != 0.0) atomicAdd(P.grad + 3 * c0 + i, v);
  }
}

// dV_nuc/dR: one thread per nucleus.
__global__ void vnuc_grad_kernel(const double* __restrict__ xyz, const double* __restrict__ Z, int natom, double* __restrict__ grad) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= natom) return;
  const double x = xyz[3 * c], y = xyz[3 * c + 1], z = xyz[3 * c + 2], zc = Z[c];
  double g[3] = {0.0, 0.0, 0.0};
  for (int d = 0; d < natom; ++d) {
    if (d == c) continue;
    const double rx = x - xyz[3 * d], ry = y - xyz[3 * d + 1], rz = z - xyz[3 * d + 2];
    const double r2 = rx * rx + ry * ry + rz * rz, ri = rsqrt(r2), f = -zc * Z[d] * ri * ri * ri;
    g[0] += f * rx; g[1] += f * ry; g[2] += f * rz;
  }
  for (int k = 0; k < 3; ++k) atomicAdd(grad + 3 * c + k, g[k]);
}

template <int LA, int LB>
static cudaError_t launch_onee_class(const OneeParams& P, cudaStream_t s) {
  dim3 grid((P.npair + ONEE_NT - 1) / ONEE_NT, (P.natom + ONEE_ATOMS - 1) / ONEE_ATOMS);
  onee_kernel<LA, LB><<<grid, ONEE_NT, 0, s>>>(P);
  return cudaGetLastError();
}

cudaError_t tdg_launch_onee(const PairHdr* hdr, const double* prim, int npair, int npp, int la, int lb, const double* xyz, const double* Z,
                            int natom, const double* Pm, const double* Wm, int nbf, double* grad, const double* rys_tab, cudaStream_t s) {
  OneeParams P{hdr, prim, npair, npp, xyz, Z, natom, Pm, Wm, nbf, grad, rys_tab};
#define ONEE_CASE(a, b) if (la == a && lb == b) return launch_onee_class<a, b>(P, s);
  ONEE_CASE(0, 0) ONEE_CASE(1, 0) ONEE_CASE(1, 1) ONEE_CASE(2, 0) ONEE_CASE(2, 1) ONEE_CASE(2, 2)
  ONEE_CASE(3, 0) ONEE_CASE(3, 1) ONEE_CASE(3, 2) ONEE_CASE(3, 3)
#undef ONEE_CASE
  return cudaErrorInvalidValue;
}

cudaError_t tdg_launch_vnuc_grad(const double* xyz, const double* Z, int natom, double* grad, cudaStream_t s) {
  vnuc_grad_kernel<<<(natom + 127) / 128, 128, 0, s>>>(xyz, Z, natom, grad);
  return cudaGetLastError();
}
