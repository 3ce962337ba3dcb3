// tdg_grad.cuh — per-class ERI-derivative + density-contraction kernel (steps a4-a8; Fig. 1).
//
// Work mapping (differs from Fig. 1's "1 thread = 1 batch"): a block work item is one bra tile of
// 32 consecutive sorted shell pairs (one per lane) times a chunk of TDG_KB sorted ket pairs (TDG_KW per warp).
// Every lane of a warp works on the SAME ket pair, so ket pair data are warp-uniform loads, the ket-centre
// gradient is reduced with warp shuffles (1 atomic per 32 quartets), and the bra-centre gradient stays in
// registers over the ket loop.  The fourth centre follows from translational invariance (eq 41).
//
// Integrals: Rys quadrature: n_r = floor((L+1)/2)+1 roots (reading S6) for the full operator and
// again for erf(omega r)/r (roots at s^2 T, x <- s^2 x, w <- s w; reading S8); 2-D recurrences of DESIGN.md
// "Rys 2-D recurrences"; centre derivative of eq 39/42 applied to the 2-D integral of
// one direction.  The derivative batch is never stored: each (component, root) term is multiplied by the
// symmetrised density product Gt (eqs 13-14) and accumulated into 9 scalars.
#pragma once
#include "tdg_common.cuh"

template <int LA, int LB, int LC, int LD>
struct QC {
  static constexpr int NA = ncart(LA), NB = ncart(LB), NC = ncart(LC), ND = ncart(LD);
  static constexpr int NCOMP = NA * NB * NC * ND;
  static constexpr int L = LA + LB + LC + LD;
  static constexpr int NR = (L + 1) / 2 + 1;
  static constexpr int DA = LA + 2, DB = LB + 2, DC = LC + 2, DD = LD + 1;
  static constexpr int NMX = LA + LB + 1, MMX = LC + LD + 1;
  static constexpr bool SMALL = NCOMP <= 27;
  static constexpr int UNR = SMALL ? 64 : 1;
};

// 2-D integrals of one direction for one root: I[i][j][k][l], i<=LA+1, j<=LB+1 (i+j<=LA+LB+1), k<=LC+1, l<=LD.
template <int LA, int LB, int LC, int LD>
__device__ __forceinline__ void build2d(double c00, double c00p, double b00, double b10, double b01, double ab,
                                        double cd, double v00,
                                        double (&I)[QC<LA, LB, LC, LD>::DA][QC<LA, LB, LC, LD>::DB][QC<LA, LB, LC, LD>::DC][QC<LA, LB, LC, LD>::DD]) {
  typedef QC<LA, LB, LC, LD> C;
  constexpr int NMX = C::NMX, MMX = C::MMX, U = C::UNR;
  double V[NMX + 1][MMX + 1];
  V[0][0] = v00;
#pragma unroll(U)
  for (int n = 0; n < NMX; ++n) V[n + 1][0] = c00 * V[n][0] + (n > 0 ? n * b10 * V[n - 1][0] : 0.0);
#pragma unroll(U)
  for (int m = 0; m < MMX; ++m) {
#pragma unroll(U)
    for (int n = 0; n <= NMX; ++n) {
      double v = c00p * V[n][m];
      if (m > 0) v += m * b01 * V[n][m - 1];
      if (n > 0) v += n * b00 * V[n - 1][m];
      V[n][m + 1] = v;
    }
  }
  // bra transfer i -> j, then ket transfer k -> l
  double W[C::DA][C::DB][MMX + 1];
#pragma unroll(U)
  for (int m = 0; m <= MMX; ++m) {
    double h[NMX + 1];
#pragma unroll(U)
    for (int i = 0; i <= NMX; ++i) h[i] = V[i][m];
#pragma unroll(U)
    for (int j = 0; j <= LB + 1; ++j) {
#pragma unroll(U)
      for (int i = 0; i <= LA + 1; ++i)
        if (i + j <= NMX) W[i][j][m] = h[i];
#pragma unroll(U)
      for (int i = 0; i + j < NMX; ++i) h[i] = h[i + 1] + ab * h[i];
    }
  }
#pragma unroll(U)
  for (int i = 0; i <= LA + 1; ++i) {
#pragma unroll(U)
    for (int j = 0; j <= LB + 1; ++j) {
      if (i + j > NMX) continue;
      double g[MMX + 1];
#pragma unroll(U)
      for (int k = 0; k <= MMX; ++k) g[k] = W[i][j][k];
#pragma unroll(U)
      for (int l = 0; l <= LD; ++l) {
#pragma unroll(U)
        for (int k = 0; k <= LC + 1; ++k)
          if (k + l <= MMX) I[i][j][k][l] = g[k];
#pragma unroll(U)
        for (int k = 0; k + l < MMX; ++k) g[k] = g[k + 1] + cd * g[k];
      }
    }
  }
}

template <int L, bool SMALL>
__device__ __forceinline__ void comp_exps(int idx, int& x, int& y, int& z) {
  if (SMALL) { x = cart_exp(L, idx, 0); y = cart_exp(L, idx, 1); z = cart_exp(L, idx, 2); }
  else { unsigned v = c_cart[L][idx]; x = v & 15; y = (v >> 4) & 15; z = (v >> 8) & 15; }
}

// Gradient contribution of one shell quartet: g[0..2] = d/dA, g[3..5] = d/dB, g[6..8] = d/dC (sum over all
// functions, primitives, roots and both operators, already multiplied by deg and the density products).
template <int LA, int LB, int LC, int LD>
__device__ __forceinline__ void quartet_grad(const KParams& P, const PairHdr& bh, const double* __restrict__ bprim,
                                             const PairHdr& kh, const double* __restrict__ kprim, double deg,
                                             double (&g)[9]) {
  typedef QC<LA, LB, LC, LD> C;
  constexpr int NA = C::NA, NB = C::NB, NC = C::NC, ND = C::ND, NR = C::NR, U = C::UNR;
  constexpr bool SM = C::SMALL;
  double GF[C::NCOMP], GL[C::NCOMP];
  {  // step a7, part 1: symmetrised density products for every function quartet
    const size_t n = (size_t)P.nbf;
#pragma unroll(U)
    for (int a = 0; a < NA; ++a)
#pragma unroll(U)
      for (int b = 0; b < NB; ++b)
#pragma unroll(U)
        for (int c = 0; c < NC; ++c)
#pragma unroll(U)
          for (int d = 0; d < ND; ++d) {
            const size_t mu = bh.offA + a, nu = bh.offB + b, la = kh.offA + c, si = kh.offB + d;
            double gj = 0.0, gk = 0.0;
            for (int q = 0; q < P.nJ; ++q) {
              const double* X = P.jp[q].X; const double* Y = P.jp[q].Y;
              gj += P.jp[q].w * (__ldg(X + mu * n + nu) * __ldg(Y + la * n + si) + __ldg(X + la * n + si) * __ldg(Y + mu * n + nu));
            }
            for (int q = 0; q < P.nK; ++q) {
              const double* X = P.kp[q].X; const double* Y = P.kp[q].Y;
              gk += P.kp[q].w * (__ldg(X + mu * n + la) * __ldg(Y + nu * n + si) + __ldg(X + nu * n + la) * __ldg(Y + mu * n + si) +
                                 __ldg(X + mu * n + si) * __ldg(Y + nu * n + la) + __ldg(X + nu * n + si) * __ldg(Y + mu * n + la));
            }
            const double cn = deg * c_cnorm[LA][a] * c_cnorm[LB][b] * c_cnorm[LC][c] * c_cnorm[LD][d];
            const int idx = ((a * NB + b) * NC + c) * ND + d;
            GF[idx] = cn * (gj + P.cK * gk);
            GL[idx] = cn * P.cLR * gk;
          }
  }
#pragma unroll
  for (int t = 0; t < 9; ++t) g[t] = 0.0;
  const double ABx = bh.AB[0], ABy = bh.AB[1], ABz = bh.AB[2];
  const double CDx = kh.AB[0], CDy = kh.AB[1], CDz = kh.AB[2];
  for (int ib = 0; ib < P.nppb; ++ib) {
    const double* bp = bprim + ib * TDG_PRIM_STRIDE;
    const double p = bp[0], Px = bp[1], Py = bp[2], Pz = bp[3], Kab = bp[4], a2 = 2.0 * bp[5], b2 = 2.0 * bp[6];
    const double PAx = Px - bh.A[0], PAy = Py - bh.A[1], PAz = Pz - bh.A[2];
    for (int ik = 0; ik < P.nppk; ++ik) {
      const double* kp = kprim + ik * TDG_PRIM_STRIDE;
      const double q = __ldg(kp + 0), Qx = __ldg(kp + 1), Qy = __ldg(kp + 2), Qz = __ldg(kp + 3), Kcd = __ldg(kp + 4), c2 = 2.0 * __ldg(kp + 5);
      const double QCx = Qx - kh.A[0], QCy = Qy - kh.A[1], QCz = Qz - kh.A[2];
      const double PQx = Px - Qx, PQy = Py - Qy, PQz = Pz - Qz;
      const double rpq = 1.0 / (p + q), rho = p * q * rpq;
      const double T = rho * (PQx * PQx + PQy * PQy + PQz * PQz);
      const double pref = 34.986836655249725693 /* 2 pi^(5/2) */ * Kab * Kcd * rpq * sqrt(rpq) / rho;
      const double rp = 1.0 / p, rq = 1.0 / q;
      for (int op = 0; op <= P.use_lr; ++op) {
        double s2 = 1.0, ss = 1.0;
        if (op == 1) { s2 = P.omega2 / (P.omega2 + rho); ss = sqrt(s2); }
        double xr[NR], wr[NR];
        rys_roots<NR>(P.rys_tab, s2 * T, xr, wr);
        const double* __restrict__ G = op == 0 ? GF : GL;
#pragma unroll(U)
        for (int r = 0; r < NR; ++r) {
          const double x = xr[r] * s2, w = wr[r] * ss * pref;
          const double b00 = 0.5 * x * rpq, b10 = (0.5 - q * b00) * rp, b01 = (0.5 - p * b00) * rq;
          const double fq = q * rpq * x, fp = p * rpq * x;
          double Ix[C::DA][C::DB][C::DC][C::DD], Iy[C::DA][C::DB][C::DC][C::DD], Iz[C::DA][C::DB][C::DC][C::DD];
          build2d<LA, LB, LC, LD>(PAx - fq * PQx, QCx + fp * PQx, b00, b10, b01, ABx, CDx, 1.0, Ix);
          build2d<LA, LB, LC, LD>(PAy - fq * PQy, QCy + fp * PQy, b00, b10, b01, ABy, CDy, 1.0, Iy);
          build2d<LA, LB, LC, LD>(PAz - fq * PQz, QCz + fp * PQz, b00, b10, b01, ABz, CDz, w, Iz);
          // step a7, part 2: contract the derivative integrals of this root with Gt
#pragma unroll(U)
          for (int a = 0; a < NA; ++a) {
            int ax, ay, az; comp_exps<LA, SM>(a, ax, ay, az);
#pragma unroll(U)
            for (int b = 0; b < NB; ++b) {
              int bx, by, bz; comp_exps<LB, SM>(b, bx, by, bz);
#pragma unroll(U)
              for (int c = 0; c < NC; ++c) {
                int cx, cy, cz; comp_exps<LC, SM>(c, cx, cy, cz);
#pragma unroll(U)
                for (int d = 0; d < ND; ++d) {
                  int dx, dy, dz; comp_exps<LD, SM>(d, dx, dy, dz);
                  const double Gv = G[((a * NB + b) * NC + c) * ND + d];
                  const double X0 = Ix[ax][bx][cx][dx], Y0 = Iy[ay][by][cy][dy], Z0 = Iz[az][bz][cz][dz];
                  const double tx = Gv * Y0 * Z0, ty = Gv * X0 * Z0, tz = Gv * X0 * Y0;
                  double dAx = a2 * Ix[ax + 1][bx][cx][dx], dAy = a2 * Iy[ay + 1][by][cy][dy], dAz = a2 * Iz[az + 1][bz][cz][dz];
                  if (ax > 0) dAx -= ax * Ix[ax - 1][bx][cx][dx];
                  if (ay > 0) dAy -= ay * Iy[ay - 1][by][cy][dy];
                  if (az > 0) dAz -= az * Iz[az - 1][bz][cz][dz];
                  double dBx = b2 * Ix[ax][bx + 1][cx][dx], dBy = b2 * Iy[ay][by + 1][cy][dy], dBz = b2 * Iz[az][bz + 1][cz][dz];
                  if (bx > 0) dBx -= bx * Ix[ax][bx - 1][cx][dx];
                  if (by > 0) dBy -= by * Iy[ay][by - 1][cy][dy];
                  if (bz > 0) dBz -= bz * Iz[az][bz - 1][cz][dz];
                  double dCx = c2 * Ix[ax][bx][cx + 1][dx], dCy = c2 * Iy[ay][by][cy + 1][dy], dCz = c2 * Iz[az][bz][cz + 1][dz];
                  if (cx > 0) dCx -= cx * Ix[ax][bx][cx - 1][dx];
                  if (cy > 0) dCy -= cy * Iy[ay][by][cy - 1][dy];
                  if (cz > 0) dCz -= cz * Iz[az][bz][cz - 1][dz];
                  g[0] += tx * dAx; g[1] += ty * dAy; g[2] += tz * dAz;
                  g[3] += tx * dBx; g[4] += ty * dBy; g[5] += tz * dBz;
                  g[6] += tx * dCx; g[7] += ty * dCy; g[8] += tz * dCz;
                }
              }
            }
          }
        }
      }
    }
  }
}

__device__ __forceinline__ void red_add(double* addr, double v) { atomicAdd(addr, v); }

template <int LA, int LB, int LC, int LD>
__global__ void __launch_bounds__(TDG_WARPS * TDG_WARP) tdg_grad_kernel(const __grid_constant__ KParams P) {
  // block work item -> (bra tile, ket chunk): largest t with cum[t] <= item
  const int item = blockIdx.x;
  int lo = 0, hi = P.ntiles;
  while (hi - lo > 1) { int mid = (lo + hi) >> 1; if (__ldg(P.cum + mid) <= item) lo = mid; else hi = mid; }
  const int tile = lo, chunk = item - __ldg(P.cum + tile);
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int bra = tile * TDG_WARP + lane;
  const bool bra_ok = bra < P.nbra;
  PairHdr bh = P.bra_hdr[bra_ok ? bra : P.nbra - 1];
  const double* bprim = P.bra_prim + (size_t)(bra_ok ? bra : P.nbra - 1) * P.nppb * TDG_PRIM_STRIDE;
  const int k0 = chunk * TDG_KB + warp * TDG_KW;
  int k1 = k0 + TDG_KW; if (k1 > P.nket) k1 = P.nket;
  double gA[3] = {0, 0, 0}, gB[3] = {0, 0, 0};
  unsigned long long n_vis = 0, n_cmp = 0, n_prim = 0;
  const int ns = P.nshell;
  for (int k = k0; k < k1; ++k) {
    const PairHdr kh = P.ket_hdr[k];
    bool act = bra_ok && (!P.same_bucket || k <= bra);
    if (act && P.tau > 0.0) {   // step a4 (reading S9)
      const double qq = bh.Q * kh.Q;
      act = qq >= P.tau;
      if (act) {
        ++n_vis;
        if (P.density_weighted) {
          const double dij = __ldg(P.dmax + (size_t)bh.ish * ns + bh.jsh), dkl = __ldg(P.dmax + (size_t)kh.ish * ns + kh.jsh);
          const double dik = __ldg(P.dmax + (size_t)bh.ish * ns + kh.ish), djl = __ldg(P.dmax + (size_t)bh.jsh * ns + kh.jsh);
          const double dil = __ldg(P.dmax + (size_t)bh.ish * ns + kh.jsh), djk = __ldg(P.dmax + (size_t)bh.jsh * ns + kh.ish);
          const double x1 = dik * djl, x2 = dil * djk;
          double W = P.CJ * dij * dkl; const double WK = P.CK * (x1 > x2 ? x1 : x2);
          if (WK > W) W = WK;
          if (qq * W < P.tau) act = false;
        }
      }
    } else if (act) ++n_vis;
    if (act && !tdg_sample_keep(bh.ish, bh.jsh, kh.ish, kh.jsh, P.sample_mod, P.sample_seed)) act = false;
    if (act) {
      ++n_cmp; n_prim += (unsigned long long)P.nppb * P.nppk;
      // all four shells on one atom: the four centre derivatives sum to zero on that atom (reading S11)
      if (bh.atomA == bh.atomB && kh.atomA == kh.atomB && bh.atomA == kh.atomA) act = false;
    }
    if (!__any_sync(0xffffffffu, act)) continue;
    double g[9];
    if (act) {
      double deg = 1.0;
      if (bh.ish == bh.jsh) deg *= 0.5;
      if (kh.ish == kh.jsh) deg *= 0.5;
      if (P.same_bucket && k == bra) deg *= 0.5;
      quartet_grad<LA, LB, LC, LD>(P, bh, bprim, kh, P.ket_prim + (size_t)k * P.nppk * TDG_PRIM_STRIDE, deg, g);
    } else {
#pragma unroll
      for (int t = 0; t < 9; ++t) g[t] = 0.0;
    }
    // step a8: bra centres stay in registers; ket centres are reduced over the warp (all lanes share this ket)
    double gC[3], gD[3];
#pragma unroll
    for (int x = 0; x < 3; ++x) {
      gA[x] += g[x]; gB[x] += g[3 + x];
      gC[x] = warp_sum(g[6 + x]);
      gD[x] = -warp_sum(g[x] + g[3 + x] + g[6 + x]);
    }
    if (lane == 0) {
#pragma unroll
      for (int x = 0; x < 3; ++x) { red_add(P.grad + 3 * kh.atomA + x, gC[x]); red_add(P.grad + 3 * kh.atomB + x, gD[x]); }
    }
  }
  if (bra_ok) {
#pragma unroll
    for (int x = 0; x < 3; ++x) {
      if (gA[x] != 0.0) red_add(P.grad + 3 * bh.atomA + x, gA[x]);
      if (gB[x] != 0.0) red_add(P.grad + 3 * bh.atomB + x, gB[x]);
    }
  }
  // stats
  for (int o = 16; o > 0; o >>= 1) {
    n_vis += __shfl_xor_sync(0xffffffffu, n_vis, o);
    n_cmp += __shfl_xor_sync(0xffffffffu, n_cmp, o);
    n_prim += __shfl_xor_sync(0xffffffffu, n_prim, o);
  }
  if (lane == 0 && n_vis) {
    atomicAdd(P.counters + 0, n_vis); atomicAdd(P.counters + 1, n_cmp); atomicAdd(P.counters + 2, n_prim);
  }
}

// Host-callable launcher of one class, defined in tdg_class_*.cu; c1 = pair class la(la+1)/2+lb of the bra.
typedef void (*tdg_launch_fn)(const KParams& P, int nblocks, cudaStream_t s);
tdg_launch_fn tdg_get_launcher(int la, int lb, int lc, int ld);
