// tdg_fock.cuh — integral-direct Fock-type (J/K) build, one thread per shell quartet (NEXT-1 of SURVEY.md 8(f)).
//
//   F_k[mn] = sum_ls [ wJ_k B_k[sl] (mn|ls) - X_k[sl] ( cK (ml|sn) + cLR (ml|sn)_lr ) ],   X_k = wK_k B_k + wKT_k B_k^T
//
// (eq 19: wJ = 2, wK = 1, wKT = 0; eqs 33-34: wJ = 4, wK = wKT = 1 -- the sigma-vector build
// of the Z-vector iterations, ~49 % of the paper's wall time.)  Same planner, work items, Schwarz-sorted
// prefix and survivor compaction as the gradient kernel (tdg_grad.cuh); undifferentiated integrals, n = floor(L/2)+1 roots.
//
// Canonical matrices (slots of the packed array, <= 4 per pass): S = (B+B^T)/2 and, where the exchange density is
// nonsymmetric, N = (B-B^T)/2.  The kernel accumulates, per slot, the "upper orientation" G of the 8 index permutations:
//   G[mn] += jw S[ls] I,  G[ls] += jw S[mn] I                       (Coulomb; jw = 2 wJ for S slots, 0 for N slots)
//   G[ms] -= kw X[ln] Ik, G[ns] -= kw X[lm] Ik, G[ml] -= kw X[sn] Ik, G[nl] -= kw X[sm] Ik     (exchange; Ik = cK I + cLR I_lr)
// with deg = (1/2)^{[i=j]+[k=l]+[ij=kl]} folded into the integrals; the other four permutations are the transposes, applied by
// fock_finalize: F = G + G^T (S slots), F = G - G^T (N slots).  G is updated with FP64 RED (no return value).
#pragma once
#include "tdg_grad.cuh"

// Plain 2-D integrals of one direction for one root: I[i][j][k][l], i<=LA, j<=LB, k<=LC, l<=LD.
template <int LA, int LB, int LC, int LD>
__device__ __forceinline__ void build2d_plain(double c00, double c00p, double b00, double b10, double b01, double ab, double cd, double v00,
                                              double (&I)[LA + 1][LB + 1][LC + 1][LD + 1]) {
  constexpr int NMX = LA + LB, MMX = LC + LD;
  double V[NMX + 1][MMX + 1];
  V[0][0] = v00;
#pragma unroll
  for (int n = 0; n < NMX; ++n) V[n + 1][0] = c00 * V[n][0] + (n > 0 ? n * b10 * V[n - 1][0] : 0.0);
#pragma unroll
  for (int m = 0; m < MMX; ++m) {
#pragma unroll
    for (int n = 0; n <= NMX; ++n) {
      double v = c00p * V[n][m];
      if (m > 0) v += m * b01 * V[n][m - 1];
      if (n > 0) v += n * b00 * V[n - 1][m];
      V[n][m + 1] = v;
    }
  }
  double W[LA + 1][LB + 1][MMX + 1];
#pragma unroll
  for (int m = 0; m <= MMX; ++m) {
    double h[NMX + 1];
#pragma unroll
    for (int i = 0; i <= NMX; ++i) h[i] = V[i][m];
#pragma unroll
    for (int j = 0; j <= LB; ++j) {
#pragma unroll
      for (int i = 0; i <= LA; ++i) W[i][j][m] = h[i];
#pragma unroll
      for (int i = 0; i + j < NMX; ++i) h[i] = h[i + 1] + ab * h[i];
    }
  }
#pragma unroll
  for (int i = 0; i <= LA; ++i) {
#pragma unroll
    for (int j = 0; j <= LB; ++j) {
      double g[MMX + 1];
#pragma unroll
      for (int k = 0; k <= MMX; ++k) g[k] = W[i][j][k];
#pragma unroll
      for (int l = 0; l <= LD; ++l) {
#pragma unroll
        for (int k = 0; k <= LC; ++k) I[i][j][k][l] = g[k];
#pragma unroll
        for (int k = 0; k + l < MMX; ++k) g[k] = g[k + 1] + cd * g[k];
      }
    }
  }
}

// Fock-build parameters that ride in KParams: G = P.grad ([4][nbf][nbf]); pair weights in MJ[0..3] (jw) and MK[0..3] (kw).
template <int LA, int LB, int LC, int LD, int AB0, int ABC>
__device__ __forceinline__ void quartet_fock(const KParams& P, const PairHdr& bh, const double* __restrict__ bprim, const PairHdr& kh,
                                             const double* __restrict__ kprim, double deg, const double* __restrict__ rys) {
  typedef QC<LA, LB, LC, LD> C;
  constexpr int NA = C::NA, NB = C::NB, NC = C::NC, ND = C::ND, KDN = NC * ND;
  constexpr int NR = (LA + LB + LC + LD) / 2 + 1;
  // integrals of this role's function quartets: IJ (1/r, for J) and IK = cK (1/r) + cLR (erf) (for K), normalisation and deg folded in
  double IJ[ABC * KDN], IK[ABC * KDN];
#pragma unroll
  for (int t = 0; t < ABC * KDN; ++t) { IJ[t] = 0.0; IK[t] = 0.0; }
  const double ABx = bh.AB[0], ABy = bh.AB[1], ABz = bh.AB[2];
  const double CDx = kh.AB[0], CDy = kh.AB[1], CDz = kh.AB[2];
  for (int ib = 0; ib < P.nppb; ++ib) {
    const d4 bp0 = ld256(bprim + ib * TDG_PRIM_STRIDE), bp1 = ld256(bprim + ib * TDG_PRIM_STRIDE + 4);
    const double p = bp0.x, Px = bp0.y, Py = bp0.z, Pz = bp0.w, Kab = 34.986836655249725693 /* 2 pi^(5/2) */ * bp1.x, rp = bp1.w;
    const double PAx = Px - bh.A[0], PAy = Py - bh.A[1], PAz = Pz - bh.A[2];
    for (int ik = 0; ik < P.nppk; ++ik) {
      const d4 kp0 = ld256(kprim + ik * TDG_PRIM_STRIDE), kp1 = ld256(kprim + ik * TDG_PRIM_STRIDE + 4);
      const double q = kp0.x, Qx = kp0.y, Qy = kp0.z, Qz = kp0.w, rq = kp1.w;
      const double QCx = Qx - kh.A[0], QCy = Qy - kh.A[1], QCz = Qz - kh.A[2];
      const double PQx = Px - Qx, PQy = Py - Qy, PQz = Pz - Qz;
      const double rs = rsqrt(p + q), rpq = rs * rs, rho = p * q * rpq;
      const double T = rho * (PQx * PQx + PQy * PQy + PQz * PQz);
      const double pref = deg * Kab * kp1.x * rs;
      for (int op = 0; op <= P.use_lr; ++op) {
        double s2 = 1.0, ss = 1.0;
        if (op == 1) { ss = P.omega * rsqrt(P.omega2 + rho); s2 = ss * ss; }
        double xr[NR], wr[NR];
        rys_eval<NR, (NR <= 4)>(rys, s2 * T, xr, wr);
        const double wj = op == 0 ? 1.0 : 0.0, wk = op == 0 ? P.cK : P.cLR;
#pragma unroll
        for (int r = 0; r < NR; ++r) {
          const double x = xr[r] * s2, w = wr[r] * ss * pref;
          const double b00 = 0.5 * x * rpq, b10 = (0.5 - q * b00) * rp, b01 = (0.5 - p * b00) * rq;
          const double fq = q * rpq * x, fp = p * rpq * x;
          double Ix[LA + 1][LB + 1][LC + 1][LD + 1], Iy[LA + 1][LB + 1][LC + 1][LD + 1], Iz[LA + 1][LB + 1][LC + 1][LD + 1];
          build2d_plain<LA, LB, LC, LD>(PAx - fq * PQx, QCx + fp * PQx, b00, b10, b01, ABx, CDx, 1.0, Ix);
          build2d_plain<LA, LB, LC, LD>(PAy - fq * PQy, QCy + fp * PQy, b00, b10, b01, ABy, CDy, 1.0, Iy);
          build2d_plain<LA, LB, LC, LD>(PAz - fq * PQz, QCz + fp * PQz, b00, b10, b01, ABz, CDz, w, Iz);
#pragma unroll
          for (int ab = AB0; ab < AB0 + ABC; ++ab) {
            const int a = ab / NB, b = ab - a * NB;
            int ax, ay, az, bx, by, bz;
            comp_exps<LA, true>(a, ax, ay, az); comp_exps<LB, true>(b, bx, by, bz);
#pragma unroll
            for (int c = 0; c < NC; ++c) {
              int cx, cy, cz; comp_exps<LC, true>(c, cx, cy, cz);
#pragma unroll
              for (int d = 0; d < ND; ++d) {
                int dx, dy, dz; comp_exps<LD, true>(d, dx, dy, dz);
                const double v = Ix[ax][bx][cx][dx] * Iy[ay][by][cy][dy] * Iz[az][bz][cz][dz];
                const int idx = ((ab - AB0) * NC + c) * ND + d;
                IJ[idx] = fma(wj, v, IJ[idx]);
                IK[idx] = fma(wk, v, IK[idx]);
              }
            }
          }
        }
      }
    }
  }
  // ---- digestion: 4 canonical matrices at once (256-bit loads of the packed blocks), FP64 RED into G[slot][row][col] ----
  const size_t n = (size_t)P.nbf, n2 = n * n;
  const double* __restrict__ pk = P.pk;
  double* __restrict__ G = P.grad;
  const int oi = bh.offA, oj = bh.offB, ok = kh.offA, ol = kh.offB;
  auto blk = [&](int rowsh_off, int nrow, int colsh_off) { return pk + 4 * ((size_t)rowsh_off * n + (size_t)nrow * colsh_off); };
  const double* bKL = blk(ok, NC, ol);   // S[l s] rows k, cols l
  const double* bIJ = blk(oi, NA, oj);
  const double* bKJ = blk(ok, NC, oj);   // X[l n]
  const double* bKI = blk(ok, NC, oi);   // X[l m]
  const double* bLJ = blk(ol, ND, oj);   // X[s n]
  const double* bLI = blk(ol, ND, oi);   // X[s m]
  auto red4 = [&](size_t row, size_t col, const double (&v)[4], const double* wgt, double sign) {
#pragma unroll
    for (int s = 0; s < 4; ++s)
      if (wgt[s] != 0.0) red_add(G + (size_t)s * n2 + row * n + col, sign * wgt[s] * v[s]);
  };
  const double* jw = P.MJ;   // [4]
  const double* kw = P.MK;   // [4]
  // normalisation of the components
  double cnab[ABC];
#pragma unroll
  for (int ab = AB0; ab < AB0 + ABC; ++ab) cnab[ab - AB0] = cnorm_c(LA, ab / NB) * cnorm_c(LB, ab % NB);
#pragma unroll
  for (int ab = AB0; ab < AB0 + ABC; ++ab)
#pragma unroll
    for (int cd = 0; cd < KDN; ++cd) {
      const double cn = cnab[ab - AB0] * cnorm_c(LC, cd / ND) * cnorm_c(LD, cd % ND);
      IJ[(ab - AB0) * KDN + cd] *= cn; IK[(ab - AB0) * KDN + cd] *= cn;
    }
  // Coulomb, bra block (i,j): G[m n] += jw S[l s] I
#pragma unroll
  for (int ab = AB0; ab < AB0 + ABC; ++ab) {
    const int a = ab / NB, b = ab - a * NB;
    double acc[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
    for (int cd = 0; cd < KDN; ++cd) {
      const d4 s = ld256(bKL + 4 * cd);
      const double v = IJ[(ab - AB0) * KDN + cd];
      acc[0] = fma(s.x, v, acc[0]); acc[1] = fma(s.y, v, acc[1]); acc[2] = fma(s.z, v, acc[2]); acc[3] = fma(s.w, v, acc[3]);
    }
    red4(oi + a, oj + b, acc, jw, 1.0);
  }
  // Coulomb, ket block (k,l): G[l s] += jw S[m n] I  (this role's share of the sum over the bra functions)
#pragma unroll
  for (int cd = 0; cd < KDN; ++cd) {
    double acc[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
    for (int ab = AB0; ab < AB0 + ABC; ++ab) {
      const d4 s = ld256(bIJ + 4 * ab);
      const double v = IJ[(ab - AB0) * KDN + cd];
      acc[0] = fma(s.x, v, acc[0]); acc[1] = fma(s.y, v, acc[1]); acc[2] = fma(s.z, v, acc[2]); acc[3] = fma(s.w, v, acc[3]);
    }
    red4(ok + cd / ND, ol + cd % ND, acc, jw, 1.0);
  }
  // exchange: four output blocks; sums over the two contracted functions
  constexpr int A0 = AB0 / NB, A1 = (AB0 + ABC - 1) / NB;   // rows a touched by this role
#pragma unroll
  for (int a = A0; a <= A1; ++a) {
#pragma unroll
    for (int d = 0; d < ND; ++d) {   // G[m s] -= kw sum_{n l} X[l n] Ik
      double acc[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
      for (int b = 0; b < NB; ++b) {
        if (a * NB + b < AB0 || a * NB + b >= AB0 + ABC) continue;
#pragma unroll
        for (int c = 0; c < NC; ++c) {
          const d4 s = ld256(bKJ + 4 * (c * NB + b));
          const double v = IK[((a * NB + b - AB0) * NC + c) * ND + d];
          acc[0] = fma(s.x, v, acc[0]); acc[1] = fma(s.y, v, acc[1]); acc[2] = fma(s.z, v, acc[2]); acc[3] = fma(s.w, v, acc[3]);
        }
      }
      red4(oi + a, ol + d, acc, kw, -1.0);
    }
#pragma unroll
    for (int c = 0; c < NC; ++c) {   // G[m l] -= kw sum_{n s} X[s n] Ik
      double acc[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
      for (int b = 0; b < NB; ++b) {
        if (a * NB + b < AB0 || a * NB + b >= AB0 + ABC) continue;
#pragma unroll
        for (int d = 0; d < ND; ++d) {
          const d4 s = ld256(bLJ + 4 * (d * NB + b));
          const double v = IK[((a * NB + b - AB0) * NC + c) * ND + d];
          acc[0] = fma(s.x, v, acc[0]); acc[1] = fma(s.y, v, acc[1]); acc[2] = fma(s.z, v, acc[2]); acc[3] = fma(s.w, v, acc[3]);
        }
      }
      red4(oi + a, ok + c, acc, kw, -1.0);
    }
  }
#pragma unroll
  for (int b = 0; b < NB; ++b) {
    bool any = false;
#pragma unroll
    for (int a = A0; a <= A1; ++a) any = any || (a * NB + b >= AB0 && a * NB + b < AB0 + ABC);
    if (!any) continue;
#pragma unroll
    for (int d = 0; d < ND; ++d) {   // G[n s] -= kw sum_{m l} X[l m] Ik
      double acc[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
      for (int a = A0; a <= A1; ++a) {
        if (a * NB + b < AB0 || a * NB + b >= AB0 + ABC) continue;
#pragma unroll
        for (int c = 0; c < NC; ++c) {
          const d4 s = ld256(bKI + 4 * (c * NA + a));
          const double v = IK[((a * NB + b - AB0) * NC + c) * ND + d];
          acc[0] = fma(s.x, v, acc[0]); acc[1] = fma(s.y, v, acc[1]); acc[2] = fma(s.z, v, acc[2]); acc[3] = fma(s.w, v, acc[3]);
        }
      }
      red4(oj + b, ol + d, acc, kw, -1.0);
    }
#pragma unroll
    for (int c = 0; c < NC; ++c) {   // G[n l] -= kw sum_{m s} X[s m] Ik
      double acc[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
      for (int a = A0; a <= A1; ++a) {
        if (a * NB + b < AB0 || a * NB + b >= AB0 + ABC) continue;
#pragma unroll
        for (int d = 0; d < ND; ++d) {
          const d4 s = ld256(bLI + 4 * (d * NA + a));
          const double v = IK[((a * NB + b - AB0) * NC + c) * ND + d];
          acc[0] = fma(s.x, v, acc[0]); acc[1] = fma(s.y, v, acc[1]); acc[2] = fma(s.z, v, acc[2]); acc[3] = fma(s.w, v, acc[3]);
        }
      }
      red4(oj + b, ok + c, acc, kw, -1.0);
    }
  }
}

template <int LA, int LB, int LC, int LD, int ROLE>
__global__ void __launch_bounds__(TDG_NT) tdg_fock_kernel(const __grid_constant__ KParams P) {
  __shared__ PairHdr s_bra[TDG_WARP];
  __shared__ PairHdr s_ket[TDG_KB];
  __shared__ double s_dij[TDG_WARP];
  extern __shared__ double2 s_dyn[];
  typedef QC<LA, LB, LC, LD> C;
  constexpr int NR = (LA + LB + LC + LD) / 2 + 1;
  constexpr bool RYS_SH = NR <= 4;
  int tile, chunk;
  find_work_item(P, blockIdx.x, tile, chunk);
  const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
  const int bra0 = tile * TDG_WARP, k0 = chunk * TDG_KB;
  const int nb = min(TDG_WARP, P.nbra - bra0);
  const bool dw = P.tau > 0.0 && P.density_weighted;
  if (t < nb) {
    const PairHdr h = P.bra_hdr[bra0 + t];
    s_bra[t] = h;
    s_dij[t] = dw ? __ldg(P.dmax + (size_t)h.ish * P.nshell + h.jsh) : 0.0;
  }
  const int k = k0 + t;
  const bool ket_ok = k < P.nket;
  if (ket_ok) s_ket[t] = P.ket_hdr[k];
  const double* rys = P.rys_tab + rys_part_off(NR);
  if (RYS_SH) {
    const double2* src = reinterpret_cast<const double2*>(rys);
    for (int i = t; i < rys_part_doubles(NR) / 2; i += TDG_NT) s_dyn[rys_sh_index<NR>(i)] = __ldg(src + i);   // conflict-free staged layout (tdg_common.cuh)
    rys = reinterpret_cast<const double*>(s_dyn);
  }
  __syncthreads();
  unsigned long long n_vis = 0, n_cmp = 0;
  const unsigned mask = ket_ok ? screen_ket(P, s_bra, s_dij, nb, bra0, k, s_ket[t], dw, n_vis, n_cmp) : 0u;
  const int cnt = __popc(mask);
  int incl = cnt;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const int v = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += v; }
  const int tot = __shfl_sync(0xffffffffu, incl, 31), pre = incl - cnt;
  static_assert(ROLE >= 0 && ROLE < C::NROLE, "role out of range");
  constexpr int AB0 = ROLE * C::ABN;
  constexpr int ABC = (AB0 + C::ABN <= C::NAB) ? C::ABN : C::NAB - AB0;
  const int kw0 = warp * TDG_KW;
  for (int base = 0; base < tot; base += TDG_WARP) {
    const int s = base + lane;
    int kt, b;
    warp_survivor(mask, pre, s < tot ? s : tot - 1, kt, b);
    if (s < tot) {
      const PairHdr& bh = s_bra[b];
      const PairHdr& kh = s_ket[kw0 + kt];
      double deg = 1.0;
      if (bh.ish == bh.jsh) deg *= 0.5;
      if (kh.ish == kh.jsh) deg *= 0.5;
      if (P.same_bucket && k0 + kw0 + kt == bra0 + b) deg *= 0.5;
      quartet_fock<LA, LB, LC, LD, AB0, ABC>(P, bh, P.bra_prim + (size_t)(bra0 + b) * P.nppb * TDG_PRIM_STRIDE, kh,
                                             P.ket_prim + (size_t)(k0 + kw0 + kt) * P.nppk * TDG_PRIM_STRIDE, deg, rys);
    }
  }
  for (int o = 16; o > 0; o >>= 1) {
    n_vis += __shfl_xor_sync(0xffffffffu, n_vis, o);
    n_cmp += __shfl_xor_sync(0xffffffffu, n_cmp, o);
  }
  if (ROLE == 0 && lane == 0 && n_vis) {
    atomicAdd(P.counters + 0, n_vis); atomicAdd(P.counters + 1, n_cmp);
    atomicAdd(P.counters + 2, n_cmp * (unsigned long long)(P.nppb * P.nppk));
  }
}
