// tdg_grad.cuh — per-class ERI-derivative + density-contraction kernel (steps a4-a8; Fig. 1).
//
// Work mapping (differs from Fig. 1's "1 thread = 1 batch" over a dense supermatrix): a block work item
// is one bra tile of 32 consecutive sorted shell pairs times a chunk of TDG_KB sorted ket pairs.  Phase 1 screens the
// 32 x TDG_KB candidates (one ket per thread) and compacts the survivors into a shared-memory list; phase 2 processes
// the survivors densely, one quartet per thread, so lanes do not idle on quartets the density-weighted test rejected.
// Gradient contributions go to per-block shared-memory accumulators (one slot per bra/ket pair centre) that are flushed
// with one FP64 atomic per touched slot.  The fourth centre follows from translational invariance (eq 41).
//
// Integrals: Rys quadrature: n_r = floor((L+1)/2)+1 roots (reading S6) for the full operator and
// again for erf(omega r)/r (roots at s^2 T, x <- s^2 x, w <- s w; reading S8); 2-D recurrences of DESIGN.md
// "Rys 2-D recurrences"; centre derivative of eq 39/42 applied to the 2-D integral of
// one direction.  The derivative batch is never stored: each (component, root) term is multiplied by the
// symmetrised density product Gt (eqs 13-14) and accumulated into 9 scalars.
#pragma once
#include "tdg_common.cuh"
#define TDG_NT (TDG_WARPS * TDG_WARP)
#define TDG_ACC_DOUBLES ((TDG_WARPS * TDG_WARP + TDG_KB) * 6)   // per-warp bra slots + ket slots (each ket belongs to one warp)
#ifndef TDG_RU_LIM
#define TDG_RU_LIM 120
#endif
#ifndef TDG_STAGE_IJ
#define TDG_STAGE_IJ 1
#endif
#ifndef TDG_DUAL_RYS
#define TDG_DUAL_RYS 0   // per class (build.py CLASS_FLAGS): -4 % on (ps|ps), -1 % on (ss|ss), +5 % on (ds|ss) (spills), neutral on (ps|ss), (pp|ss)
#endif
#ifndef TDG_STAGE_IJ_MAXAB
#define TDG_STAGE_IJ_MAXAB 3   // measured on cfg 3 (profiles/r02_variants.md): -1 % on ss and ps bras, +1..10 % on pp, ds, dp bras
#endif
#define TDG_MAX_ROLES_F 15   // f classes up to 15 roles run unrolled (cfg 2: 13.1 s -> 9.6 s against 8; each role is a 25-45 s compile)
#define TDG_MAX_ROLES 18  // classes needing more roles ((dd|dd), f shells) use the block-per-quartet kernel (tdg_gradb.cuh)
// target number of function quartets per role: 27 is the measured optimum (14: +30 %, 54: +15 % time on cfg 3), except
// (dd|dp), which needs 54 to stay within TDG_MAX_ROLES (12 roles; 10x faster than the block-per-quartet kernel on cfg 3)
__host__ __device__ constexpr int role_comps(int la, int lb, int lc, int ld) {
  return (la == 2 && lb == 2 && lc == 2 && ld == 1) ? 54 : 27;
}

template <int LA, int LB, int LC, int LD>
struct QC {
  static constexpr int NA = ncart(LA), NB = ncart(LB), NC = ncart(LC), ND = ncart(LD);
  static constexpr int NCOMP = NA * NB * NC * ND;
  static constexpr int L = LA + LB + LC + LD;
  static constexpr int NR = (L + 1) / 2 + 1;
  static constexpr int DA = LA + 2, DB = LB + 2, DC = LC + 2, DD = LD + 1;
  static constexpr int NMX = LA + LB + 1, MMX = LC + LD + 1;
  // Component slicing ("roles", grid.y): a block of role r handles the bra function pairs ab in [r*ABN, (r+1)*ABN) of
  // every surviving quartet, so that a thread holds at most ~27 density products and fully unrolled code stays in
  // registers; the 2-D integrals are rebuilt by every role.  Classes with an f shell keep rolled loops (one role).
  static constexpr bool HASF = LA == 3 || LB == 3 || LC == 3 || LD == 3;
  static constexpr int NAB = NA * NB, KDN = NC * ND;
  static constexpr int RC = role_comps(LA, LB, LC, LD);
  static constexpr int ABN1 = RC / KDN >= NAB ? NAB : (RC / KDN > 0 ? RC / KDN : 1);
  static constexpr int NROLE1 = (NAB + ABN1 - 1) / ABN1;
  // thread-per-quartet, fully unrolled code: up to 18 roles without f shells, up to 15 with (longer compiles; measured on cfg 2:
  // the block-per-quartet kernel is 5-10x slower on the small f classes, which carry most of that config's quartets)
  static constexpr bool SMALL = NCOMP <= 27 || NROLE1 <= (HASF ? TDG_MAX_ROLES_F : TDG_MAX_ROLES);
  static constexpr int NROLE = SMALL ? NROLE1 : 1;
  static constexpr int ABN = (NAB + NROLE - 1) / NROLE;
  static constexpr int UNR = SMALL ? 64 : 1;
  static constexpr bool TWO_STAGE = SMALL && NROLE <= 2;   // measured: faster for 1-2 roles, slower for classes with more roles
  static constexpr bool RYS_SH = NR <= 4;                                  // Rys table of this NR staged in shared memory
  static constexpr int RYS_SH_DOUBLES = RYS_SH ? rys_sh_doubles(NR) : 0;    // staged size (padded layout, tdg_common.cuh)
  static constexpr int RYS_SRC_DOUBLES = RYS_SH ? rys_part_doubles(NR) : 0;
  static constexpr int RUNR = (SMALL && ABN * KDN * NR <= TDG_RU_LIM) ? 64 : 1;   // root loop
  // (ij) density blocks of the 32 bras of a tile staged in shared memory, already multiplied by M_J (step a7): bra-invariant over
  // the kets of the work item, so one global gather per block instead of one per quartet
  static constexpr bool DUAL_RYS = TDG_DUAL_RYS && NR <= 2;
  static constexpr bool IJ_SH = TDG_STAGE_IJ && SMALL && NAB <= TDG_STAGE_IJ_MAXAB;
  static constexpr int IJ_SH_DOUBLES = IJ_SH ? TDG_WARP * NAB * 4 : 0;
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
  if (SMALL) {
    x = (int)((CartPack<L, 0>::v >> (4 * idx)) & 15); y = (int)((CartPack<L, 1>::v >> (4 * idx)) & 15); z = (int)((CartPack<L, 2>::v >> (4 * idx)) & 15);
  }
  else { unsigned v = c_cart[L][idx]; x = v & 15; y = (v >> 4) & 15; z = (v >> 8) & 15; }
}

// Compile-time mask of the bra exponent pairs (i, j) that occur, in any direction, among the function pairs
// ab in [AB0, AB0+ABC) of a role: stage 2 of the contraction skips the others (their H entries are never touched).
template <int LA, int LB, int AB0, int ABC>
constexpr unsigned make_touch() {   // bit i*5+j
  unsigned m = 0;
  for (int ab = AB0; ab < AB0 + ABC; ++ab) {
    const int a = ab / ncart(LB), b = ab - a * ncart(LB);
    for (int d = 0; d < 3; ++d) m |= 1u << (cart_exp(LA, a, d) * 5 + cart_exp(LB, b, d));
  }
  return m;
}
template <int LA, int LB, int AB0, int ABC> struct Touch { static constexpr unsigned v = make_touch<LA, LB, AB0, ABC>(); };

// Gradient contribution of one shell quartet: g[0..2] = d/dA, g[3..5] = d/dB, g[6..8] = d/dC (sum over all
// functions, primitives, roots and both operators, already multiplied by deg and the density products).
template <int LA, int LB, int LC, int LD, int AB0, int ABC>
__device__ __forceinline__ void quartet_grad(const KParams& P, const PairHdr& bh, const double* __restrict__ bprim,
                                             const PairHdr& kh, const double* __restrict__ kprim, double deg,
                                             const double* __restrict__ rys, const double* __restrict__ sIJ, double (&g)[9]) {
  typedef QC<LA, LB, LC, LD> C;
  constexpr int NA = C::NA, NB = C::NB, NC = C::NC, ND = C::ND, NR = C::NR, U = C::UNR, RU = C::RUNR;
  constexpr bool SM = C::SMALL;
  typedef Touch<LA, LB, AB0, ABC> TM;
  // this role's bra function pairs: ab = a*NB + b in [AB0, AB0+ABC)
  double GF[ABC * NC * ND], GL[ABC * NC * ND];
  {  // step a7, part 1: symmetrised density products for every function quartet, from the packed blocks
    //   Gt_K = u.MK.v + s.MK.t,  u = pk(ik)[a,c], v = pk(jl)[b,d], s = pk(jk)[b,c], t = pk(il)[a,d];  Gt_J = pk(ij)[a,b].MJ.pk(kl)[c,d]
    const size_t n = (size_t)P.nbf;
    const double* __restrict__ pk = P.pk;
    const double* bIK = pk + 4 * ((size_t)bh.offA * n + (size_t)NA * kh.offA);
    const double* bJL = pk + 4 * ((size_t)bh.offB * n + (size_t)NB * kh.offB);
    const double* bJK = pk + 4 * ((size_t)bh.offB * n + (size_t)NB * kh.offA);
    const double* bIL = pk + 4 * ((size_t)bh.offA * n + (size_t)NA * kh.offB);
    const double* bIJ = pk + 4 * ((size_t)bh.offA * n + (size_t)NA * bh.offB);
    const double* bKL = pk + 4 * ((size_t)kh.offA * n + (size_t)NC * kh.offB);
    // transformed small blocks: MK.v (jl), MK.t (il), MJ.(kl)
    double vJL[NB * ND][4], tIL[NA * ND][4], vKL[NC * ND][4];
#pragma unroll(U)
    for (int e = 0; e < NB * ND; ++e) {
      const d4 x = ld256(bJL + 4 * e);
#pragma unroll
      for (int m = 0; m < 4; ++m) vJL[e][m] = P.MK[4 * m] * x.x + P.MK[4 * m + 1] * x.y + P.MK[4 * m + 2] * x.z + P.MK[4 * m + 3] * x.w;
    }
#pragma unroll(U)
    for (int e = 0; e < NA * ND; ++e) {
      const d4 x = ld256(bIL + 4 * e);
#pragma unroll
      for (int m = 0; m < 4; ++m) tIL[e][m] = P.MK[4 * m] * x.x + P.MK[4 * m + 1] * x.y + P.MK[4 * m + 2] * x.z + P.MK[4 * m + 3] * x.w;
    }
#pragma unroll(U)
    for (int e = 0; e < NC * ND; ++e) {
      const d4 x = ld256(bKL + 4 * e);
      if constexpr (C::IJ_SH) { vKL[e][0] = x.x; vKL[e][1] = x.y; vKL[e][2] = x.z; vKL[e][3] = x.w; }   // M_J is already in the staged (ij) block
      else {
#pragma unroll
        for (int m = 0; m < 4; ++m) vKL[e][m] = P.MJ[4 * m] * x.x + P.MJ[4 * m + 1] * x.y + P.MJ[4 * m + 2] * x.z + P.MJ[4 * m + 3] * x.w;
      }
    }
#pragma unroll(U)
    for (int ab = AB0; ab < AB0 + ABC; ++ab) {
      {
        const int a = ab / NB, b = ab - a * NB;
        d4 jv;
        if constexpr (C::IJ_SH) {
          const double2 j0 = *reinterpret_cast<const double2*>(sIJ + 4 * ab), j1 = *reinterpret_cast<const double2*>(sIJ + 4 * ab + 2);
          jv.x = j0.x; jv.y = j0.y; jv.z = j1.x; jv.w = j1.y;
        } else jv = ld256(bIJ + 4 * (a * NB + b));
#pragma unroll(U)
        for (int c = 0; c < NC; ++c) {
          const d4 u = ld256(bIK + 4 * (a * NC + c));
          const d4 sv = ld256(bJK + 4 * (b * NC + c));
#pragma unroll(U)
          for (int d = 0; d < ND; ++d) {
            const double* v = vJL[b * ND + d]; const double* tt = tIL[a * ND + d]; const double* w = vKL[c * ND + d];
            const double gk = u.x * v[0] + u.y * v[1] + u.z * v[2] + u.w * v[3] + sv.x * tt[0] + sv.y * tt[1] + sv.z * tt[2] + sv.w * tt[3];
            const double gj = jv.x * w[0] + jv.y * w[1] + jv.z * w[2] + jv.w * w[3];
            const double cn = deg * (cnorm_c(LA, a) * cnorm_c(LB, b) * cnorm_c(LC, c) * cnorm_c(LD, d));
            const int idx = ((ab - AB0) * NC + c) * ND + d;
            GF[idx] = cn * (gj + P.cK * gk);
            GL[idx] = cn * P.cLR * gk;
          }
        }
      }
    }
  }
#pragma unroll
  for (int t = 0; t < 9; ++t) g[t] = 0.0;
  const double ABx = bh.AB[0], ABy = bh.AB[1], ABz = bh.AB[2];
  const double CDx = kh.AB[0], CDy = kh.AB[1], CDz = kh.AB[2];
  // primitive-pair record (tdg_common.cuh): p, Px, Py, Pz, K_ab/p, a, b, 1/p.  With rs = (p+q)^(-1/2):
  //   2 pi^(5/2) K_ab K_cd / (p q sqrt(p+q)) = C (K_ab/p) (K_cd/q) rs;  1/(p+q) = rs^2;  s = omega (omega^2+rho)^(-1/2)  (S8)
  for (int ib = 0; ib < P.nppb; ++ib) {
    const d4 bp0 = ld256(bprim + ib * TDG_PRIM_STRIDE), bp1 = ld256(bprim + ib * TDG_PRIM_STRIDE + 4);
    const double p = bp0.x, Px = bp0.y, Py = bp0.z, Pz = bp0.w, Kab = 34.986836655249725693 /* 2 pi^(5/2) */ * bp1.x, a2 = 2.0 * bp1.y, b2 = 2.0 * bp1.z, rp = bp1.w;
    const double PAx = Px - bh.A[0], PAy = Py - bh.A[1], PAz = Pz - bh.A[2];
    for (int ik = 0; ik < P.nppk; ++ik) {
      const d4 kp0 = ld256(kprim + ik * TDG_PRIM_STRIDE), kp1 = ld256(kprim + ik * TDG_PRIM_STRIDE + 4);
      const double q = kp0.x, Qx = kp0.y, Qy = kp0.z, Qz = kp0.w, c2 = 2.0 * kp1.y, rq = kp1.w;
      const double QCx = Qx - kh.A[0], QCy = Qy - kh.A[1], QCz = Qz - kh.A[2];
      const double PQx = Px - Qx, PQy = Py - Qy, PQz = Pz - Qz;
      const double rs = rsqrt(p + q), rpq = rs * rs, rho = p * q * rpq;
      const double T = rho * (PQx * PQx + PQy * PQy + PQz * PQz);
      const double pref = Kab * kp1.x * rs;
      // n <= 2: the rules of both operators are evaluated back to back, unconditionally, before the operator loop, so that their
      // two dependency chains (exp, Taylor row, closed-form roots) interleave; the loop then picks its set with selects
      double xa[C::DUAL_RYS ? 2 * NR : 1], wa[C::DUAL_RYS ? 2 * NR : 1];
      if constexpr (C::DUAL_RYS) {
        const double ssl = P.omega * rsqrt(P.omega2 + rho), s2l = ssl * ssl;   // omega = 0 (no long-range pass): T = 0, unused
        rys_eval<NR, C::RYS_SH>(rys, T, xa, wa);
        rys_eval<NR, C::RYS_SH>(rys, s2l * T, xa + NR, wa + NR);
#pragma unroll
        for (int r = 0; r < NR; ++r) { xa[NR + r] *= s2l; wa[NR + r] *= ssl; }
      }
      for (int op = 0; op <= P.use_lr; ++op) {
        double s2 = 1.0, ss = 1.0;
        double xr[NR], wr[NR];
        if constexpr (C::DUAL_RYS) {
#pragma unroll
          for (int r = 0; r < NR; ++r) { xr[r] = op == 0 ? xa[r] : xa[NR + r]; wr[r] = op == 0 ? wa[r] : wa[NR + r]; }
        } else {
          if (op == 1) { ss = P.omega * rsqrt(P.omega2 + rho); s2 = ss * ss; }
          rys_eval<NR, C::RYS_SH>(rys, s2 * T, xr, wr);
        }
        const double* __restrict__ G = op == 0 ? GF : GL;
#pragma unroll(RU)
        for (int r = 0; r < NR; ++r) {
          const double x = xr[r] * s2, w = wr[r] * ss * pref;
          const double b00 = 0.5 * x * rpq, b10 = (0.5 - q * b00) * rp, b01 = (0.5 - p * b00) * rq;
          const double fq = q * rpq * x, fp = p * rpq * x;
          double Ix[C::DA][C::DB][C::DC][C::DD], Iy[C::DA][C::DB][C::DC][C::DD], Iz[C::DA][C::DB][C::DC][C::DD];
          build2d<LA, LB, LC, LD>(PAx - fq * PQx, QCx + fp * PQx, b00, b10, b01, ABx, CDx, 1.0, Ix);
          build2d<LA, LB, LC, LD>(PAy - fq * PQy, QCy + fp * PQy, b00, b10, b01, ABy, CDy, 1.0, Iy);
          build2d<LA, LB, LC, LD>(PAz - fq * PQz, QCz + fp * PQz, b00, b10, b01, ABz, CDz, w, Iz);
          if constexpr (C::TWO_STAGE) {
          // step a7, part 2, two stages.  Stage 1 sums the density products times the two undifferentiated directions
          // over all functions that share the exponent tuple (i,j,k,l) of the third direction:
          //   Hx[i,j,k,l] = sum_{functions with x-exponents (i,j,k,l)} Gt * Iy * Iz   (and cyclically Hy, Hz).
          // Stage 2 applies the centre derivatives (eq 39/42) once per tuple instead of once per function quartet:
          //   g_Ax += Hx[t] (2a Ix[i+1..] - i Ix[i-1..]),  g_Bx, g_Cx likewise.
          double Hx[LA + 1][LB + 1][LC + 1][LD + 1], Hy[LA + 1][LB + 1][LC + 1][LD + 1], Hz[LA + 1][LB + 1][LC + 1][LD + 1];
#pragma unroll(U)
          for (int i = 0; i <= LA; ++i)
#pragma unroll(U)
            for (int j = 0; j <= LB; ++j)
#pragma unroll(U)
              for (int k = 0; k <= LC; ++k)
#pragma unroll(U)
                for (int l = 0; l <= LD; ++l) { Hx[i][j][k][l] = 0.0; Hy[i][j][k][l] = 0.0; Hz[i][j][k][l] = 0.0; }
#pragma unroll(U)
          for (int ab = AB0; ab < AB0 + ABC; ++ab) {
            const int a = ab / NB, b = ab - a * NB;
            int ax, ay, az; comp_exps<LA, SM>(a, ax, ay, az);
            {
              int bx, by, bz; comp_exps<LB, SM>(b, bx, by, bz);
#pragma unroll(U)
              for (int c = 0; c < NC; ++c) {
                int cx, cy, cz; comp_exps<LC, SM>(c, cx, cy, cz);
#pragma unroll(U)
                for (int d = 0; d < ND; ++d) {
                  int dx, dy, dz; comp_exps<LD, SM>(d, dx, dy, dz);
                  const double Gv = G[((ab - AB0) * NC + c) * ND + d];
                  const double X0 = Ix[ax][bx][cx][dx], Y0 = Iy[ay][by][cy][dy], Z0 = Iz[az][bz][cz][dz];
                  const double gz = Gv * Z0;
                  Hx[ax][bx][cx][dx] += gz * Y0;
                  Hy[ay][by][cy][dy] += gz * X0;
                  Hz[az][bz][cz][dz] += Gv * X0 * Y0;
                }
              }
            }
          }
#pragma unroll(U)
          for (int i = 0; i <= LA; ++i)
#pragma unroll(U)
            for (int j = 0; j <= LB; ++j) {
              if (SM && !((TM::v >> (i * 5 + j)) & 1u)) continue;   // exponent pair (i,j) of the bra not present in this role's slice
#pragma unroll(U)
              for (int k = 0; k <= LC; ++k)
#pragma unroll(U)
                for (int l = 0; l <= LD; ++l) {
                  const double hx = Hx[i][j][k][l], hy = Hy[i][j][k][l], hz = Hz[i][j][k][l];
                  double dAx = a2 * Ix[i + 1][j][k][l], dAy = a2 * Iy[i + 1][j][k][l], dAz = a2 * Iz[i + 1][j][k][l];
                  if (i > 0) { dAx -= i * Ix[i - 1][j][k][l]; dAy -= i * Iy[i - 1][j][k][l]; dAz -= i * Iz[i - 1][j][k][l]; }
                  double dBx = b2 * Ix[i][j + 1][k][l], dBy = b2 * Iy[i][j + 1][k][l], dBz = b2 * Iz[i][j + 1][k][l];
                  if (j > 0) { dBx -= j * Ix[i][j - 1][k][l]; dBy -= j * Iy[i][j - 1][k][l]; dBz -= j * Iz[i][j - 1][k][l]; }
                  double dCx = c2 * Ix[i][j][k + 1][l], dCy = c2 * Iy[i][j][k + 1][l], dCz = c2 * Iz[i][j][k + 1][l];
                  if (k > 0) { dCx -= k * Ix[i][j][k - 1][l]; dCy -= k * Iy[i][j][k - 1][l]; dCz -= k * Iz[i][j][k - 1][l]; }
                  g[0] += hx * dAx; g[1] += hy * dAy; g[2] += hz * dAz;
                  g[3] += hx * dBx; g[4] += hy * dBy; g[5] += hz * dBz;
                  g[6] += hx * dCx; g[7] += hy * dCy; g[8] += hz * dCz;
                }
            }
          } else {
          // step a7, part 2: contract the derivative integrals of this root with Gt
#pragma unroll(U)
          for (int ab = AB0; ab < AB0 + ABC; ++ab) {
            const int a = ab / NB, b = ab - a * NB;
            int ax, ay, az; comp_exps<LA, SM>(a, ax, ay, az);
            {
              int bx, by, bz; comp_exps<LB, SM>(b, bx, by, bz);
#pragma unroll(U)
              for (int c = 0; c < NC; ++c) {
                int cx, cy, cz; comp_exps<LC, SM>(c, cx, cy, cz);
#pragma unroll(U)
                for (int d = 0; d < ND; ++d) {
                  int dx, dy, dz; comp_exps<LD, SM>(d, dx, dy, dz);
                  const double Gv = G[((ab - AB0) * NC + c) * ND + d];
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
}

__device__ __forceinline__ void red_add(double* addr, double v) { atomicAdd(addr, v); }

// ---- step a4 (reading S9): one ket against the nb bras of the tile -> 32-bit survivor mask ----
__device__ __forceinline__ unsigned screen_ket(const KParams& P, const PairHdr* s_bra, const double* s_dij, int nb, int bra0, int k,
                                               const PairHdr& kh, bool dw, unsigned long long& n_vis, unsigned long long& n_cmp) {
  const int ns = P.nshell;
  const int ksh = kh.ish, lsh = kh.jsh;
  const double Qk = kh.Q;
  const double dkl = dw ? __ldg(P.dmax + (size_t)ksh * ns + lsh) : 0.0;
  const bool ket_one = kh.atomA == kh.atomB;
  unsigned mask = 0;
  for (int b = 0; b < nb; ++b) {
    if (P.same_bucket && k > bra0 + b) continue;
    const PairHdr& bh = s_bra[b];
    if (P.tau > 0.0) {
      const double qq = bh.Q * Qk;
      if (!(qq >= P.tau)) continue;
      ++n_vis;
      if (dw && P.wmode == 0 && qq * (P.CJ * s_dij[b] * dkl) < P.tau) {
        // W = max(W_J, W_K) (S9): the J-type bound alone does not keep the quartet, so gather the four K-type maxima
        const double dik = __ldg(P.dmax + (size_t)bh.ish * ns + ksh), djl = __ldg(P.dmax + (size_t)bh.jsh * ns + lsh);
        const double dil = __ldg(P.dmax + (size_t)bh.ish * ns + lsh), djk = __ldg(P.dmax + (size_t)bh.jsh * ns + ksh);
        const double x1 = dik * djl, x2 = dil * djk;
        if (qq * (P.CK * (x1 > x2 ? x1 : x2)) < P.tau) continue;
      }
      if (dw && P.wmode == 1 && qq * (P.CJ * (s_dij[b] > dkl ? s_dij[b] : dkl)) < P.tau) {
        // Fock-type build: W = max(CJ max(d_ij, d_kl), CK max(d_ik, d_il, d_jk, d_jl))  (tdg_fock.cuh)
        const double dik = __ldg(P.dmax + (size_t)bh.ish * ns + ksh), djl = __ldg(P.dmax + (size_t)bh.jsh * ns + lsh);
        const double dil = __ldg(P.dmax + (size_t)bh.ish * ns + lsh), djk = __ldg(P.dmax + (size_t)bh.jsh * ns + ksh);
        double mk = dik > djl ? dik : djl;
        if (dil > mk) mk = dil;
        if (djk > mk) mk = djk;
        if (qq * (P.CK * mk) < P.tau) continue;
      }
    } else ++n_vis;
    if (!tdg_sample_keep(bh.ish, bh.jsh, ksh, lsh, P.sample_mod, P.sample_seed)) continue;
    ++n_cmp;
    // all four shells on one atom: the four centre derivatives sum to zero on that atom (reading S11); the undifferentiated
    // integrals of the Fock-type build (wmode 1) do not vanish
    if (P.wmode == 0 && ket_one && bh.atomA == bh.atomB && bh.atomA == kh.atomA) continue;
    mask |= 1u << b;
  }
  return mask;
}

// Survivor s of a warp's list (ket-major: lane o owns ket o with survivor mask `mask` and exclusive prefix `pre`):
// owner lane = largest o with pre_o <= s; bra = position of the (s - pre_o + 1)-th set bit of its mask.
__device__ __forceinline__ void warp_survivor(unsigned mask, int pre, int s, int& o, int& b) {
  o = 0;
#pragma unroll
  for (int step = 16; step > 0; step >>= 1) { const int pv = __shfl_sync(0xffffffffu, pre, o + step); if (pv <= s) o += step; }
  const unsigned m = __shfl_sync(0xffffffffu, mask, o);
  const int r = s - __shfl_sync(0xffffffffu, pre, o);
  b = (int)__fns(m, 0, r + 1);
}

// Phase 2 of the kernel for one role (slice [AB0, AB0+ABC) of the bra function pairs).
template <int LA, int LB, int LC, int LD, int AB0, int ABC>
__device__ __forceinline__ void process_survivors(const KParams& P, const PairHdr* s_bra, const PairHdr* s_ket, unsigned mask, int pre, int tot,
                                                  double* s_gb, double* s_gk, int bra0, int k0, const double* __restrict__ rys,
                                                  const double* __restrict__ s_ij) {
  // Each warp owns the 32 kets [32 w, 32 w + 32) of the chunk and takes passes of 32 consecutive entries of its ket-major
  // survivor list.  Gradient accumulation uses no atomics (shared-memory FP64 atomics are CAS loops of ~60 iterations
  // per warp and 6 RED per quartet saturate L2; both measured): lanes with the same ket are contiguous, so the ket-centre
  // terms are summed by a segmented warp shuffle scan and added by the segment head to the ket's slot (only this warp
  // touches it); the bra-centre terms are added to this warp's private bra slots segment by segment (bras are distinct
  // within a segment).  Fourth centre: eq 41.
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  double* my_gb = s_gb + warp * (TDG_WARP * 6);
  double* my_gk = s_gk + warp * (TDG_KW * 6);
  const int kw0 = warp * TDG_KW;
  for (int base = 0; base < tot; base += TDG_WARP) {
    const int s = base + lane;
    const bool act = s < tot;
    int kt, b;
    warp_survivor(mask, pre, act ? s : tot - 1, kt, b);
    double g[9];
    if (act) {
      const PairHdr& bh = s_bra[b];
      const PairHdr& kh = s_ket[kw0 + kt];
      double deg = 1.0;
      if (bh.ish == bh.jsh) deg *= 0.5;
      if (kh.ish == kh.jsh) deg *= 0.5;
      if (P.same_bucket && k0 + kw0 + kt == bra0 + b) deg *= 0.5;
      quartet_grad<LA, LB, LC, LD, AB0, ABC>(P, bh, P.bra_prim + (size_t)(bra0 + b) * P.nppb * TDG_PRIM_STRIDE, kh,
                                             P.ket_prim + (size_t)(k0 + kw0 + kt) * P.nppk * TDG_PRIM_STRIDE, deg, rys,
                                             s_ij + b * (QC<LA, LB, LC, LD>::NAB * 4), g);
    } else {
#pragma unroll
      for (int x = 0; x < 9; ++x) g[x] = 0.0;
    }
    const int key = act ? kt : -1 - lane;
    double v[6];
#pragma unroll
    for (int x = 0; x < 3; ++x) { v[x] = g[6 + x]; v[3 + x] = -(g[x] + g[3 + x] + g[6 + x]); }
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const int ko = __shfl_down_sync(0xffffffffu, key, o);
      const bool same = (lane + o < 32) && (ko == key);
#pragma unroll
      for (int x = 0; x < 6; ++x) { const double tv = __shfl_down_sync(0xffffffffu, v[x], o); if (same) v[x] += tv; }
    }
    const int kprev = __shfl_up_sync(0xffffffffu, key, 1);
    const bool head = (lane == 0) || (kprev != key);
    if (act && head) {
#pragma unroll
      for (int x = 0; x < 6; ++x) my_gk[kt * 6 + x] += v[x];
    }
    const unsigned hm = __ballot_sync(0xffffffffu, head);
    const int seg = __popc(hm & (0xffffffffu >> (31 - lane))) - 1, nseg = __popc(hm);
    for (int sidx = 0; sidx < nseg; ++sidx) {
      if (act && seg == sidx) {
#pragma unroll
        for (int x = 0; x < 6; ++x) my_gb[b * 6 + x] += g[x];
      }
      __syncwarp();
    }
  }
}
// Block work item -> (bra tile, ket chunk): largest t with cum[t] <= item.
__device__ __forceinline__ void find_work_item(const KParams& P, int item, int& tile, int& chunk) {
  int lo = 0, hi = P.ntiles;
  while (hi - lo > 1) { int mid = (lo + hi) >> 1; if (__ldg(P.cum + mid) <= item) lo = mid; else hi = mid; }
  tile = lo; chunk = item - __ldg(P.cum + lo);
}

#ifndef TDG_MINB
#define TDG_MINB 1
#endif
// One kernel per (class, role): role R handles the bra function pairs [R*ABN, (R+1)*ABN) of every surviving quartet (QC).  Each
// role is its own translation unit (they compile in parallel and get their own register allocation).
template <int LA, int LB, int LC, int LD, int ROLE>
__global__ void __launch_bounds__(TDG_NT, TDG_MINB) tdg_grad_kernel(const __grid_constant__ KParams P) {
  __shared__ PairHdr s_bra[TDG_WARP];
  __shared__ PairHdr s_ket[TDG_KB];
  __shared__ double s_dij[TDG_WARP];
  // dynamic shared memory: accumulators (per-warp bra slots, then the ket slots), then the Rys table of this class (QC::RYS_SH)
  extern __shared__ double2 s_dyn[];
  typedef QC<LA, LB, LC, LD> C;
  double* s_gb = reinterpret_cast<double*>(s_dyn);            // [warp][bra][centre A,B][xyz]
  double* s_gk = s_gb + TDG_WARPS * TDG_WARP * 6;             // [ket][centre C,D][xyz]; ket 32 w + o belongs to warp w
  double* s_ij = s_gb + TDG_ACC_DOUBLES;                      // [bra][ab][4]: M_J . pk(ij)  (QC::IJ_SH)
  double2* s_rys = s_dyn + (TDG_ACC_DOUBLES + C::IJ_SH_DOUBLES) / 2;
  int tile, chunk;
  find_work_item(P, blockIdx.x, tile, chunk);
  const int t = threadIdx.x, lane = t & 31;
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
  for (int i = t; i < TDG_ACC_DOUBLES; i += TDG_NT) s_gb[i] = 0.0;
  if constexpr (C::IJ_SH) {   // stage M_J . pk(ij)[a,b] of the tile's bras (offsets straight from the global headers: no extra barrier)
    for (int e = t; e < nb * C::NAB; e += TDG_NT) {
      const int b = e / C::NAB, ab = e - b * C::NAB;
      const PairHdr* gh = P.bra_hdr + bra0 + b;
      const d4 x = ld256(P.pk + 4 * ((size_t)gh->offA * P.nbf + (size_t)C::NA * gh->offB) + 4 * ab);
      double* dst = s_ij + 4 * e;
#pragma unroll
      for (int m = 0; m < 4; ++m) dst[m] = P.MJ[4 * m] * x.x + P.MJ[4 * m + 1] * x.y + P.MJ[4 * m + 2] * x.z + P.MJ[4 * m + 3] * x.w;
    }
  }
  const double* rys = P.rys_tab + rys_part_off(C::NR);
  if (C::RYS_SH) {
    const double2* src = reinterpret_cast<const double2*>(rys);
    for (int i = t; i < C::RYS_SRC_DOUBLES / 2; i += TDG_NT) s_rys[rys_sh_index<C::NR>(i)] = __ldg(src + i);
    rys = reinterpret_cast<const double*>(s_rys);
  }
  __syncthreads();
  // ---- phase 1 (step a4): one ket per thread, tested against the 32 bras; warp scan of the survivor counts ----
  unsigned long long n_vis = 0, n_cmp = 0;
  const unsigned mask = ket_ok ? screen_ket(P, s_bra, s_dij, nb, bra0, k, s_ket[t], dw, n_vis, n_cmp) : 0u;
  const int cnt = __popc(mask);
  int incl = cnt;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const int v = __shfl_up_sync(0xffffffffu, incl, o); if (lane >= o) incl += v; }
  const int tot = __shfl_sync(0xffffffffu, incl, 31);
  // ---- phase 2 (steps a5-a8): each warp processes the survivors of its own 32 kets densely, one quartet per thread per pass ----
  static_assert(ROLE >= 0 && ROLE < C::NROLE, "role out of range");
  constexpr int AB0 = ROLE * C::ABN;
  constexpr int ABC = (AB0 + C::ABN <= C::NAB) ? C::ABN : C::NAB - AB0;
  process_survivors<LA, LB, LC, LD, AB0, ABC>(P, s_bra, s_ket, mask, incl - cnt, tot, s_gb, s_gk, bra0, k0, rys, s_ij);
  __syncthreads();
  // flush: sum the warps' private bra slots, one FP64 RED per touched (pair, centre, xyz)
  for (int i = t; i < (TDG_WARP + TDG_KB) * 6; i += TDG_NT) {
    double v = 0.0;
    const PairHdr* h;
    int r;
    if (i < TDG_WARP * 6) {
#pragma unroll
      for (int w = 0; w < TDG_WARPS; ++w) v += s_gb[w * (TDG_WARP * 6) + i];
      h = s_bra + i / 6; r = i % 6;
    } else {
      const int ii = i - TDG_WARP * 6;
      v = s_gk[ii];
      h = s_ket + ii / 6; r = ii % 6;
    }
    if (v != 0.0) red_add(P.grad + 3 * (r < 3 ? h->atomA : h->atomB) + (r < 3 ? r : r - 3), v);
  }
  // stats
  for (int o = 16; o > 0; o >>= 1) {
    n_vis += __shfl_xor_sync(0xffffffffu, n_vis, o);
    n_cmp += __shfl_xor_sync(0xffffffffu, n_cmp, o);
  }
  if (ROLE == 0 && lane == 0 && n_vis) {
    atomicAdd(P.counters + 0, n_vis); atomicAdd(P.counters + 1, n_cmp);
    atomicAdd(P.counters + 2, n_cmp * (unsigned long long)(P.nppb * P.nppk));
  }
}

// Host-callable launcher of one (class, role), defined in a translation unit of its own (tdg_class.cu) and registered at
// load time; tdg_num_roles = QC::NROLE of the class (1 for the block-per-quartet kernel).
typedef void (*tdg_launch_fn)(const KParams& P, int nblocks, cudaStream_t s);
#define TDG_FOCK_ROLE_BASE 32   // launcher table: roles [0, 32) = gradient kernels, [32, 64) = Fock-build kernels of the same role
void tdg_register_launcher(int la, int lb, int lc, int ld, int role, tdg_launch_fn fn);
tdg_launch_fn tdg_get_launcher(int la, int lb, int lc, int ld, int role);
int tdg_num_roles(int la, int lb, int lc, int ld);
