// tdg_gradb.cuh — block-per-quartet ERI-derivative + density-contraction kernel for the high-l classes
// ((dd|dp), (dd|dd) and every class with an f shell; steps a4-a8).
//
// Why a second kernel: with one thread per quartet the 2-D Rys integrals of these classes (192 doubles per root and
// direction for (dd|dd), 500 for (ff|ff)) and the density products (1296 / 10000 per quartet) do not fit a thread's
// registers and go to local memory -- the reason the paper's own high-l kernels are memory-bound.
// Here a block of G threads (32..128) works on ONE quartet at a time:
//   * the 2-D integrals Ix, Iy, Iz of a batch of roots live in shared memory, built cooperatively: one thread per
//     (root, direction) runs the vertical recurrence, then all threads run the two transfer recurrences
//     column by column (SURVEY.md 9.1 formulas, same as build2d of tdg_grad.cuh);
//   * the function quartets are dealt over the threads; each thread forms its symmetrised density products from the six
//     density blocks staged (and pre-multiplied by the pair-weight matrices MJ, MK) in shared memory, applies the
//     centre derivative 2 zeta I(+1) - l I(-1) (eq 39/42) on A, B, C and accumulates 9 sums
//     in registers over all primitives, both operators and all roots;
//   * the 9 sums are reduced over the block and added to the same per-block shared accumulators as in tdg_grad.cuh
//     (fourth centre by eq 41), flushed with one FP64 RED per touched slot.
// Work items, screening (phase 1) and counters are those of tdg_grad.cuh, so the planner does not distinguish the two.
#pragma once
#include "tdg_grad.cuh"
#define TDG_GRADB_SLICES 16   // grid.y of the block-per-quartet kernel: slices of a work item's 128 kets

template <int LA, int LB, int LC, int LD>
struct QB {
  typedef QC<LA, LB, LC, LD> C;
  static constexpr int NA = C::NA, NB = C::NB, NC = C::NC, ND = C::ND, NCOMP = C::NCOMP, NR = C::NR;
  static constexpr int NMX = C::NMX, MMX = C::MMX, DA = C::DA, DB = C::DB, DC = C::DC, DD = C::DD;
  static constexpr int S = MMX + 1;                         // row stride of V[n][m] and of W[i][j][m]
  static constexpr int WSZ = DA * DB * S, ISZ = DA * DB * DC * DD;
  static constexpr int TASK = ISZ + WSZ;                    // doubles per (root, direction): I (V aliased inside) + W
  static constexpr int G = NCOMP >= 512 ? 128 : (NCOMP >= 128 ? 64 : 32);   // threads per quartet (= block size)
  static constexpr int RB0 = (36 * 1024) / (3 * TASK * 8);
  static constexpr int RB = RB0 < 1 ? 1 : (RB0 > 2 * NR ? 2 * NR : RB0);    // roots per batch (both operators form one list)
  static constexpr int sA = DB * DC * DD, sB = DC * DD, sC = DD;           // index strides of I[i][j][k][l]
  // density blocks staged as 4-vectors (one entry per canonical matrix): raw IK, JK, IJ; MK.JL, MK.IL, MJ.KL
  static constexpr int O_IK = 0, O_JK = O_IK + NA * NC, O_IJ = O_JK + NB * NC, O_JL = O_IJ + NA * NB, O_IL = O_JL + NB * ND,
                       O_KL = O_IL + NA * ND, NBLK = O_KL + NC * ND;
  // Fock mode (tdg_fock.cuh): raw blocks S[ls] (k,l), S[mn] (i,j), X[ln] (k,j), X[lm] (k,i), X[sn] (l,j), X[sm] (l,i)
  static constexpr int F_KL = 0, F_IJ = F_KL + NC * ND, F_KJ = F_IJ + NA * NB, F_KI = F_KJ + NC * NB, F_LJ = F_KI + NC * NA,
                       F_LI = F_LJ + ND * NB, F_NBLK = F_LI + ND * NA;
  static_assert(F_NBLK == NBLK, "both modes stage the same number of block elements");
  static constexpr int ACC = (TDG_WARP + TDG_KB) * 6;
  static constexpr int SMEM_DOUBLES = ACC + RB * 3 * TASK + NBLK * 4 + 2 * NR * 4 + 4 * 9 + TDG_WARP + TDG_KB / 2;
};

template <int L>
__device__ __forceinline__ void comp_exps_rt(int idx, int& x, int& y, int& z) {
  x = (int)((CartPack<L, 0>::v >> (4 * idx)) & 15); y = (int)((CartPack<L, 1>::v >> (4 * idx)) & 15); z = (int)((CartPack<L, 2>::v >> (4 * idx)) & 15);
}

// MODE 0: gradient (steps a5-a8).  MODE 1: Fock-type build (NEXT-1; conventions of tdg_fock.cuh): the same 2-D integrals (read
// without the raised entries; the gradient's root count is exact for the lower degree too), each thread sums its function
// quartets' integrals over the roots of a batch and digests them into G[slot][row][col] with FP64 RED.
template <int LA, int LB, int LC, int LD, int MODE>
__global__ void __launch_bounds__(QB<LA, LB, LC, LD>::G) tdg_gradb_kernel(const __grid_constant__ KParams P) {
  typedef QB<LA, LB, LC, LD> B;
  constexpr int G = B::G, NR = B::NR, S = B::S, TASK = B::TASK;
  extern __shared__ double2 s_dyn[];
  double* s_acc = reinterpret_cast<double*>(s_dyn);      // [bra 32][6] then [ket 128][6]
  double* s_task = s_acc + B::ACC;                       // [RB][3][TASK]
  double* s_blk = s_task + B::RB * 3 * TASK;             // [NBLK][4]
  double* s_root = s_blk + B::NBLK * 4;                  // [2 NR][x, w*pref, alpha (J weight), beta (K weight)]
  double* s_red = s_root + 2 * NR * 4;                   // [4 warps][9]
  double* s_dij = s_red + 4 * 9;                         // [32]
  unsigned* s_mask = reinterpret_cast<unsigned*>(s_dij + TDG_WARP);   // [128]
  int tile, chunk;
  find_work_item(P, blockIdx.x, tile, chunk);
  const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
  const int bra0 = tile * TDG_WARP, k0 = chunk * TDG_KB;
  const int nb = min(TDG_WARP, P.nbra - bra0);
  const bool dw = P.tau > 0.0 && P.density_weighted;
  for (int i = t; i < B::ACC; i += G) s_acc[i] = 0.0;
  for (int i = t; i < nb; i += G) {
    const PairHdr& h = P.bra_hdr[bra0 + i];
    s_dij[i] = dw ? __ldg(P.dmax + (size_t)h.ish * P.nshell + h.jsh) : 0.0;
  }
  __syncthreads();
  // ---- phase 1 (step a4): the block's threads share the 128 kets of the chunk ----
  unsigned long long n_vis = 0, n_cmp = 0;
  // The classes of this kernel have few shell pairs, hence few work items (cfg 3 (dd|dd): 36): a work item is therefore cut into
  // gridDim.y slices, slice y taking the kets y, y + gridDim.y, ... of the chunk (screening and counters included), so that the launch
  // fills the GPU (ncu round 2: 4 warps per SM active with one block per work item).
  for (int kt = blockIdx.y + gridDim.y * t; kt < TDG_KB; kt += gridDim.y * G) {
    const int k = k0 + kt;
    s_mask[kt] = k < P.nket ? screen_ket(P, P.bra_hdr + bra0, s_dij, nb, bra0, k, P.ket_hdr[k], dw, n_vis, n_cmp) : 0u;
  }
  __syncthreads();
  const double* rys = P.rys_tab + rys_part_off(NR);
  const size_t n = (size_t)P.nbf;
  const double* __restrict__ pk = P.pk;
  // ---- phase 2: survivors one after another, the whole block on each ----
  for (int kt = blockIdx.y; kt < TDG_KB; kt += gridDim.y) {
    unsigned m = s_mask[kt];
    if (!m) continue;
    const PairHdr kh = P.ket_hdr[k0 + kt];
    const double* kprim = P.ket_prim + (size_t)(k0 + kt) * P.nppk * TDG_PRIM_STRIDE;
    while (m) {
      const int b = __ffs(m) - 1;
      m &= m - 1;
      const PairHdr bh = P.bra_hdr[bra0 + b];
      const double* bprim = P.bra_prim + (size_t)(bra0 + b) * P.nppb * TDG_PRIM_STRIDE;
      double deg = 1.0;
      if (bh.ish == bh.jsh) deg *= 0.5;
      if (kh.ish == kh.jsh) deg *= 0.5;
      if (P.same_bucket && k0 + kt == bra0 + b) deg *= 0.5;
      // stage the six density blocks (step a7, part 1): raw IK, JK, IJ and MK.JL, MK.IL, MJ.KL (4-vectors over the canonical matrices)
      if (MODE == 0) {
        const double* bIK = pk + 4 * ((size_t)bh.offA * n + (size_t)B::NA * kh.offA);
        const double* bJL = pk + 4 * ((size_t)bh.offB * n + (size_t)B::NB * kh.offB);
        const double* bJK = pk + 4 * ((size_t)bh.offB * n + (size_t)B::NB * kh.offA);
        const double* bIL = pk + 4 * ((size_t)bh.offA * n + (size_t)B::NA * kh.offB);
        const double* bIJ = pk + 4 * ((size_t)bh.offA * n + (size_t)B::NA * bh.offB);
        const double* bKL = pk + 4 * ((size_t)kh.offA * n + (size_t)B::NC * kh.offB);
        for (int e = t; e < B::NBLK; e += G) {
          const double* src; const double* M = nullptr;
          if (e < B::O_JK) src = bIK + 4 * e;
          else if (e < B::O_IJ) src = bJK + 4 * (e - B::O_JK);
          else if (e < B::O_JL) src = bIJ + 4 * (e - B::O_IJ);
          else if (e < B::O_IL) { src = bJL + 4 * (e - B::O_JL); M = P.MK; }
          else if (e < B::O_KL) { src = bIL + 4 * (e - B::O_IL); M = P.MK; }
          else { src = bKL + 4 * (e - B::O_KL); M = P.MJ; }
          const d4 x = ld256(src);
          double* dst = s_blk + 4 * e;
          if (M) {
#pragma unroll
            for (int q = 0; q < 4; ++q) dst[q] = M[4 * q] * x.x + M[4 * q + 1] * x.y + M[4 * q + 2] * x.z + M[4 * q + 3] * x.w;
          } else { dst[0] = x.x; dst[1] = x.y; dst[2] = x.z; dst[3] = x.w; }
        }
      } else {   // Fock mode: raw blocks in the orientation the digestion reads
        const double* src0[6] = {pk + 4 * ((size_t)kh.offA * n + (size_t)B::NC * kh.offB), pk + 4 * ((size_t)bh.offA * n + (size_t)B::NA * bh.offB),
                                 pk + 4 * ((size_t)kh.offA * n + (size_t)B::NC * bh.offB), pk + 4 * ((size_t)kh.offA * n + (size_t)B::NC * bh.offA),
                                 pk + 4 * ((size_t)kh.offB * n + (size_t)B::ND * bh.offB), pk + 4 * ((size_t)kh.offB * n + (size_t)B::ND * bh.offA)};
        constexpr int off[7] = {B::F_KL, B::F_IJ, B::F_KJ, B::F_KI, B::F_LJ, B::F_LI, B::F_NBLK};
        for (int e = t; e < B::F_NBLK; e += G) {
          int q = 0;
#pragma unroll
          for (int z = 1; z < 6; ++z) if (e >= off[z]) q = z;
          const d4 x = ld256(src0[q] + 4 * (e - off[q]));
          double* dst = s_blk + 4 * e;
          dst[0] = x.x; dst[1] = x.y; dst[2] = x.z; dst[3] = x.w;
        }
      }
      double g[9];
#pragma unroll
      for (int x = 0; x < 9; ++x) g[x] = 0.0;
      for (int ib = 0; ib < P.nppb; ++ib) {
        const double* bp = bprim + ib * TDG_PRIM_STRIDE;
        const double p = bp[0], Kab = 34.986836655249725693 /* 2 pi^(5/2) */ * bp[4], a2 = 2.0 * bp[5], b2 = 2.0 * bp[6], rp = bp[7];
        for (int ik = 0; ik < P.nppk; ++ik) {
          const double* kp = kprim + ik * TDG_PRIM_STRIDE;
          const double q = kp[0], c2 = 2.0 * kp[5], rq = kp[7];
          const double rs = rsqrt(p + q), rpq = rs * rs, rho = p * q * rpq;
          const double PQx = bp[1] - kp[1], PQy = bp[2] - kp[2], PQz = bp[3] - kp[3];
          const double T = rho * (PQx * PQx + PQy * PQy + PQz * PQz);
          const double pref = Kab * kp[4] * rs;
          __syncthreads();   // previous users of s_root / s_task / s_blk (first pass: staging above) are done
          // roots and weights of both operators (step a5; S8): warp 0 lane 0 -> 1/r, lane 1 -> erf(omega r)/r
          if (t <= P.use_lr) {
            double s2 = 1.0, ss = 1.0;
            if (t == 1) { ss = P.omega * rsqrt(P.omega2 + rho); s2 = ss * ss; }
            double xr[NR], wr[NR];
            rys_eval<NR>(rys, s2 * T, xr, wr);
#pragma unroll
            for (int r = 0; r < NR; ++r) {
              double* e = s_root + (t * NR + r) * 4;
              e[0] = xr[r] * s2; e[1] = wr[r] * ss * pref; e[2] = t == 0 ? 1.0 : 0.0; e[3] = t == 0 ? P.cK : P.cLR;
            }
          }
          __syncthreads();
          const int nroot = (1 + P.use_lr) * NR;
          for (int r0 = 0; r0 < nroot; r0 += B::RB) {
            const int nrb = min(B::RB, nroot - r0);
            const int ntask = nrb * 3;
            // (1) vertical recurrence, one thread per (root, direction)
            for (int tk = t; tk < ntask; tk += G) {
              const int r = tk / 3, dir = tk - 3 * r;
              const double x = s_root[(r0 + r) * 4], w = s_root[(r0 + r) * 4 + 1];
              const double b00 = 0.5 * x * rpq, b10 = (0.5 - q * b00) * rp, b01 = (0.5 - p * b00) * rq;
              const double PQd = bp[1 + dir] - kp[1 + dir];
              const double c00 = (bp[1 + dir] - bh.A[dir]) - q * rpq * x * PQd, c00p = (kp[1 + dir] - kh.A[dir]) + p * rpq * x * PQd;
              double* V = s_task + tk * TASK;       // V[n][m] at n*S + m, inside the I region
              V[0] = dir == 2 ? w : 1.0;
#pragma unroll 1
              for (int nn = 0; nn < B::NMX; ++nn) V[(nn + 1) * S] = c00 * V[nn * S] + (nn > 0 ? nn * b10 * V[(nn - 1) * S] : 0.0);
#pragma unroll 1
              for (int mm = 0; mm < B::MMX; ++mm)
#pragma unroll 1
                for (int nn = 0; nn <= B::NMX; ++nn) {
                  double v = c00p * V[nn * S + mm];
                  if (mm > 0) v += mm * b01 * V[nn * S + mm - 1];
                  if (nn > 0) v += nn * b00 * V[(nn - 1) * S + mm];
                  V[nn * S + mm + 1] = v;
                }
            }
            __syncthreads();
            // (2) bra transfer i -> j, one column m of one task per thread: W[i][j][m] at (i*DB + j)*S + m
            for (int it = t; it < ntask * S; it += G) {
              const int tk = it / S, mm = it - tk * S, dir = tk % 3;
              const double ab = bh.AB[dir];
              double* h = s_task + tk * TASK + mm;
              double* W = s_task + tk * TASK + B::ISZ + mm;
#pragma unroll 1
              for (int j = 0; j <= LB + 1; ++j) {
                const int imax = min(LA + 1, B::NMX - j);
                for (int i = 0; i <= imax; ++i) W[(i * B::DB + j) * S] = h[i * S];
                for (int i = 0; i + j < B::NMX; ++i) h[i * S] = h[(i + 1) * S] + ab * h[i * S];
              }
            }
            __syncthreads();
            // (3) ket transfer k -> l, one (i, j) of one task per thread: I[i][j][k][l] at ((i*DB + j)*DC + k)*DD + l
            for (int it = t; it < ntask * B::DA * B::DB; it += G) {
              const int tk = it / (B::DA * B::DB), ij = it - tk * (B::DA * B::DB), dir = tk % 3;
              const int i = ij / B::DB, j = ij - i * B::DB;
              if (i + j > B::NMX) continue;
              const double cd = kh.AB[dir];
              double* gk = s_task + tk * TASK + B::ISZ + ij * S;
              double* I = s_task + tk * TASK + ij * (B::DC * B::DD);
#pragma unroll 1
              for (int l = 0; l <= LD; ++l) {
                const int kmax = min(LC + 1, B::MMX - l);
                for (int k = 0; k <= kmax; ++k) I[k * B::DD + l] = gk[k];
                for (int k = 0; k + l < B::MMX; ++k) gk[k] = gk[k + 1] + cd * gk[k];
              }
            }
            __syncthreads();
            if constexpr (MODE == 1) {
              // (4F) this thread's function quartets: integral summed over the batch's roots, digested at once
              const size_t n2 = n * n;
              double* __restrict__ Gm = P.grad;
#pragma unroll 1
              for (int fn = t; fn < B::NCOMP; fn += G) {
                const int d = fn % B::ND, c = (fn / B::ND) % B::NC, bb = (fn / (B::ND * B::NC)) % B::NB, a = fn / (B::ND * B::NC * B::NB);
                int ax, ay, az, bx, by, bz, cx, cy, cz, dx, dy, dz;
                comp_exps_rt<LA>(a, ax, ay, az); comp_exps_rt<LB>(bb, bx, by, bz); comp_exps_rt<LC>(c, cx, cy, cz); comp_exps_rt<LD>(d, dx, dy, dz);
                const int ix = ((ax * B::DB + bx) * B::DC + cx) * B::DD + dx;
                const int iy = ((ay * B::DB + by) * B::DC + cy) * B::DD + dy + TASK;
                const int iz = ((az * B::DB + bz) * B::DC + cz) * B::DD + dz + 2 * TASK;
                double vJ = 0.0, vK = 0.0;
#pragma unroll 1
                for (int r = 0; r < nrb; ++r) {
                  const double* e = s_root + (r0 + r) * 4;
                  const double* I = s_task + r * 3 * TASK;
                  const double v = I[ix] * I[iy] * I[iz];
                  vJ = fma(e[2], v, vJ); vK = fma(e[3], v, vK);
                }
                const double cn = deg * c_cnorm[LA][a] * c_cnorm[LB][bb] * c_cnorm[LC][c] * c_cnorm[LD][d];
                vJ *= cn; vK *= cn;
                const int mu = bh.offA + a, nu = bh.offB + bb, la_ = kh.offA + c, si = kh.offB + d;
                const double* sKL = s_blk + 4 * (B::F_KL + c * B::ND + d);
                const double* sIJ = s_blk + 4 * (B::F_IJ + a * B::NB + bb);
                const double* xKJ = s_blk + 4 * (B::F_KJ + c * B::NB + bb);
                const double* xKI = s_blk + 4 * (B::F_KI + c * B::NA + a);
                const double* xLJ = s_blk + 4 * (B::F_LJ + d * B::NB + bb);
                const double* xLI = s_blk + 4 * (B::F_LI + d * B::NA + a);
#pragma unroll
                for (int sl = 0; sl < 4; ++sl) {
                  double* Gs = Gm + (size_t)sl * n2;
                  const double jw = P.MJ[sl], kw = P.MK[sl];
                  if (jw != 0.0) {
                    red_add(Gs + (size_t)mu * n + nu, jw * sKL[sl] * vJ);
                    red_add(Gs + (size_t)la_ * n + si, jw * sIJ[sl] * vJ);
                  }
                  if (kw != 0.0) {
                    red_add(Gs + (size_t)mu * n + si, -kw * xKJ[sl] * vK);
                    red_add(Gs + (size_t)nu * n + si, -kw * xKI[sl] * vK);
                    red_add(Gs + (size_t)mu * n + la_, -kw * xLJ[sl] * vK);
                    red_add(Gs + (size_t)nu * n + la_, -kw * xLI[sl] * vK);
                  }
                }
              }
            } else {
            // (4) function quartets over the threads (step a7): density products, centre derivatives, 9 sums
#pragma unroll 1
            for (int fn = t; fn < B::NCOMP; fn += G) {
              const int d = fn % B::ND, c = (fn / B::ND) % B::NC, bb = (fn / (B::ND * B::NC)) % B::NB, a = fn / (B::ND * B::NC * B::NB);
              const double* u = s_blk + 4 * (B::O_IK + a * B::NC + c);
              const double* sv = s_blk + 4 * (B::O_JK + bb * B::NC + c);
              const double* jv = s_blk + 4 * (B::O_IJ + a * B::NB + bb);
              const double* v = s_blk + 4 * (B::O_JL + bb * B::ND + d);
              const double* tt = s_blk + 4 * (B::O_IL + a * B::ND + d);
              const double* wv = s_blk + 4 * (B::O_KL + c * B::ND + d);
              const double cn = deg * c_cnorm[LA][a] * c_cnorm[LB][bb] * c_cnorm[LC][c] * c_cnorm[LD][d];
              const double gkk = cn * (u[0] * v[0] + u[1] * v[1] + u[2] * v[2] + u[3] * v[3] + sv[0] * tt[0] + sv[1] * tt[1] + sv[2] * tt[2] + sv[3] * tt[3]);
              const double gjj = cn * (jv[0] * wv[0] + jv[1] * wv[1] + jv[2] * wv[2] + jv[3] * wv[3]);
              int ax, ay, az, bx, by, bz, cx, cy, cz, dx, dy, dz;
              comp_exps_rt<LA>(a, ax, ay, az); comp_exps_rt<LB>(bb, bx, by, bz); comp_exps_rt<LC>(c, cx, cy, cz); comp_exps_rt<LD>(d, dx, dy, dz);
              const int ix = ((ax * B::DB + bx) * B::DC + cx) * B::DD + dx;
              const int iy = ((ay * B::DB + by) * B::DC + cy) * B::DD + dy + TASK;
              const int iz = ((az * B::DB + bz) * B::DC + cz) * B::DD + dz + 2 * TASK;
#pragma unroll 1
              for (int r = 0; r < nrb; ++r) {
                const double* e = s_root + (r0 + r) * 4;
                const double Gr = gjj * e[2] + gkk * e[3];
                const double* I = s_task + r * 3 * TASK;
                const double X0 = I[ix], Y0 = I[iy], Z0 = I[iz];
                const double gx = Gr * X0, gy = Gr * Y0;
                const double tx = gy * Z0, ty = gx * Z0, tz = gx * Y0;
                double dAx = a2 * I[ix + B::sA], dAy = a2 * I[iy + B::sA], dAz = a2 * I[iz + B::sA];
                if (ax > 0) dAx -= ax * I[ix - B::sA];
                if (ay > 0) dAy -= ay * I[iy - B::sA];
                if (az > 0) dAz -= az * I[iz - B::sA];
                double dBx = b2 * I[ix + B::sB], dBy = b2 * I[iy + B::sB], dBz = b2 * I[iz + B::sB];
                if (bx > 0) dBx -= bx * I[ix - B::sB];
                if (by > 0) dBy -= by * I[iy - B::sB];
                if (bz > 0) dBz -= bz * I[iz - B::sB];
                double dCx = c2 * I[ix + B::sC], dCy = c2 * I[iy + B::sC], dCz = c2 * I[iz + B::sC];
                if (cx > 0) dCx -= cx * I[ix - B::sC];
                if (cy > 0) dCy -= cy * I[iy - B::sC];
                if (cz > 0) dCz -= cz * I[iz - B::sC];
                g[0] += tx * dAx; g[1] += ty * dAy; g[2] += tz * dAz;
                g[3] += tx * dBx; g[4] += ty * dBy; g[5] += tz * dBz;
                g[6] += tx * dCx; g[7] += ty * dCy; g[8] += tz * dCz;
              }
            }
            }
            if (r0 + B::RB < nroot) __syncthreads();   // the next batch overwrites s_task
          }
        }
      }
      if constexpr (MODE == 0) {
      // block reduction of the 9 sums; thread 0 adds them to the accumulators (one quartet at a time: no races)
#pragma unroll
      for (int x = 0; x < 9; ++x) g[x] = warp_sum(g[x]);
      if (G > 32) {
        if (lane == 0) {
#pragma unroll
          for (int x = 0; x < 9; ++x) s_red[warp * 9 + x] = g[x];
        }
        __syncthreads();
        if (t == 0) {
#pragma unroll
          for (int x = 0; x < 9; ++x) { g[x] = 0.0; for (int w = 0; w < G / 32; ++w) g[x] += s_red[w * 9 + x]; }
        }
      }
      if (t == 0) {
        double* gb = s_acc + b * 6;
        double* gkp = s_acc + (TDG_WARP + kt) * 6;
#pragma unroll
        for (int x = 0; x < 3; ++x) {
          gb[x] += g[x]; gb[3 + x] += g[3 + x];
          gkp[x] += g[6 + x]; gkp[3 + x] -= g[x] + g[3 + x] + g[6 + x];
        }
      }
      } else {
        __syncthreads();   // the next quartet restages s_blk / s_task
      }
    }
  }
  __syncthreads();
  for (int i = t; MODE == 0 && i < B::ACC; i += G) {
    const double v = s_acc[i];
    if (v == 0.0) continue;
    const int r = i % 6;
    const PairHdr& h = i < TDG_WARP * 6 ? P.bra_hdr[bra0 + i / 6] : P.ket_hdr[k0 + (i - TDG_WARP * 6) / 6];
    red_add(P.grad + 3 * (r < 3 ? h.atomA : h.atomB) + (r < 3 ? r : r - 3), v);
  }
  for (int o = 16; o > 0; o >>= 1) {
    n_vis += __shfl_xor_sync(0xffffffffu, n_vis, o);
    n_cmp += __shfl_xor_sync(0xffffffffu, n_cmp, o);
  }
  if (lane == 0 && n_vis) {
    atomicAdd(P.counters + 0, n_vis); atomicAdd(P.counters + 1, n_cmp);
    atomicAdd(P.counters + 2, n_cmp * (unsigned long long)(P.nppb * P.nppk));
  }
}
