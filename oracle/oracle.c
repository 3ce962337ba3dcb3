/*
 * oracle.c — CPU ORACLE for the ERI-derivative gradient path.  TEST INFRASTRUCTURE ONLY.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call this file.  The product (paper_2407_16586_b200/csrc, libtdgrad.so) shares
 * no code, table, header or constant with it and never calls it.
 *
 * What it computes (plain definition, FP64, every centre differentiated explicitly, no
 * translational-invariance shortcut):
 *
 *   E(R) = sum_k [ wJ_k cJ J(A_k,B_k) - wK_k ( cK K(A_k,B_k) + cLR K_w(A_k,B_k) ) ]
 *   J(A,B)   = sum A_mn B_ls (mn|ls)            K(A,B) = sum A_ml B_ns (mn|ls)
 *   g_{E,x}  = dE/dR_{E,x} with the matrices held fixed
 *
 * i.e. terms 4 and 5 of PAPER.md:84-89 (eq 7) with the density products of PAPER.md:110-114
 * (eqs 13-14), the centre derivative of PAPER.md:243-253 (eqs 39-40) and the update of
 * PAPER.md:261-268 (eq 42), contracted shells of PAPER.md:268-273 (eq 43).  (mn|ls) uses 1/r
 * (eqs 3-4), K_w uses erf(w r)/r (eq 5).
 *
 * Integral algorithm: McMurchie-Davidson (Hermite Gaussians + Boys function), textbook, chosen
 * because the CUDA path uses Rys quadrature: the two share neither roots nor recurrences.
 * Steps O1..O10 are those of SURVEY.md section 8(c) / DESIGN.md "Oracle"; readings S1..S19 of the
 * paper are listed in DESIGN.md.
 *
 * Pins (tests/test_oracle_*.py, all independent of this file's arithmetic): Boys vs mpmath
 * quadrature and the incomplete gamma function; (ss|ss) closed form, both operators; p/d/f
 * integrals vs high-precision differentiation of the (ss|ss) closed form; unit self-overlap;
 * omega->infinity and omega->0 limits; derivative integrals vs finite differences; gradient vs
 * central finite differences of orc_energy; sum_A g_A = 0; N^4 loop vs unique-quartet loop;
 * K(T,T) vs explicit MO sum; energy vs numpy einsum over orc_eri_tensor; the density-weighted
 * screening rule (density_maxima, quartet_weight) vs the Cauchy-Schwarz inequality on every
 * density-weighted integral, the closed form for s shells, permutation/transpose invariance and
 * the c * n_dropped * tau error bound (tests/test_oracle_screening.py).  One-electron terms (orc_onee_*, end of
 * file): closed forms, finite differences of the pinned overlap, tight-charge limit of the pinned ERIs, mpmath
 * derivatives of the s-s closed forms, finite differences of the energy (tests/test_oracle_onee.py).
 * Paper-printed values: none exist for this path ("parity unpinned" w.r.t. printed numbers).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define LMAX 3               /* highest shell angular momentum */
#define LR (LMAX + 1)        /* raised */
#define NHERM1 (2 * LR + 1)  /* Hermite index range of one pair, one direction: t <= 2(LMAX+1) */
#define NTOT (4 * LMAX + 2)  /* t+u+v <= 4*LMAX+1 */
#define MAXM 32
#define NCMAX 10             /* ncart(3) */

static const double PI = 3.14159265358979323846264338327950288;

static int ncart(int l) { return (l + 1) * (l + 2) / 2; }

/* Cartesian component order (reading S7): lx descending, then ly descending. */
static void cart_comp(int l, int idx, int *lx, int *ly, int *lz) {
    int c = 0;
    for (int x = l; x >= 0; --x)
        for (int y = l - x; y >= 0; --y) {
            if (c == idx) { *lx = x; *ly = y; *lz = l - x - y; return; }
            ++c;
        }
    *lx = *ly = *lz = 0;
}

static double dfact(int n) { /* n!!, (-1)!! = 1 */
    double r = 1.0;
    for (; n > 1; n -= 2) r *= n;
    return r;
}

/* ---------------------------------------------------------------- O2: Boys function
 * F_m(T) = int_0^1 t^{2m} exp(-T t^2) dt.  T <= 30: series at mmax then downward recursion;
 * T > 30: F_0 from erf, upward recursion.  (PAPER.md:291 needs its moments via the Rys weight;
 * here used directly.) */
void orc_boys(int mmax, double T, double *F) {
    if (T <= 30.0) {
        /* upward recursion is unstable for T < m; series at the top, go down */
        double eT = exp(-T);
        double term = 1.0 / (2.0 * mmax + 1.0), sum = term;
        for (int k = 1; k < 400; ++k) {
            term *= 2.0 * T / (2.0 * mmax + 2.0 * k + 1.0);
            sum += term;
            if (term < 1e-17 * sum) break;
        }
        F[mmax] = eT * sum;
        for (int m = mmax; m > 0; --m) F[m - 1] = (2.0 * T * F[m] + eT) / (2.0 * m - 1.0);
    } else {
        double eT = exp(-T);
        F[0] = 0.5 * sqrt(PI / T) * erf(sqrt(T));
        for (int m = 0; m < mmax; ++m) F[m + 1] = ((2.0 * m + 1.0) * F[m] - eT) / (2.0 * T);
    }
}

/* O3: operator-specific Boys vector.  omega <= 0: full 1/r, G_n = F_n(T).
 * omega > 0: erf(omega r)/r, s^2 = omega^2/(omega^2+rho), G_n = s^{2n+1} F_n(s^2 T)
 * (eq 5; formula = reading S8). */
void orc_boys_op(int mmax, double T, double rho, double omega, double *G) {
    if (omega <= 0.0) { orc_boys(mmax, T, G); return; }
    double s2 = omega * omega / (omega * omega + rho);
    double s = sqrt(s2);
    orc_boys(mmax, s2 * T, G);
    double f = s;
    for (int n = 0; n <= mmax; ++n) { G[n] *= f; f *= s2; }
}

/* ---------------------------------------------------------------- system + O1 normalisation */
typedef struct {
    int natom, nshell, nbf;
    const double *xyz;
    const int32_t *shells; /* [nshell][4] atom,l,nprim,prim_off */
    const double *exps;
    double *cn;    /* normalised primitive coefficient of the (l,0,0)-type radial part, see below */
    int *off;      /* first function of shell */
} sys_t;

/* O1 (eq 38 "N"; eq 43).  Input d_k multiply normalised primitives.
 * N_prim(z;lx,ly,lz) = (2z/pi)^{3/4} (4z)^{l/2} / sqrt((2lx-1)!!(2ly-1)!!(2lz-1)!!).
 * Shell self-overlap S = sum_kk' d_k d_k' (2 sqrt(z z')/(z+z'))^{l+3/2}; phi = S^{-1/2} sum d_k N_prim x^lx.. e^{-z r^2}.
 * cn[k] holds d_k S^{-1/2} (2z/pi)^{3/4} (4z)^{l/2}; the component factor is applied separately. */
static double comp_norm(int lx, int ly, int lz) {
    return 1.0 / sqrt(dfact(2 * lx - 1) * dfact(2 * ly - 1) * dfact(2 * lz - 1));
}

static int sys_init(sys_t *s, int natom, const double *xyz, int nshell, const int32_t *shells,
                    int nprim_total, const double *exps, const double *coefs) {
    s->natom = natom; s->nshell = nshell; s->xyz = xyz; s->shells = shells; s->exps = exps;
    s->cn = (double *)malloc(sizeof(double) * (size_t)nprim_total);
    s->off = (int *)malloc(sizeof(int) * (size_t)(nshell + 1));
    if (!s->cn || !s->off) return -1;
    int nbf = 0;
    for (int i = 0; i < nshell; ++i) {
        int l = shells[4 * i + 1], np = shells[4 * i + 2], po = shells[4 * i + 3];
        if (l < 0 || l > LMAX || np <= 0 || shells[4 * i] < 0 || shells[4 * i] >= natom) return -2;
        s->off[i] = nbf; nbf += ncart(l);
        double S = 0.0;
        for (int k = 0; k < np; ++k)
            for (int k2 = 0; k2 < np; ++k2) {
                double a = exps[po + k], b = exps[po + k2];
                S += coefs[po + k] * coefs[po + k2] * pow(2.0 * sqrt(a * b) / (a + b), l + 1.5);
            }
        for (int k = 0; k < np; ++k) {
            double z = exps[po + k];
            s->cn[po + k] = coefs[po + k] / sqrt(S) * pow(2.0 * z / PI, 0.75) * pow(4.0 * z, 0.5 * l);
        }
    }
    s->off[nshell] = nbf; s->nbf = nbf;
    return 0;
}
static void sys_free(sys_t *s) { free(s->cn); free(s->off); }

int orc_nbf(int nshell, const int32_t *shells) {
    int n = 0;
    for (int i = 0; i < nshell; ++i) n += ncart(shells[4 * i + 1]);
    return n;
}

/* ---------------------------------------------------------------- O4: Hermite expansion, one direction
 * E[i][j][t], i<=imax, j<=jmax.  mu = ab/p, X = A_x - B_x.
 * E_0^{00} = exp(-mu X^2);
 * E_t^{i+1,j} = E_{t-1}^{ij}/(2p) - (b/p) X E_t^{ij} + (t+1) E_{t+1}^{ij}
 * E_t^{i,j+1} = E_{t-1}^{ij}/(2p) + (a/p) X E_t^{ij} + (t+1) E_{t+1}^{ij} */
typedef double herm_t[LR + 1][LR + 1][NHERM1 + 1];

static void hermite_E(int imax, int jmax, double a, double b, double X, herm_t E) {
    double p = a + b, mu = a * b / p;
    for (int i = 0; i <= imax; ++i)      /* entries with t > i+j are zero; only the used range is cleared */
        for (int j = 0; j <= jmax; ++j)
            for (int t = 0; t <= i + j + 2 && t <= NHERM1; ++t) E[i][j][t] = 0.0;
    E[0][0][0] = exp(-mu * X * X);
    for (int j = 0; j <= jmax; ++j) {
        if (j > 0) { /* raise j from (0, j-1) */
            for (int t = 0; t <= j; ++t) {
                double v = (a / p) * X * E[0][j - 1][t] + (t + 1) * E[0][j - 1][t + 1];
                if (t > 0) v += E[0][j - 1][t - 1] / (2.0 * p);
                E[0][j][t] = v;
            }
        }
        for (int i = 1; i <= imax; ++i)
            for (int t = 0; t <= i + j; ++t) {
                double v = -(b / p) * X * E[i - 1][j][t] + (t + 1) * E[i - 1][j][t + 1];
                if (t > 0) v += E[i - 1][j][t - 1] / (2.0 * p);
                E[i][j][t] = v;
            }
    }
}

/* ---------------------------------------------------------------- O5: Hermite Coulomb integrals
 * R^n_000 = (-2 rho)^n G_n;  R^n_{t+1,u,v} = t R^{n+1}_{t-1,u,v} + X R^{n+1}_{t,u,v} (same for u,v).
 * Output R0[t][u][v] = R^0_{tuv} for t+u+v <= N. */
typedef double rtab_t[NTOT + 1][NTOT + 1][NTOT + 1];

static void hermite_R(int N, double rho, const double *G, double X, double Y, double Z, rtab_t R0, double *work) {
    /* work: (N+1) tables of (N+1)^3 */
    size_t n1 = (size_t)(N + 1);
#define RW(n, t, u, v) work[(((size_t)(n) * n1 + (t)) * n1 + (u)) * n1 + (v)]
    double f = 1.0;
    for (int n = 0; n <= N; ++n) { RW(n, 0, 0, 0) = f * G[n]; f *= -2.0 * rho; }
    for (int s = 1; s <= N; ++s)            /* total order t+u+v = s */
        for (int n = 0; n <= N - s; ++n)
            for (int t = 0; t <= s; ++t)
                for (int u = 0; u <= s - t; ++u) {
                    int v = s - t - u;
                    double val;
                    if (t > 0) {
                        val = X * RW(n + 1, t - 1, u, v);
                        if (t > 1) val += (t - 1) * RW(n + 1, t - 2, u, v);
                    } else if (u > 0) {
                        val = Y * RW(n + 1, t, u - 1, v);
                        if (u > 1) val += (u - 1) * RW(n + 1, t, u - 2, v);
                    } else {
                        val = Z * RW(n + 1, t, u, v - 1);
                        if (v > 1) val += (v - 1) * RW(n + 1, t, u, v - 2);
                    }
                    RW(n, t, u, v) = val;
                }
    for (int t = 0; t <= N; ++t)
        for (int u = 0; u <= N - t; ++u)
            for (int v = 0; v <= N - t - u; ++v) R0[t][u][v] = RW(0, t, u, v);
#undef RW
}

/* ---------------------------------------------------------------- O6 + O7: contracted shell quartet
 * [ab|cd] = 2 pi^{5/2}/(p q sqrt(p+q)) sum_{tuv} E_t E_u E_v sum_{t'u'v'} (-1)^{t'+u'+v'} E'_t' E'_u' E'_v' R_{t+t',u+u',v+v'}
 * d/dA_x [ab|cd] = 2a [a+1_x b|cd] - a_x [a-1_x b|cd]   (eq 39 with the nuclear-coordinate
 * sign, eq 42); likewise B, C, D and y, z.  All 12 are evaluated; eq 41 is NOT used. */
typedef struct {
    double *rwork;                 /* (NTOT+1)^4 */
    rtab_t R;
    herm_t Eb[3], Ek[3];
    double K[7][2 * LR][2 * LR][2 * LR]; /* ket-contracted Hermite integrals per ket variant */
    double *val, *der;             /* [nfun], [12][nfun]  (full or lr, caller decides) */
    double *val2, *der2;           /* second operator */
} work_t;

static work_t *work_new(void) {
    work_t *w = (work_t *)malloc(sizeof(work_t));
    if (!w) return NULL;
    size_t nf = (size_t)NCMAX * NCMAX * NCMAX * NCMAX;
    w->rwork = (double *)malloc(sizeof(double) * (size_t)(NTOT + 1) * (NTOT + 1) * (NTOT + 1) * (NTOT + 1));
    w->val = (double *)malloc(sizeof(double) * nf);
    w->der = (double *)malloc(sizeof(double) * nf * 12);
    w->val2 = (double *)malloc(sizeof(double) * nf);
    w->der2 = (double *)malloc(sizeof(double) * nf * 12);
    return w;
}
static void work_free(work_t *w) {
    if (!w) return;
    free(w->rwork); free(w->val); free(w->der); free(w->val2); free(w->der2); free(w);
}

/* 1-D Hermite vector of a function pair in one direction, variant 0 plain,
 * 1: derivative w.r.t. first centre, 2: w.r.t. second centre. n = number of entries written. */
static int herm_vec(herm_t E, int i, int j, double a, double b, int variant, double *out) {
    if (variant == 0) {
        for (int t = 0; t <= i + j; ++t) out[t] = E[i][j][t];
        return i + j + 1;
    }
    if (variant == 1) {
        for (int t = 0; t <= i + j + 1; ++t) {
            double v = 2.0 * a * E[i + 1][j][t];
            if (i > 0) v -= i * E[i - 1][j][t];
            out[t] = v;
        }
    } else {
        for (int t = 0; t <= i + j + 1; ++t) {
            double v = 2.0 * b * E[i][j + 1][t];
            if (j > 0) v -= j * E[i][j - 1][t];
            out[t] = v;
        }
    }
    return i + j + 2;
}

/* Contracted, normalised integrals of shell quartet (si sj|sk sl) for one operator.
 * val[ni][nj][nk][nl]; if der != NULL: der[c*3+x][ni][nj][nk][nl], c = 0..3 (A,B,C,D).
 * Returns the number of primitive quartets. */
static long shell_quartet(const sys_t *s, int si, int sj, int sk, int sl, double omega, work_t *w,
                          double *val, double *der) {
    const int32_t *sh = s->shells;
    int la = sh[4 * si + 1], lb = sh[4 * sj + 1], lc = sh[4 * sk + 1], ld = sh[4 * sl + 1];
    int na = ncart(la), nb = ncart(lb), nc = ncart(lc), nd = ncart(ld);
    size_t nfun = (size_t)na * nb * nc * nd;
    const double *A = s->xyz + 3 * sh[4 * si], *B = s->xyz + 3 * sh[4 * sj];
    const double *C = s->xyz + 3 * sh[4 * sk], *D = s->xyz + 3 * sh[4 * sl];
    int dv = der ? 1 : 0;
    int N = la + lb + lc + ld + dv;
    int NB = la + lb + dv; /* max total Hermite order of the bra */
    memset(val, 0, sizeof(double) * nfun);
    if (der) memset(der, 0, sizeof(double) * nfun * 12);
    double G[MAXM];
    long nprimq = 0;
    for (int ka = 0; ka < sh[4 * si + 2]; ++ka)
    for (int kb = 0; kb < sh[4 * sj + 2]; ++kb) {
        double a = s->exps[sh[4 * si + 3] + ka], b = s->exps[sh[4 * sj + 3] + kb];
        double p = a + b;
        double P[3];
        for (int x = 0; x < 3; ++x) {
            P[x] = (a * A[x] + b * B[x]) / p;
            hermite_E(la + dv, lb + dv, a, b, A[x] - B[x], w->Eb[x]);
        }
        double cab = s->cn[sh[4 * si + 3] + ka] * s->cn[sh[4 * sj + 3] + kb];
        for (int kc = 0; kc < sh[4 * sk + 2]; ++kc)
        for (int kd = 0; kd < sh[4 * sl + 2]; ++kd) {
            double c = s->exps[sh[4 * sk + 3] + kc], d = s->exps[sh[4 * sl + 3] + kd];
            double q = c + d;
            double Qc[3], PQ[3];
            for (int x = 0; x < 3; ++x) {
                Qc[x] = (c * C[x] + d * D[x]) / q;
                PQ[x] = P[x] - Qc[x];
                hermite_E(lc + dv, ld + dv, c, d, C[x] - D[x], w->Ek[x]);
            }
            double rho = p * q / (p + q);
            double T = rho * (PQ[0] * PQ[0] + PQ[1] * PQ[1] + PQ[2] * PQ[2]);
            orc_boys_op(N, T, rho, omega, G);
            hermite_R(N, rho, G, PQ[0], PQ[1], PQ[2], w->R, w->rwork);
            double pref = 2.0 * pow(PI, 2.5) / (p * q * sqrt(p + q)) * cab *
                          s->cn[sh[4 * sk + 3] + kc] * s->cn[sh[4 * sl + 3] + kd];
            ++nprimq;
            for (int ic = 0; ic < nc; ++ic)
            for (int id = 0; id < nd; ++id) {
                int cx[3], dx[3];
                cart_comp(lc, ic, &cx[0], &cx[1], &cx[2]);
                cart_comp(ld, id, &dx[0], &dx[1], &dx[2]);
                double nk = comp_norm(cx[0], cx[1], cx[2]) * comp_norm(dx[0], dx[1], dx[2]);
                int nkv = der ? 7 : 1;
                /* ket variants: 0 plain; 1..3 dC_x,y,z; 4..6 dD_x,y,z */
                for (int kv = 0; kv < nkv; ++kv) {
                    double e[3][NHERM1 + 1]; int ne[3];
                    for (int x = 0; x < 3; ++x) {
                        int var = 0;
                        if (kv >= 1 && kv <= 3 && kv - 1 == x) var = 1;
                        if (kv >= 4 && kv - 4 == x) var = 2;
                        ne[x] = herm_vec(w->Ek[x], cx[x], dx[x], c, d, var, e[x]);
                    }
                    for (int t = 0; t <= NB; ++t)
                    for (int u = 0; u <= NB - t; ++u)
                    for (int v = 0; v <= NB - t - u; ++v) {
                        double acc = 0.0;
                        for (int t2 = 0; t2 < ne[0]; ++t2)
                        for (int u2 = 0; u2 < ne[1]; ++u2)
                        for (int v2 = 0; v2 < ne[2]; ++v2) {
                            double sg = ((t2 + u2 + v2) & 1) ? -1.0 : 1.0;
                            acc += sg * e[0][t2] * e[1][u2] * e[2][v2] * w->R[t + t2][u + u2][v + v2];
                        }
                        w->K[kv][t][u][v] = acc;
                    }
                }
                for (int ia = 0; ia < na; ++ia)
                for (int ib = 0; ib < nb; ++ib) {
                    int ax[3], bx[3];
                    cart_comp(la, ia, &ax[0], &ax[1], &ax[2]);
                    cart_comp(lb, ib, &bx[0], &bx[1], &bx[2]);
                    double f = pref * nk * comp_norm(ax[0], ax[1], ax[2]) * comp_norm(bx[0], bx[1], bx[2]);
                    size_t idx = (((size_t)ia * nb + ib) * nc + ic) * nd + id;
                    int nbv = der ? 7 : 1;
                    /* bra variants: 0 plain; 1..3 dA_x,y,z; 4..6 dB_x,y,z */
                    for (int bv = 0; bv < nbv; ++bv) {
                        double e[3][NHERM1 + 1]; int ne[3];
                        for (int x = 0; x < 3; ++x) {
                            int var = 0;
                            if (bv >= 1 && bv <= 3 && bv - 1 == x) var = 1;
                            if (bv >= 4 && bv - 4 == x) var = 2;
                            ne[x] = herm_vec(w->Eb[x], ax[x], bx[x], a, b, var, e[x]);
                        }
                        int kvlo = 0, kvhi = (bv == 0) ? nkv - 1 : 0;
                        for (int kv = kvlo; kv <= kvhi; ++kv) {
                            double acc = 0.0;
                            for (int t = 0; t < ne[0]; ++t)
                            for (int u = 0; u < ne[1]; ++u)
                            for (int v = 0; v < ne[2]; ++v)
                                acc += e[0][t] * e[1][u] * e[2][v] * w->K[kv][t][u][v];
                            acc *= f;
                            if (bv == 0 && kv == 0) val[idx] += acc;
                            else if (bv > 0) der[(size_t)(bv - 1) * nfun + idx] += acc;      /* A: 0..2, B: 3..5 */
                            else der[(size_t)(6 + kv - 1) * nfun + idx] += acc;              /* C: 6..8, D: 9..11 */
                        }
                    }
                }
            }
        }
    }
    return nprimq;
}

/* ---------------------------------------------------------------- exported helpers for the pins */
#define SYS_ARGS int natom, const double *xyz, int nshell, const int32_t *shells, int nprim_total, \
                 const double *exps, const double *coefs
#define SYS_PASS natom, xyz, nshell, shells, nprim_total, exps, coefs

/* (si sj|sk sl) block, omega<=0: 1/r, else erf(omega r)/r.  out[ni][nj][nk][nl];
 * dout (may be NULL): [4][3][ni][nj][nk][nl]. */
int orc_eri_shell(SYS_ARGS, int si, int sj, int sk, int sl, double omega, double *out, double *dout) {
    sys_t s; if (sys_init(&s, SYS_PASS)) return -1;
    work_t *w = work_new(); if (!w) return -1;
    shell_quartet(&s, si, sj, sk, sl, omega, w, w->val, dout ? w->der : NULL);
    size_t nfun = (size_t)ncart(shells[4 * si + 1]) * ncart(shells[4 * sj + 1]) * ncart(shells[4 * sk + 1]) * ncart(shells[4 * sl + 1]);
    memcpy(out, w->val, sizeof(double) * nfun);
    if (dout) memcpy(dout, w->der, sizeof(double) * nfun * 12);
    work_free(w); sys_free(&s);
    return 0;
}

/* Full nbf^4 tensor (tiny systems only). */
int orc_eri_tensor(SYS_ARGS, double omega, double *out) {
    sys_t s; if (sys_init(&s, SYS_PASS)) return -1;
    work_t *w = work_new(); if (!w) return -1;
    size_t n = (size_t)s.nbf;
    for (int i = 0; i < nshell; ++i) for (int j = 0; j < nshell; ++j)
    for (int k = 0; k < nshell; ++k) for (int l = 0; l < nshell; ++l) {
        shell_quartet(&s, i, j, k, l, omega, w, w->val, NULL);
        int ni = s.off[i + 1] - s.off[i], nj = s.off[j + 1] - s.off[j];
        int nk = s.off[k + 1] - s.off[k], nl = s.off[l + 1] - s.off[l];
        for (int a = 0; a < ni; ++a) for (int b = 0; b < nj; ++b)
        for (int c = 0; c < nk; ++c) for (int d = 0; d < nl; ++d)
            out[(((size_t)(s.off[i] + a) * n + s.off[j] + b) * n + s.off[k] + c) * n + s.off[l] + d] =
                w->val[(((size_t)a * nj + b) * nk + c) * nl + d];
    }
    work_free(w); sys_free(&s);
    return 0;
}

/* Overlap matrix S[nbf][nbf] = product over directions of E_0^{ij} sqrt(pi/p), normalised functions
 * (used only to pin O1: unit self-overlap; and the omega->0 limit). */
int orc_overlap(SYS_ARGS, double *S) {
    sys_t s; if (sys_init(&s, SYS_PASS)) return -1;
    herm_t E[3];
    size_t n = (size_t)s.nbf;
    memset(S, 0, sizeof(double) * n * n);
    for (int i = 0; i < nshell; ++i) for (int j = 0; j < nshell; ++j) {
        int la = shells[4 * i + 1], lb = shells[4 * j + 1];
        const double *A = xyz + 3 * shells[4 * i], *B = xyz + 3 * shells[4 * j];
        for (int ka = 0; ka < shells[4 * i + 2]; ++ka) for (int kb = 0; kb < shells[4 * j + 2]; ++kb) {
            double a = exps[shells[4 * i + 3] + ka], b = exps[shells[4 * j + 3] + kb], p = a + b;
            for (int x = 0; x < 3; ++x) hermite_E(la, lb, a, b, A[x] - B[x], E[x]);
            double f = s.cn[shells[4 * i + 3] + ka] * s.cn[shells[4 * j + 3] + kb] * pow(PI / p, 1.5);
            for (int ia = 0; ia < ncart(la); ++ia) for (int ib = 0; ib < ncart(lb); ++ib) {
                int ax[3], bx[3];
                cart_comp(la, ia, &ax[0], &ax[1], &ax[2]); cart_comp(lb, ib, &bx[0], &bx[1], &bx[2]);
                S[(size_t)(s.off[i] + ia) * n + s.off[j] + ib] += f * comp_norm(ax[0], ax[1], ax[2]) * comp_norm(bx[0], bx[1], bx[2]) *
                    E[0][ax[0]][bx[0]][0] * E[1][ax[1]][bx[1]][0] * E[2][ax[2]][bx[2]][0];
            }
        }
    }
    sys_free(&s);
    return 0;
}

/* Schwarz bounds (reading S9): Q_ij = sqrt(max_{m in i, n in j} (mn|mn)), full operator, normalised functions.
 * Q[nshell][nshell], symmetric. */
static void schwarz_all(const sys_t *s, double *Q) {
    int ns = s->nshell;
#pragma omp parallel
    {
        work_t *w = work_new();
#pragma omp for schedule(dynamic, 8)
        for (int i = 0; i < ns; ++i)
            for (int j = 0; j <= i; ++j) {
                shell_quartet(s, i, j, i, j, 0.0, w, w->val, NULL);
                int ni = s->off[i + 1] - s->off[i], nj = s->off[j + 1] - s->off[j];
                double m = 0.0;
                for (int a = 0; a < ni; ++a) for (int b = 0; b < nj; ++b) {
                    double v = w->val[(((size_t)a * nj + b) * ni + a) * nj + b];
                    if (v > m) m = v;
                }
                Q[(size_t)i * ns + j] = Q[(size_t)j * ns + i] = sqrt(m);
            }
        work_free(w);
    }
}

int orc_schwarz(SYS_ARGS, double *Q) {
    sys_t s; if (sys_init(&s, SYS_PASS)) return -1;
    schwarz_all(&s, Q);
    sys_free(&s);
    return 0;
}

/* ---------------------------------------------------------------- O8/O9/O10: contraction */
typedef struct {
    double tau;               /* <= 0: no screening */
    int32_t density_weighted; /* 0: Schwarz only; 1: Schwarz x density (reading S9) */
    uint32_t sample_mod, sample_seed; /* 0: all quartets (reading S12) */
} orc_options;

typedef struct {
    int64_t pairs_total, pairs_kept, quartets_visited, quartets_computed, prim_quartets;
} orc_stats;

/* S12: fixed 64-bit finaliser; canonical shell-pair indices on the INPUT shell order. */
static uint64_t mix64(uint64_t z) {
    z ^= z >> 30; z *= 0xbf58476d1ce4e5b9ULL;
    z ^= z >> 27; z *= 0x94d049bb133111ebULL;
    z ^= z >> 31;
    return z;
}
static int sample_keep(int i, int j, int k, int l, uint32_t mod, uint32_t seed) {
    if (mod == 0) return 1;
    if (i < j) { int t = i; i = j; j = t; }
    if (k < l) { int t = k; k = l; l = t; }
    uint64_t ij = (uint64_t)i * (uint64_t)(i + 1) / 2 + (uint64_t)j;
    uint64_t kl = (uint64_t)k * (uint64_t)(k + 1) / 2 + (uint64_t)l;
    uint64_t hi = ij > kl ? ij : kl, lo = ij > kl ? kl : ij;
    uint64_t key = (hi << 32) ^ lo ^ ((uint64_t)seed * 0x9E3779B97F4A7C15ULL);
    return (mix64(key) % mod) == 0;
}
int orc_sample_keep(int i, int j, int k, int l, uint32_t mod, uint32_t seed) { return sample_keep(i, j, k, l, mod, seed); }

/* S9: shell-block maxima d_ij = max over all input matrices M, m in i, n in j of max(|M_mn|,|M_nm|). */
static void density_maxima(const sys_t *s, int nmat, const double *const *M, double *d) {
    int ns = s->nshell; size_t n = (size_t)s->nbf;
#pragma omp parallel for schedule(static)
    for (int i = 0; i < ns; ++i)
        for (int j = 0; j < ns; ++j) {
            double m = 0.0;
            for (int q = 0; q < nmat; ++q)
                for (int a = s->off[i]; a < s->off[i + 1]; ++a)
                    for (int b = s->off[j]; b < s->off[j + 1]; ++b) {
                        double v = fabs(M[q][a * n + b]), v2 = fabs(M[q][b * n + a]);
                        if (v > m) m = v;
                        if (v2 > m) m = v2;
                    }
            d[(size_t)i * ns + j] = m;
        }
}

/* S9: W_ijkl = max(C_J d_ij d_kl, C_K max(d_ik d_jl, d_il d_jk)) from the shell-block maxima d[ns][ns]. */
static double quartet_weight(const double *dm, int ns, int i, int j, int k, int l, double CJ, double CK) {
    double dij = dm[(size_t)i * ns + j], dkl = dm[(size_t)k * ns + l];
    double dik = dm[(size_t)i * ns + k], djl = dm[(size_t)j * ns + l];
    double dil = dm[(size_t)i * ns + l], djk = dm[(size_t)j * ns + k];
    double x1 = dik * djl, x2 = dil * djk;
    double W = CJ * dij * dkl, WK = CK * (x1 > x2 ? x1 : x2);
    if (WK > W) W = WK;
    return W;
}

/* Test access to the two S9 quantities above (tests/test_oracle_screening.py pins them): d[ns][ns] of the 2*npair
 * matrices A_k, B_k, and W[ns][ns][ns][ns] with C_J = sum|wJ_k cJ|, C_K = (|cK|+|cLR|) sum|wK_k| as in contract_driver. */
int orc_density_weights(SYS_ARGS, int npair, const double *const *A, const double *const *B, const double *wJ,
                        const double *wK, double cJ, double cK, double cLR, double *d, double *W) {
    sys_t s; int rc = sys_init(&s, SYS_PASS); if (rc) return rc;
    int ns = nshell;
    double CJ = 0.0, CK = 0.0;
    for (int k = 0; k < npair; ++k) { CJ += fabs(wJ[k] * cJ); CK += fabs(wK[k]); }
    CK *= fabs(cK) + fabs(cLR);
    const double **M = (const double **)malloc(sizeof(double *) * 2 * (size_t)npair);
    for (int k = 0; k < npair; ++k) { M[2 * k] = A[k]; M[2 * k + 1] = B[k]; }
    density_maxima(&s, 2 * npair, M, d);
    free(M);
    if (W)
        for (int i = 0; i < ns; ++i) for (int j = 0; j < ns; ++j) for (int k = 0; k < ns; ++k) for (int l = 0; l < ns; ++l)
            W[(((size_t)i * ns + j) * ns + k) * ns + l] = quartet_weight(d, ns, i, j, k, l, CJ, CK);
    sys_free(&s);
    return 0;
}

typedef struct { int i, j; double Q; } pair_t;
static int pair_cmp(const void *a, const void *b) {
    const pair_t *x = (const pair_t *)a, *y = (const pair_t *)b;
    if (x->Q > y->Q) return -1;
    if (x->Q < y->Q) return 1;
    if (x->i != y->i) return x->i < y->i ? -1 : 1;
    return x->j < y->j ? -1 : (x->j > y->j);
}

/* mode 0: gradient (grad[natom][3]); mode 1: energy (*E).
 * Production loop of O8: unique shell quartets i>=j, k>=l, ij>=kl, degeneracy deg = (1/2)^{[i=j]+[k=l]+[ij=kl]},
 *   Gt_J = sum_k wJ_k cJ [(A_mn+A_nm)(B_ls+B_sl) + (A_ls+A_sl)(B_mn+B_nm)]
 *   Gt_K = - sum_k wK_k [A_ml B_ns + A_nl B_ms + A_ms B_nl + A_ns B_ml + A_lm B_sn + A_ln B_sm + A_sm B_ln + A_sn B_lm]
 *   g += deg [ (Gt_J + cK Gt_K) d(mn|ls) + cLR Gt_K d(mn|ls)_lr ]
 * Screening (S9): pair kept iff tau<=0 or Q_ij Q_max >= tau; quartet kept iff tau<=0 or
 *   ( Q_ij Q_kl >= tau  and  (not density_weighted or Q_ij Q_kl W_ijkl >= tau) ),
 *   W_ijkl = max(C_J d_ij d_kl, C_K max(d_ik d_jl, d_il d_jk)), C_J = sum|wJ_k cJ|, C_K = (|cK|+|cLR|) sum|wK_k|. */
static int contract_driver(int mode, SYS_ARGS, const orc_options *opt, int npair,
                           const double *const *A, const double *const *B, const double *wJ, const double *wK,
                           double cJ, double cK, double cLR, double omega, double *out, orc_stats *st) {
    sys_t s; int rc = sys_init(&s, SYS_PASS); if (rc) return rc;
    if (cLR != 0.0 && omega <= 0.0) { sys_free(&s); return -3; }
    int ns = nshell; size_t n = (size_t)s.nbf;
    double tau = opt ? opt->tau : 0.0;
    int dw = opt ? opt->density_weighted : 0;
    uint32_t smod = opt ? opt->sample_mod : 0, sseed = opt ? opt->sample_seed : 0;
    double *Q = NULL, *dm = NULL;
    double CJ = 0.0, CK = 0.0;
    for (int k = 0; k < npair; ++k) { CJ += fabs(wJ[k] * cJ); CK += fabs(wK[k]); }
    CK *= fabs(cK) + fabs(cLR);
    size_t np_all = (size_t)ns * (ns + 1) / 2;
    pair_t *pairs = (pair_t *)malloc(sizeof(pair_t) * np_all);
    size_t npk = 0;
    if (tau > 0.0) {
        Q = (double *)malloc(sizeof(double) * (size_t)ns * ns);
        schwarz_all(&s, Q);
        double Qmax = 0.0;
        for (size_t t = 0; t < (size_t)ns * ns; ++t) if (Q[t] > Qmax) Qmax = Q[t];
        for (int i = 0; i < ns; ++i) for (int j = 0; j <= i; ++j)
            if (Q[(size_t)i * ns + j] * Qmax >= tau) { pairs[npk].i = i; pairs[npk].j = j; pairs[npk].Q = Q[(size_t)i * ns + j]; ++npk; }
        if (dw) {
            const double **M = (const double **)malloc(sizeof(double *) * 2 * (size_t)npair);
            for (int k = 0; k < npair; ++k) { M[2 * k] = A[k]; M[2 * k + 1] = B[k]; }
            dm = (double *)malloc(sizeof(double) * (size_t)ns * ns);
            density_maxima(&s, 2 * npair, M, dm);
            free(M);
        }
        qsort(pairs, npk, sizeof(pair_t), pair_cmp); /* Q descending: lets the inner loop stop early */
    } else {
        for (int i = 0; i < ns; ++i) for (int j = 0; j <= i; ++j) { pairs[npk].i = i; pairs[npk].j = j; pairs[npk].Q = 1.0; ++npk; }
    }
    int nthr = 1;
#ifdef _OPENMP
    nthr = omp_get_max_threads();
#endif
    size_t nout = mode == 0 ? (size_t)3 * natom : 1;
    double *acc = (double *)calloc(nout * (size_t)nthr, sizeof(double));
    int64_t visited = 0, computed = 0, primq = 0;
    int use_lr = (cLR != 0.0);
#pragma omp parallel reduction(+ : visited, computed, primq)
    {
        int tid = 0;
#ifdef _OPENMP
        tid = omp_get_thread_num();
#endif
        double *g = acc + nout * (size_t)tid;
        work_t *w = work_new();
        double *vF = w->val, *dF = w->der, *vL = w->val2, *dL = w->der2;
#pragma omp for schedule(dynamic, 1)
        for (long pa = 0; pa < (long)npk; ++pa) {
            int i = pairs[pa].i, j = pairs[pa].j;
            double Qij = pairs[pa].Q;
            for (long pb = 0; pb <= pa; ++pb) {   /* pairs sorted: pb<=pa enumerates each unordered pair of pairs once */
                int k = pairs[pb].i, l = pairs[pb].j;
                if (tau > 0.0) {
                    /* pairs[] is sorted by Q descending, so Q_ij Q_kl only falls as pb grows: stop at the first failure */
                    double qq = Qij * pairs[pb].Q;
                    if (qq < tau) break;
                    ++visited;
                    if (dw && qq * quartet_weight(dm, ns, i, j, k, l, CJ, CK) < tau) continue;
                } else ++visited;
                if (!sample_keep(i, j, k, l, smod, sseed)) continue;
                ++computed;
                double deg = 1.0;
                if (i == j) deg *= 0.5;
                if (k == l) deg *= 0.5;
                if (i == k && j == l) deg *= 0.5;
                primq += shell_quartet(&s, i, j, k, l, 0.0, w, vF, mode == 0 ? dF : NULL);
                if (use_lr) shell_quartet(&s, i, j, k, l, omega, w, vL, mode == 0 ? dL : NULL);
                int ni = s.off[i + 1] - s.off[i], nj = s.off[j + 1] - s.off[j];
                int nk = s.off[k + 1] - s.off[k], nl = s.off[l + 1] - s.off[l];
                size_t nfun = (size_t)ni * nj * nk * nl;
                int atoms[4] = { shells[4 * i], shells[4 * j], shells[4 * k], shells[4 * l] };
                for (int a = 0; a < ni; ++a) for (int b = 0; b < nj; ++b)
                for (int c = 0; c < nk; ++c) for (int d = 0; d < nl; ++d) {
                    size_t m_ = s.off[i] + a, n_ = s.off[j] + b, l_ = s.off[k] + c, s_ = s.off[l] + d;
                    double GJ = 0.0, GK = 0.0;
                    for (int q = 0; q < npair; ++q) {
                        const double *Aq = A[q], *Bq = B[q];
                        GJ += wJ[q] * cJ * ((Aq[m_ * n + n_] + Aq[n_ * n + m_]) * (Bq[l_ * n + s_] + Bq[s_ * n + l_]) +
                                            (Aq[l_ * n + s_] + Aq[s_ * n + l_]) * (Bq[m_ * n + n_] + Bq[n_ * n + m_]));
                        GK -= wK[q] * (Aq[m_ * n + l_] * Bq[n_ * n + s_] + Aq[n_ * n + l_] * Bq[m_ * n + s_] +
                                       Aq[m_ * n + s_] * Bq[n_ * n + l_] + Aq[n_ * n + s_] * Bq[m_ * n + l_] +
                                       Aq[l_ * n + m_] * Bq[s_ * n + n_] + Aq[l_ * n + n_] * Bq[s_ * n + m_] +
                                       Aq[s_ * n + m_] * Bq[l_ * n + n_] + Aq[s_ * n + n_] * Bq[l_ * n + m_]);
                    }
                    size_t idx = (((size_t)a * nj + b) * nk + c) * nl + d;
                    double gf = deg * (GJ + cK * GK), gl = deg * cLR * GK;
                    if (mode == 1) {
                        g[0] += gf * vF[idx] + (use_lr ? gl * vL[idx] : 0.0);
                    } else {
                        for (int cen = 0; cen < 4; ++cen) for (int x = 0; x < 3; ++x) {
                            double v = gf * dF[(size_t)(cen * 3 + x) * nfun + idx];
                            if (use_lr) v += gl * dL[(size_t)(cen * 3 + x) * nfun + idx];
                            g[3 * atoms[cen] + x] += v;
                        }
                    }
                }
            }
        }
        work_free(w);
    }
    for (size_t t = 0; t < nout; ++t) {
        double sum = 0.0;
        for (int th = 0; th < nthr; ++th) sum += acc[nout * (size_t)th + t]; /* fixed order */
        out[t] = sum;
    }
    if (st) {
        st->pairs_total = (int64_t)np_all; st->pairs_kept = (int64_t)npk;
        st->quartets_visited = visited; st->quartets_computed = computed; st->prim_quartets = primq;
    }
    free(acc); free(pairs); free(Q); free(dm); sys_free(&s);
    return 0;
}

int orc_gradient(SYS_ARGS, const orc_options *opt, int npair, const double *const *A, const double *const *B,
                 const double *wJ, const double *wK, double cJ, double cK, double cLR, double omega,
                 double *grad, orc_stats *st) {
    return contract_driver(0, SYS_PASS, opt, npair, A, B, wJ, wK, cJ, cK, cLR, omega, grad, st);
}

int orc_energy(SYS_ARGS, const orc_options *opt, int npair, const double *const *A, const double *const *B,
               const double *wJ, const double *wK, double cJ, double cK, double cLR, double omega,
               double *E, orc_stats *st) {
    return contract_driver(1, SYS_PASS, opt, npair, A, B, wJ, wK, cJ, cK, cLR, omega, E, st);
}

/* Reference loop of O8 (tiny inputs): ALL nshell^4 shell quartets, no symmetry, no screening:
 *   G = sum_k wJ_k cJ A_mn B_ls,  G_K = - sum_k wK_k A_ml B_ns,
 *   g_{atom(c)} += (G + cK G_K) d_c(mn|ls) + cLR G_K d_c(mn|ls)_lr. */
int orc_gradient_n4(SYS_ARGS, int npair, const double *const *A, const double *const *B,
                    const double *wJ, const double *wK, double cJ, double cK, double cLR, double omega, double *grad) {
    sys_t s; int rc = sys_init(&s, SYS_PASS); if (rc) return rc;
    size_t n = (size_t)s.nbf;
    work_t *w = work_new();
    memset(grad, 0, sizeof(double) * 3 * (size_t)natom);
    for (int i = 0; i < nshell; ++i) for (int j = 0; j < nshell; ++j)
    for (int k = 0; k < nshell; ++k) for (int l = 0; l < nshell; ++l) {
        shell_quartet(&s, i, j, k, l, 0.0, w, w->val, w->der);
        if (cLR != 0.0) shell_quartet(&s, i, j, k, l, omega, w, w->val2, w->der2);
        int ni = s.off[i + 1] - s.off[i], nj = s.off[j + 1] - s.off[j];
        int nk = s.off[k + 1] - s.off[k], nl = s.off[l + 1] - s.off[l];
        size_t nfun = (size_t)ni * nj * nk * nl;
        int atoms[4] = { shells[4 * i], shells[4 * j], shells[4 * k], shells[4 * l] };
        for (int a = 0; a < ni; ++a) for (int b = 0; b < nj; ++b)
        for (int c = 0; c < nk; ++c) for (int d = 0; d < nl; ++d) {
            size_t m_ = s.off[i] + a, n_ = s.off[j] + b, l_ = s.off[k] + c, s_ = s.off[l] + d;
            double G = 0.0, GK = 0.0;
            for (int q = 0; q < npair; ++q) {
                G += wJ[q] * cJ * A[q][m_ * n + n_] * B[q][l_ * n + s_];
                GK -= wK[q] * A[q][m_ * n + l_] * B[q][n_ * n + s_];
            }
            size_t idx = (((size_t)a * nj + b) * nk + c) * nl + d;
            for (int cen = 0; cen < 4; ++cen) for (int x = 0; x < 3; ++x) {
                double v = (G + cK * GK) * w->der[(size_t)(cen * 3 + x) * nfun + idx];
                if (cLR != 0.0) v += cLR * GK * w->der2[(size_t)(cen * 3 + x) * nfun + idx];
                grad[3 * atoms[cen] + x] += v;
            }
        }
    }
    work_free(w); sys_free(&s);
    return 0;
}

/* ---------------------------------------------------------------- NEXT-1: Fock-type (J/K) build
 * PAPER.md:138 (eq 19), PAPER.md:197-207 (eqs 33-34).  For each input matrix B_k (general, nonsymmetric allowed):
 *
 *   F_k[mn] = sum_{ls} [ wJ_k B_k[sl] (mn|ls)  -  X_k[sl] ( cK (ml|sn) + cLR (ml|sn)_lr ) ],   X_k = wK_k B_k + wKT_k B_k^T
 *
 * Eq 34 is wJ = 4, wK = wKT = 1, cK = alpha, cLR = beta  ((ms|ln) with B[sl] is (ml|sn) with B^T[sl]);
 * eq 19 is wJ = 2, wK = 1, wKT = 0.  The XC kernel term of both equations is out of scope.
 *
 * orc_fock_n4: the definition, all nshell^4 shell quartets, no symmetry, no screening (tiny inputs). */
int orc_fock_n4(SYS_ARGS, int nmat, const double *const *B, const double *wJ, const double *wK, const double *wKT,
                double cK, double cLR, double omega, double *const *F) {
    sys_t s; int rc = sys_init(&s, SYS_PASS); if (rc) return rc;
    size_t n = (size_t)s.nbf;
    work_t *w = work_new();
    for (int q = 0; q < nmat; ++q) memset(F[q], 0, sizeof(double) * n * n);
    for (int i = 0; i < nshell; ++i) for (int j = 0; j < nshell; ++j)
    for (int k = 0; k < nshell; ++k) for (int l = 0; l < nshell; ++l) {
        shell_quartet(&s, i, j, k, l, 0.0, w, w->val, NULL);
        if (cLR != 0.0) shell_quartet(&s, i, j, k, l, omega, w, w->val2, NULL);
        int ni = s.off[i + 1] - s.off[i], nj = s.off[j + 1] - s.off[j];
        int nk = s.off[k + 1] - s.off[k], nl = s.off[l + 1] - s.off[l];
        for (int a = 0; a < ni; ++a) for (int b = 0; b < nj; ++b)
        for (int c = 0; c < nk; ++c) for (int d = 0; d < nl; ++d) {
            size_t p_ = s.off[i] + a, q_ = s.off[j] + b, r_ = s.off[k] + c, s_ = s.off[l] + d;
            size_t idx = (((size_t)a * nj + b) * nk + c) * nl + d;
            double v = w->val[idx], vk = cK * v + (cLR != 0.0 ? cLR * w->val2[idx] : 0.0);
            for (int m = 0; m < nmat; ++m) {
                /* Coulomb: this integral read as (mn|ls) = (pq|rs):  F[pq] += wJ B[sr] (pq|rs) */
                F[m][p_ * n + q_] += wJ[m] * B[m][s_ * n + r_] * v;
                /* exchange: this integral read as (ml|sn) = (pq|rs): m=p, l=q, s=r, n=s:  F[ps] -= X[s l] = X[r q] */
                F[m][p_ * n + s_] -= (wK[m] * B[m][r_ * n + q_] + wKT[m] * B[m][q_ * n + r_]) * vk;
            }
        }
    }
    work_free(w); sys_free(&s);
    return 0;
}

/* Production loop: unique shell quartets i>=j, k>=l, ij>=kl with degeneracy deg, every integral digested into the
 * blocks its 8 index permutations touch:
 *   J:  F[mn] += wJ (B[ls]+B[sl]) I,  F[nm] += same,  F[ls] += wJ (B[mn]+B[nm]) I,  F[sl] += same
 *   K:  F[ms] -= X[ln] Ik, F[ns] -= X[lm] Ik, F[ml] -= X[sn] Ik, F[nl] -= X[sm] Ik,
 *       F[ln] -= X[ms] Ik, F[sn] -= X[ml] Ik, F[lm] -= X[ns] Ik, F[sm] -= X[nl] Ik        (Ik = cK I + cLR I_lr)
 * Screening: pair kept iff tau<=0 or Q_ij Q_max >= tau; quartet kept iff Q_ij Q_kl >= tau and (if density_weighted)
 *   Q_ij Q_kl W >= tau,  W = max( CJ max(d_ij, d_kl), CK max(d_ik, d_il, d_jk, d_jl) ),  d = block maxima over all B_k (both
 *   orientations), CJ = max_k |wJ_k|, CK = (|cK|+|cLR|) max_k (|wK_k|+|wKT_k|)   ("the product of the density
 *   matrix B_k and the Schwarz upper bound ... used as the screening parameter").  Subsample rule S12. */
int orc_fock(SYS_ARGS, const orc_options *opt, int nmat, const double *const *B, const double *wJ, const double *wK,
             const double *wKT, double cK, double cLR, double omega, double *const *F, orc_stats *st) {
    sys_t s; int rc = sys_init(&s, SYS_PASS); if (rc) return rc;
    if (cLR != 0.0 && omega <= 0.0) { sys_free(&s); return -3; }
    int ns = nshell; size_t n = (size_t)s.nbf;
    double tau = opt ? opt->tau : 0.0;
    int dw = opt ? opt->density_weighted : 0;
    uint32_t smod = opt ? opt->sample_mod : 0, sseed = opt ? opt->sample_seed : 0;
    double *Q = NULL, *dm = NULL;
    double CJ = 0.0, CK = 0.0;
    for (int m = 0; m < nmat; ++m) {
        if (fabs(wJ[m]) > CJ) CJ = fabs(wJ[m]);
        if (fabs(wK[m]) + fabs(wKT[m]) > CK) CK = fabs(wK[m]) + fabs(wKT[m]);
    }
    CK *= fabs(cK) + fabs(cLR);
    size_t np_all = (size_t)ns * (ns + 1) / 2;
    pair_t *pairs = (pair_t *)malloc(sizeof(pair_t) * np_all);
    size_t npk = 0;
    if (tau > 0.0) {
        Q = (double *)malloc(sizeof(double) * (size_t)ns * ns);
        schwarz_all(&s, Q);
        double Qmax = 0.0;
        for (size_t t = 0; t < (size_t)ns * ns; ++t) if (Q[t] > Qmax) Qmax = Q[t];
        for (int i = 0; i < ns; ++i) for (int j = 0; j <= i; ++j)
            if (Q[(size_t)i * ns + j] * Qmax >= tau) { pairs[npk].i = i; pairs[npk].j = j; pairs[npk].Q = Q[(size_t)i * ns + j]; ++npk; }
        if (dw) {
            dm = (double *)malloc(sizeof(double) * (size_t)ns * ns);
            density_maxima(&s, nmat, B, dm);
        }
        qsort(pairs, npk, sizeof(pair_t), pair_cmp);
    } else {
        for (int i = 0; i < ns; ++i) for (int j = 0; j <= i; ++j) { pairs[npk].i = i; pairs[npk].j = j; pairs[npk].Q = 1.0; ++npk; }
    }
    int nthr = 1;
#ifdef _OPENMP
    nthr = omp_get_max_threads();
#endif
    size_t nout = n * n * (size_t)nmat;
    /* per-thread copies summed in a fixed order when they fit in ~1.6 GB, else one copy updated with atomic adds */
    int shared = nout * (size_t)nthr > ((size_t)1 << 27) * (size_t)(nthr > 1);
    double *acc = (double *)calloc(shared ? nout : nout * (size_t)nthr, sizeof(double));
    if (!acc) { free(pairs); free(Q); free(dm); sys_free(&s); return -4; }
    int64_t visited = 0, computed = 0, primq = 0;
    int use_lr = (cLR != 0.0);
#pragma omp parallel reduction(+ : visited, computed, primq)
    {
        int tid = 0;
#ifdef _OPENMP
        tid = omp_get_thread_num();
#endif
        double *Ft = shared ? acc : acc + nout * (size_t)tid;
        work_t *w = work_new();
#pragma omp for schedule(dynamic, 1)
        for (long pa = 0; pa < (long)npk; ++pa) {
            int i = pairs[pa].i, j = pairs[pa].j;
            double Qij = pairs[pa].Q;
            for (long pb = 0; pb <= pa; ++pb) {
                int k = pairs[pb].i, l = pairs[pb].j;
                if (tau > 0.0) {
                    double qq = Qij * pairs[pb].Q;
                    if (qq < tau) break;
                    ++visited;
                    if (dw) {
                        double dij = dm[(size_t)i * ns + j], dkl = dm[(size_t)k * ns + l];
                        double dik = dm[(size_t)i * ns + k], djl = dm[(size_t)j * ns + l];
                        double dil = dm[(size_t)i * ns + l], djk = dm[(size_t)j * ns + k];
                        double mj = dij > dkl ? dij : dkl;
                        double mk = dik; if (djl > mk) mk = djl; if (dil > mk) mk = dil; if (djk > mk) mk = djk;
                        double W = CJ * mj, WK = CK * mk;
                        if (WK > W) W = WK;
                        if (qq * W < tau) continue;
                    }
                } else ++visited;
                if (!sample_keep(i, j, k, l, smod, sseed)) continue;
                ++computed;
                double deg = 1.0;
                if (i == j) deg *= 0.5;
                if (k == l) deg *= 0.5;
                if (i == k && j == l) deg *= 0.5;
                primq += shell_quartet(&s, i, j, k, l, 0.0, w, w->val, NULL);
                if (use_lr) shell_quartet(&s, i, j, k, l, omega, w, w->val2, NULL);
                int ni = s.off[i + 1] - s.off[i], nj = s.off[j + 1] - s.off[j];
                int nk = s.off[k + 1] - s.off[k], nl = s.off[l + 1] - s.off[l];
                for (int a = 0; a < ni; ++a) for (int b = 0; b < nj; ++b)
                for (int c = 0; c < nk; ++c) for (int d = 0; d < nl; ++d) {
                    size_t m_ = s.off[i] + a, n_ = s.off[j] + b, l_ = s.off[k] + c, s_ = s.off[l] + d;
                    size_t idx = (((size_t)a * nj + b) * nk + c) * nl + d;
                    double I = deg * w->val[idx], Ik = deg * (cK * w->val[idx] + (use_lr ? cLR * w->val2[idx] : 0.0));
                    for (int m = 0; m < nmat; ++m) {
                        const double *Bm = B[m];
                        double *Fm = Ft + (size_t)m * n * n;
                        double jb = wJ[m] * (Bm[l_ * n + s_] + Bm[s_ * n + l_]) * I, jk = wJ[m] * (Bm[m_ * n + n_] + Bm[n_ * n + m_]) * I;
#define ADD(r, c, v) do { double v_ = (v); double *p_ = &Fm[(r) * n + (c)]; if (shared) { _Pragma("omp atomic") *p_ += v_; } else *p_ += v_; } while (0)
#define XX(r, c) (wK[m] * Bm[(r) * n + (c)] + wKT[m] * Bm[(c) * n + (r)])
                        ADD(m_, n_, jb); ADD(n_, m_, jb);
                        ADD(l_, s_, jk); ADD(s_, l_, jk);
                        ADD(m_, s_, -XX(l_, n_) * Ik); ADD(n_, s_, -XX(l_, m_) * Ik);
                        ADD(m_, l_, -XX(s_, n_) * Ik); ADD(n_, l_, -XX(s_, m_) * Ik);
                        ADD(l_, n_, -XX(m_, s_) * Ik); ADD(s_, n_, -XX(m_, l_) * Ik);
                        ADD(l_, m_, -XX(n_, s_) * Ik); ADD(s_, m_, -XX(n_, l_) * Ik);
#undef XX
#undef ADD
                    }
                }
            }
        }
        work_free(w);
    }
    for (int m = 0; m < nmat; ++m)
        for (size_t t = 0; t < n * n; ++t) {
            double sum = 0.0;
            for (int th = 0; th < (shared ? 1 : nthr); ++th) sum += acc[nout * (size_t)th + (size_t)m * n * n + t];
            F[m][t] = sum;
        }
    if (st) {
        st->pairs_total = (int64_t)np_all; st->pairs_kept = (int64_t)npk;
        st->quartets_visited = visited; st->quartets_computed = computed; st->prim_quartets = primq;
    }
    free(acc); free(pairs); free(Q); free(dm); sys_free(&s);
    return 0;
}

/* ---------------------------------------------------------------- NEXT-2: real solid harmonics
 * C[2l+1][ncart(l)]: function m = -l..l of a spherical shell as a combination of the NORMALISED Cartesian components (order
 * S7).  Built from the harmonic polynomials themselves (no stored coefficients): each monomial x^a y^b z^c carries the factor
 * sqrt((2a-1)!!(2b-1)!!(2c-1)!!) that its normalised Cartesian function lacks, and the row is scaled to unit norm under the
 * overlap of the normalised components, S = prod_dir (e+e'-1)!! / sqrt((2e-1)!!(2e'-1)!!) (even e+e' only).
 * l <= 1: identity.  The tests pin the result by orthonormality under orc_overlap and by harmonicity of the polynomials. */
typedef struct { int n; struct { int a, b, c; double co; } t[3]; } poly_t;
static const poly_t SPH_D[5] = {
    {1, {{1, 1, 0, 1}}}, {1, {{0, 1, 1, 1}}}, {3, {{0, 0, 2, 2}, {2, 0, 0, -1}, {0, 2, 0, -1}}}, {1, {{1, 0, 1, 1}}},
    {2, {{2, 0, 0, 1}, {0, 2, 0, -1}}}};
static const poly_t SPH_F[7] = {
    {2, {{2, 1, 0, 3}, {0, 3, 0, -1}}}, {1, {{1, 1, 1, 1}}}, {3, {{0, 1, 2, 4}, {2, 1, 0, -1}, {0, 3, 0, -1}}},
    {3, {{0, 0, 3, 2}, {2, 0, 1, -3}, {0, 2, 1, -3}}}, {3, {{1, 0, 2, 4}, {3, 0, 0, -1}, {1, 2, 0, -1}}},
    {2, {{2, 0, 1, 1}, {0, 2, 1, -1}}}, {2, {{3, 0, 0, 1}, {1, 2, 0, -3}}}};
int orc_sph_matrix(int l, double *C) {
    int nc = ncart(l), ns = 2 * l + 1;
    if (l < 0 || l > 3) return -1;
    memset(C, 0, sizeof(double) * (size_t)(l < 2 ? nc * nc : ns * nc));
    if (l < 2) { for (int i = 0; i < nc; ++i) C[i * nc + i] = 1.0; return 0; }
    const poly_t *P = l == 2 ? SPH_D : SPH_F;
    for (int m = 0; m < ns; ++m) {
        double *row = C + (size_t)m * nc;
        for (int t = 0; t < P[m].n; ++t)
            for (int i = 0; i < nc; ++i) {
                int x, y, z; cart_comp(l, i, &x, &y, &z);
                if (x == P[m].t[t].a && y == P[m].t[t].b && z == P[m].t[t].c)
                    row[i] += P[m].t[t].co * sqrt(dfact(2 * x - 1) * dfact(2 * y - 1) * dfact(2 * z - 1));
            }
        double nrm = 0.0;
        for (int i = 0; i < nc; ++i) for (int j = 0; j < nc; ++j) {
            int x, y, z, x2, y2, z2; cart_comp(l, i, &x, &y, &z); cart_comp(l, j, &x2, &y2, &z2);
            if (((x + x2) | (y + y2) | (z + z2)) & 1) continue;
            double sij = dfact(x + x2 - 1) * dfact(y + y2 - 1) * dfact(z + z2 - 1) /
                         sqrt(dfact(2 * x - 1) * dfact(2 * y - 1) * dfact(2 * z - 1) * dfact(2 * x2 - 1) * dfact(2 * y2 - 1) * dfact(2 * z2 - 1));
            nrm += row[i] * sij * row[j];
        }
        for (int i = 0; i < nc; ++i) row[i] /= sqrt(nrm);
    }
    return 0;
}

int orc_num_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---------------------------------------------------------------- NEXT-4: one-electron terms of the gradient
 * Terms 1-3 of PAPER.md:84 (eq 7):  g_A = sum_mn P_mn dH^core_mn/dA + sum_mn W_mn dS_mn/dA + dV_nuc/dA,
 * H^core = T + V,  T_mn = <m| -1/2 Laplacian |n>,  V_mn = -sum_C Z_C <m| 1/|r - R_C| |n>,  V_nuc = sum_{C<D} Z_C Z_D / R_CD,
 * with P and W held fixed (general matrices, not assumed symmetric).  The paper computes these on the CPU.
 *
 * Textbook McMurchie-Davidson, written out: per direction s_ij = E_0^{ij} sqrt(pi/p);
 *   k_ij = -1/2 [ j(j-1) s_{i,j-2} - 2b(2j+1) s_{ij} + 4b^2 s_{i,j+2} ],   T = k_x s_y s_z + s_x k_y s_z + s_x s_y k_z;
 *   V^C  = -Z_C (2 pi/p) sum_tuv E_t E_u E_v R_tuv(p, P - C),  R^n_000 = (-2p)^n F_n(p |P-C|^2).
 * Derivatives, every centre explicitly (no translational-invariance shortcut): a function on A contributes
 * d/dA_x = 2a [i+1] - i [i-1] (eq 39 with the nuclear-coordinate sign), same for B; the operator centre enters R through
 * X = P_x - C_x, so d/dC_x R_tuv = -R_{t+1,u,v}.
 * Pins (tests/test_oracle_onee.py): closed forms for s functions (S, T, V via erf), T = 1/2 sum_x d^2 S / dA_x dB_x by finite
 * differences of the pinned overlap, V as the tight-charge limit of the pinned ERIs, hydrogen-like expectation values,
 * gradient vs central finite differences of orc_onee_energy, sum over atoms = 0. */
#define L1I (LMAX + 2)
#define L1J (LMAX + 4)
typedef double herm1_t[L1I][L1J][L1I + L1J + 1];

static void hermite_E1(int imax, int jmax, double a, double b, double X, herm1_t E) {   /* same recurrences as hermite_E (O4) */
    double p = a + b, mu = a * b / p;
    for (int i = 0; i <= imax; ++i)
        for (int j = 0; j <= jmax; ++j)
            for (int t = 0; t <= L1I + L1J; ++t) E[i][j][t] = 0.0;
    E[0][0][0] = exp(-mu * X * X);
    for (int j = 0; j <= jmax; ++j) {
        if (j > 0)
            for (int t = 0; t <= j; ++t) {
                double v = (a / p) * X * E[0][j - 1][t] + (t + 1) * E[0][j - 1][t + 1];
                if (t > 0) v += E[0][j - 1][t - 1] / (2.0 * p);
                E[0][j][t] = v;
            }
        for (int i = 1; i <= imax; ++i)
            for (int t = 0; t <= i + j; ++t) {
                double v = -(b / p) * X * E[i - 1][j][t] + (t + 1) * E[i - 1][j][t + 1];
                if (t > 0) v += E[i - 1][j][t - 1] / (2.0 * p);
                E[i][j][t] = v;
            }
    }
}

/* A 1-D factor of a (possibly differentiated) function: sum of at most two monomial powers with coefficients. */
typedef struct { int n; int pw[2]; double co[2]; } lin1_t;
static lin1_t lin_plain(int i) { lin1_t r; r.n = 1; r.pw[0] = i; r.co[0] = 1.0; r.pw[1] = 0; r.co[1] = 0.0; return r; }
static lin1_t lin_deriv(int i, double zeta) {   /* d/d(centre): 2 zeta [i+1] - i [i-1] */
    lin1_t r; r.n = 1; r.pw[0] = i + 1; r.co[0] = 2.0 * zeta; r.pw[1] = 0; r.co[1] = 0.0;
    if (i > 0) { r.n = 2; r.pw[1] = i - 1; r.co[1] = -(double)i; }
    return r;
}
static double s1d(herm1_t E, int i, int j, double p) { return (i < 0 || j < 0) ? 0.0 : E[i][j][0] * sqrt(PI / p); }
static double k1d(herm1_t E, int i, int j, double b, double p) {
    return -0.5 * (j * (j - 1) * s1d(E, i, j - 2, p) - 2.0 * b * (2 * j + 1) * s1d(E, i, j, p) + 4.0 * b * b * s1d(E, i, j + 2, p));
}
static double lin_s(herm1_t E, lin1_t u, lin1_t v, double p) {
    double r = 0.0;
    for (int x = 0; x < u.n; ++x) for (int y = 0; y < v.n; ++y) r += u.co[x] * v.co[y] * s1d(E, u.pw[x], v.pw[y], p);
    return r;
}
static double lin_k(herm1_t E, lin1_t u, lin1_t v, double b, double p) {
    double r = 0.0;
    for (int x = 0; x < u.n; ++x) for (int y = 0; y < v.n; ++y) r += u.co[x] * v.co[y] * k1d(E, u.pw[x], v.pw[y], b, p);
    return r;
}
static int lin_e(herm1_t E, lin1_t u, lin1_t v, double *out) {   /* Hermite vector of the product, entries t = 0..n-1 */
    int n = 0;
    for (int t = 0; t <= L1I + L1J; ++t) out[t] = 0.0;
    for (int x = 0; x < u.n; ++x) for (int y = 0; y < v.n; ++y) {
        int top = u.pw[x] + v.pw[y];
        for (int t = 0; t <= top; ++t) out[t] += u.co[x] * v.co[y] * E[u.pw[x]][v.pw[y]][t];
        if (top + 1 > n) n = top + 1;
    }
    return n;
}

/* One shell pair (si, sj): contracted, normalised S, T, V blocks [ni][nj] (any may be NULL), and, if acc != NULL, the pair's
 * contribution sum_ab [ P_ab d(T+V)_ab + W_ab dS_ab ] to acc[3*natom] for all centres (A, B and every nucleus C). */
static void onee_pair(const sys_t *s, const double *Zn, int si, int sj, double *Sb, double *Tb, double *Vb,
                      const double *Pm, const double *Wm, double *acc, rtab_t R, double *rwork) {
    const int32_t *sh = s->shells;
    int la = sh[4 * si + 1], lb = sh[4 * sj + 1], na = ncart(la), nb = ncart(lb);
    int atA = sh[4 * si], atB = sh[4 * sj];
    const double *A = s->xyz + 3 * atA, *B = s->xyz + 3 * atB;
    size_t n = (size_t)s->nbf;
    int dv = acc ? 1 : 0;
    if (Sb) memset(Sb, 0, sizeof(double) * (size_t)na * nb);
    if (Tb) memset(Tb, 0, sizeof(double) * (size_t)na * nb);
    if (Vb) memset(Vb, 0, sizeof(double) * (size_t)na * nb);
    herm1_t E[3];
    double G[MAXM];
    for (int ka = 0; ka < sh[4 * si + 2]; ++ka)
    for (int kb = 0; kb < sh[4 * sj + 2]; ++kb) {
        double a = s->exps[sh[4 * si + 3] + ka], b = s->exps[sh[4 * sj + 3] + kb], p = a + b;
        double Pc[3];
        for (int x = 0; x < 3; ++x) { Pc[x] = (a * A[x] + b * B[x]) / p; hermite_E1(la + dv, lb + dv + 2, a, b, A[x] - B[x], E[x]); }
        double cab = s->cn[sh[4 * si + 3] + ka] * s->cn[sh[4 * sj + 3] + kb];
        for (int ia = 0; ia < na; ++ia)
        for (int ib = 0; ib < nb; ++ib) {
            int ax[3], bx[3];
            cart_comp(la, ia, &ax[0], &ax[1], &ax[2]); cart_comp(lb, ib, &bx[0], &bx[1], &bx[2]);
            double f = cab * comp_norm(ax[0], ax[1], ax[2]) * comp_norm(bx[0], bx[1], bx[2]);
            double pw = Pm ? Pm[(size_t)(s->off[si] + ia) * n + s->off[sj] + ib] : 0.0;
            double ww = Wm ? Wm[(size_t)(s->off[si] + ia) * n + s->off[sj] + ib] : 0.0;
            /* variant 0: plain; 1..3: d/dA_x,y,z; 4..6: d/dB_x,y,z */
            for (int var = 0; var < (dv ? 7 : 1); ++var) {
                lin1_t u[3], v[3];
                for (int x = 0; x < 3; ++x) {
                    u[x] = (var >= 1 && var <= 3 && var - 1 == x) ? lin_deriv(ax[x], a) : lin_plain(ax[x]);
                    v[x] = (var >= 4 && var - 4 == x) ? lin_deriv(bx[x], b) : lin_plain(bx[x]);
                }
                double sx = lin_s(E[0], u[0], v[0], p), sy = lin_s(E[1], u[1], v[1], p), sz = lin_s(E[2], u[2], v[2], p);
                double kx = lin_k(E[0], u[0], v[0], b, p), ky = lin_k(E[1], u[1], v[1], b, p), kz = lin_k(E[2], u[2], v[2], b, p);
                double Sv = f * sx * sy * sz;
                double Tv = f * (kx * sy * sz + sx * ky * sz + sx * sy * kz);
                double ex[L1I + L1J + 1], ey[L1I + L1J + 1], ez[L1I + L1J + 1];
                int nx = lin_e(E[0], u[0], v[0], ex), ny = lin_e(E[1], u[1], v[1], ey), nz = lin_e(E[2], u[2], v[2], ez);
                double Vv = 0.0;
                for (int c = 0; c < s->natom; ++c) {
                    if (Zn[c] == 0.0) continue;
                    const double *Cc = s->xyz + 3 * c;
                    double X = Pc[0] - Cc[0], Y = Pc[1] - Cc[1], Zd = Pc[2] - Cc[2];
                    int N = la + lb + 2 * dv;
                    orc_boys(N, p * (X * X + Y * Y + Zd * Zd), G);
                    hermite_R(N, p, G, X, Y, Zd, R, rwork);
                    double vc = 0.0, dC[3] = {0.0, 0.0, 0.0};
                    for (int t = 0; t < nx; ++t) for (int uu = 0; uu < ny; ++uu) for (int w = 0; w < nz; ++w) {
                        double e3 = ex[t] * ey[uu] * ez[w];
                        vc += e3 * R[t][uu][w];
                        if (var == 0 && dv) { dC[0] -= e3 * R[t + 1][uu][w]; dC[1] -= e3 * R[t][uu + 1][w]; dC[2] -= e3 * R[t][uu][w + 1]; }
                    }
                    double pref = -Zn[c] * 2.0 * PI / p * f;
                    Vv += pref * vc;
                    if (var == 0 && dv) for (int x = 0; x < 3; ++x) acc[3 * c + x] += pw * pref * dC[x];   /* operator centre */
                }
                if (var == 0) {
                    if (Sb) Sb[ia * nb + ib] += Sv;
                    if (Tb) Tb[ia * nb + ib] += Tv;
                    if (Vb) Vb[ia * nb + ib] += Vv;
                } else {
                    int at = var <= 3 ? atA : atB, x = (var - 1) % 3;
                    acc[3 * at + x] += pw * (Tv + Vv) + ww * Sv;
                }
            }
        }
    }
}

int orc_onee_matrices(SYS_ARGS, const double *Z, double *S, double *T, double *V) {
    sys_t s; int rc = sys_init(&s, SYS_PASS); if (rc) return rc;
    size_t n = (size_t)s.nbf;
    double *rwork = (double *)malloc(sizeof(double) * (size_t)(NTOT + 1) * (NTOT + 1) * (NTOT + 1) * (NTOT + 1));
    rtab_t *R = (rtab_t *)malloc(sizeof(rtab_t));
    double Sb[NCMAX * NCMAX], Tb[NCMAX * NCMAX], Vb[NCMAX * NCMAX];
    for (int i = 0; i < nshell; ++i) for (int j = 0; j < nshell; ++j) {
        onee_pair(&s, Z, i, j, Sb, Tb, Vb, NULL, NULL, NULL, *R, rwork);
        int ni = s.off[i + 1] - s.off[i], nj = s.off[j + 1] - s.off[j];
        for (int a = 0; a < ni; ++a) for (int b = 0; b < nj; ++b) {
            size_t idx = (size_t)(s.off[i] + a) * n + s.off[j] + b;
            S[idx] = Sb[a * nj + b]; T[idx] = Tb[a * nj + b]; V[idx] = Vb[a * nj + b];
        }
    }
    free(R); free(rwork); sys_free(&s);
    return 0;
}

static double vnuc(const sys_t *s, const double *Z, double *grad) {
    double e = 0.0;
    for (int c = 0; c < s->natom; ++c) for (int d = 0; d < c; ++d) {
        double r[3], r2 = 0.0;
        for (int x = 0; x < 3; ++x) { r[x] = s->xyz[3 * c + x] - s->xyz[3 * d + x]; r2 += r[x] * r[x]; }
        double rr = sqrt(r2);
        e += Z[c] * Z[d] / rr;
        if (grad) for (int x = 0; x < 3; ++x) { double gx = -Z[c] * Z[d] * r[x] / (r2 * rr); grad[3 * c + x] += gx; grad[3 * d + x] -= gx; }
    }
    return e;
}

/* E_1e = sum_mn P_mn (T + V)_mn + sum_mn W_mn S_mn + V_nuc. */
int orc_onee_energy(SYS_ARGS, const double *Z, const double *P, const double *W, double *E) {
    sys_t s; int rc = sys_init(&s, SYS_PASS); if (rc) return rc;
    size_t n = (size_t)s.nbf;
    double *rwork = (double *)malloc(sizeof(double) * (size_t)(NTOT + 1) * (NTOT + 1) * (NTOT + 1) * (NTOT + 1));
    rtab_t *R = (rtab_t *)malloc(sizeof(rtab_t));
    double Sb[NCMAX * NCMAX], Tb[NCMAX * NCMAX], Vb[NCMAX * NCMAX];
    double e = 0.0;
    for (int i = 0; i < nshell; ++i) for (int j = 0; j < nshell; ++j) {
        onee_pair(&s, Z, i, j, Sb, Tb, Vb, NULL, NULL, NULL, *R, rwork);
        int ni = s.off[i + 1] - s.off[i], nj = s.off[j + 1] - s.off[j];
        for (int a = 0; a < ni; ++a) for (int b = 0; b < nj; ++b) {
            size_t idx = (size_t)(s.off[i] + a) * n + s.off[j] + b;
            e += P[idx] * (Tb[a * nj + b] + Vb[a * nj + b]) + W[idx] * Sb[a * nj + b];
        }
    }
    *E = e + vnuc(&s, Z, NULL);
    free(R); free(rwork); sys_free(&s);
    return 0;
}

/* grad[natom][3] = dE_1e/dR with P, W fixed: terms 1-3 of eq 7.  All nshell^2 ordered shell pairs. */
int orc_onee_gradient(SYS_ARGS, const double *Z, const double *P, const double *W, double *grad) {
    sys_t s; int rc = sys_init(&s, SYS_PASS); if (rc) return rc;
    size_t ng = 3 * (size_t)natom;
    memset(grad, 0, sizeof(double) * ng);
    int nthr = 1;
#ifdef _OPENMP
    nthr = omp_get_max_threads();
#endif
    double *acc = (double *)calloc(ng * (size_t)nthr, sizeof(double));
    if (!acc) { sys_free(&s); return -1; }
#pragma omp parallel
    {
        int th = 0;
#ifdef _OPENMP
        th = omp_get_thread_num();
#endif
        double *rwork = (double *)malloc(sizeof(double) * (size_t)(NTOT + 1) * (NTOT + 1) * (NTOT + 1) * (NTOT + 1));
        rtab_t *R = (rtab_t *)malloc(sizeof(rtab_t));
#pragma omp for schedule(dynamic, 1)
        for (int i = 0; i < nshell; ++i)
            for (int j = 0; j < nshell; ++j)
                onee_pair(&s, Z, i, j, NULL, NULL, NULL, P, W, acc + ng * (size_t)th, *R, rwork);
        free(R); free(rwork);
    }
    for (int th = 0; th < nthr; ++th) for (size_t t = 0; t < ng; ++t) grad[t] += acc[ng * (size_t)th + t];
    vnuc(&s, Z, grad);
    free(acc); sys_free(&s);
    return 0;
}
