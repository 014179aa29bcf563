/*
 * gnep_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU oracle for the GNEP hot path (arxiv 2507.00528; citations "P:n" are line
 * numbers of /root/reference/PAPER.md, "S:8(c).k" are readings listed in SURVEY.md section 8(c) and
 * repeated in DESIGN.md).  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference leg may call it.  It shares no code with the CUDA path under
 * paper_2507_00528_b200/csrc and neither includes the other.
 *
 * What it computes, in the paper's order:
 *   neighbour sets            P:44 Eq.2                       orc_batch_create
 *   Chebyshev basis, cutoff   P:72 Eq.6, App.A      orc_basis
 *   harmonics b_lm, B_lm      P:251-449 App.B (l = 1..8), P:454 Eq.B9    orc_blm
 *   descriptors q_n, q_nl     P:69-85 Eq.5-8 (+ 4-body, S:8(c).4; + 5-body, R41)   orc_descriptors
 *   network F(G)              P:718 Eq.D1.1-D1.6              orc_network
 *   E, F, virial              P:39 Eq.1, Eq.3, Eq.4, P:611 Eq.C3.6   orc_predict
 *   loss                      P:93-102 Eq.9-12 (+ L2, S:8(c).8)     orc_loss
 *   analytic gradient         P:104-114 Eq.13-16, App.C/D in contraction-first form (S:8(c).9)
 *                                                             orc_loss_and_grad
 *   Adam                      P:960 ref.21 (textbook, S:8(c).11)    orc_adam_step
 * Every function is pinned by tests/test_oracle_*.py (finite differences of the plain loss/energy,
 * closed forms, invariants, brute force): nothing here is "parity unpinned".
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC gnep_oracle.c -o libgnep_oracle.so -lm
 * OpenMP is used over structures only (independent units).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define NLM_MAX 80   /* (l,m) slots for l = 1..8; slot lm = l*l - 1 + m, m = 0..2l */
#define KMAX 32

typedef struct {
  int32_t T;               /* number of species */
  int32_t NR, KR;          /* radial functions n, radial basis functions k */
  int32_t NA, KA;          /* angular radial functions, basis functions */
  int32_t L;               /* l_max 1..8 */
  int32_t use4;            /* 4-body term */
  int32_t use5;            /* 5-body term */
  int32_t Nn;              /* hidden neurons */
  int32_t loss_mode;       /* 0 = mean square (paper Eq.9-12), 1 = RMSE */
  double rcR, rcA;
  double lam_e, lam_f, lam_v, lam_2;
} orc_spec;

typedef struct {
  int S, N;
  int *aoff;               /* S+1 */
  double *pos;             /* N*3, wrapped into the cell */
  double *cell;            /* S*9 rows a,b,c */
  int *type;               /* N */
  int64_t *rptr[2];        /* N+1 : [0] radial, [1] angular */
  int *nj[2];              /* neighbour atom index (global) */
  int *nsh[2];             /* 3 ints per pair */
  double *nr[2];           /* r_ij, 3 doubles per pair */
  double *Eref, *Fref, *Wref;   /* may be NULL */
  double *we, *wf, *wv;         /* per-structure weights of the three loss terms (R40); NULL = all ones */
} orc_batch;

/* ------------------------------------------------------------------ sizes and layout (S:8(c).2) */
int orc_ndes(const orc_spec *sp) { return sp->NR + sp->NA * sp->L + (sp->use4 ? sp->NA : 0) + (sp->use5 ? sp->NA : 0); }
int orc_nlm(const orc_spec *sp) { return sp->L * (sp->L + 2); }
static int off5(const orc_spec *sp) { return sp->NR + sp->L * sp->NA + (sp->use4 ? sp->NA : 0); }   /* first 5-body descriptor */
static int64_t off_cR(const orc_spec *sp) { (void)sp; return 0; }
static int64_t off_cA(const orc_spec *sp) { return (int64_t)sp->T * sp->T * sp->NR * sp->KR; }
static int64_t off_net(const orc_spec *sp) { return off_cA(sp) + (int64_t)sp->T * sp->T * sp->NA * sp->KA; }
static int64_t net_size(const orc_spec *sp) { return (int64_t)sp->Nn * orc_ndes(sp) + 2 * sp->Nn + 1; }
int64_t orc_num_params(const orc_spec *sp) { return off_net(sp) + sp->T * net_size(sp); }
int orc_max_threads(void) {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

/* ------------------------------------------------------------------ Chebyshev basis (App.A) */
/* f_k(d) = 1/2 (T_k(xi)+1) f_c(d), xi = 2(d/rc-1)^2-1; fp = d f_k / dd.  k = 0..K-1. */
void orc_basis(double rc, int K, double d, double *f, double *fp) {
  double x = d / rc - 1.0;
  double xi = 2.0 * x * x - 1.0;                 /* A1.2 */
  double dxi = 4.0 * x / rc;                     /* d xi / d d */
  double fc, fcp;
  if (d < rc) {                                  /* A2.1, A2.2 */
    fc = 0.5 * (1.0 + cos(M_PI * d / rc));
    fcp = -(M_PI / (2.0 * rc)) * sin(M_PI * d / rc);
  } else { fc = 0.0; fcp = 0.0; }
  double Tk[KMAX], Tp[KMAX];
  for (int k = 0; k < K; ++k) {
    if (k == 0) { Tk[0] = 1.0; Tp[0] = 0.0; }                      /* A1.1, A1.3 */
    else if (k == 1) { Tk[1] = xi; Tp[1] = 1.0; }                  /* A1.4 */
    else {
      Tk[k] = 2.0 * xi * Tk[k - 1] - Tk[k - 2];                    /* A1.1 */
      Tp[k] = 2.0 * Tk[k - 1] + 2.0 * xi * Tp[k - 1] - Tp[k - 2];  /* A1.5 */
    }
    f[k] = 0.5 * (Tk[k] + 1.0) * fc;                               /* Eq.6 */
    fp[k] = 0.5 * (Tp[k] * dxi * fc + (Tk[k] + 1.0) * fcp);        /* exact derivative of Eq.6 */
  }
}

/* ------------------------------------------------------------------ harmonics (App.B) */
/* l = 5..8 (B5.1-B8.17).  Every printed b_lm is a product  Z(z, r^2) * C(x, y)  of a polynomial in z and
 * r^2 = x^2+y^2+z^2 and one of the planar polynomials printed beside it,
 *   c_m = Re (x+iy)^m :  c1 = x, c2 = x^2-y^2, c3 = x^3-3xy^2, c4 = x^4-6x^2y^2+y^4, c5 = x^5-10x^3y^2+5xy^4, ...
 *   s_m = Im (x+iy)^m :  s1 = y, s2 = 2xy,     s3 = 3x^2y-y^3, s4 = 4x^3y-4xy^3,     s5 = 5x^4y-10x^2y^3+y^5, ...
 * (m = 0: C = 1).  Slots: m = 0 first, then (c_m', s_m') for m' = 1..l.  The gradient is the product rule with
 *   dZ/dx = 2x dZ/dr2, dZ/dy = 2y dZ/dr2, dZ/dz (total) = Zz + 2z dZ/dr2,   Zz = partial dZ/dz at fixed r2,
 * and the planar derivatives written out term by term below. */
static void planar(double x, double y, double *c, double *s, double *cx, double *cy, double *sx, double *sy) {
  double x2 = x * x, y2 = y * y, x3 = x2 * x, y3 = y2 * y, x4 = x2 * x2, y4 = y2 * y2, x5 = x4 * x, y5 = y4 * y;
  double x6 = x3 * x3, y6 = y3 * y3, x7 = x6 * x, y7 = y6 * y, x8 = x4 * x4, y8 = y4 * y4;
  c[0] = 1; s[0] = 0; cx[0] = 0; cy[0] = 0; sx[0] = 0; sy[0] = 0;
  c[1] = x;                                   cx[1] = 1;                                cy[1] = 0;
  s[1] = y;                                   sx[1] = 0;                                sy[1] = 1;
  c[2] = x2 - y2;                             cx[2] = 2 * x;                            cy[2] = -2 * y;
  s[2] = 2 * x * y;                           sx[2] = 2 * y;                            sy[2] = 2 * x;
  c[3] = x3 - 3 * x * y2;                     cx[3] = 3 * x2 - 3 * y2;                  cy[3] = -6 * x * y;
  s[3] = 3 * x2 * y - y3;                     sx[3] = 6 * x * y;                        sy[3] = 3 * x2 - 3 * y2;
  c[4] = x4 - 6 * x2 * y2 + y4;               cx[4] = 4 * x3 - 12 * x * y2;             cy[4] = -12 * x2 * y + 4 * y3;
  s[4] = 4 * x3 * y - 4 * x * y3;             sx[4] = 12 * x2 * y - 4 * y3;             sy[4] = 4 * x3 - 12 * x * y2;
  c[5] = x5 - 10 * x3 * y2 + 5 * x * y4;      cx[5] = 5 * x4 - 30 * x2 * y2 + 5 * y4;   cy[5] = -20 * x3 * y + 20 * x * y3;
  s[5] = 5 * x4 * y - 10 * x2 * y3 + y5;      sx[5] = 20 * x3 * y - 20 * x * y3;        sy[5] = 5 * x4 - 30 * x2 * y2 + 5 * y4;
  c[6] = x6 - 15 * x4 * y2 + 15 * x2 * y4 - y6;
  cx[6] = 6 * x5 - 60 * x3 * y2 + 30 * x * y4;            cy[6] = -30 * x4 * y + 60 * x2 * y3 - 6 * y5;
  s[6] = 6 * x5 * y - 20 * x3 * y3 + 6 * x * y5;
  sx[6] = 30 * x4 * y - 60 * x2 * y3 + 6 * y5;            sy[6] = 6 * x5 - 60 * x3 * y2 + 30 * x * y4;
  c[7] = x7 - 21 * x5 * y2 + 35 * x3 * y4 - 7 * x * y6;
  cx[7] = 7 * x6 - 105 * x4 * y2 + 105 * x2 * y4 - 7 * y6; cy[7] = -42 * x5 * y + 140 * x3 * y3 - 42 * x * y5;
  s[7] = 7 * x6 * y - 35 * x4 * y3 + 21 * x2 * y5 - y7;
  sx[7] = 42 * x5 * y - 140 * x3 * y3 + 42 * x * y5;       sy[7] = 7 * x6 - 105 * x4 * y2 + 105 * x2 * y4 - 7 * y6;
  c[8] = x8 - 28 * x6 * y2 + 70 * x4 * y4 - 28 * x2 * y6 + y8;
  cx[8] = 8 * x7 - 168 * x5 * y2 + 280 * x3 * y4 - 56 * x * y6;
  cy[8] = -56 * x6 * y + 280 * x4 * y3 - 168 * x2 * y5 + 8 * y7;
  s[8] = 8 * x7 * y - 56 * x5 * y3 + 56 * x3 * y5 - 8 * x * y7;
  sx[8] = 56 * x6 * y - 280 * x4 * y3 + 168 * x2 * y5 - 8 * y7;
  sy[8] = 8 * x7 - 168 * x5 * y2 + 280 * x3 * y4 - 56 * x * y6;
}
/* slot lm = Z, slots lm+1 / lm+2 = Z c_m / Z s_m */
static void put_zero(int lm, double Z, double Zz, double Zr, double x, double y, double z, double *b, double (*g)[3]) {
  b[lm] = Z; g[lm][0] = 2 * x * Zr; g[lm][1] = 2 * y * Zr; g[lm][2] = Zz + 2 * z * Zr;
}
static void put_pair(int lm, int m, double Z, double Zz, double Zr, double x, double y, double z, const double *c,
                     const double *s, const double *cx, const double *cy, const double *sx, const double *sy, double *b,
                     double (*g)[3]) {
  b[lm] = Z * c[m];
  g[lm][0] = 2 * x * Zr * c[m] + Z * cx[m]; g[lm][1] = 2 * y * Zr * c[m] + Z * cy[m]; g[lm][2] = (Zz + 2 * z * Zr) * c[m];
  b[lm + 1] = Z * s[m];
  g[lm + 1][0] = 2 * x * Zr * s[m] + Z * sx[m]; g[lm + 1][1] = 2 * y * Zr * s[m] + Z * sy[m]; g[lm + 1][2] = (Zz + 2 * z * Zr) * s[m];
}
static void blm_poly_high(double x, double y, double z, double *b, double (*g)[3]) {
  double c[9], s[9], cx[9], cy[9], sx[9], sy[9];
  planar(x, y, c, s, cx, cy, sx, sy);
  double r2 = x * x + y * y + z * z, r4 = r2 * r2, r6 = r4 * r2, r8 = r4 * r4;
  double z2 = z * z, z3 = z2 * z, z4 = z2 * z2, z5 = z4 * z, z6 = z3 * z3, z7 = z6 * z, z8 = z4 * z4;
#define PAIR(lm, m, Z, Zz, Zr) put_pair(lm, m, Z, Zz, Zr, x, y, z, c, s, cx, cy, sx, sy, b, g)
  /* l = 5: B5.1-B5.11, slots 24..34 */
  put_zero(24, 63 * z5 - 70 * z3 * r2 + 15 * z * r4, 315 * z4 - 210 * z2 * r2 + 15 * r4, -70 * z3 + 30 * z * r2, x, y, z, b, g);
  PAIR(25, 1, 21 * z4 - 14 * z2 * r2 + r4, 84 * z3 - 28 * z * r2, -14 * z2 + 2 * r2);
  PAIR(27, 2, 3 * z3 - z * r2, 9 * z2 - r2, -z);
  PAIR(29, 3, 9 * z2 - r2, 18 * z, -1.0);
  PAIR(31, 4, z, 1.0, 0.0);
  PAIR(33, 5, 1.0, 0.0, 0.0);
  /* l = 6: B6.1-B6.13, slots 35..47 */
  put_zero(35, 231 * z6 - 315 * z4 * r2 + 105 * z2 * r4 - 5 * r6, 1386 * z5 - 1260 * z3 * r2 + 210 * z * r4,
           -315 * z4 + 210 * z2 * r2 - 15 * r4, x, y, z, b, g);
  PAIR(36, 1, 33 * z5 - 30 * z3 * r2 + 5 * z * r4, 165 * z4 - 90 * z2 * r2 + 5 * r4, -30 * z3 + 10 * z * r2);
  PAIR(38, 2, 33 * z4 - 18 * z2 * r2 + r4, 132 * z3 - 36 * z * r2, -18 * z2 + 2 * r2);
  PAIR(40, 3, 11 * z3 - 3 * z * r2, 33 * z2 - 3 * r2, -3 * z);
  PAIR(42, 4, 11 * z2 - r2, 22 * z, -1.0);
  PAIR(44, 5, z, 1.0, 0.0);
  PAIR(46, 6, 1.0, 0.0, 0.0);
  /* l = 7: B7.1-B7.15, slots 48..62 */
  put_zero(48, 429 * z7 - 693 * z5 * r2 + 315 * z3 * r4 - 35 * z * r6, 3003 * z6 - 3465 * z4 * r2 + 945 * z2 * r4 - 35 * r6,
           -693 * z5 + 630 * z3 * r2 - 105 * z * r4, x, y, z, b, g);
  PAIR(49, 1, 429 * z6 - 495 * z4 * r2 + 135 * z2 * r4 - 5 * r6, 2574 * z5 - 1980 * z3 * r2 + 270 * z * r4,
       -495 * z4 + 270 * z2 * r2 - 15 * r4);
  PAIR(51, 2, 143 * z5 - 110 * z3 * r2 + 15 * z * r4, 715 * z4 - 330 * z2 * r2 + 15 * r4, -110 * z3 + 30 * z * r2);
  PAIR(53, 3, 143 * z4 - 66 * z2 * r2 + 3 * r4, 572 * z3 - 132 * z * r2, -66 * z2 + 6 * r2);
  PAIR(55, 4, 13 * z3 - 3 * z * r2, 39 * z2 - 3 * r2, -3 * z);
  PAIR(57, 5, 13 * z2 - r2, 26 * z, -1.0);
  PAIR(59, 6, z, 1.0, 0.0);
  PAIR(61, 7, 1.0, 0.0, 0.0);
  /* l = 8: B8.1-B8.17, slots 63..79 */
  put_zero(63, 6435 * z8 - 12012 * z6 * r2 + 6930 * z4 * r4 - 1260 * z2 * r6 + 35 * r8,
           51480 * z7 - 72072 * z5 * r2 + 27720 * z3 * r4 - 2520 * z * r6, -12012 * z6 + 13860 * z4 * r2 - 3780 * z2 * r4 + 140 * r6,
           x, y, z, b, g);
  PAIR(64, 1, 715 * z7 - 1001 * z5 * r2 + 385 * z3 * r4 - 35 * z * r6, 5005 * z6 - 5005 * z4 * r2 + 1155 * z2 * r4 - 35 * r6,
       -1001 * z5 + 770 * z3 * r2 - 105 * z * r4);
  PAIR(66, 2, 143 * z6 - 143 * z4 * r2 + 33 * z2 * r4 - r6, 858 * z5 - 572 * z3 * r2 + 66 * z * r4, -143 * z4 + 66 * z2 * r2 - 3 * r4);
  PAIR(68, 3, 39 * z5 - 26 * z3 * r2 + 3 * z * r4, 195 * z4 - 78 * z2 * r2 + 3 * r4, -26 * z3 + 6 * z * r2);
  PAIR(70, 4, 65 * z4 - 26 * z2 * r2 + r4, 260 * z3 - 52 * z * r2, -26 * z2 + 2 * r2);
  PAIR(72, 5, 5 * z3 - z * r2, 15 * z2 - r2, -z);
  PAIR(74, 6, 15 * z2 - r2, 30 * z, -1.0);
  PAIR(76, 7, z, 1.0, 0.0);
  PAIR(78, 8, 1.0, 0.0, 0.0);
#undef PAIR
}

/* b_lm polynomials (B1.1-B4.9) in flattened order lm = l*l-1+m, and their Cartesian gradients. */
static void blm_poly(double x, double y, double z, double *b, double (*g)[3]) {
  double r2 = x * x + y * y + z * z;
  double x2 = x * x, y2 = y * y, z2 = z * z;
  /* l = 1 */
  b[0] = z;  g[0][0] = 0; g[0][1] = 0; g[0][2] = 1;
  b[1] = x;  g[1][0] = 1; g[1][1] = 0; g[1][2] = 0;
  b[2] = y;  g[2][0] = 0; g[2][1] = 1; g[2][2] = 0;
  /* l = 2 */
  b[3] = 3 * z2 - r2;  g[3][0] = -2 * x; g[3][1] = -2 * y; g[3][2] = 4 * z;
  b[4] = x * z;        g[4][0] = z; g[4][1] = 0; g[4][2] = x;
  b[5] = y * z;        g[5][0] = 0; g[5][1] = z; g[5][2] = y;
  b[6] = x2 - y2;      g[6][0] = 2 * x; g[6][1] = -2 * y; g[6][2] = 0;
  b[7] = 2 * x * y;    g[7][0] = 2 * y; g[7][1] = 2 * x; g[7][2] = 0;
  /* l = 3 */
  b[8] = 5 * z2 * z - 3 * z * r2;
  g[8][0] = -6 * x * z; g[8][1] = -6 * y * z; g[8][2] = 9 * z2 - 3 * r2;
  b[9] = (5 * z2 - r2) * x;
  g[9][0] = (5 * z2 - r2) - 2 * x2; g[9][1] = -2 * x * y; g[9][2] = 8 * x * z;
  b[10] = (5 * z2 - r2) * y;
  g[10][0] = -2 * x * y; g[10][1] = (5 * z2 - r2) - 2 * y2; g[10][2] = 8 * y * z;
  b[11] = (x2 - y2) * z;
  g[11][0] = 2 * x * z; g[11][1] = -2 * y * z; g[11][2] = x2 - y2;
  b[12] = 2 * x * y * z;
  g[12][0] = 2 * y * z; g[12][1] = 2 * x * z; g[12][2] = 2 * x * y;
  b[13] = (x2 - 3 * y2) * x;
  g[13][0] = 3 * x2 - 3 * y2; g[13][1] = -6 * x * y; g[13][2] = 0;
  b[14] = (3 * x2 - y2) * y;
  g[14][0] = 6 * x * y; g[14][1] = 3 * x2 - 3 * y2; g[14][2] = 0;
  /* l = 4 */
  b[15] = 35 * z2 * z2 - 30 * z2 * r2 + 3 * r2 * r2;
  g[15][0] = -60 * z2 * x + 12 * r2 * x; g[15][1] = -60 * z2 * y + 12 * r2 * y;
  g[15][2] = 80 * z2 * z - 48 * z * r2;
  double p = 7 * z2 * z - 3 * z * r2;
  b[16] = p * x;
  g[16][0] = p - 6 * z * x2; g[16][1] = -6 * z * x * y; g[16][2] = (15 * z2 - 3 * r2) * x;
  b[17] = p * y;
  g[17][0] = -6 * z * x * y; g[17][1] = p - 6 * z * y2; g[17][2] = (15 * z2 - 3 * r2) * y;
  double w = 7 * z2 - r2;
  b[18] = w * (x2 - y2);
  g[18][0] = -2 * x * (x2 - y2) + 2 * x * w; g[18][1] = -2 * y * (x2 - y2) - 2 * y * w;
  g[18][2] = 12 * z * (x2 - y2);
  b[19] = w * 2 * x * y;
  g[19][0] = -4 * x2 * y + 2 * y * w; g[19][1] = -4 * x * y2 + 2 * x * w; g[19][2] = 24 * x * y * z;
  b[20] = (x2 * x - 3 * x * y2) * z;
  g[20][0] = (3 * x2 - 3 * y2) * z; g[20][1] = -6 * x * y * z; g[20][2] = x2 * x - 3 * x * y2;
  b[21] = (3 * x2 * y - y2 * y) * z;
  g[21][0] = 6 * x * y * z; g[21][1] = (3 * x2 - 3 * y2) * z; g[21][2] = 3 * x2 * y - y2 * y;
  b[22] = x2 * x2 - 6 * x2 * y2 + y2 * y2;
  g[22][0] = 4 * x2 * x - 12 * x * y2; g[22][1] = -12 * x2 * y + 4 * y2 * y; g[22][2] = 0;
  b[23] = 4 * x2 * x * y - 4 * x * y2 * y;
  g[23][0] = 12 * x2 * y - 4 * y2 * y; g[23][1] = 4 * x2 * x - 12 * x * y2; g[23][2] = 0;
  blm_poly_high(x, y, z, b, g);
}

static int l_of_lm(int lm) { int l = 1; while ((l + 1) * (l + 1) - 1 <= lm) ++l; return l; }

/* raw polynomials, exported for the harmonic / homogeneity pins */
void orc_blm_raw(double x, double y, double z, double *b, double *grad /*24*3*/) {
  double g[NLM_MAX][3];
  blm_poly(x, y, z, b, g);
  for (int i = 0; i < NLM_MAX; ++i) for (int c = 0; c < 3; ++c) grad[3 * i + c] = g[i][c];
}

/* B_lm = b_lm / d^l (B9.1) and grad B_lm = grad b_lm / d^l - l b_lm r / d^(l+2) (from B9.2) */
void orc_blm(double x, double y, double z, double *B, double *dB /*24*3*/) {
  double b[NLM_MAX], g[NLM_MAX][3];
  blm_poly(x, y, z, b, g);
  double d = sqrt(x * x + y * y + z * z);
  double r[3] = {x, y, z};
  for (int lm = 0; lm < NLM_MAX; ++lm) {
    int l = l_of_lm(lm);
    double dl = pow(d, (double)l);
    B[lm] = b[lm] / dl;
    for (int c = 0; c < 3; ++c) dB[3 * lm + c] = g[lm][c] / dl - l * b[lm] * r[c] / (dl * d * d);
  }
}

/* C_lm = kappa_l * Chat_lm, kappa_l = (2l+1)/(4 pi)  (S:8(c).4; the paper never prints them) */
void orc_clm(double *C) {
  /* one entry for m = 0, then one per (cos, sin) pair; derived from the addition theorem, pinned against scipy's Legendre */
  static const double chat[NLM_MAX] = {
      1, 1, 1,
      1.0 / 4, 3, 3, 3.0 / 4, 3.0 / 4,
      1.0 / 4, 3.0 / 8, 3.0 / 8, 15.0 / 4, 15.0 / 4, 5.0 / 8, 5.0 / 8,
      1.0 / 64, 5.0 / 8, 5.0 / 8, 5.0 / 16, 5.0 / 16, 35.0 / 8, 35.0 / 8, 35.0 / 64, 35.0 / 64,
      1.0 / 64, 15.0 / 64, 15.0 / 64, 105.0 / 16, 105.0 / 16, 35.0 / 128, 35.0 / 128, 315.0 / 64, 315.0 / 64, 63.0 / 128, 63.0 / 128,
      1.0 / 256, 21.0 / 64, 21.0 / 64, 105.0 / 512, 105.0 / 512, 105.0 / 128, 105.0 / 128, 63.0 / 256, 63.0 / 256, 693.0 / 128,
      693.0 / 128, 231.0 / 512, 231.0 / 512,
      1.0 / 256, 7.0 / 1024, 7.0 / 1024, 21.0 / 512, 21.0 / 512, 21.0 / 1024, 21.0 / 1024, 231.0 / 256, 231.0 / 256, 231.0 / 1024,
      231.0 / 1024, 3003.0 / 512, 3003.0 / 512, 429.0 / 1024, 429.0 / 1024,
      1.0 / 16384, 9.0 / 1024, 9.0 / 1024, 315.0 / 2048, 315.0 / 2048, 1155.0 / 1024, 1155.0 / 1024, 693.0 / 4096, 693.0 / 4096,
      9009.0 / 1024, 9009.0 / 1024, 429.0 / 2048, 429.0 / 2048, 6435.0 / 1024, 6435.0 / 1024, 6435.0 / 16384, 6435.0 / 16384};
  for (int lm = 0; lm < NLM_MAX; ++lm) {
    int l = l_of_lm(lm);
    C[lm] = (2 * l + 1) / (4.0 * M_PI) * chat[lm];
  }
}

/* 4-body cubic invariant of the l=2 moments (S:8(c).4): q4 = kappa4 * P4(s), P4 = 108 det M */
#define KAPPA4 (-5.0 * sqrt(14.0) / (448.0 * M_PI * sqrt(M_PI)))
double orc_kappa4(void) { return KAPPA4; }
double orc_p4(const double *s, double *g /*5 or NULL*/, double *H /*25 or NULL*/) {
  double s0 = s[0], s1 = s[1], s2 = s[2], s3 = s[3], s4 = s[4];
  double P = s0 * s0 * s0 + 18 * s0 * (s1 * s1 + s2 * s2) - 9 * s0 * (s3 * s3 + s4 * s4) +
             54 * s3 * (s1 * s1 - s2 * s2) + 108 * s1 * s2 * s4;
  if (g) {
    g[0] = 3 * s0 * s0 + 18 * (s1 * s1 + s2 * s2) - 9 * (s3 * s3 + s4 * s4);
    g[1] = 36 * s0 * s1 + 108 * s3 * s1 + 108 * s2 * s4;
    g[2] = 36 * s0 * s2 - 108 * s3 * s2 + 108 * s1 * s4;
    g[3] = -18 * s0 * s3 + 54 * (s1 * s1 - s2 * s2);
    g[4] = -18 * s0 * s4 + 108 * s1 * s2;
  }
  if (H) {
    double h[5][5] = {{6 * s0, 36 * s1, 36 * s2, -18 * s3, -18 * s4},
                      {36 * s1, 36 * s0 + 108 * s3, 108 * s4, 108 * s1, 108 * s2},
                      {36 * s2, 108 * s4, 36 * s0 - 108 * s3, -108 * s2, 108 * s1},
                      {-18 * s3, 108 * s1, -108 * s2, -18 * s0, 0},
                      {-18 * s4, 108 * s2, 108 * s1, 0, -18 * s0}};
    for (int a = 0; a < 5; ++a) for (int c = 0; c < 5; ++c) H[5 * a + c] = h[a][c];
  }
  return P;
}

/* 5-body term (named at P:65; not defined in the paper; R41): the only quartic rotational invariant of
 * the l = 1 moments v = (S_n10, S_n11, S_n12) = sum_j g_n(d_ij) (z, x, y)/d is |v|^4.  Normalised like the 4-body term
 * as the contraction of four orthonormal l = 1 moments coupled pairwise to zero, (1/3) (sum_m |A_1m|^2)^2 with
 * sum_m |A_1m|^2 = 3/(4 pi) |v|^2:   q5 = kappa5 |v|^4,  kappa5 = 3 / (16 pi^2)  (= q_{n,l=1}^2 / 3). */
#define KAPPA5 (3.0 / (16.0 * M_PI * M_PI))
double orc_kappa5(void) { return KAPPA5; }
double orc_p5(const double *s, double *g /*3 or NULL*/, double *H /*9 or NULL*/) {
  double n2 = s[0] * s[0] + s[1] * s[1] + s[2] * s[2];
  if (g) for (int a = 0; a < 3; ++a) g[a] = 4 * KAPPA5 * n2 * s[a];
  if (H)
    for (int a = 0; a < 3; ++a)
      for (int c = 0; c < 3; ++c) H[3 * a + c] = 4 * KAPPA5 * (n2 * (a == c ? 1.0 : 0.0) + 2 * s[a] * s[c]);
  return KAPPA5 * n2 * n2;
}

/* ------------------------------------------------------------------ neighbour sets (Eq.2; S:8(c).3) */
static void cross3(const double *a, const double *b, double *c) {
  c[0] = a[1] * b[2] - a[2] * b[1];
  c[1] = a[2] * b[0] - a[0] * b[2];
  c[2] = a[0] * b[1] - a[1] * b[0];
}
static double dot3(const double *a, const double *b) { return a[0] * b[0] + a[1] * b[1] + a[2] * b[2]; }

/* returns 0 ok, -1 degenerate cell */
static int cell_geometry(const double *c, double *inv /*9*/, double *h /*3*/) {
  const double *a = c, *b = c + 3, *cc = c + 6;
  double bxc[3], cxa[3], axb[3];
  cross3(b, cc, bxc); cross3(cc, a, cxa); cross3(a, b, axb);
  double V = dot3(a, bxc);
  if (!(fabs(V) > 0.0)) return -1;
  h[0] = fabs(V) / sqrt(dot3(bxc, bxc));
  h[1] = fabs(V) / sqrt(dot3(cxa, cxa));
  h[2] = fabs(V) / sqrt(dot3(axb, axb));
  /* pos = u_a a + u_b b + u_c c  ->  u_a = pos . (b x c)/V etc.; inv stored as columns */
  for (int k = 0; k < 3; ++k) { inv[0 * 3 + k] = bxc[k] / V; inv[1 * 3 + k] = cxa[k] / V; inv[2 * 3 + k] = axb[k] / V; }
  return 0;
}

/* One list (cutoff rc) of one structure. Brute force over every j and every image in the range
 * ceil(rc/h) per axis; exclude only (i, zero shift).  Row order ascending (j, sa, sb, sc). */
static int64_t build_list(int n, const double *pos, const double *c, double rc, const double *h,
                          int first_atom, int64_t *rptr, int *oj, int *osh, double *orr) {
  int na = (int)ceil(rc / h[0]), nb = (int)ceil(rc / h[1]), nc = (int)ceil(rc / h[2]);
  double rc2 = rc * rc;
  int64_t cnt = 0;
  for (int i = 0; i < n; ++i) {
    if (rptr) rptr[i] = cnt;
    for (int j = 0; j < n; ++j)
      for (int sa = -na; sa <= na; ++sa)
        for (int sb = -nb; sb <= nb; ++sb)
          for (int sc = -nc; sc <= nc; ++sc) {
            if (j == i && sa == 0 && sb == 0 && sc == 0) continue;
            /* fixed operation order, no FMA contraction (bit-exactness recipe, S:8(c).3) */
            double tx = (sa * c[0] + sb * c[3]) + sc * c[6];
            double ty = (sa * c[1] + sb * c[4]) + sc * c[7];
            double tz = (sa * c[2] + sb * c[5]) + sc * c[8];
            double dx = (pos[3 * j + 0] - pos[3 * i + 0]) + tx;
            double dy = (pos[3 * j + 1] - pos[3 * i + 1]) + ty;
            double dz = (pos[3 * j + 2] - pos[3 * i + 2]) + tz;
            double d2 = (dx * dx + dy * dy) + dz * dz;
            if (d2 < rc2) {
              if (oj) {
                oj[cnt] = first_atom + j;
                osh[3 * cnt + 0] = sa; osh[3 * cnt + 1] = sb; osh[3 * cnt + 2] = sc;
                orr[3 * cnt + 0] = dx; orr[3 * cnt + 1] = dy; orr[3 * cnt + 2] = dz;
              }
              ++cnt;
            }
          }
  }
  if (rptr) rptr[n] = cnt;
  return cnt;
}

void orc_batch_destroy(orc_batch *b) {
  if (!b) return;
  free(b->aoff); free(b->pos); free(b->cell); free(b->type);
  for (int w = 0; w < 2; ++w) { free(b->rptr[w]); free(b->nj[w]); free(b->nsh[w]); free(b->nr[w]); }
  free(b->Eref); free(b->Fref); free(b->Wref);
  free(b->we); free(b->wf); free(b->wv);
  free(b);
}

static double *dupd(const double *p, size_t n) {
  if (!p) return NULL;
  double *q = (double *)malloc(n * sizeof(double));
  memcpy(q, p, n * sizeof(double));
  return q;
}

/* Copies the inputs, wraps positions by whole lattice vectors, builds both lists. NULL on error. */
orc_batch *orc_batch_create(int S, const int32_t *aoff, const double *pos, const double *cell,
                            const int32_t *type, double rcR, double rcA, const double *Eref,
                            const double *Fref, const double *Wref) {
  orc_batch *b = (orc_batch *)calloc(1, sizeof(orc_batch));
  int N = aoff[S];
  b->S = S; b->N = N;
  b->aoff = (int *)malloc((S + 1) * sizeof(int));
  for (int s = 0; s <= S; ++s) b->aoff[s] = aoff[s];
  b->pos = dupd(pos, (size_t)3 * N);
  b->cell = dupd(cell, (size_t)9 * S);
  b->type = (int *)malloc((size_t)(N > 0 ? N : 1) * sizeof(int));
  for (int i = 0; i < N; ++i) b->type[i] = type[i];
  b->Eref = dupd(Eref, S); b->Fref = dupd(Fref, (size_t)3 * N); b->Wref = dupd(Wref, (size_t)6 * S);
  double rc[2] = {rcR, rcA};
  int64_t *cnt[2];
  for (int w = 0; w < 2; ++w) {
    b->rptr[w] = (int64_t *)calloc((size_t)N + 1, sizeof(int64_t));
    cnt[w] = (int64_t *)calloc((size_t)S + 1, sizeof(int64_t));
  }
  int bad = 0;
  /* wrap (S:8(c).3): subtract floor(u) lattice vectors, same operation order as the image shifts */
  for (int s = 0; s < S; ++s) {
    double inv[9], h[3];
    const double *c = b->cell + 9 * s;
    if (cell_geometry(c, inv, h)) { bad = 1; continue; }
    for (int i = b->aoff[s]; i < b->aoff[s + 1]; ++i) {
      double *p = b->pos + 3 * i;
      double ua = (p[0] * inv[0] + p[1] * inv[1]) + p[2] * inv[2];
      double ub = (p[0] * inv[3] + p[1] * inv[4]) + p[2] * inv[5];
      double uc = (p[0] * inv[6] + p[1] * inv[7]) + p[2] * inv[8];
      double fa = floor(ua), fb = floor(ub), fc = floor(uc);
      if (fa != 0.0 || fb != 0.0 || fc != 0.0) {
        p[0] = p[0] - ((fa * c[0] + fb * c[3]) + fc * c[6]);
        p[1] = p[1] - ((fa * c[1] + fb * c[4]) + fc * c[7]);
        p[2] = p[2] - ((fa * c[2] + fb * c[5]) + fc * c[8]);
      }
    }
  }
  if (bad) { for (int w = 0; w < 2; ++w) free(cnt[w]); orc_batch_destroy(b); return NULL; }
  /* count, then fill (two passes of the same brute-force loop) */
  for (int w = 0; w < 2; ++w) {
#pragma omp parallel for schedule(dynamic)
    for (int s = 0; s < S; ++s) {
      double inv[9], h[3];
      cell_geometry(b->cell + 9 * s, inv, h);
      int n = b->aoff[s + 1] - b->aoff[s];
      cnt[w][s + 1] = build_list(n, b->pos + 3 * b->aoff[s], b->cell + 9 * s, rc[w], h, b->aoff[s],
                                 NULL, NULL, NULL, NULL);
    }
    for (int s = 0; s < S; ++s) cnt[w][s + 1] += cnt[w][s];
    int64_t tot = cnt[w][S];
    b->nj[w] = (int *)malloc((size_t)(tot > 0 ? tot : 1) * sizeof(int));
    b->nsh[w] = (int *)malloc((size_t)(tot > 0 ? tot : 1) * 3 * sizeof(int));
    b->nr[w] = (double *)malloc((size_t)(tot > 0 ? tot : 1) * 3 * sizeof(double));
#pragma omp parallel for schedule(dynamic)
    for (int s = 0; s < S; ++s) {
      double inv[9], h[3];
      cell_geometry(b->cell + 9 * s, inv, h);
      int n = b->aoff[s + 1] - b->aoff[s];
      int64_t base = cnt[w][s];
      int64_t *tmp = (int64_t *)malloc((size_t)(n + 1) * sizeof(int64_t));
      build_list(n, b->pos + 3 * b->aoff[s], b->cell + 9 * s, rc[w], h, b->aoff[s], tmp,
                 b->nj[w] + base, b->nsh[w] + 3 * base, b->nr[w] + 3 * base);
      for (int i = 0; i < n; ++i) b->rptr[w][b->aoff[s] + i] = base + tmp[i];
      free(tmp);
    }
    b->rptr[w][N] = tot;
    free(cnt[w]);
  }
  return b;
}

int64_t orc_batch_num_pairs(const orc_batch *b, int which) { return b->rptr[which][b->N]; }
int orc_batch_num_atoms(const orc_batch *b) { return b->N; }
void orc_batch_get_positions(const orc_batch *b, double *pos) { memcpy(pos, b->pos, (size_t)3 * b->N * sizeof(double)); }
void orc_batch_get_neighbors(const orc_batch *b, int which, int64_t *rptr, int32_t *j, int32_t *sh,
                             double *r) {
  int64_t tot = b->rptr[which][b->N];
  if (rptr) memcpy(rptr, b->rptr[which], ((size_t)b->N + 1) * sizeof(int64_t));
  for (int64_t p = 0; p < tot; ++p) {
    if (j) j[p] = b->nj[which][p];
    if (sh) for (int c = 0; c < 3; ++c) sh[3 * p + c] = b->nsh[which][3 * p + c];
    if (r) for (int c = 0; c < 3; ++c) r[3 * p + c] = b->nr[which][3 * p + c];
  }
}
void orc_batch_set_refs(orc_batch *b, const double *Eref, const double *Fref, const double *Wref) {
  free(b->Eref); free(b->Fref); free(b->Wref);
  b->Eref = dupd(Eref, b->S); b->Fref = dupd(Fref, (size_t)3 * b->N); b->Wref = dupd(Wref, (size_t)6 * b->S);
}

/* Per-structure loss weights (R40; the paper's sets mix structures with and without virials, and
 * Eq.10-12 weigh every structure equally): a weight is the multiplicity of the structure in the training set, so a
 * term is the weighted mean  sum_s w_s (...)_s / sum_s w_s  (forces: / (3 sum_s w_s N_s)); w = 0 masks a missing
 * label, all ones (or NULL) is Eq.10-12 as printed.  Each array has S entries or is NULL. */
void orc_batch_set_weights(orc_batch *b, const double *we, const double *wf, const double *wv) {
  free(b->we); free(b->wf); free(b->wv);
  b->we = dupd(we, b->S); b->wf = dupd(wf, b->S); b->wv = dupd(wv, b->S);
}
static double wgt(const double *w, int s) { return w ? w[s] : 1.0; }
/* normalisers Z_E = sum w_e, Z_F = sum w_f N_s, Z_V = sum w_v  (= S, N, S without weights) */
static void weight_norms(const orc_batch *b, double *Z) {
  Z[0] = Z[1] = Z[2] = 0.0;
  for (int s = 0; s < b->S; ++s) {
    double Ns = b->aoff[s + 1] - b->aoff[s];
    Z[0] += wgt(b->we, s); Z[1] += wgt(b->wf, s) * Ns; Z[2] += wgt(b->wv, s);
  }
}

/* ------------------------------------------------------------------ per-atom forward pieces */
typedef struct {
  int Ndes, NLM, P;
  const double *cR, *cA;
  double C[NLM_MAX];
} ctx_t;

static void make_ctx(const orc_spec *sp, const double *theta, ctx_t *cx) {
  cx->Ndes = orc_ndes(sp); cx->NLM = orc_nlm(sp); cx->P = (int)orc_num_params(sp);
  cx->cR = theta + off_cR(sp); cx->cA = theta + off_cA(sp);
  orc_clm(cx->C);
}
static const double *net_W0(const orc_spec *sp, const double *theta, int t) { return theta + off_net(sp) + t * net_size(sp); }

/* g_n(d) = sum_k c[I][J][n][k] f_k(d)  (Eq.6) and its derivative */
static void radial_fn(const double *c, int T, int Nf, int K, int I, int J, const double *f,
                      const double *fp, double *g, double *gp) {
  for (int n = 0; n < Nf; ++n) {
    const double *cn = c + (((int64_t)I * T + J) * Nf + n) * K;
    double a = 0, b = 0;
    for (int k = 0; k < K; ++k) { a += cn[k] * f[k]; b += cn[k] * fp[k]; }
    g[n] = a; gp[n] = b;
  }
}

/* Descriptor of atom i (unscaled q, Ndes entries) and its S_nlm (NA*24) */
static void atom_descriptor(const orc_spec *sp, const ctx_t *cx, const orc_batch *b, int i, double *q,
                            double *Snlm) {
  int I = b->type[i];
  double f[KMAX], fp[KMAX], g[KMAX], gp[KMAX];
  for (int v = 0; v < cx->Ndes; ++v) q[v] = 0.0;
  for (int x = 0; x < sp->NA * NLM_MAX; ++x) Snlm[x] = 0.0;
  /* radial, Eq.5 */
  for (int64_t p = b->rptr[0][i]; p < b->rptr[0][i + 1]; ++p) {
    const double *r = b->nr[0] + 3 * p;
    double d = sqrt(dot3(r, r));
    orc_basis(sp->rcR, sp->KR, d, f, fp);
    radial_fn(cx->cR, sp->T, sp->NR, sp->KR, I, b->type[b->nj[0][p]], f, fp, g, gp);
    for (int n = 0; n < sp->NR; ++n) q[n] += g[n];
  }
  /* angular, Eq.8 then Eq.7 */
  for (int64_t p = b->rptr[1][i]; p < b->rptr[1][i + 1]; ++p) {
    const double *r = b->nr[1] + 3 * p;
    double d = sqrt(dot3(r, r));
    double B[NLM_MAX], dB[NLM_MAX * 3];
    orc_basis(sp->rcA, sp->KA, d, f, fp);
    radial_fn(cx->cA, sp->T, sp->NA, sp->KA, I, b->type[b->nj[1][p]], f, fp, g, gp);
    orc_blm(r[0], r[1], r[2], B, dB);
    for (int n = 0; n < sp->NA; ++n)
      for (int lm = 0; lm < cx->NLM; ++lm) Snlm[n * NLM_MAX + lm] += g[n] * B[lm];
  }
  for (int n = 0; n < sp->NA; ++n) {
    for (int lm = 0; lm < cx->NLM; ++lm) {
      int l = l_of_lm(lm);
      double s = Snlm[n * NLM_MAX + lm];
      q[sp->NR + (l - 1) * sp->NA + n] += cx->C[lm] * s * s;
    }
    if (sp->use4) q[sp->NR + sp->L * sp->NA + n] = KAPPA4 * orc_p4(Snlm + n * NLM_MAX + 3, NULL, NULL);
    if (sp->use5) q[off5(sp) + n] = orc_p5(Snlm + n * NLM_MAX, NULL, NULL);
  }
}

/* Network of species t at scaled input G: E, x_mu, E'_nu = dE/dq_nu (includes q_scale) (D1.1-D1.5) */
static double atom_network(const orc_spec *sp, const ctx_t *cx, const double *theta, const double *qs,
                           int t, const double *q, double *x, double *Ep) {
  int Nd = cx->Ndes, Nn = sp->Nn;
  const double *W0 = net_W0(sp, theta, t), *b0 = W0 + (int64_t)Nn * Nd, *w1 = b0 + Nn, *b1 = w1 + Nn;
  double E = b1[0];
  for (int v = 0; v < Nd; ++v) Ep[v] = 0.0;
  for (int m = 0; m < Nn; ++m) {
    double z = b0[m];
    for (int v = 0; v < Nd; ++v) z += W0[(int64_t)m * Nd + v] * (qs[v] * q[v]);
    x[m] = tanh(z);
    E += w1[m] * x[m];
    double d1 = 1.0 - x[m] * x[m];
    for (int v = 0; v < Nd; ++v) Ep[v] += qs[v] * w1[m] * d1 * W0[(int64_t)m * Nd + v];
  }
  return E;
}

/* beta_nlm = sum_{nu in n} E'_nu dq_nu/dS_nlm   (S:8(c).6) */
static void atom_beta(const orc_spec *sp, const ctx_t *cx, const double *Ep, const double *Snlm,
                      double *beta) {
  for (int n = 0; n < sp->NA; ++n) {
    for (int lm = 0; lm < NLM_MAX; ++lm) beta[n * NLM_MAX + lm] = 0.0;
    for (int lm = 0; lm < cx->NLM; ++lm) {
      int l = l_of_lm(lm);
      beta[n * NLM_MAX + lm] = Ep[sp->NR + (l - 1) * sp->NA + n] * 2.0 * cx->C[lm] * Snlm[n * NLM_MAX + lm];
    }
    if (sp->use4) {
      double g4[5];
      orc_p4(Snlm + n * NLM_MAX + 3, g4, NULL);
      for (int m = 0; m < 5; ++m) beta[n * NLM_MAX + 3 + m] += Ep[sp->NR + sp->L * sp->NA + n] * KAPPA4 * g4[m];
    }
    if (sp->use5) {
      double g5[3];
      orc_p5(Snlm + n * NLM_MAX, g5, NULL);
      for (int m = 0; m < 3; ++m) beta[n * NLM_MAX + m] += Ep[off5(sp) + n] * g5[m];
    }
  }
}

/* workspace for one structure */
typedef struct { double *q, *S, *x, *Ep, *Ei; } swork;
static void swork_alloc(swork *w, const orc_spec *sp, int nmax) {
  int Nd = orc_ndes(sp);
  w->q = (double *)malloc((size_t)nmax * Nd * sizeof(double));
  w->S = (double *)malloc((size_t)nmax * sp->NA * NLM_MAX * sizeof(double));
  w->x = (double *)malloc((size_t)nmax * sp->Nn * sizeof(double));
  w->Ep = (double *)malloc((size_t)nmax * Nd * sizeof(double));
  w->Ei = (double *)malloc((size_t)nmax * sizeof(double));
}
static void swork_free(swork *w) { free(w->q); free(w->S); free(w->x); free(w->Ep); free(w->Ei); }

/* Forward for structure s: fills w (per atom of s), and if F!=NULL accumulates E_s, F (global
 * indexing) and W_s (6: xx,yy,zz,xy,yz,zx).  Eq.1, C3.6, Eq.3, Eq.4 (S:8(c).6-7). */
static void structure_forward(const orc_spec *sp, const ctx_t *cx, const double *theta, const double *qs,
                              const orc_batch *b, int s, swork *w, double *Es, double *F, double *Ws) {
  int a0 = b->aoff[s], a1 = b->aoff[s + 1], Nd = cx->Ndes;
  double E = 0.0;
  for (int i = a0; i < a1; ++i) {
    int li = i - a0;
    atom_descriptor(sp, cx, b, i, w->q + (size_t)li * Nd, w->S + (size_t)li * sp->NA * NLM_MAX);
    w->Ei[li] = atom_network(sp, cx, theta, qs, b->type[i], w->q + (size_t)li * Nd,
                             w->x + (size_t)li * sp->Nn, w->Ep + (size_t)li * Nd);
    E += w->Ei[li];
  }
  if (Es) *Es = E;
  if (!F) return;
  double W[6] = {0, 0, 0, 0, 0, 0};
  double f[KMAX], fp[KMAX], g[KMAX], gp[KMAX];
  double *beta = (double *)malloc((size_t)sp->NA * NLM_MAX * sizeof(double));
  for (int i = a0; i < a1; ++i) {
    int li = i - a0, I = b->type[i];
    const double *Ep = w->Ep + (size_t)li * Nd;
    for (int list = 0; list < 2; ++list) {
      if (list == 1) atom_beta(sp, cx, Ep, w->S + (size_t)li * sp->NA * NLM_MAX, beta);
      for (int64_t p = b->rptr[list][i]; p < b->rptr[list][i + 1]; ++p) {
        const double *r = b->nr[list] + 3 * p;
        int j = b->nj[list][p];
        double d = sqrt(dot3(r, r));
        double fij[3] = {0, 0, 0};
        if (list == 0) {   /* radial part: sum_n E'_n g_n'(d) rhat */
          orc_basis(sp->rcR, sp->KR, d, f, fp);
          radial_fn(cx->cR, sp->T, sp->NR, sp->KR, I, b->type[j], f, fp, g, gp);
          double sc = 0;
          for (int n = 0; n < sp->NR; ++n) sc += Ep[n] * gp[n];
          for (int c = 0; c < 3; ++c) fij[c] = sc * r[c] / d;
        } else {           /* angular part: sum_n sum_lm beta_nlm dS_nlm/dr_ij (C2.3) */
          double B[NLM_MAX], dB[NLM_MAX * 3];
          orc_basis(sp->rcA, sp->KA, d, f, fp);
          radial_fn(cx->cA, sp->T, sp->NA, sp->KA, I, b->type[j], f, fp, g, gp);
          orc_blm(r[0], r[1], r[2], B, dB);
          for (int n = 0; n < sp->NA; ++n)
            for (int lm = 0; lm < cx->NLM; ++lm) {
              double be = beta[n * NLM_MAX + lm];
              for (int c = 0; c < 3; ++c) fij[c] += be * (gp[n] * B[lm] * r[c] / d + g[n] * dB[3 * lm + c]);
            }
        }
        for (int c = 0; c < 3; ++c) { F[3 * i + c] += fij[c]; F[3 * j + c] -= fij[c]; }
        W[0] -= r[0] * fij[0]; W[1] -= r[1] * fij[1]; W[2] -= r[2] * fij[2];
        W[3] -= r[0] * fij[1]; W[4] -= r[1] * fij[2]; W[5] -= r[2] * fij[0];
      }
    }
  }
  free(beta);
  for (int c = 0; c < 6; ++c) Ws[c] = W[c];
}

static int max_struct_atoms(const orc_batch *b) {
  int m = 1;
  for (int s = 0; s < b->S; ++s) if (b->aoff[s + 1] - b->aoff[s] > m) m = b->aoff[s + 1] - b->aoff[s];
  return m;
}

/* unscaled descriptors q[N][Ndes] */
void orc_descriptors(const orc_spec *sp, const double *theta, const orc_batch *b, double *q) {
  ctx_t cx; make_ctx(sp, theta, &cx);
#pragma omp parallel
  {
    double *S = (double *)malloc((size_t)sp->NA * NLM_MAX * sizeof(double));
#pragma omp for schedule(dynamic, 16)
    for (int i = 0; i < b->N; ++i) atom_descriptor(sp, &cx, b, i, q + (size_t)i * cx.Ndes, S);
    free(S);
  }
}

/* network pin aid: E, E'(Ndes, wrt unscaled q), and the Hessian-vector product (E'' D) */
double orc_network(const orc_spec *sp, const double *theta, const double *qs, int t, const double *q,
                   double *Ep, const double *D, double *h) {
  ctx_t cx; make_ctx(sp, theta, &cx);
  int Nd = cx.Ndes, Nn = sp->Nn;
  double *x = (double *)malloc((size_t)Nn * sizeof(double));
  double E = atom_network(sp, &cx, theta, qs, t, q, x, Ep);
  if (D && h) {
    const double *W0 = net_W0(sp, theta, t), *w1 = W0 + (int64_t)Nn * Nd + Nn;
    for (int v = 0; v < Nd; ++v) h[v] = 0.0;
    for (int m = 0; m < Nn; ++m) {                         /* D1.6 contracted with D */
      double pm = 0;
      for (int v = 0; v < Nd; ++v) pm += W0[(int64_t)m * Nd + v] * qs[v] * D[v];
      double d2 = -2.0 * x[m] * (1.0 - x[m] * x[m]);
      for (int v = 0; v < Nd; ++v) h[v] += qs[v] * w1[m] * d2 * pm * W0[(int64_t)m * Nd + v];
    }
  }
  free(x);
  return E;
}

/* E_s[S], F[N*3], W_s[S*6] */
void orc_predict(const orc_spec *sp, const double *theta, const double *qs, const orc_batch *b,
                 double *Es, double *F, double *Ws) {
  ctx_t cx; make_ctx(sp, theta, &cx);
  for (int64_t x = 0; x < (int64_t)3 * b->N; ++x) F[x] = 0.0;
  int nmax = max_struct_atoms(b);
#pragma omp parallel
  {
    swork w; swork_alloc(&w, sp, nmax);
#pragma omp for schedule(dynamic)
    for (int s = 0; s < b->S; ++s)   /* F of different structures never alias */
      structure_forward(sp, &cx, theta, qs, b, s, &w, Es + s, F, Ws + 6 * s);
    swork_free(&w);
  }
}

/* loss terms from predictions: terms = {L, t_e, t_f, t_v, t_2}  (Eq.9-12; S:8(c).8; weights R40) */
static void loss_terms(const orc_spec *sp, const double *theta, const orc_batch *b, const double *Es,
                       const double *F, const double *Ws, double *terms) {
  int64_t P = orc_num_params(sp);
  double te = 0, tf = 0, tv = 0, t2 = 0, Z[3];
  weight_norms(b, Z);
  if (b->Eref && Z[0] > 0) {
    for (int s = 0; s < b->S; ++s) {
      double Ns = b->aoff[s + 1] - b->aoff[s];
      double dE = Es[s] / Ns - b->Eref[s] / Ns;
      te += wgt(b->we, s) * dE * dE;
    }
    te /= Z[0];
  }
  if (b->Fref && Z[1] > 0) {
    for (int s = 0; s < b->S; ++s)
      for (int64_t x = (int64_t)3 * b->aoff[s]; x < (int64_t)3 * b->aoff[s + 1]; ++x) {
        double d = F[x] - b->Fref[x];
        tf += wgt(b->wf, s) * d * d;
      }
    tf /= 3.0 * Z[1];
  }
  if (b->Wref && Z[2] > 0) {
    for (int s = 0; s < b->S; ++s) {
      double Ns = b->aoff[s + 1] - b->aoff[s];
      for (int c = 0; c < 6; ++c) { double d = (Ws[6 * s + c] - b->Wref[6 * s + c]) / Ns; tv += wgt(b->wv, s) * d * d; }
    }
    tv /= 6.0 * Z[2];
  }
  for (int64_t p = 0; p < P; ++p) t2 += theta[p] * theta[p];
  t2 /= (double)P;
  terms[1] = te; terms[2] = tf; terms[3] = tv; terms[4] = t2;
  if (sp->loss_mode == 0) terms[0] = sp->lam_e * te + sp->lam_f * tf + sp->lam_v * tv + sp->lam_2 * t2;
  else terms[0] = sp->lam_e * sqrt(te) + sp->lam_f * sqrt(tf) + sp->lam_v * sqrt(tv) + sp->lam_2 * sqrt(t2);
}

/* the plain loss L(theta): predictions, then Eq.9-12.  This is what the finite differences use. */
void orc_loss(const orc_spec *sp, const double *theta, const double *qs, const orc_batch *b, double *terms) {
  double *Es = (double *)malloc((size_t)(b->S + 1) * sizeof(double));
  double *F = (double *)malloc((size_t)(3 * b->N + 1) * sizeof(double));
  double *Ws = (double *)malloc((size_t)(6 * b->S + 1) * sizeof(double));
  orc_predict(sp, theta, qs, b, Es, F, Ws);
  loss_terms(sp, theta, b, Es, F, Ws, terms);
  free(Es); free(F); free(Ws);
}

/* Analytic gradient, contraction-first form of App.C/D (S:8(c).9 steps 1-7). grad[P], terms[5]. */
void orc_loss_and_grad(const orc_spec *sp, const double *theta, const double *qs, const orc_batch *b,
                       double *terms, double *grad) {
  ctx_t cx; make_ctx(sp, theta, &cx);
  int64_t P = orc_num_params(sp);
  int Nd = cx.Ndes, Nn = sp->Nn, NA = sp->NA, NR = sp->NR, T = sp->T;
  double *Es = (double *)malloc((size_t)(b->S + 1) * sizeof(double));
  double *F = (double *)malloc((size_t)(3 * b->N + 1) * sizeof(double));
  double *Ws = (double *)malloc((size_t)(6 * b->S + 1) * sizeof(double));
  orc_predict(sp, theta, qs, b, Es, F, Ws);
  loss_terms(sp, theta, b, Es, F, Ws, terms);
  /* step 1: seeds.  mode 1 multiplies each term's seed by 1/(2 sqrt(t_x)) (guard t_x = 0) */
  double me = 1, mf = 1, mv = 1, m2 = 1;
  if (sp->loss_mode == 1) {
    me = terms[1] > 0 ? 0.5 / sqrt(terms[1]) : 0; mf = terms[2] > 0 ? 0.5 / sqrt(terms[2]) : 0;
    mv = terms[3] > 0 ? 0.5 / sqrt(terms[3]) : 0; m2 = terms[4] > 0 ? 0.5 / sqrt(terms[4]) : 0;
  }
  double Z[3];
  weight_norms(b, Z);
  double *u = (double *)calloc((size_t)3 * b->N + 1, sizeof(double));
  if (b->Fref && Z[1] > 0)
    for (int s = 0; s < b->S; ++s)
      for (int64_t x = (int64_t)3 * b->aoff[s]; x < (int64_t)3 * b->aoff[s + 1]; ++x)
        u[x] = mf * 2.0 * sp->lam_f * wgt(b->wf, s) * (F[x] - b->Fref[x]) / (3.0 * Z[1]);
  for (int64_t p = 0; p < P; ++p) grad[p] = 0.0;
  int nmax = max_struct_atoms(b);
#pragma omp parallel
  {
    double *gl = (double *)calloc((size_t)P, sizeof(double));   /* thread-local gradient */
    swork w; swork_alloc(&w, sp, nmax);
    double *Dv = (double *)malloc((size_t)Nd * sizeof(double));
    double *Tn = (double *)malloc((size_t)NA * NLM_MAX * sizeof(double));
    double *pm = (double *)malloc((size_t)Nn * sizeof(double));
    double *gbar = (double *)malloc((size_t)Nd * sizeof(double));
    double *alpha = (double *)malloc((size_t)NA * NLM_MAX * sizeof(double));
    double *beta = (double *)malloc((size_t)NA * NLM_MAX * sizeof(double));
    double f[KMAX], fp[KMAX], g[KMAX], gp[KMAX];
#pragma omp for schedule(dynamic)
    for (int s = 0; s < b->S; ++s) {
      int a0 = b->aoff[s], a1 = b->aoff[s + 1];
      double Ns = a1 - a0;
      structure_forward(sp, &cx, theta, qs, b, s, &w, NULL, NULL, NULL);
      double e = 0.0, om[6] = {0, 0, 0, 0, 0, 0};
      if (b->Eref && Z[0] > 0) e = me * 2.0 * sp->lam_e * wgt(b->we, s) * (Es[s] / Ns - b->Eref[s] / Ns) / (Z[0] * Ns);
      if (b->Wref && Z[2] > 0)
        for (int c = 0; c < 6; ++c)
          om[c] = mv * 2.0 * sp->lam_v * wgt(b->wv, s) * ((Ws[6 * s + c] - b->Wref[6 * s + c]) / Ns) / (6.0 * Z[2] * Ns);
      for (int i = a0; i < a1; ++i) {
        int li = i - a0, I = b->type[i];
        const double *q = w.q + (size_t)li * Nd, *Sn = w.S + (size_t)li * NA * NLM_MAX;
        const double *x = w.x + (size_t)li * Nn, *Ep = w.Ep + (size_t)li * Nd;
        for (int v = 0; v < Nd; ++v) Dv[v] = 0.0;
        for (int z = 0; z < NA * NLM_MAX; ++z) Tn[z] = 0.0;
        /* steps 2-3: pair adjoint a_ij and directional derivatives D, T */
        for (int list = 0; list < 2; ++list)
          for (int64_t p = b->rptr[list][i]; p < b->rptr[list][i + 1]; ++p) {
            const double *r = b->nr[list] + 3 * p;
            int j = b->nj[list][p];
            double d = sqrt(dot3(r, r));
            double a[3];
            a[0] = u[3 * i + 0] - u[3 * j + 0] - (om[0] * r[0] + om[5] * r[2]);
            a[1] = u[3 * i + 1] - u[3 * j + 1] - (om[1] * r[1] + om[3] * r[0]);
            a[2] = u[3 * i + 2] - u[3 * j + 2] - (om[2] * r[2] + om[4] * r[1]);
            double ar = (a[0] * r[0] + a[1] * r[1] + a[2] * r[2]) / d;
            if (list == 0) {
              orc_basis(sp->rcR, sp->KR, d, f, fp);
              radial_fn(cx.cR, T, NR, sp->KR, I, b->type[j], f, fp, g, gp);
              for (int n = 0; n < NR; ++n) Dv[n] += gp[n] * ar;
            } else {
              double B[NLM_MAX], dB[NLM_MAX * 3];
              orc_basis(sp->rcA, sp->KA, d, f, fp);
              radial_fn(cx.cA, T, NA, sp->KA, I, b->type[j], f, fp, g, gp);
              orc_blm(r[0], r[1], r[2], B, dB);
              for (int n = 0; n < NA; ++n)
                for (int lm = 0; lm < cx.NLM; ++lm) {
                  double dBa = dB[3 * lm] * a[0] + dB[3 * lm + 1] * a[1] + dB[3 * lm + 2] * a[2];
                  Tn[n * NLM_MAX + lm] += gp[n] * B[lm] * ar + g[n] * dBa;
                }
            }
          }
        for (int n = 0; n < NA; ++n) {
          for (int lm = 0; lm < cx.NLM; ++lm) {
            int l = l_of_lm(lm);
            Dv[NR + (l - 1) * NA + n] += 2.0 * cx.C[lm] * Sn[n * NLM_MAX + lm] * Tn[n * NLM_MAX + lm];
          }
          if (sp->use4) {
            double g4[5], acc = 0;
            orc_p4(Sn + n * NLM_MAX + 3, g4, NULL);
            for (int m = 0; m < 5; ++m) acc += g4[m] * Tn[n * NLM_MAX + 3 + m];
            Dv[NR + sp->L * NA + n] = KAPPA4 * acc;
          }
          if (sp->use5) {
            double g5[3], acc = 0;
            orc_p5(Sn + n * NLM_MAX, g5, NULL);
            for (int m = 0; m < 3; ++m) acc += g5[m] * Tn[n * NLM_MAX + m];
            Dv[off5(sp) + n] = acc;
          }
        }
        /* step 4: network (species I) */
        {
          int64_t o = off_net(sp) + I * net_size(sp);
          const double *W0 = theta + o, *w1 = W0 + (int64_t)Nn * Nd + Nn;
          double *gW0 = gl + o, *gb0 = gW0 + (int64_t)Nn * Nd, *gw1 = gb0 + Nn, *gb1 = gw1 + Nn;
          for (int v = 0; v < Nd; ++v) gbar[v] = e * Ep[v];
          for (int m = 0; m < Nn; ++m) {
            double d1 = 1.0 - x[m] * x[m], d2 = -2.0 * x[m] * d1;
            double pv = 0;
            for (int v = 0; v < Nd; ++v) pv += W0[(int64_t)m * Nd + v] * qs[v] * Dv[v];
            pm[m] = pv;
            gw1[m] += e * x[m] + d1 * pv;                         /* D1.7 + D1.13 */
            double A = e * w1[m] * d1 + w1[m] * d2 * pv;          /* D1.10 + D1.17 */
            gb0[m] += A;
            for (int v = 0; v < Nd; ++v)                          /* D1.9 + D1.14 */
              gW0[(int64_t)m * Nd + v] += A * (qs[v] * q[v]) + w1[m] * d1 * qs[v] * Dv[v];
            for (int v = 0; v < Nd; ++v)                          /* h = E'' D  (D1.6, C3.8) */
              gbar[v] += qs[v] * w1[m] * d2 * pv * W0[(int64_t)m * Nd + v];
          }
          gb1[0] += e;                                            /* D1.8 (+ D1.15 = 0) */
        }
        /* step 6 prerequisites: alpha, beta */
        atom_beta(sp, &cx, Ep, Sn, beta);
        for (int n = 0; n < NA; ++n) {
          for (int lm = 0; lm < NLM_MAX; ++lm) alpha[n * NLM_MAX + lm] = 0.0;
          for (int lm = 0; lm < cx.NLM; ++lm) {
            int l = l_of_lm(lm), v = NR + (l - 1) * NA + n;
            alpha[n * NLM_MAX + lm] = gbar[v] * 2.0 * cx.C[lm] * Sn[n * NLM_MAX + lm] +
                                      Ep[v] * 2.0 * cx.C[lm] * Tn[n * NLM_MAX + lm];
          }
          if (sp->use4) {
            int v = NR + sp->L * NA + n;
            double g4[5], H4[25];
            orc_p4(Sn + n * NLM_MAX + 3, g4, H4);
            for (int m = 0; m < 5; ++m) {
              double ht = 0;
              for (int m2i = 0; m2i < 5; ++m2i) ht += H4[5 * m + m2i] * Tn[n * NLM_MAX + 3 + m2i];
              alpha[n * NLM_MAX + 3 + m] += gbar[v] * KAPPA4 * g4[m] + Ep[v] * KAPPA4 * ht;
            }
          }
          if (sp->use5) {
            int v = off5(sp) + n;
            double g5[3], H5[9];
            orc_p5(Sn + n * NLM_MAX, g5, H5);
            for (int m = 0; m < 3; ++m) {
              double ht = 0;
              for (int m2i = 0; m2i < 3; ++m2i) ht += H5[3 * m + m2i] * Tn[n * NLM_MAX + m2i];
              alpha[n * NLM_MAX + m] += gbar[v] * g5[m] + Ep[v] * ht;
            }
          }
        }
        /* steps 5-6: expansion-coefficient gradients, pair by pair */
        for (int list = 0; list < 2; ++list)
          for (int64_t p = b->rptr[list][i]; p < b->rptr[list][i + 1]; ++p) {
            const double *r = b->nr[list] + 3 * p;
            int j = b->nj[list][p], J = b->type[j];
            double d = sqrt(dot3(r, r));
            double a[3];
            a[0] = u[3 * i + 0] - u[3 * j + 0] - (om[0] * r[0] + om[5] * r[2]);
            a[1] = u[3 * i + 1] - u[3 * j + 1] - (om[1] * r[1] + om[3] * r[0]);
            a[2] = u[3 * i + 2] - u[3 * j + 2] - (om[2] * r[2] + om[4] * r[1]);
            double ar = (a[0] * r[0] + a[1] * r[1] + a[2] * r[2]) / d;
            if (list == 0) {
              orc_basis(sp->rcR, sp->KR, d, f, fp);
              double *gc = gl + off_cR(sp) + ((int64_t)I * T + J) * NR * sp->KR;
              for (int n = 0; n < NR; ++n)
                for (int k = 0; k < sp->KR; ++k) gc[n * sp->KR + k] += gbar[n] * f[k] + Ep[n] * fp[k] * ar;
            } else {
              double B[NLM_MAX], dB[NLM_MAX * 3];
              orc_basis(sp->rcA, sp->KA, d, f, fp);
              orc_blm(r[0], r[1], r[2], B, dB);
              double *gc = gl + off_cA(sp) + ((int64_t)I * T + J) * NA * sp->KA;
              for (int n = 0; n < NA; ++n) {
                double U = 0, V = 0;
                for (int lm = 0; lm < cx.NLM; ++lm) {
                  double dBa = dB[3 * lm] * a[0] + dB[3 * lm + 1] * a[1] + dB[3 * lm + 2] * a[2];
                  U += alpha[n * NLM_MAX + lm] * B[lm] + beta[n * NLM_MAX + lm] * dBa;
                  V += beta[n * NLM_MAX + lm] * B[lm];
                }
                V *= ar;
                for (int k = 0; k < sp->KA; ++k) gc[n * sp->KA + k] += U * f[k] + V * fp[k];
              }
            }
          }
      }
    }
#pragma omp critical
    for (int64_t p = 0; p < P; ++p) grad[p] += gl[p];
    free(gl); swork_free(&w); free(Dv); free(Tn); free(pm); free(gbar); free(alpha); free(beta);
  }
  /* step 7: regulariser */
  for (int64_t p = 0; p < P; ++p) grad[p] += m2 * 2.0 * sp->lam_2 * theta[p] / (double)P;
  free(Es); free(F); free(Ws); free(u);
}

/* Textbook Adam with bias correction; step is the 1-based step index t (S:8(c).11) */
void orc_adam_step(int64_t P, double *theta, double *m, double *v, const double *grad, int64_t step,
                   double lr, double beta1, double beta2, double eps) {
  double c1 = 1.0 - pow(beta1, (double)step), c2 = 1.0 - pow(beta2, (double)step);
  for (int64_t p = 0; p < P; ++p) {
    m[p] = beta1 * m[p] + (1.0 - beta1) * grad[p];
    v[p] = beta2 * v[p] + (1.0 - beta2) * grad[p] * grad[p];
    double mh = m[p] / c1, vh = v[p] / c2;
    theta[p] -= lr * mh / (sqrt(vh) + eps);
  }
}
