/* ORACLE -- TEST INFRASTRUCTURE ONLY.  Not part of the product path.
 *
 * Plain, slow, fp64 CPU implementation of the far-field mobility product M.[F,T,S] -> [U,Omega,E]
 * of Spectral Ewald Accelerated Stokesian Dynamics (Wang & Brady, arXiv 1506.08481; "PAPER.md").
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may call it.
 * It shares no code with paper_1506_08481_b200/ (the CUDA path) and neither includes the other.
 *
 * Two oracles:
 *   O1  o1_apply   -- the DEFINITION: direct Ewald sum, all lattice images within a cube of images and
 *                     all wave vectors within a cube of modes, no grid.  Tiny N only.
 *                     PAPER.md Eq. 13-15 (Faxen laws), Eq. 17 (multipole expansion), Eq. 19-23 (periodic
 *                     Stokeslet and its Hasimoto/Ewald split), Eq. 24-34 (compressible extension),
 *                     Eq. 35-37 (wave-space sum and its self term).
 *   O2  o2_apply   -- the ALGORITHM step by step: real-space pair sum over a cell list with cutoff r_c
 *                     (Sec. 3.3) + Spectral Ewald wave-space sum, hybrid size-effect variant
 *                     (Sec. 3.1-3.2: Eq. 41-46, Eq. 48, Eq. 50-52 and the "third approach"
 *                     paragraph) + self and one-body terms.  This is what the CUDA path is held to.
 *
 * Conventions: inputs are the moments the particles exert ON THE
 * FLUID, (F,T,S) = -(F^H,T^H,S^H) of Eq. 7-9; outputs are (U-U^inf, Omega-Omega^inf, -E^inf) of Eq. 11.
 * S and E are symmetric traceless, stored as 5 components (xx,xy,xz,yy,yz), zz = -(xx+yy).
 * The pressure moment s (compressible extension) keeps the paper's Eq. 25-26 sign.
 *
 * Everything in the real-space sum is generated mechanically from the Hasimoto screening function
 *     Phi(r) = r erfc(xi r) - exp(-xi^2 r^2)/(xi sqrt(pi))                            [Eq. 22]
 * by a small symbolic algebra on functions of the form
 *     sum_e  ce[e] erfc(xi r) r^e  +  sum_{e,p} cg[e][p] xi^p r^e exp(-xi^2 r^2)/sqrt(pi)
 * with INTEGER coefficients, closed under (1/r)d/dr and the radial Laplacian.  Cartesian derivative
 * tensors of a radial function psi follow from psi_n = ((1/r)d/dr)^n psi:
 *     d_a psi = x_a psi_1;  d_a d_b psi = delta_ab psi_1 + x_a x_b psi_2;  (and so on to rank 4).
 * No hand-expanded pair formulas appear in this file.
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

/* ------------------------------------------------------------------------------------------------
 * Symbolic radial functions
 * ---------------------------------------------------------------------------------------------- */
#define EOFF 14               /* index e <-> r^(e - EOFF) */
#define NE 24
#define POFF 1                /* index p <-> xi^(p - POFF) */
#define NPW 20

typedef struct { double ce[NE]; double cg[NE][NPW]; } rsym;   /* integer-valued coefficients */
typedef struct { double ce[NE]; double cg[NE]; } rnum;        /* numeric at a given xi        */

static void rsym_zero(rsym *f) { memset(f, 0, sizeof(*f)); }

/* o = (1/r) d/dr f.
 *   (1/r) d/dr [erfc(xi r) r^e]        = e erfc(xi r) r^(e-2) - (2 xi/sqrt(pi)) exp(-xi^2 r^2) r^(e-1)
 *   (1/r) d/dr [exp(-xi^2 r^2) r^e]    = e exp(-xi^2 r^2) r^(e-2) - 2 xi^2 exp(-xi^2 r^2) r^e          */
static void rsym_D1(const rsym *f, rsym *o)
{
    rsym t; rsym_zero(&t);
    for (int k = 0; k < NE; ++k) {
        const double e = (double)(k - EOFF);
        if (f->ce[k] != 0.0) {
            if (k < 2) abort();
            t.ce[k - 2] += e * f->ce[k];
            t.cg[k - 1][1 + POFF] += -2.0 * f->ce[k];
        }
        for (int p = 0; p < NPW; ++p) if (f->cg[k][p] != 0.0) {
            if (k < 2 || p + 2 >= NPW) abort();
            t.cg[k - 2][p] += e * f->cg[k][p];
            t.cg[k][p + 2] += -2.0 * f->cg[k][p];
        }
    }
    *o = t;
}

/* o = r^2 f */
static void rsym_mulr2(const rsym *f, rsym *o)
{
    rsym t; rsym_zero(&t);
    for (int k = 0; k < NE; ++k) {
        if (f->ce[k] != 0.0) { if (k + 2 >= NE) abort(); t.ce[k + 2] = f->ce[k]; }
        for (int p = 0; p < NPW; ++p) if (f->cg[k][p] != 0.0) { if (k + 2 >= NE) abort(); t.cg[k + 2][p] = f->cg[k][p]; }
    }
    *o = t;
}

/* o = laplacian f = f'' + 2 f'/r = 3 f_1 + r^2 f_2  with f_n = ((1/r) d/dr)^n f */
static void rsym_lap(const rsym *f, rsym *o)
{
    rsym f1, f2, r2f2, t;
    rsym_D1(f, &f1);
    rsym_D1(&f1, &f2);
    rsym_mulr2(&f2, &r2f2);
    rsym_zero(&t);
    for (int k = 0; k < NE; ++k) {
        t.ce[k] = 3.0 * f1.ce[k] + r2f2.ce[k];
        for (int p = 0; p < NPW; ++p) t.cg[k][p] = 3.0 * f1.cg[k][p] + r2f2.cg[k][p];
    }
    *o = t;
}

static void rsym_to_num(const rsym *f, double xi, rnum *o)
{
    for (int k = 0; k < NE; ++k) {
        o->ce[k] = f->ce[k];
        double s = 0.0;
        for (int p = 0; p < NPW; ++p) if (f->cg[k][p] != 0.0) s += f->cg[k][p] * pow(xi, (double)(p - POFF));
        o->cg[k] = s / sqrt(M_PI);
    }
}

static double rnum_eval(const rnum *f, double erfc_xr, double gauss, const double rpow[NE])
{
    double s = 0.0;
    for (int k = 0; k < NE; ++k) {
        const double c = f->ce[k] * erfc_xr + f->cg[k] * gauss;
        if (c != 0.0) s += c * rpow[k];
    }
    return s;
}

/* Families: 0 Phi, 1 B = lap Phi, 2 C = lap^2 Phi, 3 D = lap^3 Phi, 4 X = erfc(xi r)/r, 5 lap X.
 * Orders n = 0..4 of ((1/r) d/dr)^n.  Integer tables are xi-independent; numeric tables are per xi. */
#define NFAM 6
#define NORD 5
typedef struct { double xi; rnum t[NFAM][NORD]; } radtab;

static void radtab_build(double xi, radtab *rt)
{
    rsym fam[NFAM];
    rsym_zero(&fam[0]);
    fam[0].ce[1 + EOFF] = 1.0;                 /* r erfc(xi r)                    [Eq. 22] */
    fam[0].cg[0 + EOFF][-1 + POFF] = -1.0;     /* -exp(-xi^2 r^2)/(xi sqrt(pi))   [Eq. 22] */
    rsym_lap(&fam[0], &fam[1]);
    rsym_lap(&fam[1], &fam[2]);
    rsym_lap(&fam[2], &fam[3]);
    rsym_zero(&fam[4]);
    fam[4].ce[-1 + EOFF] = 1.0;                /* erfc(xi r)/r                    [Eq. 34] */
    rsym_lap(&fam[4], &fam[5]);
    rt->xi = xi;
    for (int f = 0; f < NFAM; ++f) {
        rsym cur = fam[f];
        for (int n = 0; n < NORD; ++n) {
            rsym_to_num(&cur, xi, &rt->t[f][n]);
            if (n + 1 < NORD) { rsym nxt; rsym_D1(&cur, &nxt); cur = nxt; }
        }
    }
}

/* Values base[f][n] of every family/order at separation r. */
static void radtab_eval(const radtab *rt, double r, double base[NFAM][NORD])
{
    double rpow[NE];
    const double rinv = 1.0 / r;
    rpow[EOFF] = 1.0;
    for (int k = EOFF + 1; k < NE; ++k) rpow[k] = rpow[k - 1] * r;
    for (int k = EOFF - 1; k >= 0; --k) rpow[k] = rpow[k + 1] * rinv;
    const double e = erfc(rt->xi * r), g = exp(-rt->xi * rt->xi * r * r);
    for (int f = 0; f < NFAM; ++f)
        for (int n = 0; n < NORD; ++n) base[f][n] = rnum_eval(&rt->t[f][n], e, g, rpow);
}

/* Exported for the pins: value of family f, order n at (xi, r). */
double oracle_radial(int fam, int order, double xi, double r)
{
    radtab rt; double base[NFAM][NORD];
    radtab_build(xi, &rt);
    radtab_eval(&rt, r, base);
    return base[fam][order];
}

/* ------------------------------------------------------------------------------------------------
 * Cartesian derivative tensors of a radial function
 * ---------------------------------------------------------------------------------------------- */
static double kd(int a, int b) { return a == b ? 1.0 : 0.0; }
static double eps3(int a, int b, int c)
{
    if (a == b || b == c || a == c) return 0.0;
    return ((b - a + 3) % 3 == 1) ? 1.0 : -1.0;
}

typedef struct { double d1[3], d2[3][3], d3[3][3][3], d4[3][3][3][3]; } dtens;

/* p[n] = psi_n, n = 1..4 (p[0] unused here). */
static void dtens_build(const double p[NORD], const double x[3], dtens *t)
{
    for (int a = 0; a < 3; ++a) {
        t->d1[a] = x[a] * p[1];
        for (int b = 0; b < 3; ++b) {
            t->d2[a][b] = kd(a, b) * p[1] + x[a] * x[b] * p[2];
            for (int c = 0; c < 3; ++c) {
                t->d3[a][b][c] = (kd(a, b) * x[c] + kd(a, c) * x[b] + kd(b, c) * x[a]) * p[2]
                               + x[a] * x[b] * x[c] * p[3];
                for (int d = 0; d < 3; ++d)
                    t->d4[a][b][c][d] =
                        (kd(a, b) * kd(c, d) + kd(a, c) * kd(b, d) + kd(a, d) * kd(b, c)) * p[2]
                      + (kd(a, b) * x[c] * x[d] + kd(a, c) * x[b] * x[d] + kd(a, d) * x[b] * x[c]
                       + kd(b, c) * x[a] * x[d] + kd(b, d) * x[a] * x[c] + kd(c, d) * x[a] * x[b]) * p[3]
                      + x[a] * x[b] * x[c] * x[d] * p[4];
            }
        }
    }
}

/* Psi = Phi + (ci+cj) B + ci cj C and Lambda = lap Psi = B + (ci+cj) C + ci cj D, all orders. */
static void psi_lambda(const double base[NFAM][NORD], double ci, double cj, double psi[NORD], double lam[NORD])
{
    for (int n = 0; n < NORD; ++n) {
        psi[n] = base[0][n] + (ci + cj) * base[1][n] + ci * cj * base[2][n];
        lam[n] = base[1][n] + (ci + cj) * base[2][n] + ci * cj * base[3][n];
    }
}

static void s5_to_33(const double *s5, double S[3][3])
{
    S[0][0] = s5[0]; S[0][1] = S[1][0] = s5[1]; S[0][2] = S[2][0] = s5[2];
    S[1][1] = s5[3]; S[1][2] = S[2][1] = s5[4]; S[2][2] = -(s5[0] + s5[3]);
}

/* Per-particle accumulators in full Cartesian form. */
typedef struct { double U[3], W[3], E[3][3], p; } acc_t;

/* Real-space contribution of source j (moments F,T,S on the fluid, pressure moment s) at separation
 * x = r_i - r_j - R_n to target i, accumulated into acc.
 *
 * Disturbance velocity of source j (Eq. 17 with J -> J_R = (I lap - grad grad) Phi, Eq. 22, and the
 * a_j^2 terms read as Laplacians; Q of Eq. 26 with 1/r -> erfc(xi r)/r, Eq. 34):
 *   v_a = k0 [ (delta_ab lap - d_a d_b)(Phi + cF_j lap Phi) F_b + (1/2) eps_agm d_g (lap Phi) T_m
 *              - d_g (delta_ab lap - d_a d_b)(Phi + cS_j lap Phi) S_bg ]  +  d_a psi_R s,
 *   k0 = 1/(8 pi eta0),  psi_R = -(1/(16 pi eta0)) erfc(xi r)/r,
 * followed by the Faxen laws (Eq. 13-15): U = (1 + cF_i lap) v, Omega = (1/2) curl v,
 * E = (1 + cS_i lap) sym grad v.  Pressure (Eq. 29-31): p' = -(1/4pi)[(1+cF_j lap) d_b chi F_b
 * - (1+cS_j lap) d_b d_g chi S_bg], chi = erfc(xi r)/r.
 * With Psi, Lambda as in psi_lambda() every coupling is one line of derivative tensors; the (ci, cj)
 * pair of each coupling is (size operator at the target end, size operator at the source end).     */
static void pair_real(const radtab *rt, const double x[3], double ai, double aj, double eta0,
                      const double F[3], const double T[3], const double S[3][3], double s, acc_t *acc)
{
    const double r = sqrt(x[0] * x[0] + x[1] * x[1] + x[2] * x[2]);
    double base[NFAM][NORD];
    radtab_eval(rt, r, base);
    const double k0 = 1.0 / (8.0 * M_PI * eta0);
    const double cFi = ai * ai / 6.0, cFj = aj * aj / 6.0, cSi = ai * ai / 10.0, cSj = aj * aj / 10.0;
    double psi[NORD], lam[NORD];
    dtens P, Lm;

    /* U <- F : k0 [delta_ab Lambda - d_a d_b Psi],                      (cF_i, cF_j) */
    psi_lambda(base, cFi, cFj, psi, lam); dtens_build(psi, x, &P);
    for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b)
        acc->U[a] += k0 * (kd(a, b) * lam[0] - P.d2[a][b]) * F[b];
    /* U <- T : (k0/2) eps_agm d_g Lambda,                               (cF_i, 0)    */
    psi_lambda(base, cFi, 0.0, psi, lam); dtens_build(lam, x, &Lm);
    for (int a = 0; a < 3; ++a) for (int g = 0; g < 3; ++g) for (int m = 0; m < 3; ++m)
        acc->U[a] += 0.5 * k0 * eps3(a, g, m) * Lm.d1[g] * T[m];
    /* U <- S : -k0 [delta_ab d_g Lambda - d_a d_b d_g Psi],             (cF_i, cS_j) */
    psi_lambda(base, cFi, cSj, psi, lam); dtens_build(psi, x, &P); dtens_build(lam, x, &Lm);
    for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b) for (int g = 0; g < 3; ++g)
        acc->U[a] += -k0 * (kd(a, b) * Lm.d1[g] - P.d3[a][b][g]) * S[b][g];

    /* Omega <- F : (k0/2) eps_agb d_g Lambda,                           (0, cF_j)    */
    psi_lambda(base, 0.0, cFj, psi, lam); dtens_build(lam, x, &Lm);
    for (int a = 0; a < 3; ++a) for (int g = 0; g < 3; ++g) for (int b = 0; b < 3; ++b)
        acc->W[a] += 0.5 * k0 * eps3(a, g, b) * Lm.d1[g] * F[b];
    /* Omega <- T : (k0/4) [d_a d_m Lambda - delta_am lap Lambda],       (0, 0): Lambda = B, lap Lambda = C */
    psi_lambda(base, 0.0, 0.0, psi, lam); dtens_build(lam, x, &Lm);
    for (int a = 0; a < 3; ++a) for (int m = 0; m < 3; ++m)
        acc->W[a] += 0.25 * k0 * (Lm.d2[a][m] - kd(a, m) * base[2][0]) * T[m];
    /* Omega <- S : -(k0/2) eps_apb d_p d_g Lambda,                      (0, cS_j)    */
    psi_lambda(base, 0.0, cSj, psi, lam); dtens_build(lam, x, &Lm);
    for (int a = 0; a < 3; ++a) for (int p = 0; p < 3; ++p) for (int b = 0; b < 3; ++b) for (int g = 0; g < 3; ++g)
        acc->W[a] += -0.5 * k0 * eps3(a, p, b) * Lm.d2[p][g] * S[b][g];

    /* E <- F : k0 [(1/2)(delta_ac d_b + delta_bc d_a) Lambda - d_a d_b d_c Psi],   (cS_i, cF_j) */
    psi_lambda(base, cSi, cFj, psi, lam); dtens_build(psi, x, &P); dtens_build(lam, x, &Lm);
    for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b) for (int c = 0; c < 3; ++c)
        acc->E[a][b] += k0 * (0.5 * (kd(a, c) * Lm.d1[b] + kd(b, c) * Lm.d1[a]) - P.d3[a][b][c]) * F[c];
    /* E <- T : (k0/4) [eps_agm d_b d_g + eps_bgm d_a d_g] Lambda,                  (cS_i, 0)    */
    psi_lambda(base, cSi, 0.0, psi, lam); dtens_build(lam, x, &Lm);
    for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b) for (int g = 0; g < 3; ++g) for (int m = 0; m < 3; ++m)
        acc->E[a][b] += 0.25 * k0 * (eps3(a, g, m) * Lm.d2[b][g] + eps3(b, g, m) * Lm.d2[a][g]) * T[m];
    /* E <- S : -k0 [(1/2)(delta_ac d_b + delta_bc d_a) d_d Lambda - d_a d_b d_c d_d Psi], (cS_i, cS_j) */
    psi_lambda(base, cSi, cSj, psi, lam); dtens_build(psi, x, &P); dtens_build(lam, x, &Lm);
    for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b) for (int c = 0; c < 3; ++c) for (int d = 0; d < 3; ++d)
        acc->E[a][b] += -k0 * (0.5 * (kd(a, c) * Lm.d2[b][d] + kd(b, c) * Lm.d2[a][d]) - P.d4[a][b][c][d]) * S[c][d];

    /* Compressible extension (Eq. 24-34).  chi = X (family 4), lap chi (family 5). */
    {
        const double kq = -1.0 / (16.0 * M_PI * eta0);      /* psi_R = kq chi */
        double q[NORD];
        dtens Q;
        if (s != 0.0) {
            /* U_a <- s : d_a (psi_R + cF_i lap psi_R) s */
            for (int n = 0; n < NORD; ++n) q[n] = kq * (base[4][n] + cFi * base[5][n]);
            dtens_build(q, x, &Q);
            for (int a = 0; a < 3; ++a) acc->U[a] += Q.d1[a] * s;
            /* E_ab <- s : d_a d_b (psi_R + cS_i lap psi_R) s  (trace removed by the caller) */
            for (int n = 0; n < NORD; ++n) q[n] = kq * (base[4][n] + cSi * base[5][n]);
            dtens_build(q, x, &Q);
            for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b) acc->E[a][b] += Q.d2[a][b] * s;
        }
        /* p <- F_b : -(1/4pi) d_b (chi + cF_j lap chi) */
        for (int n = 0; n < NORD; ++n) q[n] = base[4][n] + cFj * base[5][n];
        dtens_build(q, x, &Q);
        for (int b = 0; b < 3; ++b) acc->p += -(1.0 / (4.0 * M_PI)) * Q.d1[b] * F[b];
        /* p <- S_bg : +(1/4pi) d_b d_g (chi + cS_j lap chi) */
        for (int n = 0; n < NORD; ++n) q[n] = base[4][n] + cSj * base[5][n];
        dtens_build(q, x, &Q);
        for (int b = 0; b < 3; ++b) for (int g = 0; g < 3; ++g) acc->p += (1.0 / (4.0 * M_PI)) * Q.d2[b][g] * S[b][g];
    }
}

/* Self terms of the wave-space sum, removed because that sum runs over j = i too:
 *   UF: Eq. 37 as printed; Omega-T and E-S: same integral for the other couplings (reading 6):
 *   xi^3 5/(12 pi^{3/2} eta0) and xi^3 (25 - 42 a^2 xi^2 + 27 a^4 xi^4)/(50 pi^{3/2} eta0).            */
static void self_coeffs(double a, double xi, double eta0, double *sUF, double *sWT, double *sES)
{
    const double p32 = pow(M_PI, 1.5), a2 = a * a * xi * xi;
    *sUF = xi * (9.0 - 10.0 * a2 + 7.0 * a2 * a2) / (18.0 * p32 * eta0);
    *sWT = 5.0 * xi * xi * xi / (12.0 * p32 * eta0);
    *sES = xi * xi * xi * (25.0 - 42.0 * a2 + 27.0 * a2 * a2) / (50.0 * p32 * eta0);
}

/* One-body terms of the Faxen laws, Eq. 13-15. */
static void onebody_coeffs(double a, double eta0, double *bU, double *bW, double *bE)
{
    *bU = 1.0 / (6.0 * M_PI * eta0 * a);
    *bW = 1.0 / (8.0 * M_PI * eta0 * a * a * a);
    *bE = 1.0 / ((20.0 / 3.0) * M_PI * eta0 * a * a * a);
}

void oracle_self_coeffs(double a, double xi, double eta0, double out[3]) { self_coeffs(a, xi, eta0, &out[0], &out[1], &out[2]); }

enum { PART_REAL = 1, PART_WAVE = 2, PART_SELF = 4, PART_ONEBODY = 8 };

static void acc_finish(const acc_t *acc, int64_t N, const double *rad, double *U, double *W, double *E5, double *s_out)
{
    for (int64_t i = 0; i < N; ++i) {
        for (int d = 0; d < 3; ++d) { U[3 * i + d] = acc[i].U[d]; W[3 * i + d] = acc[i].W[d]; }
        const double tr3 = (acc[i].E[0][0] + acc[i].E[1][1] + acc[i].E[2][2]) / 3.0;   /* traceless part, Eq. 15 overline */
        E5[5 * i + 0] = acc[i].E[0][0] - tr3;
        E5[5 * i + 1] = 0.5 * (acc[i].E[0][1] + acc[i].E[1][0]);
        E5[5 * i + 2] = 0.5 * (acc[i].E[0][2] + acc[i].E[2][0]);
        E5[5 * i + 3] = acc[i].E[1][1] - tr3;
        E5[5 * i + 4] = 0.5 * (acc[i].E[1][2] + acc[i].E[2][1]);
        if (s_out) s_out[i] = 4.0 * M_PI * rad[i] * rad[i] * rad[i] * acc[i].p;          /* Eq. 28, interaction part */
    }
}

static void add_self_onebody(acc_t *acc, int64_t N, const double *rad, double xi, double eta0, unsigned parts,
                             const double *F, const double *T, const double *S5)
{
    for (int64_t i = 0; i < N; ++i) {
        double S[3][3]; s5_to_33(S5 + 5 * i, S);
        double cU = 0.0, cW = 0.0, cE = 0.0, a, b, c;
        if (parts & PART_SELF) { self_coeffs(rad[i], xi, eta0, &a, &b, &c); cU -= a; cW -= b; cE -= c; }
        if (parts & PART_ONEBODY) { onebody_coeffs(rad[i], eta0, &a, &b, &c); cU += a; cW += b; cE += c; }
        for (int d = 0; d < 3; ++d) {
            acc[i].U[d] += cU * F[3 * i + d];
            acc[i].W[d] += cW * T[3 * i + d];
            for (int e = 0; e < 3; ++e) acc[i].E[d][e] += cE * S[d][e];
        }
    }
}

/* ------------------------------------------------------------------------------------------------
 * O1: direct Ewald sum (the definition)
 * ---------------------------------------------------------------------------------------------- */
/* pos [N][3], rad [N], F,T [N][3], S5 [N][5], s_in [N] or NULL; outputs U,W [N][3], E5 [N][5], s_out [N] or NULL.
 * Real part: every lattice image R_n = L n, |n_d| <= nimg, of every pair (i,j), excluding r = 0.
 * Wave part: every k = (2 pi/L) j, |j_d| <= kmax, k != 0, including j = i.                         */
int o1_apply(int64_t N, double L, const double *pos, const double *rad, double xi, double eta0,
             int nimg, int kmax, unsigned parts,
             const double *F, const double *T, const double *S5, const double *s_in,
             double *U, double *W, double *E5, double *s_out)
{
    acc_t *acc = (acc_t *)calloc((size_t)N, sizeof(acc_t));
    if (!acc) return 1;
    const double V = L * L * L;

    if (parts & PART_REAL) {
        radtab rt; radtab_build(xi, &rt);
        #pragma omp parallel for schedule(dynamic)
        for (int64_t i = 0; i < N; ++i)
            for (int64_t j = 0; j < N; ++j) {
                double S[3][3]; s5_to_33(S5 + 5 * j, S);
                for (int n0 = -nimg; n0 <= nimg; ++n0) for (int n1 = -nimg; n1 <= nimg; ++n1) for (int n2 = -nimg; n2 <= nimg; ++n2) {
                    if (i == j && n0 == 0 && n1 == 0 && n2 == 0) continue;
                    const double x[3] = { pos[3 * i] - pos[3 * j] - L * n0, pos[3 * i + 1] - pos[3 * j + 1] - L * n1,
                                          pos[3 * i + 2] - pos[3 * j + 2] - L * n2 };
                    pair_real(&rt, x, rad[i], rad[j], eta0, F + 3 * j, T + 3 * j, S, s_in ? s_in[j] : 0.0, &acc[i]);
                }
            }
    }

    if (parts & PART_WAVE) {
        for (int j0 = -kmax; j0 <= kmax; ++j0) for (int j1 = -kmax; j1 <= kmax; ++j1) for (int j2 = -kmax; j2 <= kmax; ++j2) {
            if (j0 == 0 && j1 == 0 && j2 == 0) continue;                            /* k != 0, Eq. 19 */
            const double k[3] = { 2.0 * M_PI * j0 / L, 2.0 * M_PI * j1 / L, 2.0 * M_PI * j2 / L };
            const double k2 = k[0] * k[0] + k[1] * k[1] + k[2] * k[2];
            /* f_k = sum_j e^{ik.r_j} [(1 - cF_j k^2) F_j + (i/2) T_j x k + i (1 - cS_j k^2) S_j.k]   (from Eq. 17) */
            double complex f[3] = { 0, 0, 0 }, sk = 0;
            for (int64_t j = 0; j < N; ++j) {
                double S[3][3]; s5_to_33(S5 + 5 * j, S);
                const double cF = rad[j] * rad[j] / 6.0, cS = rad[j] * rad[j] / 10.0;
                const double *Fj = F + 3 * j, *Tj = T + 3 * j;
                const double complex ph = cexp(I * (k[0] * pos[3 * j] + k[1] * pos[3 * j + 1] + k[2] * pos[3 * j + 2]));
                const double Txk[3] = { Tj[1] * k[2] - Tj[2] * k[1], Tj[2] * k[0] - Tj[0] * k[2], Tj[0] * k[1] - Tj[1] * k[0] };
                for (int a = 0; a < 3; ++a) {
                    const double Sk = S[a][0] * k[0] + S[a][1] * k[1] + S[a][2] * k[2];
                    f[a] += ph * ((1.0 - cF * k2) * Fj[a] + 0.5 * I * Txk[a] + I * (1.0 - cS * k2) * Sk);
                }
                if (s_in) sk += ph * s_in[j];
            }
            /* v_k = (1/eta0 V) (1 + k^2/4xi^2) e^{-k^2/4xi^2} (I - kk/k^2)/k^2 . f_k     [Eq. 23, 35, 36]
             *       + (i k/(4 eta0 V k^2)) e^{-k^2/4xi^2} s_k                           [Eq. 33, 34]   */
            const double ew = exp(-k2 / (4.0 * xi * xi));
            const double hk = (1.0 + k2 / (4.0 * xi * xi)) * ew;
            const double complex kf = k[0] * f[0] + k[1] * f[1] + k[2] * f[2];
            double complex v[3];
            for (int a = 0; a < 3; ++a)
                v[a] = hk / (eta0 * V * k2) * (f[a] - k[a] * kf / k2) + I * k[a] / (4.0 * eta0 * V * k2) * ew * sk;
            /* p_k = (1/V) (i k.f_k / k^2) e^{-k^2/4xi^2}                                 [Eq. 29-31, 34] */
            const double complex pk = I * kf / (V * k2) * ew;
            for (int64_t i = 0; i < N; ++i) {
                const double cF = rad[i] * rad[i] / 6.0, cS = rad[i] * rad[i] / 10.0;
                const double complex ph = cexp(-I * (k[0] * pos[3 * i] + k[1] * pos[3 * i + 1] + k[2] * pos[3 * i + 2]));
                /* grad -> -ik on e^{-ik.x} */
                double complex g[3] = { -I * k[0], -I * k[1], -I * k[2] };
                for (int a = 0; a < 3; ++a) acc[i].U[a] += creal((1.0 - cF * k2) * ph * v[a]);            /* Eq. 13 */
                acc[i].W[0] += creal(0.5 * ph * (g[1] * v[2] - g[2] * v[1]));                            /* Eq. 14 */
                acc[i].W[1] += creal(0.5 * ph * (g[2] * v[0] - g[0] * v[2]));
                acc[i].W[2] += creal(0.5 * ph * (g[0] * v[1] - g[1] * v[0]));
                for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b)
                    acc[i].E[a][b] += creal((1.0 - cS * k2) * ph * 0.5 * (g[a] * v[b] + g[b] * v[a]));    /* Eq. 15 */
                acc[i].p += creal(ph * pk);
            }
        }
    }

    add_self_onebody(acc, N, rad, xi, eta0, parts, F, T, S5);
    acc_finish(acc, N, rad, U, W, E5, s_out);
    free(acc);
    return 0;
}

/* ------------------------------------------------------------------------------------------------
 * O2: the algorithm, step by step
 * ---------------------------------------------------------------------------------------------- */
static double wrap_box(double x, double L) { return x - L * floor(x / L); }          /* step 2: wrap */

/* ---- real-space part: cell list (Sec. 3.3) or, for fewer than 3 cells per axis, all pairs ---- */
static void min_image(const double *ri, const double *rj, double L, double x[3])
{
    for (int d = 0; d < 3; ++d) { double dd = ri[d] - rj[d]; x[d] = dd - L * nearbyint(dd / L); }
}

/* Brute-force real-space sum for the listed targets (all j, nearest image, r^2 < rc^2).  Used as the
 * one-by-one oracle for sampled outputs at full size and as the pin of the cell list.  posw = wrapped. */
static void real_targets(int64_t N, double L, const double *posw, const double *rad, double xi, double rc, double eta0,
                         const double *F, const double *T, const double *S5, const double *s_in,
                         int64_t ntgt, const int64_t *tgt, acc_t *acc /* [ntgt] */)
{
    radtab rt; radtab_build(xi, &rt);
    #pragma omp parallel for schedule(dynamic)
    for (int64_t t = 0; t < ntgt; ++t) {
        const int64_t i = tgt[t];
        for (int64_t j = 0; j < N; ++j) {
            if (j == i) continue;
            double x[3]; min_image(posw + 3 * i, posw + 3 * j, L, x);
            const double r2 = x[0] * x[0] + x[1] * x[1] + x[2] * x[2];
            if (!(r2 < rc * rc) || r2 == 0.0) continue;
            double S[3][3]; s5_to_33(S5 + 5 * j, S);
            pair_real(&rt, x, rad[i], rad[j], eta0, F + 3 * j, T + 3 * j, S, s_in ? s_in[j] : 0.0, &acc[t]);
        }
    }
}

static int real_celllist(int64_t N, double L, const double *posw, const double *rad, double xi, double rc, double eta0,
                         const double *F, const double *T, const double *S5, const double *s_in, acc_t *acc)
{
    int nc = (int)floor(L / rc);
    if (nc < 3) {                                    /* tiny systems: all pairs, minimum image */
        int64_t *all = (int64_t *)malloc(sizeof(int64_t) * (size_t)N);
        if (!all) return 1;
        for (int64_t i = 0; i < N; ++i) all[i] = i;
        real_targets(N, L, posw, rad, xi, rc, eta0, F, T, S5, s_in, N, all, acc);
        free(all);
        return 0;
    }
    if (nc > 1024) nc = 1024;
    const double h = L / nc;                         /* cell edge >= rc */
    const int64_t ncell = (int64_t)nc * nc * nc;
    int64_t *head = (int64_t *)malloc(sizeof(int64_t) * (size_t)ncell), *next = (int64_t *)malloc(sizeof(int64_t) * (size_t)N);
    int *cidx = (int *)malloc(sizeof(int) * 3 * (size_t)N);
    if (!head || !next || !cidx) { free(head); free(next); free(cidx); return 1; }
    for (int64_t c = 0; c < ncell; ++c) head[c] = -1;
    for (int64_t i = 0; i < N; ++i) {
        int c[3];
        for (int d = 0; d < 3; ++d) { c[d] = (int)floor(posw[3 * i + d] / h); c[d] = ((c[d] % nc) + nc) % nc; cidx[3 * i + d] = c[d]; }
        const int64_t ci = ((int64_t)c[0] * nc + c[1]) * nc + c[2];
        next[i] = head[ci]; head[ci] = i;
    }
    radtab rt; radtab_build(xi, &rt);
    #pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < N; ++i) {
        for (int dx = -1; dx <= 1; ++dx) for (int dy = -1; dy <= 1; ++dy) for (int dz = -1; dz <= 1; ++dz) {
            const int cx = (cidx[3 * i] + dx + nc) % nc, cy = (cidx[3 * i + 1] + dy + nc) % nc, cz = (cidx[3 * i + 2] + dz + nc) % nc;
            for (int64_t j = head[((int64_t)cx * nc + cy) * nc + cz]; j >= 0; j = next[j]) {
                if (j == i) continue;
                double x[3]; min_image(posw + 3 * i, posw + 3 * j, L, x);
                const double r2 = x[0] * x[0] + x[1] * x[1] + x[2] * x[2];
                if (!(r2 < rc * rc) || r2 == 0.0) continue;
                double S[3][3]; s5_to_33(S5 + 5 * j, S);
                pair_real(&rt, x, rad[i], rad[j], eta0, F + 3 * j, T + 3 * j, S, s_in ? s_in[j] : 0.0, &acc[i]);
            }
        }
    }
    free(head); free(next); free(cidx);
    return 0;
}

/* ---- plain complex FFT: radix-2 when M is a power of two, O(M^2) DFT otherwise ---- */
static void dft_line(double complex *x, int M, const double complex *w /* w[q] = e^{sign 2 pi i q/M} */, double complex *tmp)
{
    if ((M & (M - 1)) == 0) {
        for (int i = 1, j = 0; i < M; ++i) {                 /* bit reversal */
            int bit = M >> 1;
            for (; j & bit; bit >>= 1) j ^= bit;
            j ^= bit;
            if (i < j) { double complex t = x[i]; x[i] = x[j]; x[j] = t; }
        }
        for (int len = 2; len <= M; len <<= 1) {
            const int step = M / len;
            for (int i = 0; i < M; i += len)
                for (int q = 0; q < len / 2; ++q) {
                    const double complex u = x[i + q], v = x[i + q + len / 2] * w[q * step];
                    x[i + q] = u + v; x[i + q + len / 2] = u - v;
                }
        }
    } else {
        for (int q = 0; q < M; ++q) {
            double complex s = 0;
            for (int n = 0; n < M; ++n) s += x[n] * w[(int)(((int64_t)q * n) % M)];
            tmp[q] = s;
        }
        memcpy(x, tmp, sizeof(double complex) * (size_t)M);
    }
}

/* In-place 3-D transform  X_q = sum_n x_n e^{sign 2 pi i q.n/M}  of an [M][M][M] array (last index fastest). */
static int fft3d(double complex *a, int M, int sign)
{
    double complex *w = (double complex *)malloc(sizeof(double complex) * (size_t)M);
    if (!w) return 1;
    for (int q = 0; q < M; ++q) w[q] = cexp(sign * 2.0 * M_PI * I * (double)q / (double)M);
    const int64_t stride[3] = { (int64_t)M * M, M, 1 };
    int fail = 0;
    for (int ax = 0; ax < 3; ++ax) {
        const int o1 = (ax + 1) % 3, o2 = (ax + 2) % 3;
        #pragma omp parallel
        {
            double complex *line = (double complex *)malloc(sizeof(double complex) * 2 * (size_t)M);
            if (!line) { fail = 1; }
            else {
                #pragma omp for collapse(2)
                for (int i1 = 0; i1 < M; ++i1) for (int i2 = 0; i2 < M; ++i2) {
                    double complex *base = a + i1 * stride[o1] + i2 * stride[o2];
                    for (int n = 0; n < M; ++n) line[n] = base[n * stride[ax]];
                    dft_line(line, M, w, line + M);
                    for (int n = 0; n < M; ++n) base[n * stride[ax]] = line[n];
                }
                free(line);
            }
        }
    }
    free(w);
    return fail;
}

typedef struct { double Delta, alpha, eta_se, gnorm; int M, P; } se_consts;

/* Step 1: constants.  Delta = L/M; eta_se = (P Delta xi/m)^2 [= theta L^2/4pi^2 of Eq. 46];
 * alpha = 2 xi^2/eta_se; gamma(d) = (alpha/pi)^{3/2} e^{-alpha |d|^2}  (Eq. 41 in physical coordinates). */
static se_consts se_constants(double L, double xi, int M, int P, double m)
{
    se_consts c;
    c.M = M; c.P = P;
    c.Delta = L / M;
    c.eta_se = (P * c.Delta * xi / m) * (P * c.Delta * xi / m);
    c.alpha = 2.0 * xi * xi / c.eta_se;
    c.gnorm = pow(c.alpha / M_PI, 1.5);
    return c;
}

/* Step 2: support of a particle along one axis: u = x (M/L); first grid index n0 (unwrapped). */
static int support_start(double u, int P)
{
    return (P % 2 == 0) ? (int)floor(u) - P / 2 + 1 : (int)floor(u + 0.5) - (P - 1) / 2;
}

static int64_t gidx(int M, int n0, int n1, int n2)
{
    const int i0 = ((n0 % M) + M) % M, i1 = ((n1 % M) + M) % M, i2 = ((n2 % M) + M) % M;
    return ((int64_t)i0 * M + i1) * M + i2;
}

/* Optional staged outputs (any may be NULL):
 *   gridH   [3 or 4][M^3]  spread grids H_x,H_y,H_z (+ scalar grid of the pressure moments when s_in)
 *   gridOut [6 or 7][M^3]  returned real grids u~ (3), w~ (3) (+ p~ when s_out)
 * parts: PART_REAL | PART_WAVE | PART_SELF | PART_ONEBODY.                                       */
int o2_apply(int64_t N, double L, const double *pos, const double *rad, double xi, double rc,
             int M, int P, double m, double eta0, unsigned parts,
             const double *F, const double *T, const double *S5, const double *s_in,
             double *U, double *W, double *E5, double *s_out, double *gridH, double *gridOut)
{
    if (N < 1 || M < 2 || (M % 2) || P < 2 || P > M || !(rc > 0.0) || rc > 0.5 * L) return 2;
    acc_t *acc = (acc_t *)calloc((size_t)N, sizeof(acc_t));
    double *posw = (double *)malloc(sizeof(double) * 3 * (size_t)N);
    if (!acc || !posw) { free(acc); free(posw); return 1; }
    for (int64_t i = 0; i < 3 * N; ++i) posw[i] = wrap_box(pos[i], L);
    int status = 0;

    if (parts & PART_REAL)                                                          /* step 8 */
        status = real_celllist(N, L, posw, rad, xi, rc, eta0, F, T, S5, s_in, acc);

    if (!status && (parts & PART_WAVE)) {
        const se_consts c = se_constants(L, xi, M, P, m);
        const double al = c.alpha, D = c.Delta, V = L * L * L;
        const int64_t G = (int64_t)M * M * M;
        const int nin = s_in ? 4 : 3, nout = s_out ? 7 : 6;
        double *H = (double *)calloc((size_t)(nin * G), sizeof(double));
        double complex *Hk = (double complex *)malloc(sizeof(double complex) * (size_t)(nin * G));
        double *Gr = (double *)malloc(sizeof(double) * (size_t)(nout * G));
        double complex *work = (double complex *)malloc(sizeof(double complex) * (size_t)G);
        if (!H || !Hk || !Gr || !work) status = 1;

        if (!status) {
            /* step 3: spread (Eq. 42, Gaussian derivatives of Eq. 48 carried out analytically):
             * H(x_n) = sum_j gamma(d) [ F_j (1 + cF_j (4 al^2 d^2 - 6 al)) - al d x T_j
             *                           + 2 al (S_j.d)(1 + cS_j (4 al^2 d^2 - 10 al)) ],  d = x_n - r_j  */
            for (int64_t j = 0; j < N; ++j) {
                double S[3][3]; s5_to_33(S5 + 5 * j, S);
                const double cF = rad[j] * rad[j] / 6.0, cS = rad[j] * rad[j] / 10.0;
                const double *Fj = F + 3 * j, *Tj = T + 3 * j;
                double u[3]; int n0[3];
                for (int d = 0; d < 3; ++d) { u[d] = posw[3 * j + d] * ((double)M / L); n0[d] = support_start(u[d], P); }
                for (int a0 = 0; a0 < P; ++a0) for (int a1 = 0; a1 < P; ++a1) for (int a2 = 0; a2 < P; ++a2) {
                    const double d[3] = { ((n0[0] + a0) - u[0]) * D, ((n0[1] + a1) - u[1]) * D, ((n0[2] + a2) - u[2]) * D };
                    const double d2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
                    const double gam = c.gnorm * exp(-al * d2);
                    const double dxT[3] = { d[1] * Tj[2] - d[2] * Tj[1], d[2] * Tj[0] - d[0] * Tj[2], d[0] * Tj[1] - d[1] * Tj[0] };
                    const int64_t idx = gidx(M, n0[0] + a0, n0[1] + a1, n0[2] + a2);
                    for (int a = 0; a < 3; ++a) {
                        const double Sd = S[a][0] * d[0] + S[a][1] * d[1] + S[a][2] * d[2];
                        H[a * G + idx] += gam * (Fj[a] * (1.0 + cF * (4.0 * al * al * d2 - 6.0 * al)) - al * dxT[a]
                                                 + 2.0 * al * Sd * (1.0 + cS * (4.0 * al * al * d2 - 10.0 * al)));
                    }
                    if (s_in) H[3 * G + idx] += gam * s_in[j];
                }
            }
            if (gridH) memcpy(gridH, H, sizeof(double) * (size_t)(nin * G));

            /* step 4: H_k = sum_n H(x_n) e^{+ik.x_n},  k = (2 pi/L) j */
            for (int64_t q = 0; q < nin * G; ++q) Hk[q] = H[q];
            for (int a = 0; a < nin && !status; ++a) status = fft3d(Hk + a * G, M, +1);
        }

        /* steps 5-6, one returned grid at a time:
         *   u_k = [Delta^3/(eta0 V)] (1 + k^2/4xi^2) e^{-(1-eta_se) k^2/4xi^2}/k^2 (H_k - k (k.H_k)/k^2)   [Eq. 43 + 36]
         *         + [Delta^3/(4 eta0 V)] (i k/k^2) e^{-(1-eta_se) k^2/4xi^2} Hs_k                           [Eq. 33-34]
         *   w_k = -k^2 u_k                                                                               [hybrid, Eq. 50-51]
         *   p_k = [Delta^3/V] (i k.H_k/k^2) e^{-(1-eta_se) k^2/4xi^2}                                      [Eq. 29-31, 34]
         *   all zero for k = 0 (Eq. 43) and on the Nyquist planes j_d = -M/2 (reading 13);
         *   u~(x_n) = sum_k u_k e^{-ik.x_n} (unnormalised).                                               */
        for (int og = 0; og < nout && !status; ++og) {
            #pragma omp parallel for
            for (int i0 = 0; i0 < M; ++i0) for (int i1 = 0; i1 < M; ++i1) for (int i2 = 0; i2 < M; ++i2) {
                const int j0 = i0 < M / 2 ? i0 : i0 - M, j1 = i1 < M / 2 ? i1 : i1 - M, j2 = i2 < M / 2 ? i2 : i2 - M;
                const int64_t q = ((int64_t)i0 * M + i1) * M + i2;
                if ((j0 == 0 && j1 == 0 && j2 == 0) || j0 == -M / 2 || j1 == -M / 2 || j2 == -M / 2) { work[q] = 0; continue; }
                const double k[3] = { 2.0 * M_PI * j0 / L, 2.0 * M_PI * j1 / L, 2.0 * M_PI * j2 / L };
                const double k2 = k[0] * k[0] + k[1] * k[1] + k[2] * k[2];
                const double dec = exp(-(1.0 - c.eta_se) * k2 / (4.0 * xi * xi));
                const double sc = D * D * D / (eta0 * V) * (1.0 + k2 / (4.0 * xi * xi)) * dec / k2;
                const double complex h[3] = { Hk[q], Hk[G + q], Hk[2 * G + q] };
                const double complex kh = k[0] * h[0] + k[1] * h[1] + k[2] * h[2];
                if (og < 6) {
                    const int a = og % 3;
                    double complex uk = sc * (h[a] - k[a] * kh / k2);
                    if (s_in) uk += D * D * D / (4.0 * eta0 * V) * (I * k[a] / k2) * dec * Hk[3 * G + q];
                    work[q] = (og < 3) ? uk : -k2 * uk;
                } else {
                    work[q] = D * D * D / V * (I * kh / k2) * dec;
                }
            }
            status = fft3d(work, M, -1);
            if (!status) for (int64_t q = 0; q < G; ++q) Gr[og * G + q] = creal(work[q]);
        }
        if (!status && gridOut) memcpy(gridOut, Gr, sizeof(double) * (size_t)(nout * G));

        if (!status) {
            /* step 7: gather (Eq. 45/52 by the trapezoidal rule):
             *   U_i = D^3 sum_n gamma(d) (u~ + cF_i w~);  Omega_i = D^3 sum_n al gamma(d) d x u~;
             *   E_i = D^3 sum_n al gamma(d) (d q + q d), q = u~ + cS_i w~ (trace removed at the end);
             *   s_i = 4 pi a_i^3 D^3 sum_n gamma(d) p~,   d = x_n - r_i over the same P^3 support.     */
            const double D3 = D * D * D;
            #pragma omp parallel for schedule(static)
            for (int64_t i = 0; i < N; ++i) {
                const double cF = rad[i] * rad[i] / 6.0, cS = rad[i] * rad[i] / 10.0;
                double u[3]; int n0[3];
                for (int d = 0; d < 3; ++d) { u[d] = posw[3 * i + d] * ((double)M / L); n0[d] = support_start(u[d], P); }
                double aU[3] = { 0, 0, 0 }, aW[3] = { 0, 0, 0 }, aE[3][3] = { { 0 } }, ap = 0.0;
                for (int a0 = 0; a0 < P; ++a0) for (int a1 = 0; a1 < P; ++a1) for (int a2 = 0; a2 < P; ++a2) {
                    const double d[3] = { ((n0[0] + a0) - u[0]) * D, ((n0[1] + a1) - u[1]) * D, ((n0[2] + a2) - u[2]) * D };
                    const double gam = c.gnorm * exp(-al * (d[0] * d[0] + d[1] * d[1] + d[2] * d[2]));
                    const int64_t idx = gidx(M, n0[0] + a0, n0[1] + a1, n0[2] + a2);
                    const double ut[3] = { Gr[idx], Gr[G + idx], Gr[2 * G + idx] };
                    const double wt[3] = { Gr[3 * G + idx], Gr[4 * G + idx], Gr[5 * G + idx] };
                    double q[3];
                    for (int a = 0; a < 3; ++a) { aU[a] += gam * (ut[a] + cF * wt[a]); q[a] = ut[a] + cS * wt[a]; }
                    aW[0] += al * gam * (d[1] * ut[2] - d[2] * ut[1]);
                    aW[1] += al * gam * (d[2] * ut[0] - d[0] * ut[2]);
                    aW[2] += al * gam * (d[0] * ut[1] - d[1] * ut[0]);
                    for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b) aE[a][b] += al * gam * (d[a] * q[b] + q[a] * d[b]);
                    if (s_out) ap += gam * Gr[6 * G + idx];
                }
                for (int a = 0; a < 3; ++a) {
                    acc[i].U[a] += D3 * aU[a]; acc[i].W[a] += D3 * aW[a];
                    for (int b = 0; b < 3; ++b) acc[i].E[a][b] += D3 * aE[a][b];
                }
                acc[i].p += D3 * ap;
            }
        }
        free(H); free(Hk); free(Gr); free(work);
    }

    if (!status) {
        add_self_onebody(acc, N, rad, xi, eta0, parts, F, T, S5);                    /* step 9 (epilogue) */
        acc_finish(acc, N, rad, U, W, E5, s_out);
    }
    free(acc); free(posw);
    return status;
}

/* Real-space part of O2 for selected targets only, by brute force over all j (no cell list).
 * Outputs are [ntgt][3], [ntgt][3], [ntgt][5], [ntgt].                                            */
int o2_real_targets(int64_t N, double L, const double *pos, const double *rad, double xi, double rc, double eta0,
                    const double *F, const double *T, const double *S5, const double *s_in,
                    int64_t ntgt, const int64_t *tgt, double *U, double *W, double *E5, double *s_out)
{
    acc_t *acc = (acc_t *)calloc((size_t)ntgt, sizeof(acc_t));
    double *posw = (double *)malloc(sizeof(double) * 3 * (size_t)N);
    double *radt = (double *)malloc(sizeof(double) * (size_t)ntgt);
    if (!acc || !posw || !radt) { free(acc); free(posw); free(radt); return 1; }
    for (int64_t i = 0; i < 3 * N; ++i) posw[i] = wrap_box(pos[i], L);
    for (int64_t t = 0; t < ntgt; ++t) radt[t] = rad[tgt[t]];
    real_targets(N, L, posw, rad, xi, rc, eta0, F, T, S5, s_in, ntgt, tgt, acc);
    acc_finish(acc, ntgt, radt, U, W, E5, s_out);
    free(acc); free(posw); free(radt);
    return 0;
}

/* The SE constants of step 1, exported so tests can state them: out = {Delta, eta_se, alpha, gnorm}. */
void oracle_se_constants(double L, double xi, int M, int P, double m, double out[4])
{
    const se_consts c = se_constants(L, xi, M, P, m);
    out[0] = c.Delta; out[1] = c.eta_se; out[2] = c.alpha; out[3] = c.gnorm;
}

/* ================================================================================================
 * Sheared (Lees-Edwards) lattice, SURVEY 8f-2.  PAPER.md Sec. 3.1 L245-253 (fractional coordinates t, r = A.t,
 * k = B.q, k^2 = q.B^T.B.q), Eq. 39-45 (the Gaussian h(t) of Eq. 41 is ISOTROPIC in the fractional coordinate; the
 * lattice enters through the metric B^T.B of the derivatives and through g1(B.q)), L300-302 (simple shear:
 * a1 = (L,0,0), a2 = (gamma L, L, 0), a3 = (0,0,L), Eq. 48), L501 (same accuracy at gamma = 0.5).
 * New functions; the cubic O1 / O2 above are left as they were pinned.  For gamma = 0 they compute the same numbers.
 *
 *   A = L [[1, gamma, 0], [0, 1, 0], [0, 0, 1]]  (columns a1, a2, a3),  V = L^3,
 *   lattice images  R_n = A.n = L (n0 + gamma n1, n1, n2),
 *   wave vectors    k = 2 pi A^{-T}.j = (2 pi/L) (j0, j1 - gamma j0, j2),    k.r = 2 pi j.t.
 * ============================================================================================== */

/* O1 under shear: the definition.  Image and mode cubes are widened along the sheared directions so that they still
 * contain the spheres the cubic version sums over. */
int o1_apply_sheared(int64_t N, double L, double gamma, const double *pos, const double *rad, double xi, double eta0,
                     int nimg, int kmax, unsigned parts,
                     const double *F, const double *T, const double *S5, const double *s_in,
                     double *U, double *W, double *E5, double *s_out)
{
    acc_t *acc = (acc_t *)calloc((size_t)N, sizeof(acc_t));
    if (!acc) return 1;
    const double V = L * L * L;
    const int nx = nimg + (int)ceil(fabs(gamma) * nimg), ky = kmax + (int)ceil(fabs(gamma) * kmax);

    if (parts & PART_REAL) {
        radtab rt; radtab_build(xi, &rt);
        #pragma omp parallel for schedule(dynamic)
        for (int64_t i = 0; i < N; ++i)
            for (int64_t j = 0; j < N; ++j) {
                double S[3][3]; s5_to_33(S5 + 5 * j, S);
                for (int n0 = -nx; n0 <= nx; ++n0) for (int n1 = -nimg; n1 <= nimg; ++n1) for (int n2 = -nimg; n2 <= nimg; ++n2) {
                    if (i == j && n0 == 0 && n1 == 0 && n2 == 0) continue;
                    const double x[3] = { pos[3 * i] - pos[3 * j] - L * (n0 + gamma * n1), pos[3 * i + 1] - pos[3 * j + 1] - L * n1,
                                          pos[3 * i + 2] - pos[3 * j + 2] - L * n2 };
                    pair_real(&rt, x, rad[i], rad[j], eta0, F + 3 * j, T + 3 * j, S, s_in ? s_in[j] : 0.0, &acc[i]);
                }
            }
    }

    if (parts & PART_WAVE) {
        for (int j0 = -kmax; j0 <= kmax; ++j0) for (int j1 = -ky; j1 <= ky; ++j1) for (int j2 = -kmax; j2 <= kmax; ++j2) {
            if (j0 == 0 && j1 == 0 && j2 == 0) continue;
            const double k[3] = { 2.0 * M_PI * j0 / L, 2.0 * M_PI * (j1 - gamma * j0) / L, 2.0 * M_PI * j2 / L };
            const double k2 = k[0] * k[0] + k[1] * k[1] + k[2] * k[2];
            double complex f[3] = { 0, 0, 0 }, sk = 0;
            for (int64_t j = 0; j < N; ++j) {
                double S[3][3]; s5_to_33(S5 + 5 * j, S);
                const double cF = rad[j] * rad[j] / 6.0, cS = rad[j] * rad[j] / 10.0;
                const double *Fj = F + 3 * j, *Tj = T + 3 * j;
                const double complex ph = cexp(I * (k[0] * pos[3 * j] + k[1] * pos[3 * j + 1] + k[2] * pos[3 * j + 2]));
                const double Txk[3] = { Tj[1] * k[2] - Tj[2] * k[1], Tj[2] * k[0] - Tj[0] * k[2], Tj[0] * k[1] - Tj[1] * k[0] };
                for (int a = 0; a < 3; ++a) {
                    const double Sk = S[a][0] * k[0] + S[a][1] * k[1] + S[a][2] * k[2];
                    f[a] += ph * ((1.0 - cF * k2) * Fj[a] + 0.5 * I * Txk[a] + I * (1.0 - cS * k2) * Sk);
                }
                if (s_in) sk += ph * s_in[j];
            }
            const double ew = exp(-k2 / (4.0 * xi * xi));
            const double hk = (1.0 + k2 / (4.0 * xi * xi)) * ew;
            const double complex kf = k[0] * f[0] + k[1] * f[1] + k[2] * f[2];
            double complex v[3];
            for (int a = 0; a < 3; ++a)
                v[a] = hk / (eta0 * V * k2) * (f[a] - k[a] * kf / k2) + I * k[a] / (4.0 * eta0 * V * k2) * ew * sk;
            const double complex pk = I * kf / (V * k2) * ew;
            for (int64_t i = 0; i < N; ++i) {
                const double cF = rad[i] * rad[i] / 6.0, cS = rad[i] * rad[i] / 10.0;
                const double complex ph = cexp(-I * (k[0] * pos[3 * i] + k[1] * pos[3 * i + 1] + k[2] * pos[3 * i + 2]));
                double complex g[3] = { -I * k[0], -I * k[1], -I * k[2] };
                for (int a = 0; a < 3; ++a) acc[i].U[a] += creal((1.0 - cF * k2) * ph * v[a]);
                acc[i].W[0] += creal(0.5 * ph * (g[1] * v[2] - g[2] * v[1]));
                acc[i].W[1] += creal(0.5 * ph * (g[2] * v[0] - g[0] * v[2]));
                acc[i].W[2] += creal(0.5 * ph * (g[0] * v[1] - g[1] * v[0]));
                for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b)
                    acc[i].E[a][b] += creal((1.0 - cS * k2) * ph * 0.5 * (g[a] * v[b] + g[b] * v[a]));
                acc[i].p += creal(ph * pk);
            }
        }
    }
    add_self_onebody(acc, N, rad, xi, eta0, parts, F, T, S5);
    acc_finish(acc, N, rad, U, W, E5, s_out);
    free(acc);
    return 0;
}

/* Minimum image on the sheared lattice (r_c <= L/2: at most one image of a pair lies within r_c, and it is this one):
 * the y and z images are fixed by rounding, then the x image given the shift gamma L of the chosen y image. */
static void min_image_sheared(const double *ri, const double *rj, double L, double gamma, double x[3])
{
    const double dy = ri[1] - rj[1], dz = ri[2] - rj[2];
    const double n1 = nearbyint(dy / L);
    const double dx = (ri[0] - rj[0]) - gamma * L * n1;
    x[0] = dx - L * nearbyint(dx / L);
    x[1] = dy - L * n1;
    x[2] = dz - L * nearbyint(dz / L);
}

/* O2 under shear, step by step.  Differences from o2_apply:
 *   2. fractional coordinates t = A^{-1} r = ((x - gamma y)/L, y/L, z/L), wrapped to [0,1); u_d = t_d M; same support rule.
 *   3. grid offsets d_d = (n_d - u_d) Delta (fractional offset times L); the Gaussian is isotropic in them (Eq. 41),
 *      gam = (alpha/pi)^{3/2} e^{-alpha |d|^2}; its physical gradient is grad gam = -2 alpha D gam with the metric vector
 *          D = L^2 A^{-T}A^{-1} (r - r_j) = (d0, d1 - gamma d0, d2),    Mt = L^2 A^{-T}A^{-1} = [[1,-gamma,0],[-gamma,1+gamma^2,0],[0,0,1]],
 *      lap gam = (4 alpha^2 D.D - 2 alpha tr Mt) gam,  grad lap gam = [8 alpha^2 Mt.D - 2 alpha D (4 alpha^2 D.D - 2 alpha tr Mt)] gam
 *      (the braces of Eq. 48: tr Mt = 3 + gamma^2, D.D = (1+gamma^2) d0^2 + d1^2 + d2^2 - 2 gamma d0 d1), so
 *          H = gam { F [1 + cF (4 al^2 D.D - 2 al trMt)] - al D x T + 2 al (S.D) [1 + cS (4 al^2 D.D - 2 al trMt)] - 8 al^2 cS S.(Mt.D) }
 *      = F (1 + cF lap) gam + (1/2) grad gam x T - S.grad (1 + cS lap) gam, as in the cubic case.
 *   5. k = (2 pi/L)(j0, j1 - gamma j0, j2) in the Green's function, the projector and w = -k^2 u; the deconvolution of the two
 *      Gaussians uses the FRACTIONAL wave number: e^{+eta_se kq^2/4xi^2}, kq^2 = (2 pi/L)^2 |j|^2 (theta q^2 of Eq. 39, 43).
 *   7. gather with D in place of d:  Omega = D^3 sum al gam D x u~,  E = D^3 sum al gam (D q + q D).
 *   8. real part: all pairs, sheared minimum image, r^2 < r_c^2 (brute force: this oracle is for N <= ~1e4).         */
int o2_apply_sheared(int64_t N, double L, double gamma, const double *pos, const double *rad, double xi, double rc,
                     int M, int P, double m, double eta0, unsigned parts,
                     const double *F, const double *T, const double *S5, const double *s_in,
                     double *U, double *W, double *E5, double *s_out, double *gridH, double *gridOut)
{
    if (N < 1 || M < 2 || (M % 2) || P < 2 || P > M || !(rc > 0.0) || rc > 0.5 * L) return 2;
    acc_t *acc = (acc_t *)calloc((size_t)N, sizeof(acc_t));
    double *uu = (double *)malloc(sizeof(double) * 3 * (size_t)N);              /* u_d = wrapped fractional coordinate * M */
    if (!acc || !uu) { free(acc); free(uu); return 1; }
    const double invL = 1.0 / L;
    for (int64_t i = 0; i < N; ++i) {
        const double t[3] = { (pos[3 * i] - gamma * pos[3 * i + 1]) * invL, pos[3 * i + 1] * invL, pos[3 * i + 2] * invL };
        for (int d = 0; d < 3; ++d) uu[3 * i + d] = (t[d] - floor(t[d])) * (double)M;
    }
    int status = 0;

    if (parts & PART_REAL) {
        radtab rt; radtab_build(xi, &rt);
        #pragma omp parallel for schedule(dynamic, 16)
        for (int64_t i = 0; i < N; ++i)
            for (int64_t j = 0; j < N; ++j) {
                if (j == i) continue;
                double x[3]; min_image_sheared(pos + 3 * i, pos + 3 * j, L, gamma, x);
                const double r2 = x[0] * x[0] + x[1] * x[1] + x[2] * x[2];
                if (!(r2 < rc * rc) || r2 == 0.0) continue;
                double S[3][3]; s5_to_33(S5 + 5 * j, S);
                pair_real(&rt, x, rad[i], rad[j], eta0, F + 3 * j, T + 3 * j, S, s_in ? s_in[j] : 0.0, &acc[i]);
            }
    }

    if (parts & PART_WAVE) {
        const se_consts c = se_constants(L, xi, M, P, m);
        const double al = c.alpha, D = c.Delta, V = L * L * L, trM = 3.0 + gamma * gamma;
        const int64_t G = (int64_t)M * M * M;
        const int nin = s_in ? 4 : 3, nout = s_out ? 7 : 6;
        double *H = (double *)calloc((size_t)(nin * G), sizeof(double));
        double complex *Hk = (double complex *)malloc(sizeof(double complex) * (size_t)(nin * G));
        double *Gr = (double *)malloc(sizeof(double) * (size_t)(nout * G));
        double complex *work = (double complex *)malloc(sizeof(double complex) * (size_t)G);
        if (!H || !Hk || !Gr || !work) status = 1;

        if (!status) {
            for (int64_t j = 0; j < N; ++j) {                                         /* step 3 */
                double S[3][3]; s5_to_33(S5 + 5 * j, S);
                const double cF = rad[j] * rad[j] / 6.0, cS = rad[j] * rad[j] / 10.0;
                const double *Fj = F + 3 * j, *Tj = T + 3 * j, *u = uu + 3 * j;
                int n0[3];
                for (int d = 0; d < 3; ++d) n0[d] = support_start(u[d], P);
                for (int a0 = 0; a0 < P; ++a0) for (int a1 = 0; a1 < P; ++a1) for (int a2 = 0; a2 < P; ++a2) {
                    const double d[3] = { ((n0[0] + a0) - u[0]) * D, ((n0[1] + a1) - u[1]) * D, ((n0[2] + a2) - u[2]) * D };
                    const double gam = c.gnorm * exp(-al * (d[0] * d[0] + d[1] * d[1] + d[2] * d[2]));
                    const double Dv[3] = { d[0], d[1] - gamma * d[0], d[2] };
                    const double MD[3] = { Dv[0] - gamma * Dv[1], -gamma * Dv[0] + (1.0 + gamma * gamma) * Dv[1], Dv[2] };
                    const double DD = Dv[0] * Dv[0] + Dv[1] * Dv[1] + Dv[2] * Dv[2];
                    const double lapf = 4.0 * al * al * DD - 2.0 * al * trM;
                    const double DxT[3] = { Dv[1] * Tj[2] - Dv[2] * Tj[1], Dv[2] * Tj[0] - Dv[0] * Tj[2], Dv[0] * Tj[1] - Dv[1] * Tj[0] };
                    const int64_t idx = gidx(M, n0[0] + a0, n0[1] + a1, n0[2] + a2);
                    for (int a = 0; a < 3; ++a) {
                        const double SD = S[a][0] * Dv[0] + S[a][1] * Dv[1] + S[a][2] * Dv[2];
                        const double SMD = S[a][0] * MD[0] + S[a][1] * MD[1] + S[a][2] * MD[2];
                        H[a * G + idx] += gam * (Fj[a] * (1.0 + cF * lapf) - al * DxT[a] + 2.0 * al * SD * (1.0 + cS * lapf)
                                                 - 8.0 * al * al * cS * SMD);
                    }
                    if (s_in) H[3 * G + idx] += gam * s_in[j];
                }
            }
            if (gridH) memcpy(gridH, H, sizeof(double) * (size_t)(nin * G));
            for (int64_t q = 0; q < nin * G; ++q) Hk[q] = H[q];                       /* step 4: e^{+2 pi i j.t_n} */
            for (int a = 0; a < nin && !status; ++a) status = fft3d(Hk + a * G, M, +1);
        }

        for (int og = 0; og < nout && !status; ++og) {                               /* steps 5-6 */
            #pragma omp parallel for
            for (int i0 = 0; i0 < M; ++i0) for (int i1 = 0; i1 < M; ++i1) for (int i2 = 0; i2 < M; ++i2) {
                const int j0 = i0 < M / 2 ? i0 : i0 - M, j1 = i1 < M / 2 ? i1 : i1 - M, j2 = i2 < M / 2 ? i2 : i2 - M;
                const int64_t q = ((int64_t)i0 * M + i1) * M + i2;
                if ((j0 == 0 && j1 == 0 && j2 == 0) || j0 == -M / 2 || j1 == -M / 2 || j2 == -M / 2) { work[q] = 0; continue; }
                const double k[3] = { 2.0 * M_PI * j0 / L, 2.0 * M_PI * (j1 - gamma * j0) / L, 2.0 * M_PI * j2 / L };
                const double k2 = k[0] * k[0] + k[1] * k[1] + k[2] * k[2];
                const double kq2 = (2.0 * M_PI / L) * (2.0 * M_PI / L) * ((double)j0 * j0 + (double)j1 * j1 + (double)j2 * j2);
                const double dec = exp(-k2 / (4.0 * xi * xi) + c.eta_se * kq2 / (4.0 * xi * xi));
                const double sc = D * D * D / (eta0 * V) * (1.0 + k2 / (4.0 * xi * xi)) * dec / k2;
                const double complex h[3] = { Hk[q], Hk[G + q], Hk[2 * G + q] };
                const double complex kh = k[0] * h[0] + k[1] * h[1] + k[2] * h[2];
                if (og < 6) {
                    const int a = og % 3;
                    double complex uk = sc * (h[a] - k[a] * kh / k2);
                    if (s_in) uk += D * D * D / (4.0 * eta0 * V) * (I * k[a] / k2) * dec * Hk[3 * G + q];
                    work[q] = (og < 3) ? uk : -k2 * uk;
                } else {
                    work[q] = D * D * D / V * (I * kh / k2) * dec;
                }
            }
            status = fft3d(work, M, -1);
            if (!status) for (int64_t q = 0; q < G; ++q) Gr[og * G + q] = creal(work[q]);
        }
        if (!status && gridOut) memcpy(gridOut, Gr, sizeof(double) * (size_t)(nout * G));

        if (!status) {                                                                /* step 7 */
            const double D3 = D * D * D;
            #pragma omp parallel for schedule(static)
            for (int64_t i = 0; i < N; ++i) {
                const double cF = rad[i] * rad[i] / 6.0, cS = rad[i] * rad[i] / 10.0;
                const double *u = uu + 3 * i;
                int n0[3];
                for (int d = 0; d < 3; ++d) n0[d] = support_start(u[d], P);
                double aU[3] = { 0, 0, 0 }, aW[3] = { 0, 0, 0 }, aE[3][3] = { { 0 } }, ap = 0.0;
                for (int a0 = 0; a0 < P; ++a0) for (int a1 = 0; a1 < P; ++a1) for (int a2 = 0; a2 < P; ++a2) {
                    const double d[3] = { ((n0[0] + a0) - u[0]) * D, ((n0[1] + a1) - u[1]) * D, ((n0[2] + a2) - u[2]) * D };
                    const double gam = c.gnorm * exp(-al * (d[0] * d[0] + d[1] * d[1] + d[2] * d[2]));
                    const double Dv[3] = { d[0], d[1] - gamma * d[0], d[2] };
                    const int64_t idx = gidx(M, n0[0] + a0, n0[1] + a1, n0[2] + a2);
                    const double ut[3] = { Gr[idx], Gr[G + idx], Gr[2 * G + idx] };
                    const double wt[3] = { Gr[3 * G + idx], Gr[4 * G + idx], Gr[5 * G + idx] };
                    double q[3];
                    for (int a = 0; a < 3; ++a) { aU[a] += gam * (ut[a] + cF * wt[a]); q[a] = ut[a] + cS * wt[a]; }
                    aW[0] += al * gam * (Dv[1] * ut[2] - Dv[2] * ut[1]);
                    aW[1] += al * gam * (Dv[2] * ut[0] - Dv[0] * ut[2]);
                    aW[2] += al * gam * (Dv[0] * ut[1] - Dv[1] * ut[0]);
                    for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b) aE[a][b] += al * gam * (Dv[a] * q[b] + q[a] * Dv[b]);
                    if (s_out) ap += gam * Gr[6 * G + idx];
                }
                for (int a = 0; a < 3; ++a) {
                    acc[i].U[a] += D3 * aU[a]; acc[i].W[a] += D3 * aW[a];
                    for (int b = 0; b < 3; ++b) acc[i].E[a][b] += D3 * aE[a][b];
                }
                acc[i].p += D3 * ap;
            }
        }
        free(H); free(Hk); free(Gr); free(work);
    }

    if (!status) {
        add_self_onebody(acc, N, rad, xi, eta0, parts, F, T, S5);
        acc_finish(acc, N, rad, U, W, E5, s_out);
    }
    free(acc); free(uu);
    return status;
}

/* ------------------------------------------------------------------------------------------------
 * O2, the other two ways of bringing in the particle size (Sec. 3.2), cubic box.
 * Both differ from o2_apply (the hybrid approach) in the wave part only; steps are numbered as there.
 *
 *   variant 1, "real space" (L298-304): the size terms are derivatives of the shape function on BOTH sides.
 *     spread  : H of Eq. 42 as in o2_apply (step 3);
 *     k space : u_k only (steps 5-6 without w_k): 3 grids to wave space, 3 back (+1 +1 for the pressure);
 *     gather  : U_i = D^3 sum_n [(1 + cF lap) gamma](d) u~            = D^3 sum gamma (1 + cF (4 al^2 d^2 -  6 al)) u~
 *               E_i = D^3 sum_n -(1/2)[grad (1 + cS lap) gamma] u~ + T = D^3 sum al gamma (1 + cS (4 al^2 d^2 - 10 al)) (d u~ + u~ d)
 *               Om_i as in o2_apply.          (lap gamma = (4 al^2 d^2 - 6 al) gamma, grad gamma = -2 al d gamma)
 *
 *   variant 2, "wave space" (L306-322, Eq. 49-52): only gamma itself is spread and gathered; every derivative is a
 *     multiplication by the wave vector.  With the transform conventions of o2_apply (H_k = sum_n H e^{+ik.x},
 *     returned grids sum_k (.) e^{-ik.x}) a gradient acting on gamma(x - r_j) in the spreading becomes -ik, and a
 *     gradient acting on a returned grid becomes -ik as well.
 *     spread  : H'_F = sum gamma F, H''_F = sum gamma a^2 F, H_T = sum gamma T, H'_S = sum gamma S, H''_S = sum gamma a^2 S   (Eq. 49)
 *     k space : Heff_k = (H'_F - (k^2/6) H''_F) - (i/2) k x H_T + i (H'_S - (k^2/10) H''_S).k                     (Eq. 50, bracket)
 *               [this is the transform of Eq. 42's H: F (1 + a^2/6 lap) gamma + (1/2) grad gamma x T - (1 + a^2/10 lap) S.grad gamma]
 *               u_k as in o2_apply from Heff_k;   w_k = -k^2 u_k (Eq. 51);   om_k = -(i/2) k x u_k;
 *               e0_k[ab] = -(i/2)(k_a u_b + k_b u_a);   e2_k = -k^2 e0_k
 *     gather  : U_i = D^3 sum gamma (u~ + cF_i w~) (Eq. 52);  Om_i = D^3 sum gamma om~;  E_i = D^3 sum gamma (e0~ + cS_i e2~).
 *     Grid count: the paper quotes 20 pairs with a symmetric S of six components; this restatement carries six
 *     components for S, a^2 S, e0 and e2 (21 to wave space, 21 back) and removes the trace at the end like o2_apply.
 *   Pressure moment and pressure (a9): the scalar grid Hs and the returned p~ carry no size terms and are spread and
 *   gathered with gamma in every variant; p_k uses Heff_k in variant 2.
 * ---------------------------------------------------------------------------------------------- */
int o2_apply_variant(int variant, int64_t N, double L, const double *pos, const double *rad, double xi, double rc,
                     int M, int P, double m, double eta0, unsigned parts,
                     const double *F, const double *T, const double *S5, const double *s_in,
                     double *U, double *W, double *E5, double *s_out)
{
    if (variant != 1 && variant != 2) return 2;
    if (N < 1 || M < 2 || (M % 2) || P < 2 || P > M || !(rc > 0.0) || rc > 0.5 * L) return 2;
    acc_t *acc = (acc_t *)calloc((size_t)N, sizeof(acc_t));
    double *posw = (double *)malloc(sizeof(double) * 3 * (size_t)N);
    if (!acc || !posw) { free(acc); free(posw); return 1; }
    for (int64_t i = 0; i < 3 * N; ++i) posw[i] = wrap_box(pos[i], L);
    int status = 0;

    if (parts & PART_REAL) status = real_celllist(N, L, posw, rad, xi, rc, eta0, F, T, S5, s_in, acc);   /* step 8 */

    if (!status && (parts & PART_WAVE)) {
        const se_consts c = se_constants(L, xi, M, P, m);
        const double al = c.alpha, D = c.Delta, V = L * L * L, D3 = D * D * D;
        const int64_t G = (int64_t)M * M * M;
        /* grid tables.  variant 1: in 0-2 H (3 s);            out 0-2 u~ (3 p~)
         *               variant 2: in 0-2 F, 3-5 a^2 F, 6-8 T, 9-14 S, 15-20 a^2 S (21 s);
         *                          out 0-2 u~, 3-5 w~, 6-8 om~, 9-14 e0~, 15-20 e2~ (21 p~);  pairs (a,b) in the order below */
        static const int PA[6] = { 0, 0, 0, 1, 1, 2 }, PB[6] = { 0, 1, 2, 1, 2, 2 };
        const int nbase = variant == 1 ? 3 : 21;
        const int nin = nbase + (s_in ? 1 : 0), nout = nbase + (s_out ? 1 : 0);
        double *H = (double *)calloc((size_t)(nin * G), sizeof(double));
        double complex *Hk = (double complex *)malloc(sizeof(double complex) * (size_t)(nin * G));
        double *Gr = (double *)malloc(sizeof(double) * (size_t)(nout * G));
        double complex *work = (double complex *)malloc(sizeof(double complex) * (size_t)G);
        if (!H || !Hk || !Gr || !work) status = 1;

        if (!status) {                                                              /* step 3: spread */
            for (int64_t j = 0; j < N; ++j) {
                double S[3][3]; s5_to_33(S5 + 5 * j, S);
                const double a2 = rad[j] * rad[j], cF = a2 / 6.0, cS = a2 / 10.0;
                const double *Fj = F + 3 * j, *Tj = T + 3 * j;
                double u[3]; int n0[3];
                for (int d = 0; d < 3; ++d) { u[d] = posw[3 * j + d] * ((double)M / L); n0[d] = support_start(u[d], P); }
                for (int a0 = 0; a0 < P; ++a0) for (int a1 = 0; a1 < P; ++a1) for (int a2i = 0; a2i < P; ++a2i) {
                    const double d[3] = { ((n0[0] + a0) - u[0]) * D, ((n0[1] + a1) - u[1]) * D, ((n0[2] + a2i) - u[2]) * D };
                    const double d2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
                    const double gam = c.gnorm * exp(-al * d2);
                    const int64_t idx = gidx(M, n0[0] + a0, n0[1] + a1, n0[2] + a2i);
                    if (variant == 1) {
                        const double dxT[3] = { d[1] * Tj[2] - d[2] * Tj[1], d[2] * Tj[0] - d[0] * Tj[2], d[0] * Tj[1] - d[1] * Tj[0] };
                        for (int a = 0; a < 3; ++a) {
                            const double Sd = S[a][0] * d[0] + S[a][1] * d[1] + S[a][2] * d[2];
                            H[a * G + idx] += gam * (Fj[a] * (1.0 + cF * (4.0 * al * al * d2 - 6.0 * al)) - al * dxT[a]
                                                     + 2.0 * al * Sd * (1.0 + cS * (4.0 * al * al * d2 - 10.0 * al)));
                        }
                    } else {
                        for (int a = 0; a < 3; ++a) {
                            H[a * G + idx] += gam * Fj[a];
                            H[(3 + a) * G + idx] += gam * a2 * Fj[a];
                            H[(6 + a) * G + idx] += gam * Tj[a];
                        }
                        for (int e = 0; e < 6; ++e) {
                            H[(9 + e) * G + idx] += gam * S[PA[e]][PB[e]];
                            H[(15 + e) * G + idx] += gam * a2 * S[PA[e]][PB[e]];
                        }
                    }
                    if (s_in) H[nbase * G + idx] += gam * s_in[j];
                }
            }
            for (int64_t q = 0; q < nin * G; ++q) Hk[q] = H[q];                     /* step 4 */
            for (int a = 0; a < nin && !status; ++a) status = fft3d(Hk + a * G, M, +1);
        }

        for (int og = 0; og < nout && !status; ++og) {                              /* steps 5-6, one returned grid at a time */
            #pragma omp parallel for
            for (int i0 = 0; i0 < M; ++i0) for (int i1 = 0; i1 < M; ++i1) for (int i2 = 0; i2 < M; ++i2) {
                const int j0 = i0 < M / 2 ? i0 : i0 - M, j1 = i1 < M / 2 ? i1 : i1 - M, j2 = i2 < M / 2 ? i2 : i2 - M;
                const int64_t q = ((int64_t)i0 * M + i1) * M + i2;
                if ((j0 == 0 && j1 == 0 && j2 == 0) || j0 == -M / 2 || j1 == -M / 2 || j2 == -M / 2) { work[q] = 0; continue; }
                const double k[3] = { 2.0 * M_PI * j0 / L, 2.0 * M_PI * j1 / L, 2.0 * M_PI * j2 / L };
                const double k2 = k[0] * k[0] + k[1] * k[1] + k[2] * k[2];
                const double dec = exp(-(1.0 - c.eta_se) * k2 / (4.0 * xi * xi));
                const double sc = D3 / (eta0 * V) * (1.0 + k2 / (4.0 * xi * xi)) * dec / k2;
                double complex h[3];
                if (variant == 1) { h[0] = Hk[q]; h[1] = Hk[G + q]; h[2] = Hk[2 * G + q]; }
                else {
                    double complex Tk[3], Sk[3][3];
                    for (int a = 0; a < 3; ++a) Tk[a] = Hk[(6 + a) * G + q];
                    for (int e = 0; e < 6; ++e)
                        Sk[PA[e]][PB[e]] = Sk[PB[e]][PA[e]] = Hk[(9 + e) * G + q] - (k2 / 10.0) * Hk[(15 + e) * G + q];
                    const double complex kxT[3] = { k[1] * Tk[2] - k[2] * Tk[1], k[2] * Tk[0] - k[0] * Tk[2], k[0] * Tk[1] - k[1] * Tk[0] };
                    for (int a = 0; a < 3; ++a)
                        h[a] = Hk[a * G + q] - (k2 / 6.0) * Hk[(3 + a) * G + q] - 0.5 * I * kxT[a]
                               + I * (Sk[a][0] * k[0] + Sk[a][1] * k[1] + Sk[a][2] * k[2]);
                }
                const double complex kh = k[0] * h[0] + k[1] * h[1] + k[2] * h[2];
                double complex uk[3];
                for (int a = 0; a < 3; ++a) {
                    uk[a] = sc * (h[a] - k[a] * kh / k2);
                    if (s_in) uk[a] += D3 / (4.0 * eta0 * V) * (I * k[a] / k2) * dec * Hk[nbase * G + q];
                }
                if (og == nbase) work[q] = D3 / V * (I * kh / k2) * dec;                                   /* p_k */
                else if (og < 3) work[q] = uk[og];
                else if (og < 6) work[q] = -k2 * uk[og - 3];
                else if (og < 9) {
                    const double complex kxu[3] = { k[1] * uk[2] - k[2] * uk[1], k[2] * uk[0] - k[0] * uk[2], k[0] * uk[1] - k[1] * uk[0] };
                    work[q] = -0.5 * I * kxu[og - 6];
                } else {
                    const int e = (og - 9) % 6, a = PA[e], b = PB[e];
                    const double complex e0 = -0.5 * I * (k[a] * uk[b] + k[b] * uk[a]);
                    work[q] = og < 15 ? e0 : -k2 * e0;
                }
            }
            status = fft3d(work, M, -1);
            if (!status) for (int64_t q = 0; q < G; ++q) Gr[og * G + q] = creal(work[q]);
        }

        if (!status) {                                                              /* step 7: gather */
            #pragma omp parallel for schedule(static)
            for (int64_t i = 0; i < N; ++i) {
                const double cF = rad[i] * rad[i] / 6.0, cS = rad[i] * rad[i] / 10.0;
                double u[3]; int n0[3];
                for (int d = 0; d < 3; ++d) { u[d] = posw[3 * i + d] * ((double)M / L); n0[d] = support_start(u[d], P); }
                double aU[3] = { 0, 0, 0 }, aW[3] = { 0, 0, 0 }, aE[3][3] = { { 0 } }, ap = 0.0;
                for (int a0 = 0; a0 < P; ++a0) for (int a1 = 0; a1 < P; ++a1) for (int a2i = 0; a2i < P; ++a2i) {
                    const double d[3] = { ((n0[0] + a0) - u[0]) * D, ((n0[1] + a1) - u[1]) * D, ((n0[2] + a2i) - u[2]) * D };
                    const double d2 = d[0] * d[0] + d[1] * d[1] + d[2] * d[2];
                    const double gam = c.gnorm * exp(-al * d2);
                    const int64_t idx = gidx(M, n0[0] + a0, n0[1] + a1, n0[2] + a2i);
                    if (variant == 1) {
                        const double ut[3] = { Gr[idx], Gr[G + idx], Gr[2 * G + idx] };
                        const double fU = 1.0 + cF * (4.0 * al * al * d2 - 6.0 * al), fE = 1.0 + cS * (4.0 * al * al * d2 - 10.0 * al);
                        for (int a = 0; a < 3; ++a) aU[a] += gam * fU * ut[a];
                        aW[0] += al * gam * (d[1] * ut[2] - d[2] * ut[1]);
                        aW[1] += al * gam * (d[2] * ut[0] - d[0] * ut[2]);
                        aW[2] += al * gam * (d[0] * ut[1] - d[1] * ut[0]);
                        for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b) aE[a][b] += al * gam * fE * (d[a] * ut[b] + ut[a] * d[b]);
                    } else {
                        for (int a = 0; a < 3; ++a) {
                            aU[a] += gam * (Gr[a * G + idx] + cF * Gr[(3 + a) * G + idx]);
                            aW[a] += gam * Gr[(6 + a) * G + idx];
                        }
                        for (int e = 0; e < 6; ++e) {
                            const double v = gam * (Gr[(9 + e) * G + idx] + cS * Gr[(15 + e) * G + idx]);
                            aE[PA[e]][PB[e]] += v;
                            if (PA[e] != PB[e]) aE[PB[e]][PA[e]] += v;
                        }
                    }
                    if (s_out) ap += gam * Gr[nbase * G + idx];
                }
                for (int a = 0; a < 3; ++a) {
                    acc[i].U[a] += D3 * aU[a]; acc[i].W[a] += D3 * aW[a];
                    for (int b = 0; b < 3; ++b) acc[i].E[a][b] += D3 * aE[a][b];
                }
                acc[i].p += D3 * ap;
            }
        }
        free(H); free(Hk); free(Gr); free(work);
    }

    if (!status) {
        add_self_onebody(acc, N, rad, xi, eta0, parts, F, T, S5);                    /* step 9 */
        acc_finish(acc, N, rad, U, W, E5, s_out);
    }
    free(acc); free(posw);
    return status;
}

/* ------------------------------------------------------------------------------------------------
 * The real-space and wave-space size variants on the SHEARED lattice (Fig. 2 shows both at gamma = 0.5).
 * o2_apply_variant with the changes o2_apply_sheared makes to o2_apply (its header): wrapped fractional coordinates, the
 * Gaussian isotropic in the grid offsets d, physical derivatives through D = (d0, d1 - gamma d0, d2) and Mt, k = B.q in every
 * wave-vector factor, deconvolution in the fractional wave number, brute-force real part with the sheared minimum image.
 *   variant 1: spread as o2_apply_sheared; u~ only; gather with the SAME operators on the Gaussian (the adjoint of the spreading):
 *       U  = D^3 sum gam [1 + cF lapf] u~,                           lapf = 4 al^2 D.D - 2 al tr Mt
 *       Om = D^3 sum al gam D x u~
 *       E  = D^3 sum gam { al [1 + cS lapf] (D u~ + u~ D) - 4 al^2 cS (Mt.D u~ + u~ Mt.D) }     [-(1/2) grad (1 + cS lap) gam, symmetrised]
 *   variant 2: plain gam on both sides, k = B.q in H_eff, u, w, om, e0, e2 as in o2_apply_variant.
 * ---------------------------------------------------------------------------------------------- */
int o2_apply_variant_sheared(int variant, int64_t N, double L, double gamma, const double *pos, const double *rad, double xi, double rc,
                             int M, int P, double m, double eta0, unsigned parts,
                             const double *F, const double *T, const double *S5, const double *s_in,
                             double *U, double *W, double *E5, double *s_out)
{
    if (variant != 1 && variant != 2) return 2;
    if (N < 1 || M < 2 || (M % 2) || P < 2 || P > M || !(rc > 0.0) || rc > 0.5 * L) return 2;
    acc_t *acc = (acc_t *)calloc((size_t)N, sizeof(acc_t));
    double *uu = (double *)malloc(sizeof(double) * 3 * (size_t)N);
    if (!acc || !uu) { free(acc); free(uu); return 1; }
    const double invL = 1.0 / L;
    for (int64_t i = 0; i < N; ++i) {                                              /* step 2 */
        const double t[3] = { (pos[3 * i] - gamma * pos[3 * i + 1]) * invL, pos[3 * i + 1] * invL, pos[3 * i + 2] * invL };
        for (int d = 0; d < 3; ++d) uu[3 * i + d] = (t[d] - floor(t[d])) * (double)M;
    }
    int status = 0;

    if (parts & PART_REAL) {                                                        /* step 8 */
        radtab rt; radtab_build(xi, &rt);
        #pragma omp parallel for schedule(dynamic, 16)
        for (int64_t i = 0; i < N; ++i)
            for (int64_t j = 0; j < N; ++j) {
                if (j == i) continue;
                double x[3]; min_image_sheared(pos + 3 * i, pos + 3 * j, L, gamma, x);
                const double r2 = x[0] * x[0] + x[1] * x[1] + x[2] * x[2];
                if (!(r2 < rc * rc) || r2 == 0.0) continue;
                double S[3][3]; s5_to_33(S5 + 5 * j, S);
                pair_real(&rt, x, rad[i], rad[j], eta0, F + 3 * j, T + 3 * j, S, s_in ? s_in[j] : 0.0, &acc[i]);
            }
    }

    if (parts & PART_WAVE) {
        const se_consts c = se_constants(L, xi, M, P, m);
        const double al = c.alpha, D = c.Delta, V = L * L * L, D3 = D * D * D, trM = 3.0 + gamma * gamma;
        const int64_t G = (int64_t)M * M * M;
        static const int PA[6] = { 0, 0, 0, 1, 1, 2 }, PB[6] = { 0, 1, 2, 1, 2, 2 };
        const int nbase = variant == 1 ? 3 : 21;
        const int nin = nbase + (s_in ? 1 : 0), nout = nbase + (s_out ? 1 : 0);
        double *H = (double *)calloc((size_t)(nin * G), sizeof(double));
        double complex *Hk = (double complex *)malloc(sizeof(double complex) * (size_t)(nin * G));
        double *Gr = (double *)malloc(sizeof(double) * (size_t)(nout * G));
        double complex *work = (double complex *)malloc(sizeof(double complex) * (size_t)G);
        if (!H || !Hk || !Gr || !work) status = 1;

        if (!status) {                                                              /* step 3 */
            for (int64_t j = 0; j < N; ++j) {
                double S[3][3]; s5_to_33(S5 + 5 * j, S);
                const double a2 = rad[j] * rad[j], cF = a2 / 6.0, cS = a2 / 10.0;
                const double *Fj = F + 3 * j, *Tj = T + 3 * j, *u = uu + 3 * j;
                int n0[3];
                for (int d = 0; d < 3; ++d) n0[d] = support_start(u[d], P);
                for (int a0 = 0; a0 < P; ++a0) for (int a1 = 0; a1 < P; ++a1) for (int a2i = 0; a2i < P; ++a2i) {
                    const double d[3] = { ((n0[0] + a0) - u[0]) * D, ((n0[1] + a1) - u[1]) * D, ((n0[2] + a2i) - u[2]) * D };
                    const double gam = c.gnorm * exp(-al * (d[0] * d[0] + d[1] * d[1] + d[2] * d[2]));
                    const int64_t idx = gidx(M, n0[0] + a0, n0[1] + a1, n0[2] + a2i);
                    if (variant == 1) {
                        const double Dv[3] = { d[0], d[1] - gamma * d[0], d[2] };
                        const double MD[3] = { Dv[0] - gamma * Dv[1], -gamma * Dv[0] + (1.0 + gamma * gamma) * Dv[1], Dv[2] };
                        const double lapf = 4.0 * al * al * (Dv[0] * Dv[0] + Dv[1] * Dv[1] + Dv[2] * Dv[2]) - 2.0 * al * trM;
                        const double DxT[3] = { Dv[1] * Tj[2] - Dv[2] * Tj[1], Dv[2] * Tj[0] - Dv[0] * Tj[2], Dv[0] * Tj[1] - Dv[1] * Tj[0] };
                        for (int a = 0; a < 3; ++a) {
                            const double SD = S[a][0] * Dv[0] + S[a][1] * Dv[1] + S[a][2] * Dv[2];
                            const double SMD = S[a][0] * MD[0] + S[a][1] * MD[1] + S[a][2] * MD[2];
                            H[a * G + idx] += gam * (Fj[a] * (1.0 + cF * lapf) - al * DxT[a] + 2.0 * al * SD * (1.0 + cS * lapf)
                                                     - 8.0 * al * al * cS * SMD);
                        }
                    } else {
                        for (int a = 0; a < 3; ++a) {
                            H[a * G + idx] += gam * Fj[a];
                            H[(3 + a) * G + idx] += gam * a2 * Fj[a];
                            H[(6 + a) * G + idx] += gam * Tj[a];
                        }
                        for (int e = 0; e < 6; ++e) {
                            H[(9 + e) * G + idx] += gam * S[PA[e]][PB[e]];
                            H[(15 + e) * G + idx] += gam * a2 * S[PA[e]][PB[e]];
                        }
                    }
                    if (s_in) H[nbase * G + idx] += gam * s_in[j];
                }
            }
            for (int64_t q = 0; q < nin * G; ++q) Hk[q] = H[q];                     /* step 4 */
            for (int a = 0; a < nin && !status; ++a) status = fft3d(Hk + a * G, M, +1);
        }

        for (int og = 0; og < nout && !status; ++og) {                              /* steps 5-6 */
            #pragma omp parallel for
            for (int i0 = 0; i0 < M; ++i0) for (int i1 = 0; i1 < M; ++i1) for (int i2 = 0; i2 < M; ++i2) {
                const int j0 = i0 < M / 2 ? i0 : i0 - M, j1 = i1 < M / 2 ? i1 : i1 - M, j2 = i2 < M / 2 ? i2 : i2 - M;
                const int64_t q = ((int64_t)i0 * M + i1) * M + i2;
                if ((j0 == 0 && j1 == 0 && j2 == 0) || j0 == -M / 2 || j1 == -M / 2 || j2 == -M / 2) { work[q] = 0; continue; }
                const double k[3] = { 2.0 * M_PI * j0 / L, 2.0 * M_PI * (j1 - gamma * j0) / L, 2.0 * M_PI * j2 / L };
                const double k2 = k[0] * k[0] + k[1] * k[1] + k[2] * k[2];
                const double kq2 = (2.0 * M_PI / L) * (2.0 * M_PI / L) * ((double)j0 * j0 + (double)j1 * j1 + (double)j2 * j2);
                const double dec = exp(-k2 / (4.0 * xi * xi) + c.eta_se * kq2 / (4.0 * xi * xi));
                const double sc = D3 / (eta0 * V) * (1.0 + k2 / (4.0 * xi * xi)) * dec / k2;
                double complex h[3];
                if (variant == 1) { h[0] = Hk[q]; h[1] = Hk[G + q]; h[2] = Hk[2 * G + q]; }
                else {
                    double complex Tk[3], Sk[3][3];
                    for (int a = 0; a < 3; ++a) Tk[a] = Hk[(6 + a) * G + q];
                    for (int e = 0; e < 6; ++e)
                        Sk[PA[e]][PB[e]] = Sk[PB[e]][PA[e]] = Hk[(9 + e) * G + q] - (k2 / 10.0) * Hk[(15 + e) * G + q];
                    const double complex kxT[3] = { k[1] * Tk[2] - k[2] * Tk[1], k[2] * Tk[0] - k[0] * Tk[2], k[0] * Tk[1] - k[1] * Tk[0] };
                    for (int a = 0; a < 3; ++a)
                        h[a] = Hk[a * G + q] - (k2 / 6.0) * Hk[(3 + a) * G + q] - 0.5 * I * kxT[a]
                               + I * (Sk[a][0] * k[0] + Sk[a][1] * k[1] + Sk[a][2] * k[2]);
                }
                const double complex kh = k[0] * h[0] + k[1] * h[1] + k[2] * h[2];
                double complex uk[3];
                for (int a = 0; a < 3; ++a) {
                    uk[a] = sc * (h[a] - k[a] * kh / k2);
                    if (s_in) uk[a] += D3 / (4.0 * eta0 * V) * (I * k[a] / k2) * dec * Hk[nbase * G + q];
                }
                if (og == nbase) work[q] = D3 / V * (I * kh / k2) * dec;
                else if (og < 3) work[q] = uk[og];
                else if (og < 6) work[q] = -k2 * uk[og - 3];
                else if (og < 9) {
                    const double complex kxu[3] = { k[1] * uk[2] - k[2] * uk[1], k[2] * uk[0] - k[0] * uk[2], k[0] * uk[1] - k[1] * uk[0] };
                    work[q] = -0.5 * I * kxu[og - 6];
                } else {
                    const int e = (og - 9) % 6, a = PA[e], b = PB[e];
                    const double complex e0 = -0.5 * I * (k[a] * uk[b] + k[b] * uk[a]);
                    work[q] = og < 15 ? e0 : -k2 * e0;
                }
            }
            status = fft3d(work, M, -1);
            if (!status) for (int64_t q = 0; q < G; ++q) Gr[og * G + q] = creal(work[q]);
        }

        if (!status) {                                                              /* step 7 */
            #pragma omp parallel for schedule(static)
            for (int64_t i = 0; i < N; ++i) {
                const double cF = rad[i] * rad[i] / 6.0, cS = rad[i] * rad[i] / 10.0;
                const double *u = uu + 3 * i;
                int n0[3];
                for (int d = 0; d < 3; ++d) n0[d] = support_start(u[d], P);
                double aU[3] = { 0, 0, 0 }, aW[3] = { 0, 0, 0 }, aE[3][3] = { { 0 } }, ap = 0.0;
                for (int a0 = 0; a0 < P; ++a0) for (int a1 = 0; a1 < P; ++a1) for (int a2i = 0; a2i < P; ++a2i) {
                    const double d[3] = { ((n0[0] + a0) - u[0]) * D, ((n0[1] + a1) - u[1]) * D, ((n0[2] + a2i) - u[2]) * D };
                    const double gam = c.gnorm * exp(-al * (d[0] * d[0] + d[1] * d[1] + d[2] * d[2]));
                    const int64_t idx = gidx(M, n0[0] + a0, n0[1] + a1, n0[2] + a2i);
                    if (variant == 1) {
                        const double Dv[3] = { d[0], d[1] - gamma * d[0], d[2] };
                        const double MD[3] = { Dv[0] - gamma * Dv[1], -gamma * Dv[0] + (1.0 + gamma * gamma) * Dv[1], Dv[2] };
                        const double lapf = 4.0 * al * al * (Dv[0] * Dv[0] + Dv[1] * Dv[1] + Dv[2] * Dv[2]) - 2.0 * al * trM;
                        const double ut[3] = { Gr[idx], Gr[G + idx], Gr[2 * G + idx] };
                        for (int a = 0; a < 3; ++a) aU[a] += gam * (1.0 + cF * lapf) * ut[a];
                        aW[0] += al * gam * (Dv[1] * ut[2] - Dv[2] * ut[1]);
                        aW[1] += al * gam * (Dv[2] * ut[0] - Dv[0] * ut[2]);
                        aW[2] += al * gam * (Dv[0] * ut[1] - Dv[1] * ut[0]);
                        for (int a = 0; a < 3; ++a) for (int b = 0; b < 3; ++b)
                            aE[a][b] += gam * (al * (1.0 + cS * lapf) * (Dv[a] * ut[b] + ut[a] * Dv[b])
                                               - 4.0 * al * al * cS * (MD[a] * ut[b] + ut[a] * MD[b]));
                    } else {
                        for (int a = 0; a < 3; ++a) {
                            aU[a] += gam * (Gr[a * G + idx] + cF * Gr[(3 + a) * G + idx]);
                            aW[a] += gam * Gr[(6 + a) * G + idx];
                        }
                        for (int e = 0; e < 6; ++e) {
                            const double v = gam * (Gr[(9 + e) * G + idx] + cS * Gr[(15 + e) * G + idx]);
                            aE[PA[e]][PB[e]] += v;
                            if (PA[e] != PB[e]) aE[PB[e]][PA[e]] += v;
                        }
                    }
                    if (s_out) ap += gam * Gr[nbase * G + idx];
                }
                for (int a = 0; a < 3; ++a) {
                    acc[i].U[a] += D3 * aU[a]; acc[i].W[a] += D3 * aW[a];
                    for (int b = 0; b < 3; ++b) acc[i].E[a][b] += D3 * aE[a][b];
                }
                acc[i].p += D3 * ap;
            }
        }
        free(H); free(Hk); free(Gr); free(work);
    }

    if (!status) {
        add_self_onebody(acc, N, rad, xi, eta0, parts, F, T, S5);                    /* step 9 */
        acc_finish(acc, N, rad, U, W, E5, s_out);
    }
    free(acc); free(uu);
    return status;
}
