/* me_oracle.c -- CPU ORACLE.  TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * call this.  It shares no code with the CUDA path (paper_2510_05392_b200/csrc, .../gen) and is
 * never tuned for speed.
 *
 * What it computes ("takes as input an array of particle momenta for many events
 * ... returns an array of matrix elements"; PAPER.md:95-98,124 helicity sum; PAPER.md:117-119,
 * 243, 264-269 Eq. 1: quadratic form J^H (C) J with a real symmetric colour matrix):
 *
 *     me = (1/denom) * sum_{helicities h} sum_{colours} |M_h|^2        (tree level, LO)
 *
 * for g g -> t tbar + (n-2) g and for e+ e- -> mu+ mu-.  The paper reaches this number through
 * explicit Feynman diagrams (HELAS routines) and a leading-colour-flow basis; the oracle takes an
 * INDEPENDENT route to the same, plainly defined number:
 *   - colour-ordered Berends-Giele recursion for the n! partial amplitudes A(sigma)
 *     (PAPER.md:641, 708 name BG recursion as the alternative to diagrams),
 *   - the colour matrix C_{sigma sigma'} by brute force over all SU(3) colour indices with
 *     explicit Gell-Mann matrices,
 *   - Dirac-representation gamma matrices and helicity spinors (the CUDA path uses a chiral,
 *     HELAS-like representation), explicit 4x4 matrix algebra, no shortcuts.
 *
 * Conventions (textbook Feynman rules):
 *   metric (+,-,-,-);  T^a = lambda^a/2;  [T^a,T^b] = i f^{abc} T^c;  g = sqrt(4 pi alpha_s);
 *   colour decomposition  M = sum_sigma (T^{a_s1} ... T^{a_sn})_{i jbar} A(sigma), first T next to the top;
 *   all-incoming gluon momenta k (k = p for the beams, k = -p for final gluons);
 *   eps(p,lambda) for incoming gluons, eps^* for outgoing; ubar(p_t) and v(p_tbar) with physical helicities;
 *   top propagator (qslash + m)/(q^2 - m^2 + i m Gamma): width in the denominator only (reading A4).
 *   Helicity index h = sum_i b_i 2^(npar-1-i), b_i = 0 <-> lambda_i = -1 (reading A2).
 *
 * Pins (tests/test_oracle_pins.py): P1 e+e- closed form, P2 analytic gg->ttbar, P3 gauge invariance,
 * P4 colour-dressed brute force with explicit f^{abc} (numpy, in the test), P5 colour-matrix
 * invariants, P6 Lorentz/Bose/parity symmetry, P10 double vs long double.
 * Parity with MG5aMC/CUDACPP output itself is UNPINNED: the paper prints mean MEs only for
 * unspecified momenta, SURVEY.md P9.
 *
 * Precision: fp64 (`real` = double); compile with -DORC_LONG_DOUBLE for the 80-bit arbiter build.
 */
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>

#ifdef ORC_LONG_DOUBLE
#define ORC_REAL long double
#define R_SQRT sqrtl
#define R_CONJ conjl
#define R_RE creall
#define R_IM cimagl
#else
#define ORC_REAL double
#define R_SQRT sqrt
#define R_CONJ conj
#define R_RE creal
#define R_IM cimag
#endif
#define R_PI ((real)3.14159265358979323846264338327950288L)
typedef ORC_REAL real;
typedef ORC_REAL _Complex cplx;

#define MAXG 6            /* max number of gluons (g g -> t tbar g g g g: Table 2) */
#define MAXPERM 720
#define NCODE 262144      /* 8^6 tuple codes, digits 1..6 */

/* ------------------------------------------------------------------------------------------ */
/* permutations of n in lexicographic order                                                    */
static int perms_lex(int n, int perm[][MAXG])
{
    int a[MAXG], cnt = 0;
    for (int i = 0; i < n; i++) a[i] = i;
    for (;;) {
        memcpy(perm[cnt++], a, sizeof(int) * MAXG);
        int i = n - 2;
        while (i >= 0 && a[i] > a[i + 1]) i--;
        if (i < 0) break;
        int j = n - 1;
        while (a[j] < a[i]) j--;
        int t = a[i]; a[i] = a[j]; a[j] = t;
        for (int l = i + 1, r = n - 1; l < r; l++, r--) { t = a[l]; a[l] = a[r]; a[r] = t; }
    }
    return cnt;
}

/* ------------------------------------------------------------------------------------------ */
/* SU(3): T^a = lambda^a / 2 with the eight Gell-Mann matrices                                 */
static void su3_generators(double _Complex T[8][3][3])
{
    memset(T, 0, sizeof(double _Complex) * 72);
    const double s3 = 1.0 / sqrt(3.0);
    T[0][0][1] = 1; T[0][1][0] = 1;
    T[1][0][1] = -I; T[1][1][0] = I;
    T[2][0][0] = 1; T[2][1][1] = -1;
    T[3][0][2] = 1; T[3][2][0] = 1;
    T[4][0][2] = -I; T[4][2][0] = I;
    T[5][1][2] = 1; T[5][2][1] = 1;
    T[6][1][2] = -I; T[6][2][1] = I;
    T[7][0][0] = s3; T[7][1][1] = s3; T[7][2][2] = -2 * s3;
    for (int a = 0; a < 8; a++)
        for (int i = 0; i < 3; i++)
            for (int j = 0; j < 3; j++) T[a][i][j] *= 0.5;
}

void orc_su3_generators(double* out /* [8][3][3][2] */)
{
    double _Complex T[8][3][3];
    su3_generators(T);
    for (int a = 0; a < 8; a++)
        for (int i = 0; i < 3; i++)
            for (int j = 0; j < 3; j++) {
                out[((a * 3 + i) * 3 + j) * 2 + 0] = creal(T[a][i][j]);
                out[((a * 3 + i) * 3 + j) * 2 + 1] = cimag(T[a][i][j]);
            }
}

/* C_{ss'} = sum_{a_1..a_n = 1..8} sum_{i,j=1..3} (T^{a_s1}...T^{a_sn})_{ij} conj((T^{a_s'1}...T^{a_s'n})_{ij})
 * by brute force.  Permutations in lexicographic order.  Returns n!; the largest
 * |imaginary part| met (must be rounding noise) is written to *max_imag.                       */
int orc_color_matrix(int n, double* C /* [n!][n!] */, double* max_imag)
{
    if (n < 1 || n > MAXG) return -1;
    double _Complex T[8][3][3];
    su3_generators(T);
    static int perm[MAXPERM][MAXG];
    int np = perms_lex(n, perm);
    long nassign = 1;
    for (int i = 0; i < n; i++) nassign *= 8;
    double _Complex* acc = calloc((size_t)np * np, sizeof(double _Complex));
#pragma omp parallel
    {
        double _Complex* loc = calloc((size_t)np * np, sizeof(double _Complex));
        double _Complex (*chain)[3][3] = malloc(sizeof(double _Complex) * 9 * np);
#pragma omp for schedule(static)
        for (long code = 0; code < nassign; code++) {
            int a[MAXG];
            long c = code;
            for (int i = 0; i < n; i++) { a[i] = (int)(c % 8); c /= 8; }
            for (int s = 0; s < np; s++) {
                double _Complex M[3][3], N[3][3];
                memcpy(M, T[a[perm[s][0]]], sizeof(M));
                for (int k = 1; k < n; k++) {
                    const double _Complex (*X)[3] = T[a[perm[s][k]]];
                    for (int i = 0; i < 3; i++)
                        for (int j = 0; j < 3; j++) {
                            double _Complex v = 0;
                            for (int l = 0; l < 3; l++) v += M[i][l] * X[l][j];
                            N[i][j] = v;
                        }
                    memcpy(M, N, sizeof(M));
                }
                memcpy(chain[s], M, sizeof(M));
            }
            for (int s = 0; s < np; s++)
                for (int t = 0; t < np; t++) {
                    double _Complex v = 0;
                    for (int i = 0; i < 3; i++)
                        for (int j = 0; j < 3; j++) v += chain[s][i][j] * conj(chain[t][i][j]);
                    loc[(size_t)s * np + t] += v;
                }
        }
#pragma omp critical
        for (size_t i = 0; i < (size_t)np * np; i++) acc[i] += loc[i];
        free(loc);
        free(chain);
    }
    double mi = 0;
    for (size_t i = 0; i < (size_t)np * np; i++) {
        C[i] = creal(acc[i]);
        if (fabs(cimag(acc[i])) > mi) mi = fabs(cimag(acc[i]));
    }
    if (max_imag) *max_imag = mi;
    free(acc);
    return np;
}

/* First row only, C_{id,s'} for all s', by the same brute force.  With 6 gluons the full double loop over (s, s')
 * inside the 8^6 colour assignments is out of reach (1.2e12 3x3 products); renaming the summed adjoint indices
 * a_i -> a_{s(i)} in the definition gives C_{s s'} = C_{id, s^-1 o s'}, which the Python front end uses to fill the
 * matrix from this row.  The identity itself is pinned against the full brute force for n <= 5
 * (tests/test_oracle_pins.py).  Returns n!.                                                    */
int orc_color_matrix_row0(int n, double* row /* [n!] */, double* max_imag)
{
    if (n < 1 || n > MAXG) return -1;
    double _Complex T[8][3][3];
    su3_generators(T);
    static int perm[MAXPERM][MAXG];
    int np = perms_lex(n, perm);
    long nassign = 1;
    for (int i = 0; i < n; i++) nassign *= 8;
    double _Complex* acc = calloc((size_t)np, sizeof(double _Complex));
#pragma omp parallel
    {
        double _Complex* loc = calloc((size_t)np, sizeof(double _Complex));
#pragma omp for schedule(static)
        for (long code = 0; code < nassign; code++) {
            int a[MAXG];
            long c = code;
            for (int i = 0; i < n; i++) { a[i] = (int)(c % 8); c /= 8; }
            double _Complex M0[3][3];
            for (int s = 0; s < np; s++) {
                double _Complex M[3][3], N[3][3];
                memcpy(M, T[a[perm[s][0]]], sizeof(M));
                for (int k = 1; k < n; k++) {
                    const double _Complex (*X)[3] = T[a[perm[s][k]]];
                    for (int i = 0; i < 3; i++)
                        for (int j = 0; j < 3; j++) {
                            double _Complex v = 0;
                            for (int l = 0; l < 3; l++) v += M[i][l] * X[l][j];
                            N[i][j] = v;
                        }
                    memcpy(M, N, sizeof(M));
                }
                if (s == 0) memcpy(M0, M, sizeof(M));      /* lexicographic order: permutation 0 is the identity */
                double _Complex v = 0;
                for (int i = 0; i < 3; i++)
                    for (int j = 0; j < 3; j++) v += M0[i][j] * conj(M[i][j]);
                loc[s] += v;
            }
        }
#pragma omp critical
        for (int i = 0; i < np; i++) acc[i] += loc[i];
        free(loc);
    }
    double mi = 0;
    for (int i = 0; i < np; i++) {
        row[i] = creal(acc[i]);
        if (fabs(cimag(acc[i])) > mi) mi = fabs(cimag(acc[i]));
    }
    if (max_imag) *max_imag = mi;
    free(acc);
    return np;
}

/* ------------------------------------------------------------------------------------------ */
/* Lorentz and Dirac algebra, Dirac representation:                                            */
/*   gamma^0 = diag(1,1,-1,-1),  gamma^i = [[0, sigma_i], [-sigma_i, 0]],  gamma_5 = [[0,1],[1,0]] */

static cplx mdot(const cplx a[4], const cplx b[4])
{   /* Minkowski product, no complex conjugation */
    return a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3];
}

static void slash(const cplx a[4], cplx S[4][4])
{   /* a_mu gamma^mu = a0 gamma^0 - a1 gamma^1 - a2 gamma^2 - a3 gamma^3 */
    const cplx a0 = a[0], ax = a[1], ay = a[2], az = a[3];
    /* sigma . a = [[az, ax - i ay], [ax + i ay, -az]] */
    const cplx s00 = az, s01 = ax - I * ay, s10 = ax + I * ay, s11 = -az;
    S[0][0] = a0;  S[0][1] = 0;   S[0][2] = -s00; S[0][3] = -s01;
    S[1][0] = 0;   S[1][1] = a0;  S[1][2] = -s10; S[1][3] = -s11;
    S[2][0] = s00; S[2][1] = s01; S[2][2] = -a0;  S[2][3] = 0;
    S[3][0] = s10; S[3][1] = s11; S[3][2] = 0;    S[3][3] = -a0;
}

static void row_times_mat(const cplx r[4], const cplx M[4][4], cplx out[4])
{
    for (int j = 0; j < 4; j++) {
        cplx v = 0;
        for (int i = 0; i < 4; i++) v += r[i] * M[i][j];
        out[j] = v;
    }
}

static void mat_times_col(const cplx M[4][4], const cplx c[4], cplx out[4])
{
    for (int i = 0; i < 4; i++) {
        cplx v = 0;
        for (int j = 0; j < 4; j++) v += M[i][j] * c[j];
        out[i] = v;
    }
}

/* two-component helicity eigenstates chi_lambda of sigma.p/|p| (lambda = +1, -1) */
static void chi(const real p[4], int lambda, cplx x[2])
{
    const real pp = R_SQRT(p[1] * p[1] + p[2] * p[2] + p[3] * p[3]);
    const real ppz = pp + p[3];
    if (pp == 0 || ppz <= pp * 1e-14) {           /* at rest, or along -z: phi := 0 */
        if (pp == 0) { if (lambda > 0) { x[0] = 1; x[1] = 0; } else { x[0] = 0; x[1] = 1; } }
        else         { if (lambda > 0) { x[0] = 0; x[1] = 1; } else { x[0] = -1; x[1] = 0; } }
        return;
    }
    const real nrm = 1 / R_SQRT(2 * pp * ppz);
    if (lambda > 0) { x[0] = ppz * nrm; x[1] = (p[1] + I * p[2]) * nrm; }
    else            { x[0] = (-p[1] + I * p[2]) * nrm; x[1] = ppz * nrm; }
}

/* u(p, lambda): fermion of mass m, helicity lambda; normalised ubar u = 2m, u^dagger u = 2E */
static void spinor_u(const real p[4], real m, int lambda, cplx u[4])
{
    cplx x[2];
    chi(p, lambda, x);
    const real a = R_SQRT(p[0] + m), b = lambda * R_SQRT(p[0] - m > 0 ? p[0] - m : 0);
    u[0] = a * x[0]; u[1] = a * x[1]; u[2] = b * x[0]; u[3] = b * x[1];
}

/* v(p, lambda): antifermion of physical helicity lambda, built on chi_{-lambda} */
static void spinor_v(const real p[4], real m, int lambda, cplx v[4])
{
    cplx x[2];
    chi(p, -lambda, x);
    const real a = R_SQRT(p[0] + m), b = -lambda * R_SQRT(p[0] - m > 0 ? p[0] - m : 0);
    v[0] = b * x[0]; v[1] = b * x[1]; v[2] = a * x[0]; v[3] = a * x[1];
}

static void dirac_bar(const cplx u[4], cplx ub[4])
{   /* u^dagger gamma^0 */
    ub[0] = R_CONJ(u[0]); ub[1] = R_CONJ(u[1]); ub[2] = -R_CONJ(u[2]); ub[3] = -R_CONJ(u[3]);
}

/* polarisation vector of a massless vector, helicity lambda = +-1, helicity basis:
 *   eps(lambda) = (0, (-lambda e1 - i e2)/sqrt2),  e1 = d p^/d theta, e2 = z^ x p^ / sin theta    */
static void polvec(const real p[4], int lambda, cplx e[4])
{
    const real pt = R_SQRT(p[1] * p[1] + p[2] * p[2]);
    const real pp = R_SQRT(pt * pt + p[3] * p[3]);
    real ct = p[3] / pp, st = pt / pp, cf = 1, sf = 0;
    if (pt > pp * 1e-14) { cf = p[1] / pt; sf = p[2] / pt; } else { st = 0; ct = p[3] > 0 ? 1 : -1; }
    const real e1[3] = { ct * cf, ct * sf, -st };
    const real e2[3] = { -sf, cf, 0 };
    const real r = 1 / R_SQRT((real)2);
    e[0] = 0;
    for (int i = 0; i < 3; i++) e[1 + i] = (-lambda * e1[i] - I * e2[i]) * r;
}

/* ------------------------------------------------------------------------------------------ */
/* colour-ordered Berends-Giele recursion:
 *   J(i) = eps_i ;  K_{i..j} = sum k
 *   J(i..j) = (1/K^2) { -g sum_m V3[J(i..m),K_{i..m}; J(m+1..j),K_{m+1..j}]
 *                       + g^2 sum_{m<m'} V4[J(i..m), J(m+1..m'), J(m'+1..j)] }
 *   V3[A,KA;B,KB] = (A.B)(KA-KB) + ((2KB+KA).A) B - ((2KA+KB).B) A
 *   V4[A,B,C]     = 2(A.C)B - (A.B)C - (B.C)A
 *   Psibar() = ubar(p_t);  Psibar(1..k) = -g [sum_{i<k} Psibar(1..i) Jslash(i+1..k)] (qslash_k + m)/(q_k^2 - m^2 + i m Gamma),
 *              q_k = p_t - K_{1..k}
 *   A(1..n) = g sum_{i<n} Psibar(1..i) Jslash(i+1..n) v(p_tbar)                                   */

typedef struct {
    int n;                   /* number of gluons */
    real k[MAXG][4];         /* all-incoming gluon momenta */
    cplx eps[MAXG][4];
    real pt[4], ptb[4];
    cplx ubar[4], v[4];
    real m, w, g;
    cplx (*J)[4];            /* [NCODE] gluon currents by ordered tuple */
    cplx (*P)[4];            /* [NCODE] quark-line currents by ordered prefix */
    unsigned char* haveJ;
    unsigned char* haveP;
} bg_t;

static int tcode(const int* t, int len)
{   /* ordered tuple -> code (base 8, digits 1..6) */
    int c = 0;
    for (int i = len - 1; i >= 0; i--) c = c * 8 + (t[i] + 1);
    return c;
}

static void tuple_momentum(const bg_t* s, const int* t, int len, cplx K[4])
{
    for (int mu = 0; mu < 4; mu++) {
        real v = 0;
        for (int i = 0; i < len; i++) v += s->k[t[i]][mu];
        K[mu] = v;
    }
}

static const cplx* gluon_current(bg_t* s, const int* t, int len)
{
    const int code = tcode(t, len);
    if (s->haveJ[code]) return s->J[code];
    cplx out[4] = { 0, 0, 0, 0 };
    if (len == 1) {
        for (int mu = 0; mu < 4; mu++) out[mu] = s->eps[t[0]][mu];
    } else {
        cplx K[4];
        tuple_momentum(s, t, len, K);
        /* three-gluon vertices */
        for (int m = 1; m < len; m++) {
            const cplx* A = gluon_current(s, t, m);
            const cplx* B = gluon_current(s, t + m, len - m);
            cplx KA[4], KB[4], d[4], ea[4], eb[4];
            tuple_momentum(s, t, m, KA);
            tuple_momentum(s, t + m, len - m, KB);
            for (int mu = 0; mu < 4; mu++) {
                d[mu] = KA[mu] - KB[mu];
                ea[mu] = 2 * KB[mu] + KA[mu];
                eb[mu] = 2 * KA[mu] + KB[mu];
            }
            const cplx ab = mdot(A, B), xa = mdot(ea, A), xb = mdot(eb, B);
            for (int mu = 0; mu < 4; mu++) out[mu] += -s->g * (ab * d[mu] + xa * B[mu] - xb * A[mu]);
        }
        /* four-gluon vertices */
        for (int m = 1; m < len; m++)
            for (int m2 = m + 1; m2 < len; m2++) {
                const cplx* A = gluon_current(s, t, m);
                const cplx* B = gluon_current(s, t + m, m2 - m);
                const cplx* C = gluon_current(s, t + m2, len - m2);
                const cplx ac = mdot(A, C), ab = mdot(A, B), bc = mdot(B, C);
                for (int mu = 0; mu < 4; mu++)
                    out[mu] += s->g * s->g * (2 * ac * B[mu] - ab * C[mu] - bc * A[mu]);
            }
        const cplx K2 = mdot(K, K);
        for (int mu = 0; mu < 4; mu++) out[mu] /= K2;
    }
    for (int mu = 0; mu < 4; mu++) s->J[code][mu] = out[mu];
    s->haveJ[code] = 1;
    return s->J[code];
}

static const cplx* quark_current(bg_t* s, const int* t, int len)
{   /* Psibar(t[0..len)) as a row spinor */
    const int code = tcode(t, len);
    if (s->haveP[code]) return s->P[code];
    cplx out[4] = { 0, 0, 0, 0 };
    if (len == 0) {
        for (int a = 0; a < 4; a++) out[a] = s->ubar[a];
    } else {
        cplx acc[4] = { 0, 0, 0, 0 };
        for (int i = 0; i < len; i++) {
            const cplx* psi = quark_current(s, t, i);
            const cplx* Jc = gluon_current(s, t + i, len - i);
            cplx S[4][4], r[4];
            slash(Jc, S);
            row_times_mat(psi, S, r);
            for (int a = 0; a < 4; a++) acc[a] += r[a];
        }
        cplx K[4], q[4], S[4][4], r[4];
        tuple_momentum(s, t, len, K);
        for (int mu = 0; mu < 4; mu++) q[mu] = s->pt[mu] - K[mu];
        slash(q, S);
        for (int a = 0; a < 4; a++) S[a][a] += s->m;
        row_times_mat(acc, S, r);
        const cplx den = mdot(q, q) - s->m * s->m + I * s->m * s->w;
        for (int a = 0; a < 4; a++) out[a] = -s->g * r[a] / den;
    }
    for (int a = 0; a < 4; a++) s->P[code][a] = out[a];
    s->haveP[code] = 1;
    return s->P[code];
}

static cplx partial_amplitude(bg_t* s, const int* sigma)
{
    cplx A = 0;
    for (int i = 0; i < s->n; i++) {
        const cplx* psi = quark_current(s, sigma, i);
        const cplx* Jc = gluon_current(s, sigma + i, s->n - i);
        cplx S[4][4], c[4];
        slash(Jc, S);
        mat_times_col(S, s->v, c);
        for (int a = 0; a < 4; a++) A += psi[a] * c[a];
    }
    return s->g * A;
}

static void bg_alloc(bg_t* s)
{
    s->J = malloc(sizeof(cplx) * 4 * NCODE);
    s->P = malloc(sizeof(cplx) * 4 * NCODE);
    s->haveJ = malloc(NCODE);
    s->haveP = malloc(NCODE);
}

static void bg_free(bg_t* s)
{
    free(s->J); free(s->P); free(s->haveJ); free(s->haveP);
}

/* Set up one (event, helicity): particle order g g t tbar g...; gluon list = particles 0,1,4,5,.. */
static void bg_setup(bg_t* s, int n, const double* mom /* [n+2][4] */, const int* hel /* [n+2], +-1 */,
                     real mt, real wt, real gs, const double* eps_override /* [n][4][2] or NULL */)
{
    s->n = n; s->m = mt; s->w = wt; s->g = gs;
    memset(s->haveJ, 0, NCODE);
    memset(s->haveP, 0, NCODE);
    for (int ig = 0; ig < n; ig++) {
        const int ip = ig < 2 ? ig : ig + 2;
        real p[4];
        for (int mu = 0; mu < 4; mu++) p[mu] = mom[ip * 4 + mu];
        const real sgn = ig < 2 ? 1 : -1;
        for (int mu = 0; mu < 4; mu++) s->k[ig][mu] = sgn * p[mu];
        cplx e[4];
        polvec(p, hel[ip], e);
        if (ig >= 2) for (int mu = 0; mu < 4; mu++) e[mu] = R_CONJ(e[mu]);
        if (eps_override)
            for (int mu = 0; mu < 4; mu++)
                e[mu] = eps_override[(ig * 4 + mu) * 2] + I * eps_override[(ig * 4 + mu) * 2 + 1];
        for (int mu = 0; mu < 4; mu++) s->eps[ig][mu] = e[mu];
    }
    for (int mu = 0; mu < 4; mu++) { s->pt[mu] = mom[2 * 4 + mu]; s->ptb[mu] = mom[3 * 4 + mu]; }
    cplx u[4];
    spinor_u(s->pt, mt, hel[2], u);
    dirac_bar(u, s->ubar);
    spinor_v(s->ptb, mt, hel[3], s->v);
}

/* Partial amplitudes A(sigma), sigma over the n! lexicographic permutations of the gluon list,
 * for one event and one helicity assignment.  eps_override lets a test replace polarisations
 * (gauge-invariance pin P3).                                                                  */
int orc_ggttx_partial(int n, const double* mom, const int* hel, double mt, double wt, double gs,
                      const double* eps_override, double* A /* [n!][2] */)
{
    if (n < 2 || n > MAXG) return -1;
    static int perm[MAXPERM][MAXG];
    int np;
#pragma omp critical(orc_perm)
    np = perms_lex(n, perm);
    bg_t s;
    bg_alloc(&s);
    bg_setup(&s, n, mom, hel, mt, wt, gs, eps_override);
    for (int i = 0; i < np; i++) {
        cplx a = partial_amplitude(&s, perm[i]);
        A[2 * i] = (double)R_RE(a);
        A[2 * i + 1] = (double)R_IM(a);
    }
    bg_free(&s);
    return np;
}

/* me[e] = (1/denom) sum_h sum_{ss'} conj(A_h(s)) C_{ss'} A_h(s');  me_hel (nullable) gets the
 * per-helicity terms sum_{ss'}(...)/denom, [nevt][2^npar], helicity index as in reading A2.     */
int orc_me_ggttx(int n, const double* mom /* [nevt][n+2][4] */, long nevt, double mt, double wt, double gs,
                 const double* C /* [n!][n!] */, double denom, double* me, double* me_hel)
{
    if (n < 2 || n > MAXG) return -1;
    const int npar = n + 2, ncomb = 1 << npar;
    static int perm[MAXPERM][MAXG];
    const int np = perms_lex(n, perm);
#pragma omp parallel
    {
        bg_t s;
        bg_alloc(&s);
        cplx* A = malloc(sizeof(cplx) * np);
#pragma omp for schedule(dynamic, 1)
        for (long e = 0; e < nevt; e++) {
            real tot = 0;
            for (int h = 0; h < ncomb; h++) {
                int hel[MAXG + 2];
                for (int i = 0; i < npar; i++) hel[i] = ((h >> (npar - 1 - i)) & 1) ? 1 : -1;
                bg_setup(&s, n, mom + e * npar * 4, hel, mt, wt, gs, NULL);
                for (int i = 0; i < np; i++) A[i] = partial_amplitude(&s, perm[i]);
                cplx q = 0;
                for (int i = 0; i < np; i++)
                    for (int j = 0; j < np; j++) q += R_CONJ(A[i]) * (real)C[(size_t)i * np + j] * A[j];
                const real meh = R_RE(q) / denom;
                if (me_hel) me_hel[e * ncomb + h] = (double)meh;
                tot += meh;
            }
            me[e] = (double)tot;
        }
        free(A);
        bg_free(&s);
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------ */
/* e+ e- -> mu+ mu-  (BASELINE.json config 1; particle order e+ e- mu+ mu-), photon + Z, s-channel:
 *   M_h = sum_V [vbar(e+) gamma^mu G_V u(e-)] [ubar(mu-) gamma_mu G_V v(mu+)] P_V
 *   G_gamma = -e (Q = -1), P_gamma = 1/s;  G_Z = gL PL + gR PR, P_Z = 1/(s - mZ^2 + i mZ wZ)
 *   gL = e(-1/2 + sW^2)/(sW cW), gR = e sW/cW, e = sqrt(4 pi alpha), sW^2 = 1 - mW^2/mZ^2.
 * The k^mu k^nu/mZ^2 propagator term vanishes for massless leptons.  denom = 4.                 */
int orc_me_eemumu(const double* mom /* [nevt][4][4] */, long nevt, double alpha, double mZ, double wZ, double mW,
                  double* me, double* me_hel /* nullable [nevt][16] */)
{
    const real ee = R_SQRT(4 * R_PI * alpha);
    const real sw2 = 1 - (real)mW * mW / ((real)mZ * mZ);
    const real sw = R_SQRT(sw2), cw = R_SQRT(1 - sw2);
    const real gL = ee * (-(real)0.5 + sw2) / (sw * cw), gR = ee * sw / cw;
#pragma omp parallel for schedule(static)
    for (long e = 0; e < nevt; e++) {
        real p[4][4];
        for (int i = 0; i < 4; i++)
            for (int mu = 0; mu < 4; mu++) p[i][mu] = mom[(e * 4 + i) * 4 + mu];
        real q[4];
        for (int mu = 0; mu < 4; mu++) q[mu] = p[0][mu] + p[1][mu];
        const real s = q[0] * q[0] - q[1] * q[1] - q[2] * q[2] - q[3] * q[3];
        const cplx PZ = 1 / (s - (real)mZ * mZ + I * (real)mZ * wZ);
        const real PA = 1 / s;
        real tot = 0;
        for (int h = 0; h < 16; h++) {
            int hel[4];
            for (int i = 0; i < 4; i++) hel[i] = ((h >> (3 - i)) & 1) ? 1 : -1;
            cplx vep[4], vbar[4], uem[4], umu[4], ubar[4], vmu[4];
            spinor_v(p[0], 0, hel[0], vep);  dirac_bar(vep, vbar);      /* incoming e+  : vbar */
            spinor_u(p[1], 0, hel[1], uem);                              /* incoming e-  : u    */
            spinor_v(p[2], 0, hel[2], vmu);                              /* outgoing mu+ : v    */
            spinor_u(p[3], 0, hel[3], umu);  dirac_bar(umu, ubar);      /* outgoing mu- : ubar */
            /* chiral projections in the Dirac representation: gamma5 = [[0,1],[1,0]] */
            cplx uL[4], uR[4], vL[4], vR[4];
            for (int a = 0; a < 2; a++) {
                uL[a] = (uem[a] - uem[a + 2]) / 2; uL[a + 2] = -uL[a];
                uR[a] = (uem[a] + uem[a + 2]) / 2; uR[a + 2] = uR[a];
                vL[a] = (vmu[a] - vmu[a + 2]) / 2; vL[a + 2] = -vL[a];
                vR[a] = (vmu[a] + vmu[a + 2]) / 2; vR[a + 2] = vR[a];
            }
            cplx M = 0;
            for (int mu = 0; mu < 4; mu++) {
                cplx unit[4] = { 0, 0, 0, 0 }, G[4][4], c[4];
                unit[mu] = 1;                      /* slash(unit) = gamma^mu with lower index contracted: g_{mu mu} handled below */
                slash(unit, G);                    /* = g_{mu mu} gamma^mu */
                const real gmm = mu == 0 ? 1 : -1; /* so gamma^mu = gmm * G */
                cplx eA = 0, eL = 0, eR = 0, mA = 0, mL = 0, mR = 0;
                mat_times_col(G, uem, c); for (int a = 0; a < 4; a++) eA += vbar[a] * c[a];
                mat_times_col(G, uL, c);  for (int a = 0; a < 4; a++) eL += vbar[a] * c[a];
                mat_times_col(G, uR, c);  for (int a = 0; a < 4; a++) eR += vbar[a] * c[a];
                mat_times_col(G, vmu, c); for (int a = 0; a < 4; a++) mA += ubar[a] * c[a];
                mat_times_col(G, vL, c);  for (int a = 0; a < 4; a++) mL += ubar[a] * c[a];
                mat_times_col(G, vR, c);  for (int a = 0; a < 4; a++) mR += ubar[a] * c[a];
                /* J_e^mu J_mu,mu = sum_mu g_{mu mu} J^mu J^mu, and J^mu = gmm * (bar G .) each: gmm^3 = gmm */
                M += gmm * ((-ee * eA) * (-ee * mA) * PA + (gL * eL + gR * eR) * (gL * mL + gR * mR) * PZ);
            }
            const real meh = (R_RE(M) * R_RE(M) + R_IM(M) * R_IM(M)) / 4;
            if (me_hel) me_hel[e * 16 + h] = (double)meh;
            tot += meh;
        }
        me[e] = (double)tot;
    }
    return 0;
}

int orc_real_bits(void) { return (int)(8 * sizeof(real)); }
