/*
 * ris_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, CPU-only oracle for the TDDFT-ris derivative-integral contractions
 *   G_J [A,x] = sum_{mu nu} sum_P D_{mu nu} c_P  d(mu nu|P)/dR_{A,x}
 *   G_K [A,x] = sum_P sum_{mu nu} Gamma^P_{mu nu} d(mu nu|P)/dR_{A,x}
 *   G_PQ[A,x] = sum_{PQ} c_P d_Q d(P|Q)/dR_{A,x}
 * i.e. the integral-derivative factors of the first two terms and of the third term of
 * Eq. 27, for the three-centre integrals (pq|A) and metric M_AB=(A|B) of
 * Eqs. 21-22, with the minimal auxiliary basis of one s-type Gaussian
 * per atom.  (pq|sr) is in charge-cloud notation, Eq. 7.
 * The derivative is the TOTAL nuclear derivative (xi is a nuclear coordinate, Eq. 8,
 * PAPER.md:62-65): every centre that sits on atom A moves.
 *
 * The paper does not describe the integral evaluation ("We will not discuss the details of
 * these integral evaluation algorithms"), so the oracle writes out the
 * textbook McMurchie-Davidson definition, step by step, with no
 * blocking, screening (except the documented opt-in primitive cutoff), symmetry or
 * translational-invariance shortcuts: all ORDERED (mu,nu) pairs are visited and the three
 * centre derivatives are computed explicitly.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg
 * may call this file.  It shares no code with paper_2511_18233_b200/csrc.
 *
 * Pins (tests/test_oracle_pins.py): closed-form sss value and gradient, Boys reference
 * values / erf / incomplete gamma / quadrature, the worked example of SURVEY.md 8(c) P4-P5,
 * finite differences, translational invariance, brute-force quadrature, far-aux limit.
 * Nothing in this file is "parity unpinned".
 *
 * NEXT-2 ("a single GTO for each angular momentum component (up to l = 2) on each atom",
 * PAPER.md:168 "s- and p-type for Coulomb, only s-type for exchange"): the J-fit auxiliary set may hold p-type functions.
 * An auxiliary FUNCTION is (atom, l in {0,1}, Cartesian component i, exponent); the p function
 *   chi_{P,i}(r) = N_p (r - C)_i exp(-alpha |r-C|^2),  N_p = (2 alpha/pi)^(3/4) 2 sqrt(alpha)   (normalised)
 * is the centre derivative of the s primitive, (r-C)_i e^{..} = (1/2 alpha) d/dC_i e^{..}, so in the Hermite basis it only
 * shifts the Coulomb tensor: [ab|p_i] = -(1/2 alpha) pref sum E_tuv R_{tuv + 1_i}.  mol->naux_fn = 0 selects the default
 * set (one s function per atom, exponent aux_exponents[atom]).
 *
 * Conventions: atomic units; row-major double arrays; Cartesian component order inside a
 * shell: lx descending, then ly descending (xx,xy,xz,yy,yz,zz; ...).  prim_coef is applied
 * as-is to UNnormalised primitives; the aux function carries N_P = (2 alpha/pi)^(3/4).
 */
#include <math.h>
#include <tgmath.h>            /* exp / sqrt / pow / fabs pick the precision of their argument */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define LMAX 3                 /* shells up to f */
#define EMAX (LMAX + 1)        /* one raised by the derivative */
#define TMAX (2 * EMAX + 2)    /* Hermite order bound (+1 for the aux derivative) */
#define MMAX (TMAX + 1)

/* Working precision of every intermediate (E, R, Boys values, prefactors, per-pair buffers).  The oracle IS the
 * default build (double: "FP64 unless the paper fixes the precision"); `-DORACLE_REAL="long double"` builds the same
 * source with x87 extended intermediates, used only by tests/test_oracle_pins.py to measure the oracle's own FP64
 * rounding error (the evidence behind the parity tolerance, reading R-tol).  Inputs / outputs stay double. */
#ifndef ORACLE_REAL
#define ORACLE_REAL double
#endif
typedef ORACLE_REAL real;

static const real PI = (real)3.14159265358979323846264338327950288L;

/* ---------------------------------------------------------------- O1: Boys function
 * F_m(T) = int_0^1 t^(2m) exp(-T t^2) dt.
 * T < 35: F_M = e^-T sum_k (2T)^k / [(2M+1)(2M+3)...(2M+2k+1)] at M = mmax, then downward
 *         F_m = (2T F_{m+1} + e^-T)/(2m+1).
 * T >= 35: F_0 = 1/2 sqrt(pi/T) erf(sqrt T), upward F_{m+1} = ((2m+1)F_m - e^-T)/(2T).
 */
static void boys_real(int mmax, real T, real *F)
{
    if (T < 35.0) {
        long double t = (long double)T;
        long double et = expl(-t);
        long double term = 1.0L / (2 * mmax + 1);
        long double sum = term;
        for (int k = 1; k < 2000; ++k) {
            term *= 2.0L * t / (2 * mmax + 2 * k + 1);
            sum += term;
            if (term < 1e-22L * sum) break;
        }
        long double f = et * sum;
        F[mmax] = (real)f;
        for (int m = mmax - 1; m >= 0; --m) {
            f = (2.0L * t * f + et) / (2 * m + 1);
            F[m] = (real)f;
        }
    } else {
        long double t = (long double)T;
        long double et = expl(-t);
        long double f = 0.5L * sqrtl(3.14159265358979323846264338327950288L / t) * erfl(sqrtl(t));
        F[0] = (real)f;
        for (int m = 0; m < mmax; ++m) {
            f = ((2 * m + 1) * f - et) / (2.0L * t);
            F[m + 1] = (real)f;
        }
    }
}

void ris_oracle_boys(int mmax, double T, double *F)
{
    real Fr[64];
    boys_real(mmax, (real)T, Fr);
    for (int m = 0; m <= mmax; ++m) F[m] = (double)Fr[m];
}

/* ---------------------------------------------------------------- O2: Hermite expansion
 * E[i][j][t], 0<=i<=imax, 0<=j<=jmax, one Cartesian direction.  Q = A_x - B_x.
 *   E^{00}_0 = exp(-q Q^2),  q = ab/p
 *   E^{i+1,j}_t = E^{ij}_{t-1}/(2p) - (q Q/a) E^{ij}_t + (t+1) E^{ij}_{t+1}
 *   E^{i,j+1}_t = E^{ij}_{t-1}/(2p) + (q Q/b) E^{ij}_t + (t+1) E^{ij}_{t+1}
 */
typedef real Etab[EMAX + 1][EMAX + 1][2 * EMAX + 2];

static void hermite_E(int imax, int jmax, real a, real b, real Q, Etab E)
{
    real p = a + b, q = a * b / p;
    memset(E, 0, sizeof(Etab));
    E[0][0][0] = exp(-q * Q * Q);
    for (int i = 0; i <= imax; ++i) {
        for (int j = 0; j <= jmax; ++j) {
            if (i == 0 && j == 0) continue;
            for (int t = 0; t <= i + j; ++t) {
                real lo, mid, hi;
                if (j == 0) {           /* raise i from (i-1, 0) */
                    lo = (t > 0) ? E[i - 1][j][t - 1] : 0.0;
                    mid = E[i - 1][j][t];
                    hi = (t + 1 <= i - 1 + j) ? E[i - 1][j][t + 1] : 0.0;
                    E[i][j][t] = lo / (2 * p) - (q * Q / a) * mid + (t + 1) * hi;
                } else {                /* raise j from (i, j-1) */
                    lo = (t > 0) ? E[i][j - 1][t - 1] : 0.0;
                    mid = E[i][j - 1][t];
                    hi = (t + 1 <= i + j - 1) ? E[i][j - 1][t + 1] : 0.0;
                    E[i][j][t] = lo / (2 * p) + (q * Q / b) * mid + (t + 1) * hi;
                }
            }
        }
    }
}

/* ---------------------------------------------------------------- O3: Hermite Coulomb
 * R^n_{000} = (-2 rho)^n F_n(T);  R^n_{t+1,u,v} = t R^{n+1}_{t-1,u,v} + X_x R^{n+1}_{t,u,v}
 * (same in y and z).  Output R[t][u][v] = R^0_{tuv} for t+u+v <= nmax.
 */
typedef real Rtab[TMAX + 1][TMAX + 1][TMAX + 1];

static void hermite_R(int nmax, real rho, const real X[3], Rtab R0)
{
    real F[MMAX + 1];
    real T = rho * (X[0] * X[0] + X[1] * X[1] + X[2] * X[2]);
    boys_real(nmax, T, F);
    /* Rn[n][t][u][v]; every entry read below has been written before it is read */
    int N = nmax + 1;
    real Rn[N][N][N][N];
    real pw = 1.0;
    for (int n = 0; n <= nmax; ++n) { Rn[n][0][0][0] = pw * F[n]; pw *= -2.0 * rho; }
    for (int tot = 1; tot <= nmax; ++tot)
        for (int t = 0; t <= tot; ++t)
            for (int u = 0; u <= tot - t; ++u) {
                int v = tot - t - u;
                for (int n = 0; n <= nmax - tot; ++n) {
                    real val;
                    if (t > 0)
                        val = ((t > 1) ? (t - 1) * Rn[n + 1][t - 2][u][v] : 0.0) + X[0] * Rn[n + 1][t - 1][u][v];
                    else if (u > 0)
                        val = ((u > 1) ? (u - 1) * Rn[n + 1][t][u - 2][v] : 0.0) + X[1] * Rn[n + 1][t][u - 1][v];
                    else
                        val = ((v > 1) ? (v - 1) * Rn[n + 1][t][u][v - 2] : 0.0) + X[2] * Rn[n + 1][t][u][v - 1];
                    Rn[n][t][u][v] = val;
                }
            }
    for (int t = 0; t <= nmax; ++t)
        for (int u = 0; u <= nmax - t; ++u)
            for (int v = 0; v <= nmax - t - u; ++v) R0[t][u][v] = Rn[0][t][u][v];
}

/* sum_{tuv} Ex[t] Ey[u] Ez[v] R[t+dt][u+du][v+dv] */
static real hsum(const real *Ex, int nx, const real *Ey, int ny, const real *Ez, int nz,
                 Rtab R, int dt, int du, int dv)
{
    long double s = 0.0L;
    for (int t = 0; t <= nx; ++t)
        for (int u = 0; u <= ny; ++u)
            for (int v = 0; v <= nz; ++v) s += (long double)(Ex[t] * Ey[u] * Ez[v]) * R[t + dt][u + du][v + dv];
    return (real)s;
}

/* ---------------------------------------------------------------- O4/O5: one primitive integral
 * Unnormalised Cartesian primitives la=(lax,lay,laz) at A (exponent a), lb at B (exponent b);
 * s-type aux exp(-alpha |r-C|^2) WITHOUT N_P.
 *   [ab|P]       = 2 pi^{5/2}/(p alpha sqrt(p+alpha)) sum_{tuv} E_t E_u E_v R^0_{tuv}
 *   d/dA_x[ab|P] = 2a [a+1_x,b|P] - a_x [a-1_x,b|P]          (same for B with b)
 *   d/dC_x[ab|P] = -pref sum E_tuv R^0_{t+1,u,v}              (explicit aux derivative)
 * out[0] = value, out[1..3] = d/dA, out[4..6] = d/dB, out[7..9] = d/dC.
 */
void ris_oracle_prim3c_aux(const int la[3], const int lb[3], double a_, double b_, double alpha_,
                           const double A[3], const double B[3], const double C[3], int aux_l, int aux_comp, double out[10]);

void ris_oracle_prim3c(const int la[3], const int lb[3], double a_, double b_, double alpha_,
                       const double A[3], const double B[3], const double C[3], double out[10])
{
    ris_oracle_prim3c_aux(la, lb, a_, b_, alpha_, A, B, C, 0, 0, out);
}

/* The same for an unnormalised auxiliary primitive of type aux_l (0: s, 1: p with component aux_comp):
 *   [ab|p_i] = (1/2 alpha) d/dC_i [ab|s] = -(1/2 alpha) pref sum E_tuv R_{tuv + 1_i}           (R depends on P - C)
 * i.e. the Coulomb tensor is read with the shift sh = 1_i and the factor fP = -1/(2 alpha) (s: sh = 0, fP = 1);
 * d/dC_d shifts once more and flips the sign. */
void ris_oracle_prim3c_aux(const int la[3], const int lb[3], double a_, double b_, double alpha_,
                           const double A[3], const double B[3], const double C[3], int aux_l, int aux_comp, double out[10])
{
    real a = a_, b = b_, alpha = alpha_;
    const int sh0 = (aux_l == 1 && aux_comp == 0), sh1 = (aux_l == 1 && aux_comp == 1), sh2 = (aux_l == 1 && aux_comp == 2);
    const real fP = aux_l == 1 ? -1.0 / (2.0 * alpha) : 1.0;
    real p = a + b, rho = p * alpha / (p + alpha);
    real P[3], X[3];
    Etab E[3];
    for (int d = 0; d < 3; ++d) {
        P[d] = (a * A[d] + b * B[d]) / p;
        X[d] = P[d] - C[d];
        hermite_E(la[d] + 1, lb[d] + 1, a, b, (real)A[d] - B[d], E[d]);
    }
    int L = la[0] + la[1] + la[2] + lb[0] + lb[1] + lb[2];
    Rtab *R = malloc(sizeof(Rtab));
    hermite_R(L + 2 + aux_l, rho, X, *R);
    real pref = fP * 2.0 * pow(PI, (real)2.5) / (p * alpha * sqrt(p + alpha));
#define EE(d, i, j) E[d][i][j], (i) + (j)
    out[0] = pref * hsum(EE(0, la[0], lb[0]), EE(1, la[1], lb[1]), EE(2, la[2], lb[2]), *R, sh0, sh1, sh2);
    for (int d = 0; d < 3; ++d) {
        int ia[3] = {la[0], la[1], la[2]}, ib[3] = {lb[0], lb[1], lb[2]};
        real up, dn;
        /* bra centre A */
        ia[d] = la[d] + 1;
        up = hsum(EE(0, ia[0], ib[0]), EE(1, ia[1], ib[1]), EE(2, ia[2], ib[2]), *R, sh0, sh1, sh2);
        dn = 0.0;
        if (la[d] > 0) {
            ia[d] = la[d] - 1;
            dn = hsum(EE(0, ia[0], ib[0]), EE(1, ia[1], ib[1]), EE(2, ia[2], ib[2]), *R, sh0, sh1, sh2);
        }
        out[1 + d] = pref * (2.0 * a * up - la[d] * dn);
        ia[d] = la[d];
        /* ket-side bra centre B */
        ib[d] = lb[d] + 1;
        up = hsum(EE(0, ia[0], ib[0]), EE(1, ia[1], ib[1]), EE(2, ia[2], ib[2]), *R, sh0, sh1, sh2);
        dn = 0.0;
        if (lb[d] > 0) {
            ib[d] = lb[d] - 1;
            dn = hsum(EE(0, ia[0], ib[0]), EE(1, ia[1], ib[1]), EE(2, ia[2], ib[2]), *R, sh0, sh1, sh2);
        }
        out[4 + d] = pref * (2.0 * b * up - lb[d] * dn);
        ib[d] = lb[d];
        /* aux centre C, explicitly */
        out[7 + d] = -pref * hsum(EE(0, la[0], lb[0]), EE(1, la[1], lb[1]), EE(2, la[2], lb[2]), *R,
                                  sh0 + (d == 0), sh1 + (d == 1), sh2 + (d == 2));
    }
#undef EE
    free(R);
}

/* ---------------------------------------------------------------- O7: two-centre term
 * (P|Q) = 2 pi^{5/2}/(alpha beta sqrt(alpha+beta)) F_0(rho R^2), rho = alpha beta/(alpha+beta)
 * d/dR_P = -2 rho (R_P-R_Q) * 2 pi^{5/2}/(alpha beta sqrt(alpha+beta)) * F_1(rho R^2) = -d/dR_Q.
 * WITHOUT N_P N_Q.  out[0]=value, out[1..3] = d/dR_P.
 */
void ris_oracle_prim2c(double alpha_, double beta_, const double RP[3], const double RQ[3], double out[4])
{
    real alpha = alpha_, beta = beta_;
    real rho = alpha * beta / (alpha + beta);
    real X[3] = {(real)RP[0] - RQ[0], (real)RP[1] - RQ[1], (real)RP[2] - RQ[2]};
    real F[2];
    boys_real(1, rho * (X[0] * X[0] + X[1] * X[1] + X[2] * X[2]), F);
    real pref = 2.0 * pow(PI, (real)2.5) / (alpha * beta * sqrt(alpha + beta));
    out[0] = pref * F[0];
    for (int d = 0; d < 3; ++d) out[1 + d] = -2.0 * rho * X[d] * pref * F[1];
}

/* Two-centre integral between unnormalised auxiliary primitives of type (lP, iP) at RP and (lQ, iQ) at RQ (l in {0,1}):
 * in the Hermite basis, with X = RP - RQ,
 *   (Lambda_t^P | Lambda_u^Q) = (-1)^|u| kappa R_{t+u}(rho, X),  kappa = 2 pi^{5/2}/(alpha beta sqrt(alpha+beta)),
 * and p_i = Lambda_{1_i}/(2 exponent).  out[0] = value, out[1..3] = d/dR_P (= -d/dR_Q: a function of X only). */
void ris_oracle_prim2c_lm(double alpha_, double beta_, int lP, int iP, int lQ, int iQ, const double RP[3], const double RQ[3],
                          double out[4])
{
    real alpha = alpha_, beta = beta_;
    real rho = alpha * beta / (alpha + beta);
    real X[3] = {(real)RP[0] - RQ[0], (real)RP[1] - RQ[1], (real)RP[2] - RQ[2]};
    Rtab *R = malloc(sizeof(Rtab));
    hermite_R(lP + lQ + 1, rho, X, *R);
    int sh[3] = {0, 0, 0};
    if (lP == 1) sh[iP] += 1;
    if (lQ == 1) sh[iQ] += 1;
    real g = 2.0 * pow(PI, (real)2.5) / (alpha * beta * sqrt(alpha + beta));
    if (lP == 1) g /= 2.0 * alpha;
    if (lQ == 1) g /= -2.0 * beta;          /* (-1)^|u| */
    out[0] = (double)(g * (*R)[sh[0]][sh[1]][sh[2]]);
    for (int d = 0; d < 3; ++d) out[1 + d] = (double)(g * (*R)[sh[0] + (d == 0)][sh[1] + (d == 1)][sh[2] + (d == 2)]);
    free(R);
}

/* ---------------------------------------------------------------- molecule description */
typedef struct {
    int natoms;
    const double *coords;          /* [natoms][3] */
    int nshells;
    const int32_t *shell_atom, *shell_l, *shell_nprim, *shell_prim_off;
    const double *prim_exp, *prim_coef;
    const double *aux_exponents;   /* [natoms]: the default set, one s function per atom */
    /* optional explicit auxiliary FUNCTION list (NEXT-2, the J-fit set); naux_fn = 0: the default set above */
    int naux_fn;
    const int32_t *aux_atom, *aux_l, *aux_comp;    /* [naux_fn] */
    const double *aux_exp;                         /* [naux_fn] */
} ris_oracle_mol;

static int aux_count(const ris_oracle_mol *m) { return m->naux_fn > 0 ? m->naux_fn : m->natoms; }
static int aux_atom_of(const ris_oracle_mol *m, int P) { return m->naux_fn > 0 ? m->aux_atom[P] : P; }
static int aux_l_of(const ris_oracle_mol *m, int P) { return m->naux_fn > 0 ? m->aux_l[P] : 0; }
static int aux_comp_of(const ris_oracle_mol *m, int P) { return m->naux_fn > 0 ? m->aux_comp[P] : 0; }
static double aux_exp_of(const ris_oracle_mol *m, int P) { return m->naux_fn > 0 ? m->aux_exp[P] : m->aux_exponents[P]; }

static int ncart(int l) { return (l + 1) * (l + 2) / 2; }

static void cart_components(int l, int comp[][3])
{
    int n = 0;
    for (int lx = l; lx >= 0; --lx)
        for (int ly = l - lx; ly >= 0; --ly) {
            comp[n][0] = lx; comp[n][1] = ly; comp[n][2] = l - lx - ly; ++n;
        }
}

static real aux_norm(real alpha) { return pow(2.0 * alpha / PI, (real)0.75); }
/* normalised Cartesian p: N_p = (2 alpha/pi)^(3/4) (4 alpha)^(1/2) */
static real aux_norm_l(real alpha, int l) { return l == 1 ? aux_norm(alpha) * 2.0 * sqrt(alpha) : aux_norm(alpha); }

/* ---------------------------------------------------------------- O6: contraction for one aux P
 * For aux function P (on atom P) and nmat dense matrices G_s[nao][nao] with scale factors
 * scale[s]:
 *   eacc[s]        += scale[s] sum_{mu nu} G_s[mu,nu] (mu nu|P)
 *   gacc[s][A][x]  += scale[s] sum_{mu nu} G_s[mu,nu] d(mu nu|P)/dR_{A,x}
 * over ALL ordered (mu,nu).  J-type: G = D, scale = c_P.  K-type: G = Gamma^P, scale = 1.
 * atom_mask (nullable): when given, only triplets that touch a masked atom are visited and
 * only masked atoms' rows of gacc are meaningful (used to sample outputs at full size).
 * prim_cutoff: a primitive pair is skipped when |d_a d_b| K_ab (pi/p)^{3/2} < prim_cutoff
 * (0 = no cutoff; 1e-22 for the 300-atom config only).
 * Accumulation in long double.
 */
int ris_oracle_contract_P(const ris_oracle_mol *mol, int P, int nmat, const double *G,
                          const double *scale, const uint8_t *atom_mask, double prim_cutoff,
                          long double *gacc, long double *eacc)
{
    int natoms = mol->natoms, nsh = mol->nshells;
    int *ao_off = malloc(sizeof(int) * (size_t)(nsh + 1));
    ao_off[0] = 0;
    for (int s = 0; s < nsh; ++s) {
        if (mol->shell_l[s] < 0 || mol->shell_l[s] > LMAX) { free(ao_off); return -1; }
        ao_off[s + 1] = ao_off[s] + ncart(mol->shell_l[s]);
    }
    int nao = ao_off[nsh];
    real alpha = aux_exp_of(mol, P);
    const int lP = aux_l_of(mol, P), iP = aux_comp_of(mol, P), atP = aux_atom_of(mol, P);
    /* s: Coulomb tensor as it is; p_i: shifted by 1_i, factor -1/(2 alpha) (see ris_oracle_prim3c_aux) */
    const int sh0 = (lP == 1 && iP == 0), sh1 = (lP == 1 && iP == 1), sh2 = (lP == 1 && iP == 2);
    real NP = lP == 1 ? aux_norm_l(alpha, 1) * (-1.0 / (2.0 * alpha)) : aux_norm(alpha);
    const double *C = mol->coords + 3 * atP;
    int Pmasked = atom_mask ? atom_mask[atP] : 1;
    size_t ng = (size_t)nmat * natoms * 3;

#pragma omp parallel
    {
        long double *gl = calloc(ng, sizeof(long double));
        long double *el = calloc((size_t)nmat, sizeof(long double));
        real *buf = malloc(sizeof(real) * 10 * 10 * 10);   /* [ca][cb][10] */
#pragma omp for schedule(dynamic, 1)
        for (int sa = 0; sa < nsh; ++sa) {
            int la = mol->shell_l[sa], at_a = mol->shell_atom[sa];
            int na = ncart(la);
            int compa[10][3];
            cart_components(la, compa);
            const double *A = mol->coords + 3 * at_a;
            for (int sb = 0; sb < nsh; ++sb) {
                int lb = mol->shell_l[sb], at_b = mol->shell_atom[sb];
                if (atom_mask && !Pmasked && !atom_mask[at_a] && !atom_mask[at_b]) continue;
                int nb = ncart(lb);
                int compb[10][3];
                cart_components(lb, compb);
                const double *Bc = mol->coords + 3 * at_b;
                memset(buf, 0, sizeof(real) * 1000);
                real AB2 = 0.0;
                for (int d = 0; d < 3; ++d) AB2 += ((real)A[d] - Bc[d]) * ((real)A[d] - Bc[d]);
                for (int ka = 0; ka < mol->shell_nprim[sa]; ++ka) {
                    real a = mol->prim_exp[mol->shell_prim_off[sa] + ka];
                    real da = mol->prim_coef[mol->shell_prim_off[sa] + ka];
                    for (int kb = 0; kb < mol->shell_nprim[sb]; ++kb) {
                        real b = mol->prim_exp[mol->shell_prim_off[sb] + kb];
                        real db = mol->prim_coef[mol->shell_prim_off[sb] + kb];
                        real p = a + b;
                        if (prim_cutoff > 0.0 &&
                            fabs(da * db) * exp(-a * b / p * AB2) * pow(PI / p, (real)1.5) < prim_cutoff)
                            continue;
                        /* O2-O5 for every Cartesian component pair of this primitive pair */
                        real rho = p * alpha / (p + alpha);
                        real Pc[3], X[3];
                        Etab E[3];
                        for (int d = 0; d < 3; ++d) {
                            Pc[d] = (a * A[d] + b * Bc[d]) / p;
                            X[d] = Pc[d] - C[d];
                            hermite_E(la + 1, lb + 1, a, b, (real)A[d] - Bc[d], E[d]);
                        }
                        Rtab R;
                        hermite_R(la + lb + 2 + lP, rho, X, R);
                        real pref = NP * da * db * 2.0 * pow(PI, (real)2.5) / (p * alpha * sqrt(p + alpha));
                        for (int ca = 0; ca < na; ++ca)
                            for (int cb = 0; cb < nb; ++cb) {
                                const int *ia = compa[ca], *ib = compb[cb];
                                real *o = buf + (ca * 10 + cb) * 10;
#define EE(d, i, j) E[d][i][j], (i) + (j)
                                o[0] += pref * hsum(EE(0, ia[0], ib[0]), EE(1, ia[1], ib[1]), EE(2, ia[2], ib[2]), R, sh0, sh1, sh2);
                                for (int d = 0; d < 3; ++d) {
                                    int ja[3] = {ia[0], ia[1], ia[2]}, jb[3] = {ib[0], ib[1], ib[2]};
                                    real up, dn = 0.0;
                                    ja[d] = ia[d] + 1;
                                    up = hsum(EE(0, ja[0], jb[0]), EE(1, ja[1], jb[1]), EE(2, ja[2], jb[2]), R, sh0, sh1, sh2);
                                    if (ia[d] > 0) {
                                        ja[d] = ia[d] - 1;
                                        dn = hsum(EE(0, ja[0], jb[0]), EE(1, ja[1], jb[1]), EE(2, ja[2], jb[2]), R, sh0, sh1, sh2);
                                    }
                                    o[1 + d] += pref * (2.0 * a * up - ia[d] * dn);
                                    ja[d] = ia[d];
                                    jb[d] = ib[d] + 1;
                                    up = hsum(EE(0, ja[0], jb[0]), EE(1, ja[1], jb[1]), EE(2, ja[2], jb[2]), R, sh0, sh1, sh2);
                                    dn = 0.0;
                                    if (ib[d] > 0) {
                                        jb[d] = ib[d] - 1;
                                        dn = hsum(EE(0, ja[0], jb[0]), EE(1, ja[1], jb[1]), EE(2, ja[2], jb[2]), R, sh0, sh1, sh2);
                                    }
                                    o[4 + d] += pref * (2.0 * b * up - ib[d] * dn);
                                    o[7 + d] += -pref * hsum(EE(0, ia[0], ib[0]), EE(1, ia[1], ib[1]), EE(2, ia[2], ib[2]), R,
                                                             sh0 + (d == 0), sh1 + (d == 1), sh2 + (d == 2));
                                }
#undef EE
                            }
                    }
                }
                /* O6: multiply by G and scale, add to the three atoms */
                for (int s = 0; s < nmat; ++s) {
                    const double *Gs = G + (size_t)s * nao * nao;
                    long double *g = gl + (size_t)s * natoms * 3;
                    for (int ca = 0; ca < na; ++ca)
                        for (int cb = 0; cb < nb; ++cb) {
                            long double w = (long double)scale[s] * Gs[(size_t)(ao_off[sa] + ca) * nao + ao_off[sb] + cb];
                            const real *o = buf + (ca * 10 + cb) * 10;
                            el[s] += w * o[0];
                            for (int d = 0; d < 3; ++d) {
                                g[at_a * 3 + d] += w * o[1 + d];
                                g[at_b * 3 + d] += w * o[4 + d];
                                g[atP * 3 + d] += w * o[7 + d];
                            }
                        }
                }
            }
        }
#pragma omp critical
        {
            for (size_t i = 0; i < ng; ++i) gacc[i] += gl[i];
            for (int s = 0; s < nmat; ++s) eacc[s] += el[s];
        }
        free(gl); free(el); free(buf);
    }
    free(ao_off);
    return 0;
}

/* ---------------------------------------------------------------- undifferentiated integral matrix
 * out[mu][nu] = (mu nu|P) for aux P, all ordered (mu, nu)  (first factor of Eq. 21; O2-O4 with
 * N_P and the contraction coefficients).  Used by the fitting step (NEXT-1): T^P = C_occ^T (mu nu|P) C_vir.
 */
int ris_oracle_int3c_P(const ris_oracle_mol *mol, int P, double prim_cutoff, double *out)
{
    int nsh = mol->nshells;
    int *ao_off = malloc(sizeof(int) * (size_t)(nsh + 1));
    ao_off[0] = 0;
    for (int s = 0; s < nsh; ++s) {
        if (mol->shell_l[s] < 0 || mol->shell_l[s] > LMAX) { free(ao_off); return -1; }
        ao_off[s + 1] = ao_off[s] + ncart(mol->shell_l[s]);
    }
    int nao = ao_off[nsh];
    real alpha = aux_exp_of(mol, P);
    const int lP = aux_l_of(mol, P), iP = aux_comp_of(mol, P);
    const int sh0 = (lP == 1 && iP == 0), sh1 = (lP == 1 && iP == 1), sh2 = (lP == 1 && iP == 2);
    real NP = lP == 1 ? aux_norm_l(alpha, 1) * (-1.0 / (2.0 * alpha)) : aux_norm(alpha);
    const double *C = mol->coords + 3 * aux_atom_of(mol, P);
#pragma omp parallel for schedule(dynamic, 1)
    for (int sa = 0; sa < nsh; ++sa) {
        int la = mol->shell_l[sa], na = ncart(la);
        int compa[10][3];
        cart_components(la, compa);
        const double *A = mol->coords + 3 * mol->shell_atom[sa];
        for (int sb = 0; sb < nsh; ++sb) {
            int lb = mol->shell_l[sb], nb = ncart(lb);
            int compb[10][3];
            cart_components(lb, compb);
            const double *Bc = mol->coords + 3 * mol->shell_atom[sb];
            real buf[100];
            memset(buf, 0, sizeof buf);
            real AB2 = 0.0;
            for (int d = 0; d < 3; ++d) AB2 += ((real)A[d] - Bc[d]) * ((real)A[d] - Bc[d]);
            for (int ka = 0; ka < mol->shell_nprim[sa]; ++ka) {
                real a = mol->prim_exp[mol->shell_prim_off[sa] + ka];
                real da = mol->prim_coef[mol->shell_prim_off[sa] + ka];
                for (int kb = 0; kb < mol->shell_nprim[sb]; ++kb) {
                    real b = mol->prim_exp[mol->shell_prim_off[sb] + kb];
                    real db = mol->prim_coef[mol->shell_prim_off[sb] + kb];
                    real p = a + b;
                    if (prim_cutoff > 0.0 && fabs(da * db) * exp(-a * b / p * AB2) * pow(PI / p, (real)1.5) < prim_cutoff)
                        continue;
                    real rho = p * alpha / (p + alpha);
                    real X[3];
                    Etab E[3];
                    for (int d = 0; d < 3; ++d) {
                        X[d] = (a * A[d] + b * Bc[d]) / p - C[d];
                        hermite_E(la, lb, a, b, (real)A[d] - Bc[d], E[d]);
                    }
                    Rtab R;
                    hermite_R(la + lb + lP, rho, X, R);
                    real pref = NP * da * db * 2.0 * pow(PI, (real)2.5) / (p * alpha * sqrt(p + alpha));
                    for (int ca = 0; ca < na; ++ca)
                        for (int cb = 0; cb < nb; ++cb) {
                            const int *ia = compa[ca], *ib = compb[cb];
                            buf[ca * 10 + cb] += pref * hsum(E[0][ia[0]][ib[0]], ia[0] + ib[0], E[1][ia[1]][ib[1]], ia[1] + ib[1],
                                                             E[2][ia[2]][ib[2]], ia[2] + ib[2], R, sh0, sh1, sh2);
                        }
                }
            }
            for (int ca = 0; ca < na; ++ca)
                for (int cb = 0; cb < nb; ++cb)
                    out[(size_t)(ao_off[sa] + ca) * nao + ao_off[sb] + cb] = (double)buf[ca * 10 + cb];
        }
    }
    free(ao_off);
    return 0;
}

/* ---------------------------------------------------------------- O7: G_PQ and E_PQ
 * gacc[s][A][x] += sum_{PQ} c^s_P d^s_Q d(P|Q)/dR_{A,x};  eacc[s] += sum_{PQ} c_P d_Q (P|Q),
 * with N_P N_Q included.  P and Q run over all ordered pairs; P = Q contributes no gradient.
 */
int ris_oracle_grad_PQ(const ris_oracle_mol *mol, int nbatch, const double *c, const double *dq,
                       long double *gacc, long double *eacc)
{
    int n = aux_count(mol), nat = mol->natoms;
    for (int s = 0; s < nbatch; ++s)
        for (int P = 0; P < n; ++P)
            for (int Q = 0; Q < n; ++Q) {
                double o[4];
                double aP = aux_exp_of(mol, P), aQ = aux_exp_of(mol, Q);
                int lP = aux_l_of(mol, P), lQ = aux_l_of(mol, Q), atP = aux_atom_of(mol, P), atQ = aux_atom_of(mol, Q);
                if (lP == 0 && lQ == 0) ris_oracle_prim2c(aP, aQ, mol->coords + 3 * atP, mol->coords + 3 * atQ, o);
                else ris_oracle_prim2c_lm(aP, aQ, lP, aux_comp_of(mol, P), lQ, aux_comp_of(mol, Q), mol->coords + 3 * atP,
                                          mol->coords + 3 * atQ, o);
                long double w = (long double)c[s * n + P] * dq[s * n + Q] * (double)aux_norm_l(aP, lP) * (double)aux_norm_l(aQ, lQ);
                eacc[s] += w * o[0];
                if (atP == atQ) continue;          /* both functions move together: the integral depends on R_P - R_Q only */
                for (int d = 0; d < 3; ++d) {
                    gacc[((size_t)s * nat + atP) * 3 + d] += w * o[1 + d];
                    gacc[((size_t)s * nat + atQ) * 3 + d] -= w * o[1 + d];
                }
            }
    return 0;
}

int ris_oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
