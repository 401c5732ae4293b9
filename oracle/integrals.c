/* ORACLE -- test infrastructure, NOT the product.  Plain, slow, CPU-only McMurchie-Davidson
 * integrals for contracted Cartesian s/p/d Gaussians, written from the textbook definitions the
 * paper cites (refs 88-91) and DESIGN.md section "Oracle".  Shares no code with
 * paper_2601_16949_b200/csrc.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call it.
 *
 * Conventions: AO order = shell order, p components x, y, z; d components (Cartesian, 6 per shell, SURVEY 8(f)
 * NEXT-4, "6-31G*") xx, xy, xz, yy, yz, zz.  `ncoef[k]` are the FINAL
 * coefficients multiplying the bare primitive  x^i y^j z^k exp(-a r^2)  (primitive norm,
 * contraction coefficient and the contracted-shell renormalisation already folded in by
 * oracle/integrals.py, which computes them from this file's own overlap routine).  Reading R11 for d shells:
 * EVERY Cartesian component is normalised, <phi|phi> = 1; ncoef normalises xx (and yy, zz, which share its norm),
 * and xy, xz, yz carry the extra factor sqrt(3) = sqrt(<xx|xx> / <xy|xy>) (cart_norm below).
 *
 * Every function follows the definitions step by step; there is no blocking or reordering.
 */
#define _GNU_SOURCE
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <stdint.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define LMAX 2       /* highest shell angular momentum: s, p, d */
#define LMAX_TOT 8   /* l_a+l_b+l_c+l_d */
#define NR (LMAX_TOT + 1)
/* Hermite table R^n_{tuv}, n, t, u, v <= L, stored compactly with stride L + 1 (the variable L of the enclosing function) */
#define RT(n, t, u, v) Rt[((((n) * (L + 1)) + (t)) * (L + 1) + (u)) * (L + 1) + (v)]
#define NCART(l) (((l) + 1) * ((l) + 2) / 2)
#define NCMAX 6      /* NCART(LMAX) */
#define NQMAX 1296   /* NCMAX^4 */

typedef struct {
    int nshells;
    const double *centers; /* [ncenters][3] */
    const int32_t *sh_center, *sh_l, *sh_nprim, *sh_off, *ao_off;
    const double *exps, *ncoef;
} basis_t;

/* ---- Boys function F_n(T) = int_0^1 t^(2n) exp(-T t^2) dt, n = 0..nmax -------------------- */
/* T <= 35: series F_m(T) = exp(-T) sum_k (2T)^k / ((2m+1)(2m+3)...(2m+2k+1)) at m = nmax,
 *          then downward F_(n-1) = (2T F_n + exp(-T)) / (2n-1).
 * T  > 35: F_0 = 1/2 sqrt(pi/T) erf(sqrt T), upward F_(n+1) = ((2n+1) F_n - exp(-T)) / (2T). */
void oracle_boys(int nmax, double T, double *F)
{
    if (T <= 35.0) {
        long double term = 1.0L / (2 * nmax + 1), sum = term;
        for (int k = 1; k < 2000; ++k) {
            term *= 2.0L * T / (2 * nmax + 2 * k + 1);
            sum += term;
            if (term < 1e-19L * sum) break;
        }
        long double emt = expl(-(long double)T);
        long double f = emt * sum;
        F[nmax] = (double)f;
        for (int n = nmax; n >= 1; --n) {
            f = (2.0L * T * f + emt) / (2 * n - 1);
            F[n - 1] = (double)f;
        }
    } else {
        long double emt = expl(-(long double)T);
        long double f = 0.5L * sqrtl(M_PIl / T) * erfl(sqrtl((long double)T));
        F[0] = (double)f;
        for (int n = 0; n < nmax; ++n) {
            f = ((2 * n + 1) * f - emt) / (2.0L * T);
            F[n + 1] = (double)f;
        }
    }
}

/* ---- 1-D Hermite expansion coefficients E_t^{ij}, i,j <= LMAX, t <= i+j ------------------- */
/* E_0^{00} = exp(-mu X_AB^2);
 * E_t^{i+1,j} = E_{t-1}^{ij}/(2p) + X_PA E_t^{ij} + (t+1) E_{t+1}^{ij}
 * E_t^{i,j+1} = E_{t-1}^{ij}/(2p) + X_PB E_t^{ij} + (t+1) E_{t+1}^{ij};  E_t = 0 for t<0, t>i+j;
 * filled for i <= li, j <= lj (the shells' angular momenta), zero beyond */
static void hermite_E(int li, int lj, double a, double b, double Ax, double Bx, double E[LMAX + 1][LMAX + 1][2 * LMAX + 1])
{
    double p = a + b, mu = a * b / p, XAB = Ax - Bx;
    double Px = (a * Ax + b * Bx) / p, XPA = Px - Ax, XPB = Px - Bx;
    memset(E, 0, sizeof(double) * (LMAX + 1) * (LMAX + 1) * (2 * LMAX + 1));
    E[0][0][0] = exp(-mu * XAB * XAB);
    /* i -> i+1 at j = 0 */
    for (int i = 0; i < li; ++i)
        for (int t = 0; t <= i + 1; ++t) {
            double em = (t - 1 >= 0) ? E[i][0][t - 1] : 0.0;
            double e0 = (t <= i) ? E[i][0][t] : 0.0;
            double ep = (t + 1 <= i) ? E[i][0][t + 1] : 0.0;
            E[i + 1][0][t] = em / (2 * p) + XPA * e0 + (t + 1) * ep;
        }
    /* j -> j+1 at every i */
    for (int i = 0; i <= li; ++i)
        for (int j = 0; j < lj; ++j)
            for (int t = 0; t <= i + j + 1; ++t) {
                double em = (t - 1 >= 0) ? E[i][j][t - 1] : 0.0;
                double e0 = (t <= i + j) ? E[i][j][t] : 0.0;
                double ep = (t + 1 <= i + j) ? E[i][j][t + 1] : 0.0;
                E[i][j + 1][t] = em / (2 * p) + XPB * e0 + (t + 1) * ep;
            }
}

/* Cartesian powers of component c of a shell with angular momentum l (s: 000; p: x, y, z; d: xx, xy, xz, yy, yz, zz). */
static void cart_pow(int l, int c, int pw[3])
{
    static const int dpow[6][3] = {{2, 0, 0}, {1, 1, 0}, {1, 0, 1}, {0, 2, 0}, {0, 1, 1}, {0, 0, 2}};
    pw[0] = pw[1] = pw[2] = 0;
    if (l == 1) pw[c] = 1;
    if (l == 2) { pw[0] = dpow[c][0]; pw[1] = dpow[c][1]; pw[2] = dpow[c][2]; }
}

/* Norm of component c relative to component 0 of its shell (R11 for d shells, see the header): for one radial part
 * int x^4 e^{-2ar^2} = 3 int x^2 y^2 e^{-2ar^2}, so xy, xz, yz need sqrt(3) to reach <phi|phi> = 1. */
static double cart_norm(int l, int c)
{
    return (l == 2 && (c == 1 || c == 2 || c == 4)) ? sqrt(3.0) : 1.0;
}

/* ---- one-electron: overlap and dipole (origin O) for one shell pair ----------------------- */
/* <g_a|g_b> = E_0^x E_0^y E_0^z (pi/p)^{3/2};
 * <g_a| x-O_x |g_b> = (E_1^x + (P_x - O_x) E_0^x) E_0^y E_0^z (pi/p)^{3/2}. */
static void shell_pair_1e(const basis_t *B, int sa, int sb, const double *O,
                          double *S, double *D /* [3][na*nb] or NULL */)
{
    int la = B->sh_l[sa], lb = B->sh_l[sb], na = NCART(la), nb = NCART(lb);
    const double *A = B->centers + 3 * B->sh_center[sa], *Bc = B->centers + 3 * B->sh_center[sb];
    for (int i = 0; i < na * nb; ++i) {
        S[i] = 0.0;
        if (D) D[i] = D[na * nb + i] = D[2 * na * nb + i] = 0.0;
    }
    for (int ka = 0; ka < B->sh_nprim[sa]; ++ka)
        for (int kb = 0; kb < B->sh_nprim[sb]; ++kb) {
            double a = B->exps[B->sh_off[sa] + ka], b = B->exps[B->sh_off[sb] + kb];
            double cc = B->ncoef[B->sh_off[sa] + ka] * B->ncoef[B->sh_off[sb] + kb];
            double p = a + b, pref = pow(M_PI / p, 1.5);
            double E[3][LMAX + 1][LMAX + 1][2 * LMAX + 1], P[3];
            for (int x = 0; x < 3; ++x) {
                hermite_E(la, lb, a, b, A[x], Bc[x], E[x]);
                P[x] = (a * A[x] + b * Bc[x]) / p;
            }
            for (int ca = 0; ca < na; ++ca)
                for (int cb = 0; cb < nb; ++cb) {
                    int pa[3], pb[3];
                    cart_pow(la, ca, pa);
                    cart_pow(lb, cb, pb);
                    double e0[3], e1[3];
                    for (int x = 0; x < 3; ++x) {
                        e0[x] = E[x][pa[x]][pb[x]][0];
                        e1[x] = E[x][pa[x]][pb[x]][1];
                    }
                    double cn = cart_norm(la, ca) * cart_norm(lb, cb);
                    S[ca * nb + cb] += cn * (cc * pref * e0[0] * e0[1] * e0[2]);
                    if (D)
                        for (int x = 0; x < 3; ++x) {
                            double m = e1[x] + (P[x] - O[x]) * e0[x];
                            int y = (x + 1) % 3, z = (x + 2) % 3;
                            D[x * na * nb + ca * nb + cb] += cn * (cc * pref * m * e0[y] * e0[z]);
                        }
                }
        }
}

static basis_t mk_basis(int nshells, const double *centers, const int32_t *sh_center,
                        const int32_t *sh_l, const int32_t *sh_nprim, const int32_t *sh_off,
                        const int32_t *ao_off, const double *exps, const double *ncoef)
{
    basis_t B = {nshells, centers, sh_center, sh_l, sh_nprim, sh_off, ao_off, exps, ncoef};
    return B;
}

#define BASIS_ARGS int nshells, const double *centers, const int32_t *sh_center, \
    const int32_t *sh_l, const int32_t *sh_nprim, const int32_t *sh_off,       \
    const int32_t *ao_off, const double *exps, const double *ncoef
#define BASIS_MK mk_basis(nshells, centers, sh_center, sh_l, sh_nprim, sh_off, ao_off, exps, ncoef)

/* S [nao][nao], D [3][nao][nao] (D may be NULL); origin O[3]. */
void oracle_one_electron(BASIS_ARGS, int nao, const double *O, double *S, double *D)
{
    basis_t B = BASIS_MK;
    for (int sa = 0; sa < nshells; ++sa)
        for (int sb = 0; sb < nshells; ++sb) {
            double s[NCMAX * NCMAX], d[3 * NCMAX * NCMAX];
            int na = NCART(sh_l[sa]), nb = NCART(sh_l[sb]);
            shell_pair_1e(&B, sa, sb, O, s, D ? d : NULL);
            for (int ca = 0; ca < na; ++ca)
                for (int cb = 0; cb < nb; ++cb) {
                    size_t idx = (size_t)(ao_off[sa] + ca) * nao + ao_off[sb] + cb;
                    S[idx] = s[ca * nb + cb];
                    if (D)
                        for (int x = 0; x < 3; ++x)
                            D[(size_t)x * nao * nao + idx] = d[x * na * nb + ca * nb + cb];
                }
        }
}

/* ---- Hermite Coulomb integrals R^n_{tuv}(alpha, R_PQ) -------------------------------------- */
/* R^n_{000} = (-2 alpha)^n F_n(alpha |R|^2);
 * R^n_{t+1,u,v} = t R^{n+1}_{t-1,u,v} + X R^{n+1}_{t,u,v}  (same in u with Y, v with Z). */
/* Range-separated operator erf(omega r12)/r12 (NEXT-4: the long-range exchange of CAM-type functionals): with
 * theta^2 = omega^2 / (alpha + omega^2) the Hermite integrals are those of 1/r12 with alpha -> alpha theta^2 and an
 * overall factor theta:  R^n_{000} = theta (-2 alpha theta^2)^n F_n(alpha theta^2 |R|^2).  omega <= 0 means 1/r12. */
static void hermite_R(int L, double alpha, double omega, const double *R, double *Rt /* RT(n,t,u,v), (L+1)^4 entries */)
{
    double F[LMAX_TOT + 1];
    double theta = 1.0;
    if (omega > 0.0) {
        double th2 = omega * omega / (alpha + omega * omega);
        theta = sqrt(th2);
        alpha *= th2;
    }
    double T = alpha * (R[0] * R[0] + R[1] * R[1] + R[2] * R[2]);
    oracle_boys(L, T, F);
    for (int n = 0; n <= L; ++n)        /* only n, t, u, v <= L are ever touched */
        for (int t = 0; t <= L; ++t)
            for (int u = 0; u <= L; ++u)
                for (int v = 0; v <= L; ++v) RT(n, t, u, v) = 0.0;
    double m2a = theta;
    for (int n = 0; n <= L; ++n) {
        RT(n, 0, 0, 0) = m2a * F[n];
        m2a *= -2.0 * alpha;
    }
    for (int N = 1; N <= L; ++N) /* total order t+u+v = N needs n <= L-N */
        for (int t = 0; t <= N; ++t)
            for (int u = 0; u <= N - t; ++u) {
                int v = N - t - u;
                for (int n = 0; n <= L - N; ++n) {
                    double val;
                    if (t > 0)
                        val = (t - 1 > 0 ? (t - 1) * RT(n + 1, t - 2, u, v) : 0.0) +
                              R[0] * RT(n + 1, t - 1, u, v);
                    else if (u > 0)
                        val = (u - 1 > 0 ? (u - 1) * RT(n + 1, t, u - 2, v) : 0.0) +
                              R[1] * RT(n + 1, t, u - 1, v);
                    else
                        val = (v - 1 > 0 ? (v - 1) * RT(n + 1, t, u, v - 2) : 0.0) +
                              R[2] * RT(n + 1, t, u, v - 1);
                    RT(n, t, u, v) = val;
                }
            }
}

/* ---- contracted shell quartet (ab|cd): out[na][nb][nc][nd] --------------------------------- */
/* primitive: (ab|cd) = 2 pi^{5/2} / (p q sqrt(p+q)) sum_{tuv} E^{ab}_{tuv}
 *                       sum_{t'u'v'} (-1)^{t'+u'+v'} E^{cd}_{t'u'v'} R^0_{t+t',u+u',v+v'}          */
static void shell_quartet_op(const basis_t *B, int sa, int sb, int sc, int sd, double omega, double *out)
{
    int l[4] = {B->sh_l[sa], B->sh_l[sb], B->sh_l[sc], B->sh_l[sd]};
    int n[4] = {NCART(l[0]), NCART(l[1]), NCART(l[2]), NCART(l[3])};
    int L = l[0] + l[1] + l[2] + l[3];
    const double *A = B->centers + 3 * B->sh_center[sa], *Bc = B->centers + 3 * B->sh_center[sb];
    const double *C = B->centers + 3 * B->sh_center[sc], *D = B->centers + 3 * B->sh_center[sd];
    int ntot = n[0] * n[1] * n[2] * n[3];
    long double acc[NQMAX];
    for (int i = 0; i < ntot; ++i) acc[i] = 0.0L;
    for (int ka = 0; ka < B->sh_nprim[sa]; ++ka)
    for (int kb = 0; kb < B->sh_nprim[sb]; ++kb) {
        double a = B->exps[B->sh_off[sa] + ka], b = B->exps[B->sh_off[sb] + kb];
        double cab = B->ncoef[B->sh_off[sa] + ka] * B->ncoef[B->sh_off[sb] + kb];
        double p = a + b, P[3], Eab[3][LMAX + 1][LMAX + 1][2 * LMAX + 1];
        for (int x = 0; x < 3; ++x) {
            P[x] = (a * A[x] + b * Bc[x]) / p;
            hermite_E(l[0], l[1], a, b, A[x], Bc[x], Eab[x]);
        }
        for (int kc = 0; kc < B->sh_nprim[sc]; ++kc)
        for (int kd = 0; kd < B->sh_nprim[sd]; ++kd) {
            double c = B->exps[B->sh_off[sc] + kc], d = B->exps[B->sh_off[sd] + kd];
            double ccd = B->ncoef[B->sh_off[sc] + kc] * B->ncoef[B->sh_off[sd] + kd];
            double q = c + d, Q[3], Ecd[3][LMAX + 1][LMAX + 1][2 * LMAX + 1], RPQ[3];
            for (int x = 0; x < 3; ++x) {
                Q[x] = (c * C[x] + d * D[x]) / q;
                hermite_E(l[2], l[3], c, d, C[x], D[x], Ecd[x]);
                RPQ[x] = P[x] - Q[x];
            }
            double alpha = p * q / (p + q);
            double Rt[NR * NR * NR * NR];          /* only the first (L+1)^4 entries are used */
            hermite_R(L, alpha, omega, RPQ, Rt);
            double pref = 2.0 * pow(M_PI, 2.5) / (p * q * sqrt(p + q)) * cab * ccd;
            int idx = 0;
            for (int ca = 0; ca < n[0]; ++ca)
            for (int cb = 0; cb < n[1]; ++cb)
            for (int cc = 0; cc < n[2]; ++cc)
            for (int cd = 0; cd < n[3]; ++cd, ++idx) {
                int pa[3], pb[3], pc[3], pd[3];
                cart_pow(l[0], ca, pa); cart_pow(l[1], cb, pb);
                cart_pow(l[2], cc, pc); cart_pow(l[3], cd, pd);
                double s = 0.0;
                for (int t = 0; t <= pa[0] + pb[0]; ++t)
                for (int u = 0; u <= pa[1] + pb[1]; ++u)
                for (int v = 0; v <= pa[2] + pb[2]; ++v) {
                    double eab = Eab[0][pa[0]][pb[0]][t] * Eab[1][pa[1]][pb[1]][u] *
                                 Eab[2][pa[2]][pb[2]][v];
                    for (int t2 = 0; t2 <= pc[0] + pd[0]; ++t2)
                    for (int u2 = 0; u2 <= pc[1] + pd[1]; ++u2)
                    for (int v2 = 0; v2 <= pc[2] + pd[2]; ++v2) {
                        double ecd = Ecd[0][pc[0]][pd[0]][t2] * Ecd[1][pc[1]][pd[1]][u2] *
                                     Ecd[2][pc[2]][pd[2]][v2];
                        double sgn = ((t2 + u2 + v2) & 1) ? -1.0 : 1.0;
                        s += eab * sgn * ecd * RT(0, t + t2, u + u2, v + v2);
                    }
                }
                double cn = cart_norm(l[0], ca) * cart_norm(l[1], cb) * cart_norm(l[2], cc) * cart_norm(l[3], cd);
                acc[idx] += (long double)(cn * (pref * s));
            }
        }
    }
    for (int i = 0; i < ntot; ++i) out[i] = (double)acc[i];
}

static void shell_quartet(const basis_t *B, int sa, int sb, int sc, int sd, double *out)
{
    shell_quartet_op(B, sa, sb, sc, sd, 0.0, out);
}

void oracle_shell_quartet(BASIS_ARGS, int sa, int sb, int sc, int sd, double *out)
{
    basis_t B = BASIS_MK;
    shell_quartet(&B, sa, sb, sc, sd, out);
}

/* One primitive (un-contracted, coefficient 1) ERI class block, for the pins: centres and exponents
 * given directly.  out[na][nb][nc][nd]. */
void oracle_primitive_eri(const double *ctr /* [4][3] */, const double *ex /* [4] */,
                          const int32_t *l4, double *out)
{
    int32_t sh_center[4] = {0, 1, 2, 3}, sh_nprim[4] = {1, 1, 1, 1}, sh_off[4] = {0, 1, 2, 3};
    int32_t ao_off[4];
    double ncoef[4] = {1.0, 1.0, 1.0, 1.0};
    int o = 0;
    for (int i = 0; i < 4; ++i) { ao_off[i] = o; o += NCART(l4[i]); }
    basis_t B = mk_basis(4, ctr, sh_center, l4, sh_nprim, sh_off, ao_off, ex, ncoef);
    shell_quartet(&B, 0, 1, 2, 3, out);
}

/* Same for the operator erf(omega r12)/r12 (omega <= 0: 1/r12). */
void oracle_primitive_eri_erf(const double *ctr, const double *ex, const int32_t *l4, double omega, double *out)
{
    int32_t sh_center[4] = {0, 1, 2, 3}, sh_nprim[4] = {1, 1, 1, 1}, sh_off[4] = {0, 1, 2, 3};
    int32_t ao_off[4];
    double ncoef[4] = {1.0, 1.0, 1.0, 1.0};
    int o = 0;
    for (int i = 0; i < 4; ++i) { ao_off[i] = o; o += NCART(l4[i]); }
    basis_t B = mk_basis(4, ctr, sh_center, l4, sh_nprim, sh_off, ao_off, ex, ncoef);
    shell_quartet_op(&B, 0, 1, 2, 3, omega, out);
}

void oracle_eri_tensor_erf(BASIS_ARGS, int nao, double omega, double *eri);

/* Full AO tensor (mu nu|lam sig), [nao]^4, NO symmetry used (tiny systems only). */
void oracle_eri_tensor(BASIS_ARGS, int nao, double *eri)
{
    oracle_eri_tensor_erf(nshells, centers, sh_center, sh_l, sh_nprim, sh_off, ao_off, exps, ncoef, nao, 0.0, eri);
}

/* Full AO tensor of erf(omega r12)/r12 (omega <= 0: 1/r12). */
void oracle_eri_tensor_erf(BASIS_ARGS, int nao, double omega, double *eri)
{
    basis_t B = BASIS_MK;
    #pragma omp parallel for schedule(dynamic) collapse(2)
    for (int sa = 0; sa < nshells; ++sa)
    for (int sb = 0; sb < nshells; ++sb)
        for (int sc = 0; sc < nshells; ++sc)
        for (int sd = 0; sd < nshells; ++sd) {
            double blk[NQMAX];
            shell_quartet_op(&B, sa, sb, sc, sd, omega, blk);
            int n0 = NCART(sh_l[sa]), n1 = NCART(sh_l[sb]), n2 = NCART(sh_l[sc]),
                n3 = NCART(sh_l[sd]), idx = 0;
            for (int ca = 0; ca < n0; ++ca)
            for (int cb = 0; cb < n1; ++cb)
            for (int cc = 0; cc < n2; ++cc)
            for (int cd = 0; cd < n3; ++cd, ++idx) {
                size_t m = ao_off[sa] + ca, nu = ao_off[sb] + cb, la = ao_off[sc] + cc,
                       si = ao_off[sd] + cd;
                eri[((m * nao + nu) * nao + la) * nao + si] = blk[idx];
            }
        }
}

/* All integrals (mu nu|lam sig) with (lam, sig) running over the AOs of ONE shell pair (sc, sd):
 * out[nao][nao][nc][nd], no symmetry used in (mu, nu) except that the shell quartet (sa sb|sc sd) with sa >= sb is
 * evaluated once and written to both (mu nu) and (nu mu).  Shell quartets with Q_ab Q_cd < tau are left zero
 * (tau <= 0: none skipped).  Building block of the dense A of the 400-AO configuration (SURVEY 8(c5) route ii). */
void oracle_eri_pair_block(BASIS_ARGS, int nao, int sc, int sd, double tau, const double *Qs, double *out)
{
    basis_t B = BASIS_MK;
    int nc = NCART(sh_l[sc]), nd = NCART(sh_l[sd]);
    memset(out, 0, sizeof(double) * (size_t)nao * nao * nc * nd);
    double qcd = Qs[(size_t)sc * nshells + sd];
    #pragma omp parallel for schedule(dynamic, 2)
    for (int sa = 0; sa < nshells; ++sa)
        for (int sb = 0; sb <= sa; ++sb) {
            if (tau > 0.0 && Qs[(size_t)sa * nshells + sb] * qcd < tau) continue;
            double blk[NQMAX];
            shell_quartet(&B, sa, sb, sc, sd, blk);
            int na = NCART(sh_l[sa]), nb = NCART(sh_l[sb]), idx = 0;
            for (int ca = 0; ca < na; ++ca)
            for (int cb = 0; cb < nb; ++cb)
            for (int cc = 0; cc < nc; ++cc)
            for (int cd = 0; cd < nd; ++cd, ++idx) {
                size_t m = ao_off[sa] + ca, n = ao_off[sb] + cb;
                out[((m * nao + n) * nc + cc) * nd + cd] = blk[idx];
                out[((n * nao + m) * nc + cc) * nd + cd] = blk[idx];
            }
        }
}

/* ---- the same shell quartet with EVERY intermediate in x87 long double --------------------------------------
 * (Boys function, Hermite E and R recursions, contraction; same formulas, same order as shell_quartet_op with
 * omega = 0).  Used to measure the rounding noise of the FP64 integral values themselves: at cond(S) ~ 1e4-1e5 the
 * back transform C_o^T F C_v amplifies per-integral relative errors of 1e-15 to the 1e-10 level of the sigma
 * tolerance. */
static void boys_ld(int nmax, long double T, long double *F)
{
    if (T <= 35.0L) {
        long double term = 1.0L / (2 * nmax + 1), sum = term;
        for (int k = 1; k < 4000; ++k) {
            term *= 2.0L * T / (2 * nmax + 2 * k + 1);
            sum += term;
            if (term < 1e-21L * sum) break;
        }
        long double emt = expl(-T), f = emt * sum;
        F[nmax] = f;
        for (int n = nmax; n >= 1; --n) { f = (2.0L * T * f + emt) / (2 * n - 1); F[n - 1] = f; }
    } else {
        long double emt = expl(-T), f = 0.5L * sqrtl(M_PIl / T) * erfl(sqrtl(T));
        F[0] = f;
        for (int n = 0; n < nmax; ++n) { f = ((2 * n + 1) * f - emt) / (2.0L * T); F[n + 1] = f; }
    }
}

static void hermite_E_ld(int li, int lj, long double a, long double b, long double Ax, long double Bx,
                         long double E[LMAX + 1][LMAX + 1][2 * LMAX + 1])
{
    long double p = a + b, mu = a * b / p, XAB = Ax - Bx;
    long double Px = (a * Ax + b * Bx) / p, XPA = Px - Ax, XPB = Px - Bx;
    for (int i = 0; i < (LMAX + 1) * (LMAX + 1) * (2 * LMAX + 1); ++i) ((long double *)E)[i] = 0.0L;
    E[0][0][0] = expl(-mu * XAB * XAB);
    for (int i = 0; i < li; ++i)
        for (int t = 0; t <= i + 1; ++t) {
            long double em = (t - 1 >= 0) ? E[i][0][t - 1] : 0.0L;
            long double e0 = (t <= i) ? E[i][0][t] : 0.0L;
            long double ep = (t + 1 <= i) ? E[i][0][t + 1] : 0.0L;
            E[i + 1][0][t] = em / (2 * p) + XPA * e0 + (t + 1) * ep;
        }
    for (int i = 0; i <= li; ++i)
        for (int j = 0; j < lj; ++j)
            for (int t = 0; t <= i + j + 1; ++t) {
                long double em = (t - 1 >= 0) ? E[i][j][t - 1] : 0.0L;
                long double e0 = (t <= i + j) ? E[i][j][t] : 0.0L;
                long double ep = (t + 1 <= i + j) ? E[i][j][t + 1] : 0.0L;
                E[i][j + 1][t] = em / (2 * p) + XPB * e0 + (t + 1) * ep;
            }
}

static void shell_quartet_ld(const basis_t *B, int sa, int sb, int sc, int sd, long double *out)
{
    int l[4] = {B->sh_l[sa], B->sh_l[sb], B->sh_l[sc], B->sh_l[sd]};
    int n[4] = {NCART(l[0]), NCART(l[1]), NCART(l[2]), NCART(l[3])};
    int L = l[0] + l[1] + l[2] + l[3];
    const double *A = B->centers + 3 * B->sh_center[sa], *Bc = B->centers + 3 * B->sh_center[sb];
    const double *C = B->centers + 3 * B->sh_center[sc], *D = B->centers + 3 * B->sh_center[sd];
    int ntot = n[0] * n[1] * n[2] * n[3];
    for (int i = 0; i < ntot; ++i) out[i] = 0.0L;
    for (int ka = 0; ka < B->sh_nprim[sa]; ++ka)
    for (int kb = 0; kb < B->sh_nprim[sb]; ++kb) {
        long double a = B->exps[B->sh_off[sa] + ka], b = B->exps[B->sh_off[sb] + kb];
        long double cab = (long double)B->ncoef[B->sh_off[sa] + ka] * B->ncoef[B->sh_off[sb] + kb];
        long double p = a + b, P[3], Eab[3][LMAX + 1][LMAX + 1][2 * LMAX + 1];
        for (int x = 0; x < 3; ++x) { P[x] = (a * A[x] + b * Bc[x]) / p; hermite_E_ld(l[0], l[1], a, b, A[x], Bc[x], Eab[x]); }
        for (int kc = 0; kc < B->sh_nprim[sc]; ++kc)
        for (int kd = 0; kd < B->sh_nprim[sd]; ++kd) {
            long double c = B->exps[B->sh_off[sc] + kc], d = B->exps[B->sh_off[sd] + kd];
            long double ccd = (long double)B->ncoef[B->sh_off[sc] + kc] * B->ncoef[B->sh_off[sd] + kd];
            long double q = c + d, Q[3], Ecd[3][LMAX + 1][LMAX + 1][2 * LMAX + 1], R[3];
            for (int x = 0; x < 3; ++x) { Q[x] = (c * C[x] + d * D[x]) / q; hermite_E_ld(l[2], l[3], c, d, C[x], D[x], Ecd[x]); R[x] = P[x] - Q[x]; }
            long double alpha = p * q / (p + q), F[LMAX_TOT + 1];
            boys_ld(L, alpha * (R[0] * R[0] + R[1] * R[1] + R[2] * R[2]), F);
            static __thread long double Rt[NR * NR * NR * NR];
            for (int nn = 0; nn <= L; ++nn)
                for (int t = 0; t <= L; ++t)
                    for (int u = 0; u <= L; ++u)
                        for (int v = 0; v <= L; ++v) RT(nn, t, u, v) = 0.0L;
            long double m2a = 1.0L;
            for (int nn = 0; nn <= L; ++nn) { RT(nn, 0, 0, 0) = m2a * F[nn]; m2a *= -2.0L * alpha; }
            for (int N = 1; N <= L; ++N)
                for (int t = 0; t <= N; ++t)
                    for (int u = 0; u <= N - t; ++u) {
                        int v = N - t - u;
                        for (int nn = 0; nn <= L - N; ++nn) {
                            long double val;
                            if (t > 0) val = (t - 1 > 0 ? (t - 1) * RT(nn + 1, t - 2, u, v) : 0.0L) + R[0] * RT(nn + 1, t - 1, u, v);
                            else if (u > 0) val = (u - 1 > 0 ? (u - 1) * RT(nn + 1, t, u - 2, v) : 0.0L) + R[1] * RT(nn + 1, t, u - 1, v);
                            else val = (v - 1 > 0 ? (v - 1) * RT(nn + 1, t, u, v - 2) : 0.0L) + R[2] * RT(nn + 1, t, u, v - 1);
                            RT(nn, t, u, v) = val;
                        }
                    }
            long double pref = 2.0L * powl(M_PIl, 2.5L) / (p * q * sqrtl(p + q)) * cab * ccd;
            int idx = 0;
            for (int ca = 0; ca < n[0]; ++ca)
            for (int cb = 0; cb < n[1]; ++cb)
            for (int cc = 0; cc < n[2]; ++cc)
            for (int cd = 0; cd < n[3]; ++cd, ++idx) {
                int pa[3], pb[3], pc[3], pd[3];
                cart_pow(l[0], ca, pa); cart_pow(l[1], cb, pb); cart_pow(l[2], cc, pc); cart_pow(l[3], cd, pd);
                long double s = 0.0L;
                for (int t = 0; t <= pa[0] + pb[0]; ++t)
                for (int u = 0; u <= pa[1] + pb[1]; ++u)
                for (int v = 0; v <= pa[2] + pb[2]; ++v) {
                    long double eab = Eab[0][pa[0]][pb[0]][t] * Eab[1][pa[1]][pb[1]][u] * Eab[2][pa[2]][pb[2]][v];
                    for (int t2 = 0; t2 <= pc[0] + pd[0]; ++t2)
                    for (int u2 = 0; u2 <= pc[1] + pd[1]; ++u2)
                    for (int v2 = 0; v2 <= pc[2] + pd[2]; ++v2) {
                        long double ecd = Ecd[0][pc[0]][pd[0]][t2] * Ecd[1][pc[1]][pd[1]][u2] * Ecd[2][pc[2]][pd[2]][v2];
                        long double sgn = ((t2 + u2 + v2) & 1) ? -1.0L : 1.0L;
                        s += eab * sgn * ecd * RT(0, t + t2, u + u2, v + v2);
                    }
                }
                long double cn = 1.0L;     /* sqrt(3) per mixed d component, in long double */
                { int pw[4][3]; cart_pow(l[0], ca, pw[0]); cart_pow(l[1], cb, pw[1]); cart_pow(l[2], cc, pw[2]); cart_pow(l[3], cd, pw[3]);
                  for (int k = 0; k < 4; ++k) if (l[k] == 2 && pw[k][0] < 2 && pw[k][1] < 2 && pw[k][2] < 2) cn *= sqrtl(3.0L); }
                out[idx] += cn * (pref * s);
            }
        }
    }
}

/* Full AO tensor in long double, [nao]^4 (small systems only: 16 bytes per element). */
void oracle_eri_tensor_ld(BASIS_ARGS, int nao, long double *eri)
{
    basis_t B = BASIS_MK;
    #pragma omp parallel for schedule(dynamic) collapse(2)
    for (int sa = 0; sa < nshells; ++sa)
    for (int sb = 0; sb < nshells; ++sb)
        for (int sc = 0; sc < nshells; ++sc)
        for (int sd = 0; sd < nshells; ++sd) {
            long double blk[NQMAX];
            shell_quartet_ld(&B, sa, sb, sc, sd, blk);
            int n0 = NCART(sh_l[sa]), n1 = NCART(sh_l[sb]), n2 = NCART(sh_l[sc]), n3 = NCART(sh_l[sd]), idx = 0;
            for (int ca = 0; ca < n0; ++ca)
            for (int cb = 0; cb < n1; ++cb)
            for (int cc = 0; cc < n2; ++cc)
            for (int cd = 0; cd < n3; ++cd, ++idx) {
                size_t m = ao_off[sa] + ca, nu = ao_off[sb] + cb, la = ao_off[sc] + cc, si = ao_off[sd] + cd;
                eri[((m * nao + nu) * nao + la) * nao + si] = blk[idx];
            }
        }
}

/* Schwarz bounds Q_ab = sqrt(max_{mu in a, nu in b} (mu nu|mu nu)), [nshells][nshells] (R14). */
void oracle_schwarz(BASIS_ARGS, double *Q)
{
    basis_t B = BASIS_MK;
    #pragma omp parallel for schedule(dynamic)
    for (int sa = 0; sa < nshells; ++sa)
        for (int sb = 0; sb <= sa; ++sb) {
            double blk[NQMAX];
            shell_quartet(&B, sa, sb, sa, sb, blk);
            int na = NCART(sh_l[sa]), nb = NCART(sh_l[sb]);
            double m = 0.0;
            for (int ca = 0; ca < na; ++ca)
                for (int cb = 0; cb < nb; ++cb) {
                    double v = blk[((ca * nb + cb) * na + ca) * nb + cb];
                    if (v > m) m = v;
                }
            Q[(size_t)sa * nshells + sb] = Q[(size_t)sb * nshells + sa] = sqrt(m);
        }
}

/* ---- matrix-free J[T], K[T] over Schwarz-screened unique shell quartets -------------------- */
/* Definitions: J_{mu nu} = sum_{lam sig} (mu nu|lam sig) T_{lam sig},
 *                          K_{mu lam} = sum_{nu sig} (mu nu|lam sig) T_{nu sig},  T NOT symmetric.
 * Unique quartets: a>=b, c>=d, pair(ab) >= pair(cd); each integral is applied through all 8
 * index images with weight 1/2 per coincidence (a==b, c==d, ab==cd), the standard degeneracy
 * rule; tests pin this against the plain N^4 contraction of oracle_eri_tensor.
 * T, J, K: [nvec][nao][nao].  Returns the number of unique shell quartets with Q_ab Q_cd >= tau
 * (R14) through *nquartets, primitive quartets through *nprimq.  tau <= 0 disables screening. */
/* oracle_jk_strided visits only the bra pairs ab with ab % ab_stride == ab_phase (all their kets): a
 * BOUNDED SAMPLE of the same loop, used only to time the oracle on workloads whose full pass takes
 * tens of minutes (bench.py cpu_baseline); its J/K are then partial sums.  oracle_jk = stride 1. */
void oracle_jk_strided_op(BASIS_ARGS, int nao, int nvec, const double *T, double tau, const double *Qs,
                          int ab_stride, int ab_phase, double omega,
                          double *J, double *K, int64_t *nquartets, int64_t *nprimq);

void oracle_jk_strided(BASIS_ARGS, int nao, int nvec, const double *T, double tau, const double *Qs,
                       int ab_stride, int ab_phase,
                       double *J, double *K, int64_t *nquartets, int64_t *nprimq)
{
    oracle_jk_strided_op(nshells, centers, sh_center, sh_l, sh_nprim, sh_off, ao_off, exps, ncoef, nao, nvec, T, tau, Qs,
                         ab_stride, ab_phase, 0.0, J, K, nquartets, nprimq);
}

/* The same loop for the operator erf(omega r12)/r12 (omega <= 0: 1/r12).  The screening bounds Qs stay those of
 * 1/r12, which dominate the attenuated integrals (erf <= 1). */
void oracle_jk_strided_op(BASIS_ARGS, int nao, int nvec, const double *T, double tau, const double *Qs,
                          int ab_stride, int ab_phase, double omega,
                          double *J, double *K, int64_t *nquartets, int64_t *nprimq)
{
    basis_t B = BASIS_MK;
    size_t nn = (size_t)nao * nao;
    memset(J, 0, sizeof(double) * nn * nvec);
    memset(K, 0, sizeof(double) * nn * nvec);
    int64_t nq_tot = 0, npq_tot = 0;
    int npair = nshells * (nshells + 1) / 2;
    #pragma omp parallel
    {
        double *Jl = calloc(nn * nvec, sizeof(double)), *Kl = calloc(nn * nvec, sizeof(double));
        int64_t nq = 0, npq = 0;
        #pragma omp for schedule(dynamic, 4)
        for (int ab = npair - 1; ab >= 0; --ab) {
            if (ab_stride > 1 && ab % ab_stride != ab_phase) continue;
            int sa = (int)((sqrt(8.0 * ab + 1.0) - 1.0) / 2.0);
            while ((sa + 1) * (sa + 2) / 2 <= ab) ++sa;
            while (sa * (sa + 1) / 2 > ab) --sa;
            int sb = ab - sa * (sa + 1) / 2;
            double qab = Qs[(size_t)sa * nshells + sb];
            for (int cd = 0; cd <= ab; ++cd) {
                int sc = (int)((sqrt(8.0 * cd + 1.0) - 1.0) / 2.0);
                while ((sc + 1) * (sc + 2) / 2 <= cd) ++sc;
                while (sc * (sc + 1) / 2 > cd) --sc;
                int sd = cd - sc * (sc + 1) / 2;
                if (tau > 0.0 && qab * Qs[(size_t)sc * nshells + sd] < tau) continue;
                ++nq;
                npq += (int64_t)sh_nprim[sa] * sh_nprim[sb] * sh_nprim[sc] * sh_nprim[sd];
                double blk[NQMAX];
                shell_quartet_op(&B, sa, sb, sc, sd, omega, blk);
                double w = 1.0;
                if (sa == sb) w *= 0.5;
                if (sc == sd) w *= 0.5;
                if (ab == cd) w *= 0.5;
                int n0 = NCART(sh_l[sa]), n1 = NCART(sh_l[sb]), n2 = NCART(sh_l[sc]),
                    n3 = NCART(sh_l[sd]), idx = 0;
                for (int ca = 0; ca < n0; ++ca)
                for (int cb = 0; cb < n1; ++cb)
                for (int cc = 0; cc < n2; ++cc)
                for (int cdd = 0; cdd < n3; ++cdd, ++idx) {
                    double I = w * blk[idx];
                    size_t m = ao_off[sa] + ca, n = ao_off[sb] + cb, l = ao_off[sc] + cc,
                           s = ao_off[sd] + cdd;
                    /* the 8 images (m n|l s) (n m|l s) (m n|s l) (n m|s l) and bra<->ket */
                    size_t im[8][4] = {{m, n, l, s}, {n, m, l, s}, {m, n, s, l}, {n, m, s, l},
                                       {l, s, m, n}, {s, l, m, n}, {l, s, n, m}, {s, l, n, m}};
                    for (int v = 0; v < nvec; ++v) {
                        const double *Tv = T + v * nn;
                        double *Jv = Jl + v * nn, *Kv = Kl + v * nn;
                        for (int g = 0; g < 8; ++g) {
                            size_t i0 = im[g][0], i1 = im[g][1], i2 = im[g][2], i3 = im[g][3];
                            Jv[i0 * nao + i1] += I * Tv[i2 * nao + i3];
                            Kv[i0 * nao + i2] += I * Tv[i1 * nao + i3];
                        }
                    }
                }
            }
        }
        #pragma omp critical
        {
            for (size_t i = 0; i < nn * nvec; ++i) { J[i] += Jl[i]; K[i] += Kl[i]; }
            nq_tot += nq;
            npq_tot += npq;
        }
        free(Jl);
        free(Kl);
    }
    if (nquartets) *nquartets = nq_tot;
    if (nprimq) *nprimq = npq_tot;
}

void oracle_jk(BASIS_ARGS, int nao, int nvec, const double *T, double tau, const double *Qs,
               double *J, double *K, int64_t *nquartets, int64_t *nprimq)
{
    oracle_jk_strided(nshells, centers, sh_center, sh_l, sh_nprim, sh_off, ao_off, exps, ncoef, nao, nvec, T,
                      tau, Qs, 1, 0, J, K, nquartets, nprimq);
}

/* Extended-precision route of oracle_jk ("accumulate J/K sums ... in long double"): the same loop
 * over unique screened quartets and the same 8-image rule, but the densities arrive as long double, every product
 * I * T and every partial sum (per thread and across threads) is x87 80-bit long double, and J, K are returned as
 * long double.  Only the integral values themselves are FP64 (shell_quartet).  Layout: T, J, K are [nao][nao][nvec]
 * (vector index fastest) so that one integral meets the nvec densities at consecutive addresses.  Used for the
 * stored samples at 1280 AOs and by the test that bounds the noise floor of the FP64 route above. */
void oracle_jk_ld(BASIS_ARGS, int nao, int nvec, const long double *T, double tau, const double *Qs,
                  long double *J, long double *K, int64_t *nquartets, int64_t *nprimq)
{
    basis_t B = BASIS_MK;
    size_t nn = (size_t)nao * nao;
    for (size_t i = 0; i < nn * nvec; ++i) J[i] = K[i] = 0.0L;
    int64_t nq_tot = 0, npq_tot = 0;
    int npair = nshells * (nshells + 1) / 2;
    #pragma omp parallel
    {
        long double *Jl = calloc(nn * nvec, sizeof(long double)), *Kl = calloc(nn * nvec, sizeof(long double));
        int64_t nq = 0, npq = 0;
        #pragma omp for schedule(dynamic, 4)
        for (int ab = npair - 1; ab >= 0; --ab) {
            int sa = (int)((sqrt(8.0 * ab + 1.0) - 1.0) / 2.0);
            while ((sa + 1) * (sa + 2) / 2 <= ab) ++sa;
            while (sa * (sa + 1) / 2 > ab) --sa;
            int sb = ab - sa * (sa + 1) / 2;
            double qab = Qs[(size_t)sa * nshells + sb];
            for (int cd = 0; cd <= ab; ++cd) {
                int sc = (int)((sqrt(8.0 * cd + 1.0) - 1.0) / 2.0);
                while ((sc + 1) * (sc + 2) / 2 <= cd) ++sc;
                while (sc * (sc + 1) / 2 > cd) --sc;
                int sd = cd - sc * (sc + 1) / 2;
                if (tau > 0.0 && qab * Qs[(size_t)sc * nshells + sd] < tau) continue;
                ++nq;
                npq += (int64_t)sh_nprim[sa] * sh_nprim[sb] * sh_nprim[sc] * sh_nprim[sd];
                double blk[NQMAX];
                shell_quartet(&B, sa, sb, sc, sd, blk);
                long double w = 1.0L;
                if (sa == sb) w *= 0.5L;
                if (sc == sd) w *= 0.5L;
                if (ab == cd) w *= 0.5L;
                int n0 = NCART(sh_l[sa]), n1 = NCART(sh_l[sb]), n2 = NCART(sh_l[sc]),
                    n3 = NCART(sh_l[sd]), idx = 0;
                for (int ca = 0; ca < n0; ++ca)
                for (int cb = 0; cb < n1; ++cb)
                for (int cc = 0; cc < n2; ++cc)
                for (int cdd = 0; cdd < n3; ++cdd, ++idx) {
                    long double I = w * (long double)blk[idx];
                    size_t m = ao_off[sa] + ca, n = ao_off[sb] + cb, l = ao_off[sc] + cc,
                           s = ao_off[sd] + cdd;
                    size_t im[8][4] = {{m, n, l, s}, {n, m, l, s}, {m, n, s, l}, {n, m, s, l},
                                       {l, s, m, n}, {s, l, m, n}, {l, s, n, m}, {s, l, n, m}};
                    for (int g = 0; g < 8; ++g) {
                        size_t i0 = im[g][0], i1 = im[g][1], i2 = im[g][2], i3 = im[g][3];
                        long double *Jr = Jl + (i0 * nao + i1) * nvec, *Kr = Kl + (i0 * nao + i2) * nvec;
                        const long double *Tj = T + (i2 * nao + i3) * nvec, *Tk = T + (i1 * nao + i3) * nvec;
                        for (int v = 0; v < nvec; ++v) {
                            Jr[v] += I * Tj[v];
                            Kr[v] += I * Tk[v];
                        }
                    }
                }
            }
        }
        #pragma omp critical
        {
            for (size_t i = 0; i < nn * nvec; ++i) { J[i] += Jl[i]; K[i] += Kl[i]; }
            nq_tot += nq;
            npq_tot += npq;
        }
        free(Jl);
        free(Kl);
    }
    if (nquartets) *nquartets = nq_tot;
    if (nprimq) *nprimq = npq_tot;
}

/* Sampled elements of J[T] and K[T] straight from the definitions (no symmetry, no screening):
 * for each sample s with AO pair (mu, nu): J = sum_{lam sig} (mu nu|lam sig) T[lam][sig],
 * K = sum_{lam sig} (mu lam|nu sig) T[lam][sig].  Jout, Kout: [nsamp][nvec]. */
void oracle_jk_samples(BASIS_ARGS, int nao, int nvec, const double *T, int nsamp,
                       const int32_t *smu, const int32_t *snu, double *Jout, double *Kout)
{
    basis_t B = BASIS_MK;
    size_t nn = (size_t)nao * nao;
    int32_t *ao2sh = malloc(sizeof(int32_t) * nao);
    for (int s = 0; s < nshells; ++s)
        for (int c = 0; c < NCART(sh_l[s]); ++c) ao2sh[ao_off[s] + c] = s;
    #pragma omp parallel for schedule(dynamic)
    for (int smp = 0; smp < nsamp; ++smp) {
        int mu = smu[smp], nu = snu[smp], sa = ao2sh[mu], sb = ao2sh[nu];
        int ca = mu - ao_off[sa], cb = nu - ao_off[sb];
        int na = NCART(sh_l[sa]), nb = NCART(sh_l[sb]);
        (void)na;
        long double Jacc[64], Kacc[64];
        for (int v = 0; v < nvec; ++v) Jacc[v] = Kacc[v] = 0.0L;
        for (int sc = 0; sc < nshells; ++sc)
            for (int sd = 0; sd < nshells; ++sd) {
                int nc = NCART(sh_l[sc]), nd = NCART(sh_l[sd]);
                double bj[NQMAX], bk[NQMAX];
                shell_quartet(&B, sa, sb, sc, sd, bj); /* (mu nu|lam sig) */
                shell_quartet(&B, sa, sc, sb, sd, bk); /* (mu lam|nu sig) */
                for (int cc = 0; cc < nc; ++cc)
                    for (int cd = 0; cd < nd; ++cd) {
                        size_t lam = ao_off[sc] + cc, sig = ao_off[sd] + cd;
                        double ij = bj[((ca * nb + cb) * nc + cc) * nd + cd];
                        double ik = bk[((ca * nc + cc) * nb + cb) * nd + cd];
                        for (int v = 0; v < nvec; ++v) {
                            double t = T[v * nn + lam * nao + sig];
                            Jacc[v] += (long double)(ij * t);
                            Kacc[v] += (long double)(ik * t);
                        }
                    }
            }
        for (int v = 0; v < nvec; ++v) {
            Jout[(size_t)smp * nvec + v] = (double)Jacc[v];
            Kout[(size_t)smp * nvec + v] = (double)Kacc[v];
        }
    }
    free(ao2sh);
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
