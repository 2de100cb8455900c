// sldg_tables.cpp -- host-side constants of the SLDG scheme (product code; independent of oracle/).
//
//  * Gauss-Legendre rules on [0,1] from their closed forms (n <= 5)
//  * A_jl(alpha), B_jl(alpha) of eq. (3) as explicit polynomials in alpha.  The paper defers the
//    matrices to Einkemmer (2019); they follow from "translate, then L2-project cell-wise"
//    (Fig. 1) with the diagonal GL-Lagrange mass matrix (reading A):
//        A_jl = 1/w_j int_alpha^1 l_j(x) l_l(x - alpha) dx,   B_jl = 1/w_j int_0^alpha l_j(x) l_l(x - alpha + 1) dx.
//    Here the integrals are done in closed form on the monomial expansion of the Lagrange basis (long double),
//    which gives every entry as a polynomial of degree <= 2k+1 in alpha (stored re-expanded around alpha = 1/2);
//    the host evaluates it by Horner in long double, the device in fp64.
//  * fused transfer + DFT matrices of the Poisson solve (reading P1).
#include <math.h>
#include <string.h>

#include "sldg_internal.h"

typedef long double ld;
typedef __float128 qd;   // coefficient construction only: the monomial route cancels ~1e5, harmless at 1e-34

void sldg_gl_rule(int n, double* xi, double* w)
{
    ld t[SLDG_MAXK1], wt[SLDG_MAXK1];
    switch (n) {
    case 1: t[0] = 0; wt[0] = 2; break;
    case 2: t[0] = -1 / sqrtl(3.0L); t[1] = -t[0]; wt[0] = wt[1] = 1; break;
    case 3:
        t[0] = -sqrtl(3.0L / 5.0L); t[1] = 0; t[2] = -t[0];
        wt[0] = wt[2] = 5.0L / 9.0L; wt[1] = 8.0L / 9.0L; break;
    case 4: {
        ld a = sqrtl(3.0L / 7.0L - 2.0L / 7.0L * sqrtl(6.0L / 5.0L));
        ld b = sqrtl(3.0L / 7.0L + 2.0L / 7.0L * sqrtl(6.0L / 5.0L));
        ld wa = (18.0L + sqrtl(30.0L)) / 36.0L, wb = (18.0L - sqrtl(30.0L)) / 36.0L;
        t[0] = -b; t[1] = -a; t[2] = a; t[3] = b;
        wt[0] = wb; wt[1] = wa; wt[2] = wa; wt[3] = wb; break;
    }
    default: {
        ld a = sqrtl(5.0L - 2.0L * sqrtl(10.0L / 7.0L)) / 3.0L;
        ld b = sqrtl(5.0L + 2.0L * sqrtl(10.0L / 7.0L)) / 3.0L;
        ld wa = (322.0L + 13.0L * sqrtl(70.0L)) / 900.0L, wb = (322.0L - 13.0L * sqrtl(70.0L)) / 900.0L;
        t[0] = -b; t[1] = -a; t[2] = 0; t[3] = a; t[4] = b;
        wt[0] = wb; wt[1] = wa; wt[2] = 128.0L / 225.0L; wt[3] = wa; wt[4] = wb; break;
    }
    }
    for (int i = 0; i < n; i++) {
        xi[i] = (double)((t[i] + 1.0L) / 2.0L);
        w[i] = (double)(wt[i] / 2.0L);
    }
}

// monomial coefficients (ascending) of the Lagrange basis on the nodes xi
static void lagrange_monomials(int n, const double* xi, qd c[SLDG_MAXK1][SLDG_MAXK1])
{
    for (int l = 0; l < n; l++) {
        qd p[SLDG_MAXK1 + 1];
        for (int q = 0; q <= SLDG_MAXK1; q++) p[q] = 0;
        p[0] = 1;
        int deg = 0;
        for (int m = 0; m < n; m++) {
            if (m == l) continue;
            qd den = (qd)xi[l] - (qd)xi[m], r = (qd)xi[m];
            // p <- p * (z - r) / den
            for (int q = deg + 1; q >= 0; q--) {
                qd lower = (q > 0) ? p[q - 1] : (qd)0;
                qd same = (q <= deg) ? p[q] : (qd)0;
                p[q] = (lower - r * same) / den;
            }
            deg++;
        }
        for (int q = 0; q < n; q++) c[l][q] = p[q];
    }
}

static qd binom(int n, int r)
{
    qd b = 1;
    for (int i = 1; i <= r; i++) b = b * (qd)(n - r + i) / (qd)i;
    return b;
}

void sldg_build_poly(int k, const double* xi, const double* w, ABPoly* out, ABPolyLD* outld)
{
    int n = k + 1;
    qd c[SLDG_MAXK1][SLDG_MAXK1];
    lagrange_monomials(n, xi, c);
    memset(out, 0, sizeof(*out));
    memset(outld, 0, sizeof(*outld));
    for (int j = 0; j < n; j++)
        for (int l = 0; l < n; l++) {
            qd pa[SLDG_MAXPOLY], pb[SLDG_MAXPOLY];
            for (int i = 0; i < SLDG_MAXPOLY; i++) { pa[i] = 0; pb[i] = 0; }
            for (int m = 0; m < n; m++)
                for (int q = 0; q < n; q++) {
                    qd cc = c[j][m] * c[l][q];
                    // A: int_alpha^1 x^m (x-alpha)^q dx = sum_r C(m,r) alpha^(m-r) (1-alpha)^(r+q+1) / (r+q+1)
                    for (int r = 0; r <= m; r++) {
                        int p = r + q + 1;
                        qd f = cc * binom(m, r) / (qd)p;
                        for (int t = 0; t <= p; t++)
                            pa[m - r + t] += f * binom(p, t) * ((t & 1) ? (qd)-1 : (qd)1);
                    }
                    // B: int_0^alpha x^m (x+1-alpha)^q dx = sum_r C(q,r) (1-alpha)^(q-r) alpha^(m+r+1) / (m+r+1)
                    for (int r = 0; r <= q; r++) {
                        int p = q - r;
                        qd f = cc * binom(q, r) / (qd)(m + r + 1);
                        for (int t = 0; t <= p; t++)
                            pb[m + r + 1 + t] += f * binom(p, t) * ((t & 1) ? (qd)-1 : (qd)1);
                    }
                }
            // re-expand around alpha = 1/2 (t = alpha - 1/2, |t| <= 1/2): sum |c_i| |t|^i drops from ~380 to ~20
            // for k = 4, which keeps the fp64 Horner evaluation on the device within a few 1e-15.
            const int deg = 2 * k + 1;
            for (int m = 0; m <= deg; m++) {
                qd sa = 0, sb = 0, half = 1;
                for (int i = m; i <= deg; i++) {
                    sa += pa[i] * binom(i, m) * half;
                    sb += pb[i] * binom(i, m) * half;
                    half *= (qd)0.5;
                }
                qd ca = sa / (qd)w[j], cb = sb / (qd)w[j];
                outld->c[0][j * n + l][m] = (ld)ca; outld->c[1][j * n + l][m] = (ld)cb;
                out->c[0][j * n + l][m] = (double)ca; out->c[1][j * n + l][m] = (double)cb;
            }
        }
}

void sldg_eval_AB_host(const ABPolyLD* p, int k, double alpha, double* A, double* B)
{
    int n = k + 1, deg = 2 * k + 1;
    const ld x = (ld)alpha - 0.5L;
    for (int e = 0; e < n * n; e++) {
        ld a = p->c[0][e][deg], b = p->c[1][e][deg];
        for (int t = deg - 1; t >= 0; t--) {
            a = a * x + p->c[0][e][t];
            b = b * x + p->c[1][e][t];
        }
        A[e] = (double)a; B[e] = (double)b;
    }
}

static ld lagrange_at(int n, const double* xi, int l, ld z)
{
    ld r = 1;
    for (int m = 0; m < n; m++)
        if (m != l) r *= (z - (ld)xi[m]) / ((ld)xi[l] - (ld)xi[m]);
    return r;
}

void sldg_build_dft(int k, const double* xi, int ncell, double* fwdT, double* invT)
{
    const ld twopi = 6.28318530717958647692528676655900577L;
    int n = k + 1;
    long D = (long)ncell * n;
    // P[mm][l] = l_l(eta_mm), eta_mm = (mm + 1/2)/(k+1)  (equidistant points of one cell)
    // and its inverse in closed form: the map back from the equidistant points to the GL nodes evaluates the
    // interpolation polynomial through the equidistant values, Pinv[l][mm] = (Lagrange basis of eta_mm)(xi_l)
    ld P[SLDG_MAXK1][SLDG_MAXK1], Pinv[SLDG_MAXK1][SLDG_MAXK1];
    for (int mm = 0; mm < n; mm++)
        for (int l = 0; l < n; l++) {
            P[mm][l] = lagrange_at(n, xi, l, ((ld)mm + 0.5L) / (ld)n);
            ld r = 1;                                         // exact rational nodes: (mm + 1/2)/n
            for (int m2 = 0; m2 < n; m2++)
                if (m2 != mm) r *= ((ld)xi[l] - ((ld)m2 + 0.5L) / (ld)n) / ((ld)(mm - m2) / (ld)n);
            Pinv[l][mm] = r;
        }
    std::vector<ld> cs(D), sn(D);
    for (long r = 0; r < D; r++) {
        cs[r] = cosl(twopi * (ld)r / (ld)D);
        sn[r] = sinl(twopi * (ld)r / (ld)D);
    }
    double* fre = fwdT; double* fim = fwdT + D * D;
    double* ire = invT; double* iim = invT + D * D;
    for (long m = 0; m < D; m++)             // frequency index
        for (long i = 0; i < ncell; i++)
            for (int l = 0; l < n; l++) {    // node index within the cell
                ld gr = 0, gi = 0, hr = 0, hi = 0;
                for (int mm = 0; mm < n; mm++) {
                    long r = (m * (i * n + mm)) % D;
                    gr += cs[r] * P[mm][l];  gi += -sn[r] * P[mm][l];          // e^{-2 pi i m e / D}
                    hr += cs[r] * Pinv[l][mm]; hi += sn[r] * Pinv[l][mm];  // e^{+2 pi i m e / D}
                }
                long node = i * n + l;
                // forward G[m][node] stored transposed at [node][m]
                fre[node * D + m] = (double)gr; fim[node * D + m] = (double)gi;
                // inverse H[node][m] stored transposed at [m][node]
                ire[m * D + node] = (double)(hr / (ld)D); iim[m * D + node] = (double)(hi / (ld)D);
            }
}
