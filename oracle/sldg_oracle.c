/*
 * sldg_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Plain, slow, fp64 CPU statement of the split-step semi-Lagrangian discontinuous
 * Galerkin (SLDG) Vlasov-Poisson scheme of Einkemmer & Moriggl (arXiv 2110.14557),
 * written from the paper (/root/reference/PAPER.md, cited as P:line) and from the
 * readings fixed in SURVEY.md section 8(c) / DESIGN.md ("reading X").
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may load this.  It shares no code, table, constant generator or helper with the
 * CUDA path under paper_2110_14557_b200/csrc/.  No blocking, fusion or reordering
 * beyond what the definitions state; "#pragma omp parallel for" over independent
 * lines is the only concession to run time and does not change any arithmetic.
 *
 * Parity pins (tests/test_oracle_*.py):  every function below is pinned by at least
 * one of p1..p13 of DESIGN.md section 3.  "parity unpinned": the two-stream growth
 * rate (not in the paper) and the internals of the authors' own FFT solver (reading
 * P1 is pinned only by the closed forms p10/p11 and the physics pin p12); for the NEXT rows at the end of
 * this file: E from the dG potential (reading U), sigma for k = 1 (reading T) and which quantities the single
 * precision mode keeps in fp64 (reading W) are readings pinned by convergence / closed forms only.
 *
 * Layout of f (reading E): flat index n = n_0 + D_0 (n_1 + D_1 (n_2 + ...)),
 * axis order x_1..x_dx, v_1..v_dv (x_1 fastest), per-axis node index
 * n_a = i_a (k+1) + j_a (cell-major, Gauss-Legendre nodes interleaved), value stored
 * = f at coordinate lo_a + (i_a + xi_j) h_a.
 *
 * Build: gcc -O2 -ffp-contract=off -fopenmp -shared -fPIC  (see oracle/build.py).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_MAXDIM 6
#define ORC_MAXK 8

typedef struct orc_ctx {
    int dx, dv, d, k;
    int cells[ORC_MAXDIM];
    long D[ORC_MAXDIM];      /* nodes per axis = cells*(k+1)            */
    double lo[ORC_MAXDIM], hi[ORC_MAXDIM], h[ORC_MAXDIM];
    long nf, X, V;           /* |f|, prod of x nodes, prod of v nodes   */
    double xi[ORC_MAXK + 1], w[ORC_MAXK + 1];
    int threads;
} orc_ctx;

/* ------------------------------------------------------------------ O1 constants */

/* (n)-point Gauss-Legendre rule mapped to [0,1]: xi=(t+1)/2, w=w_t/2.
 * Newton iteration on the Legendre polynomial P_n in long double. */
void orc_gauss_legendre(int n, double *xi, double *w)
{
    const long double pi = 3.14159265358979323846264338327950288L;
    for (int i = 0; i < n; i++) {
        long double t = cosl(pi * ((long double)i + 0.75L) / ((long double)n + 0.5L));
        long double dp = 1.0L;
        for (int it = 0; it < 100; it++) {
            long double p0 = 1.0L, p1 = t;
            for (int m = 2; m <= n; m++) {
                long double p2 = ((2.0L * m - 1.0L) * t * p1 - (m - 1.0L) * p0) / m;
                p0 = p1; p1 = p2;
            }
            dp = n * (t * p1 - p0) / (t * t - 1.0L);   /* P_n'(t) */
            long double dt = p1 / dp;
            t -= dt;
            if (fabsl(dt) < 1e-21L) break;
        }
        /* recompute derivative at the converged root for the weight */
        long double p0 = 1.0L, p1 = t;
        for (int m = 2; m <= n; m++) {
            long double p2 = ((2.0L * m - 1.0L) * t * p1 - (m - 1.0L) * p0) / m;
            p0 = p1; p1 = p2;
        }
        dp = n * (t * p1 - p0) / (t * t - 1.0L);
        long double wt = 2.0L / ((1.0L - t * t) * dp * dp);
        /* roots come out descending in t; store ascending */
        xi[n - 1 - i] = (double)((t + 1.0L) / 2.0L);
        w[n - 1 - i] = (double)(wt / 2.0L);
    }
}

/* Lagrange basis l_l(z) = prod_{m != l} (z - xi_m)/(xi_l - xi_m), product form so that
 * l_l(xi_q) = delta_lq exactly. */
double orc_lagrange(int n, const double *xi, int l, double z)
{
    double r = 1.0;
    for (int m = 0; m < n; m++)
        if (m != l) r *= (z - xi[m]) / (xi[l] - xi[m]);
    return r;
}

/* ------------------------------------------------------------------ O2  A(alpha), B(alpha) */

/* Translate the piecewise polynomial by alpha cells (0 <= alpha < 1) and L2-project
 * cell-wise (Fig. 1).  The GL-Lagrange mass matrix is diagonal
 * (int l_j l_l = w_j delta_jl), hence (reading A)
 *   A_jl = (1/w_j) int_alpha^1 l_j(x) l_l(x - alpha)     dx   (donor = same cell,  i-s)
 *   B_jl = (1/w_j) int_0^alpha l_j(x) l_l(x - alpha + 1) dx   (donor = left cell, i-s-1)
 * Each integrand has degree 2k on its sub-interval, so the (k+1)-point GL rule mapped
 * to that sub-interval is exact.  A, B row-major (k+1)x(k+1). */
void orc_AB(int k, double alpha, double *A, double *B)
{
    int n = k + 1;
    double xi[ORC_MAXK + 1], w[ORC_MAXK + 1];
    orc_gauss_legendre(n, xi, w);
    for (int j = 0; j < n; j++) {
        for (int l = 0; l < n; l++) {
            double sa = 0.0, sb = 0.0;
            for (int q = 0; q < n; q++) {
                /* quadrature point on [alpha,1] */
                double xa = alpha + (1.0 - alpha) * xi[q];
                sa += (1.0 - alpha) * w[q] * orc_lagrange(n, xi, j, xa) * orc_lagrange(n, xi, l, xa - alpha);
                /* quadrature point on [0,alpha] */
                double xb = alpha * xi[q];
                sb += alpha * w[q] * orc_lagrange(n, xi, j, xb) * orc_lagrange(n, xi, l, xb - alpha + 1.0);
            }
            A[j * n + l] = sa / w[j];
            B[j * n + l] = sb / w[j];
        }
    }
}

/* ------------------------------------------------------------------ O3  1-D sweep */

static long pmod(long a, long n) { long r = a % n; return r < 0 ? r + n : r; }

/* One line, eq. (3) with reading B, given s mod N, alpha and A(alpha), B(alpha):
 *   u_i^new = A u_{(i-s) mod N} + B u_{(i-s-1) mod N},   i = 0..N-1.
 * alpha == 0 is a pure copy (integer shift = exact permutation, bit for bit).
 * uin/uout: node n of the line is at [n*stride]; N cells of k+1 nodes. */
static void sweep_line_AB(int k, int N, long s, double alpha, const double *A, const double *B,
                          const double *uin, double *uout, long stride)
{
    int n = k + 1;
    for (long i = 0; i < N; i++) {
        long ia = pmod(i - s, N);
        long ib = pmod(i - s - 1, N);
        for (int j = 0; j < n; j++) {
            if (alpha == 0.0) {
                uout[(i * n + j) * stride] = uin[(ia * n + j) * stride];
            } else {
                double acc = 0.0;
                for (int l = 0; l < n; l++) acc += A[j * n + l] * uin[(ia * n + l) * stride];
                for (int l = 0; l < n; l++) acc += B[j * n + l] * uin[(ib * n + l) * stride];
                uout[(i * n + j) * stride] = acc;
            }
        }
    }
}

/* s = floor(delta), alpha = delta - s in [0,1)  (reading B); s is returned mod N so that
 * donors stay correct for |s| >= N (reading O). */
static void split_delta(double delta, int N, long *s, double *alpha)
{
    double sd = floor(delta);
    *alpha = delta - sd;
    *s = (long)fmod(sd, (double)N);
}

/* One line shifted by delta cells. */
void orc_sweep_line(int k, int N, double delta, const double *uin, double *uout, long stride)
{
    long s; double alpha;
    double A[(ORC_MAXK + 1) * (ORC_MAXK + 1)], B[(ORC_MAXK + 1) * (ORC_MAXK + 1)];
    split_delta(delta, N, &s, &alpha);
    if (alpha != 0.0) orc_AB(k, alpha, A, B);
    sweep_line_AB(k, N, s, alpha, A, B, uin, uout, stride);
}

/* ------------------------------------------------------------------ context */

orc_ctx *orc_create(int dx, int dv, const int *cells, int k, const double *domain)
{
    if (dx < 1 || dv < 1 || dx + dv > ORC_MAXDIM || k < 0 || k > ORC_MAXK) return NULL;
    orc_ctx *c = (orc_ctx *)calloc(1, sizeof(orc_ctx));
    c->dx = dx; c->dv = dv; c->d = dx + dv; c->k = k;
    c->nf = 1; c->X = 1; c->V = 1;
    for (int a = 0; a < c->d; a++) {
        c->cells[a] = cells[a];
        c->D[a] = (long)cells[a] * (k + 1);
        c->lo[a] = domain[2 * a]; c->hi[a] = domain[2 * a + 1];
        c->h[a] = (c->hi[a] - c->lo[a]) / (double)cells[a];
        c->nf *= c->D[a];
        if (a < dx) c->X *= c->D[a]; else c->V *= c->D[a];
    }
    orc_gauss_legendre(k + 1, c->xi, c->w);
    c->threads = 1;
    return c;
}
void orc_destroy(orc_ctx *c) { free(c); }
void orc_set_threads(orc_ctx *c, int t) { c->threads = t < 1 ? 1 : t; }
int orc_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
long orc_field_elems(const orc_ctx *c) { return c->nf; }
long orc_rho_elems(const orc_ctx *c) { return c->X; }

/* coordinate of node n = i(k+1)+j on axis a:  lo + (i + xi_j) h */
static double node_coord(const orc_ctx *c, int a, long n)
{
    long i = n / (c->k + 1); int j = (int)(n % (c->k + 1));
    return c->lo[a] + ((double)i + c->xi[j]) * c->h[a];
}
void orc_node_coords(const orc_ctx *c, int axis, double *out)
{
    for (long n = 0; n < c->D[axis]; n++) out[n] = node_coord(c, axis, n);
}

/* Sweep every line along `axis`.  The line at (inner p, outer q) is shifted by
 * delta[idx(p,q)]:
 *   mode 0: idx = node index along axis `saxis` (> axis)        -- x-sweeps
 *   mode 1: idx = flat index over the x axes (all < axis)       -- v-sweeps */
void orc_sweep_axis(const orc_ctx *c, const double *fin, double *fout, int axis,
                    const double *delta, int mode, int saxis)
{
    long inner = 1, outer = 1, Da = c->D[axis];
    for (int a = 0; a < axis; a++) inner *= c->D[a];
    for (int a = axis + 1; a < c->d; a++) outer *= c->D[a];
    long sdiv = 1;
    if (mode == 0) for (int a = axis + 1; a < saxis; a++) sdiv *= c->D[a];
    long lines = inner * outer;
    /* A, B depend only on the advection speed and "can be precomputed": once per shift index */
    long nidx = (mode == 0) ? c->D[saxis] : c->X;
    int nn = (c->k + 1) * (c->k + 1);
    long *S = (long *)malloc(sizeof(long) * nidx);
    double *AL = (double *)malloc(sizeof(double) * nidx);
    double *AB = (double *)malloc(sizeof(double) * nidx * 2 * nn);
    for (long i = 0; i < nidx; i++) {
        split_delta(delta[i], c->cells[axis], &S[i], &AL[i]);
        if (AL[i] != 0.0) orc_AB(c->k, AL[i], AB + i * 2 * nn, AB + i * 2 * nn + nn);
    }
#pragma omp parallel for schedule(static) num_threads(c->threads)
    for (long t = 0; t < lines; t++) {
        long p = t % inner, q = t / inner;
        long idx = (mode == 0) ? (q / sdiv) % c->D[saxis] : p % c->X;
        long base = q * Da * inner + p;
        sweep_line_AB(c->k, c->cells[axis], S[idx], AL[idx], AB + idx * 2 * nn, AB + idx * 2 * nn + nn,
                      fin + base, fout + base, inner);
    }
    free(S); free(AL); free(AB);
}

/* x-advection, steps 1a-1c: for d = 1..dx  f(x_d - v_d tau), i.e. speed c = v_d,
 * delta = (c*tau)/h_{x_d} in that operation order (reading O3).  Result in f; tmp is |f| scratch. */
void orc_advect_x(const orc_ctx *c, double *f, double *tmp, double tau)
{
    for (int d = 0; d < c->dx; d++) {
        int b = c->dx + d;
        double *delta = (double *)malloc(sizeof(double) * c->D[b]);
        for (long n = 0; n < c->D[b]; n++) delta[n] = (node_coord(c, b, n) * tau) / c->h[d];
        orc_sweep_axis(c, f, tmp, d, delta, 0, b);
        memcpy(f, tmp, sizeof(double) * c->nf);
        free(delta);
    }
}

/* v-advection, steps 3a-3c: f(x, v_d + E_d(x) tau): speed c = -E_d(x-node)
 * (sign from eq. (1); reading H), only v_1..v_dx move (reading D).
 * E is [dx][X] component-major. */
void orc_advect_v(const orc_ctx *c, double *f, double *tmp, const double *E, double tau)
{
    for (int d = 0; d < c->dx; d++) {
        int a = c->dx + d;
        double *delta = (double *)malloc(sizeof(double) * c->X);
        for (long n = 0; n < c->X; n++) delta[n] = ((-E[d * c->X + n]) * tau) / c->h[a];
        orc_sweep_axis(c, f, tmp, a, delta, 1, -1);
        memcpy(f, tmp, sizeof(double) * c->nf);
        free(delta);
    }
}

/* ------------------------------------------------------------------ O4  rho */

/* rho[x] = sum_v (prod_d h_{v_d} w_{j_d}) f[x,v]  -- exact integral of the dG polynomial
 * (P:54).  long double accumulation. */
void orc_density(const orc_ctx *c, const double *f, double *rho)
{
    long X = c->X, V = c->V;
    double *W = (double *)malloc(sizeof(double) * V);
    for (long v = 0; v < V; v++) {
        long r = v; double wv = 1.0;
        for (int a = c->dx; a < c->d; a++) {
            long n = r % c->D[a]; r /= c->D[a];
            wv *= c->h[a] * c->w[n % (c->k + 1)];
        }
        W[v] = wv;
    }
#pragma omp parallel for schedule(static) num_threads(c->threads)
    for (long x = 0; x < X; x++) {
        long double acc = 0.0L;
        for (long v = 0; v < V; v++) acc += (long double)W[v] * (long double)f[v * X + x];
        rho[x] = (double)acc;
    }
    free(W);
}

/* ------------------------------------------------------------------ O5  Poisson / E (reading P1) */

/* apply an (n x n) matrix M to every cell along x-axis `a` of a [X] array (in place) */
static void apply_cellwise(const orc_ctx *c, double *g, int a, const double *M)
{
    int n = c->k + 1;
    long inner = 1, outer = 1;
    for (int b = 0; b < a; b++) inner *= c->D[b];
    for (int b = a + 1; b < c->dx; b++) outer *= c->D[b];
    double t[ORC_MAXK + 1];
    for (long q = 0; q < outer; q++)
        for (long p = 0; p < inner; p++)
            for (long i = 0; i < c->cells[a]; i++) {
                double *u = g + q * c->D[a] * inner + p + i * n * inner;
                for (int m = 0; m < n; m++) {
                    double acc = 0.0;
                    for (int l = 0; l < n; l++) acc += M[m * n + l] * u[l * inner];
                    t[m] = acc;
                }
                for (int m = 0; m < n; m++) u[m * inner] = t[m];
            }
}

/* naive O(D^2) DFT along x-axis `a` of a complex [X] array (re, im), sign = -1 forward, +1 inverse
 * (no scaling).  Twiddle argument reduced with integer (m*n) mod D. */
static void dft_axis(const orc_ctx *c, double *re, double *im, int a, int sign)
{
    const long double twopi = 6.28318530717958647692528676655900577L;
    long D = c->D[a], inner = 1, outer = 1;
    for (int b = 0; b < a; b++) inner *= c->D[b];
    for (int b = a + 1; b < c->dx; b++) outer *= c->D[b];
    double *cs = (double *)malloc(sizeof(double) * D), *sn = (double *)malloc(sizeof(double) * D);
    for (long r = 0; r < D; r++) {
        cs[r] = (double)cosl(twopi * (long double)r / (long double)D);
        sn[r] = (double)sinl(twopi * (long double)r / (long double)D);
    }
    double *tr = (double *)malloc(sizeof(double) * D), *ti = (double *)malloc(sizeof(double) * D);
    for (long q = 0; q < outer; q++)
        for (long p = 0; p < inner; p++) {
            double *lr = re + q * D * inner + p, *li = im + q * D * inner + p;
            for (long m = 0; m < D; m++) {
                double ar = 0.0, ai = 0.0;
                for (long n = 0; n < D; n++) {
                    long r = (m * n) % D;
                    double cr = cs[r], ci = sign * sn[r];      /* e^{sign * 2 pi i m n / D} */
                    double xr = lr[n * inner], xi_ = li[n * inner];
                    ar += xr * cr - xi_ * ci;
                    ai += xr * ci + xi_ * cr;
                }
                tr[m] = ar; ti[m] = ai;
            }
            for (long m = 0; m < D; m++) { lr[m * inner] = tr[m]; li[m * inner] = ti[m]; }
        }
    free(cs); free(sn); free(tr); free(ti);
}

/* invert a small matrix by Gauss-Jordan with partial pivoting (long double) */
static void invert_small(int n, const double *M, double *Minv)
{
    long double a[(ORC_MAXK + 1)][2 * (ORC_MAXK + 1)];
    for (int i = 0; i < n; i++)
        for (int j = 0; j < n; j++) { a[i][j] = M[i * n + j]; a[i][n + j] = (i == j); }
    for (int col = 0; col < n; col++) {
        int piv = col;
        for (int r = col + 1; r < n; r++) if (fabsl(a[r][col]) > fabsl(a[piv][col])) piv = r;
        for (int j = 0; j < 2 * n; j++) { long double t = a[col][j]; a[col][j] = a[piv][j]; a[piv][j] = t; }
        long double d = a[col][col];
        for (int j = 0; j < 2 * n; j++) a[col][j] /= d;
        for (int r = 0; r < n; r++) if (r != col) {
            long double fct = a[r][col];
            for (int j = 0; j < 2 * n; j++) a[r][j] -= fct * a[col][j];
        }
    }
    for (int i = 0; i < n; i++) for (int j = 0; j < n; j++) Minv[i * n + j] = (double)a[i][n + j];
}

/* -Laplace(phi) = 1 - rho periodic, E = -grad(phi), at the x DG nodes.
 * Reading P1 ("FFT based ... interpolation to and from the equidistant grid"):
 *  (i)  per axis, evaluate each cell's degree-k interpolant at the k+1 equidistant points
 *       eta_m = (m+1/2)/(k+1)  (matrix P_ml = l_l(eta_m)) -> uniform periodic grid;
 *  (ii) forward DFT;  (iii) E^_d = i kappa_d rho^ / |kappa|^2 for kappa != 0, 0 for kappa = 0,
 *       kappa_d := 0 in the numerator at the Nyquist index of an even-length axis;
 *  (iv) inverse DFT, real part;  (v) per cell map the equidistant values back with P^-1.
 * E is [dx][X] component-major. */
void orc_poisson(const orc_ctx *c, const double *rho, double *E)
{
    const long double twopi = 6.28318530717958647692528676655900577L;
    int n = c->k + 1, dx = c->dx;
    long X = c->X;
    double P[(ORC_MAXK + 1) * (ORC_MAXK + 1)], Pinv[(ORC_MAXK + 1) * (ORC_MAXK + 1)];
    for (int m = 0; m < n; m++)
        for (int l = 0; l < n; l++)
            P[m * n + l] = orc_lagrange(n, c->xi, l, ((double)m + 0.5) / (double)n);
    invert_small(n, P, Pinv);

    double *gr = (double *)malloc(sizeof(double) * X), *gi = (double *)calloc(X, sizeof(double));
    memcpy(gr, rho, sizeof(double) * X);
    for (int a = 0; a < dx; a++) apply_cellwise(c, gr, a, P);          /* (i)  */
    for (int a = 0; a < dx; a++) dft_axis(c, gr, gi, a, -1);           /* (ii) */

    double *er = (double *)malloc(sizeof(double) * X), *ei = (double *)malloc(sizeof(double) * X);
    for (int d = 0; d < dx; d++) {
        for (long t = 0; t < X; t++) {                                 /* (iii) */
            long r = t; double k2 = 0.0, kd = 0.0;
            for (int a = 0; a < dx; a++) {
                long m = r % c->D[a]; r /= c->D[a];
                long mm = (2 * m < c->D[a]) ? m : m - c->D[a];         /* signed frequency */
                double kap = (double)(twopi * (long double)mm / (long double)(c->hi[a] - c->lo[a]));
                k2 += kap * kap;
                if (a == d) kd = (2 * m == c->D[a]) ? 0.0 : kap;       /* Nyquist -> 0 */
            }
            if (k2 == 0.0) { er[t] = 0.0; ei[t] = 0.0; }
            else {                                                      /* i*kd*(gr + i gi)/k2 */
                er[t] = -kd * gi[t] / k2;
                ei[t] = kd * gr[t] / k2;
            }
        }
        for (int a = 0; a < dx; a++) dft_axis(c, er, ei, a, +1);       /* (iv) */
        for (long t = 0; t < X; t++) er[t] = er[t] / (double)X;
        for (int a = 0; a < dx; a++) apply_cellwise(c, er, a, Pinv);   /* (v)  */
        memcpy(E + d * X, er, sizeof(double) * X);
    }
    free(gr); free(gi); free(er); free(ei);
}

/* ------------------------------------------------------------------ O6  Strang step, O7 diagnostics */

/* x(dt/2) -> rho -> E -> v(dt) -> x(dt/2).  rho [X], E [dx][X] are outputs too. */
void orc_step(const orc_ctx *c, double *f, double *tmp, double *rho, double *E, double dt)
{
    orc_advect_x(c, f, tmp, dt / 2.0);
    orc_density(c, f, rho);
    orc_poisson(c, rho, E);
    orc_advect_v(c, f, tmp, E, dt);
    orc_advect_x(c, f, tmp, dt / 2.0);
}

/* mass = sum_n (prod_a h_a w_{j_a}) f_n */
double orc_mass(const orc_ctx *c, const double *f)
{
    long double acc = 0.0L;
    for (long t = 0; t < c->nf; t++) {
        long r = t; double wn = 1.0;
        for (int a = 0; a < c->d; a++) {
            long n = r % c->D[a]; r /= c->D[a];
            wn *= c->h[a] * c->w[n % (c->k + 1)];
        }
        acc += (long double)wn * (long double)f[t];
    }
    return (double)acc;
}

/* electric energy = 1/2 sum_x W_x |E(x)|^2 */
double orc_electric_energy(const orc_ctx *c, const double *E)
{
    long double acc = 0.0L;
    for (long t = 0; t < c->X; t++) {
        long r = t; double wn = 1.0;
        for (int a = 0; a < c->dx; a++) {
            long n = r % c->D[a]; r /= c->D[a];
            wn *= c->h[a] * c->w[n % (c->k + 1)];
        }
        long double e2 = 0.0L;
        for (int d = 0; d < c->dx; d++) e2 += (long double)E[d * c->X + t] * (long double)E[d * c->X + t];
        acc += (long double)wn * e2;
    }
    return (double)(0.5L * acc);
}

/* ================================================================== NEXT row
 * CGdG Poisson solver: SIPG discretisation + mean-preserving CG   (Appendix, Algorithm 1)
 *
 * Readings (I / T / U / V):
 *  I  M, B of P:525-527 are garbled; taken from eq. (4) with [v] = v^- - v^+, {v} = (v^- + v^+)/2,
 *     reference basis on [0,1], weights summing to 1, everything times 1/h:
 *       M_ab = sum_l w_l phi_a'(xi_l) phi_b'(xi_l)
 *              + 1/2 phi_b'(0) phi_a(0) + 1/2 phi_b(0) phi_a'(0) + sigma phi_b(0) phi_a(0)
 *              - 1/2 phi_b'(1) phi_a(1) - 1/2 phi_b(1) phi_a'(1) + sigma phi_b(1) phi_a(1)
 *       B_ab = -1/2 phi_a'(0) phi_b(1) + 1/2 phi_a(0) phi_b'(1) - sigma phi_a(0) phi_b(1)
 *     (A_hat u)_i = M u_i + B u_{i-1} + B^T u_{i+1}, periodic;  A_x = A_hat / h_x.
 *  T  sigma "set to its minimum allowed value", sigma >= k^2: k^2 for k >= 2; for k = 1 the
 *     value k^2 = 1 leaves a second null vector and first-order convergence, so 2 is used; k = 0 is rejected.
 *  U  E = -grad phi is the cell-wise derivative of phi^DG at the Gauss-Legendre nodes (paper silent).
 *  V  mean(.) in Algorithm 1 is the arithmetic mean of the coefficient vector (the null vector of A is the
 *     constant coefficient vector); the loop is entered only if ||r_0|| >= tol ||b|| and r_0 != 0.
 * Pins: tests/test_oracle_cgdg.py. */

/* d/dz of the Lagrange basis l_l at z */
double orc_lagrange_deriv(int n, const double *xi, int l, double z)
{
    long double s = 0.0L;
    for (int m = 0; m < n; m++) {
        if (m == l) continue;
        long double p = 1.0L / ((long double)xi[l] - (long double)xi[m]);
        for (int q = 0; q < n; q++)
            if (q != l && q != m) p *= ((long double)z - (long double)xi[q]) / ((long double)xi[l] - (long double)xi[q]);
        s += p;
    }
    return (double)s;
}

double orc_sipg_sigma_default(int k) { return k >= 2 ? (double)(k * k) : 2.0; }

/* M, B of reading I, row-major (k+1)x(k+1) */
void orc_sipg_MB(int k, double sigma, double *M, double *B)
{
    int n = k + 1;
    double xi[ORC_MAXK + 1], w[ORC_MAXK + 1];
    orc_gauss_legendre(n, xi, w);
    for (int a = 0; a < n; a++)
        for (int b = 0; b < n; b++) {
            double vol = 0.0;
            for (int l = 0; l < n; l++)
                vol += w[l] * orc_lagrange_deriv(n, xi, a, xi[l]) * orc_lagrange_deriv(n, xi, b, xi[l]);
            double pa0 = orc_lagrange(n, xi, a, 0.0), pa1 = orc_lagrange(n, xi, a, 1.0);
            double pb0 = orc_lagrange(n, xi, b, 0.0), pb1 = orc_lagrange(n, xi, b, 1.0);
            double da0 = orc_lagrange_deriv(n, xi, a, 0.0), da1 = orc_lagrange_deriv(n, xi, a, 1.0);
            double db0 = orc_lagrange_deriv(n, xi, b, 0.0), db1 = orc_lagrange_deriv(n, xi, b, 1.0);
            M[a * n + b] = vol + 0.5 * db0 * pa0 + 0.5 * pb0 * da0 + sigma * pb0 * pa0
                               - 0.5 * db1 * pa1 - 0.5 * pb1 * da1 + sigma * pb1 * pa1;
            B[a * n + b] = -0.5 * da0 * pb1 + 0.5 * pa0 * db1 - sigma * pa0 * pb1;
        }
}

/* out = A u on the x grid [X]:  A = sum_d (prod_{e != d} h_e W_e) (x) A_hat_d / h_d */
void orc_sipg_apply(const orc_ctx *c, double sigma, const double *u, double *out)
{
    int n = c->k + 1;
    double M[(ORC_MAXK + 1) * (ORC_MAXK + 1)], B[(ORC_MAXK + 1) * (ORC_MAXK + 1)];
    orc_sipg_MB(c->k, sigma, M, B);
    for (long x = 0; x < c->X; x++) out[x] = 0.0;
    for (int d = 0; d < c->dx; d++) {
        long inner = 1;
        for (int b = 0; b < d; b++) inner *= c->D[b];
        long N = c->cells[d];
        for (long x = 0; x < c->X; x++) {
            /* node indices of x on every axis; weight of the other axes */
            long rem = x, nd = 0;
            double wo = 1.0;
            for (int e = 0; e < c->dx; e++) {
                long ne = rem % c->D[e];
                rem /= c->D[e];
                if (e == d) nd = ne;
                else wo *= c->h[e] * c->w[ne % n];
            }
            long i = nd / n, a = nd % n;
            long base = x - nd * inner;                       /* node 0 of this line */
            long im = pmod(i - 1, N), ip = pmod(i + 1, N);
            double acc = 0.0;
            for (int b = 0; b < n; b++) acc += M[a * n + b] * u[base + (i * n + b) * inner];
            for (int b = 0; b < n; b++) acc += B[a * n + b] * u[base + (im * n + b) * inner];
            for (int b = 0; b < n; b++) acc += B[b * n + a] * u[base + (ip * n + b) * inner];
            out[x] += wo * (acc / c->h[d]);
        }
    }
}

/* E_d = -(1/h_d) d/dxi phi^DG at the x DG nodes (reading U); E is [dx][X] */
void orc_grad_phi(const orc_ctx *c, const double *phi, double *E)
{
    int n = c->k + 1;
    double Dm[(ORC_MAXK + 1) * (ORC_MAXK + 1)];               /* Dm[a][b] = phi_b'(xi_a) */
    for (int a = 0; a < n; a++)
        for (int b = 0; b < n; b++) Dm[a * n + b] = orc_lagrange_deriv(n, c->xi, b, c->xi[a]);
    for (int d = 0; d < c->dx; d++) {
        long inner = 1;
        for (int b = 0; b < d; b++) inner *= c->D[b];
        for (long x = 0; x < c->X; x++) {
            long nd = (x / inner) % c->D[d];
            long i = nd / n, a = nd % n;
            long base = x - nd * inner;
            double acc = 0.0;
            for (int b = 0; b < n; b++) acc += Dm[a * n + b] * phi[base + (i * n + b) * inner];
            E[d * c->X + x] = -(acc / c->h[d]);
        }
    }
}

static double vec_mean(const double *v, long n)
{
    long double s = 0.0L;
    for (long i = 0; i < n; i++) s += v[i];
    return (double)(s / (long double)n);
}
static double vec_dot(const double *a, const double *b, long n)
{
    long double s = 0.0L;
    for (long i = 0; i < n; i++) s += (long double)a[i] * (long double)b[i];
    return (double)s;
}

/* b = W_x (1 - rho): right-hand side of eq. (4) with the diagonal Gauss-Legendre mass matrix */
void orc_sipg_rhs(const orc_ctx *c, const double *rho, double *b)
{
    int n = c->k + 1;
    for (long x = 0; x < c->X; x++) {
        long rem = x;
        double wx = 1.0;
        for (int e = 0; e < c->dx; e++) { wx *= c->h[e] * c->w[(rem % c->D[e]) % n]; rem /= c->D[e]; }
        b[x] = wx * (1.0 - rho[x]);
    }
}

/* Algorithm 1, mean-preserving CG, step by step in the paper's order and notation.
 * phi: in = starting vector u_0 (its mean is removed first), out = solution.  E = -grad phi (reading U).
 * info[0] = ||r||_2 / ||b||_2 at exit, info[1] = eta.  Returns the number of iterations performed. */
int orc_poisson_cg(const orc_ctx *c, double sigma, const double *rho, double *phi, double *E, double tol,
                   int maxiter, double *info)
{
    long X = c->X;
    double *b = malloc(sizeof(double) * X), *r = malloc(sizeof(double) * X);
    double *p = malloc(sizeof(double) * X), *w = malloc(sizeof(double) * X);
    double *u = phi;
    orc_sipg_rhs(c, rho, b);
    double m = vec_mean(u, X);                                 /* mean(u_0) = 0 */
    for (long x = 0; x < X; x++) u[x] -= m;
    orc_sipg_apply(c, sigma, u, w);
    for (long x = 0; x < X; x++) r[x] = b[x] - w[x];           /* r_0 = b - A u_0 */
    m = vec_mean(r, X);
    for (long x = 0; x < X; x++) { r[x] -= m; p[x] = r[x]; }   /* r_0 = r_0 - mean(r_0), p_0 = r_0 */
    double eta = 0.0;
    for (long x = 0; x < X; x++) eta += (b[x] + r[x]) * u[x];  /* eta = (b + r_0)^T u_0 */
    double bb = vec_dot(b, b, X), rr = vec_dot(r, r, X);
    int it = 0;
    if (rr > 0.0 && !(sqrt(rr) < tol * sqrt(bb))) {            /* reading V */
        while (it < maxiter) {
            orc_sipg_apply(c, sigma, p, w);                    /* [w_i, mean_w] = A p_i */
            double mw = vec_mean(w, X);
            double alpha = rr / vec_dot(p, w, X);              /* alpha_i = r_i^T r_i / p_i^T w_i */
            for (long x = 0; x < X; x++) u[x] += alpha * p[x];
            for (long x = 0; x < X; x++) r[x] -= alpha * (w[x] - mw);
            eta += alpha * rr;
            double rr1 = vec_dot(r, r, X);
            it++;
            if (sqrt(rr1) < tol * sqrt(bb)) { rr = rr1; break; }
            double beta = rr1 / rr;                            /* beta_i = r_{i+1}^T r_{i+1} / r_i^T r_i */
            for (long x = 0; x < X; x++) p[x] = r[x] + beta * p[x];
            rr = rr1;
        }
    }
    if (info) { info[0] = bb > 0.0 ? sqrt(rr / bb) : 0.0; info[1] = eta; }
    orc_grad_phi(c, u, E);
    free(b); free(r); free(p); free(w);
    return it;
}

/* ================================================================== NEXT row
 * Single precision mode ("running simulations ... in single precision is a viable option. This reduces
 * memory consumption by a factor of two"; Tables 3-4 report fp32 throughout).
 *
 * Reading W: f is STORED in fp32 and the sweep arithmetic of eq. (3) runs in fp32
 * (coefficients A, B rounded to fp32, every product and sum rounded to fp32); everything that is O(X) stays
 * fp64: the shift delta, s = floor(delta), alpha and A(alpha), B(alpha) before rounding, rho (fp64 sum of the
 * fp32 values), the field solve and E.  So integer decisions are taken in fp64 exactly as in the fp64 path.
 * Same functions as above with float storage; no other change of order. */

static void sweep_line_AB_f32(int k, int N, long s, double alpha, const float *A, const float *B,
                              const float *uin, float *uout, long stride)
{
    int n = k + 1;
    for (long i = 0; i < N; i++) {
        long ia = pmod(i - s, N);
        long ib = pmod(i - s - 1, N);
        for (int j = 0; j < n; j++) {
            if (alpha == 0.0) {
                uout[(i * n + j) * stride] = uin[(ia * n + j) * stride];
            } else {
                float acc = 0.0f;
                for (int l = 0; l < n; l++) acc += A[j * n + l] * uin[(ia * n + l) * stride];
                for (int l = 0; l < n; l++) acc += B[j * n + l] * uin[(ib * n + l) * stride];
                uout[(i * n + j) * stride] = acc;
            }
        }
    }
}

void orc_sweep_axis_f32(const orc_ctx *c, const float *fin, float *fout, int axis,
                        const double *delta, int mode, int saxis)
{
    long inner = 1, outer = 1, Da = c->D[axis];
    for (int a = 0; a < axis; a++) inner *= c->D[a];
    for (int a = axis + 1; a < c->d; a++) outer *= c->D[a];
    long sdiv = 1;
    if (mode == 0) for (int a = axis + 1; a < saxis; a++) sdiv *= c->D[a];
    long lines = inner * outer;
    long nidx = (mode == 0) ? c->D[saxis] : c->X;
    int nn = (c->k + 1) * (c->k + 1);
    long *S = (long *)malloc(sizeof(long) * nidx);
    double *AL = (double *)malloc(sizeof(double) * nidx);
    float *AB = (float *)malloc(sizeof(float) * nidx * 2 * nn);
    double A64[(ORC_MAXK + 1) * (ORC_MAXK + 1)], B64[(ORC_MAXK + 1) * (ORC_MAXK + 1)];
    for (long i = 0; i < nidx; i++) {
        split_delta(delta[i], c->cells[axis], &S[i], &AL[i]);              /* fp64 decision */
        if (AL[i] != 0.0) {
            orc_AB(c->k, AL[i], A64, B64);
            for (int m = 0; m < nn; m++) { AB[i * 2 * nn + m] = (float)A64[m]; AB[i * 2 * nn + nn + m] = (float)B64[m]; }
        }
    }
#pragma omp parallel for schedule(static) num_threads(c->threads)
    for (long t = 0; t < lines; t++) {
        long p = t % inner, q = t / inner;
        long idx = (mode == 0) ? (q / sdiv) % c->D[saxis] : p % c->X;
        long base = q * Da * inner + p;
        sweep_line_AB_f32(c->k, c->cells[axis], S[idx], AL[idx], AB + idx * 2 * nn, AB + idx * 2 * nn + nn,
                          fin + base, fout + base, inner);
    }
    free(S); free(AL); free(AB);
}

void orc_advect_x_f32(const orc_ctx *c, float *f, float *tmp, double tau)
{
    for (int d = 0; d < c->dx; d++) {
        int b = c->dx + d;
        double *delta = (double *)malloc(sizeof(double) * c->D[b]);
        for (long n = 0; n < c->D[b]; n++) delta[n] = (node_coord(c, b, n) * tau) / c->h[d];
        orc_sweep_axis_f32(c, f, tmp, d, delta, 0, b);
        memcpy(f, tmp, sizeof(float) * c->nf);
        free(delta);
    }
}

void orc_advect_v_f32(const orc_ctx *c, float *f, float *tmp, const double *E, double tau)
{
    for (int d = 0; d < c->dx; d++) {
        int a = c->dx + d;
        double *delta = (double *)malloc(sizeof(double) * c->X);
        for (long n = 0; n < c->X; n++) delta[n] = ((-E[d * c->X + n]) * tau) / c->h[a];
        orc_sweep_axis_f32(c, f, tmp, a, delta, 1, -1);
        memcpy(f, tmp, sizeof(float) * c->nf);
        free(delta);
    }
}

/* rho in fp64 from the fp32 values (reading W) */
void orc_density_f32(const orc_ctx *c, const float *f, double *rho)
{
    long X = c->X, V = c->V;
    double *W = (double *)malloc(sizeof(double) * V);
    for (long v = 0; v < V; v++) {
        long r = v; double wv = 1.0;
        for (int a = c->dx; a < c->d; a++) {
            long n = r % c->D[a]; r /= c->D[a];
            wv *= c->h[a] * c->w[n % (c->k + 1)];
        }
        W[v] = wv;
    }
#pragma omp parallel for schedule(static) num_threads(c->threads)
    for (long x = 0; x < X; x++) {
        long double acc = 0.0L;
        for (long v = 0; v < V; v++) acc += (long double)W[v] * (long double)f[v * X + x];
        rho[x] = (double)acc;
    }
    free(W);
}

void orc_step_f32(const orc_ctx *c, float *f, float *tmp, double *rho, double *E, double dt)
{
    orc_advect_x_f32(c, f, tmp, dt / 2.0);
    orc_density_f32(c, f, rho);
    orc_poisson(c, rho, E);
    orc_advect_v_f32(c, f, tmp, E, dt);
    orc_advect_x_f32(c, f, tmp, dt / 2.0);
}

double orc_mass_f32(const orc_ctx *c, const float *f)
{
    long double acc = 0.0L;
    for (long t = 0; t < c->nf; t++) {
        long r = t; double wn = 1.0;
        for (int a = 0; a < c->d; a++) {
            long n = r % c->D[a]; r /= c->D[a];
            wn *= c->h[a] * c->w[n % (c->k + 1)];
        }
        acc += (long double)wn * (long double)f[t];
    }
    return (double)acc;
}
