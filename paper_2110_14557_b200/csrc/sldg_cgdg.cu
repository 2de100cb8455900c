// sldg_cgdg.cu -- CGdG Poisson solver: symmetric interior penalty (SIPG) dG discretisation
// of -Laplace phi = 1 - rho on the x grid + the mean-preserving conjugate gradient method of Algorithm 1
// (P:496-567), matrix-free, warm-started from the previous potential, E = -grad phi, sm_100a.
//
// Readings: I (M, B from eq. (4)), T (sigma: k^2, 2 for k = 1), U (E = cell-wise
// derivative of phi^DG at the nodes), V (arithmetic mean; loop entered only if ||r_0|| >= tol ||b||).
//
// The x grid is small (X <= ~1e5 unknowns), so the solve is latency bound: the WHOLE iteration runs in ONE
// cooperative launch (<= one 256-thread block per SM, grid-wide barriers between the phases of an iteration), no
// host round trip, no per-iteration launches.  Dot products are deterministic: block partials in a fixed slot,
// summed by every block in the same fixed order after the barrier, so every thread takes the same termination
// decision and two runs give the same bits.
#include <cooperative_groups.h>
#include <math.h>

#include "sldg_internal.h"

namespace cg = cooperative_groups;

namespace {

constexpr int CG_THREADS = 256;
constexpr int CG_SLOT = 512;          // doubles per reduction slot (>= blocks of the launch)

struct CgParams {
    int dx, K1;
    long long X;
    long long D[3];
    int N[3];
    double invh[3];
    const double* Wx[3];              // h_a w_j per node of x axis a
    double M[SLDG_MAXNN], B[SLDG_MAXNN], Dm[SLDG_MAXNN];   // reading I; Dm[a][b] = phi_b'(xi_a)
    double tol;
    int maxiter;
    const double* rho;
    double *phi, *r, *p, *w, *b, *E, *red, *info;
};

// block partial -> slot, fixed order
__device__ __forceinline__ void put_partial(double v, double* slot)
{
    __shared__ double sh[CG_THREADS / 32];
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    const int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (lane == 0) sh[wid] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        double s = 0.0;
        for (int i = 0; i < CG_THREADS / 32; i++) s += sh[i];
        slot[blockIdx.x] = s;
    }
    __syncthreads();
}
// after the grid barrier: every block sums the partials in the same order -> the same value everywhere
__device__ __forceinline__ double get_total(const double* slot)
{
    __shared__ double tot;
    if (threadIdx.x < 32) {
        double s = 0.0;
        for (int i = threadIdx.x; i < (int)gridDim.x; i += 32) s += __ldcg(slot + i);
        for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
        if (threadIdx.x == 0) tot = s;
    }
    __syncthreads();
    const double v = tot;
    __syncthreads();
    return v;
}

struct NodeIdx { long long n[3]; };
__device__ __forceinline__ NodeIdx split(const CgParams& P, long long x)
{
    NodeIdx q;
    for (int e = 0; e < 3; e++) {
        if (e < P.dx) { q.n[e] = x % P.D[e]; x /= P.D[e]; } else q.n[e] = 0;
    }
    return q;
}

// (A u)[x],  A = sum_d (prod_{e != d} h_e W_e) (x) A_hat_d / h_d
__device__ __forceinline__ double apply_A(const CgParams& P, const double* __restrict__ u, long long x)
{
    const int n = P.K1;
    const NodeIdx q = split(P, x);
    double out = 0.0;
    long long inner = 1;
    for (int d = 0; d < P.dx; d++) {
        double wo = 1.0;
        for (int e = 0; e < P.dx; e++)
            if (e != d) wo *= __ldg(P.Wx[e] + q.n[e]);
        const int i = (int)(q.n[d] / n), a = (int)(q.n[d] - (long long)i * n);
        const long long base = x - q.n[d] * inner;
        const int im = (i == 0) ? P.N[d] - 1 : i - 1, ip = (i == P.N[d] - 1) ? 0 : i + 1;
        double acc = 0.0;
        for (int b = 0; b < n; b++) acc += P.M[a * n + b] * __ldcg(u + base + ((long long)i * n + b) * inner);
        for (int b = 0; b < n; b++) acc += P.B[a * n + b] * __ldcg(u + base + ((long long)im * n + b) * inner);
        for (int b = 0; b < n; b++) acc += P.B[b * n + a] * __ldcg(u + base + ((long long)ip * n + b) * inner);
        out += wo * (acc * P.invh[d]);
        inner *= P.D[d];
    }
    return out;
}

// Algorithm 1 in the paper's order.  slots: 0 sum(u) / pw, 1 sum(r) / sw, 2 bb, 3 rr
__global__ void __launch_bounds__(CG_THREADS) cgdg_kernel(const CgParams P)
{
    cg::grid_group grid = cg::this_grid();
    const long long X = P.X;
    const long long g0 = (long long)blockIdx.x * CG_THREADS + threadIdx.x, gs = (long long)gridDim.x * CG_THREADS;
    double* const s0 = P.red, * const s1 = P.red + CG_SLOT, * const s2 = P.red + 2 * CG_SLOT,
          * const s3 = P.red + 3 * CG_SLOT;
    const double invX = 1.0 / (double)X;

    // b = W_x (1 - rho)  (right-hand side of eq. (4) with the diagonal mass matrix);  mean(u_0) = 0
    double acc = 0.0;
    for (long long x = g0; x < X; x += gs) {
        const NodeIdx q = split(P, x);
        double wx = 1.0;
        for (int e = 0; e < P.dx; e++) wx *= __ldg(P.Wx[e] + q.n[e]);
        P.b[x] = wx * (1.0 - __ldg(P.rho + x));
        acc += __ldcg(P.phi + x);
    }
    put_partial(acc, s0);
    grid.sync();
    const double mu = get_total(s0) * invX;
    for (long long x = g0; x < X; x += gs) __stcg(P.phi + x, __ldcg(P.phi + x) - mu);
    grid.sync();
    // r_0 = b - A u_0;  r_0 -= mean(r_0);  p_0 = r_0
    double sr = 0.0, bb = 0.0;
    for (long long x = g0; x < X; x += gs) {
        const double bx = P.b[x], rx = bx - apply_A(P, P.phi, x);
        P.r[x] = rx;
        sr += rx; bb += bx * bx;
    }
    put_partial(sr, s1);
    put_partial(bb, s2);
    grid.sync();
    const double mr = get_total(s1) * invX;
    bb = get_total(s2);
    acc = 0.0;
    for (long long x = g0; x < X; x += gs) {
        const double rx = P.r[x] - mr;
        P.r[x] = rx;
        __stcg(P.p + x, rx);
        acc += rx * rx;
    }
    put_partial(acc, s3);
    grid.sync();
    double rr = get_total(s3);
    int it = 0;
    if (rr > 0.0 && !(sqrt(rr) < P.tol * sqrt(bb))) {                       // reading V
        while (it < P.maxiter) {
            // [w_i, mean_w] = A p_i
            double pw = 0.0, sw = 0.0;
            for (long long x = g0; x < X; x += gs) {
                const double wx = apply_A(P, P.p, x);
                P.w[x] = wx;
                pw += __ldcg(P.p + x) * wx; sw += wx;
            }
            put_partial(pw, s0);
            put_partial(sw, s1);
            grid.sync();
            const double alpha = rr / get_total(s0);                        // alpha_i = r_i^T r_i / p_i^T w_i
            const double mw = get_total(s1) * invX;
            acc = 0.0;
            for (long long x = g0; x < X; x += gs) {
                __stcg(P.phi + x, __ldcg(P.phi + x) + alpha * __ldcg(P.p + x));   // u_{i+1} = u_i + alpha_i p_i
                const double rx = P.r[x] - alpha * (P.w[x] - mw);           // r_{i+1} = r_i - alpha_i (w_i - mean_w)
                P.r[x] = rx;
                acc += rx * rx;
            }
            put_partial(acc, s3);
            grid.sync();
            const double rr1 = get_total(s3);
            it++;
            if (sqrt(rr1) < P.tol * sqrt(bb)) { rr = rr1; break; }          // ||r_{i+1}||_2 < tol ||b||_2
            const double beta = rr1 / rr;                                   // beta_i
            for (long long x = g0; x < X; x += gs) __stcg(P.p + x, P.r[x] + beta * __ldcg(P.p + x));
            rr = rr1;
            grid.sync();
        }
    }
    grid.sync();
    // E_d = -(1/h_d) d/dxi phi^DG at the nodes (reading U)
    const int n = P.K1;
    for (long long x = g0; x < X; x += gs) {
        const NodeIdx q = split(P, x);
        long long inner = 1;
        for (int d = 0; d < P.dx; d++) {
            const int i = (int)(q.n[d] / n), a = (int)(q.n[d] - (long long)i * n);
            const long long base = x - q.n[d] * inner;
            double dv = 0.0;
            for (int b = 0; b < n; b++) dv += P.Dm[a * n + b] * __ldcg(P.phi + base + ((long long)i * n + b) * inner);
            P.E[(long long)d * X + x] = -(dv * P.invh[d]);
            inner *= P.D[d];
        }
    }
    if (g0 == 0) { P.info[0] = (double)it; P.info[1] = bb > 0.0 ? sqrt(rr / bb) : 0.0; }
}

long double lag(int n, const double* xi, int l, long double z)
{
    long double p = 1.0L;
    for (int m = 0; m < n; m++)
        if (m != l) p *= (z - (long double)xi[m]) / ((long double)xi[l] - (long double)xi[m]);
    return p;
}
long double dlag(int n, const double* xi, int l, long double z)
{
    long double s = 0.0L;
    for (int m = 0; m < n; m++) {
        if (m == l) continue;
        long double p = 1.0L / ((long double)xi[l] - (long double)xi[m]);
        for (int q = 0; q < n; q++)
            if (q != l && q != m) p *= (z - (long double)xi[q]) / ((long double)xi[l] - (long double)xi[q]);
        s += p;
    }
    return s;
}

}  // namespace

double sldg_sipg_sigma_default(int k) { return k >= 2 ? (double)(k * k) : 2.0; }

// M, B (reading I) and the nodal derivative matrix, row-major (k+1)x(k+1); host, long double
void sldg_sipg_tables(int k, const double* xi, const double* w, double sigma, double* M, double* B, double* Dm)
{
    const int n = k + 1;
    for (int a = 0; a < n; a++)
        for (int b = 0; b < n; b++) {
            long double vol = 0.0L;
            for (int l = 0; l < n; l++) vol += (long double)w[l] * dlag(n, xi, a, xi[l]) * dlag(n, xi, b, xi[l]);
            const long double pa0 = lag(n, xi, a, 0.0L), pa1 = lag(n, xi, a, 1.0L), pb0 = lag(n, xi, b, 0.0L),
                              pb1 = lag(n, xi, b, 1.0L), da0 = dlag(n, xi, a, 0.0L), da1 = dlag(n, xi, a, 1.0L),
                              db0 = dlag(n, xi, b, 0.0L), db1 = dlag(n, xi, b, 1.0L), s = sigma;
            M[a * n + b] = (double)(vol + 0.5L * (db0 * pa0 + pb0 * da0) + s * pb0 * pa0
                                        - 0.5L * (db1 * pa1 + pb1 * da1) + s * pb1 * pa1);
            B[a * n + b] = (double)(-0.5L * da0 * pb1 + 0.5L * pa0 * db1 - s * pa0 * pb1);
            Dm[a * n + b] = (double)dlag(n, xi, b, xi[a]);
        }
}

cudaError_t sldg_launch_poisson_cg(sldg_ctx* c, const double* rho, double* E, double tol, int maxiter, double sigma)
{
    CgParams P;
    P.dx = c->dx; P.K1 = c->K1; P.X = c->X;
    for (int a = 0; a < 3; a++) {
        P.D[a] = a < c->dx ? c->D[a] : 1; P.N[a] = a < c->dx ? c->cells[a] : 1;
        P.invh[a] = a < c->dx ? 1.0 / c->h[a] : 1.0; P.Wx[a] = a < c->dx ? c->dWx[a] : nullptr;
    }
    sldg_sipg_tables(c->k, c->xi, c->w, sigma, P.M, P.B, P.Dm);
    P.tol = tol; P.maxiter = maxiter;
    P.rho = rho; P.phi = c->phi; P.r = c->cplx[0]; P.p = c->cplx[1]; P.w = c->cplx[2]; P.b = c->cplx[3];
    P.E = E; P.red = c->red; P.info = c->cg_info;
    long long blocks = (c->X + CG_THREADS - 1) / CG_THREADS;
    int occ = 0;
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, cgdg_kernel, CG_THREADS, 0);
    if (e != cudaSuccess) return e;
    if (occ < 1) return cudaErrorInvalidConfiguration;
    if (blocks > c->sm_count) blocks = c->sm_count;          // one block per SM: cheap grid barriers
    if (blocks > CG_SLOT) blocks = CG_SLOT;
    void* args[] = {(void*)&P};
    return cudaLaunchCooperativeKernel((const void*)cgdg_kernel, dim3((unsigned)blocks), dim3(CG_THREADS), args, 0,
                                       c->stream);
}
