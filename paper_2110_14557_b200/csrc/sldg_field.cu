// sldg_field.cu -- rho reduction, Poisson/E solve, v-sweep shift tables and diagnostics, sm_100a.
//
//  rho[x] = sum_v W_v f[x,v]   HBM-bound: one read of f
//  -Laplace phi = 1 - rho, E = -grad phi  (reading P1)     tiny, latency-bound
//  per-x-node shift tables of the v-sweeps
#include "sldg_async.h"
#include "sldg_internal.h"
#include "sldg_tmap.h"

// The polynomial coefficients of A(alpha), B(alpha) depend on the degree: each context owns its device copy (c->dPoly),
// so contexts of different degree can live side by side.
cudaError_t sldg_upload_poly(sldg_ctx* c)
{
    cudaError_t e = cudaMalloc((void**)&c->dPoly, sizeof(ABPoly));
    if (e != cudaSuccess) return e;
    return cudaMemcpy(c->dPoly, &c->poly, sizeof(ABPoly), cudaMemcpyHostToDevice);
}

#define SLDG_RHO_U 8          // loads in flight per thread of the rho kernel

namespace {

// ------------------------------------------------------------------ v-sweep shift table (row a5)
// delta = ((-E) * tau) / h_v in exactly this operation order (reading O3); s = floor(delta), alpha = delta - s.
// A(alpha), B(alpha) by Horner on the polynomial coefficients.  Output SoA: AB[m][X].
template <int K1, class TAB>
__global__ void vtable_kernel(const ABPoly* __restrict__ poly, const double* __restrict__ Ed, double tau, double hv, int N,
                              long long X, int* __restrict__ S, TAB* __restrict__ AB)
{
    long long x = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (x >= X) return;
    constexpr int NN = K1 * K1;
    double delta = __ddiv_rn(__dmul_rn(-Ed[x], tau), hv);
    double sd = floor(delta);
    double alpha = delta - sd;
    double sm = fmod(sd, (double)N);
    int s = (int)sm;
    if (s < 0) s += N;
    bool cp = (alpha == 0.0);
    S[x] = s | (cp ? SLDG_COPY_BIT : 0);
    const double xc = alpha - 0.5;              // coefficients are in powers of (alpha - 1/2)
#pragma unroll
    for (int m = 0; m < NN; m++) {
        double a = sldg_horner<K1>(*poly, 0, m, xc), b = sldg_horner<K1>(*poly, 1, m, xc);
        if (cp) { a = (m % (K1 + 1) == 0) ? 1.0 : 0.0; b = 0.0; }
        AB[(long long)m * X + x] = (TAB)a;
        AB[(long long)(NN + m) * X + x] = (TAB)b;
    }
}

// ------------------------------------------------------------------ velocity quadrature weights W_v
struct WvParams { int dv; long long Dv[3]; const double* w[3]; long long V; };
__global__ void wv_kernel(WvParams P, double* __restrict__ Wv)
{
    long long v = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (v >= P.V) return;
    long long r = v;
    double wv = 1.0;
    for (int a = 0; a < P.dv; a++) {
        long long n = r % P.Dv[a]; r /= P.Dv[a];
        wv *= P.w[a][n];
    }
    Wv[v] = wv;
}

// ------------------------------------------------------------------ rho (row a3)
// f seen as [V][X] (X contiguous).  Block = 128 threads x 2 values along x; grid.y splits V into chunks.
// Each chunk writes a partial sum; a second kernel adds the partials in a fixed order (deterministic).
template <class T> struct Pair;
template <> struct Pair<double> { typedef double2 type; };
template <> struct Pair<float> { typedef float2 type; };

template <int VEC, class T>
__global__ void __launch_bounds__(128) rho_partial_kernel(const T* __restrict__ f, const double* __restrict__ Wv,
                                                          long long X, long long V, long long vchunk,
                                                          double* __restrict__ part)
{
    long long x = ((long long)blockIdx.x * blockDim.x + threadIdx.x) * VEC;
    if (x >= X) return;
    long long v0 = (long long)blockIdx.y * vchunk;
    long long v1 = v0 + vchunk; if (v1 > V) v1 = V;
    double acc[VEC] = {0};
    constexpr int U = SLDG_RHO_U;
    long long v = v0;
    for (; v + U <= v1; v += U) {
        T t[U][VEC];
#pragma unroll
        for (int u = 0; u < U; u++) {
            const T* p = f + (v + u) * X + x;
            if (VEC == 2) { typename Pair<T>::type d = __ldcs(reinterpret_cast<const typename Pair<T>::type*>(p)); t[u][0] = d.x; t[u][VEC - 1] = d.y; }
            else t[u][0] = __ldcs(p);
        }
#pragma unroll
        for (int u = 0; u < U; u++) {
            double wv = __ldg(Wv + v + u);
#pragma unroll
            for (int e = 0; e < VEC; e++) acc[e] = fma(wv, (double)t[u][e], acc[e]);
        }
    }
    for (; v < v1; v++) {
        double wv = __ldg(Wv + v);
#pragma unroll
        for (int e = 0; e < VEC; e++) acc[e] = fma(wv, (double)__ldcs(f + v * X + x + e), acc[e]);
    }
#pragma unroll
    for (int e = 0; e < VEC; e++) part[(long long)blockIdx.y * X + x + e] = acc[e];
}

// rho by TMA (large problems): f seen as [V][X]; a block owns a tile of 32 x values and a chunk of v rows and streams boxes
// of 32 x RHO_ROWS values (2-d tensor copies into a full/empty mbarrier ring; profiles/r2_probe_load_rate.md: this path streams at
// 1.05-1.1 of the device-copy rate, the plain-load kernel above at 0.95).  Lane = two x values, warp w sums rows w, w + 8, ... of
// every box in ascending v with fma(W_v, f, acc); the eight warps' sums are added in warp order: deterministic.
constexpr int RHO_WX = 64, RHO_ROWS = 32, RHO_WARPS = 8;     // lane = TWO x values (one 16-byte / 8-byte load per row)
struct RhoTmaParams { const double* Wv; double* part; long long X, V, vchunk; int ntiles, slots; uint32_t slot_bytes; };

template <class T>
__global__ void __launch_bounds__(RHO_WARPS * 32) rho_tma_kernel(const __grid_constant__ CUtensorMap tmap, const RhoTmaParams P)
{
    using namespace sldg_async;
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    const int ST = P.slots;
    const uint32_t ring_s = smem_u32(smem_raw);
    const uint32_t full_s = ring_s + (uint32_t)ST * P.slot_bytes, empty_s = full_s + 8u * ST;
    const int t = threadIdx.x, lane = t & 31, w = t >> 5;
    const int tile = (int)(blockIdx.x % (unsigned)P.ntiles);
    const long long chunk = blockIdx.x / (unsigned)P.ntiles;
    const long long v0 = chunk * P.vchunk;
    const long long v1 = min(P.V, v0 + P.vchunk);
    const int total = (int)((v1 - v0 + RHO_ROWS - 1) / RHO_ROWS);
    if (t == 0) {
        for (int s = 0; s < ST; s++) { mbar_init(full_s + 8u * s, 1); mbar_init(empty_s + 8u * s, RHO_WARPS); }
        mbar_init_fence();
    }
    __syncthreads();
    const uint32_t box_bytes = (uint32_t)(RHO_ROWS * RHO_WX * sizeof(T));
    int pst = 0, pn = 0, pi = 0;
    auto produce = [&]() {
        if (pi >= total) return;
        if (pn > 0) mbar_wait(empty_s + 8u * pst, (uint32_t)((pn - 1) & 1));
        mbar_expect_tx(full_s + 8u * pst, box_bytes);
        asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                     ::"r"(ring_s + (uint32_t)pst * P.slot_bytes), "l"(&tmap), "r"(tile * RHO_WX), "r"((int)(v0 + (long long)pi * RHO_ROWS)),
                       "r"(full_s + 8u * pst) : "memory");
        if (++pst == ST) { pst = 0; pn++; }
        pi++;
    };
    if (t == 0) for (int i = 0; i < ST - 1; i++) produce();
    int st = 0; uint32_t ph = 0;
    double acc0[2] = {0.0, 0.0}, acc1[2] = {0.0, 0.0};              // [x value of the lane], even / odd rows of this warp
    for (int i = 0; i < total; i++) {
        if (t == 0) produce();
        const long long vb = v0 + (long long)i * RHO_ROWS;
        double wv[RHO_ROWS / RHO_WARPS];                            // the weights do not depend on the box: loaded before the wait
#pragma unroll
        for (int r = 0; r < RHO_ROWS / RHO_WARPS; r++) {
            const long long v = vb + w + r * RHO_WARPS;
            wv[r] = (v < v1) ? __ldg(P.Wv + v) : 0.0;               // rows past the chunk (zero-filled, or the next chunk's) count 0
        }
        mbar_wait(full_s + 8u * st, ph);
        typedef typename Pair<T>::type T2;
        const T2* box = reinterpret_cast<const T2*>(smem_raw + (size_t)st * P.slot_bytes) + lane;
        T2 val[RHO_ROWS / RHO_WARPS];
#pragma unroll
        for (int r = 0; r < RHO_ROWS / RHO_WARPS; r++) val[r] = box[(w + r * RHO_WARPS) * (RHO_WX / 2)];
        fence_async_smem();                                         // generic-proxy reads -> the slot's refill by the async proxy
        __syncwarp();
        if (lane == 0) mbar_arrive(empty_s + 8u * st);
#pragma unroll
        for (int r = 0; r < RHO_ROWS / RHO_WARPS; r += 2) {
            acc0[0] = fma(wv[r], (double)val[r].x, acc0[0]);         acc0[1] = fma(wv[r], (double)val[r].y, acc0[1]);
            acc1[0] = fma(wv[r + 1], (double)val[r + 1].x, acc1[0]); acc1[1] = fma(wv[r + 1], (double)val[r + 1].y, acc1[1]);
        }
        if (++st == ST) { st = 0; ph ^= 1u; }
    }
    __syncthreads();                                                // the ring is drained: reuse it for the warps' sums
    double* red = reinterpret_cast<double*>(smem_raw);
    red[w * RHO_WX + 2 * lane] = acc0[0] + acc1[0];
    red[w * RHO_WX + 2 * lane + 1] = acc0[1] + acc1[1];
    __syncthreads();
    if (w < 2) {                                                    // warp 0: x values 0..31 of the tile, warp 1: 32..63
        const int xi = w * 32 + lane;
        double s = 0.0;
#pragma unroll
        for (int u = 0; u < RHO_WARPS; u++) s += red[u * RHO_WX + xi];
        const long long x = (long long)tile * RHO_WX + xi;
        if (x < P.X) P.part[chunk * P.X + x] = s;
    }
}

__global__ void rho_final_kernel(const double* __restrict__ part, long long X, int nchunk, double* __restrict__ rho)
{
    long long x = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (x >= X) return;
    double acc = 0.0;
    for (int c = 0; c < nchunk; c++) acc += part[(long long)c * X + x];
    rho[x] = acc;
}

// ------------------------------------------------------------------ Poisson / E (row a4)
// out[q][m][p] = sum_n M[m][n] in[q][n][p], complex; M stored transposed MT[n][m] (re block, then im block).
// HAS_IM = 0: the input is real.
// A small complex GEMM per axis (D <= a few hundred): blocks of 16 x 16 outputs (m, column c = q * inner + p), the
// n loop staged through shared memory in chunks of 32 so that M and the input are read from L2 once per tile and not
// once per output.  Per output the sum runs over n in ascending order with the same fused multiply-adds as a plain
// loop, so results do not depend on the tiling.
template <int HAS_IM>
__global__ void __launch_bounds__(256) apply_axis_kernel(const double* __restrict__ inr, const double* __restrict__ ini,
                                                         const double* __restrict__ MT, long long D, long long inner,
                                                         long long total, double* __restrict__ outr,
                                                         double* __restrict__ outi)
{
    constexpr int TM = 16, TC = 16, KC = 32;
    __shared__ double sMr[KC][TM + 1], sMi[KC][TM + 1], sXr[KC][TC + 1], sXi[KC][TC + 1];
    const long long ncols = total / D;
    const int tc = threadIdx.x % TC, tm = threadIdx.x / TC;            // column fastest: coalesced when inner >= 16
    const long long c = (long long)blockIdx.x * TC + tc;
    const long long m = (long long)blockIdx.y * TM + tm;
    const bool colok = c < ncols, ok = colok && m < D;
    const long long q = colok ? c / inner : 0, pp = colok ? c - q * inner : 0;
    const long long xbase = q * D * inner + pp;
    double ar = 0.0, ai = 0.0;
    for (long long n0 = 0; n0 < D; n0 += KC) {
        // stage M[m-tile][n0..n0+KC) (stored transposed: MT[n][m]) and in[n0..n0+KC)[column tile]
        for (int e = threadIdx.x; e < KC * TM; e += 256) {
            const int kn = e / TM, km = e - kn * TM;
            const long long n = n0 + kn, mm = (long long)blockIdx.y * TM + km;
            const bool v = n < D && mm < D;
            sMr[kn][km] = v ? __ldg(MT + n * D + mm) : 0.0;
            sMi[kn][km] = v ? __ldg(MT + D * D + n * D + mm) : 0.0;
        }
        for (int e = threadIdx.x; e < KC * TC; e += 256) {
            const int kn = e / TC, kc = e - kn * TC;
            const long long n = n0 + kn, cc = (long long)blockIdx.x * TC + kc;
            double vr = 0.0, vi = 0.0;
            if (n < D && cc < ncols) {
                const long long qq = cc / inner, p2 = cc - qq * inner;
                vr = inr[qq * D * inner + n * inner + p2];
                if (HAS_IM) vi = ini[qq * D * inner + n * inner + p2];
            }
            sXr[kn][kc] = vr; sXi[kn][kc] = vi;
        }
        __syncthreads();
        const int kmax = (int)min((long long)KC, D - n0);
        for (int k = 0; k < kmax; k++) {
            const double mr = sMr[k][tm], mi = sMi[k][tm], vr = sXr[k][tc];
            ar = fma(mr, vr, ar); ai = fma(mi, vr, ai);
            if (HAS_IM) {
                const double vi = sXi[k][tc];
                ar = fma(-mi, vi, ar); ai = fma(mr, vi, ai);
            }
        }
        __syncthreads();
    }
    if (ok) {
        const long long o = xbase + m * inner;
        outr[o] = ar;
        if (outi) outi[o] = ai;
    }
}

// E^_d = i kappa_d rho^ / |kappa|^2 (kappa != 0), 0 at kappa = 0; kappa_d := 0 at the Nyquist index of an even axis.
struct SpecParams { int dx; long long D[3]; const double* kap[3]; long long X; };
__global__ void spectral_kernel(SpecParams P, int d, const double* __restrict__ rr, const double* __restrict__ ri,
                                double* __restrict__ er, double* __restrict__ ei)
{
    long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= P.X) return;
    long long r = t;
    double k2 = 0.0, kd = 0.0;
    for (int a = 0; a < P.dx; a++) {
        long long m = r % P.D[a]; r /= P.D[a];
        double kap = P.kap[a][m];
        k2 += kap * kap;
        if (a == d) kd = (2 * m == P.D[a]) ? 0.0 : kap;
    }
    if (k2 == 0.0) { er[t] = 0.0; ei[t] = 0.0; }
    else { er[t] = -kd * ri[t] / k2; ei[t] = kd * rr[t] / k2; }
}

// Small x grids (X <= 1024 nodes, e.g. BASELINE config 1: 256): the whole solve in ONE single-block launch with the
// six complex work arrays in shared memory, instead of 8 (dim_x = 2) or 15 (dim_x = 3) launches of a few microseconds
// each.  Every output is the same fma chain over n = 0..D-1 as in apply_axis_kernel and the same spectral formula, so
// the result is bit-identical to the multi-launch route.
struct SmallParams { int dx; long long D[3]; const double* kap[3]; const double* fwdT[3]; const double* invT[3]; long long X; };

template <bool HAS_IM, bool OUT_IM>
__device__ __forceinline__ void small_axis(const double* __restrict__ inr, const double* __restrict__ ini,
                                           const double* __restrict__ MT, long long D, long long inner, long long X,
                                           double* __restrict__ outr, double* __restrict__ outi)
{
    for (long long t = threadIdx.x; t < X; t += blockDim.x) {
        const long long pp = t % inner, m = (t / inner) % D, q = t / (inner * D);
        const long long base = q * D * inner + pp;
        double ar = 0.0, ai = 0.0;
        for (long long n = 0; n < D; n++) {
            const double mr = __ldg(MT + n * D + m), mi = __ldg(MT + D * D + n * D + m), vr = inr[base + n * inner];
            ar = fma(mr, vr, ar); ai = fma(mi, vr, ai);
            if (HAS_IM) {
                const double vi = ini[base + n * inner];
                ar = fma(-mi, vi, ar); ai = fma(mr, vi, ai);
            }
        }
        outr[t] = ar;
        if (OUT_IM) outi[t] = ai;
    }
    __syncthreads();
}

__global__ void __launch_bounds__(256) poisson_small_kernel(SmallParams P, const double* __restrict__ rho, double* __restrict__ E)
{
    extern __shared__ double sm_small[];
    const long long X = P.X;
    double *ar = sm_small, *ai = ar + X, *br = ai + X, *bi = br + X, *rr = bi + X, *ri = rr + X;
    // forward: transfer to the equidistant grid + DFT, axis by axis (as sldg_launch_poisson)
    const double* sr = rho; const double* si = nullptr;
    long long inner = 1;
    for (int a = 0; a < P.dx; a++) {
        const bool last = (a == P.dx - 1);
        double* dr = last ? rr : ((a & 1) ? br : ar);
        double* di = last ? ri : ((a & 1) ? bi : ai);
        if (si) small_axis<true, true>(sr, si, P.fwdT[a], P.D[a], inner, X, dr, di);
        else small_axis<false, true>(sr, si, P.fwdT[a], P.D[a], inner, X, dr, di);
        sr = dr; si = di; inner *= P.D[a];
    }
    for (int d = 0; d < P.dx; d++) {
        for (long long t = threadIdx.x; t < X; t += blockDim.x) {
            long long r = t;
            double k2 = 0.0, kd = 0.0;
            for (int a = 0; a < P.dx; a++) {
                long long m = r % P.D[a]; r /= P.D[a];
                double kap = P.kap[a][m];
                k2 += kap * kap;
                if (a == d) kd = (2 * m == P.D[a]) ? 0.0 : kap;
            }
            if (k2 == 0.0) { ar[t] = 0.0; ai[t] = 0.0; }
            else { ar[t] = -kd * ri[t] / k2; ai[t] = kd * rr[t] / k2; }
        }
        __syncthreads();
        double *pr = ar, *pi = ai, *qr = br, *qi = bi;
        inner = 1;
        for (int a = 0; a < P.dx; a++) {
            const bool last = (a == P.dx - 1);
            if (last) small_axis<true, false>(pr, pi, P.invT[a], P.D[a], inner, X, E + (long long)d * X, nullptr);
            else small_axis<true, true>(pr, pi, P.invT[a], P.D[a], inner, X, qr, qi);
            double* t2;
            t2 = pr; pr = qr; qr = t2;
            t2 = pi; pi = qi; qi = t2;
            inner *= P.D[a];
        }
    }
}

// ------------------------------------------------------------------ diagnostics
struct WgtParams { int nd; long long D[SLDG_MAX_DIM]; const double* w[SLDG_MAX_DIM]; long long total; };

__device__ __forceinline__ double block_sum(double v)
{
    __shared__ double sh[32];
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    int lane = threadIdx.x & 31, wid = threadIdx.x >> 5;
    if (lane == 0) sh[wid] = v;
    __syncthreads();
    if (wid == 0) {
        v = (lane < (blockDim.x >> 5)) ? sh[lane] : 0.0;
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    }
    return v;
}

// partial[b] = sum over a grid-stride slice of  W_n * g(n);  NCOMP = 0: g = f[n];  NCOMP > 0: g = sum_d E_d[n]^2
template <class T>
__global__ void __launch_bounds__(256) weighted_sum_kernel(WgtParams P, const T* __restrict__ a, int ncomp,
                                                           double* __restrict__ partial)
{
    double acc = 0.0;
    for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < P.total;
         t += (long long)gridDim.x * blockDim.x) {
        long long r = t;
        double wn = 1.0;
        for (int d = 0; d < P.nd; d++) { long long n = r % P.D[d]; r /= P.D[d]; wn *= P.w[d][n]; }
        double g;
        if (ncomp == 0) g = (double)a[t];
        else { g = 0.0; for (int d = 0; d < ncomp; d++) { double e = (double)a[(long long)d * P.total + t]; g = fma(e, e, g); } }
        acc = fma(wn, g, acc);
    }
    acc = block_sum(acc);
    if (threadIdx.x == 0) partial[blockIdx.x] = acc;
}
__global__ void __launch_bounds__(256) final_sum_kernel(const double* __restrict__ partial, int n, double scale,
                                                        double* __restrict__ out)
{
    double acc = 0.0;
    for (int t = threadIdx.x; t < n; t += blockDim.x) acc += partial[t];
    acc = block_sum(acc);
    if (threadIdx.x == 0) out[0] = acc * scale;
}

}  // namespace

template <class TAB>
static void vtable_dispatch(sldg_ctx* c, const double* Ed, double tau, double hv, int N, int* S, TAB* AB)
{
    int block = 128;
    unsigned grid = (unsigned)((c->X + block - 1) / block);
    switch (c->K1) {
    case 1: vtable_kernel<1, TAB><<<grid, block, 0, c->stream>>>(c->dPoly, Ed, tau, hv, N, c->X, S, AB); break;
    case 2: vtable_kernel<2, TAB><<<grid, block, 0, c->stream>>>(c->dPoly, Ed, tau, hv, N, c->X, S, AB); break;
    case 3: vtable_kernel<3, TAB><<<grid, block, 0, c->stream>>>(c->dPoly, Ed, tau, hv, N, c->X, S, AB); break;
    case 4: vtable_kernel<4, TAB><<<grid, block, 0, c->stream>>>(c->dPoly, Ed, tau, hv, N, c->X, S, AB); break;
    case 5: vtable_kernel<5, TAB><<<grid, block, 0, c->stream>>>(c->dPoly, Ed, tau, hv, N, c->X, S, AB); break;
    }
}

// A, B are evaluated in fp64 and stored in the sweep's type (float in single precision mode, reading W)
cudaError_t sldg_launch_vtable(sldg_ctx* c, const double* Ed, double tau, double hv, int N, int* S, double* AB)
{
    if (c->prec == SLDG_F32) vtable_dispatch<float>(c, Ed, tau, hv, N, S, reinterpret_cast<float*>(AB));
    else vtable_dispatch<double>(c, Ed, tau, hv, N, S, AB);
    return cudaGetLastError();
}

cudaError_t sldg_launch_wv(sldg_ctx* c)
{
    WvParams P;
    P.dv = c->dv; P.V = c->V;
    for (int a = 0; a < c->dv; a++) { P.Dv[a] = c->D[c->dx + a]; P.w[a] = c->dWx[c->dx + a]; }
    int block = 256;
    wv_kernel<<<(unsigned)((c->V + block - 1) / block), block, 0, c->stream>>>(P, c->Wv);
    return cudaGetLastError();
}

// rho through the TMA kernel when the problem is large enough to fill the GPU with x tiles x v chunks; cudaErrorNotSupported otherwise
static cudaError_t density_tma(sldg_ctx* c, const double* f, double* rho)
{
    const long long X = c->X, V = c->V;
    const size_t es = c->esize;
    if (!c->opt_rho_tma || ((X * (long long)es) & 15) || (((uintptr_t)f) & 15) || X < RHO_WX || V < 4 * RHO_ROWS) return cudaErrorNotSupported;
    if (X >= (1LL << 31) || V >= (1LL << 31)) return cudaErrorNotSupported;
    SldgEncodeTiled enc = sldg_encode_tiled();
    if (!enc) return cudaErrorNotSupported;
    RhoTmaParams P;
    P.Wv = c->Wv; P.part = c->part; P.X = X; P.V = V;
    P.ntiles = (int)((X + RHO_WX - 1) / RHO_WX);
    // chunks of whole boxes: about 20 waves of blocks (two are resident per SM), so that the last, partial wave does not show
    // (measured on cfg4: 1000 blocks = 3.4 waves ran 8 % slower than the plain-load kernel); no more than the partial-sum buffer holds
    long long nchunk = ((long long)c->sm_count * 40 + P.ntiles - 1) / P.ntiles;
    const long long nbox = (V + RHO_ROWS - 1) / RHO_ROWS;
    if (nchunk > nbox / 4) nchunk = nbox / 4;
    if (nchunk > c->part_cap / X) nchunk = c->part_cap / X;
    if (nchunk < 1) nchunk = 1;
    long long bpc = (nbox + nchunk - 1) / nchunk;                       // boxes per chunk
    P.vchunk = bpc * RHO_ROWS;
    nchunk = (V + P.vchunk - 1) / P.vchunk;
    if ((long long)P.ntiles * nchunk < 2LL * c->sm_count) return cudaErrorNotSupported;
    P.slot_bytes = (uint32_t)(RHO_ROWS * RHO_WX * es);
    P.slots = 6;
    const size_t smem = (size_t)P.slots * P.slot_bytes + 16 * (size_t)P.slots + 64;
    CUtensorMap tm;
    const cuuint64_t gdim[2] = {(cuuint64_t)X, (cuuint64_t)V};
    const cuuint64_t gstr[1] = {(cuuint64_t)X * es};
    const cuuint32_t box[2] = {(cuuint32_t)RHO_WX, (cuuint32_t)RHO_ROWS};
    const cuuint32_t estr[2] = {1u, 1u};
    if (enc(&tm, es == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<double*>(f), gdim, gstr, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return cudaErrorNotSupported;
    const unsigned grid = (unsigned)((long long)P.ntiles * nchunk);
    cudaError_t e;
    if (es == 8) {
        e = cudaFuncSetAttribute(rho_tma_kernel<double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        rho_tma_kernel<double><<<grid, RHO_WARPS * 32, smem, c->stream>>>(tm, P);
    } else {
        e = cudaFuncSetAttribute(rho_tma_kernel<float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        rho_tma_kernel<float><<<grid, RHO_WARPS * 32, smem, c->stream>>>(tm, P);
    }
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    rho_final_kernel<<<(unsigned)((X + 255) / 256), 256, 0, c->stream>>>(c->part, X, (int)nchunk, rho);
    c->launches += 2;
    return cudaGetLastError();
}

cudaError_t sldg_launch_density(sldg_ctx* c, const double* f, double* rho)
{
    {
        const cudaError_t et = density_tma(c, f, rho);
        if (et != cudaErrorNotSupported) return et;
    }
    const long long X = c->X, V = c->V;
    const bool f32 = c->prec == SLDG_F32;
    int vec = ((X & 1) == 0 && (((uintptr_t)f) & (f32 ? 7 : 15)) == 0) ? 2 : 1;
    if (c->opt_rho_vec == 1) vec = 1;
    long long xtiles = (X + 128LL * vec - 1) / (128LL * vec);
    // ONE wave of equal blocks: at most opt_rho_blocks (8) blocks per SM, rounded DOWN so that no second, partial
    // wave forms (measured on B200: 1.2x between a grid of 1.03 waves and one of 0.5 or 4.0 waves)
    long long want = (long long)c->sm_count * c->opt_rho_blocks;
    long long nchunk = want / xtiles;
    if (nchunk > V / 16) nchunk = V / 16;
    if (nchunk > c->part_cap / X) nchunk = c->part_cap / X;
    if (nchunk > 65535) nchunk = 65535;
    if (nchunk < 1) nchunk = 1;
    long long vchunk = (V + nchunk - 1) / nchunk;
    nchunk = (V + vchunk - 1) / vchunk;
    dim3 grid((unsigned)xtiles, (unsigned)nchunk);
    const float* f4 = reinterpret_cast<const float*>(f);
    if (f32 && vec == 2) rho_partial_kernel<2, float><<<grid, 128, 0, c->stream>>>(f4, c->Wv, X, V, vchunk, c->part);
    else if (f32) rho_partial_kernel<1, float><<<grid, 128, 0, c->stream>>>(f4, c->Wv, X, V, vchunk, c->part);
    else if (vec == 2) rho_partial_kernel<2, double><<<grid, 128, 0, c->stream>>>(f, c->Wv, X, V, vchunk, c->part);
    else rho_partial_kernel<1, double><<<grid, 128, 0, c->stream>>>(f, c->Wv, X, V, vchunk, c->part);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    rho_final_kernel<<<(unsigned)((X + 255) / 256), 256, 0, c->stream>>>(c->part, X, (int)nchunk, rho);
    c->launches += 2;
    return cudaGetLastError();
}

cudaError_t sldg_launch_poisson(sldg_ctx* c, const double* rho, double* E)
{
    const long long X = c->X;
    if (X <= 1024 && c->opt_poisson_small) {
        SmallParams S;
        S.dx = c->dx; S.X = X;
        for (int a = 0; a < c->dx; a++) { S.D[a] = c->D[a]; S.kap[a] = c->dKap[a]; S.fwdT[a] = c->dFwdT[a]; S.invT[a] = c->dInvT[a]; }
        poisson_small_kernel<<<1, 256, (size_t)(6 * X * sizeof(double)), c->stream>>>(S, rho, E);
        c->launches++;
        return cudaGetLastError();
    }
    const int block = 128;
    const unsigned grid = (unsigned)((X + block - 1) / block);
    double *ar = c->cplx[0], *ai = c->cplx[1], *br = c->cplx[2], *bi = c->cplx[3], *rr = c->cplx[4], *ri = c->cplx[5];
    // forward: transfer to the equidistant grid + DFT, axis by axis
    const double* sr = rho; const double* si = nullptr;
    long long inner = 1;
    for (int a = 0; a < c->dx; a++) {
        bool last = (a == c->dx - 1);
        double* dr = last ? rr : ((a & 1) ? br : ar);
        double* di = last ? ri : ((a & 1) ? bi : ai);
        const dim3 ag((unsigned)((X / c->D[a] + 15) / 16), (unsigned)((c->D[a] + 15) / 16));
        if (si) apply_axis_kernel<1><<<ag, 256, 0, c->stream>>>(sr, si, c->dFwdT[a], c->D[a], inner, X, dr, di);
        else apply_axis_kernel<0><<<ag, 256, 0, c->stream>>>(sr, si, c->dFwdT[a], c->D[a], inner, X, dr, di);
        c->launches++;
        sr = dr; si = di; inner *= c->D[a];
    }
    SpecParams S;
    S.dx = c->dx; S.X = X;
    for (int a = 0; a < c->dx; a++) { S.D[a] = c->D[a]; S.kap[a] = c->dKap[a]; }
    for (int d = 0; d < c->dx; d++) {
        spectral_kernel<<<grid, block, 0, c->stream>>>(S, d, rr, ri, ar, ai);
        c->launches++;
        double *pr = ar, *pi = ai, *qr = br, *qi = bi;
        inner = 1;
        for (int a = 0; a < c->dx; a++) {
            bool last = (a == c->dx - 1);
            const dim3 ag((unsigned)((X / c->D[a] + 15) / 16), (unsigned)((c->D[a] + 15) / 16));
            apply_axis_kernel<1><<<ag, 256, 0, c->stream>>>(pr, pi, c->dInvT[a], c->D[a], inner, X,
                                                                last ? E + (long long)d * X : qr, last ? nullptr : qi);
            c->launches++;
            double* t;
            t = pr; pr = qr; qr = t;
            t = pi; pi = qi; qi = t;
            inner *= c->D[a];
        }
    }
    return cudaGetLastError();
}

template <class T>
static cudaError_t weighted_sum(sldg_ctx* c, const T* a, int nd, int axis0, int ncomp, long long total,
                                double scale, double* out1)
{
    WgtParams P;
    P.nd = nd; P.total = total;
    for (int d = 0; d < nd; d++) { P.D[d] = c->D[axis0 + d]; P.w[d] = c->dWx[axis0 + d]; }
    long long nb = (total + 255) / 256;
    if (nb > 2048) nb = 2048;
    weighted_sum_kernel<T><<<(unsigned)nb, 256, 0, c->stream>>>(P, a, ncomp, c->red);
    final_sum_kernel<<<1, 256, 0, c->stream>>>(c->red, (int)nb, scale, out1);
    c->launches += 2;
    return cudaGetLastError();
}

cudaError_t sldg_launch_energy(sldg_ctx* c, const double* E, double* out1)
{
    return weighted_sum(c, E, c->dx, 0, c->dx, c->X, 0.5, out1);
}

cudaError_t sldg_launch_mass(sldg_ctx* c, const double* f, double* out1)
{
    if (c->prec == SLDG_F32) return weighted_sum(c, reinterpret_cast<const float*>(f), c->d, 0, 0, c->nf, 1.0, out1);
    return weighted_sum(c, f, c->d, 0, 0, c->nf, 1.0, out1);
}
