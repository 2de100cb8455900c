// sldg_sweep_fused.cu -- the x_1 and x_2 sweeps of an x advection in ONE pass over f, sm_100a.
//
// eq. (3), reading B, applied twice:  first along x_1 (axis 0, contiguous), then along x_2 (axis 1).
// The x sweeps commute and act on different axes, so both can be applied while a value passes through the
// SM once: 16 B of HBM traffic per value for TWO sweeps (two separate passes move 32 B).
//
// The array is seen as [planes q][D_1 rows][D_0] with a row = one contiguous x_1 line.  A block owns PB planes
// and has one thread per (plane, x_1 node).  Every thread WALKS along x_2 exactly like sldg_sweep_walk.cu (cell j
// in registers, cell j+1 loaded U cells ahead, output cell (j + s_2 + 1) mod N_1 written, first cell kept for the
// periodic wrap), but the values that enter the walk are x_1-swept first: the freshly loaded rows are exchanged
// through shared memory (one row = one x_1 line, so both x_1 donor cells of every node are in the same row) and
// each thread combines its 2(k+1) donor values with its row of A_1, B_1.  The loads of chunk c+1 are issued before
// chunk c is computed (register double buffering), shared memory is double buffered: one __syncthreads per chunk.
// Every value is read once and written once; the shift of x_1 depends on the plane's v_1 node, that of x_2 on
// its v_2 node (one (s, A, B) each per thread).  Out of place only (fin != fout).
#include "sldg_internal.h"

namespace {

#ifndef SLDG_FUSED_U2
#define SLDG_FUSED_U2 4
#endif
#ifndef SLDG_FUSED_U3
#define SLDG_FUSED_U3 4
#endif
template <int K1> struct FUnroll {
    static constexpr int U = (K1 == 1) ? 8 : (K1 == 2) ? SLDG_FUSED_U2 : (K1 == 3) ? SLDG_FUSED_U3 : 2;
};

struct FusedParams {
    const double* fin;
    double* fout;
    long long planes;             // prod of D_b, b >= 2
    int N0, N1, PB;               // cells along x_1, x_2; planes per block
    long long sdiv0, sdiv1;       // shift index of plane q: (q / sdiv) % smod, per axis
    long long smod0, smod1;
    ShiftTable t0, t1;
};

template <int K1>
__global__ void __launch_bounds__(256) sweep_fused_kernel(const FusedParams P)
{
    constexpr int U = FUnroll<K1>::U;
    constexpr int NN = K1 * K1;
    constexpr int ROWS = U * K1;                      // rows exchanged per chunk
    extern __shared__ __align__(16) double sm[];      // [2][ROWS][PB * D0]
    const int N0 = P.N0, N1 = P.N1, D0 = N0 * K1;
    const int W = P.PB * D0;                          // threads that own a node (== blockDim.x)
    const int t = threadIdx.x;
    const int pl = t / D0, n0 = t - pl * D0;
    const long long q = (long long)blockIdx.x * P.PB + pl;
    const bool live = q < P.planes;
    const long long qq = live ? q : P.planes - 1;     // dead threads shadow the last plane (no loads, no stores)

    // ---- x_1: this thread's row of A_1, B_1 and the offsets of its two donor cells inside a row
    double a1[K1], b1[K1];
    int da, db;
    bool cp1;
    {
        const long long idx = (qq / P.sdiv0) % P.smod0;
        const int sv = __ldg(P.t0.S + idx);
        cp1 = (sv & SLDG_COPY_BIT) != 0;
        const int s = sv & SLDG_S_MASK;
        const int cell = n0 / K1, jj = n0 - cell * K1;
        int ia = cell - s; if (ia < 0) ia += N0;
        int ib = ia - 1; if (ib < 0) ib += N0;
        da = pl * D0 + ia * K1; db = pl * D0 + ib * K1;
        const double* ab = static_cast<const double*>(P.t0.AB) + idx * P.t0.strideIdx;
#pragma unroll
        for (int m = 0; m < K1; m++) {
            a1[m] = __ldg(ab + (jj * K1 + m) * P.t0.strideM);
            b1[m] = __ldg(ab + (NN + jj * K1 + m) * P.t0.strideM);
        }
        if (cp1) da += jj;                            // copy: the donor VALUE itself
    }
    // ---- x_2: full A_2, B_2
    double A[NN], B[NN];
    int s2;
    bool cp2;
    {
        const long long idx = (qq / P.sdiv1) % P.smod1;
        const int sv = __ldg(P.t1.S + idx);
        cp2 = (sv & SLDG_COPY_BIT) != 0;
        s2 = sv & SLDG_S_MASK;
        const double* ab = static_cast<const double*>(P.t1.AB) + idx * P.t1.strideIdx;
#pragma unroll
        for (int m = 0; m < NN; m++) {
            A[m] = __ldg(ab + m * P.t1.strideM);
            B[m] = __ldg(ab + (NN + m) * P.t1.strideM);
        }
    }

    const long long base = qq * (long long)N1 * K1 * D0 + n0;
    const double* in = P.fin + base;
    double* out = P.fout + base;

    // x_1-swept value of this thread's node in exchanged row r of buffer `buf`
    auto swept = [&](const double* buf, int r) {
        const double* row = buf + r * W;
        if (cp1) return row[da];
        double acc = 0.0;
#pragma unroll
        for (int m = 0; m < K1; m++) acc += a1[m] * row[da + m];
#pragma unroll
        for (int m = 0; m < K1; m++) acc += b1[m] * row[db + m];
        return acc;
    };

    double* const buf0 = sm;
    double* const buf1 = sm + ROWS * W;
    double first[K1], prev[K1], raw[U][K1];

    // loads of cells c0+1 .. c0+U (those that exist) into raw
    auto load_chunk = [&](int c0) {
#pragma unroll
        for (int u = 0; u < U; u++) {
            const int c = c0 + 1 + u;
            if (c < N1 && live) {
#pragma unroll
                for (int j = 0; j < K1; j++) raw[u][j] = __ldcs(in + ((long long)c * K1 + j) * D0);
            }
        }
    };

    // round 0: cell 0 alone
#pragma unroll
    for (int j = 0; j < K1; j++) buf0[j * W + t] = live ? __ldcs(in + (long long)j * D0) : 0.0;
    __syncthreads();
    load_chunk(0);
#pragma unroll
    for (int j = 0; j < K1; j++) { first[j] = swept(buf0, j); prev[j] = first[j]; }

    int io = s2 + 1; if (io >= N1) io -= N1;          // output cell of the current donor pair
    int b = 1;
    for (int jc = 0; jc < N1; jc += U) {
        double* const buf = b ? buf1 : buf0;
#pragma unroll
        for (int u = 0; u < U; u++) {
            if (jc + 1 + u < N1) {
#pragma unroll
                for (int j = 0; j < K1; j++) buf[(u * K1 + j) * W + t] = raw[u][j];
            }
        }
        __syncthreads();
        load_chunk(jc + U);                           // next chunk's loads fly while this one is computed
#pragma unroll
        for (int u = 0; u < U; u++) {
            if (jc + u < N1) {
                double nxt[K1], r[K1];
                if (jc + 1 + u < N1) {
#pragma unroll
                    for (int j = 0; j < K1; j++) nxt[j] = swept(buf, u * K1 + j);
                } else {
#pragma unroll
                    for (int j = 0; j < K1; j++) nxt[j] = first[j];
                }
#pragma unroll
                for (int j = 0; j < K1; j++) {
                    double acc = 0.0;
#pragma unroll
                    for (int l = 0; l < K1; l++) acc += A[j * K1 + l] * nxt[l];
#pragma unroll
                    for (int l = 0; l < K1; l++) acc += B[j * K1 + l] * prev[l];
                    r[j] = cp2 ? nxt[j] : acc;
                }
                if (live) {
#pragma unroll
                    for (int j = 0; j < K1; j++) __stcs(out + ((long long)io * K1 + j) * D0, r[j]);
                }
                io++; if (io >= N1) io = 0;
#pragma unroll
                for (int j = 0; j < K1; j++) prev[j] = nxt[j];
            }
        }
        b ^= 1;
    }
}

template <int K1>
cudaError_t launch(sldg_ctx* c, const FusedParams& P, int threads, size_t smem)
{
    auto kern = sweep_fused_kernel<K1>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const long long grid = (P.planes + P.PB - 1) / P.PB;
    if (grid > 0x7fffffffLL) return cudaErrorNotSupported;
    kern<<<(unsigned)grid, threads, smem, c->stream>>>(P);
    return cudaGetLastError();
}

}  // namespace

// g0, g1: geometry of axis 0 and axis 1 (SweepGeom of sldg_api.cu).  Returns cudaErrorNotSupported when the
// shape does not fit (caller runs the two sweeps separately).
cudaError_t sldg_launch_sweep_fused(sldg_ctx* c, const double* fin, double* fout, const SweepGeom& g0,
                                    const SweepGeom& g1, const ShiftTable& t0, const ShiftTable& t1)
{
    if (g1.outer == 0) return cudaSuccess;
    const long long D0 = (long long)g0.N * g0.K1, D1 = (long long)g1.N * g1.K1;
    if (fin == fout || g1.inner != D0 || g0.mode != 0 || g1.mode != 0) return cudaErrorNotSupported;
    if (D0 > c->opt_fused_threads || g0.sdiv % D1 != 0) return cudaErrorNotSupported;
    FusedParams P;
    P.fin = fin; P.fout = fout; P.planes = g1.outer;
    P.N0 = g0.N; P.N1 = g1.N;
    long long PB = c->opt_fused_threads / D0;
    if (PB < 1) PB = 1;
    if (PB > P.planes) PB = P.planes;
    P.PB = (int)PB;
    P.sdiv0 = g0.sdiv / D1; P.smod0 = g0.smod;       // axis-0 lines are numbered row + D_1 * plane
    P.sdiv1 = g1.sdiv; P.smod1 = g1.smod;
    P.t0 = t0; P.t1 = t1;
    const int threads = (int)(PB * D0);
    int U;
    switch (g0.K1) { case 1: U = FUnroll<1>::U; break; case 2: U = FUnroll<2>::U; break; case 3: U = FUnroll<3>::U; break;
                     case 4: U = FUnroll<4>::U; break; default: U = FUnroll<5>::U; }
    const size_t smem = (size_t)2 * U * g0.K1 * threads * 8;
    if (smem > 227 * 1024) return cudaErrorNotSupported;
    switch (g0.K1) {
    case 1: return launch<1>(c, P, threads, smem);
    case 2: return launch<2>(c, P, threads, smem);
    case 3: return launch<3>(c, P, threads, smem);
    case 4: return launch<4>(c, P, threads, smem);
    case 5: return launch<5>(c, P, threads, smem);
    }
    return cudaErrorInvalidValue;
}
