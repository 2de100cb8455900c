// sldg_sweep_tma.cu -- 1-D SLDG sweep along the FASTEST axis (inner == 1), sm_100a.
//
// eq. (3), reading B:   u_i <- A(alpha) u_{(i-s) mod N} + B(alpha) u_{(i-s-1) mod N}.
//
// Lines along axis 0 are contiguous (D_0 = N (k+1) values) and stacked contiguously, so a tile of L whole
// lines is one contiguous chunk.  A CTA brings its tile into shared memory with ONE 1-D TMA bulk copy
// (cp.async.bulk ... mbarrier::complete_tx), every thread computes output cells from shared memory (both
// donor cells come from SMEM, nothing is re-read from HBM), results go to a second SMEM buffer and leave
// with ONE TMA bulk store.  Because a tile holds whole lines and is fully resident before anything is
// written, the sweep may run IN PLACE (fin == fout).  Tiles whose address or size is not a multiple of 16 B
// (odd D_0 only) take a plain ld/st path inside the same kernel.
#include "sldg_internal.h"

namespace {

struct TmaParams {
    const double* fin;
    double* fout;
    long long nlines;
    int N, L;              // cells per line, lines per tile
    long long sdiv, smod;  // shift index of line q: (q / sdiv) % smod
    ShiftTable t;
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t* bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t phase)
{
    uint32_t ok;
    do {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(ok) : "r"(smem_u32(bar)), "r"(phase) : "memory");
    } while (!ok);
}
__device__ __forceinline__ void tma_load_1d(void* smem_dst, const void* gsrc, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_u32(smem_dst)), "l"(gsrc), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void tma_store_1d(void* gdst, const void* smem_src, uint32_t bytes)
{
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
                 ::"l"(gdst), "r"(smem_u32(smem_src)), "r"(bytes) : "memory");
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
}
__device__ __forceinline__ void tma_store_wait_read()
{
    asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
}

template <int K1>
__global__ void __launch_bounds__(256) sweep_tma_kernel(const TmaParams P)
{
    constexpr int NN = K1 * K1;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int N = P.N, D0 = N * K1;
    const long long q0 = (long long)blockIdx.x * P.L;
    const int nl = (int)min((long long)P.L, P.nlines - q0);
    const int nval = nl * D0;
    const uint32_t bytes = (uint32_t)nval * 8u;
    const int cap = P.L * D0;
    double* sin_ = reinterpret_cast<double*>(smem_raw);
    double* sout = sin_ + ((cap + 1) & ~1);
    uint64_t* bar = reinterpret_cast<uint64_t*>(sout + ((cap + 1) & ~1));
    const double* gin = P.fin + q0 * D0;
    double* gout = P.fout + q0 * D0;
    const bool tma = ((bytes & 15u) == 0) && ((((uintptr_t)gin) | ((uintptr_t)gout)) & 15) == 0;

    if (tma) {
        if (threadIdx.x == 0) {
            mbar_init(bar, 1);
            asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
            mbar_expect_tx(bar, bytes);
            tma_load_1d(sin_, gin, bytes, bar);
        }
        __syncthreads();               // barrier init visible to all waiters
        mbar_wait(bar, 0);
    } else {
        for (int t = threadIdx.x; t < nval; t += blockDim.x) sin_[t] = gin[t];
        __syncthreads();
    }

    double A[NN], B[NN];
    long long cur = -1;
    int s = 0;
    bool cp = false;
    const int ncell = nl * N;
    for (int c = threadIdx.x; c < ncell; c += blockDim.x) {
        int l = c / N, i = c - l * N;
        long long idx = ((q0 + l) / P.sdiv) % P.smod;
        if (idx != cur) {
            cur = idx;
            int sv = __ldg(P.t.S + idx);
            cp = (sv & SLDG_COPY_BIT) != 0;
            s = sv & SLDG_S_MASK;
            const double* ab = static_cast<const double*>(P.t.AB) + idx * P.t.strideIdx;
#pragma unroll
            for (int m = 0; m < NN; m++) {
                A[m] = __ldg(ab + m * P.t.strideM);
                B[m] = __ldg(ab + (NN + m) * P.t.strideM);
            }
        }
        int ia = i - s; if (ia < 0) ia += N;
        int ib = ia - 1; if (ib < 0) ib += N;
        const double* ua = sin_ + (l * N + ia) * K1;
        const double* ub = sin_ + (l * N + ib) * K1;
        double a[K1], b[K1];
        if (K1 == 2) {
            double2 ta = *reinterpret_cast<const double2*>(ua), tb = *reinterpret_cast<const double2*>(ub);
            a[0] = ta.x; a[K1 - 1] = ta.y; b[0] = tb.x; b[K1 - 1] = tb.y;
        } else {
#pragma unroll
            for (int j = 0; j < K1; j++) { a[j] = ua[j]; b[j] = ub[j]; }
        }
        double r[K1];
#pragma unroll
        for (int j = 0; j < K1; j++) {
            double acc = 0.0;
#pragma unroll
            for (int m = 0; m < K1; m++) acc += A[j * K1 + m] * a[m];
#pragma unroll
            for (int m = 0; m < K1; m++) acc += B[j * K1 + m] * b[m];
            r[j] = cp ? a[j] : acc;
        }
        double* uo = sout + c * K1;
        if (K1 == 2) {
            *reinterpret_cast<double2*>(uo) = make_double2(r[0], r[K1 - 1]);
        } else {
#pragma unroll
            for (int j = 0; j < K1; j++) uo[j] = r[j];
        }
    }

    if (tma) {
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic-proxy writes -> async proxy
        __syncthreads();
        if (threadIdx.x == 0) {
            tma_store_1d(gout, sout, bytes);
            tma_store_wait_read();
        }
    } else {
        __syncthreads();
        for (int t = threadIdx.x; t < nval; t += blockDim.x) gout[t] = sout[t];
    }
}

template <int K1>
cudaError_t launch(sldg_ctx* c, const TmaParams& P, int D0)
{
    long long grid = (P.nlines + P.L - 1) / P.L;
    if (grid > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    int cap = (P.L * D0 + 1) & ~1;
    size_t smem = (size_t)cap * 16 + 16;
    if (smem > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(sweep_tma_kernel<K1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    sweep_tma_kernel<K1><<<(unsigned)grid, 256, smem, c->stream>>>(P);
    return cudaGetLastError();
}

}  // namespace

cudaError_t sldg_launch_sweep_tma(sldg_ctx* c, const double* fin, double* fout, const SweepGeom& g,
                                  const ShiftTable& t)
{
    TmaParams P;
    P.fin = fin; P.fout = fout;
    P.nlines = g.outer; P.N = g.N;
    P.sdiv = g.sdiv; P.smod = g.smod; P.t = t;
    if (g.outer == 0) return cudaSuccess;
    int D0 = g.N * g.K1;
    long long line_bytes = (long long)D0 * 8;
    if (2 * line_bytes + 64 > 200 * 1024) return cudaErrorInvalidConfiguration;   // one line must fit twice
    long long L = c->opt_tile_bytes / line_bytes;
    if (L < 1) L = 1;
    if (L > 1) L &= ~1LL;                     // even: keeps tile starts 16-byte aligned for odd D_0
    while (2 * L * line_bytes + 64 > 200 * 1024 && L > 1) L >>= 1;
    if (L > g.outer) L = g.outer;
    P.L = (int)L;
    switch (g.K1) {
    case 1: return launch<1>(c, P, D0);
    case 2: return launch<2>(c, P, D0);
    case 3: return launch<3>(c, P, D0);
    case 4: return launch<4>(c, P, D0);
    case 5: return launch<5>(c, P, D0);
    }
    return cudaErrorInvalidValue;
}
