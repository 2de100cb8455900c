// sldg_sweep_walk.cu -- 1-D SLDG sweep along a SLOW axis (inner > 1), sm_100a.
//
// eq. (3), reading B:   u_i <- A(alpha) u_{(i-s) mod N} + B(alpha) u_{(i-s-1) mod N}.
//
// The array is seen as [outer][D_a = N (k+1)][inner] with `inner` contiguous.  Threads are spread over the
// flattened (inner / VEC, outer) index, so a warp reads 32*VEC consecutive values of one row: coalesced,
// 128-bit when VEC == 2.  Each thread WALKS its line along the donor index j: it keeps cell j in registers,
// loads cell j+1 (U cells ahead, all loads issued before the first use), and writes output cell
// (j + s + 1) mod N = A u_{j+1} + B u_j.  The first cell is kept to close the periodic wrap, so every value
// is read exactly once and written exactly once (16 B per value, the algorithmic minimum).
#include "sldg_internal.h"
#include "sldg_real.h"

namespace {

struct WalkParams {
    const real* fin;
    real* fout;
    long long innerV, inner, nwork;
    int N;
    long long sdiv, smod;
    ShiftTable t;
};

template <int VEC> struct Vec;
template <> struct Vec<1> {
    real v[1];
    __device__ __forceinline__ void load(const real* p) { v[0] = __ldcs(p); }
    __device__ __forceinline__ void store(real* p) const { __stcs(p, v[0]); }
};
template <> struct Vec<2> {
    real v[2];
    __device__ __forceinline__ void load(const real* p)
    {
        real2 t = __ldcs(reinterpret_cast<const real2*>(p));
        v[0] = t.x; v[1] = t.y;
    }
    __device__ __forceinline__ void store(real* p) const
    {
        __stcs(reinterpret_cast<real2*>(p), make_real2(v[0], v[1]));
    }
};

// cells loaded ahead of the one being computed (loads in flight per thread = U * K1 * VEC values)
template <int K1> struct Unroll {
#ifdef SLDG_REAL_FLOAT
    static constexpr int U = (K1 == 3) ? 8 : 4;            // measured: cfg2 (k=2) prefers 8 cells in flight, cfg4 (k=1) 4
#else
    static constexpr int U = (K1 == 1) ? 8 : (K1 <= 4) ? 4 : 2;             // measured on B200 (cfg2-5)
#endif
};

// MODE 0: one shift per thread (x-sweep, shift indexed by a digit of the outer index)
// MODE 1: one shift per VALUE (v-sweep, shift indexed by the x node = inner index mod X)
template <int K1, int VEC, int MODE>
__global__ void __launch_bounds__(256) sweep_walk_kernel(const WalkParams P)
{
    constexpr int NS = (MODE == 1) ? VEC : 1;
    constexpr int U = Unroll<K1>::U;
    constexpr int NN = K1 * K1;
    long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= P.nwork) return;
    long long q, p;
    if (P.nwork < (1LL << 31)) {           // 32-bit divide when it fits
        unsigned gg = (unsigned)g, iv = (unsigned)P.innerV;
        unsigned qq = gg / iv;
        q = qq; p = (long long)(gg - qq * iv) * VEC;
    } else {
        q = g / P.innerV; p = (g - q * P.innerV) * VEC;
    }

    real A[NS][NN], B[NS][NN];
    int s[NS];
    bool cp[NS];
#pragma unroll
    for (int e = 0; e < NS; e++) {
        long long idx = (MODE == 0) ? (q / P.sdiv) % P.smod : (p + e) % P.smod;
        int sv = __ldg(P.t.S + idx);
        cp[e] = (sv & SLDG_COPY_BIT) != 0;
        s[e] = sv & SLDG_S_MASK;
        const real* ab = static_cast<const real*>(P.t.AB) + idx * P.t.strideIdx;
#pragma unroll
        for (int m = 0; m < NN; m++) {
            A[e][m] = __ldg(ab + m * P.t.strideM);
            B[e][m] = __ldg(ab + (NN + m) * P.t.strideM);
        }
    }

    const int N = P.N;
    const long long rs = P.inner;                       // row stride (elements)
    const long long base = q * (long long)N * K1 * rs + p;
    const real* in = P.fin + base;
    real* out = P.fout + base;

    Vec<VEC> first[K1], prev[K1], nxt[U][K1];
#pragma unroll
    for (int j = 0; j < K1; j++) { first[j].load(in + j * rs); prev[j] = first[j]; }

    int io[NS];                                         // output cell of the current donor pair
#pragma unroll
    for (int e = 0; e < NS; e++) { io[e] = s[e] + 1; if (io[e] >= N) io[e] -= N; }

    for (int jc = 0; jc < N; jc += U) {
        // issue all loads of this chunk first (cells jc+1 .. jc+U)
#pragma unroll
        for (int u = 0; u < U; u++) {
            int c = jc + 1 + u;
            if (c < N) {
#pragma unroll
                for (int j = 0; j < K1; j++) nxt[u][j].load(in + ((long long)c * K1 + j) * rs);
            } else if (c == N) {
#pragma unroll
                for (int j = 0; j < K1; j++) nxt[u][j] = first[j];
            }
        }
#pragma unroll
        for (int u = 0; u < U; u++) {
            if (jc + u < N) {
                Vec<VEC> r[K1];
#pragma unroll
                for (int e = 0; e < VEC; e++) {
                    const int es = (NS == 1) ? 0 : e;
#pragma unroll
                    for (int j = 0; j < K1; j++) {
                        real acc = 0;
#pragma unroll
                        for (int l = 0; l < K1; l++) acc += A[es][j * K1 + l] * nxt[u][l].v[e];
#pragma unroll
                        for (int l = 0; l < K1; l++) acc += B[es][j * K1 + l] * prev[l].v[e];
                        r[j].v[e] = cp[es] ? nxt[u][j].v[e] : acc;
                    }
                }
                bool same = true;
                if (NS == 2) same = (io[0] == io[NS - 1]);
                if (same) {
#pragma unroll
                    for (int j = 0; j < K1; j++) r[j].store(out + ((long long)io[0] * K1 + j) * rs);
                } else {
#pragma unroll
                    for (int e = 0; e < VEC; e++)
#pragma unroll
                        for (int j = 0; j < K1; j++)
                            __stcs(out + ((long long)io[(NS == 1) ? 0 : e] * K1 + j) * rs + e, r[j].v[e]);
                }
#pragma unroll
                for (int e = 0; e < NS; e++) { io[e]++; if (io[e] >= N) io[e] = 0; }
#pragma unroll
                for (int j = 0; j < K1; j++) prev[j] = nxt[u][j];
            }
        }
    }
}

template <int K1, int VEC, int MODE>
cudaError_t launch(sldg_ctx* c, const WalkParams& P)
{
    int block = c->opt_walk_block;
    long long grid = (P.nwork + block - 1) / block;
    if (grid > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    sweep_walk_kernel<K1, VEC, MODE><<<(unsigned)grid, block, 0, c->stream>>>(P);
    return cudaGetLastError();
}

template <int K1>
cudaError_t dispatch(sldg_ctx* c, const WalkParams& P, int vec, int mode)
{
    if (mode == 0) return vec == 2 ? launch<K1, 2, 0>(c, P) : launch<K1, 1, 0>(c, P);
    return vec == 2 ? launch<K1, 2, 1>(c, P) : launch<K1, 1, 1>(c, P);
}

}  // namespace

cudaError_t SLDG_SFX(sldg_launch_sweep_walk)(sldg_ctx* c, const void* fin, void* fout, const SweepGeom& g,
                                             const ShiftTable& t)
{
    WalkParams P;
    P.fin = static_cast<const real*>(fin); P.fout = static_cast<real*>(fout);
    P.inner = g.inner; P.N = g.N;
    P.sdiv = g.sdiv; P.smod = g.smod; P.t = t;
    // Measured on B200: one value per thread (64-bit loads, more threads, more loads in
    // flight) beats 128-bit loads except for x-sweeps of degree >= 2, where the thread count is ample either way.
#ifdef SLDG_REAL_FLOAT
    // fp32 (measured on cfg2 / cfg4 with smooth fields): 64-bit loads win on every slow axis.  (With a field that is
    // round-off noise of random sign neighbouring x nodes get different s and the paired store splits: 2x slower,
    // physically irrelevant.)
    int vec = 2;
#else
    int vec = (g.mode == 0 && g.K1 >= 3) ? 2 : 1;
#endif
    if (c->opt_walk_vec) vec = c->opt_walk_vec;
    if ((g.inner & 1) || (((uintptr_t)fin | (uintptr_t)fout) & (2 * sizeof(real) - 1))) vec = 1;
    P.innerV = g.inner / vec;
    P.nwork = P.innerV * g.outer;
    if (P.nwork == 0) return cudaSuccess;
    switch (g.K1) {
    case 1: return dispatch<1>(c, P, vec, g.mode);
    case 2: return dispatch<2>(c, P, vec, g.mode);
    case 3: return dispatch<3>(c, P, vec, g.mode);
    case 4: return dispatch<4>(c, P, vec, g.mode);
    case 5: return dispatch<5>(c, P, vec, g.mode);
    }
    return cudaErrorInvalidValue;
}
