// sldg_sweep_fused3.cu -- the x_1, x_2 AND x_3 sweeps of a 3-d x advection in ONE pass over f, sm_100a.
//
// eq. (3), reading B, applied three times in the order x_1, x_2, x_3 (the sweeps commute):
// 16 B (fp64) of HBM traffic per value for THREE sweeps instead of 48 B.  Same machinery as
// sldg_sweep_fused_cell.cu (1-D TMA bulk copies into a ring of shared-memory stages, one thread per cell, register
// walk along the slowest of the fused axes, bulk stores out), one axis deeper:
//
//   f is seen as [cubes q][N_2 cells][k+1 planes][D_1 rows][D_0].  A block owns one cube q (all its shifts are those
//   of q's v_1, v_2, v_3 nodes) and a STRIP of S consecutive x_2 cells, all of x_1, and walks along x_3.
//   Per x_3 cell it needs, in each of the k+1 planes, the rows of the S+1 x_2 cells that are the donors of its
//   strip (one halo cell; contiguous in memory up to the periodic wrap: one or two bulk copies per plane).
//   A thread owns one (x_1 cell, x_2 cell): it x_1-sweeps the rows of its two x_2 donor cells from shared memory,
//   combines them with A_2, B_2, and walks along x_3 with the resulting (k+1)^3 block in registers (previous cell
//   and first cell kept), writing output cell (j + s_3 + 1) mod N_2 to a shared output stage that leaves by one
//   bulk store per plane.  The halo cell is read by two neighbouring strips of the same cube (adjacent blocks,
//   normally an L2 hit); everything else is read once and written once.
//
// Arithmetic per value is identical (same operands, same order) to the three separate sweeps.  Out of place only;
// degree <= 1 (k+1 <= 2: the (k+1)^3 blocks must stay in registers); the k+1 rows of a cell must be a multiple of
// 16 bytes.
#include "sldg_async.h"
#include "sldg_internal.h"
#include "sldg_real.h"

namespace {

using namespace sldg_async;

struct F3Params {
    const real* fin;
    real* fout;
    long long cubes;              // prod of D_b, b >= 3
    int N0, N1, N2, S, nstrips, stages;
    long long sdiv[3], smod[3];   // shift index of cube q on axis a: (q / sdiv[a]) % smod[a]
    ShiftTable t[3];
};

constexpr int F3_OST = 2;

template <int K1> struct V3 {
    real v[K1];
    __device__ __forceinline__ void load(const real* p)
    {
        if constexpr (K1 == 2) { real2 t = *reinterpret_cast<const real2*>(p); v[0] = t.x; v[1] = t.y; }
        else v[0] = p[0];
    }
    __device__ __forceinline__ void store(real* p) const
    {
        if constexpr (K1 == 2) *reinterpret_cast<real2*>(p) = make_real2(v[0], v[1]);
        else p[0] = v[0];
    }
};

template <int K1>
__device__ __forceinline__ void load_table(const ShiftTable& t, long long idx, real (&A)[K1 * K1], real (&B)[K1 * K1],
                                           int& s, bool& cp)
{
    constexpr int NN = K1 * K1;
    const int sv = __ldg(t.S + idx);
    cp = (sv & SLDG_COPY_BIT) != 0;
    s = sv & SLDG_S_MASK;
    const real* ab = static_cast<const real*>(t.AB) + idx * t.strideIdx;
#pragma unroll
    for (int m = 0; m < NN; m++) {
        A[m] = __ldg(ab + m * t.strideM);
        B[m] = __ldg(ab + (NN + m) * t.strideM);
    }
}

// CP = false: no entry of the three tables has alpha == 0 (the host knows), the copy selects are compiled out.
// The block has one extra warp whose first thread (the PRODUCER) issues every bulk copy, so that no compute warp
// carries the address arithmetic of the copies or is late at the per-step barrier.
template <int K1, bool CP>
__global__ void __launch_bounds__(288) sweep_fused3_kernel(const F3Params P)
{
    constexpr int NN = K1 * K1, N3 = K1 * K1 * K1;
    constexpr uint32_t ES = (uint32_t)sizeof(real);
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int N0 = P.N0, N1 = P.N1, N2 = P.N2, S = P.S, ST = P.stages, D0 = N0 * K1;
    const int CELL = K1 * D0;                  // values of the k+1 rows of one x_2 cell
    const int TP = (S + 1) * CELL;             // one plane of an input tile (S cells + 1 halo cell)
    const int SS = K1 * TP;                    // input stage: the k+1 planes of one x_3 cell
    const int OP = S * CELL, OS = K1 * OP;     // output plane / stage
    real* const sin_ = reinterpret_cast<real*>(smem_raw);
    real* const sout = sin_ + (size_t)ST * SS;
    const uint32_t sin_s = smem_u32(sin_), sout_s = smem_u32(sout);
    const uint32_t bars_s = (smem_u32(sout + (size_t)F3_OST * OS) + 7u) & ~7u;

    const int t = threadIdx.x;
    const int NT = S * N0;                                 // compute threads; the producer is thread roundup32(NT)
    const bool lead = (t == (int)blockDim.x - 32);
    const int e1 = t / N0, i0 = t - e1 * N0;
    const long long q = (long long)(blockIdx.x / (unsigned)P.nstrips);
    const int strip = (int)(blockIdx.x - (unsigned)q * (unsigned)P.nstrips);
    const int c0 = strip * S;
    const int nS = min(S, N1 - c0);
    const bool active = t < NT && e1 < nS;
    const long long D1 = (long long)N1 * K1, D2 = (long long)N2 * K1;
    const real* const gin = P.fin + q * D2 * D1 * D0;
    real* const gout = P.fout + q * D2 * D1 * D0;

    real A1[NN], B1[NN], A2[NN], B2[NN], A3[NN], B3[NN];
    int s1, s2, s3;
    bool cp1, cp2, cp3;
    long long ix[3];
    if (P.cubes < (1LL << 31)) {                           // 32-bit divisions when they fit (the usual case)
#pragma unroll
        for (int a = 0; a < 3; a++) ix[a] = ((unsigned)q / (unsigned)P.sdiv[a]) % (unsigned)P.smod[a];
    } else {
#pragma unroll
        for (int a = 0; a < 3; a++) ix[a] = (q / P.sdiv[a]) % P.smod[a];
    }
    load_table<K1>(P.t[0], ix[0], A1, B1, s1, cp1);
    load_table<K1>(P.t[1], ix[1], A2, B2, s2, cp2);
    load_table<K1>(P.t[2], ix[2], A3, B3, s3, cp3);
    int ia = i0 - s1; if (ia < 0) ia += N0;
    int ib = ia - 1; if (ib < 0) ib += N0;
    const int oa = ia * K1, ob = ib * K1;
    int d0 = c0 - s2 - 1; if (d0 < 0) d0 += N1;            // first donor cell of the strip: slot m <-> cell (d0+m) mod N_1
    const int run1 = min(nS + 1, N1 - d0);                 // cells before the periodic wrap
    const uint32_t cellb = (uint32_t)CELL * ES;

    int lst = 0;                                           // producer: stage of the next load (loads are issued in order)
    auto issue_load = [&](int j) {                         // x_3 cell j -> stage j % ST
        if (lead && j < N2) {
            const int st = lst;
            if (++lst == ST) lst = 0;
            const uint32_t bar = bars_s + (uint32_t)st * 8u;
            mbar_expect_tx(bar, (uint32_t)(K1 * (nS + 1)) * cellb);
#pragma unroll
            for (int j3 = 0; j3 < K1; j3++) {
                const real* src = gin + ((long long)(j * K1 + j3) * D1) * D0;
                const uint32_t dst = sin_s + (uint32_t)(st * SS + j3 * TP) * ES;
                bulk_load(dst, src + (long long)d0 * CELL, (uint32_t)run1 * cellb, bar);
                if (run1 < nS + 1) bulk_load(dst + (uint32_t)run1 * cellb, src, (uint32_t)(nS + 1 - run1) * cellb, bar);
            }
        }
    };

    if (lead) {
        for (int st = 0; st < ST; st++) mbar_init(bars_s + (uint32_t)st * 8u, 1);
        mbar_init_fence();
    }
    __syncthreads();
    for (int j = 0; j < ST; j++) issue_load(j);

    // x_1- then x_2-swept (k+1)^3 block [j3][j2][j1] of this thread's (x_1 cell, x_2 cell) from one input stage.
    // Addresses: four per-thread bases (A / B donor slot x the two x_1 donor cells), computed once, plus block-uniform
    // offsets j3 * TP + j2 * D0: no index arithmetic per load.
    const int pAa = ((e1 + 1) * K1) * D0 + oa, pAb = ((e1 + 1) * K1) * D0 + ob;
    const int pBa = (e1 * K1) * D0 + oa, pBb = (e1 * K1) * D0 + ob;
    auto swept12 = [&](const real* stage, real (&N)[N3]) {
        const real* const qAa = stage + pAa;
        const real* const qAb = stage + pAb;
        const real* const qBa = stage + pBa;
        const real* const qBb = stage + pBb;
#pragma unroll
        for (int j3 = 0; j3 < K1; j3++) {
            real sw[2][NN];                                // [A-donor cell c-s_2 | B-donor cell c-s_2-1][j2'][j1]
#pragma unroll
            for (int dn = 0; dn < 2; dn++) {
#pragma unroll
                for (int j2 = 0; j2 < K1; j2++) {
                    const int uo = j3 * TP + j2 * D0;      // block-uniform
                    V3<K1> a, b;
                    a.load((dn ? qBa : qAa) + uo);
                    b.load((dn ? qBb : qAb) + uo);
#pragma unroll
                    for (int j1 = 0; j1 < K1; j1++) {
                        real acc = 0;
#pragma unroll
                        for (int m = 0; m < K1; m++) acc += A1[j1 * K1 + m] * a.v[m];
#pragma unroll
                        for (int m = 0; m < K1; m++) acc += B1[j1 * K1 + m] * b.v[m];
                        sw[dn][j2 * K1 + j1] = (CP && cp1) ? a.v[j1] : acc;
                    }
                }
            }
#pragma unroll
            for (int j2 = 0; j2 < K1; j2++)
#pragma unroll
                for (int j1 = 0; j1 < K1; j1++) {
                    real acc = 0;
#pragma unroll
                    for (int l = 0; l < K1; l++) acc += A2[j2 * K1 + l] * sw[0][l * K1 + j1];
#pragma unroll
                    for (int l = 0; l < K1; l++) acc += B2[j2 * K1 + l] * sw[1][l * K1 + j1];
                    N[(j3 * K1 + j2) * K1 + j1] = (CP && cp2) ? sw[0][j2 * K1 + j1] : acc;
                }
        }
    };

    real first[N3], prev[N3];
    if (active) {
        mbar_wait(bars_s, 0u);                             // x_3 cell 0
        swept12(sin_, first);
    }
#pragma unroll
    for (int m = 0; m < N3; m++) prev[m] = first[m];
    fence_async_smem();                                    // generic-proxy reads of stage 0 -> its refill by the async proxy
    __syncthreads();
    issue_load(ST);

    int io3 = s3 + 1; if (io3 >= N2) io3 -= N2;            // output x_3 cell of the current donor pair
    int cst = (ST > 1) ? 1 : 0;                            // consumers: stage and phase of the next input cell (cell 1)
    uint32_t cph = (ST > 1) ? 0u : 1u;
    const int cofs = (e1 * K1) * D0 + i0 * K1;             // this thread's cell inside an output plane
    // one step of the x_3 walk: nxt <- swept block of input cell h+1 (or the first one), output cell from (nxt, prv).
    // The walk alternates between `prev` and `alt` (two steps per trip): no register moves between steps.
    real alt[N3];
    auto step3 = [&](int h, real (&nxt)[N3], const real (&prv)[N3]) {
        const int j = h + 1;
        if (j < N2) {
            if (active) {
                mbar_wait(bars_s + (uint32_t)cst * 8u, cph);
                swept12(sin_ + cst * SS, nxt);
            }
            if (++cst == ST) { cst = 0; cph ^= 1u; }
        } else {
#pragma unroll
            for (int m = 0; m < N3; m++) nxt[m] = first[m];
        }
        if (active) {
            real* obase = sout + (h & 1) * OS + cofs;
#pragma unroll
            for (int j3 = 0; j3 < K1; j3++)
#pragma unroll
                for (int j2 = 0; j2 < K1; j2++) {
                    V3<K1> r;
#pragma unroll
                    for (int j1 = 0; j1 < K1; j1++) {
                        real acc = 0;
#pragma unroll
                        for (int l = 0; l < K1; l++) acc += A3[j3 * K1 + l] * nxt[(l * K1 + j2) * K1 + j1];
#pragma unroll
                        for (int l = 0; l < K1; l++) acc += B3[j3 * K1 + l] * prv[(l * K1 + j2) * K1 + j1];
                        r.v[j1] = (CP && cp3) ? nxt[(j3 * K1 + j2) * K1 + j1] : acc;
                    }
                    r.store(obase + j3 * OP + j2 * D0);
                }
        }
        fence_async_smem();
        if (lead) bulk_wait_read<0>();                     // the stores of step h-1 have left their output stage
        __syncthreads();
        if (lead) {
#pragma unroll
            for (int j3 = 0; j3 < K1; j3++)
                bulk_store(gout + (((long long)(io3 * K1 + j3)) * D1 + (long long)c0 * K1) * D0,
                           sout_s + (uint32_t)((h & 1) * OS + j3 * OP) * ES, (uint32_t)nS * cellb);
            bulk_commit();
        }
        issue_load(j + ST);
        io3++; if (io3 >= N2) io3 = 0;
    };
    {
        int h = 0;
        for (; h + 1 < N2; h += 2) { step3(h, alt, prev); step3(h + 1, prev, alt); }
        if (h < N2) step3(h, alt, prev);
    }
    if (lead) bulk_wait_read<0>();
}

template <int K1, bool CP>
cudaError_t launch(sldg_ctx* c, const F3Params& P, int threads, size_t smem)
{
    auto kern = sweep_fused3_kernel<K1, CP>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const long long grid = P.cubes * P.nstrips;
    if (grid > 0x7fffffffLL) return cudaErrorNotSupported;
    kern<<<(unsigned)grid, ((threads + 31) & ~31) + 32, smem, c->stream>>>(P);
    return cudaGetLastError();
}

}  // namespace

// g0, g1, g2: geometry of axes 0, 1, 2.  cudaErrorNotSupported when the shape does not fit (the caller plans the
// fused x_1+x_2 pass plus a separate x_3 sweep instead).
cudaError_t SLDG_SFX(sldg_launch_sweep_fused3)(sldg_ctx* c, const void* fin, void* fout, const SweepGeom* g,
                                               const ShiftTable* t, int any_copy)
{
    if (g[2].outer == 0) return cudaSuccess;
    const int K1 = g[0].K1;
    const long long D0 = (long long)g[0].N * K1, D1 = (long long)g[1].N * K1, D2 = (long long)g[2].N * K1;
    if (fin == fout || K1 > 2 || g[1].inner != D0 || g[2].inner != D0 * D1) return cudaErrorNotSupported;
    if (g[0].mode != 0 || g[1].mode != 0 || g[2].mode != 0) return cudaErrorNotSupported;
    if (g[0].sdiv % (D1 * D2) != 0 || g[1].sdiv % D2 != 0) return cudaErrorNotSupported;
    const long long cellb = (long long)K1 * D0 * sizeof(real);
    if ((cellb & 15) || ((((uintptr_t)fin) | ((uintptr_t)fout)) & 15) || g[0].N > 256) return cudaErrorNotSupported;
    F3Params P;
    P.fin = static_cast<const real*>(fin); P.fout = static_cast<real*>(fout);
    P.cubes = g[2].outer; P.N0 = g[0].N; P.N1 = g[1].N; P.N2 = g[2].N;
    // strip: about opt_f3_threads threads per block, strips of (nearly) equal size
    long long S = c->opt_f3_threads / g[0].N;
    if (S < 1) S = 1;
    if (S > g[1].N) S = g[1].N;
    long long nstrips = (g[1].N + S - 1) / S;
    S = (g[1].N + nstrips - 1) / nstrips;
    nstrips = (g[1].N + S - 1) / S;
    int stages = c->opt_f3_stages;
    auto smem_of = [&](long long s, int st) { return (size_t)K1 * (st * (s + 1) + F3_OST * s) * cellb + 8 * st + 16; };
    while (smem_of(S, stages) > 227 * 1024 && stages > 2) stages--;
    if (smem_of(S, stages) > 227 * 1024) return cudaErrorNotSupported;
    P.S = (int)S; P.nstrips = (int)nstrips; P.stages = stages;
    P.sdiv[0] = g[0].sdiv / (D1 * D2); P.sdiv[1] = g[1].sdiv / D2; P.sdiv[2] = g[2].sdiv;
    for (int a = 0; a < 3; a++) { P.smod[a] = g[a].smod; P.t[a] = t[a]; }
    const int threads = (int)(S * g[0].N);
    const size_t smem = smem_of(S, stages);
    if (any_copy) return K1 == 1 ? launch<1, true>(c, P, threads, smem) : launch<2, true>(c, P, threads, smem);
    return K1 == 1 ? launch<1, false>(c, P, threads, smem) : launch<2, false>(c, P, threads, smem);
}
