// sldg_sweep_fused3d.cu -- TWO consecutive x half steps of a 3x3v run (x_1, x_2, x_3, x_1, x_2, x_3 with the same
// tables) in ONE pass over f, sm_100a.
//
// Inside a run of Strang steps the second x half step of step n is followed directly by the first x half step of step
// n+1 (same time increment, no field solve in between).  sldg_steps runs the two as one pass: 16 B (fp64) of
// HBM traffic per value for SIX sweeps of eq. (3).  Same machinery as sldg_sweep_fused3.cu (a block owns one
// cube q = one (v_1, v_2, v_3) node, a strip of S x_2 cells and all of x_1, and walks along x_3; 1-D TMA bulk copies
// into a ring of input stages, issued by the first thread of an extra warp; bulk stores out), with a second triple
// stacked on the first one:
//
//   first triple T1:  a thread owns one (x_1 cell, MID x_2 cell); the mid cells are the S+1 donors of the strip's S
//                     output cells, so T1 reads S+2 input cells per plane (two halo cells: L2 hits for the neighbouring
//                     strips).  Its output cells go to a shared "mid" stage laid out like an input stage.
//   second triple T2: after a block barrier the threads of the S output cells read the mid stage as the donors of the
//                     second x_1 sweep and run a second x_2 combination and x_3 walk.
//   T1 emits the x_3 cells of the mid array in cyclic order starting at cell s_3 + 1, which is all a periodic walk
//   needs; T2 pairs consecutive ones, so its outputs trail by one cell and the wrap cell comes last.  T2(k-1) and
//   T1(k) share one loop trip (two mid stages): ONE __syncthreads per x_3 cell.
//
// Arithmetic per value is identical (same operands, same order) to two launches of sweep_fused3_kernel, hence to six
// separate sweeps: bit-identical.  Out of place only; degree <= 1; the k+1 rows of a cell a multiple of 16 bytes.
#include "sldg_async.h"
#include "sldg_internal.h"
#include "sldg_real.h"

namespace {

using namespace sldg_async;

struct F3DParams {
    const real* fin;
    real* fout;
    long long cubes;              // prod of D_b, b >= 3
    int N0, N1, N2, S, nstrips, stages;
    long long sdiv[3], smod[3];   // shift index of cube q on axis a: (q / sdiv[a]) % smod[a]
    ShiftTable t[3];
};

template <int K1> struct V3D {
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
__device__ __forceinline__ void f3d_table(const ShiftTable& t, long long idx, real (&A)[K1 * K1], real (&B)[K1 * K1],
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

constexpr int F3D_MAXT = 256;     // compute threads per block (one extra warp issues the copies)

// CP = false: no entry of the three tables has alpha == 0 (the host knows), the copy selects are compiled out.
template <int K1, bool CP>
__global__ void __launch_bounds__(F3D_MAXT + 32) sweep_fused3d_kernel(const F3DParams P)
{
    constexpr int NN = K1 * K1, N3 = K1 * K1 * K1;
    constexpr uint32_t ES = (uint32_t)sizeof(real);
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int N0 = P.N0, N1 = P.N1, N2 = P.N2, S = P.S, ST = P.stages, D0 = N0 * K1;
    const int CELL = K1 * D0;                  // values of the k+1 rows of one x_2 cell
    const int TPI = (S + 2) * CELL, SSI = K1 * TPI;        // input plane / stage: S + 2 cells (two halo cells)
    const int TPM = (S + 1) * CELL, SSM = K1 * TPM;        // mid plane / stage: the S + 1 donors of the strip
    const int OP = S * CELL, OS = K1 * OP;                 // output plane / stage
    const int NTC = (int)blockDim.x - 32;                  // compute threads (whole warps)
    real* const sin_ = reinterpret_cast<real*>(smem_raw);
    real* const smid = sin_ + (size_t)ST * SSI;
    real* const sout = smid + 2 * (size_t)SSM;
    real* const park = sout + 2 * (size_t)OS;              // first blocks of the two walks: [2][N3][NTC]
    const uint32_t sin_s = smem_u32(sin_), sout_s = smem_u32(sout);
    const uint32_t bars_s = (smem_u32(park + 2 * (size_t)N3 * NTC) + 7u) & ~7u;

    const int t = threadIdx.x;
    const bool lead = (t == NTC);                          // first thread of the extra warp: every bulk copy
    const int mu = t / N0, i0 = t - mu * N0;               // mid x_2 slot (T1) = output x_2 slot (T2), x_1 cell
    const long long q = (long long)(blockIdx.x / (unsigned)P.nstrips);
    const int strip = (int)(blockIdx.x - (unsigned)q * (unsigned)P.nstrips);
    const int c0 = strip * S;
    const int nS = min(S, N1 - c0);
    const bool act1 = t < NTC && mu <= nS, act2 = t < NTC && mu < nS;
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
    f3d_table<K1>(P.t[0], ix[0], A1, B1, s1, cp1);
    f3d_table<K1>(P.t[1], ix[1], A2, B2, s2, cp2);
    f3d_table<K1>(P.t[2], ix[2], A3, B3, s3, cp3);
    int ia = i0 - s1; if (ia < 0) ia += N0;
    int ib = ia - 1; if (ib < 0) ib += N0;
    const int oa = ia * K1, ob = ib * K1;
    int dm = c0 - s2 - 1; if (dm < 0) dm += N1;            // first mid cell:   mid slot m   <-> cell (dm + m) mod N_1
    int di = dm - s2 - 1; if (di < 0) di += N1;            // first input cell: input slot m <-> cell (di + m) mod N_1
    const uint32_t cellb = (uint32_t)CELL * ES;

    int lst = 0;                                           // producer: stage of the next load
    auto issue_load = [&](int j) {                         // x_3 cell j -> the next stage of the ring
        if (lead && j < N2) {
            const uint32_t bar = bars_s + (uint32_t)lst * 8u;
            mbar_expect_tx(bar, (uint32_t)(K1 * (nS + 2)) * cellb);
#pragma unroll
            for (int j3 = 0; j3 < K1; j3++) {
                const real* src = gin + ((long long)(j * K1 + j3) * D1) * D0;
                uint32_t dst = sin_s + (uint32_t)(lst * SSI + j3 * TPI) * ES;
                int rem = nS + 2, pos = di;                // contiguous up to the periodic wrap(s)
                while (rem > 0) {
                    const int n = min(rem, N1 - pos);
                    bulk_load(dst, src + (long long)pos * CELL, (uint32_t)n * cellb, bar);
                    dst += (uint32_t)n * cellb; rem -= n; pos = 0;
                }
            }
            if (++lst == ST) lst = 0;
        }
    };

    if (lead) {
        for (int st = 0; st < ST; st++) mbar_init(bars_s + (uint32_t)st * 8u, 1);
        mbar_init_fence();
    }
    __syncthreads();
    for (int j = 0; j < ST; j++) issue_load(j);

    // x_1- then x_2-swept (k+1)^3 block [j3][j2][j1] of this thread's (x_1 cell, x_2 slot mu) from a stage whose planes
    // are `tp` values apart: donors are the stage's slots mu + 1 (A) and mu (B).  Addresses: four per-thread bases (A / B
    // donor slot x the two x_1 donor cells), computed once, plus block-uniform offsets j3 * tp + j2 * D0 -- nothing is
    // recomputed per load (the first version of this kernel spent a quarter of its issue slots on index arithmetic).
    const int pAa = ((mu + 1) * K1) * D0 + oa, pAb = ((mu + 1) * K1) * D0 + ob;
    const int pBa = (mu * K1) * D0 + oa, pBb = (mu * K1) * D0 + ob;
    auto swept12 = [&](const real* stage, int tp, real (&N)[N3]) {
        const real* const qAa = stage + pAa;
        const real* const qAb = stage + pAb;
        const real* const qBa = stage + pBa;
        const real* const qBb = stage + pBb;
#pragma unroll
        for (int j3 = 0; j3 < K1; j3++) {
            real sw[2][NN];                                // [A-donor | B-donor][j2'][j1]
#pragma unroll
            for (int dn = 0; dn < 2; dn++) {
#pragma unroll
                for (int j2 = 0; j2 < K1; j2++) {
                    const int uo = j3 * tp + j2 * D0;      // block-uniform
                    V3D<K1> a, b;
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
    // x_3 combination of two swept blocks -> the k+1 planes (stride `op`) of this thread's cell at `obase`
    auto emit3 = [&](real* obase, int op, const real (&nxt)[N3], const real (&prv)[N3]) {
#pragma unroll
        for (int j3 = 0; j3 < K1; j3++)
#pragma unroll
            for (int j2 = 0; j2 < K1; j2++) {
                V3D<K1> r;
#pragma unroll
                for (int j1 = 0; j1 < K1; j1++) {
                    real acc = 0;
#pragma unroll
                    for (int l = 0; l < K1; l++) acc += A3[j3 * K1 + l] * nxt[(l * K1 + j2) * K1 + j1];
#pragma unroll
                    for (int l = 0; l < K1; l++) acc += B3[j3 * K1 + l] * prv[(l * K1 + j2) * K1 + j1];
                    r.v[j1] = (CP && cp3) ? nxt[(j3 * K1 + j2) * K1 + j1] : acc;
                }
                r.store(obase + (j3 * op + j2 * D0));      // block-uniform offset
            }
    };
    const int cofs = (mu * K1) * D0 + i0 * K1;             // this thread's cell inside a mid / output plane

    real a1[2][N3], a2[2][N3];
    if (act1) {
        mbar_wait(bars_s, 0u);                             // x_3 cell 0
        swept12(sin_, TPI, a1[0]);
#pragma unroll
        for (int m = 0; m < N3; m++) park[m * NTC + t] = a1[0][m];
    }
    fence_async_smem();                                    // generic-proxy reads of stage 0 -> its refill by the async proxy
    __syncthreads();
    issue_load(ST);

    int cst = (ST > 1) ? 1 : 0;                            // consumers: stage and phase of the next input cell
    uint32_t cph = (ST > 1) ? 0u : 1u;
    int io3 = 2 * s3 + 2; io3 %= N2;                       // output x_3 cell of T2's first donor pair
    auto store_out = [&](int buf) {                        // producer: the S output cells of x_3 cell io3, one copy per plane
#pragma unroll
        for (int j3 = 0; j3 < K1; j3++)
            bulk_store(gout + (((long long)(io3 * K1 + j3)) * D1 + (long long)c0 * K1) * D0,
                       sout_s + (uint32_t)(buf * OS + j3 * OP) * ES, (uint32_t)nS * cellb);
        bulk_commit();
        if (++io3 == N2) io3 = 0;
    };
    // One loop trip k: T2(k-1) (mid cell k-1 -> output) and T1(k) (input cell k+1 -> mid cell k), then ONE barrier.
    auto trip = [&](int k, real (&nx1)[N3], const real (&pv1)[N3], real (&nx2)[N3], const real (&pv2)[N3]) {
        if (k >= 1 && act2) {
            swept12(smid + ((k - 1) & 1) * SSM, TPM, nx2);
            if (k == 1) {                                  // the first block of the second walk only initialises it
#pragma unroll
                for (int m = 0; m < N3; m++) park[(N3 + m) * NTC + t] = nx2[m];
            } else {
                emit3(sout + ((k - 1) & 1) * OS + cofs, OP, nx2, pv2);
            }
        }
        if (k < N2) {
            const bool fresh = k + 1 < N2;                 // else: the first input cell closes the periodic wrap
            if (act1) {
                if (fresh) {
                    mbar_wait(bars_s + (uint32_t)cst * 8u, cph);
                    swept12(sin_ + cst * SSI, TPI, nx1);
                } else {
#pragma unroll
                    for (int m = 0; m < N3; m++) nx1[m] = park[m * NTC + t];
                }
                emit3(smid + (k & 1) * SSM + cofs, TPM, nx1, pv1);
            }
            if (fresh) { if (++cst == ST) { cst = 0; cph ^= 1u; } }
        }
        fence_async_smem();
        if (lead) bulk_wait_read<0>();                     // the stores of the previous trip have left their output stage
        __syncthreads();
        if (lead && k >= 2) store_out((k - 1) & 1);
        issue_load(k + 1 + ST);
    };
    {
        int k = 0;
        for (; k + 1 <= N2; k += 2) { trip(k, a1[1], a1[0], a2[1], a2[0]); trip(k + 1, a1[0], a1[1], a2[0], a2[1]); }
        if (k <= N2) trip(k, a1[1], a1[0], a2[1], a2[0]);
    }
    // the periodic wrap of the second walk: its first block again, after the last one (written by T2(N_2 - 1))
    if (act2) {
        real f2[N3];
#pragma unroll
        for (int m = 0; m < N3; m++) f2[m] = park[(N3 + m) * NTC + t];
        real* const o = sout + (N2 & 1) * OS + cofs;
        if ((N2 - 1) & 1) emit3(o, OP, f2, a2[1]);
        else emit3(o, OP, f2, a2[0]);
    }
    fence_async_smem();
    if (lead) bulk_wait_read<0>();
    __syncthreads();
    if (lead) { store_out(N2 & 1); bulk_wait_read<0>(); }
}

template <int K1, bool CP>
cudaError_t launch(sldg_ctx* c, const F3DParams& P, int threads, size_t smem)
{
    auto kern = sweep_fused3d_kernel<K1, CP>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const long long grid = P.cubes * P.nstrips;
    if (grid > 0x7fffffffLL) return cudaErrorNotSupported;
    kern<<<(unsigned)grid, threads, smem, c->stream>>>(P);
    return cudaGetLastError();
}

// strip size, ring depth and shared memory of a launch: every rule the launcher applies
struct F3DShape { int S, nstrips, stages, threads; size_t smem; };

bool shape(const sldg_ctx* c, F3DShape* o)
{
    const int K1 = c->K1, N0 = c->cells[0], N1 = c->cells[1];
    if (c->dx != 3 || K1 > 2 || 2 * N0 > F3D_MAXT) return false;
    const long long cellb = (long long)K1 * c->D[0] * (long long)sizeof(real);
    if (cellb & 15) return false;
    // strip: about opt_f3d_threads threads for the S + 1 mid cells, strips of (nearly) equal size
    long long S = c->opt_f3d_threads / N0 - 1;
    if (S < 1) S = 1;
    if (S > N1) S = N1;
    long long nstrips = (N1 + S - 1) / S;
    S = (N1 + nstrips - 1) / nstrips;
    nstrips = (N1 + S - 1) / S;
    if ((S + 1) * N0 > F3D_MAXT) return false;
    const int threads = (int)(((S + 1) * N0 + 31) / 32 * 32);
    int stages = c->opt_f3_stages;
    auto smem_of = [&](int st) {
        return (size_t)K1 * (st * (S + 2) + 2 * (S + 1) + 2 * S) * cellb + (size_t)2 * K1 * K1 * K1 * threads * sizeof(real) + 8 * st + 16;
    };
    while (smem_of(stages) > 227 * 1024 && stages > 2) stages--;
    if (smem_of(stages) > 227 * 1024) return false;
    if (o) { o->S = (int)S; o->nstrips = (int)nstrips; o->stages = stages; o->threads = threads + 32; o->smem = smem_of(stages); }
    return true;
}

}  // namespace

bool SLDG_SFX(sldg_fused3d_shape)(const sldg_ctx* c) { return shape(c, nullptr); }

// g: geometry of axes 0, 1, 2; t: their shift tables.  cudaErrorNotSupported when the shape does not fit.
cudaError_t SLDG_SFX(sldg_launch_sweep_fused3d)(sldg_ctx* c, const void* fin, void* fout, const SweepGeom* g,
                                                const ShiftTable* t, int any_copy)
{
    if (g[2].outer == 0) return cudaSuccess;
    const int K1 = g[0].K1;
    const long long D0 = (long long)g[0].N * K1, D1 = (long long)g[1].N * K1, D2 = (long long)g[2].N * K1;
    F3DShape sh;
    if (fin == fout || !shape(c, &sh) || g[1].inner != D0 || g[2].inner != D0 * D1) return cudaErrorNotSupported;
    if (g[0].mode != 0 || g[1].mode != 0 || g[2].mode != 0) return cudaErrorNotSupported;
    if (g[0].sdiv % (D1 * D2) != 0 || g[1].sdiv % D2 != 0) return cudaErrorNotSupported;
    if ((((uintptr_t)fin) | ((uintptr_t)fout)) & 15) return cudaErrorNotSupported;
    F3DParams P;
    P.fin = static_cast<const real*>(fin); P.fout = static_cast<real*>(fout);
    P.cubes = g[2].outer; P.N0 = g[0].N; P.N1 = g[1].N; P.N2 = g[2].N;
    P.S = sh.S; P.nstrips = sh.nstrips; P.stages = sh.stages;
    P.sdiv[0] = g[0].sdiv / (D1 * D2); P.sdiv[1] = g[1].sdiv / D2; P.sdiv[2] = g[2].sdiv;
    for (int a = 0; a < 3; a++) { P.smod[a] = g[a].smod; P.t[a] = t[a]; }
    if (any_copy) return K1 == 1 ? launch<1, true>(c, P, sh.threads, sh.smem) : launch<2, true>(c, P, sh.threads, sh.smem);
    return K1 == 1 ? launch<1, false>(c, P, sh.threads, sh.smem) : launch<2, false>(c, P, sh.threads, sh.smem);
}
