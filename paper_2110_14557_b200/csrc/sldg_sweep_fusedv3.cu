// sldg_sweep_fusedv3.cu -- the v_1, v_2 AND v_3 sweeps of a 3x3v v advection in ONE pass over f, sm_100a.
//
// eq. (3), reading B, applied three times in the order v_1, v_2, v_3 (E does not change during the
// v sweeps; the paper's single-GPU study is the 3x3v case, P:258, 9 advections = 18 accesses per step):
//     u_i <- A(alpha) u_{(i-s) mod N} + B(alpha) u_{(i-s-1) mod N},   delta = -E_d(x) dt / h_{v_d}  per x node.
// 16 B (fp64) of HBM traffic per value for THREE sweeps instead of 48 B.
//
//   f is seen as [D_3 rows][D_2 rows][D_1 rows][X]  (X = all x nodes, contiguous).  Every shift of the three sweeps
//   is that of the x node, so the thread that owns an x node keeps A_d, B_d (d = 1..3) of that node in registers.
//   A block owns a tile of WX consecutive x nodes, ALL of v_1, and a STRIP of S consecutive v_2 donor pairs
//   (input cells c0 .. c0+S, the last one being the halo: read by two neighbouring strips, normally an L2 hit),
//   and walks along v_3.  Per (v_3 cell, v_2 cell) ONE 4-d TMA tensor copy (box WX x D_1 x (k+1) x (k+1)) brings
//   [j3][j2][D_1][WX] into a slot of a ring of shared-memory slots; full/empty mbarriers pace the ring, thread 0
//   issues the copies between its own boxes, no __syncthreads in the loop.
//   A thread owns one (x node, v_1 cell).  Per box it v_1-sweeps the (k+1)^2 rows of its two v_1 donor cells from
//   shared memory; two consecutive boxes give, by A_2, B_2, the v_1v_2-swept (k+1)^3 block of a donor pair; that
//   block and the one of the previous v_3 cell (kept in registers, one per pair of the strip) give, by A_3, B_3,
//   the output cell (v_2: (c0+p + s_2 + 1) mod N_2, v_3: (j + s_3 + 1) mod N_3), stored straight from registers
//   (lanes over x: coalesced WX * 8 B pieces).  The first v_3 cell is streamed in once more to close the periodic
//   wrap (1/N_3 of the reads).
//
// Arithmetic per value is identical (same operands, same order) to sweep_walk_kernel on v_1, v_2, v_3 in turn, so
// the fused and the unfused plans agree bit for bit.  Out of place only; dim_x = dim_v = 3; degree <= 1;
// D_1 <= 256 (one TMA box); X * sizeof(real) a multiple of 16.
#include <type_traits>

#include "sldg_async.h"
#include "sldg_internal.h"
#include "sldg_real.h"
#include "sldg_tmap.h"

namespace {

using namespace sldg_async;

constexpr int FV3_MAXT = 320;      // threads per block: one block per SM, up to 200 registers per thread
constexpr int FV3_MAXS = 5;        // v_2 donor pairs per strip (each keeps a (k+1)^3 block in registers)

struct FV3Params {
    real* fout;
    long long X;
    int N1, N2, N3, WX, S, nstrips, ntiles, slots;
    int pw;                       // 1: the block's LAST warp is a dedicated producer (issues every tensor copy), the others only consume
    uint32_t slot_bytes;          // ring slot stride (>= (k+1)^2 * D_1 * WX * sizeof(real), multiple of 1024)
    ShiftTable t1, t2, t3;
};

template <int K1>
__device__ __forceinline__ void fv3_table(const ShiftTable& t, long long idx, real (&A)[K1 * K1], real (&B)[K1 * K1],
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

// WXT: x nodes per tile as a compile-time constant (shared-memory offsets become immediates), 0 = P.WX at run time
template <int K1, int S, int WXT>
__global__ void __launch_bounds__(FV3_MAXT + 32)
    sweep_fusedv3_kernel(const __grid_constant__ CUtensorMap tmap, const FV3Params P)
{
    constexpr int NN = K1 * K1, N3V = K1 * K1 * K1;
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    const int ST = P.slots, WX = WXT ? WXT : P.WX, N1 = P.N1, N2 = P.N2, N3 = P.N3;
    const int D1 = N1 * K1, D2 = N2 * K1;
    const uint32_t ring_s = smem_u32(smem_raw);
    const uint32_t full_s = ring_s + (uint32_t)ST * P.slot_bytes;       // ST full barriers, then ST empty barriers
    const uint32_t empty_s = full_s + (uint32_t)ST * 8u;

    const int t = threadIdx.x;
    const bool PW = P.pw != 0;
    const int NTR = (int)blockDim.x - (PW ? 32 : 0);                    // consumer threads (whole warps)
    const int LAG = ST >= 4 ? 2 : 1;                                    // the producer refills the slot of box i - LAG
    const int DEP = ST - LAG;                                           // boxes in flight ahead of the consumers
    const int strip = (int)(blockIdx.x % (unsigned)P.nstrips);          // neighbouring strips (shared halo) run together
    const int tile = (int)(blockIdx.x / (unsigned)P.nstrips);
    const int c0 = strip * S;
    const int nS = min(S, N2 - c0);                                     // donor pairs of this strip
    const int nB = nS + 1;                                              // boxes (v_2 cells) per v_3 cell
    const long long x0 = (long long)tile * WX;
    const int total = (N3 + 1) * nB;                                    // v_3 cell 0 is streamed in once more

    if (t == 0) {
        for (int s = 0; s < ST; s++) { mbar_init(full_s + 8u * s, 1); mbar_init(empty_s + 8u * s, NTR / 32); }
        mbar_init_fence();
    }
    __syncthreads();

    // ---------------- producer (thread 0, between its own boxes): one tensor copy per ring slot
    const uint32_t box_bytes = (uint32_t)NN * (uint32_t)D1 * (uint32_t)WX * (uint32_t)sizeof(real);
    int pst = 0, pn = 0, pm = 0, pj = 0, pi = 0;
    auto produce = [&]() {
        if (pi >= total) return;
        if (pn > 0) mbar_wait(empty_s + 8u * pst, (uint32_t)((pn - 1) & 1));
        mbar_expect_tx(full_s + 8u * pst, box_bytes);
        int cell2 = c0 + pm; if (cell2 >= N2) cell2 -= N2;
        const int cell3 = (pj == N3) ? 0 : pj;
        tma_load_4d(ring_s + (uint32_t)pst * P.slot_bytes, &tmap, (int)x0, 0, cell2 * K1, cell3 * K1, full_s + 8u * pst);
        if (++pm == nB) { pm = 0; pj++; }
        if (++pst == ST) { pst = 0; pn++; }
        pi++;
    };
    if (PW) {                                                           // dedicated producer: the whole ring in flight at once
        if (t == NTR)
            for (int i = 0; i < ST; i++) produce();
    } else if (t == 0) {
        for (int i = 0; i < DEP; i++) produce();
    }

    // ---------------- consumers
    const int c = t / WX, x = t - c * WX;
    const bool active = (c < N1) && (x0 + x < P.X);
    real A1[NN], B1[NN], A2[NN], B2[NN], A3[NN], B3[NN];
    int s1 = 0, s2 = 0, s3 = 0;
    bool cp1 = false, cp2 = false, cp3 = false;
#pragma unroll
    for (int m = 0; m < NN; m++) { A1[m] = B1[m] = A2[m] = B2[m] = A3[m] = B3[m] = 0; }
    if (active) {
        const long long idx = x0 + x;
        fv3_table<K1>(P.t1, idx, A1, B1, s1, cp1);
        fv3_table<K1>(P.t2, idx, A2, B2, s2, cp2);
        fv3_table<K1>(P.t3, idx, A3, B3, s3, cp3);
    }
    int ia = 0, ib = 0;
    if (active) {
        ia = c - s1; if (ia < 0) ia += N1;
        ib = ia - 1; if (ib < 0) ib += N1;
    }
    // k = 1: A_2, B_2, A_3, B_3 of the tile's x nodes live in shared memory (one padded record per x node: rows
    // [A_2[j][.] | B_2[j][.]] then [A_3[j][.] | B_3[j][.]], read as 2-value vectors; lanes of equal x broadcast, the
    // 8 lanes of a 128-bit phase fall on different banks).  With all six tables and the per-pair (k+1)^3 blocks in
    // registers ptxas spills (168 registers at 10 warps per SM).
    constexpr bool T23S = (K1 == 2);
    constexpr int PAD = 4 * NN + 2;
    real* const tab = reinterpret_cast<real*>(smem_raw + (size_t)ST * P.slot_bytes + 16 * (size_t)ST) + x * PAD;
    if (T23S) {
        if (c == 0) {
#pragma unroll
            for (int j = 0; j < K1; j++)
#pragma unroll
                for (int l = 0; l < K1; l++) {
                    tab[j * 2 * K1 + l] = A2[j * K1 + l]; tab[j * 2 * K1 + K1 + l] = B2[j * K1 + l];
                    tab[2 * NN + j * 2 * K1 + l] = A3[j * K1 + l]; tab[2 * NN + j * 2 * K1 + K1 + l] = B3[j * K1 + l];
                }
        }
        __syncthreads();
    }
    if (PW && t >= NTR) {
        // Producer warp: lane 0 refills each slot as soon as every consumer warp has arrived on its empty barrier.  No consumer
        // ever waits on an empty barrier or issues a copy, so a box is delayed only by the slowest warp's reads, not by warp 0's
        // position in its own arithmetic.  The block's shared memory outlives this warp: the consumers wait for every full
        // barrier before they finish.
        if (t == NTR)
            while (pi < total) produce();
        return;
    }
    // the alpha == 0 copy selects are compiled out for warps none of whose x nodes has the copy bit (the usual case)
    const bool anycp = __any_sync(0xffffffffu, cp1 || cp2 || cp3);

    const real* const ring = reinterpret_cast<const real*>(smem_raw);
    const real* const pa0 = ring + ia * K1 * WX + x;                    // donor rows of slot 0
    const real* const pb0 = ring + ib * K1 * WX + x;
    const int slot_vals = (int)(P.slot_bytes / sizeof(real));
    const int rowvals = D1 * WX;                                        // one (j3, j2) row group of a box
    const bool warp_lead = (t & 31) == 0;
    const long long X = P.X;
    const long long rowX = (long long)D1 * X;                           // one v_2 row, in values
    const long long cell2X = (long long)K1 * rowX;                      // one v_2 cell
    const long long row3X = (long long)D2 * rowX;                       // one v_3 row
    const long long cell3X = (long long)K1 * row3X;                     // one v_3 cell

    int st = 0, soff = 0;
    uint32_t ph = 0, fbar = full_s;

    auto body = [&](auto cpt) {
        constexpr bool CP = decltype(cpt)::value;
        // next box of the ring -> the v_1-swept (k+1)^3 block [j3][j2][j1] of this thread's v_1 cell
        auto swept_box = [&](real (&g)[N3V]) {
            if (!PW && t == 0) produce();
            mbar_wait(fbar, ph);
            real a[NN][K1], b[NN][K1];
            const real* pa = pa0 + soff;
            const real* pb = pb0 + soff;
#pragma unroll
            for (int r = 0; r < NN; r++) {
#pragma unroll
                for (int m = 0; m < K1; m++) { a[r][m] = pa[m * WX]; b[r][m] = pb[m * WX]; }
                pa += rowvals; pb += rowvals;
            }
            // The slot is read: hand it back.  It is refilled by the ASYNC proxy (TMA) once every warp has arrived, so the
            // generic-proxy reads above are ordered before that write by a proxy fence.  (Tried instead: an arrive placed
            // after the arithmetic that consumes the loads, with the results as unused operands of the asm statement.  The
            // dependency exists only in the compiler's IR, not in the PTX that ptxas schedules: the drift test failed, 256
            // wrong values, and the time did not change: 13.9 against 13.7 ms on cfg4.)
            fence_async_smem();
            __syncwarp();
            if (warp_lead) mbar_arrive(fbar + 8u * (uint32_t)ST);
            st++; soff += slot_vals; fbar += 8u;
            if (st == ST) { st = 0; soff = 0; fbar = full_s; ph ^= 1u; }
#pragma unroll
            for (int r = 0; r < NN; r++)
#pragma unroll
                for (int j = 0; j < K1; j++) {
                    real acc = 0;
#pragma unroll
                    for (int m = 0; m < K1; m++) acc += A1[j * K1 + m] * a[r][m];
#pragma unroll
                    for (int m = 0; m < K1; m++) acc += B1[j * K1 + m] * b[r][m];
                    g[r * K1 + j] = (CP && cp1) ? a[r][j] : acc;
                }
        };

        real P3[S][N3V];                                                // v_1v_2-swept block of the previous v_3 cell, per pair
        int ov2_0 = c0 + s2 + 1; if (ov2_0 >= N2) ov2_0 -= N2;          // output v_2 cell of pair 0
        int io3 = s3 + 1; if (io3 >= N3) io3 -= N3;                     // output v_3 cell of the donor pair (j-1, j), j = 1
        // Output pointers advance by uniform strides only (no per-store index arithmetic): o3 = output v_3 cell and the
        // strip's first output v_2 cell, o2 walks the strip's pairs, the stores of a pair walk (j2, j1) on both v_3 rows.
        const long long wrap2 = (long long)N2 * cell2X, wrap3 = (long long)N3 * cell3X;
        const long long stepX = X, stepRow = rowX - (long long)(K1 - 1) * X;
        real* o3 = P.fout + (long long)(c * K1) * X + x0 + x + (long long)io3 * cell3X + (long long)ov2_0 * cell2X;

        // one v_3 cell: FIRST = the cell that only initialises the walk (no output); peeled so that the walk's loop carries no
        // `first cell?` branches
        auto cell = [&](auto first_t) {
            constexpr bool FIRST = decltype(first_t)::value;
            real g[2][N3V];
            real* o2 = o3;
            int ov2 = ov2_0;
#pragma unroll
            for (int m = 0; m <= S; m++) {
                if (m < nB) {
                    swept_box(g[m & 1]);
                    if (m >= 1) {
                        const int p = m - 1;
                        const real (&nxt)[N3V] = g[m & 1];
                        const real (&prv)[N3V] = g[(m - 1) & 1];
                        real t2[2 * NN], t3[2 * NN];                    // rows [A[j][.] | B[j][.]] of v_2 and v_3
                        if (T23S) {
#pragma unroll
                            for (int e = 0; e < NN; e++) {              // 2 NN is even: whole 2-value vectors
                                const real2 u2 = *reinterpret_cast<const real2*>(tab + 2 * e);
                                const real2 u3 = *reinterpret_cast<const real2*>(tab + 2 * NN + 2 * e);
                                t2[2 * e] = u2.x; t2[2 * e + 1] = u2.y; t3[2 * e] = u3.x; t3[2 * e + 1] = u3.y;
                            }
                        } else {
#pragma unroll
                            for (int jj = 0; jj < K1; jj++)
#pragma unroll
                                for (int l = 0; l < K1; l++) {
                                    t2[jj * 2 * K1 + l] = A2[jj * K1 + l]; t2[jj * 2 * K1 + K1 + l] = B2[jj * K1 + l];
                                    t3[jj * 2 * K1 + l] = A3[jj * K1 + l]; t3[jj * 2 * K1 + K1 + l] = B3[jj * K1 + l];
                                }
                        }
                        real* q[K1];                                    // store pointers, one per output v_3 row
#pragma unroll
                        for (int j3 = 0; j3 < K1; j3++) q[j3] = o2 + (long long)j3 * row3X;
#pragma unroll
                        for (int j2 = 0; j2 < K1; j2++)
#pragma unroll
                            for (int j1 = 0; j1 < K1; j1++) {
                                real h[K1];                             // v_2-swept values [j3] of this (j2, j1)
#pragma unroll
                                for (int j3 = 0; j3 < K1; j3++) {
                                    real acc = 0;
#pragma unroll
                                    for (int l = 0; l < K1; l++) acc += t2[j2 * 2 * K1 + l] * nxt[(j3 * K1 + l) * K1 + j1];
#pragma unroll
                                    for (int l = 0; l < K1; l++) acc += t2[j2 * 2 * K1 + K1 + l] * prv[(j3 * K1 + l) * K1 + j1];
                                    h[j3] = (CP && cp2) ? nxt[(j3 * K1 + j2) * K1 + j1] : acc;
                                }
                                if constexpr (!FIRST) {
#pragma unroll
                                    for (int j3 = 0; j3 < K1; j3++) {
                                        real acc = 0;
#pragma unroll
                                        for (int l = 0; l < K1; l++) acc += t3[j3 * 2 * K1 + l] * h[l];
#pragma unroll
                                        for (int l = 0; l < K1; l++) acc += t3[j3 * 2 * K1 + K1 + l] * P3[p][(l * K1 + j2) * K1 + j1];
                                        const real r = (CP && cp3) ? h[j3] : acc;
                                        if (active) __stcs(q[j3], r);
                                        q[j3] += (j1 == K1 - 1) ? stepRow : stepX;
                                    }
                                }
#pragma unroll
                                for (int j3 = 0; j3 < K1; j3++) P3[p][(j3 * K1 + j2) * K1 + j1] = h[j3];
                            }
                        o2 += cell2X;
                        if (++ov2 == N2) { ov2 = 0; o2 -= wrap2; }
                    }
                }
            }
            if constexpr (!FIRST) {
                o3 += cell3X;
                if (++io3 == N3) { io3 = 0; o3 -= wrap3; }
            }
        };
        cell(std::true_type{});
#pragma unroll 1
        for (int j = 1; j <= N3; j++) cell(std::false_type{});
    };
    if (anycp) body(std::true_type{});
    else body(std::false_type{});
}

template <int K1, int S, int WXT>
cudaError_t launch(sldg_ctx* c, const CUtensorMap& tm, const FV3Params& P, int threads, size_t smem)
{
    auto kern = sweep_fusedv3_kernel<K1, S, WXT>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const long long grid = (long long)P.ntiles * P.nstrips;
    if (grid > 0x7fffffffLL) return cudaErrorNotSupported;
    kern<<<(unsigned)grid, threads + (P.pw ? 32 : 0), smem, c->stream>>>(tm, P);
    return cudaGetLastError();
}

template <int K1>
cudaError_t dispatch(sldg_ctx* c, const CUtensorMap& tm, const FV3Params& P, int threads, size_t smem)
{
    switch (P.S) {
    case 1: return P.WX == 16 ? launch<K1, 1, 16>(c, tm, P, threads, smem) : launch<K1, 1, 0>(c, tm, P, threads, smem);
    case 2: return P.WX == 16 ? launch<K1, 2, 16>(c, tm, P, threads, smem) : launch<K1, 2, 0>(c, tm, P, threads, smem);
    case 3: return P.WX == 16 ? launch<K1, 3, 16>(c, tm, P, threads, smem) : launch<K1, 3, 0>(c, tm, P, threads, smem);
    case 4: return P.WX == 16 ? launch<K1, 4, 16>(c, tm, P, threads, smem) : launch<K1, 4, 0>(c, tm, P, threads, smem);
    case 5: return P.WX == 16 ? launch<K1, 5, 16>(c, tm, P, threads, smem) : launch<K1, 5, 0>(c, tm, P, threads, smem);
    }
    return cudaErrorNotSupported;
}

// strip size, ring depth and shared memory of a launch: every rule the launcher applies, so that a plan that passed
// the shape test never meets cudaErrorNotSupported
struct FV3Shape { int wx, threads, S, nstrips, slots; uint32_t slot_bytes; size_t smem; };

bool shape(const sldg_ctx* c, FV3Shape* o)
{
    const int K1 = c->K1;
    if (c->dx != 3 || c->dv != 3 || K1 > 2) return false;
    const long long D1 = c->D[3], D2 = c->D[4], D3 = c->D[5];
    const int N1 = c->cells[3], N2 = c->cells[4];
    if (D1 > 256 || ((c->X * (long long)sizeof(real)) & 15)) return false;
    if (c->X >= (1LL << 31) || D2 >= (1LL << 31) || D3 >= (1LL << 31)) return false;
    if (!c->dry && !sldg_encode_tiled()) return false;
    // x nodes per tile: rows of 128 B when the thread budget allows, never below 32 B
    int wx = c->opt_fv3_wx > 0 ? c->opt_fv3_wx : (int)(128 / sizeof(real));
    if (sizeof(real) == 4 && c->opt_fv3_wx <= 0) wx = 16;              // fp32: 64-byte rows (a 128-byte tile would need 2x the threads)
    while (wx * (int)sizeof(real) > 32 && (long long)wx * N1 > FV3_MAXT) wx /= 2;
    if ((long long)wx * N1 > FV3_MAXT || ((wx * (int)sizeof(real)) & 15) || wx > 256) return false;
    // strip size: fp64 at degree 1 keeps a (k+1)^3 block per pair in registers; with 4 pairs ptxas spills at the 168-register cap
    // of a 9..12-warp block (3 warps share a 16384-register sub-partition), with 3 it does not: measured on B200, cfg5, 28.1 -> 25.3 ms
    // although 7 strips re-read more halo cells than 5 (profiles/r3_fusedv3.md)
    int S = c->opt_fv3_strip > 0 ? c->opt_fv3_strip : ((sizeof(real) == 8 && K1 == 2) ? 3 : 4);
    if (S > FV3_MAXS) S = FV3_MAXS;
    if (S > N2) S = N2;
    int nstrips = (N2 + S - 1) / S;
    S = (N2 + nstrips - 1) / nstrips;                                  // strips of (nearly) equal size
    nstrips = (N2 + S - 1) / S;
    const uint32_t slot_bytes = (uint32_t)(((size_t)K1 * K1 * D1 * wx * sizeof(real) + 1023) / 1024 * 1024);
    auto smem_of = [&](int st) { return (size_t)st * slot_bytes + 16 * (size_t)st + (size_t)wx * (4 * K1 * K1 + 2) * sizeof(real) + 128; };
    // ring depth: measured on B200 (cfg4, 20 KB boxes) 6 slots beat the 11 that fit by 4-10 % (the deeper ring lets the
    // strips of an x tile drift apart, and their shared halo cells stop hitting in L2)
    // An explicit option value is honoured down to 2 slots (LAG = 1 in the kernel: tests/test_gpu_fusedv3.py runs 2 and 3);
    // the 4-slot floor applies to the automatic choice only.
    int slots = c->opt_fv3_slots > 0 ? c->opt_fv3_slots : (int)((120 * 1024) / slot_bytes);
    if (c->opt_fv3_slots <= 0 && slots < 4) slots = 4;
    if (slots < 2) slots = 2;
    while (slots > 2 && smem_of(slots) > 227 * 1024) slots--;
    if (smem_of(slots) > 227 * 1024) return false;
    if (o) { o->wx = wx; o->threads = (int)(((long long)wx * N1 + 31) / 32 * 32); o->S = S; o->nstrips = nstrips;
             o->slots = slots; o->slot_bytes = slot_bytes; o->smem = smem_of(slots); }
    return true;
}

}  // namespace

bool SLDG_SFX(sldg_fusedv3_shape)(const sldg_ctx* c) { return shape(c, nullptr); }

// t1, t2, t3: the shift tables of v_1, v_2, v_3 (one entry per x node).  cudaErrorNotSupported when the shape does not fit.
cudaError_t SLDG_SFX(sldg_launch_sweep_fusedv3)(sldg_ctx* c, const void* fin, void* fout, const ShiftTable& t1,
                                                const ShiftTable& t2, const ShiftTable& t3)
{
    FV3Shape sh;
    if (fin == fout || !shape(c, &sh)) return cudaErrorNotSupported;
    if ((((uintptr_t)fin) | ((uintptr_t)fout)) & 15) return cudaErrorNotSupported;
    SldgEncodeTiled enc = sldg_encode_tiled();
    if (!enc) return cudaErrorNotSupported;
    const int K1 = c->K1;
    const long long D1 = c->D[3], D2 = c->D[4], D3 = c->D[5];

    FV3Params P;
    P.fout = static_cast<real*>(fout);
    P.X = c->X; P.N1 = c->cells[3]; P.N2 = c->cells[4]; P.N3 = c->cells[5]; P.WX = sh.wx;
    P.S = sh.S; P.nstrips = sh.nstrips; P.ntiles = (int)((c->X + sh.wx - 1) / sh.wx);
    P.slots = sh.slots; P.slot_bytes = sh.slot_bytes; P.pw = c->opt_fv3_pw ? 1 : 0;
    P.t1 = t1; P.t2 = t2; P.t3 = t3;

    CUtensorMap tm;
    const cuuint64_t gdim[4] = {(cuuint64_t)c->X, (cuuint64_t)D1, (cuuint64_t)D2, (cuuint64_t)D3};
    const cuuint64_t gstr[3] = {(cuuint64_t)c->X * sizeof(real), (cuuint64_t)c->X * D1 * sizeof(real),
                                (cuuint64_t)c->X * D1 * D2 * sizeof(real)};
    const cuuint32_t box[4] = {(cuuint32_t)sh.wx, (cuuint32_t)D1, (cuuint32_t)K1, (cuuint32_t)K1};
    const cuuint32_t estr[4] = {1u, 1u, 1u, 1u};
    const CUtensorMapDataType dt = sizeof(real) == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32;
    if (enc(&tm, dt, 4, const_cast<void*>(fin), gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_NONE, sldg_l2_promotion(c->opt_fv_l2), CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return cudaErrorNotSupported;
    return K1 == 1 ? dispatch<1>(c, tm, P, sh.threads, sh.smem) : dispatch<2>(c, tm, P, sh.threads, sh.smem);
}
