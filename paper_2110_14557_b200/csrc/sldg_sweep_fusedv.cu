// sldg_sweep_fusedv.cu -- the v_1 AND v_2 sweeps of a v advection in ONE pass over f, sm_100a.
//
// eq. (3), reading B, applied twice in the order v_1, v_2 (E does not change during the v sweeps):
//     u_i <- A(alpha) u_{(i-s) mod N} + B(alpha) u_{(i-s-1) mod N},   delta = -E_d(x) dt / h_{v_d}  per x node.
// 16 B (fp64) of HBM traffic per value for TWO sweeps instead of 32 B.
//
//   f is seen as [planes q][D_2 = N_2 (k+1) rows][D_1 = N_1 (k+1) rows][X]  (X = all x nodes, contiguous; v_1 is the
//   fastest velocity axis, v_2 the next; q runs over everything above v_2).  Every shift of both sweeps is that of
//   the x node, so a thread that owns one x node keeps A_1, B_1, A_2, B_2 of that node in registers.
//   A block owns a tile of WX consecutive x nodes and ALL of v_1, and walks along v_2 (and on through `ppb`
//   consecutive planes: the rows of a tile are one arithmetic sequence in memory, and the tables do not change).
//   One 3-d TMA tensor copy (box WX x D_1 x RPS; RPS = k+1 rows = a whole v_2 cell at k <= 1, one row at k = 2) brings
//   [RPS][D_1][WX] into a slot of a ring of shared-memory stages;
//   thread 0 issues them between its own rows (two rows behind the consumers' releases, so it rarely waits),
//   full/empty mbarriers pace the ring, no __syncthreads in the loop.
//   A thread owns one (x node, v_1 cell): per v_2 row it reads the k+1 rows of its two v_1 donor cells from shared
//   memory (lanes run over x: conflict free) and applies A_1, B_1; after the k+1 rows of a v_2 cell it holds the
//   v_1-swept (k+1)^2 block, combines it with the previous block by A_2, B_2 (register walk, as in
//   sldg_sweep_walk.cu) and stores output cell (j + s_2 + 1) mod N_2 straight from registers (lanes over x:
//   coalesced WX * 8 B pieces).  The first block closes the periodic wrap: kept in registers for k <= 1, streamed
//   in once more (k+1 extra rows per plane, 1/N_2 of the reads) for k = 2.
//
// Arithmetic per value is identical (same operands, same order) to sweep_walk_kernel on v_1 then on v_2, so the
// fused and the unfused plans agree bit for bit.  Out of place only; degree <= 3; D_1 <= 256 (one TMA box);
// X * sizeof(real) a multiple of 16.
#include <type_traits>

#include "sldg_async.h"
#include "sldg_internal.h"
#include "sldg_real.h"
#include "sldg_tmap.h"

namespace {

using namespace sldg_async;

struct FVParams {
    real* fout;
    long long X, planes;
    int N1, N2, WX, stages, ppb, ntiles, cps;
    uint32_t stage_bytes;         // ring slot stride (>= D_1 * WX * sizeof(real), multiple of 128)
    ShiftTable t1, t2;
};

template <int K1> struct FVTraits {
    static constexpr bool KEEP = (K1 <= 2);        // first v_2 block kept in registers (else streamed in again)
    // threads per block.  Registers are split over the 4 SM sub-partitions: 16 warps leave 128 registers per thread
    // (what the (k+1)^2 blocks and four tables of k = 2 need), 20 warps 96.
    static constexpr int MAXT = (K1 <= 2) ? 640 : (K1 == 3) ? 512 : 256;   // k = 3: 8 warps, up to 255 registers
    // k = 2: A_2, B_2 of the tile's x nodes live in shared memory (rows [A_2[j][.] | B_2[j][.]], one padded record per
    // x node, read as 2-value vectors: lanes of equal x broadcast, different x fall on different banks); with all four
    // tables in registers the kernel spills (ncu: a third of the issue slots stalled on local loads).
    static constexpr bool T2S = (K1 >= 3);
    static constexpr int PAD = 2 * K1 * K1 + (K1 == 4 ? 6 : 4);        // record stride = 12 banks mod 32: conflict free
    // v_2 rows per tensor copy (= per ring slot).  Measured: a whole cell per copy is faster at k = 1 (cfg3 3.6 -> 3.0 ms:
    // half the barrier traffic), a row per copy at k = 2 (cfg2 4.3 against 5.0 ms with 36 KB copies).
    static constexpr int RPS = (K1 >= 3) ? 1 : K1;
};

template <int K1>
__global__ void __launch_bounds__(FVTraits<K1>::MAXT)
    sweep_fusedv_kernel(const __grid_constant__ CUtensorMap tmap, const FVParams P)
{
    constexpr int NN = K1 * K1;
    constexpr bool KEEP = FVTraits<K1>::KEEP;
    constexpr bool T2S = FVTraits<K1>::T2S;
    constexpr int PAD = FVTraits<K1>::PAD;
    constexpr int RPS = FVTraits<K1>::RPS, SPC = K1 / RPS;             // rows per ring slot, slots per v_2 cell
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    const int ST = P.stages, WX = P.WX, N1 = P.N1, N2 = P.N2;
    const int D1 = N1 * K1, D2 = N2 * K1;
    const uint32_t ring_s = smem_u32(smem_raw);
    const uint32_t full_s = ring_s + (uint32_t)ST * P.stage_bytes;      // ST full barriers, then ST empty barriers
    const uint32_t empty_s = full_s + (uint32_t)ST * 8u;

    const int t = threadIdx.x;
    const int NTR = (int)blockDim.x;                                    // whole warps
    const int LAG = ST >= 4 ? 2 : 1;                                    // the producer refills the slot of row i - LAG
    const int DEP = ST - LAG;                                           // rows in flight ahead of the consumers
    const int tile = (int)(blockIdx.x % (unsigned)P.ntiles);
    const int chunk = (int)(blockIdx.x / (unsigned)P.ntiles);
    const long long q0 = (long long)chunk * P.ppb;
    const int nq = (int)min((long long)P.ppb, P.planes - q0);
    const long long x0 = (long long)tile * WX;
    const int CPP = N2 + (KEEP ? 0 : 1);                                // v_2 cells streamed per plane
    // k <= 1: a ring slot holds `cps` whole v_2 cells; the block's cells are one run of rows, so the last slot may reach
    // past it (into the next plane, or zero-filled past the end of f) and is simply not read to the end
    const int cps = (RPS == K1) ? P.cps : 1;
    const int total = (RPS == K1) ? (nq * CPP + cps - 1) / cps : nq * CPP * SPC;   // ring slots this block streams

    if (t == 0) {
        for (int s = 0; s < ST; s++) { mbar_init(full_s + 8u * s, 1); mbar_init(empty_s + 8u * s, NTR / 32); }
        mbar_init_fence();
    }
    __syncthreads();

    // ---------------- producer (thread 0, between its own rows): one tensor copy (box WX x D_1 x RPS) per ring slot
    const uint32_t slot_bytes = (uint32_t)(RPS * cps) * (uint32_t)D1 * (uint32_t)WX * (uint32_t)sizeof(real);
    int pst = 0, pn = 0, pc = 0, psub = 0, pi = 0;
    long long prow0 = q0 * D2;                                          // first row of the producer's current plane
    auto produce = [&]() {
        if (pi >= total) return;
        if (pn > 0) mbar_wait(empty_s + 8u * pst, (uint32_t)((pn - 1) & 1));
        mbar_expect_tx(full_s + 8u * pst, slot_bytes);
        if constexpr (RPS == K1) {
            tma_load_3d(ring_s + (uint32_t)pst * P.stage_bytes, &tmap, (int)x0, 0, (int)(prow0 + (long long)pi * (K1 * cps)),
                        full_s + 8u * pst);
        } else {
            const int cc = (pc >= N2) ? 0 : pc;                         // k = 2: cell 0 of the plane once more
            tma_load_3d(ring_s + (uint32_t)pst * P.stage_bytes, &tmap, (int)x0, 0, (int)(prow0 + cc * K1 + psub * RPS),
                        full_s + 8u * pst);
            if (++psub == SPC) { psub = 0; if (++pc == CPP) { pc = 0; prow0 += D2; } }
        }
        if (++pst == ST) { pst = 0; pn++; }
        pi++;
    };
    if (t == 0)
        for (int i = 0; i < DEP; i++) produce();

    // ---------------- consumers
    const int c = t / WX, x = t - c * WX;
    const bool active = (c < N1) && (x0 + x < P.X);
    real A1[NN], B1[NN], A2[NN], B2[NN];
    int s1 = 0, s2 = 0;
    bool cp1 = false, cp2 = false;
#pragma unroll
    for (int m = 0; m < NN; m++) { A1[m] = B1[m] = A2[m] = B2[m] = 0; }
    if (active) {
        const long long idx = x0 + x;
        const int sv1 = __ldg(P.t1.S + idx), sv2 = __ldg(P.t2.S + idx);
        cp1 = (sv1 & SLDG_COPY_BIT) != 0; s1 = sv1 & SLDG_S_MASK;
        cp2 = (sv2 & SLDG_COPY_BIT) != 0; s2 = sv2 & SLDG_S_MASK;
        const real* ab1 = static_cast<const real*>(P.t1.AB) + idx * P.t1.strideIdx;
        const real* ab2 = static_cast<const real*>(P.t2.AB) + idx * P.t2.strideIdx;
#pragma unroll
        for (int m = 0; m < NN; m++) {
            A1[m] = __ldg(ab1 + m * P.t1.strideM); B1[m] = __ldg(ab1 + (NN + m) * P.t1.strideM);
            A2[m] = __ldg(ab2 + m * P.t2.strideM); B2[m] = __ldg(ab2 + (NN + m) * P.t2.strideM);
        }
    }
    int ia = 0, ib = 0;
    if (active) {
        ia = c - s1; if (ia < 0) ia += N1;
        ib = ia - 1; if (ib < 0) ib += N1;
    }
    real* const tab2 = reinterpret_cast<real*>(smem_raw + (size_t)ST * P.stage_bytes + 16 * (size_t)ST) + x * PAD;
    if (T2S) {
        if (c == 0) {
#pragma unroll
            for (int j = 0; j < K1; j++)
#pragma unroll
                for (int l = 0; l < K1; l++) { tab2[j * 2 * K1 + l] = A2[j * K1 + l]; tab2[j * 2 * K1 + K1 + l] = B2[j * K1 + l]; }
        }
        __syncthreads();
    }
    // the alpha == 0 copy selects are compiled out for warps none of whose x nodes has the copy bit (the usual case)
    const bool anycp = __any_sync(0xffffffffu, cp1 || cp2);

    const real* const ring = reinterpret_cast<const real*>(smem_raw);
    const real* const pa0 = ring + ia * K1 * WX + x;                    // donor rows of stage 0
    const real* const pb0 = ring + ib * K1 * WX + x;
    const int stage_vals = (int)(P.stage_bytes / sizeof(real));
    const bool warp_lead = (t & 31) == 0;
    const long long X = P.X;
    const long long rowX = (long long)D1 * X;                          // one v_2 row of a plane, in values
    const long long cellX = (long long)K1 * rowX, planeX = (long long)D2 * rowX;

    int csub = 0;                                                      // cell inside the current ring slot (k <= 1)
    int st = 0, soff = 0;                                              // ring slot of the next row, its offset in values
    uint32_t ph = 0, fbar = full_s;

    auto body = [&](auto cpt) {
        constexpr bool CP = decltype(cpt)::value;
        // one v_2 cell of the ring -> the v_1-swept (k+1)^2 block [j2][j1] of this thread's v_1 cell
        auto swept_cell = [&](real* g) {
            const int rowvals = D1 * WX;
#pragma unroll
            for (int j2 = 0; j2 < K1; j2++) {
                const int jr = j2 % RPS;                                // row inside the ring slot (of its cell)
                if (jr == 0 && csub == 0) {
                    if (t == 0) produce();
                    mbar_wait(fbar, ph);
                }
                const int ro = soff + (csub * RPS + jr) * rowvals;
                real a[K1], b[K1];
#pragma unroll
                for (int m = 0; m < K1; m++) { a[m] = pa0[ro + m * WX]; b[m] = pb0[ro + m * WX]; }
                const bool last = jr == RPS - 1 && csub == cps - 1;
                if (last) {                                             // the slot is read: hand it back
                    // The slot is refilled by the ASYNC proxy (TMA) once every warp has arrived: the generic-proxy reads
                    // above must be ordered before that write by a proxy fence.  Without it single lanes read a row of the
                    // NEXT copy (seen at full size only, where long multi-plane walks let the warps drift apart: a few
                    // wrong values per launch, caught by the mass check of tests/test_gpu_fullsize.py).
                    fence_async_smem();
                    __syncwarp();
                    if (warp_lead) mbar_arrive(fbar + 8u * (uint32_t)ST);
                }
#pragma unroll
                for (int j = 0; j < K1; j++) {
                    real acc = 0;
#pragma unroll
                    for (int m = 0; m < K1; m++) acc += A1[j * K1 + m] * a[m];
#pragma unroll
                    for (int m = 0; m < K1; m++) acc += B1[j * K1 + m] * b[m];
                    g[j2 * K1 + j] = (CP && cp1) ? a[j] : acc;
                }
                if (last) {
                    st++; soff += stage_vals; fbar += 8u;
                    if (st == ST) { st = 0; soff = 0; fbar = full_s; ph ^= 1u; }
                }
            }
            if (RPS == K1) { if (++csub == cps) csub = 0; }
        };
        // output cell *o <- A_2 nxt + B_2 prev   (blocks are [j2][j1])
        auto emit = [&](real* o, const real (&nxt)[NN], const real (&prev)[NN]) {
#pragma unroll
            for (int j2 = 0; j2 < K1; j2++) {
                real ab[2 * K1];                                       // A_2[j2][.] then B_2[j2][.]
                if (T2S) {
#pragma unroll
                    for (int l = 0; l < K1; l++) {                      // 2 K1 is even: whole 2-value vectors
                        const real2 v = *reinterpret_cast<const real2*>(tab2 + j2 * 2 * K1 + 2 * l);
                        ab[2 * l] = v.x; ab[2 * l + 1] = v.y;
                    }
                } else {
#pragma unroll
                    for (int l = 0; l < K1; l++) { ab[l] = A2[j2 * K1 + l]; ab[K1 + l] = B2[j2 * K1 + l]; }
                }
                real* p = o;
#pragma unroll
                for (int j1 = 0; j1 < K1; j1++) {
                    real acc = 0;
#pragma unroll
                    for (int l = 0; l < K1; l++) acc += ab[l] * nxt[l * K1 + j1];
#pragma unroll
                    for (int l = 0; l < K1; l++) acc += ab[K1 + l] * prev[l * K1 + j1];
                    const real r = (CP && cp2) ? nxt[j2 * K1 + j1] : acc;
                    if (active) __stcs(p, r);
                    p += X;
                }
                o += rowX;
            }
        };

        for (int iq = 0; iq < nq; iq++) {
            real* const oplane = P.fout + (q0 + iq) * planeX + (long long)(c * K1) * X + x0 + x;
            int io2 = s2 + 1; if (io2 >= N2) io2 -= N2;                // output v_2 cell of the current donor pair
            real* o = oplane + (long long)io2 * cellX;
            real u[2][NN], first[KEEP ? NN : 1];
            auto get = [&](real (&dst)[NN], int jc) {                  // v_1-swept block of v_2 cell jc (N_2 = cell 0 again)
                if (!KEEP || jc < N2) {
                    swept_cell(dst);
                } else {
#pragma unroll
                    for (int m = 0; m < NN; m++) dst[m] = first[KEEP ? m : 0];
                }
            };
            auto step = [&](real (&nxt)[NN], const real (&prev)[NN], int jc) {
                get(nxt, jc);
                emit(o, nxt, prev);
                o += cellX;
                if (++io2 == N2) { io2 = 0; o -= planeX; }
            };
            get(u[0], 0);
            if (KEEP) {
#pragma unroll
                for (int m = 0; m < NN; m++) first[KEEP ? m : 0] = u[0][m];
            }
            // two cells per trip so that the blocks alternate between u[0] and u[1] without register moves
#pragma unroll 1
            for (int jc = 1; jc <= N2; jc += 2) {
                step(u[1], u[0], jc);
                if (jc + 1 > N2) {                                      // odd N_2: the pair ends on u[1]; not reached again
                    break;
                }
                step(u[0], u[1], jc + 1);
            }
        }
    };
    if (anycp) body(std::true_type{});
    else body(std::false_type{});
}

template <int K1>
cudaError_t launch(sldg_ctx* c, const CUtensorMap& tm, const FVParams& P, int threads, size_t smem)
{
    auto kern = sweep_fusedv_kernel<K1>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const long long nchunks = (P.planes + P.ppb - 1) / P.ppb;
    const long long grid = nchunks * P.ntiles;
    if (grid > 0x7fffffffLL) return cudaErrorNotSupported;
    kern<<<(unsigned)grid, threads, smem, c->stream>>>(tm, P);
    return cudaGetLastError();
}

}  // namespace

// The shape rules of the fused v_1+v_2 pass.  wx / threads / stage_bytes of the launch are returned when non-null.
bool SLDG_SFX(sldg_fusedv_shape)(const sldg_ctx* c, int* wx_out, int* threads_out)
{
    const int K1 = c->K1;
    if (c->dx < 2 || K1 > 4) return false;
    const long long D1 = c->D[c->dx];
    if (D1 > 256 || c->cells[c->dx] < 1) return false;
    if ((c->X * (long long)sizeof(real)) & 15) return false;
    // 32-bit tensor coordinates, and the driver's tensor-map encoder must be reachable (no libcuda link)
    if (c->X >= (1LL << 31) || c->V / D1 >= (1LL << 31) || (!c->dry && !sldg_encode_tiled())) return false;
    const int cap = (K1 <= 2) ? FVTraits<1>::MAXT : (K1 == 3) ? FVTraits<3>::MAXT : FVTraits<4>::MAXT;  // threads allowed
    // x nodes per tile: rows of 128 B when the thread budget allows, else 64 B; never below 32 B
    int wx = c->opt_fv_wx > 0 ? c->opt_fv_wx : (int)(128 / sizeof(real));
    if (K1 == 4 && c->opt_fv_wx <= 0) {
        // k = 3: one block of at most 256 threads per SM (212 registers): fill it -- as many x nodes as fit, whole 16 B
        const int q16 = 16 / (int)sizeof(real);
        wx = (int)(cap / c->cells[c->dx]) / q16 * q16;
        if (wx > 256 / (int)sizeof(real)) wx = 256 / (int)sizeof(real);
        if (wx < 32 / (int)sizeof(real)) wx = 32 / (int)sizeof(real);
    }
    while (wx * (int)sizeof(real) > 32 && (long long)wx * c->cells[c->dx] > cap) wx /= 2;
    if ((long long)wx * c->cells[c->dx] > cap) return false;
    if ((wx * (int)sizeof(real)) & 15) return false;
    if (wx > 256) return false;
    if (wx_out) *wx_out = wx;
    if (threads_out) *threads_out = (int)(((long long)wx * c->cells[c->dx] + 31) / 32 * 32);
    return true;
}

// t1, t2: the shift tables of v_1 and v_2 (one entry per x node).  cudaErrorNotSupported when the shape does not fit.
cudaError_t SLDG_SFX(sldg_launch_sweep_fusedv)(sldg_ctx* c, const void* fin, void* fout, const ShiftTable& t1,
                                               const ShiftTable& t2)
{
    int wx = 0, threads = 0;
    if (fin == fout || !SLDG_SFX(sldg_fusedv_shape)(c, &wx, &threads)) return cudaErrorNotSupported;
    if ((((uintptr_t)fin) | ((uintptr_t)fout)) & 15) return cudaErrorNotSupported;
    SldgEncodeTiled enc = sldg_encode_tiled();
    if (!enc) return cudaErrorNotSupported;
    const int K1 = c->K1, a1 = c->dx, a2 = c->dx + 1;
    const long long D1 = c->D[a1], D2 = c->D[a2];
    const long long planes = c->V / (D1 * D2);
    const long long rows = D2 * planes;
    if (c->X >= (1LL << 31) || rows >= (1LL << 31)) return cudaErrorNotSupported;

    FVParams P;
    P.fout = static_cast<real*>(fout);
    P.X = c->X; P.planes = planes; P.N1 = c->cells[a1]; P.N2 = c->cells[a2]; P.WX = wx;
    P.ntiles = (int)((c->X + wx - 1) / wx);
    int cps = (K1 >= 3) ? 1 : (c->opt_fv_cps > 0 ? c->opt_fv_cps : 1);   // v_2 cells per tensor copy (k <= 1)
    if (cps > c->cells[a2]) cps = c->cells[a2];
    P.cps = cps;
    const int rps = (K1 >= 3 ? 1 : K1) * cps;                           // rows per ring slot
    P.stage_bytes = (uint32_t)(((size_t)rps * D1 * wx * sizeof(real) + 1023) / 1024 * 1024);
    // ring depth: about opt_fv_inflight bytes in flight per SM
    const size_t regs_blocks = (K1 <= 2) ? (size_t)(65536 / 96) / threads : 1;
    size_t bps = regs_blocks < 1 ? 1 : regs_blocks;
    if (bps > 4) bps = 4;
    int stages = c->opt_fv_stages > 0 ? c->opt_fv_stages : (int)((size_t)c->opt_fv_inflight * (K1 <= 2 ? 4 : 3) / 3 / bps / P.stage_bytes);   // measured: 96 KB at k <= 1, 72 KB at k = 2
    if (stages < 3) stages = 3;
    if (stages > 24) stages = 24;
    auto smem_of = [&](int st) { return (size_t)st * P.stage_bytes + 16 * (size_t)st + (size_t)wx * (2 * K1 * K1 + 6) * sizeof(real) + 128; };
    while (stages > 2 && smem_of(stages) > 227 * 1024) stages--;
    if (smem_of(stages) > 227 * 1024) return cudaErrorNotSupported;
    P.stages = stages;
    // planes per block: long walks (tables and pipeline fill amortised), yet enough blocks to fill the GPU evenly
    long long ppb = c->opt_fv_ppb > 0 ? c->opt_fv_ppb : 1;
    if (c->opt_fv_ppb <= 0) {
        const long long slots = (long long)c->sm_count * (long long)bps;
        while (ppb < planes && D2 * ppb < 512 && (planes / (ppb * 2)) * P.ntiles >= 8 * slots) ppb *= 2;
    }
    if (ppb > planes) ppb = planes;
    P.ppb = (int)ppb;
    P.t1 = t1; P.t2 = t2;

    CUtensorMap tm;
    const cuuint64_t gdim[3] = {(cuuint64_t)c->X, (cuuint64_t)D1, (cuuint64_t)rows};
    const cuuint64_t gstr[2] = {(cuuint64_t)c->X * sizeof(real), (cuuint64_t)c->X * D1 * sizeof(real)};
    const cuuint32_t box[3] = {(cuuint32_t)wx, (cuuint32_t)D1, (cuuint32_t)rps};
    const cuuint32_t estr[3] = {1u, 1u, 1u};
    const CUtensorMapDataType dt = sizeof(real) == 8 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT64 : CU_TENSOR_MAP_DATA_TYPE_FLOAT32;
    const CUtensorMapL2promotion l2 = sldg_l2_promotion(c->opt_fv_l2);
    if (enc(&tm, dt, 3, const_cast<void*>(fin), gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_NONE, l2, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return cudaErrorNotSupported;
    const size_t smem = smem_of(stages);
    switch (K1) {
    case 1: return launch<1>(c, tm, P, threads, smem);
    case 2: return launch<2>(c, tm, P, threads, smem);
    case 3: return launch<3>(c, tm, P, threads, smem);
    case 4: return launch<4>(c, tm, P, threads, smem);
    }
    return cudaErrorNotSupported;
}
