// sldg_sweep_fused_cell.cu -- the x_1 and x_2 sweeps of an x advection in ONE pass over f, sm_100a: the production
// kernel of the fused pass (sldg_sweep_fused.cu keeps the node-per-thread variant as the fallback).
//
// eq. (3), reading B, applied twice: first along x_1 (axis 0, contiguous), then along x_2 (axis 1).  The x
// sweeps commute and act on different axes, so both are applied while a value passes through the SM once:
// 16 B of HBM traffic per value for TWO sweeps.
//
// The array is seen as [planes q][N_1 cells][k+1 rows][D_0] with a row = one contiguous x_1 line, so the k+1 rows
// of CR consecutive x_2 cells of one plane are ONE contiguous chunk.  A block owns PB planes:
//
//   plane leader:  cp.async.bulk global -> shared (1-D TMA, mbarrier complete_tx) of its plane's chunks into a
//                  ring of input stages, issued `stages` chunks ahead: the HBM latency is covered by bytes in
//                  flight, not by occupancy or registers;
//   every thread:  owns ONE x_1 CELL of one plane.  Per x_2 cell it reads its two x_1 donor cells of each of the
//                  k+1 rows from shared memory (2 shared loads per value instead of 2(k+1) with a thread per
//                  node), applies A_1, B_1, and then WALKS along x_2 exactly like sldg_sweep_walk.cu with a
//                  (k+1) x (k+1) block of x_1-swept values in registers (previous cell kept, first cell kept for
//                  the periodic wrap), writing output cell (j + s_2 + 1) mod N_1 into a shared output stage;
//   plane leader:  cp.async.bulk shared -> global of the CR output cells (two copies when they wrap around).
//
// One __syncthreads per chunk releases the input stage and publishes the output stage.  Every value is read once
// and written once.  The shift of x_1 depends on the plane's v_1 node, that of x_2 on its v_2 node.  Out of place
// only (fin != fout); the k+1 rows of a cell must be a multiple of 16 bytes (rule of the bulk copies).
#include "sldg_async.h"
#include "sldg_internal.h"
#include "sldg_real.h"

namespace {

using namespace sldg_async;

struct CellParams {
    const real* fin;
    real* fout;
    long long planes;             // prod of D_b, b >= 2
    int N0, N1, PB, CR, stages;   // cells along x_1, x_2; planes per block; x_2 cells per chunk; input stages
    long long sdiv0, sdiv1;       // shift index of plane q: (q / sdiv) % smod, per axis
    long long smod0, smod1;
    ShiftTable t0, t1;
};

constexpr int OST = 2;            // output stages

template <int K1> struct CellV {
    real v[K1];
    __device__ __forceinline__ void load(const real* p)
    {
        if constexpr (K1 % 2 == 0) {
#pragma unroll
            for (int j = 0; j < K1; j += 2) {
                real2 t = *reinterpret_cast<const real2*>(p + j);
                v[j] = t.x; v[j + 1] = t.y;
            }
        } else {
#pragma unroll
            for (int j = 0; j < K1; j++) v[j] = p[j];
        }
    }
    __device__ __forceinline__ void store(real* p) const
    {
        if constexpr (K1 % 2 == 0) {
#pragma unroll
            for (int j = 0; j < K1; j += 2) *reinterpret_cast<real2*>(p + j) = make_real2(v[j], v[j + 1]);
        } else {
#pragma unroll
            for (int j = 0; j < K1; j++) p[j] = v[j];
        }
    }
};

// DBL: the sweep pair is applied TWICE (x_1, x_2, x_1, x_2 with the same tables): the second x half step of a Strang
// step followed by the first x half step of the next one (same time increment, nothing in between), in one pass.
// The first pair's output cells go to a shared "mid" stage in the layout of an input chunk instead of to global
// memory; after a block barrier the same threads read them as the donors of the second x_1 sweep and run a second
// x_2 walk (its own previous / first block).  The first pair emits its cells in cyclic order starting at cell
// s_2 + 1, which is all a periodic walk needs, so the second pair's outputs trail by one cell and the wrap cell joins
// the last group.  Same operands and order as two launches of the single pass: bit-identical.
// CPS = false: no entry of the two shift tables has alpha == 0 (the host knows): the copy selects are compiled out.
template <int K1, int MINB, bool DBL, bool CPS>
__global__ void __launch_bounds__(128, MINB) sweep_fused_cell_kernel(const CellParams P)
{
    constexpr int NN = K1 * K1;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int N0 = P.N0, N1 = P.N1, D0 = N0 * K1, CR = P.CR, ST = P.stages;
    const int PC = CR * K1 * D0;                       // doubles of one plane's chunk
    const int SS = P.PB * PC;                          // doubles of one stage
    real* const sin_ = reinterpret_cast<real*>(smem_raw);
    const int PCO = DBL ? (CR + 1) * K1 * D0 : PC;      // doubles of one plane's output group (DBL: + the wrap cell)
    const int SSO = P.PB * PCO;                        // doubles of one output stage
    real* const smid = sin_ + (size_t)ST * SS;         // DBL: the first pair's output group, read back as input
    real* const sout = smid + (DBL ? SS : 0);
    const uint32_t sin_s = smem_u32(sin_), sout_s = smem_u32(sout);
    const uint32_t bars_s = (smem_u32(sout + (size_t)OST * SSO) + 7u) & ~7u;

    const int t = threadIdx.x;
    const int pl = t / N0, i = t - pl * N0;
    const long long q0 = (long long)blockIdx.x * P.PB;
    const long long q = q0 + pl;
    const bool live = q < P.planes && pl < P.PB;
    const bool leader = live && i == 0;
    const int nlive = (int)min((long long)P.PB, P.planes - q0);
    const long long qq = live ? q : P.planes - 1;      // dead threads shadow the last plane (no copies, no stores)
    const long long D1 = (long long)N1 * K1;
    const real* const gin = P.fin + qq * D1 * D0;
    real* const gout = P.fout + qq * D1 * D0;
    const int NCH = 1 + (N1 - 1 + CR - 1) / CR;        // input chunks: cell 0 alone, then CR cells each
    const uint32_t cell_bytes = (uint32_t)(K1 * D0) * (uint32_t)sizeof(real);

    auto issue_load = [&](int j) {                     // plane leaders only
        if (leader && j < NCH) {
            const int st = j % ST;
            const int c0 = (j == 0) ? 0 : (j - 1) * CR + 1;
            const int nc = (j == 0) ? 1 : min(CR, N1 - c0);
            const uint32_t bar = bars_s + (uint32_t)st * 8u;
            mbar_expect_tx(bar, nc * cell_bytes);
            bulk_load(sin_s + (uint32_t)(st * SS + pl * PC) * (uint32_t)sizeof(real), gin + (long long)c0 * K1 * D0, nc * cell_bytes, bar);
        }
    };

    if (t == 0) {
        for (int st = 0; st < ST; st++) mbar_init(bars_s + (uint32_t)st * 8u, nlive);
        mbar_init_fence();
    }
    __syncthreads();
    for (int j = 0; j < ST; j++) issue_load(j);

    // ---- x_1: A_1, B_1 and the offsets of the two donor cells inside a row
    real A1[NN], B1[NN];
    int oa, ob;
    bool cp1;
    {
        const long long idx = (qq / P.sdiv0) % P.smod0;
        const int sv = __ldg(P.t0.S + idx);
        cp1 = (sv & SLDG_COPY_BIT) != 0;
        const int s = sv & SLDG_S_MASK;
        int ia = i - s; if (ia < 0) ia += N0;
        int ib = ia - 1; if (ib < 0) ib += N0;
        oa = ia * K1; ob = ib * K1;
        const real* ab = static_cast<const real*>(P.t0.AB) + idx * P.t0.strideIdx;
#pragma unroll
        for (int m = 0; m < NN; m++) {
            A1[m] = __ldg(ab + m * P.t0.strideM);
            B1[m] = __ldg(ab + (NN + m) * P.t0.strideM);
        }
    }
    // ---- x_2: A_2, B_2, shift
    real A2[NN], B2[NN];
    int s2;
    bool cp2;
    {
        const long long idx = (qq / P.sdiv1) % P.smod1;
        const int sv = __ldg(P.t1.S + idx);
        cp2 = (sv & SLDG_COPY_BIT) != 0;
        s2 = sv & SLDG_S_MASK;
        const real* ab = static_cast<const real*>(P.t1.AB) + idx * P.t1.strideIdx;
#pragma unroll
        for (int m = 0; m < NN; m++) {
            A2[m] = __ldg(ab + m * P.t1.strideM);
            B2[m] = __ldg(ab + (NN + m) * P.t1.strideM);
        }
    }

    // x_1-swept (k+1) x (k+1) block [x_2 node j2][x_1 node j1] of this thread's cell from the k+1 rows at `rows`
    auto swept = [&](const real* rows, real (&N)[NN]) {
#pragma unroll
        for (int j2 = 0; j2 < K1; j2++) {
            const real* row = rows + j2 * D0;
            CellV<K1> a, b;
            a.load(row + oa);
            b.load(row + ob);
#pragma unroll
            for (int j1 = 0; j1 < K1; j1++) {
                real acc = 0;
#pragma unroll
                for (int m = 0; m < K1; m++) acc += A1[j1 * K1 + m] * a.v[m];
#pragma unroll
                for (int m = 0; m < K1; m++) acc += B1[j1 * K1 + m] * b.v[m];
                N[j2 * K1 + j1] = (CPS && cp1) ? a.v[j1] : acc;
            }
        }
    };

    // the x_1-swept first cell closes the periodic wrap at the end of the walk: in registers for k <= 2, parked in
    // shared memory (one column per thread, conflict free) for k = 3 where the four matrices fill the register file
    constexpr bool FS = K1 >= 4;
    static_assert(!(DBL && K1 >= 4), "the double pass keeps both walks in registers: degree <= 2");
    real* const first_s = reinterpret_cast<real*>(smem_raw + (((size_t)(ST + OST) * SS * sizeof(real) + 8 * ST + 31) & ~(size_t)15));
    real first[FS ? 1 : NN], prev[NN];
    // chunk 0: cell 0 alone
    mbar_wait(bars_s, 0u);
    swept(sin_ + pl * PC, prev);
#pragma unroll
    for (int m = 0; m < NN; m++) {
        if constexpr (FS) first_s[m * blockDim.x + t] = prev[m];
        else first[m] = prev[m];
    }
    fence_async_smem();                                // generic-proxy reads of stage 0 -> its refill by the async proxy
    __syncthreads();
    issue_load(ST);

    // output cell <- A_2 nxt + B_2 prev, its k+1 rows written at `orow` (row stride D0)
    auto emit = [&](real* orow, const real (&nxt)[NN], const real (&prv)[NN]) {
#pragma unroll
        for (int j2 = 0; j2 < K1; j2++) {
            CellV<K1> r;
#pragma unroll
            for (int j1 = 0; j1 < K1; j1++) {
                real acc = 0;
#pragma unroll
                for (int l = 0; l < K1; l++) acc += A2[j2 * K1 + l] * nxt[l * K1 + j1];
#pragma unroll
                for (int l = 0; l < K1; l++) acc += B2[j2 * K1 + l] * prv[l * K1 + j1];
                r.v[j1] = (CPS && cp2) ? nxt[j2 * K1 + j1] : acc;
            }
            r.store(orow + j2 * D0);
        }
    };

    const int H = (N1 + CR - 1) / CR;                  // output groups of CR cells
    int io0 = s2 + 1; if (io0 >= N1) io0 -= N1;        // first output cell of the group (of the first pair)
    int io2 = io0 + s2 + 1; if (io2 >= N1) io2 -= N1;  // DBL: first output cell of the second pair's next group
    real first2[DBL ? NN : 1], prev2[DBL ? NN : 1], alt2[DBL ? NN : 1], alt[NN];
    for (int h = 0; h < H; h++) {
        const int j = h + 1;                           // input chunk that feeds this group
        const int st = j % ST;
        const int nin = min(CR, N1 - 1 - h * CR);      // cells of that chunk (<= 0: none, the wrap cell is `first`)
        const int nout = min(CR, N1 - h * CR);
        if (nin > 0) mbar_wait(bars_s + (uint32_t)st * 8u, (uint32_t)((j / ST) & 1));
        const real* ibase = sin_ + st * SS + pl * PC;
        real* obase = (DBL ? smid : sout + (h & 1) * SS) + pl * PC + i * K1;
        // the walk alternates between `prev` and `alt` (two cells per trip: no register moves); an odd tail copies once
        auto cell1 = [&](int e, real (&nx)[NN], const real (&pv)[NN]) {
            if (e < nin) swept(ibase + e * K1 * D0, nx);
            else {
#pragma unroll
                for (int m = 0; m < NN; m++) {
                    if constexpr (FS) nx[m] = first_s[m * blockDim.x + t];
                    else nx[m] = first[m];
                }
            }
            emit(obase + e * K1 * D0, nx, pv);
        };
        {
            int e = 0;
            for (; e + 1 < nout; e += 2) { cell1(e, alt, prev); cell1(e + 1, prev, alt); }
            if (e < nout) {
                cell1(e, alt, prev);
#pragma unroll
                for (int m = 0; m < NN; m++) prev[m] = alt[m];
            }
        }
        int ncells = nout;                             // cells the leader stores for this group
        if constexpr (DBL) {
            fence_async_smem();                        // the generic-proxy reads of the input stage -> its refill by the async proxy
            __syncthreads();                           // the mid stage is complete, the input stage is free
            issue_load(j + ST);
            real* o2 = sout + (h & 1) * SSO + pl * PCO + i * K1;
            ncells = 0;
            auto cell2 = [&](int e, real (&nx)[DBL ? NN : 1], const real (&pv)[DBL ? NN : 1]) {
                swept(smid + pl * PC + e * K1 * D0, nx);
                emit(o2 + ncells * K1 * D0, nx, pv);
                ncells++;
            };
            int e = 0;
            if (h == 0) {                              // the first cell of the second walk only initialises it
                swept(smid + pl * PC, prev2);
#pragma unroll
                for (int m = 0; m < NN; m++) first2[DBL ? m : 0] = prev2[DBL ? m : 0];
                e = 1;
            }
            for (; e + 1 < nout; e += 2) { cell2(e, alt2, prev2); cell2(e + 1, prev2, alt2); }
            if (e < nout) {
                cell2(e, alt2, prev2);
#pragma unroll
                for (int m = 0; m < NN; m++) prev2[DBL ? m : 0] = alt2[DBL ? m : 0];
            }
            if (h == H - 1) {                          // the periodic wrap of the second walk
                emit(o2 + ncells * K1 * D0, first2, prev2);
                ncells++;
            }
        }
        fence_async_smem();                            // generic-proxy writes of the output stage -> async proxy
        if (leader) bulk_wait_read<0>();               // the store of group h-1 has left its output stage
        __syncthreads();
        if (leader && ncells > 0) {
            const uint32_t src = sout_s + (uint32_t)((h & 1) * SSO + pl * PCO) * (uint32_t)sizeof(real);
            const int ofirst = DBL ? io2 : io0;
            const int n1 = min(ncells, N1 - ofirst);
            bulk_store(gout + (long long)ofirst * K1 * D0, src, (uint32_t)n1 * cell_bytes);
            if (ncells > n1) bulk_store(gout, src + (uint32_t)n1 * cell_bytes, (uint32_t)(ncells - n1) * cell_bytes);
            bulk_commit();
        }
        if constexpr (!DBL) issue_load(j + ST);
        io0 += CR; if (io0 >= N1) io0 -= N1;
        io2 += ncells; if (io2 >= N1) io2 -= N1;
    }
    if (leader) bulk_wait_read<0>();                   // shared memory must outlive the bulk stores reading it
}

template <int K1, int MINB, bool DBL>
cudaError_t launch(sldg_ctx* c, const CellParams& P, int threads, size_t smem, bool any_copy)
{
    auto kern = any_copy ? sweep_fused_cell_kernel<K1, MINB, DBL, true> : sweep_fused_cell_kernel<K1, MINB, DBL, false>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const long long grid = (P.planes + P.PB - 1) / P.PB;
    if (grid > 0x7fffffffLL) return cudaErrorNotSupported;
    kern<<<(unsigned)grid, threads, smem, c->stream>>>(P);
    return cudaGetLastError();
}

}  // namespace

// g0, g1: geometry of axis 0 and axis 1.  Returns cudaErrorNotSupported when the shape does not fit (the caller
// falls back to the node-per-thread fused kernel, then to separate sweeps).
static cudaError_t launch_cell(sldg_ctx* c, const void* fin, void* fout, const SweepGeom& g0, const SweepGeom& g1,
                               const ShiftTable& t0, const ShiftTable& t1, bool dbl, bool any_copy)
{
    if (g1.outer == 0) return cudaSuccess;
    const long long D0 = (long long)g0.N * g0.K1, D1 = (long long)g1.N * g1.K1;
    const int K1 = g0.K1;
    if (fin == fout || g1.inner != D0 || g0.mode != 0 || g1.mode != 0 || g0.sdiv % D1 != 0) return cudaErrorNotSupported;
    if (K1 > 4 || (((long long)K1 * D0 * sizeof(real)) & 15) || g0.N > 128) return cudaErrorNotSupported;
    if (dbl && K1 > 3) return cudaErrorNotSupported;
    if ((((uintptr_t)fin) | ((uintptr_t)fout)) & 15) return cudaErrorNotSupported;
    CellParams P;
    P.fin = static_cast<const real*>(fin); P.fout = static_cast<real*>(fout); P.planes = g1.outer;
    P.N0 = g0.N; P.N1 = g1.N;
    long long PB = c->opt_cell_threads / g0.N;
    if (PB < 1) PB = 1;
    if (PB > P.planes) PB = P.planes;
    const long long cellb = (long long)K1 * D0 * sizeof(real);            // bytes of one x_2 cell of one plane
    // Measured on B200 (cfg2-5): 64-thread blocks, 2 input stages of about 9 KB each, i.e. many small resident
    // blocks, reach the copy rate; larger stages or deeper rings lose occupancy and run slower.
    long long CR = c->opt_cell_rows > 0 ? c->opt_cell_rows : c->opt_cell_bytes / (PB * cellb);
    if (CR < 1) CR = 1;
    if (CR > g1.N) CR = g1.N;
    int stages = c->opt_cell_stages;
    const size_t smem_max = 227 * 1024;
    auto smem_of = [&](long long pb, long long cr, int st) {
        if (dbl) return (size_t)(st + 1) * pb * cr * cellb + (size_t)OST * pb * (cr + 1) * cellb + 8 * st + 48;
        return (size_t)(st + OST) * pb * cr * cellb + 8 * st + 48 + (K1 >= 4 ? (size_t)pb * g0.N * K1 * K1 * sizeof(real) : 0);
    };
    while (smem_of(PB, CR, stages) > smem_max && CR > 1) CR--;
    while (smem_of(PB, CR, stages) > smem_max && stages > 2) stages--;
    while (smem_of(PB, CR, stages) > smem_max && PB > 1) PB--;
    if (smem_of(PB, CR, stages) > smem_max) return cudaErrorNotSupported;
    P.PB = (int)PB; P.CR = (int)CR; P.stages = stages;
    P.sdiv0 = g0.sdiv / D1; P.smod0 = g0.smod;       // axis-0 lines are numbered row + D_1 * plane
    P.sdiv1 = g1.sdiv; P.smod1 = g1.smod;
    P.t0 = t0; P.t1 = t1;
    const int threads = (int)(PB * g0.N);
    const size_t smem = smem_of(PB, CR, stages);
    if (dbl) {
        switch (K1) {
        case 1: return launch<1, 4, true>(c, P, threads, smem, any_copy);
        case 2: return launch<2, 4, true>(c, P, threads, smem, any_copy);
        case 3: return launch<3, 2, true>(c, P, threads, smem, any_copy);
        }
        return cudaErrorNotSupported;
    }
    switch (K1) {
    case 1: return launch<1, 4, false>(c, P, threads, smem, any_copy);
    case 2: return launch<2, 4, false>(c, P, threads, smem, any_copy);
    case 3: return launch<3, 3, false>(c, P, threads, smem, any_copy);
    case 4: return launch<4, 2, false>(c, P, threads, smem, any_copy);
    }
    return cudaErrorNotSupported;
}

cudaError_t SLDG_SFX(sldg_launch_sweep_fused_cell)(sldg_ctx* c, const void* fin, void* fout, const SweepGeom& g0,
                                                   const SweepGeom& g1, const ShiftTable& t0, const ShiftTable& t1, int any_copy)
{
    return launch_cell(c, fin, fout, g0, g1, t0, t1, false, any_copy != 0);
}

// The sweep pair applied twice (x_1, x_2, x_1, x_2) in one pass: two consecutive x half steps with the same tables.
cudaError_t SLDG_SFX(sldg_launch_sweep_fused_cell2)(sldg_ctx* c, const void* fin, void* fout, const SweepGeom& g0,
                                                    const SweepGeom& g1, const ShiftTable& t0, const ShiftTable& t1, int any_copy)
{
    return launch_cell(c, fin, fout, g0, g1, t0, t1, true, any_copy != 0);
}
