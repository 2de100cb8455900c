// sldg_sweep_line.cu -- 1-D SLDG sweep along the FASTEST axis (inner == 1), sm_100a: the production kernel.
//
// eq. (3), reading B:   u_i <- A(alpha) u_{(i-s) mod N} + B(alpha) u_{(i-s-1) mod N}.
//
// Lines along axis 0 are contiguous (D_0 = N (k+1) values) and stacked contiguously, so L whole lines are ONE
// contiguous chunk of memory.  The kernel is persistent (grid = SMs x resident CTAs) and every WARP runs its own
// software pipeline over chunks, with no block-level barrier:
//
//   lane 0:  cp.async.bulk global -> shared (1-D TMA, mbarrier complete_tx) into a ring of STAGES input buffers,
//            issued STAGES chunks ahead, so the HBM latency is covered by bytes in flight, not by occupancy;
//   warp:    waits on the chunk's mbarrier, computes every output cell from shared memory (both donor cells come
//            from SMEM: each value of f is read from HBM exactly once), writes a shared output buffer (2-deep);
//   lane 0:  cp.async.bulk shared -> global (bulk_group) and refills the input stage just consumed.
//
// Work distribution is dynamic: a warp claims BATCH consecutive chunks at a time from a global counter (one
// atomic per batch, fired one batch ahead so its latency is never waited for), which keeps the two dies and all
// SMs busy until the end; the last warp to leave resets the counter for the next launch.
//
// A chunk holds whole lines and is resident before anything is written, so the sweep may run IN PLACE
// (fin == fout).  Chunks whose address or size is not a multiple of 16 B (odd D_0 only) take a plain ld/st path
// inside the same kernel.  The shift index of line q is (q / sdiv) % smod; it is computed once per batch and
// tracked incrementally inside it; A, B are re-read from the (L1-resident) table only when the index changes.
#include "sldg_internal.h"
#include "sldg_real.h"

namespace {

constexpr int WARPS = 8;          // warps per CTA
constexpr int OSTAGES = 2;        // output buffers per warp
constexpr int MAXBATCH = 8;       // chunks per claim: STAGES <= batch <= MAXBATCH (issue side at most one batch ahead)

struct LineParams {
    const real* fin;
    real* fout;
    unsigned long long* counter;  // [0] next batch, [1] warps done
    long long nlines, nchunks;
    int N, L;                     // cells per line, lines per chunk
    int batch;                    // chunks per claim
    int cap;                      // doubles per stage buffer (even)
    int last_nl;                  // lines of the last chunk
    int full_tma, last_tma;       // may full chunks / the last chunk use bulk copies (16-byte rule)
    long long sdiv; int smod;     // shift index of line q: (q / sdiv) % smod
    ShiftTable t;
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t phase)
{
    uint32_t ok;
    do {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(ok) : "r"(bar), "r"(phase) : "memory");
    } while (!ok);
}
__device__ __forceinline__ void bulk_load(uint32_t smem_dst, const void* gsrc, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 ::"r"(smem_dst), "l"(gsrc), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void bulk_store(void* gdst, uint32_t smem_src, uint32_t bytes)
{
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;"
                 ::"l"(gdst), "r"(smem_src), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }

template <int K1> struct Cell {
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

template <int K1, int STAGES>
__global__ void __launch_bounds__(WARPS * 32) sweep_line_kernel(const LineParams P)
{
    static_assert(STAGES <= MAXBATCH, "issue side may be at most one batch ahead of the consume side");
    const int BATCH = P.batch;
    constexpr int NN = K1 * K1;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int lane = threadIdx.x & 31, wib = threadIdx.x >> 5;
    const int N = P.N, D0 = N * K1, cap = P.cap;
    const long long nchunks = P.nchunks;
    const long long chunk_vals = (long long)P.L * D0;

    // per-warp shared memory: STAGES input buffers, OSTAGES output buffers; barriers behind all buffers
    real* wbase = reinterpret_cast<real*>(smem_raw) + (size_t)wib * (STAGES + OSTAGES) * cap;
    const uint32_t wbase_s = smem_u32(wbase);
    const uint32_t bars_s = smem_u32(reinterpret_cast<real*>(smem_raw) + (size_t)WARPS * (STAGES + OSTAGES) * cap) +
                            (uint32_t)wib * STAGES * 8u;

    // claim(): lane 0 fires the atomic; the value is read (shuffled) one batch later
    unsigned long long pending = 0;
    auto fire_claim = [&]() { if (lane == 0) pending = atomicAdd(P.counter, 1ULL); };
    auto take_claim = [&]() { return (long long)__shfl_sync(0xffffffffu, pending, 0) * BATCH; };

    auto issue_load = [&](long long c, int st) {          // called by all lanes, acts on lane 0
        if (lane == 0 && c < nchunks) {
            const bool last = (c == nchunks - 1);
            if (last ? P.last_tma : P.full_tma) {
                const uint32_t bytes = (uint32_t)((last ? P.last_nl : P.L) * D0) * (uint32_t)sizeof(real);
                mbar_expect_tx(bars_s + st * 8u, bytes);
                bulk_load(wbase_s + (uint32_t)(st * cap) * (uint32_t)sizeof(real), P.fin + c * chunk_vals, bytes, bars_s + st * 8u);
            }
        }
    };

    if (lane == 0) {
#pragma unroll
        for (int st = 0; st < STAGES; st++) mbar_init(bars_s + st * 8u, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    fire_claim();
    __syncwarp();
    long long ibase = take_claim();       // batch the issue side works in
    fire_claim();                         // ... and the one after it, in flight
    int ioff = 0;
    long long cbase = ibase;              // batch the consume side works in
    int coff = 0;
#pragma unroll
    for (int st = 0; st < STAGES; st++) { issue_load(ibase + ioff, st); ioff++; }

    const int dl32 = 32 / N, di32 = 32 - dl32 * N;       // a stride of 32 cells = dl32 lines + di32 cells
    const int sdivc = (int)min(P.sdiv, (long long)(1 << 30));
    int lane_l = 0, lane_i = lane;                        // (line, cell) of the lane's first cell in a chunk
    while (lane_i >= N) { lane_i -= N; lane_l++; }

    real A[NN], B[NN];
    int cur = -1, s = 0;
    bool cp = false;
    uint32_t phases = 0;          // bit st = parity the next wait on barrier st expects
    int r0c = 0, idx0 = 0;        // first line of the current chunk: lines left before the index changes, index
    bool newbatch = true;

    for (int it = 0;; it++) {
        const long long c = cbase + coff;
        if (c >= nchunks) break;
        const int st = it % STAGES;
        const int ost = it % OSTAGES;
        const bool last = (c == nchunks - 1);
        const int nl = last ? P.last_nl : P.L;
        const int nval = nl * D0;
        const bool tma = (last ? P.last_tma : P.full_tma) != 0;
        real* sin_ = wbase + st * cap;
        real* sout = wbase + (STAGES + ost) * cap;

        if (newbatch) {           // the only integer divisions of the kernel: once per batch
            const long long q0 = c * P.L;
            const long long qd = q0 / P.sdiv;
            const long long r = q0 - qd * P.sdiv;
            idx0 = (int)(qd % P.smod);
            r0c = (int)min(P.sdiv - r, (long long)(1 << 30));
            newbatch = false;
        }

        if (tma) {
            mbar_wait(bars_s + st * 8u, (phases >> st) & 1u);
            phases ^= 1u << st;
        } else {
            const real* gin = P.fin + c * chunk_vals;
            for (int t = lane; t < nval; t += 32) sin_[t] = gin[t];
        }
        // the bulk store that read sout two turns ago must have finished reading shared memory
        if (lane == 0) asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory");
        __syncwarp();

        // per-lane walk over the cells lane, lane + 32, ... of the chunk
        {
            int i = lane_i;
            int left = r0c - lane_l;                       // lines before the shift index changes
            int idxl = idx0;
            while (left <= 0) { left += sdivc; idxl = (idxl + 1 == P.smod) ? 0 : idxl + 1; }
            const real* pl = sin_ + lane_l * D0;         // start of the lane's current line
            real* po = sout + lane * K1;
            const real* pend = sout + nl * D0;
            for (; po < pend; po += 32 * K1) {
                if (idxl != cur) {
                    cur = idxl;
                    const int sv = __ldg(P.t.S + idxl);
                    cp = (sv & SLDG_COPY_BIT) != 0;
                    s = sv & SLDG_S_MASK;
                    const real* ab = static_cast<const real*>(P.t.AB) + (long long)idxl * P.t.strideIdx;
#pragma unroll
                    for (int m = 0; m < NN; m++) {
                        A[m] = __ldg(ab + m * P.t.strideM);
                        B[m] = __ldg(ab + (NN + m) * P.t.strideM);
                    }
                }
                int ia = i - s; if (ia < 0) ia += N;
                int ib = ia - 1; if (ib < 0) ib += N;
                Cell<K1> a, b, r;
                a.load(pl + ia * K1);
                if (!cp) {
                    b.load(pl + ib * K1);
#pragma unroll
                    for (int j = 0; j < K1; j++) {
                        real acc = 0;
#pragma unroll
                        for (int m = 0; m < K1; m++) acc += A[j * K1 + m] * a.v[m];
#pragma unroll
                        for (int m = 0; m < K1; m++) acc += B[j * K1 + m] * b.v[m];
                        r.v[j] = acc;
                    }
                } else {
#pragma unroll
                    for (int j = 0; j < K1; j++) r.v[j] = a.v[j];
                }
                r.store(po);
                // advance by 32 cells
                int dl = dl32;
                i += di32;
                if (i >= N) { i -= N; dl++; }
                pl += dl * D0;
                left -= dl;
                while (left <= 0) { left += sdivc; idxl = (idxl + 1 == P.smod) ? 0 : idxl + 1; }
            }
        }

        if (tma) {
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic-proxy writes -> async proxy
            __syncwarp();
            if (lane == 0) bulk_store(P.fout + c * chunk_vals, wbase_s + (uint32_t)((STAGES + ost) * cap) * (uint32_t)sizeof(real),
                                      (uint32_t)nval * (uint32_t)sizeof(real));
        } else {
            asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic-proxy reads of sin_ -> a refill by the async proxy
            __syncwarp();
            real* gout = P.fout + c * chunk_vals;
            for (int t = lane; t < nval; t += 32) gout[t] = sout[t];
            __syncwarp();
        }
        // one group per turn (empty on the plain path): "at most one group pending" == "the output buffer of two
        // turns ago is free"
        if (lane == 0) bulk_commit();

        // every lane has read sin_ (ordered by the __syncwarp above): refill this stage, STAGES chunks ahead
        if (ioff == BATCH) { ibase = take_claim(); fire_claim(); ioff = 0; }
        issue_load(ibase + ioff, st);
        ioff++;

        // next chunk of the consume side
        coff++;
        if (coff == BATCH) { cbase = ibase; coff = 0; newbatch = true; }
        else {
            r0c -= P.L;
            while (r0c <= 0) { r0c += sdivc; idx0 = (idx0 + 1 == P.smod) ? 0 : idx0 + 1; }
        }
    }
    // shared memory must outlive the bulk stores that read it
    if (lane == 0) {
        asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
        // all claims of this warp have returned (`pending` was produced by the last one): the last warp to leave
        // re-arms the counter for the next launch on this stream
        const unsigned long long W = (unsigned long long)gridDim.x * WARPS;
        if (pending != ~0ULL) __threadfence();
        if (atomicAdd(P.counter + 1, 1ULL) == W - 1) {
            P.counter[0] = 0; P.counter[1] = 0;
            __threadfence();
        }
    }
}

template <int K1, int STAGES>
cudaError_t launch(sldg_ctx* c, LineParams& P, size_t smem)
{
    auto kern = sweep_line_kernel<K1, STAGES>;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    int occ = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, WARPS * 32, smem);
    if (e != cudaSuccess) return e;
    if (occ < 1) return cudaErrorInvalidConfiguration;
    long long grid = (long long)c->sm_count * occ;
    // small problems: short batches so that every warp of the grid gets work
    long long batch = P.nchunks / (4 * grid * WARPS);
    if (batch > MAXBATCH) batch = MAXBATCH;
    if (batch < STAGES) batch = STAGES;
    P.batch = (int)batch;
    const long long need = (P.nchunks + WARPS * batch - 1) / (WARPS * batch);
    if (grid > need) grid = need;
    kern<<<(unsigned)grid, WARPS * 32, smem, c->stream>>>(P);
    return cudaGetLastError();
}

template <int K1>
cudaError_t dispatch(sldg_ctx* c, LineParams& P, int stages, size_t smem)
{
    switch (stages) {
    case 1: return launch<K1, 1>(c, P, smem);
    case 2: return launch<K1, 2>(c, P, smem);
    case 3: return launch<K1, 3>(c, P, smem);
    default: return launch<K1, 4>(c, P, smem);
    }
}

}  // namespace

// Shared memory of one CTA for `stages` input buffers of `cap` doubles per warp.
static size_t line_smem(int stages, long long cap) { return (size_t)WARPS * (stages + OSTAGES) * cap * sizeof(real) + WARPS * 4 * 8 + 16; }

// Returns cudaErrorNotSupported when a line is too long for the per-warp pipelines (caller falls back).
cudaError_t SLDG_SFX(sldg_launch_sweep_line)(sldg_ctx* c, const void* fin, void* fout, const SweepGeom& g,
                                             const ShiftTable& t)
{
    if (g.outer == 0) return cudaSuccess;
    if (g.smod > 0x7fffffffLL || !c->dCounter) return cudaErrorNotSupported;
    const long long D0 = (long long)g.N * g.K1;
    const long long line_bytes = D0 * (long long)sizeof(real);
    const long long Q = 16 / (long long)sizeof(real);            // values per 16 bytes
    const size_t smem_max = 227 * 1024;
    int stages = c->opt_tile_stages;
    if (stages < 1) stages = 1;
    if (stages > 4) stages = 4;
    // lines per chunk: the tile_bytes target, at least one line, an even number of lines when D_0 is odd
    // (keeps chunk starts 16-byte aligned), and no more than fits STAGES + OSTAGES times per warp
    long long L = c->opt_tile_bytes / line_bytes;
    if (L < 1) L = 1;
    auto cap_of = [&](long long l) { return (l * D0 + Q - 1) / Q * Q; };
    while (L > 1 && line_smem(stages, cap_of(L)) > smem_max) L--;
    while (stages > 1 && line_smem(stages, cap_of(L)) > smem_max) stages--;
    if (line_smem(stages, cap_of(L)) > smem_max) return cudaErrorNotSupported;
    // small problems: shorter chunks so that there are a few chunks per warp
    const long long want_chunks = 4LL * c->sm_count * WARPS * stages;
    if (g.outer / L < want_chunks) { L = g.outer / want_chunks; if (L < 1) L = 1; }
    if ((D0 % Q) && L >= Q) L = L / Q * Q;                        // chunk starts stay 16-byte aligned
    if (L > g.outer) L = g.outer;
    LineParams P;
    P.fin = static_cast<const real*>(fin); P.fout = static_cast<real*>(fout); P.counter = c->dCounter;
    P.nlines = g.outer; P.N = g.N; P.L = (int)L; P.batch = MAXBATCH; P.cap = (int)cap_of(L);
    P.nchunks = (g.outer + L - 1) / L;
    P.last_nl = (int)(g.outer - (P.nchunks - 1) * L);
    const bool base_ok = ((((uintptr_t)fin) | ((uintptr_t)fout)) & 15) == 0;
    const bool starts_ok = ((L * line_bytes) & 15) == 0 || P.nchunks == 1;     // every chunk start 16-byte aligned
    P.full_tma = base_ok && ((L * line_bytes) & 15) == 0;
    P.last_tma = base_ok && starts_ok && (((long long)P.last_nl * line_bytes) & 15) == 0;
    P.sdiv = g.sdiv; P.smod = (int)g.smod; P.t = t;
    const size_t smem = line_smem(stages, P.cap);
    switch (g.K1) {
    case 1: return dispatch<1>(c, P, stages, smem);
    case 2: return dispatch<2>(c, P, stages, smem);
    case 3: return dispatch<3>(c, P, stages, smem);
    case 4: return dispatch<4>(c, P, stages, smem);
    case 5: return dispatch<5>(c, P, stages, smem);
    }
    return cudaErrorInvalidValue;
}
