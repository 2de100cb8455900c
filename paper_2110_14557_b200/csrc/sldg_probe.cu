// sldg_probe.cu -- load-path probe (diagnostic entry point sldg_probe_load_rate, include/sldg.h): how fast can an SM
// pull the strided row tiles that the fused v passes gather ([rows][WX] pieces of a [R][X] fp64 array, X contiguous),
// with nothing else going on?  Three ways of bringing the same bytes into the SM are timed:
//   mode 0: 2-d TMA tensor copies (cp.async.bulk.tensor, box WX x ROWS) into a ring of shared-memory slots,
//   mode 1: 1-d TMA bulk copies (cp.async.bulk), one per row piece (WX * 8 bytes each), same ring,
//   mode 2: plain 128-bit global loads by all threads (each thread one 16-byte piece of a row, DEPTH loads in flight).
// No arithmetic, no stores (mode 2 folds the loaded values into one guarded store so that the loads are not removed).
// DESIGN.md section 6 quotes the rates; tests/test_gpu_probe.py runs it.
#include <string.h>

#include "sldg_async.h"
#include "sldg_internal.h"
#include "sldg_tmap.h"

namespace {

using namespace sldg_async;

struct ProbeParams {
    const double* src;
    double* sink;
    long long X, R;               // row length (values), rows
    int WX, ROWS, depth, ntiles, nchunks, cpb;   // tile width (values), rows per box, ring depth, x tiles, row chunks, chunks per block
    uint32_t slot_bytes;
};

// modes 0 and 1: thread 0 issues, every warp waits on the full barrier and releases the slot (as the fused v kernels do)
template <int MODE>
__global__ void __launch_bounds__(256) probe_tma_kernel(const __grid_constant__ CUtensorMap tmap, const ProbeParams P)
{
    extern __shared__ __align__(1024) unsigned char smem_raw[];
    const int ST = P.depth;
    const uint32_t ring_s = smem_u32(smem_raw);
    const uint32_t full_s = ring_s + (uint32_t)ST * P.slot_bytes, empty_s = full_s + 8u * ST;
    const int t = threadIdx.x;
    const int tile = (int)(blockIdx.x % (unsigned)P.ntiles);
    const int c0 = (int)(blockIdx.x / (unsigned)P.ntiles) * P.cpb;
    const int total = min(P.cpb, P.nchunks - c0);
    if (t == 0) {
        for (int s = 0; s < ST; s++) { mbar_init(full_s + 8u * s, 1); mbar_init(empty_s + 8u * s, blockDim.x / 32); }
        mbar_init_fence();
    }
    __syncthreads();
    const uint32_t box_bytes = (uint32_t)P.ROWS * (uint32_t)P.WX * 8u;
    int pst = 0, pn = 0, pi = 0;
    auto produce = [&]() {
        if (pi >= total) return;
        if (pn > 0) mbar_wait(empty_s + 8u * pst, (uint32_t)((pn - 1) & 1));
        mbar_expect_tx(full_s + 8u * pst, box_bytes);
        const long long row0 = (long long)(c0 + pi) * P.ROWS;
        if (MODE == 0) {
            asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
                         ::"r"(ring_s + (uint32_t)pst * P.slot_bytes), "l"(&tmap), "r"(tile * P.WX), "r"((int)row0), "r"(full_s + 8u * pst) : "memory");
        } else {
            for (int r = 0; r < P.ROWS; r++)
                bulk_load(ring_s + (uint32_t)pst * P.slot_bytes + (uint32_t)r * (uint32_t)P.WX * 8u,
                          P.src + (row0 + r) * P.X + (long long)tile * P.WX, (uint32_t)P.WX * 8u, full_s + 8u * pst);
        }
        if (++pst == ST) { pst = 0; pn++; }
        pi++;
    };
    if (t == 0) for (int i = 0; i < ST - 1; i++) produce();
    int st = 0; uint32_t ph = 0;
    double acc = 0.0;
    for (int i = 0; i < total; i++) {
        if (t == 0) produce();
        mbar_wait(full_s + 8u * st, ph);
        acc += reinterpret_cast<const double*>(smem_raw + (size_t)st * P.slot_bytes)[t % (P.ROWS * P.WX)];
        fence_async_smem();
        __syncwarp();
        if ((t & 31) == 0) mbar_arrive(empty_s + 8u * st);
        if (++st == ST) { st = 0; ph ^= 1u; }
    }
    if (acc == 1.2345e300) P.sink[0] = acc;
}

// mode 2: thread -> (row, 16-byte piece) of a box; a box needs ROWS * WX / 2 pieces; DEPTH boxes' loads are issued
// before the first one is consumed
template <int DEPTH>
__global__ void __launch_bounds__(256) probe_ldg_kernel(const ProbeParams P)
{
    const int t = threadIdx.x, NT = blockDim.x;
    const int tile = (int)(blockIdx.x % (unsigned)P.ntiles);
    const int c0 = (int)(blockIdx.x / (unsigned)P.ntiles) * P.cpb;
    const int total = min(P.cpb, P.nchunks - c0);
    const int ppr = P.WX / 2, pieces = P.ROWS * ppr;     // 16-byte pieces per row / per box
    double acc = 0.0;
    for (int i = 0; i < total; i += DEPTH) {
        double2 v[DEPTH][4];
#pragma unroll
        for (int d = 0; d < DEPTH; d++) {
            const long long row0 = (long long)(c0 + i + d) * P.ROWS;
#pragma unroll
            for (int u = 0; u < 4; u++) {
                const int pc = t + u * NT;
                v[d][u] = make_double2(0.0, 0.0);
                if (i + d < total && pc < pieces) {
                    const int r = pc / ppr, q = pc - r * ppr;
                    v[d][u] = __ldcs(reinterpret_cast<const double2*>(P.src + (row0 + r) * P.X + (long long)tile * P.WX + 2 * q));
                }
            }
        }
#pragma unroll
        for (int d = 0; d < DEPTH; d++)
#pragma unroll
            for (int u = 0; u < 4; u++) acc += v[d][u].x + v[d][u].y;
    }
    if (acc == 1.2345e300) P.sink[0] = acc;
}

}  // namespace

// src: [R][X] doubles (device).  Returns the elapsed milliseconds of `reps` launches in *ms_out (host); synchronises.
extern "C" int sldg_probe_load_rate(sldg_ctx* c, const double* src, long long X, long long R, int mode, int wx, int rows,
                                    int depth, int threads, int chunks_per_block, int reps, double* ms_out)
{
    if (!c || !src || !ms_out || mode < 0 || mode > 2 || wx < 2 || (wx & 1) || wx > 256 || rows < 1 || rows > 256 || depth < 2 ||
        depth > 16 || threads < 32 || threads > 256 || (threads & 31) || chunks_per_block < 1 || reps < 1 || X < wx || R < rows)
        return SLDG_EINVAL;
    if (!c->ws_ready) return SLDG_ENOWORKSPACE;
    ProbeParams P;
    P.src = src; P.sink = c->red; P.X = X; P.R = R; P.WX = wx; P.ROWS = rows; P.depth = depth;
    P.ntiles = (int)(X / wx); P.nchunks = (int)(R / rows); P.cpb = chunks_per_block;
    P.slot_bytes = (uint32_t)(((size_t)rows * wx * 8 + 1023) / 1024 * 1024);
    const size_t smem = (size_t)depth * P.slot_bytes + 16 * (size_t)depth + 64;
    if (smem > 227 * 1024) return SLDG_EINVAL;
    const long long nblk = (long long)P.ntiles * ((P.nchunks + P.cpb - 1) / P.cpb);
    if (nblk < 1 || nblk > 0x7fffffffLL) return SLDG_EINVAL;
    if (mode == 2 && (long long)rows * (wx / 2) > 4LL * threads) return SLDG_EINVAL;
    CUtensorMap tm;
    memset(&tm, 0, sizeof(tm));
    if (mode == 0) {
        SldgEncodeTiled enc = sldg_encode_tiled();
        if (!enc) { c->last_cuda = (int)cudaErrorNotSupported; return SLDG_ECUDA; }
        const cuuint64_t gdim[2] = {(cuuint64_t)X, (cuuint64_t)R};
        const cuuint64_t gstr[1] = {(cuuint64_t)X * 8};
        const cuuint32_t box[2] = {(cuuint32_t)wx, (cuuint32_t)rows};
        const cuuint32_t estr[2] = {1u, 1u};
        if (enc(&tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<double*>(src), gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                CU_TENSOR_MAP_SWIZZLE_NONE, sldg_l2_promotion(c->opt_fv_l2), CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS) {
            c->last_cuda = (int)cudaErrorInvalidValue; return SLDG_ECUDA;
        }
    }
    cudaEvent_t e0, e1;
    if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return SLDG_ECUDA;
    cudaError_t e = cudaSuccess;
    if (mode == 0) e = cudaFuncSetAttribute(probe_tma_kernel<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (mode == 1) e = cudaFuncSetAttribute(probe_tma_kernel<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    for (int r = -1; r < reps && e == cudaSuccess; r++) {             // one untimed launch first
        if (r == 0) cudaEventRecord(e0, c->stream);
        if (mode == 0) probe_tma_kernel<0><<<(unsigned)nblk, threads, smem, c->stream>>>(tm, P);
        else if (mode == 1) probe_tma_kernel<1><<<(unsigned)nblk, threads, smem, c->stream>>>(tm, P);
        else if (depth >= 4) probe_ldg_kernel<4><<<(unsigned)nblk, threads, 0, c->stream>>>(P);
        else probe_ldg_kernel<2><<<(unsigned)nblk, threads, 0, c->stream>>>(P);
        e = cudaGetLastError();
    }
    cudaEventRecord(e1, c->stream);
    if (e == cudaSuccess) e = cudaEventSynchronize(e1);
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    if (e != cudaSuccess) { c->last_cuda = (int)e; return SLDG_ECUDA; }
    *ms_out = (double)ms;
    return SLDG_OK;
}
