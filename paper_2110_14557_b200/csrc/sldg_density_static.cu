// sldg_density_static.cu -- rho = int f dv (row a3) for callers that cannot allocate device memory.
//
// Who this is for.  sldg_density needs a context, and a context is built with cudaMalloc (small tables) plus a
// caller-supplied workspace that holds the partial sums of the two-stage reduction.  Some users of the library cannot
// do either at the point where they need rho:
//   * a time loop whose host application has already handed all of HBM to its own pool (on the 6-d configs the two f
//     buffers alone are 113 GB of the 180 GB; a framework's caching allocator typically owns the rest), so a fresh
//     cudaMalloc fails or forces that pool to give memory back;
//   * a latency-sensitive loop that runs next to other streams: cudaMalloc / cudaFree synchronise the whole device, so
//     one allocation in a diagnostic call stalls every stream of the process;
//   * a plug-in or callback that is handed device pointers and a stream by its host code and is, by that host's rules,
//     not allowed to create or release device memory of its own.
// For them this file offers ONE context-free call, sldg_density_static: inputs and the output are the caller's, and the
// partial sums live in a fixed array that is part of the library image itself (g_rho_scratch below, 8 MiB).  The call
// performs no cudaMalloc / cudaFree / cudaMallocAsync and calls no library routine that allocates.
//
// Price of that array: every GPU on which this library's device code gets loaded keeps those 8 MiB until the process
// exits, whether or not the call is ever used, and problems whose x grid has more than SLDG_DENSITY_STATIC_MAX_X nodes
// are refused (SLDG_ETOOLARGE) instead of being served more slowly.
//
// Nothing else in the library uses this file, and it uses nothing of the rest (no context, no workspace): the existing
// sldg_density path is unchanged.
#include <cuda_runtime.h>
#include <stdint.h>

#include <mutex>

#include "../../include/sldg.h"

namespace {

// The scratch: partial sums part[chunk][x], chunk-major, at most SLDG_DENSITY_STATIC_MAX_X doubles in total.
// IN HOST CODE THIS NAME IS NOT A DEVICE ADDRESS (it is the host-side shadow symbol the runtime uses as a look-up key);
// the launcher below asks the runtime for the real address once per device and hands that pointer to the kernels.
static __device__ __align__(256) double g_rho_scratch[SLDG_DENSITY_STATIC_MAX_X];

template <class T> struct Pair2;
template <> struct Pair2<double> { typedef double2 type; };
template <> struct Pair2<float> { typedef float2 type; };

constexpr int ST_THREADS = 128;     // threads per block
constexpr int ST_U = 8;             // rows of f in flight per thread

// Stage 1.  f seen as [V][X] (x contiguous).  Block (bx, by): 128 threads x VEC consecutive x values, rows
// v in [by * vchunk, min(V, (by + 1) * vchunk)) in ascending order, acc = fma(W_v, f, acc) in fp64 (f may be float).
// Writes part[by][x] for EVERY x < X of its tile, also when the chunk is short: stage 2 never reads a stale value,
// so the shared array needs no clearing between calls.
template <int VEC, class T>
__global__ void __launch_bounds__(ST_THREADS) rho_static_partial_kernel(const T* __restrict__ f, const double* __restrict__ Wv,
                                                                         long long X, long long V, long long vchunk,
                                                                         double* __restrict__ part)
{
    const long long x = ((long long)blockIdx.x * ST_THREADS + threadIdx.x) * VEC;
    if (x >= X) return;
    const long long v0 = (long long)blockIdx.y * vchunk;
    long long v1 = v0 + vchunk;
    if (v1 > V) v1 = V;
    double acc[VEC];
#pragma unroll
    for (int e = 0; e < VEC; e++) acc[e] = 0.0;
    long long v = v0;
    for (; v + ST_U <= v1; v += ST_U) {
        T t[ST_U][VEC];
#pragma unroll
        for (int u = 0; u < ST_U; u++) {
            const T* p = f + (v + u) * X + x;
            if (VEC == 2) {
                typedef typename Pair2<T>::type T2;
                const T2 d = __ldcs(reinterpret_cast<const T2*>(p));
                t[u][0] = d.x; t[u][VEC - 1] = d.y;
            } else {
                t[u][0] = __ldcs(p);
            }
        }
#pragma unroll
        for (int u = 0; u < ST_U; u++) {
            const double wv = __ldg(Wv + v + u);
#pragma unroll
            for (int e = 0; e < VEC; e++) acc[e] = fma(wv, (double)t[u][e], acc[e]);
        }
    }
    for (; v < v1; v++) {
        const double wv = __ldg(Wv + v);
#pragma unroll
        for (int e = 0; e < VEC; e++) acc[e] = fma(wv, (double)__ldcs(f + v * X + x + e), acc[e]);
    }
#pragma unroll
    for (int e = 0; e < VEC; e++) part[(long long)blockIdx.y * X + x + e] = acc[e];
}

// Stage 2: rho[x] = part[0][x] + part[1][x] + ... in chunk order (fixed order: repeated calls give the same bits).
__global__ void __launch_bounds__(256) rho_static_final_kernel(const double* __restrict__ part, long long X, int nchunk,
                                                               double* __restrict__ rho)
{
    const long long x = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (x >= X) return;
    double acc = 0.0;
    for (int c = 0; c < nchunk; c++) acc += part[(long long)c * X + x];
    rho[x] = acc;
}

// What the launcher has to know about a device, looked up once per device under a lock.
constexpr int ST_MAX_DEVICES = 64;
struct StaticDev { bool ready; double* scratch; int sm_count; };
StaticDev g_dev[ST_MAX_DEVICES];
std::mutex g_dev_mu;

// Set-up for the CURRENT device (the one cudaGetDevice reports; the caller's f, Wv and rho must live on it):
// resolve the device address of g_rho_scratch with cudaGetSymbolAddress and read the SM count.  Neither allocates;
// the first of them may make the runtime load this library's device code onto that GPU, which is why the first call
// on a device should be made at start-up, outside any stream capture.
cudaError_t static_setup(int dev, StaticDev* out)
{
    std::lock_guard<std::mutex> lock(g_dev_mu);
    StaticDev& d = g_dev[dev];
    if (!d.ready) {
        double* p = nullptr;
        cudaError_t e = cudaGetSymbolAddress((void**)&p, g_rho_scratch);
        if (e != cudaSuccess) return e;
        if (p == nullptr) return cudaErrorInvalidSymbol;
        int sm = 0;
        e = cudaDeviceGetAttribute(&sm, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return e;
        d.scratch = p; d.sm_count = sm > 0 ? sm : 1; d.ready = true;
    }
    *out = d;
    return cudaSuccess;
}

template <class T>
cudaError_t launch_static(const T* f, const double* Wv, long long X, long long V, double* rho, cudaStream_t st,
                          const StaticDev& d)
{
    const int vec = ((X & 1) == 0 && (((uintptr_t)f) & (2 * sizeof(T) - 1)) == 0) ? 2 : 1;
    const long long xtiles = (X + (long long)ST_THREADS * vec - 1) / ((long long)ST_THREADS * vec);
    // about one wave of 8 blocks per SM, never more chunks than the fixed array holds rows of X partial sums
    long long nchunk = ((long long)d.sm_count * 8) / xtiles;
    if (nchunk > V / 16) nchunk = V / 16;
    if (nchunk > (long long)SLDG_DENSITY_STATIC_MAX_X / X) nchunk = (long long)SLDG_DENSITY_STATIC_MAX_X / X;
    if (nchunk > 65535) nchunk = 65535;
    if (nchunk < 1) nchunk = 1;
    const long long vchunk = (V + nchunk - 1) / nchunk;
    nchunk = (V + vchunk - 1) / vchunk;
    const dim3 grid((unsigned)xtiles, (unsigned)nchunk);
    if (vec == 2) rho_static_partial_kernel<2, T><<<grid, ST_THREADS, 0, st>>>(f, Wv, X, V, vchunk, d.scratch);
    else rho_static_partial_kernel<1, T><<<grid, ST_THREADS, 0, st>>>(f, Wv, X, V, vchunk, d.scratch);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    rho_static_final_kernel<<<(unsigned)((X + 255) / 256), 256, 0, st>>>(d.scratch, X, (int)nchunk, rho);
    return cudaGetLastError();
}

}  // namespace

extern "C" long long sldg_density_static_max_x(void) { return (long long)SLDG_DENSITY_STATIC_MAX_X; }

extern "C" int sldg_density_static(const void* f, const double* Wv, long long X, long long V, int precision, double* rho,
                                   void* stream, int* cuda_error_host)
{
    if (cuda_error_host) *cuda_error_host = 0;
    if (!f || !Wv || !rho || X < 1 || V < 1) return SLDG_EINVAL;
    if (precision != SLDG_F64 && precision != SLDG_F32) return SLDG_EINVAL;
    if (X > (long long)SLDG_DENSITY_STATIC_MAX_X) return SLDG_ETOOLARGE;        // before anything touches the device
    if (V > (1LL << 40)) return SLDG_EINVAL;                                    // index range of v * X
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    StaticDev d = {false, nullptr, 0};
    if (e == cudaSuccess && (dev < 0 || dev >= ST_MAX_DEVICES)) e = cudaErrorInvalidDevice;
    if (e == cudaSuccess) e = static_setup(dev, &d);
    if (e == cudaSuccess) {
        cudaStream_t st = (cudaStream_t)stream;
        e = precision == SLDG_F32 ? launch_static<float>((const float*)f, Wv, X, V, rho, st, d)
                                  : launch_static<double>((const double*)f, Wv, X, V, rho, st, d);
    }
    if (e != cudaSuccess) {
        if (cuda_error_host) *cuda_error_host = (int)e;
        return SLDG_ECUDA;
    }
    return SLDG_OK;
}
