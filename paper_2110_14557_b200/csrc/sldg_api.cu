// sldg_api.cu -- the C-ABI of include/sldg.h: context, host tables, launch sequencing.
// No CPU fallback anywhere: every compute entry point enqueues sm_100a kernels or returns an error.
#include <math.h>
#include <stdlib.h>
#include <string.h>

#include <new>

#include "sldg_internal.h"

#define CK(call)                                                      \
    do {                                                              \
        cudaError_t e_ = (call);                                      \
        if (e_ != cudaSuccess) { c->last_cuda = (int)e_; return SLDG_ECUDA; } \
    } while (0)

static size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// ------------------------------------------------------------------ instrumentation
void sldg_ev_begin(sldg_ctx* c, int kind, int axis)
{
    if (!c->timing) return;
    EventRec r;
    if (!c->ev_free.empty()) { r = c->ev_free.back(); c->ev_free.pop_back(); }
    else {
        if (cudaEventCreate(&r.a) != cudaSuccess) { c->ev_failed = true; c->last_cuda = (int)cudaGetLastError(); return; }
        if (cudaEventCreate(&r.b) != cudaSuccess) { cudaEventDestroy(r.a); c->ev_failed = true; c->last_cuda = (int)cudaGetLastError(); return; }
    }
    r.kind = kind; r.axis = axis;
    cudaEventRecord(r.a, c->stream);
    c->ev.push_back(r);
}
// a launcher declined (cudaErrorNotSupported): forget the event opened for it
static void ev_cancel(sldg_ctx* c)
{
    if (!c->timing || c->ev.empty() || c->ev_failed) return;
    c->ev_free.push_back(c->ev.back());
    c->ev.pop_back();
}
void sldg_ev_end(sldg_ctx* c)
{
    if (!c->timing || c->ev.empty() || c->ev_failed) return;
    cudaEventRecord(c->ev.back().b, c->stream);
}

// ------------------------------------------------------------------ layout of the workspace
struct WsLayout { size_t f2, vS, vAB, vS2, vAB2, vS3, vAB3, Wv, rho, E, part, cplx[6], red, phi, cg_info, total; long long part_cap; };

static WsLayout ws_layout(const sldg_ctx* c)
{
    WsLayout L;
    size_t off = 0;
    const size_t X = (size_t)c->X, NN2 = 2 * (size_t)c->K1 * c->K1;
    auto take = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes, 256); return o; };
    L.f2 = take((size_t)c->nf * c->esize);
    L.vS = take(X * 4);
    L.vAB = take(X * NN2 * 8);
    L.vS2 = take(X * 4);
    L.vAB2 = take(X * NN2 * 8);
    L.vS3 = take(c->dx == 3 ? X * 4 : 0);
    L.vAB3 = take(c->dx == 3 ? X * NN2 * 8 : 0);
    L.Wv = take((size_t)c->V * 8);
    L.rho = take(X * 8);
    L.E = take(X * 8 * c->dx);
    // rho partial sums: enough chunks to fill the GPU (see sldg_launch_density), at least 1
    long long xtiles = (c->X + 255) / 256;
    long long nchunk = ((long long)c->sm_count * 64 + xtiles - 1) / xtiles;
    if (nchunk > c->V / 16) nchunk = c->V / 16;
    if (nchunk < 1) nchunk = 1;
    nchunk += 1;
    L.part_cap = nchunk * c->X;
    L.part = take((size_t)L.part_cap * 8);
    for (int i = 0; i < 6; i++) L.cplx[i] = take(X * 8);
    L.red = take(4096 * 8);
    L.phi = take(X * 8);
    L.cg_info = take(4 * 8);
    L.total = off;
    return L;
}

// ------------------------------------------------------------------ lifetime
extern "C" int sldg_create(sldg_ctx** out, int dim_x, int dim_v, const int* cells, int degree, const double* domain)
{
    return sldg_create_prec(out, dim_x, dim_v, cells, degree, domain, SLDG_F64);
}

extern "C" int sldg_precision(const sldg_ctx* c) { return c ? c->prec : SLDG_EINVAL; }

// precision dispatch of the kernels that exist as _f64 and _f32 (sldg_real.h)
cudaError_t sldg_launch_sweep_walk(sldg_ctx* c, const double* fin, double* fout, const SweepGeom& g, const ShiftTable& t)
{
    return c->prec == SLDG_F32 ? sldg_launch_sweep_walk_f32(c, fin, fout, g, t) : sldg_launch_sweep_walk_f64(c, fin, fout, g, t);
}
cudaError_t sldg_launch_sweep_line(sldg_ctx* c, const double* fin, double* fout, const SweepGeom& g, const ShiftTable& t)
{
    return c->prec == SLDG_F32 ? sldg_launch_sweep_line_f32(c, fin, fout, g, t) : sldg_launch_sweep_line_f64(c, fin, fout, g, t);
}
cudaError_t sldg_launch_sweep_fused_cell(sldg_ctx* c, const double* fin, double* fout, const SweepGeom& g0,
                                         const SweepGeom& g1, const ShiftTable& t0, const ShiftTable& t1, int any_copy)
{
    return c->prec == SLDG_F32 ? sldg_launch_sweep_fused_cell_f32(c, fin, fout, g0, g1, t0, t1, any_copy)
                               : sldg_launch_sweep_fused_cell_f64(c, fin, fout, g0, g1, t0, t1, any_copy);
}

// host_only: the host fields only, no device (the dry-run context of sldg_plan_query)
static int create_impl(sldg_ctx** out, int dim_x, int dim_v, const int* cells, int degree, const double* domain,
                       int precision, bool host_only)
{
    if (!out || !cells || !domain) return SLDG_EINVAL;
    if (precision != SLDG_F64 && precision != SLDG_F32) return SLDG_EINVAL;
    if (dim_x < 1 || dim_x > 3 || dim_v < dim_x || dim_v > 3) return SLDG_EINVAL;
    if (degree < 0 || degree > SLDG_MAX_DEGREE) return SLDG_EINVAL;
    const int d = dim_x + dim_v;
    for (int a = 0; a < d; a++) {
        if (cells[a] < 1 || cells[a] >= (1 << 24)) return SLDG_EINVAL;
        if (!(domain[2 * a + 1] > domain[2 * a])) return SLDG_EINVAL;
    }
    sldg_ctx* c = new (std::nothrow) sldg_ctx();
    if (!c) return SLDG_ENOMEM;
    c->dry = false; c->dry_safe = 0; c->dry_x = c->dry_v = c->dry_rho = c->dry_field = c->dry_copies = 0;
    c->dx = dim_x; c->dv = dim_v; c->d = d; c->k = degree; c->K1 = degree + 1;
    c->prec = precision; c->esize = precision == SLDG_F32 ? 4 : 8;
    c->nf = 1; c->X = 1; c->V = 1;
    for (int a = 0; a < d; a++) {
        c->cells[a] = cells[a];
        c->D[a] = (long long)cells[a] * c->K1;
        c->lo[a] = domain[2 * a]; c->hi[a] = domain[2 * a + 1];
        c->h[a] = (c->hi[a] - c->lo[a]) / (double)cells[a];
        c->nf *= c->D[a];
        if (a < dim_x) c->X *= c->D[a]; else c->V *= c->D[a];
    }
    sldg_gl_rule(c->K1, c->xi, c->w);
    sldg_build_poly(c->k, c->xi, c->w, &c->poly, &c->poly_ld);
    c->stream = 0; c->last_cuda = 0; c->sm_count = 148;
    c->ws = nullptr; c->ws_bytes = 0; c->ws_ready = false;
    c->timing = false; c->launches = 0;
    c->cap_stream = nullptr; c->graph_exec = nullptr; c->graph_f = nullptr; c->graph_dt = 0.0; c->graph_launches = 0; c->opt_graph = 1;
    c->phi = nullptr; c->cg_info = nullptr; c->poisson_solver = 0; c->cg_tol = 1e-3; c->cg_sigma = sldg_sipg_sigma_default(degree);
    c->cg_maxiter = 0;
    memset(c->t_launch, 0, sizeof(c->t_launch)); memset(c->t_ms, 0, sizeof(c->t_ms));
    memset(c->a_launch, 0, sizeof(c->a_launch)); memset(c->a_ms, 0, sizeof(c->a_ms));
    c->opt_tile_bytes = 3584; c->opt_tile_stages = 2; c->opt_axis0_impl = 0; c->opt_walk_block = 128; c->opt_walk_vec = 0; c->opt_rho_vec = 0; c->opt_rho_tma = 1; c->opt_fuse_x = 1; c->opt_fused_threads = 256; c->opt_inplace_walk = 1; c->opt_rho_blocks = 8;
    c->opt_fused_impl = 0; c->opt_x_copy = 0; c->opt_fuse3 = 1; c->opt_f3_threads = 128; c->opt_f3_stages = 3; c->opt_f3d_threads = 128; c->opt_cell_threads = 64; c->opt_cell_rows = 0; c->opt_cell_bytes = 9216; c->opt_cell_stages = 2;
    c->opt_poisson_small = 1; c->opt_x_double = 1; c->opt_fuse_v = 1; c->opt_fv_wx = 0; c->opt_fv_stages = 0; c->opt_fv_inflight = 72 * 1024; c->opt_fv_ppb = 0; c->opt_fv_l2 = 3; c->opt_fv_cps = 1;
    c->opt_decline = 0; c->opt_fuse_v3 = 1; c->opt_fv3_wx = 0; c->opt_fv3_strip = 0; c->opt_fv3_slots = 0; c->opt_fv3_pw = 1;
    for (int a = 0; a < SLDG_MAX_DIM; a++) { c->tab_safe[a] = false; c->tab_anycp[a] = true; c->dWx[a] = nullptr; }
    for (int a = 0; a < 3; a++) for (int i = 0; i < SLDG_XTAB_SLOTS; i++) { XTab& x = c->xtab[a][i]; x.dS = nullptr; x.dAB = nullptr; x.tau = 0.0; x.valid = x.anycp = x.safe = false; x.used = 0; }
    c->xtab_clock = 0; c->ev_failed = false;
    for (int a = 0; a < 3; a++) { c->dFwdT[a] = c->dInvT[a] = c->dKap[a] = nullptr; }
    c->dS_hook = nullptr; c->dAB_hook = nullptr; c->hook_cap = 0;
    c->dPoly = nullptr; c->dScalar = nullptr; c->dCounter = nullptr; c->hS = nullptr; c->hAB = nullptr; c->hcap = 0;

    if (host_only) { *out = c; return SLDG_OK; }                            // sldg_plan_query

    // device side: needs a CUDA device.  Without one the context is unusable -> fail loudly.
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e == cudaSuccess) {
        int sm = 0;
        if (cudaDeviceGetAttribute(&sm, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && sm > 0) c->sm_count = sm;
        e = sldg_upload_poly(c);
    }
    const size_t NN2 = 2 * (size_t)c->K1 * c->K1;
    long long maxD = 0;
    for (int a = 0; a < d; a++) if (c->D[a] > maxD) maxD = c->D[a];
    c->hcap = maxD;
    if (e == cudaSuccess) e = cudaMallocHost((void**)&c->hS, (size_t)maxD * 4);
    if (e == cudaSuccess) e = cudaMallocHost((void**)&c->hAB, (size_t)maxD * NN2 * 8);
    if (e == cudaSuccess) e = cudaMalloc((void**)&c->dScalar, 8);
    if (e == cudaSuccess) e = cudaMalloc((void**)&c->dCounter, 16);
    if (e == cudaSuccess) e = cudaMemset(c->dCounter, 0, 16);
    for (int a = 0; a < dim_x && e == cudaSuccess; a++) {
        long long Ds = c->D[dim_x + a];
        for (int i = 0; i < SLDG_XTAB_SLOTS && e == cudaSuccess; i++) {
            e = cudaMalloc((void**)&c->xtab[a][i].dS, (size_t)Ds * 4);
            if (e == cudaSuccess) e = cudaMalloc((void**)&c->xtab[a][i].dAB, (size_t)Ds * NN2 * 8);
        }
    }
    if (e == cudaSuccess) { e = cudaMalloc((void**)&c->dS_hook, (size_t)maxD * 4); }
    if (e == cudaSuccess) { e = cudaMalloc((void**)&c->dAB_hook, (size_t)maxD * NN2 * 8); c->hook_cap = maxD; }
    // per-axis quadrature weights h_a w_j
    for (int a = 0; a < d && e == cudaSuccess; a++) {
        std::vector<double> wa((size_t)c->D[a]);
        for (long long n = 0; n < c->D[a]; n++) wa[(size_t)n] = c->h[a] * c->w[n % c->K1];
        e = cudaMalloc((void**)&c->dWx[a], (size_t)c->D[a] * 8);
        if (e == cudaSuccess) e = cudaMemcpy(c->dWx[a], wa.data(), (size_t)c->D[a] * 8, cudaMemcpyHostToDevice);
    }
    // Poisson tables
    for (int a = 0; a < dim_x && e == cudaSuccess; a++) {
        const long long D = c->D[a];
        std::vector<double> fw((size_t)(2 * D * D)), iv((size_t)(2 * D * D)), kap((size_t)D);
        sldg_build_dft(c->k, c->xi, c->cells[a], fw.data(), iv.data());
        const long double twopi = 6.28318530717958647692528676655900577L;
        for (long long m = 0; m < D; m++) {
            long long mm = (2 * m < D) ? m : m - D;
            kap[(size_t)m] = (double)(twopi * (long double)mm / (long double)(c->hi[a] - c->lo[a]));
        }
        e = cudaMalloc((void**)&c->dFwdT[a], (size_t)(2 * D * D) * 8);
        if (e == cudaSuccess) e = cudaMalloc((void**)&c->dInvT[a], (size_t)(2 * D * D) * 8);
        if (e == cudaSuccess) e = cudaMalloc((void**)&c->dKap[a], (size_t)D * 8);
        if (e == cudaSuccess) e = cudaMemcpy(c->dFwdT[a], fw.data(), (size_t)(2 * D * D) * 8, cudaMemcpyHostToDevice);
        if (e == cudaSuccess) e = cudaMemcpy(c->dInvT[a], iv.data(), (size_t)(2 * D * D) * 8, cudaMemcpyHostToDevice);
        if (e == cudaSuccess) e = cudaMemcpy(c->dKap[a], kap.data(), (size_t)D * 8, cudaMemcpyHostToDevice);
    }
    if (e != cudaSuccess) {
        c->last_cuda = (int)e;
        sldg_destroy(c);
        return (e == cudaErrorMemoryAllocation) ? SLDG_ENOMEM : SLDG_ECUDA;
    }
    *out = c;
    return SLDG_OK;
}

extern "C" int sldg_create_prec(sldg_ctx** out, int dim_x, int dim_v, const int* cells, int degree, const double* domain,
                                int precision)
{
    return create_impl(out, dim_x, dim_v, cells, degree, domain, precision, false);
}

extern "C" int sldg_destroy(sldg_ctx* c)
{
    if (!c) return SLDG_EINVAL;
    sldg_graph_drop(c);
    if (c->cap_stream) cudaStreamDestroy(c->cap_stream);
    for (int a = 0; a < SLDG_MAX_DIM; a++) {
        if (c->dWx[a]) cudaFree(c->dWx[a]);
    }
    for (int a = 0; a < 3; a++) {
        for (int i = 0; i < SLDG_XTAB_SLOTS; i++) {
            if (c->xtab[a][i].dS) cudaFree(c->xtab[a][i].dS);
            if (c->xtab[a][i].dAB) cudaFree(c->xtab[a][i].dAB);
        }
        if (c->dFwdT[a]) cudaFree(c->dFwdT[a]);
        if (c->dInvT[a]) cudaFree(c->dInvT[a]);
        if (c->dKap[a]) cudaFree(c->dKap[a]);
    }
    if (c->dS_hook) cudaFree(c->dS_hook);
    if (c->dAB_hook) cudaFree(c->dAB_hook);
    if (c->dPoly) cudaFree(c->dPoly);
    if (c->dScalar) cudaFree(c->dScalar);
    if (c->dCounter) cudaFree(c->dCounter);
    if (c->hS) cudaFreeHost(c->hS);
    if (c->hAB) cudaFreeHost(c->hAB);
    for (auto& r : c->ev) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
    for (auto& r : c->ev_free) { cudaEventDestroy(r.a); cudaEventDestroy(r.b); }
    delete c;
    return SLDG_OK;
}

extern "C" int sldg_set_stream(sldg_ctx* c, void* stream)
{
    if (!c) return SLDG_EINVAL;
    sldg_graph_drop(c);
    c->stream = (cudaStream_t)stream;
    return SLDG_OK;
}

extern "C" size_t sldg_workspace_bytes(const sldg_ctx* c) { return c ? ws_layout(c).total : 0; }

extern "C" int sldg_set_workspace(sldg_ctx* c, void* dev, size_t bytes)
{
    if (!c || !dev) return SLDG_EINVAL;
    if (((uintptr_t)dev) & 255) return SLDG_EINVAL;
    WsLayout L = ws_layout(c);
    if (bytes < L.total) return SLDG_ENOWORKSPACE;
    sldg_graph_drop(c);
    char* b = (char*)dev;
    c->ws = b; c->ws_bytes = bytes;
    c->f2 = (double*)(b + L.f2); c->vS = (int*)(b + L.vS); c->vAB = (double*)(b + L.vAB);
    c->vS2 = (int*)(b + L.vS2); c->vAB2 = (double*)(b + L.vAB2);
    c->vS3 = (int*)(b + L.vS3); c->vAB3 = (double*)(b + L.vAB3);
    c->Wv = (double*)(b + L.Wv); c->rho = (double*)(b + L.rho); c->E = (double*)(b + L.E);
    c->part = (double*)(b + L.part); c->part_cap = L.part_cap;
    for (int i = 0; i < 6; i++) c->cplx[i] = (double*)(b + L.cplx[i]);
    c->red = (double*)(b + L.red);
    c->phi = (double*)(b + L.phi); c->cg_info = (double*)(b + L.cg_info);
    if (cudaMemsetAsync(c->phi, 0, (size_t)c->X * 8 + 0, c->stream) != cudaSuccess ||
        cudaMemsetAsync(c->cg_info, 0, 32, c->stream) != cudaSuccess) { c->ws_ready = false; return SLDG_ECUDA; }
    sldg_ev_begin(c, KIND_TABLE, -1);
    cudaError_t e = sldg_launch_wv(c);
    sldg_ev_end(c);
    c->launches++;
    if (e != cudaSuccess) { c->last_cuda = (int)e; c->ws_ready = false; return SLDG_ECUDA; }
    c->ws_ready = true;
    return SLDG_OK;
}

// ------------------------------------------------------------------ geometry / tables
static SweepGeom geom_of(const sldg_ctx* c, int axis)
{
    SweepGeom g;
    g.inner = 1; g.outer = 1;
    for (int b = 0; b < axis; b++) g.inner *= c->D[b];
    for (int b = axis + 1; b < c->d; b++) g.outer *= c->D[b];
    g.N = c->cells[axis]; g.K1 = c->K1;
    if (axis < c->dx) {
        g.mode = 0;
        int sa = c->dx + axis;
        g.sdiv = 1;
        for (int b = axis + 1; b < sa; b++) g.sdiv *= c->D[b];
        g.smod = c->D[sa];
    } else {
        g.mode = 1; g.sdiv = 1; g.smod = c->X;
    }
    return g;
}

// host: split delta into (s mod N | copy bit) and A(alpha), B(alpha)   (reading B, O)
static void host_entry(const sldg_ctx* c, double delta, int N, int* S, double* AB)
{
    const int NN = c->K1 * c->K1;
    double sd = floor(delta);
    double alpha = delta - sd;
    int s = (int)fmod(sd, (double)N);
    if (s < 0) s += N;
    if (alpha == 0.0) {
        *S = s | SLDG_COPY_BIT;
        for (int m = 0; m < NN; m++) { AB[m] = (m % (c->K1 + 1) == 0) ? 1.0 : 0.0; AB[NN + m] = 0.0; }
    } else {
        *S = s;
        sldg_eval_AB_host(&c->poly_ld, c->k, alpha, AB, AB + NN);
    }
}

static int upload_table(sldg_ctx* c, const double* delta, long long n, int N, int* dS, double* dAB)
{
    const size_t NN2 = 2 * (size_t)c->K1 * c->K1;
    if (n > c->hcap) return SLDG_EINVAL;
    for (long long i = 0; i < n; i++)
        if (!isfinite(delta[i])) return SLDG_EINVAL;       // a NaN / Inf shift has no floor(): nothing is enqueued
    // the pinned staging buffers may still be in flight from a previous upload on this stream: SYNCHRONISES
    // (include/sldg.h marks the calls that can get here)
    CK(cudaStreamSynchronize(c->stream));
    for (long long i = 0; i < n; i++) host_entry(c, delta[i], N, c->hS + i, c->hAB + (size_t)i * NN2);
    if (c->prec == SLDG_F32) {          // A, B were evaluated in long double; the sweep takes them rounded to fp32
        std::vector<float> h4((size_t)n * NN2);
        for (size_t i = 0; i < h4.size(); i++) h4[i] = (float)c->hAB[i];
        memcpy(c->hAB, h4.data(), h4.size() * 4);
    }
    sldg_ev_begin(c, KIND_UPLOAD, -1);
    CK(cudaMemcpyAsync(dS, c->hS, (size_t)n * 4, cudaMemcpyHostToDevice, c->stream));
    CK(cudaMemcpyAsync(dAB, c->hAB, (size_t)n * NN2 * c->esize, cudaMemcpyHostToDevice, c->stream));
    sldg_ev_end(c);
    return SLDG_OK;
}

static int copy_back(sldg_ctx* c, double* dst, const double* src);

// `scratch`: the buffer of the pair that is neither read nor written (used only if an in-place request has to be
// served by an out-of-place kernel).
static int run_sweep(sldg_ctx* c, const double* fin, double* fout, double* scratch, int axis, const ShiftTable& t,
                     bool inplace_walk_ok = false)
{
    SweepGeom g = geom_of(c, axis);
    cudaError_t e;
    if (c->dry) {
        if (g.inner != 1 && fin == fout && !inplace_walk_ok) return SLDG_EINVAL;
        (axis < c->dx ? c->dry_x : c->dry_v)++;
        c->launches++;
        return SLDG_OK;
    }
    if (g.inner == 1) {
        // contiguous lines: per-warp TMA pipelines; block-wide tiles when a line is too long for a warp's ring;
        // the (uncoalesced) register walk when it does not even fit a block's shared memory
        sldg_ev_begin(c, KIND_SWEEP0, axis);
        e = cudaErrorNotSupported;
        if (c->opt_axis0_impl == 0 || c->opt_axis0_impl == 1) e = sldg_launch_sweep_line(c, fin, fout, g, t);
        if (e == cudaErrorNotSupported && c->opt_axis0_impl != 3 && c->prec == SLDG_F64) {
            e = sldg_launch_sweep_tma(c, fin, fout, g, t);
            if (e == cudaErrorInvalidConfiguration) e = cudaErrorNotSupported;
        }
        if (e == cudaErrorNotSupported) {
            if (fin == fout) {
                if (!scratch || scratch == fin) { sldg_ev_end(c); return SLDG_EINVAL; }
                e = sldg_launch_sweep_walk(c, fin, scratch, g, t);
                sldg_ev_end(c);
                c->launches++;
                if (e != cudaSuccess) { c->last_cuda = (int)e; return SLDG_ECUDA; }
                return copy_back(c, fout, scratch);
            }
            e = sldg_launch_sweep_walk(c, fin, fout, g, t);
        }
    } else {
        // a slow-axis walk may run in place only when every shift of its table is s in {0, -1} (see x_plan)
        if (fin == fout && !inplace_walk_ok) return SLDG_EINVAL;
        sldg_ev_begin(c, KIND_SWEEP, axis);
        e = sldg_launch_sweep_walk(c, fin, fout, g, t);
    }
    sldg_ev_end(c);
    c->launches++;
    if (e != cudaSuccess) { c->last_cuda = (int)e; return SLDG_ECUDA; }
    return SLDG_OK;
}

static int copy_back(sldg_ctx* c, double* dst, const double* src)
{
    if (c->dry) { c->dry_copies++; return SLDG_OK; }
    sldg_ev_begin(c, KIND_COPY, -1);
    cudaError_t e = cudaMemcpyAsync(dst, src, (size_t)c->nf * c->esize, cudaMemcpyDeviceToDevice, c->stream);
    sldg_ev_end(c);
    if (e != cudaSuccess) { c->last_cuda = (int)e; return SLDG_ECUDA; }
    return SLDG_OK;
}

static int check_f(const sldg_ctx* c, const void* f)
{
    if (!c || !f) return SLDG_EINVAL;
    if (((uintptr_t)f) & 15) return SLDG_EINVAL;
    if (!c->ws_ready) return SLDG_ENOWORKSPACE;
    return SLDG_OK;
}

// Run sweeps along axes[0..n) in order on the buffer pair (*cur, *oth); on return *cur holds the result.
// A sweep along a slow axis is out of place (it flips cur/oth).  The sweep along axis 0 stages whole lines in
// shared memory, so it may run in place or out of place: `flip0` selects out of place, which lets the caller fix
// the parity of the flips so that a sequence ends in the caller's buffer without a device copy.
static int run_sweeps(sldg_ctx* c, double** cur, double** oth, const int* axes, const ShiftTable* tabs, int n,
                      bool flip0, int (*prep)(sldg_ctx*, int, void*), void* prep_arg)
{
    for (int i = 0; i < n; i++) {
        if (prep) { int r = prep(c, i, prep_arg); if (r) return r; }
        SweepGeom g = geom_of(c, axes[i]);
        const bool oop = (g.inner != 1) || flip0;
        int r = run_sweep(c, *cur, oop ? *oth : *cur, oop ? nullptr : *oth, axes[i], tabs[i]);
        if (r) return r;
        if (oop) { double* t = *cur; *cur = *oth; *oth = t; }
    }
    return SLDG_OK;
}

// ------------------------------------------------------------------ hot path
// Host-built x-sweep tables for time increment dt (cached per axis).  Also records whether a slow-axis walk with
// this table may run IN PLACE: the walk writes output cell (j + s + 1) mod N after reading cells j and j+1, which
// never overtakes its own reads iff every entry has s mod N in {0, N-1} (|delta| < 1, the BASELINE regime).
static int build_x_tables(sldg_ctx* c, double dt, ShiftTable* tabs)
{
    const long long NN2 = 2LL * c->K1 * c->K1;
    if (c->dry) {
        for (int a = 0; a < c->dx; a++) { c->tab_safe[a] = c->dry_safe != 0; c->tab_anycp[a] = false; tabs[a] = ShiftTable(); }
        return SLDG_OK;
    }
    if (!isfinite(dt)) return SLDG_EINVAL;
    for (int a = 0; a < c->dx; a++) {
        const int b = c->dx + a;
        XTab* x = nullptr;
        for (int i = 0; i < SLDG_XTAB_SLOTS; i++)
            if (c->xtab[a][i].valid && c->xtab[a][i].tau == dt) x = &c->xtab[a][i];
        if (!x) {
            x = &c->xtab[a][0];                             // a free slot, else the least recently used one
            for (int i = 1; i < SLDG_XTAB_SLOTS; i++)
                if (x->valid && (!c->xtab[a][i].valid || c->xtab[a][i].used < x->used)) x = &c->xtab[a][i];
            std::vector<double> delta((size_t)c->D[b]);
            for (long long n = 0; n < c->D[b]; n++) {
                // node coordinate lo + (i + xi_j) h, then delta = (v * dt) / h_x   (reading O3)
                volatile double cell = (double)(n / c->K1) + c->xi[n % c->K1];
                volatile double off = cell * c->h[b];
                volatile double v = c->lo[b] + off;
                volatile double vt = v * dt;
                delta[(size_t)n] = vt / c->h[a];
            }
            sldg_graph_drop(c);                 // a captured step reads these device tables
            x->valid = false;
            int r = upload_table(c, delta.data(), c->D[b], c->cells[a], x->dS, x->dAB);
            if (r) return r;
            bool safe = true, anycp = false;
            for (long long n = 0; n < c->D[b]; n++) {
                if (c->hS[n] & SLDG_COPY_BIT) anycp = true;
                const int sv = c->hS[n] & SLDG_S_MASK;
                if (sv != 0 && sv != c->cells[a] - 1) safe = false;
            }
            x->safe = safe; x->anycp = anycp; x->valid = true; x->tau = dt;
        }
        x->used = ++c->xtab_clock;
        c->tab_safe[a] = x->safe; c->tab_anycp[a] = x->anycp;
        tabs[a].S = x->dS; tabs[a].AB = x->dAB; tabs[a].strideIdx = NN2; tabs[a].strideM = 1;
    }
    return SLDG_OK;
}

// Plan of one x advection: x_1 and x_2 in one fused pass or separately, which sweeps run in place, such that the
// number of buffer flips has the requested parity.  Fewest passes over f wins; ties go to fewer in-place walks.
struct XPlan { bool ok, fused, fused3, x1_oop; bool inplace[3]; int passes, flips; };

static bool fused_possible(const sldg_ctx* c)
{
    if (!c->opt_fuse_x || c->dx < 2) return false;
    if (c->prec == SLDG_F32)            // only the cell-per-thread kernel exists in fp32: its shape rules
        return c->opt_fused_impl != 2 && c->K1 <= 4 && c->cells[0] <= 128 && ((c->K1 * c->D[0] * 4) & 15) == 0 &&
               (size_t)4 * c->K1 * c->D[0] * 4 + 64 <= 227 * 1024;
    return c->D[0] <= c->opt_fused_threads;
}

// the shape rules of sldg_launch_sweep_fused3 (sldg_sweep_fused3.cu), so that a plan never meets NotSupported
static bool fused3_possible(const sldg_ctx* c)
{
    if (!c->opt_fuse3 || !c->opt_fuse_x || c->dx != 3 || c->K1 > 2 || c->cells[0] > 256) return false;
    const long long cellb = (long long)c->K1 * c->D[0] * (long long)c->esize;
    if (cellb & 15) return false;
    long long S = c->opt_f3_threads / c->cells[0];
    if (S < 1) S = 1;
    if (S > c->cells[1]) S = c->cells[1];
    const long long nstrips = (c->cells[1] + S - 1) / S;
    S = (c->cells[1] + nstrips - 1) / nstrips;
    return (size_t)c->K1 * (2 * (S + 1) + 2 * S) * cellb + 64 <= 227 * 1024;
}

static XPlan x_plan(const sldg_ctx* c, bool flip)
{
    XPlan best; best.ok = false; best.fused3 = false; best.passes = 1 << 30; best.flips = 0;
    const int dx = c->dx;
    if (flip && fused3_possible(c)) {       // all three sweeps in one out-of-place pass: one flip
        best.ok = true; best.fused3 = true; best.fused = false; best.x1_oop = true; best.passes = 1; best.flips = 1;
        for (int i = 0; i < 3; i++) best.inplace[i] = false;
        return best;
    }
    for (int fused = fused_possible(c) ? 1 : 0; fused >= 0; fused--) {
        const int first_slow = fused ? 2 : 1;
        const int nslow = dx > first_slow ? dx - first_slow : 0;
        for (int x1oop = fused ? 1 : 0; x1oop <= 1; x1oop++) {
            for (int mask = 0; mask < (1 << nslow); mask++) {
                bool legal = true;
                int nin = 0;
                for (int i = 0; i < nslow; i++)
                    if (mask >> i & 1) { nin++; if (!c->tab_safe[first_slow + i] || !c->opt_inplace_walk) legal = false; }
                if (!legal) continue;
                const int flips = x1oop + nslow - nin, passes = 1 + nslow;
                if ((flips & 1) != (flip ? 1 : 0)) continue;
                const int score = passes * 16 + nin;
                if (!best.ok || score < best.passes) {
                    best.ok = true; best.passes = score; best.fused = fused != 0; best.x1_oop = x1oop != 0;
                    best.flips = flips;
                    for (int i = 0; i < 3; i++) best.inplace[i] = false;
                    for (int i = 0; i < nslow; i++) best.inplace[first_slow + i] = (mask >> i & 1) != 0;
                }
            }
        }
    }
    best.passes /= 16;
    return best;
}

// x-sweeps on (*cur, *oth); `flip` = false: the result ends in the buffer it started in, true: in the other one.
static int advect_x_impl(sldg_ctx* c, double** cur, double** oth, double dt, bool flip)
{
    ShiftTable tabs[3];
    int r = build_x_tables(c, dt, tabs);
    if (r) return r;
    XPlan p = x_plan(c, flip);
    if (!p.ok) return SLDG_EINVAL;          // cannot happen: the unfused plan reaches either parity
    int a = 0;
    if (c->dry && (p.fused3 || p.fused)) {
        c->dry_x++; c->launches++;
        double* t = *cur; *cur = *oth; *oth = t;
        if (p.fused3) return SLDG_OK;
        a = 2;
    } else
    if (p.fused3) {
        SweepGeom g3[3] = {geom_of(c, 0), geom_of(c, 1), geom_of(c, 2)};
        sldg_ev_begin(c, KIND_FUSED, 3);                       // axis field of a fused event = number of fused axes
        const int anycp = (c->tab_anycp[0] || c->tab_anycp[1] || c->tab_anycp[2]) ? 1 : 0;
        cudaError_t e = (c->opt_decline & 4) ? cudaErrorNotSupported
                      : c->prec == SLDG_F32 ? sldg_launch_sweep_fused3_f32(c, *cur, *oth, g3, tabs, anycp)
                                            : sldg_launch_sweep_fused3_f64(c, *cur, *oth, g3, tabs, anycp);
        if (e == cudaErrorNotSupported) {                  // the launcher declined a shape the planner accepted: the
            ev_cancel(c);                                   // same flip parity without the three-sweep pass
            const int keep = c->opt_fuse3;
            c->opt_fuse3 = 0;
            r = advect_x_impl(c, cur, oth, dt, flip);
            c->opt_fuse3 = keep;
            return r;
        }
        sldg_ev_end(c);
        c->launches++;
        if (e != cudaSuccess) { c->last_cuda = (int)e; return SLDG_ECUDA; }
        double* t = *cur; *cur = *oth; *oth = t;
        return SLDG_OK;
    }
    if (p.fused && !c->dry) {
        sldg_ev_begin(c, KIND_FUSED, 0);
        cudaError_t e = cudaErrorNotSupported;
        if (c->opt_fused_impl != 2 && !(c->opt_decline & 8)) e = sldg_launch_sweep_fused_cell(c, *cur, *oth, geom_of(c, 0), geom_of(c, 1), tabs[0], tabs[1], (c->tab_anycp[0] || c->tab_anycp[1]) ? 1 : 0);
        if (e == cudaErrorNotSupported && c->prec == SLDG_F64 && !(c->opt_decline & 8)) e = sldg_launch_sweep_fused(c, *cur, *oth, geom_of(c, 0), geom_of(c, 1), tabs[0], tabs[1]);
        if (e == cudaErrorNotSupported) {                  // both fused kernels declined: the same flip parity from separate sweeps
            ev_cancel(c);
            const int keep = c->opt_fuse_x;
            c->opt_fuse_x = 0;
            r = advect_x_impl(c, cur, oth, dt, flip);
            c->opt_fuse_x = keep;
            return r;
        }
        sldg_ev_end(c);
        c->launches++;
        if (e != cudaSuccess) { c->last_cuda = (int)e; return SLDG_ECUDA; }
        double* t = *cur; *cur = *oth; *oth = t;
        a = 2;
    }
    for (; a < c->dx; a++) {
        const bool oop = (a == 0) ? p.x1_oop : !p.inplace[a];
        r = run_sweep(c, *cur, oop ? *oth : *cur, oop ? nullptr : *oth, a, tabs[a], /*inplace_walk_ok=*/!oop);
        if (r) return r;
        if (oop) { double* t = *cur; *cur = *oth; *oth = t; }
    }
    return SLDG_OK;
}

extern "C" int sldg_advect_x(sldg_ctx* c, double* f, double dt)
{
    int r = check_f(c, f);
    if (r) return r;
    double *cur = f, *oth = c->f2;
    if (c->opt_x_copy) {                                // testing knob: the odd-parity plan (for dim_x = 2 the only
        if ((r = advect_x_impl(c, &cur, &oth, dt, true))) return r;   // one with the fused pass) plus one device copy
        return copy_back(c, f, cur);
    }
    return advect_x_impl(c, &cur, &oth, dt, false);     // ends in f: no copy
}

struct VPrep { const double* E; double dt; };
static int vtable_into(sldg_ctx* c, const VPrep* p, int i, int* S, double* AB)
{
    const int a = c->dx + i;
    if (c->dry) return SLDG_OK;
    sldg_ev_begin(c, KIND_TABLE, a);
    cudaError_t e = sldg_launch_vtable(c, p->E + (long long)i * c->X, p->dt, c->h[a], c->cells[a], S, AB);
    sldg_ev_end(c);
    c->launches++;
    if (e != cudaSuccess) { c->last_cuda = (int)e; return SLDG_ECUDA; }
    return SLDG_OK;
}
static int vprep(sldg_ctx* c, int i, void* arg) { return vtable_into(c, (VPrep*)arg, i, c->vS, c->vAB); }
struct VPrepOff { VPrep p; int first; };
static int vprep_off(sldg_ctx* c, int i, void* arg)
{
    VPrepOff* o = (VPrepOff*)arg;
    return vtable_into(c, &o->p, o->first + i, c->vS, c->vAB);
}

// the fused v_1+v_2 pass (sldg_sweep_fusedv.cu) is planned when its shape rules hold
static bool fusedv_possible(const sldg_ctx* c)
{
    if (!c->opt_fuse_v || c->dx < 2) return false;
    int wx = 0;
    if (!(c->prec == SLDG_F32 ? sldg_fusedv_shape_f32(c, &wx, nullptr) : sldg_fusedv_shape_f64(c, &wx, nullptr))) return false;
    if (c->opt_fuse_v == 2) return true;
    // single precision: a thread moves half the bytes per row for the same per-row work, and the tile rows shrink to
    // 32-64 bytes.  Measured: a small loss for dim_x = 2 (cfg2 7.73 against 7.66 ms per step), a small gain for dim_x = 3
    // (cfg4 35.4 against 36.4, cfg5 57.7 against 59.3: the even number of v flips also lets every x half step of a
    // single step be the one-pass x_1+x_2+x_3 sweep)
    if (c->prec == SLDG_F32 && c->dx < 3) return false;
    // auto: a block walks all of v_2 serially, so the pass pays only when its independent walks (x tiles times planes
    // above v_2) fill the GPU; small problems (BASELINE config 1: 16 tiles) are faster with two wide walk launches
    const long long walks = ((c->X + wx - 1) / wx) * (c->V / (c->D[c->dx] * c->D[c->dx + 1]));
    return walks >= 2LL * c->sm_count;
}
// the fused v_1+v_2+v_3 pass (sldg_sweep_fusedv3.cu): dim_x = dim_v = 3, degree <= 1
static bool fusedv3_possible(const sldg_ctx* c)
{
    if (!c->opt_fuse_v3 || c->dx != 3) return false;
    if (!(c->prec == SLDG_F32 ? sldg_fusedv3_shape_f32(c) : sldg_fusedv3_shape_f64(c))) return false;
    if (c->opt_fuse_v3 == 2) return true;
    // auto: a block walks all of v_3 serially; the pass pays only when its walks (x tiles times v_2 strips) fill the GPU
    const long long walks = ((c->X + 15) / 16) * ((c->cells[4] + 3) / 4);
    return walks >= 2LL * c->sm_count;
}

// How a v advection runs: every sweep a walk (VM_WALKS), v_1+v_2 in one pass and v_3 a walk (VM_FUSED2), or all of
// v_1..v_3 in one pass (VM_FUSED3).  Buffer flips and cost in tenths of a walk pass (measured on B200: the fused
// v_1+v_2 pass 1.3, the fused v_1+v_2+v_3 pass 1.5 walk passes).
enum { VM_WALKS = 0, VM_FUSED2 = 1, VM_FUSED3 = 2 };
static bool v_mode_possible(const sldg_ctx* c, int mode)
{
    return mode == VM_WALKS || (mode == VM_FUSED2 && fusedv_possible(c)) || (mode == VM_FUSED3 && fusedv3_possible(c));
}
static int v_flips(const sldg_ctx* c, int mode) { return mode == VM_FUSED3 ? 1 : mode == VM_FUSED2 ? c->dx - 1 : c->dx; }
static int v_cost(const sldg_ctx* c, int mode) { return mode == VM_FUSED3 ? 15 : mode == VM_FUSED2 ? 13 + 10 * (c->dx - 2) : 10 * c->dx; }
static bool v_mode_forced(const sldg_ctx* c, int mode)       // tests: option value 2 takes the pass whenever the shape allows
{
    return (mode == VM_FUSED3 && c->opt_fuse_v3 == 2) || (mode == VM_FUSED2 && c->opt_fuse_v == 2 && !(c->opt_fuse_v3 == 2 && fusedv3_possible(c)));
}
// the cheapest mode of a v advection inside a run of steps (any buffer parity)
static int v_mode_best(const sldg_ctx* c)
{
    int best = VM_WALKS, cost = 1 << 30;
    for (int m = VM_WALKS; m <= VM_FUSED3; m++) {
        if (!v_mode_possible(c, m)) continue;
        if (v_mode_forced(c, m)) return m;
        if (v_cost(c, m) < cost) { cost = v_cost(c, m); best = m; }
    }
    return best;
}
// the cheapest mode of a v advection on its own whose result must end in the buffer it started in (a copy = 10)
static int v_mode_standalone(const sldg_ctx* c)
{
    int best = VM_WALKS, cost = 1 << 30;
    for (int m = VM_WALKS; m <= VM_FUSED3; m++) {
        if (!v_mode_possible(c, m)) continue;
        if (v_mode_forced(c, m)) return m;
        const int k = v_cost(c, m) + ((v_flips(c, m) & 1) ? 10 : 0);
        if (k < cost) { cost = k; best = m; }
    }
    return best;
}

static int advect_v_impl(sldg_ctx* c, double** cur, double** oth, const double* E, double dt, int mode);
// A fused v pass declined by its launcher (cudaErrorNotSupported for a shape the planner accepted): the separate walks run
// instead, and one device copy restores the buffer parity the plan counted on when theirs differs.  Results are the same
// bits either way (include/sldg.h: the options change speed only).
static int v_fallback(sldg_ctx* c, double** cur, double** oth, const double* E, double dt, int flips_planned)
{
    double* const want = (flips_planned & 1) ? *oth : *cur;
    int r = advect_v_impl(c, cur, oth, E, dt, VM_WALKS);
    if (r) return r;
    if (*cur != want) {
        if ((r = copy_back(c, want, *cur))) return r;
        double* t = *cur; *cur = *oth; *oth = t;
    }
    return SLDG_OK;
}

// v-sweeps on (*cur, *oth) in the given mode; every pass is out of place and flips the pair.
static int advect_v_impl(sldg_ctx* c, double** cur, double** oth, const double* E, double dt, int mode)
{
    int axes[3];
    ShiftTable tabs[3];
    for (int i = 0; i < c->dx; i++) {
        axes[i] = c->dx + i;
        tabs[i].S = c->vS; tabs[i].AB = c->vAB; tabs[i].strideIdx = 1; tabs[i].strideM = c->X;
    }
    VPrep p = {E, dt};
    if (!v_mode_possible(c, mode)) mode = VM_WALKS;
    if (mode == VM_FUSED3) {
        int r;
        if ((r = vtable_into(c, &p, 0, c->vS, c->vAB))) return r;
        if ((r = vtable_into(c, &p, 1, c->vS2, c->vAB2))) return r;
        if ((r = vtable_into(c, &p, 2, c->vS3, c->vAB3))) return r;
        ShiftTable t2 = tabs[1], t3 = tabs[2];
        t2.S = c->vS2; t2.AB = c->vAB2; t3.S = c->vS3; t3.AB = c->vAB3;
        if (!c->dry) {
            sldg_ev_begin(c, KIND_FUSEDV3, c->dx);
            cudaError_t e = (c->opt_decline & 2) ? cudaErrorNotSupported
                          : c->prec == SLDG_F32 ? sldg_launch_sweep_fusedv3_f32(c, *cur, *oth, tabs[0], t2, t3)
                                                : sldg_launch_sweep_fusedv3_f64(c, *cur, *oth, tabs[0], t2, t3);
            if (e == cudaErrorNotSupported) { ev_cancel(c); return v_fallback(c, cur, oth, E, dt, v_flips(c, VM_FUSED3)); }
            sldg_ev_end(c);
            if (e != cudaSuccess) { c->last_cuda = (int)e; return SLDG_ECUDA; }
        } else c->dry_v++;
        c->launches++;
        double* t = *cur; *cur = *oth; *oth = t;
        return SLDG_OK;
    }
    if (mode == VM_FUSED2) {
        int r;
        if ((r = vtable_into(c, &p, 0, c->vS, c->vAB))) return r;
        if ((r = vtable_into(c, &p, 1, c->vS2, c->vAB2))) return r;
        ShiftTable t2 = tabs[1];
        t2.S = c->vS2; t2.AB = c->vAB2;
        if (!c->dry) {
            sldg_ev_begin(c, KIND_FUSEDV, c->dx);                  // axis field: first of the two fused axes
            cudaError_t e = (c->opt_decline & 1) ? cudaErrorNotSupported
                          : c->prec == SLDG_F32 ? sldg_launch_sweep_fusedv_f32(c, *cur, *oth, tabs[0], t2)
                                                : sldg_launch_sweep_fusedv_f64(c, *cur, *oth, tabs[0], t2);
            if (e == cudaErrorNotSupported) { ev_cancel(c); return v_fallback(c, cur, oth, E, dt, v_flips(c, VM_FUSED2)); }
            sldg_ev_end(c);
            if (e != cudaSuccess) { c->last_cuda = (int)e; return SLDG_ECUDA; }
        } else c->dry_v++;
        c->launches++;
        double* t = *cur; *cur = *oth; *oth = t;
        if (c->dx == 2) return SLDG_OK;
        VPrepOff o = {p, 2};
        return run_sweeps(c, cur, oth, axes + 2, tabs + 2, c->dx - 2, false, vprep_off, &o);
    }
    return run_sweeps(c, cur, oth, axes, tabs, c->dx, false, vprep, &p);
}

extern "C" int sldg_advect_v(sldg_ctx* c, double* f, const double* E, double dt)
{
    int r = check_f(c, f);
    if (r) return r;
    if (!E) return SLDG_EINVAL;
    double *cur = f, *oth = c->f2;
    if ((r = advect_v_impl(c, &cur, &oth, E, dt, v_mode_standalone(c)))) return r;
    // an odd number of v passes (dim_x = 1 or 3) leaves the result in the workspace: one device copy.
    // sldg_step avoids it by fixing the parity in its second x half step.
    if (cur != f) return copy_back(c, f, cur);
    return SLDG_OK;
}

extern "C" int sldg_density(sldg_ctx* c, const double* f, double* rho)
{
    int r = check_f(c, f);
    if (r) return r;
    if (!rho) return SLDG_EINVAL;
    if (c->dry) { c->dry_rho++; return SLDG_OK; }
    sldg_ev_begin(c, KIND_RHO, -1);
    cudaError_t e = sldg_launch_density(c, f, rho);
    sldg_ev_end(c);
    if (e != cudaSuccess) { c->last_cuda = (int)e; return SLDG_ECUDA; }
    return SLDG_OK;
}

extern "C" int sldg_poisson(sldg_ctx* c, const double* rho, double* E)
{
    if (!c || !rho || !E) return SLDG_EINVAL;
    if (!c->ws_ready) return SLDG_ENOWORKSPACE;
    if (c->dry) { c->dry_field++; return SLDG_OK; }
    sldg_ev_begin(c, KIND_POISSON, -1);
    cudaError_t e = sldg_launch_poisson(c, rho, E);
    sldg_ev_end(c);
    if (e != cudaSuccess) { c->last_cuda = (int)e; return SLDG_ECUDA; }
    return SLDG_OK;
}

// ---- CGdG Poisson solver
static int cg_default_maxiter(const sldg_ctx* c)
{
    // convergence within about (prod_l N_l (k+1))^(1/dx) iterations, times a safety factor (4, + 20)
    return 4 * (int)llround(pow((double)c->X, 1.0 / c->dx)) + 20;
}

extern "C" int sldg_poisson_cg(sldg_ctx* c, const double* rho, double* E, double tol, int maxiter)
{
    if (!c || !rho || !E || !(tol >= 0.0) || maxiter < 0) return SLDG_EINVAL;
    if (c->k < 1) return SLDG_EINVAL;                       // sigma >= k^2 = 0 gives no penalty: not defined for k = 0
    if (!c->ws_ready) return SLDG_ENOWORKSPACE;
    if (maxiter == 0) maxiter = c->cg_maxiter > 0 ? c->cg_maxiter : cg_default_maxiter(c);
    sldg_ev_begin(c, KIND_POISSON, -1);
    cudaError_t e = sldg_launch_poisson_cg(c, rho, E, tol, maxiter, c->cg_sigma);
    sldg_ev_end(c);
    c->launches++;
    if (e != cudaSuccess) { c->last_cuda = (int)e; return SLDG_ECUDA; }
    return SLDG_OK;
}

extern "C" int sldg_set_poisson_solver(sldg_ctx* c, int solver, double tol, int maxiter, double sigma)
{
    if (!c || solver < 0 || solver > 1 || !(tol >= 0.0) || maxiter < 0) return SLDG_EINVAL;
    if (solver == 1 && c->k < 1) return SLDG_EINVAL;
    sldg_graph_drop(c);
    c->poisson_solver = solver; c->cg_tol = tol; c->cg_maxiter = maxiter;
    c->cg_sigma = sigma > 0.0 ? sigma : sldg_sipg_sigma_default(c->k);
    return SLDG_OK;
}

extern "C" int sldg_cg_reset(sldg_ctx* c)
{
    if (!c) return SLDG_EINVAL;
    if (!c->ws_ready) return SLDG_ENOWORKSPACE;
    CK(cudaMemsetAsync(c->phi, 0, (size_t)c->X * 8, c->stream));
    return SLDG_OK;
}

extern "C" int sldg_cg_info(sldg_ctx* c, int* iters_host, double* relres_host)
{
    if (!c) return SLDG_EINVAL;
    if (!c->ws_ready) return SLDG_ENOWORKSPACE;
    double h[2];
    CK(cudaMemcpyAsync(h, c->cg_info, 16, cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    if (iters_host) *iters_host = (int)h[0];
    if (relres_host) *relres_host = h[1];
    return SLDG_OK;
}

extern "C" const double* sldg_last_phi(const sldg_ctx* c) { return (c && c->ws_ready) ? c->phi : nullptr; }

extern "C" int sldg_sipg_matrices(int degree, double sigma, double* hostM, double* hostB)
{
    if (degree < 1 || degree > SLDG_MAX_DEGREE || !hostM || !hostB) return SLDG_EINVAL;
    double xi[SLDG_MAXK1], w[SLDG_MAXK1], Dm[SLDG_MAXNN];
    sldg_gl_rule(degree + 1, xi, w);
    sldg_sipg_tables(degree, xi, w, sigma > 0.0 ? sigma : sldg_sipg_sigma_default(degree), hostM, hostB, Dm);
    return SLDG_OK;
}

// Two consecutive x half steps with the same time increment (the second of a Strang step and the first of the next
// one) as ONE pass of the fused cell kernel applying the sweep pair twice (sldg_sweep_fused_cell.cu, DBL).
static bool x_double_possible(const sldg_ctx* c)
{
    // dim_x = 3 (sldg_sweep_fused3d.cu): built, bit-identical, and measured SLOWER than two one-pass half steps on B200 (the
    // pass is bound by fp64 issue, not by HBM: cfg4 22.1 against 2 x 11.9 ms at the best tiling, cfg5 43.8 against 2 x 17.5
    // ms), so it is planned only when forced (option x_double = 2)
    if (c->dx == 3) {
        if (c->opt_x_double != 2 || !c->opt_fuse_x || !c->opt_fuse3) return false;
        return c->prec == SLDG_F32 ? sldg_fused3d_shape_f32(c) : sldg_fused3d_shape_f64(c);
    }
    if (!c->opt_x_double || !c->opt_fuse_x || c->dx != 2 || c->K1 > 3 || c->opt_fused_impl == 2) return false;
    if (c->cells[0] > 128 || ((c->K1 * c->D[0] * (long long)c->esize) & 15)) return false;
    return (size_t)(2 + 1) * c->K1 * c->D[0] * c->esize + (size_t)2 * 2 * c->K1 * c->D[0] * c->esize + 64 <= 227 * 1024;
}
static int advect_x_double(sldg_ctx* c, double** cur, double** oth, double tau)
{
    ShiftTable tabs[3];
    int r = build_x_tables(c, tau, tabs);
    if (r) return r;
    if (c->dry) { c->dry_x++; c->launches++; double* t = *cur; *cur = *oth; *oth = t; return SLDG_OK; }
    if (c->dx == 3) {
        SweepGeom g3[3] = {geom_of(c, 0), geom_of(c, 1), geom_of(c, 2)};
        const int anycp3 = (c->tab_anycp[0] || c->tab_anycp[1] || c->tab_anycp[2]) ? 1 : 0;
        sldg_ev_begin(c, KIND_FUSEDX3D, 0);
        cudaError_t e3 = (c->opt_decline & 16) ? cudaErrorNotSupported
                       : c->prec == SLDG_F32 ? sldg_launch_sweep_fused3d_f32(c, *cur, *oth, g3, tabs, anycp3)
                                             : sldg_launch_sweep_fused3d_f64(c, *cur, *oth, g3, tabs, anycp3);
        if (e3 == cudaErrorNotSupported) {                 // declined: the two half steps one after the other (one flip in all)
            ev_cancel(c);
            if ((r = advect_x_impl(c, cur, oth, tau, true))) return r;
            return advect_x_impl(c, cur, oth, tau, false);
        }
        sldg_ev_end(c);
        c->launches++;
        if (e3 != cudaSuccess) { c->last_cuda = (int)e3; return SLDG_ECUDA; }
        double* t3 = *cur; *cur = *oth; *oth = t3;
        return SLDG_OK;
    }
    const int anycp = (c->tab_anycp[0] || c->tab_anycp[1]) ? 1 : 0;
    sldg_ev_begin(c, KIND_FUSEDX2, 0);
    cudaError_t e = (c->opt_decline & 16) ? cudaErrorNotSupported
                  : c->prec == SLDG_F32 ? sldg_launch_sweep_fused_cell2_f32(c, *cur, *oth, geom_of(c, 0), geom_of(c, 1), tabs[0], tabs[1], anycp)
                                        : sldg_launch_sweep_fused_cell2_f64(c, *cur, *oth, geom_of(c, 0), geom_of(c, 1), tabs[0], tabs[1], anycp);
    if (e == cudaErrorNotSupported) {                      // declined: the two half steps one after the other (one flip in all)
        ev_cancel(c);
        if ((r = advect_x_impl(c, cur, oth, tau, true))) return r;
        return advect_x_impl(c, cur, oth, tau, false);
    }
    sldg_ev_end(c);
    c->launches++;
    if (e != cudaSuccess) { c->last_cuda = (int)e; return SLDG_ECUDA; }
    double* t = *cur; *cur = *oth; *oth = t;
    return SLDG_OK;
}

// passes over f of the two x half steps of one Strang step whose total number of buffer flips has parity `flip_total`,
// given the flips of its v advection; *p1 = flip parity of the first x half step that achieves it
static int step_cost(const sldg_ctx* c, bool flip_total, int* p1, int vflips)
{
    int best = 1 << 30;
    for (int q1 = 0; q1 < 2; q1++) {
        const int q2 = (q1 + vflips + (flip_total ? 1 : 0)) & 1;
        XPlan a = x_plan(c, q1 != 0), b = x_plan(c, q2 != 0);
        if (a.ok && b.ok && a.passes + b.passes < best) { best = a.passes + b.passes; if (p1) *p1 = q1; }
    }
    return best;
}
// The cheapest plan of one Strang step in tenths of a pass over f: x passes as above plus the v advection in one of its
// modes (v_cost).  For dim_x = 2 a single step that must end in its own buffer is cheaper WITHOUT the fused v pass (its
// odd flip would cost a two-pass in-place x half step: 43 against 40); for dim_x = 3 such a step takes the fused
// v_1+v_2 pass + the v_3 walk (two flips: both x half steps stay one-pass), while steps that may end in the other buffer
// (sldg_steps) take the one-pass v advection.
static int step_best(const sldg_ctx* c, bool flip_total, int* p1, int* vmode)
{
    int best = 1 << 30, bm = VM_WALKS, bp = 0;
    for (int m = VM_WALKS; m <= VM_FUSED3; m++) {
        if (!v_mode_possible(c, m)) continue;
        int q = 0;
        const int k = 10 * step_cost(c, flip_total, &q, v_flips(c, m)) + v_cost(c, m);
        if (v_mode_forced(c, m)) { best = k; bm = m; bp = q; break; }
        if (k < best) { best = k; bm = m; bp = q; }
    }
    if (p1) *p1 = bp;
    if (vmode) *vmode = bm;
    return best;
}

// One Strang step on the pair (*cur, *oth).  The dx v-sweeps flip the pair dx times; the two x half steps choose
// their flip parities so that the step ends in the buffer it started in (flip_total = false: no device copy for
// the caller's f) or in the other one (flip_total = true: sldg_steps alternates), at the fewest passes over f.
static int step_core(sldg_ctx* c, double** cur, double** oth, double dt, bool flip_total)
{
    int r;
    double* const start = *cur;
    ShiftTable tabs[3];
    if ((r = build_x_tables(c, dt / 2.0, tabs))) return r;
    int p1 = 0;
    int vmode = VM_WALKS;
    step_best(c, flip_total, &p1, &vmode);
    if ((r = advect_x_impl(c, cur, oth, dt / 2.0, p1 != 0))) return r;
    if ((r = sldg_density(c, *cur, c->rho))) return r;
    if ((r = c->poisson_solver == 1 ? sldg_poisson_cg(c, c->rho, c->E, c->cg_tol, 0) : sldg_poisson(c, c->rho, c->E))) return r;
    if ((r = advect_v_impl(c, cur, oth, c->E, dt, vmode))) return r;
    const bool want_other = flip_total;                       // where the step has to end, relative to `start`
    const bool now_other = (*cur != start);
    return advect_x_impl(c, cur, oth, dt / 2.0, now_other != want_other);
}

static int step_enqueue(sldg_ctx* c, double* f, double dt)
{
    double *cur = f, *oth = c->f2;
    int r = step_core(c, &cur, &oth, dt, false);
    if (r) return r;
    if (cur != f) return copy_back(c, f, cur);                                  // unreachable by construction
    return SLDG_OK;
}

// Out-of-place Strang step: the pair (f_in, f_out) takes the place of (f, workspace buffer) and the step is planned to END IN
// THE OTHER BUFFER (flip_total = true), which is the cheapest parity for dim_x = 3 (one-pass x half steps + the one-flip
// v_1v_2v_3 pass: 3 passes + rho) and lets dim_x = 2 use the fused v pass.
extern "C" int sldg_step_to(sldg_ctx* c, double* f_in, double* f_out, double dt, int end_of_step_field)
{
    int r = check_f(c, f_in);
    if (r) return r;
    if ((r = check_f(c, f_out))) return r;
    if (f_in == f_out) return SLDG_EINVAL;
    double *cur = f_in, *oth = f_out;
    if ((r = step_core(c, &cur, &oth, dt, true))) return r;
    if (cur != f_out && (r = copy_back(c, f_out, cur))) return r;              // unreachable by construction
    if (end_of_step_field) {                                                    // rho, E of f(t_{n+1}) for the diagnostics
        if ((r = sldg_density(c, f_out, c->rho))) return r;
        if ((r = c->poisson_solver == 1 ? sldg_poisson_cg(c, c->rho, c->E, c->cg_tol, 0) : sldg_poisson(c, c->rho, c->E))) return r;
    }
    return SLDG_OK;
}
extern "C" double* sldg_workspace_field(const sldg_ctx* c) { return (c && c->ws_ready) ? c->f2 : nullptr; }

void sldg_graph_drop(sldg_ctx* c)
{
    if (c->graph_exec) { cudaGraphExecDestroy(c->graph_exec); c->graph_exec = nullptr; }
}

// Small problems (BASELINE config 1: 2 MB) are launch-latency bound: the ~16 launches of a Strang step are
// captured once into a CUDA graph and replayed.  The graph is keyed on (f, dt) and
// dropped whenever an option, the stream, the workspace or the solver changes.  Not used with timing on (events
// cannot be recorded inside a capture) or with the CG solver (cooperative launch).
extern "C" int sldg_step(sldg_ctx* c, double* f, double dt)
{
    int r = check_f(c, f);
    if (r) return r;
    const bool small = (size_t)c->nf * c->esize <= ((size_t)256 << 20);
    const bool use_graph = !c->timing && c->poisson_solver == 0 && (c->opt_graph == 2 || (c->opt_graph == 1 && small));
    if (!use_graph) return step_enqueue(c, f, dt);
    if (c->graph_exec && c->graph_f == f && c->graph_dt == dt) {
        CK(cudaGraphLaunch(c->graph_exec, c->stream));
        c->launches += c->graph_launches;
        return SLDG_OK;
    }
    sldg_graph_drop(c);
    ShiftTable tabs[3];
    if ((r = build_x_tables(c, dt / 2.0, tabs))) return r;       // host tables + upload (synchronises): before the capture
    const long long l0 = c->launches;
    // A capture cannot be started on the legacy default stream (or the per-thread one): the step is then recorded on a
    // stream of the context's own.  Nothing executes during a capture, so no ordering between the two streams is needed;
    // the instantiated graph is launched on the caller's stream.
    cudaStream_t const user = c->stream;
    cudaStream_t cap = user;
    if (user == 0 || user == cudaStreamLegacy || user == cudaStreamPerThread) {
        if (!c->cap_stream && cudaStreamCreateWithFlags(&c->cap_stream, cudaStreamNonBlocking) != cudaSuccess) {
            c->cap_stream = nullptr;
            cudaGetLastError();
            return step_enqueue(c, f, dt);
        }
        cap = c->cap_stream;
    }
    if (cudaStreamBeginCapture(cap, cudaStreamCaptureModeThreadLocal) != cudaSuccess) {
        cudaGetLastError();
        return step_enqueue(c, f, dt);
    }
    c->stream = cap;
    r = step_enqueue(c, f, dt);
    c->stream = user;
    cudaGraph_t g = nullptr;
    cudaError_t e = cudaStreamEndCapture(cap, &g);
    if (r || e != cudaSuccess || !g) {
        if (g) cudaGraphDestroy(g);
        cudaGetLastError();
        c->launches = l0;
        if (r) return r;
        return step_enqueue(c, f, dt);                          // capture not possible: plain launches
    }
    e = cudaGraphInstantiate(&c->graph_exec, g, 0);
    cudaGraphDestroy(g);
    if (e != cudaSuccess) { c->graph_exec = nullptr; cudaGetLastError(); c->launches = l0; return step_enqueue(c, f, dt); }
    c->graph_f = f; c->graph_dt = dt; c->graph_launches = c->launches - l0;
    CK(cudaGraphLaunch(c->graph_exec, c->stream));
    return SLDG_OK;
}

extern "C" int sldg_graph_active(const sldg_ctx* c) { return (c && c->graph_exec) ? 1 : 0; }

// nsteps Strang steps.  Consecutive steps may leave their result in alternate buffers when that saves passes (for
// dim_x = 3 both x half steps of a step can then be the one-pass fused x_1+x_2+x_3 sweep); the last step restores
// the parity, so the result is in f.  Same arithmetic as nsteps calls of sldg_step, bit for bit.
extern "C" int sldg_steps(sldg_ctx* c, double* f, double dt, int nsteps)
{
    int r = check_f(c, f);
    if (r) return r;
    if (nsteps < 0) return SLDG_EINVAL;
    const bool small = (size_t)c->nf * c->esize <= ((size_t)256 << 20);
    if (!c->timing && c->poisson_solver == 0 && (c->opt_graph == 2 || (c->opt_graph == 1 && small))) {
        for (int s = 0; s < nsteps; s++)
            if ((r = sldg_step(c, f, dt))) return r;            // small problems: graph replay per step
        return SLDG_OK;
    }
    ShiftTable tabs[3];
    if ((r = build_x_tables(c, dt / 2.0, tabs))) return r;      // fills tab_safe, which the plans depend on
    double *cur = f, *oth = c->f2;
    // n - 1 merged passes save n - 1 passes over f; restoring the buffer parity at the end costs one of them back when
    // the number of flips is odd (2 steps with an even number of v flips: nothing gained, the plain plan runs)
    const int vm = v_mode_best(c);
    if (x_double_possible(c) && (nsteps >= 3 || (nsteps == 2 && (v_flips(c, vm) & 1)))) {
        // x(dt/2) | rho, E, v(dt) | x(dt/2) x(dt/2) as one pass | rho, E, v(dt) | ... | x(dt/2): the same sweeps in the
        // same order as nsteps single steps.  The last half step restores the buffer parity.
        if ((r = advect_x_impl(c, &cur, &oth, dt / 2.0, true))) return r;
        // The closing half step is one pass only if it may flip the buffers, i.e. if the flips before it are odd in
        // number: 1 + nsteps * v_flips + (nsteps - 1).  With a one-flip v pass that count is even: the LAST v advection
        // then runs in the cheapest mode of the other flip parity (dim_x = 2: two walks, 0.7 pass more; dim_x = 3: the
        // fused v_1+v_2 pass + the v_3 walk, 0.8 pass more) when that costs less than the x pass it saves.
        int vm_last = vm;
        if ((1 + nsteps * v_flips(c, vm) + (nsteps - 1)) % 2 == 0) {
            const int gain = 10 * (x_plan(c, false).passes - x_plan(c, true).passes);
            int extra = gain;
            for (int m = VM_WALKS; m <= VM_FUSED3; m++)
                if (v_mode_possible(c, m) && ((v_flips(c, m) ^ v_flips(c, vm)) & 1) && v_cost(c, m) - v_cost(c, vm) < extra) {
                    extra = v_cost(c, m) - v_cost(c, vm); vm_last = m;
                }
        }
        for (int s = 0; s < nsteps; s++) {
            if ((r = sldg_density(c, cur, c->rho))) return r;
            if ((r = c->poisson_solver == 1 ? sldg_poisson_cg(c, c->rho, c->E, c->cg_tol, 0) : sldg_poisson(c, c->rho, c->E))) return r;
            if ((r = advect_v_impl(c, &cur, &oth, c->E, dt, s == nsteps - 1 ? vm_last : vm))) return r;
            if (s < nsteps - 1) r = advect_x_double(c, &cur, &oth, dt / 2.0);
            else r = advect_x_impl(c, &cur, &oth, dt / 2.0, cur != f);
            if (r) return r;
        }
        if (cur != f) return copy_back(c, f, cur);              // unreachable by construction
        return SLDG_OK;
    }
    for (int s = 0; s < nsteps; s++) {
        bool flip;
        if (s == nsteps - 1) flip = (cur != f);                 // the last step ends in f
        else flip = step_best(c, true, nullptr, nullptr) < step_best(c, false, nullptr, nullptr);
        if ((r = step_core(c, &cur, &oth, dt, flip))) return r;
    }
    if (cur != f) return copy_back(c, f, cur);                  // unreachable by construction
    return SLDG_OK;
}

// Host-only: run the planning code of sldg_step (nsteps == 0) or sldg_steps(nsteps) on a context without a device and
// count what it would launch.  The same functions plan and launch (c->dry only replaces the launches), so the counts
// are those of the real calls.
static int plan_query_impl(int dim_x, int dim_v, const int* cells, int degree, int precision, int nsteps,
                           int shifts_below_one, int fuse_v, int fuse_v3, int x_double, long long* counts, bool step_to)
{
    if (!counts || nsteps < 0 || fuse_v < 0 || fuse_v > 2 || fuse_v3 < 0 || fuse_v3 > 2 || x_double < 0 || x_double > 2) return SLDG_EINVAL;
    if (precision != SLDG_F64 && precision != SLDG_F32) return SLDG_EINVAL;
    if (dim_x < 1 || dim_x > 3) return SLDG_EINVAL;
    double dom[2 * SLDG_MAX_DIM];
    for (int a = 0; a < SLDG_MAX_DIM; a++) { dom[2 * a] = 0.0; dom[2 * a + 1] = 1.0; }
    sldg_ctx* c = nullptr;
    int r = create_impl(&c, dim_x, dim_v, cells, degree, dom, precision, true);
    if (r) return r;
    c->dry = true; c->dry_safe = shifts_below_one; c->opt_graph = 0; c->opt_fuse_v = fuse_v; c->opt_fuse_v3 = fuse_v3; c->opt_x_double = x_double;
    c->ws_ready = true;
    // distinct, aligned, never dereferenced: the planner only compares and swaps them
    double* f = reinterpret_cast<double*>((uintptr_t)0x10000);
    c->f2 = reinterpret_cast<double*>((uintptr_t)0x20000);
    c->rho = c->E = reinterpret_cast<double*>((uintptr_t)0x30000);
    if (step_to) r = sldg_step_to(c, f, reinterpret_cast<double*>((uintptr_t)0x40000), 0.1, nsteps);   // nsteps carries end_of_step_field
    else r = nsteps == 0 ? sldg_step(c, f, 0.1) : sldg_steps(c, f, 0.1, nsteps);
    counts[0] = c->dry_x; counts[1] = c->dry_v; counts[2] = c->dry_rho; counts[3] = c->dry_field; counts[4] = c->dry_copies;
    counts[5] = c->launches;
    delete c;
    return r;
}

extern "C" int sldg_plan_query(int dim_x, int dim_v, const int* cells, int degree, int precision, int nsteps,
                               int shifts_below_one, int fuse_v, int fuse_v3, int x_double, long long* counts)
{
    return plan_query_impl(dim_x, dim_v, cells, degree, precision, nsteps, shifts_below_one, fuse_v, fuse_v3, x_double, counts, false);
}
extern "C" int sldg_plan_query_step_to(int dim_x, int dim_v, const int* cells, int degree, int precision, int end_of_step_field,
                                       int shifts_below_one, int fuse_v, int fuse_v3, int x_double, long long* counts)
{
    if (end_of_step_field < 0 || end_of_step_field > 1) return SLDG_EINVAL;
    return plan_query_impl(dim_x, dim_v, cells, degree, precision, end_of_step_field, shifts_below_one, fuse_v, fuse_v3, x_double, counts, true);
}

extern "C" int sldg_step_host(sldg_ctx* c, double* f_host, double* f_dev, double* E_host, double dt, int nsteps)
{
    int r = check_f(c, f_dev);
    if (r) return r;
    if (!f_host || nsteps < 0) return SLDG_EINVAL;
    CK(cudaMemcpyAsync(f_dev, f_host, (size_t)c->nf * c->esize, cudaMemcpyHostToDevice, c->stream));
    if ((r = sldg_steps(c, f_dev, dt, nsteps))) return r;
    CK(cudaMemcpyAsync(f_host, f_dev, (size_t)c->nf * c->esize, cudaMemcpyDeviceToHost, c->stream));
    if (E_host) CK(cudaMemcpyAsync(E_host, c->E, (size_t)c->X * 8 * c->dx, cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    return SLDG_OK;
}

extern "C" int sldg_advect_axis(sldg_ctx* c, double* f, int axis, const double* delta_host)
{
    int r = check_f(c, f);
    if (r) return r;
    if (!delta_host || axis < 0 || axis >= c->d) return SLDG_EINVAL;
    ShiftTable t;
    const long long NN2 = 2LL * c->K1 * c->K1;
    if (axis < c->dx) {
        const int b = c->dx + axis;
        r = upload_table(c, delta_host, c->D[b], c->cells[axis], c->dS_hook, c->dAB_hook);
        if (r) return r;
        t.S = c->dS_hook; t.AB = c->dAB_hook; t.strideIdx = NN2; t.strideM = 1;
    } else {
        // per-x-node table, built on the host with the same host routine, stored SoA like the device-built one
        const long long X = c->X;
        const int NN = c->K1 * c->K1;
        std::vector<int> S((size_t)X);
        std::vector<double> AB((size_t)(X * NN2)), ent((size_t)NN2);
        for (long long x = 0; x < X; x++)
            if (!isfinite(delta_host[x])) return SLDG_EINVAL;
        for (long long x = 0; x < X; x++) {
            host_entry(c, delta_host[x], c->cells[axis], &S[(size_t)x], ent.data());
            for (int m = 0; m < 2 * NN; m++) AB[(size_t)((long long)m * X + x)] = ent[(size_t)m];
        }
        CK(cudaStreamSynchronize(c->stream));
        CK(cudaMemcpy(c->vS, S.data(), (size_t)X * 4, cudaMemcpyHostToDevice));
        if (c->prec == SLDG_F32) {
            std::vector<float> AB4(AB.size());
            for (size_t i = 0; i < AB.size(); i++) AB4[i] = (float)AB[i];
            CK(cudaMemcpy(c->vAB, AB4.data(), AB4.size() * 4, cudaMemcpyHostToDevice));
        } else
            CK(cudaMemcpy(c->vAB, AB.data(), (size_t)(X * NN2) * 8, cudaMemcpyHostToDevice));
        t.S = c->vS; t.AB = c->vAB; t.strideIdx = 1; t.strideM = X;
    }
    int axes[1] = {axis};
    double *cur = f, *oth = c->f2;
    if ((r = run_sweeps(c, &cur, &oth, axes, &t, 1, false, nullptr, nullptr))) return r;
    if (cur != f) return copy_back(c, f, cur);
    return SLDG_OK;
}

// ------------------------------------------------------------------ helpers
extern "C" long long sldg_field_elems(const sldg_ctx* c) { return c ? c->nf : 0; }
extern "C" long long sldg_rho_elems(const sldg_ctx* c) { return c ? c->X : 0; }
extern "C" int sldg_nodes(const sldg_ctx* c, int axis)
{
    if (!c || axis < 0 || axis >= c->d) return SLDG_EINVAL;
    return (int)c->D[axis];
}
extern "C" int sldg_node_coords(const sldg_ctx* c, int axis, double* host_out)
{
    if (!c || !host_out || axis < 0 || axis >= c->d) return SLDG_EINVAL;
    for (long long n = 0; n < c->D[axis]; n++) {
        volatile double cell = (double)(n / c->K1) + c->xi[n % c->K1];
        volatile double off = cell * c->h[axis];
        host_out[n] = c->lo[axis] + off;
    }
    return SLDG_OK;
}
extern "C" const double* sldg_last_rho(const sldg_ctx* c) { return (c && c->ws_ready) ? c->rho : nullptr; }
extern "C" const double* sldg_last_E(const sldg_ctx* c) { return (c && c->ws_ready) ? c->E : nullptr; }

static int scalar_out(sldg_ctx* c, cudaError_t e, double* host_out)
{
    if (e != cudaSuccess) { c->last_cuda = (int)e; return SLDG_ECUDA; }
    CK(cudaMemcpyAsync(host_out, c->dScalar, 8, cudaMemcpyDeviceToHost, c->stream));
    CK(cudaStreamSynchronize(c->stream));
    return SLDG_OK;
}
extern "C" int sldg_electric_energy(sldg_ctx* c, const double* E, double* host_out)
{
    if (!c || !E || !host_out) return SLDG_EINVAL;
    if (!c->ws_ready) return SLDG_ENOWORKSPACE;
    return scalar_out(c, sldg_launch_energy(c, E, c->dScalar), host_out);
}
extern "C" int sldg_mass(sldg_ctx* c, const double* f, double* host_out)
{
    if (!c || !f || !host_out) return SLDG_EINVAL;
    if (!c->ws_ready) return SLDG_ENOWORKSPACE;
    return scalar_out(c, sldg_launch_mass(c, f, c->dScalar), host_out);
}
extern "C" int sldg_abi_version(void) { return SLDG_ABI_VERSION; }
extern "C" const char* sldg_strerror(int code)
{
    switch (code) {
    case SLDG_OK: return "ok";
    case SLDG_EINVAL: return "invalid argument";
    case SLDG_ENOMEM: return "out of memory";
    case SLDG_ECUDA: return "CUDA runtime error (see sldg_last_cuda_error); no CPU fallback exists";
    case SLDG_ENOWORKSPACE: return "workspace missing or too small";
    case SLDG_ETOOLARGE: return "x grid exceeds SLDG_DENSITY_STATIC_MAX_X nodes: sldg_density_static has a fixed scratch array; use sldg_density";
    }
    return "unknown error";
}
extern "C" int sldg_last_cuda_error(const sldg_ctx* c) { return c ? c->last_cuda : 0; }

template <int K1>
static void ab_device_arith(const ABPoly& p, double alpha, double* A, double* B)
{
    const double xc = alpha - 0.5;
    for (int m = 0; m < K1 * K1; m++) { A[m] = sldg_horner<K1>(p, 0, m, xc); B[m] = sldg_horner<K1>(p, 1, m, xc); }
}

extern "C" int sldg_AB(int degree, double alpha, int device_arith, double* A, double* B)
{
    if (degree < 0 || degree > SLDG_MAX_DEGREE || !A || !B || !(alpha >= 0.0 && alpha <= 1.0)) return SLDG_EINVAL;
    double xi[SLDG_MAXK1], w[SLDG_MAXK1];
    sldg_gl_rule(degree + 1, xi, w);
    ABPoly* p = new (std::nothrow) ABPoly;
    ABPolyLD* pl = new (std::nothrow) ABPolyLD;
    if (!p || !pl) { delete p; delete pl; return SLDG_ENOMEM; }
    sldg_build_poly(degree, xi, w, p, pl);
    if (!device_arith) sldg_eval_AB_host(pl, degree, alpha, A, B);
    else switch (degree) {
        case 0: ab_device_arith<1>(*p, alpha, A, B); break;
        case 1: ab_device_arith<2>(*p, alpha, A, B); break;
        case 2: ab_device_arith<3>(*p, alpha, A, B); break;
        case 3: ab_device_arith<4>(*p, alpha, A, B); break;
        default: ab_device_arith<5>(*p, alpha, A, B); break;
    }
    delete p; delete pl;
    return SLDG_OK;
}

extern "C" int sldg_gauss_legendre(int degree, double* xi, double* w)
{
    if (degree < 0 || degree > SLDG_MAX_DEGREE || !xi || !w) return SLDG_EINVAL;
    sldg_gl_rule(degree + 1, xi, w);
    return SLDG_OK;
}

// ------------------------------------------------------------------ instrumentation API
extern "C" int sldg_timing_enable(sldg_ctx* c, int on)
{
    if (!c) return SLDG_EINVAL;
    c->timing = on != 0;
    return SLDG_OK;
}
extern "C" int sldg_timing_read(sldg_ctx* c, long long* launches, double* ms)
{
    if (!c || !launches || !ms) return SLDG_EINVAL;
    CK(cudaStreamSynchronize(c->stream));
    if (c->ev_failed) {                                     // some launches went unrecorded: no partial figures
        for (auto& r : c->ev) c->ev_free.push_back(r);
        c->ev.clear(); c->ev_failed = false;
        return SLDG_ECUDA;
    }
    memset(c->t_launch, 0, sizeof(c->t_launch)); memset(c->t_ms, 0, sizeof(c->t_ms));
    memset(c->a_launch, 0, sizeof(c->a_launch)); memset(c->a_ms, 0, sizeof(c->a_ms));
    for (auto& r : c->ev) {
        float t = 0.f;
        if (cudaEventElapsedTime(&t, r.a, r.b) == cudaSuccess) {
            c->t_launch[r.kind]++; c->t_ms[r.kind] += t;
            if ((r.kind == KIND_SWEEP0 || r.kind == KIND_SWEEP) && r.axis >= 0) { c->a_launch[r.axis]++; c->a_ms[r.axis] += t; }
            if (r.kind == KIND_FUSED) { const int nf = r.axis == 3 ? 3 : 2; for (int a = 0; a < nf; a++) { c->a_launch[a]++; c->a_ms[a] += t / nf; } }
            if (r.kind == KIND_FUSEDX2) { for (int a = 0; a < 2; a++) { c->a_launch[a] += 2; c->a_ms[a] += t / 2; } }   // four sweeps
            if (r.kind == KIND_FUSEDV3) { for (int a = r.axis; a < r.axis + 3; a++) { c->a_launch[a]++; c->a_ms[a] += t / 3; } }
            if (r.kind == KIND_FUSEDX3D) { for (int a = 0; a < 3; a++) { c->a_launch[a] += 2; c->a_ms[a] += t / 3; } }    // six sweeps
            if (r.kind == KIND_FUSEDV) { for (int a = r.axis; a < r.axis + 2; a++) { c->a_launch[a]++; c->a_ms[a] += t / 2; } }
        }
        c->ev_free.push_back(r);
    }
    c->ev.clear();
    for (int i = 0; i < SLDG_NKINDS; i++) { launches[i] = c->t_launch[i]; ms[i] = c->t_ms[i]; }
    return SLDG_OK;
}
extern "C" int sldg_timing_axis(const sldg_ctx* c, long long* launches, double* ms)
{
    if (!c || !launches || !ms) return SLDG_EINVAL;
    for (int i = 0; i < SLDG_MAX_DIM; i++) { launches[i] = c->a_launch[i]; ms[i] = c->a_ms[i]; }
    return SLDG_OK;
}
extern "C" long long sldg_launch_count(const sldg_ctx* c) { return c ? c->launches : 0; }

extern "C" int sldg_set_option(sldg_ctx* c, const char* name, long long value)
{
    if (!c || !name) return SLDG_EINVAL;
    sldg_graph_drop(c);
    if (!strcmp(name, "graph")) { if (value < 0 || value > 2) return SLDG_EINVAL; c->opt_graph = (int)value; return SLDG_OK; }
    if (!strcmp(name, "tile_bytes")) { if (value < 256 || value > 96 * 1024) return SLDG_EINVAL; c->opt_tile_bytes = (int)value; return SLDG_OK; }
    if (!strcmp(name, "axis0_impl")) { if (value < 0 || value > 3) return SLDG_EINVAL; c->opt_axis0_impl = (int)value; return SLDG_OK; }
    if (!strcmp(name, "tile_stages")) { if (value < 1 || value > 4) return SLDG_EINVAL; c->opt_tile_stages = (int)value; return SLDG_OK; }
    if (!strcmp(name, "walk_block")) { if (value < 32 || value > 256 || (value & 31)) return SLDG_EINVAL; c->opt_walk_block = (int)value; return SLDG_OK; }
    if (!strcmp(name, "fuse_x")) { if (value < 0 || value > 1) return SLDG_EINVAL; c->opt_fuse_x = (int)value; return SLDG_OK; }
    if (!strcmp(name, "inplace_walk")) { if (value < 0 || value > 1) return SLDG_EINVAL; c->opt_inplace_walk = (int)value; return SLDG_OK; }
    if (!strcmp(name, "fused_threads")) { if (value < 1 || value > 256) return SLDG_EINVAL; c->opt_fused_threads = (int)value; return SLDG_OK; }
    if (!strcmp(name, "fuse3")) { if (value < 0 || value > 1) return SLDG_EINVAL; c->opt_fuse3 = (int)value; return SLDG_OK; }
    if (!strcmp(name, "f3_threads")) { if (value < 1 || value > 256) return SLDG_EINVAL; c->opt_f3_threads = (int)value; return SLDG_OK; }
    if (!strcmp(name, "f3d_threads")) { if (value < 1 || value > 256) return SLDG_EINVAL; c->opt_f3d_threads = (int)value; return SLDG_OK; }
    if (!strcmp(name, "f3_stages")) { if (value < 2 || value > 4) return SLDG_EINVAL; c->opt_f3_stages = (int)value; return SLDG_OK; }
    if (!strcmp(name, "x_copy")) { if (value < 0 || value > 1) return SLDG_EINVAL; c->opt_x_copy = (int)value; return SLDG_OK; }
    if (!strcmp(name, "fused_impl")) { if (value < 0 || value > 2) return SLDG_EINVAL; c->opt_fused_impl = (int)value; return SLDG_OK; }
    if (!strcmp(name, "cell_threads")) { if (value < 1 || value > 128) return SLDG_EINVAL; c->opt_cell_threads = (int)value; return SLDG_OK; }
    if (!strcmp(name, "cell_rows")) { if (value < 0 || value > 1024) return SLDG_EINVAL; c->opt_cell_rows = (int)value; return SLDG_OK; }
    if (!strcmp(name, "cell_bytes")) { if (value < 256 || value > 96 * 1024) return SLDG_EINVAL; c->opt_cell_bytes = (int)value; return SLDG_OK; }
    if (!strcmp(name, "cell_stages")) { if (value < 2 || value > 6) return SLDG_EINVAL; c->opt_cell_stages = (int)value; return SLDG_OK; }
    if (!strcmp(name, "poisson_small")) { if (value < 0 || value > 1) return SLDG_EINVAL; c->opt_poisson_small = (int)value; return SLDG_OK; }
    if (!strcmp(name, "x_double")) { if (value < 0 || value > 2) return SLDG_EINVAL; c->opt_x_double = (int)value; return SLDG_OK; }
    if (!strcmp(name, "fuse_v")) { if (value < 0 || value > 2) return SLDG_EINVAL; c->opt_fuse_v = (int)value; return SLDG_OK; }
    if (!strcmp(name, "decline")) { if (value < 0 || value > 31) return SLDG_EINVAL; c->opt_decline = (int)value; return SLDG_OK; }
    if (!strcmp(name, "fuse_v3")) { if (value < 0 || value > 2) return SLDG_EINVAL; c->opt_fuse_v3 = (int)value; return SLDG_OK; }
    if (!strcmp(name, "fv3_wx")) { if (value < 0 || value > 256) return SLDG_EINVAL; c->opt_fv3_wx = (int)value; return SLDG_OK; }
    if (!strcmp(name, "fv3_strip")) { if (value < 0 || value > 5) return SLDG_EINVAL; c->opt_fv3_strip = (int)value; return SLDG_OK; }
    if (!strcmp(name, "fv3_pw")) { if (value < 0 || value > 1) return SLDG_EINVAL; c->opt_fv3_pw = (int)value; return SLDG_OK; }
    if (!strcmp(name, "fv3_slots")) { if (value < 0 || value > 24) return SLDG_EINVAL; c->opt_fv3_slots = (int)value; return SLDG_OK; }
    if (!strcmp(name, "fv_wx")) { if (value < 0 || value > 256) return SLDG_EINVAL; c->opt_fv_wx = (int)value; return SLDG_OK; }
    if (!strcmp(name, "fv_stages")) { if (value < 0 || value > 24) return SLDG_EINVAL; c->opt_fv_stages = (int)value; return SLDG_OK; }
    if (!strcmp(name, "fv_inflight")) { if (value < 1024 || value > 220 * 1024) return SLDG_EINVAL; c->opt_fv_inflight = (int)value; return SLDG_OK; }
    if (!strcmp(name, "fv_ppb")) { if (value < 0 || value > (1 << 20)) return SLDG_EINVAL; c->opt_fv_ppb = (int)value; return SLDG_OK; }
    if (!strcmp(name, "fv_cps")) { if (value < 1 || value > 8) return SLDG_EINVAL; c->opt_fv_cps = (int)value; return SLDG_OK; }
    if (!strcmp(name, "fv_l2")) { if (value < 0 || value > 3) return SLDG_EINVAL; c->opt_fv_l2 = (int)value; return SLDG_OK; }
    if (!strcmp(name, "rho_tma")) { if (value < 0 || value > 1) return SLDG_EINVAL; c->opt_rho_tma = (int)value; return SLDG_OK; }
    if (!strcmp(name, "rho_vec")) { if (value < 0 || value > 2) return SLDG_EINVAL; c->opt_rho_vec = (int)value; return SLDG_OK; }
    if (!strcmp(name, "rho_blocks")) { if (value < 1 || value > 64) return SLDG_EINVAL; c->opt_rho_blocks = (int)value; return SLDG_OK; }
    if (!strcmp(name, "walk_vec")) { if (value < 0 || value > 2) return SLDG_EINVAL; c->opt_walk_vec = (int)value; return SLDG_OK; }
    return SLDG_EINVAL;
}
