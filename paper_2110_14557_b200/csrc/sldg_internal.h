// sldg_internal.h -- private declarations of the sm_100a SLDG library (see include/sldg.h).
// Nothing in this directory includes, links or calls anything under oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

#include <vector>

#include "../../include/sldg.h"

#define SLDG_MAXK1 (SLDG_MAX_DEGREE + 1)
#define SLDG_MAXNN (SLDG_MAXK1 * SLDG_MAXK1)
#define SLDG_MAXPOLY (2 * SLDG_MAX_DEGREE + 2)   // A_jl(alpha) has degree <= 2k+1

// bit 30 of a table's s-entry marks alpha == 0 (pure copy, exact permutation)
#define SLDG_COPY_BIT (1 << 30)
#define SLDG_S_MASK (SLDG_COPY_BIT - 1)

enum { KIND_SWEEP0 = 0, KIND_SWEEP = 1, KIND_RHO = 2, KIND_POISSON = 3, KIND_TABLE = 4, KIND_COPY = 5, KIND_FUSED = 6, KIND_FUSEDV = 7, KIND_FUSEDX2 = 8, KIND_FUSEDV3 = 9, KIND_FUSEDX3D = 10, KIND_UPLOAD = 11 };

// Polynomial coefficients of A_jl(alpha), B_jl(alpha) in powers of (alpha - 1/2), ascending, row-major
// [2][K1*K1][SLDG_MAXPOLY]; the fp64 copy is uploaded per context (dPoly) for the device-side table kernel.
struct ABPoly {
    double c[2][SLDG_MAXNN][SLDG_MAXPOLY];
};
struct ABPolyLD {
    long double c[2][SLDG_MAXNN][SLDG_MAXPOLY];
};

// fp64 Horner evaluation of entry m of A (which = 0) or B (which = 1) at xc = alpha - 1/2: the arithmetic of the
// device-side table kernel; also compiled for the host so that CPU tests can check it (sldg_AB, device_arith = 1).
#ifdef __CUDACC__
#define SLDG_HD __host__ __device__ __forceinline__
#else
#define SLDG_HD inline
#endif
template <int K1, class Coef>
SLDG_HD double sldg_horner(const Coef& c, int which, int m, double xc)
{
    constexpr int DEG = 2 * K1 - 1;
    double a = c.c[which][m][DEG];
#pragma unroll
    for (int t = DEG - 1; t >= 0; t--) a = fma(a, xc, c.c[which][m][t]);
    return a;
}

struct ShiftTable {          // device-resident shift table of one sweep
    const int* S;            // [n]  (s mod N) | copy bit
    const void* AB;          // A then B (double, or float in single precision mode), element m of index i at AB[i*strideIdx + m*strideM]
    long long strideIdx, strideM;
};

struct SweepGeom {
    long long inner, outer;  // prod of D_b below / above the axis
    int N, K1;               // cells along the axis, nodes per cell
    // shift index of the line at (inner p, outer q):
    //   mode 0: (q / sdiv) % smod      (x-sweeps: node of the matching v axis)
    //   mode 1: p % smod               (v-sweeps: flat x node, smod = X)
    int mode;
    long long sdiv, smod;
};

struct EventRec { cudaEvent_t a, b; int kind, axis; };

#define SLDG_XTAB_SLOTS 2
struct XTab {                   // one cached x-sweep shift table (device): [D_{dx+a}] and [D_{dx+a}][2 K1^2]
    int* dS; double* dAB;
    double tau;                 // time increment it was built for
    bool valid, anycp, safe;
    unsigned long long used;    // last use (context clock)
};

struct sldg_ctx {
    int dx, dv, d, k, K1;
    int prec;                       // SLDG_F64 / SLDG_F32: storage and sweep arithmetic type of f (reading W)
    size_t esize;                   // bytes per value of f
    int cells[SLDG_MAX_DIM];
    long long D[SLDG_MAX_DIM];
    double lo[SLDG_MAX_DIM], hi[SLDG_MAX_DIM], h[SLDG_MAX_DIM];
    long long nf, X, V;
    double xi[SLDG_MAXK1], w[SLDG_MAXK1];
    ABPoly poly;
    ABPolyLD poly_ld;

    cudaStream_t stream;
    int last_cuda;
    int sm_count;

    // ctx-owned small device tables
    // x-sweep shift tables: per x axis a cache of SLDG_XTAB_SLOTS tables (a Strang run alternates between dt/2 and, through
    // sldg_advect_x, other increments: two slots keep both resident, least recently used evicted)
    XTab xtab[3][SLDG_XTAB_SLOTS];
    unsigned long long xtab_clock;
    bool tab_anycp[SLDG_MAX_DIM];   // of the table selected by the last build_x_tables: some entry has alpha == 0 (copy bit)
    bool tab_safe[SLDG_MAX_DIM];    //   "   : every shift is 0 or -1: a walk may run in place
    bool ev_failed;                 // an instrumentation event could not be created: sldg_timing_read reports it
    int* dS_hook; double* dAB_hook; long long hook_cap;   // test-hook tables (x axes)
    double* dFwdT[3];               // forward transfer+DFT matrices, transposed [n][m], re then im
    double* dInvT[3];               // inverse DFT+transfer matrices, transposed
    double* dKap[3];                // signed wave numbers per x axis [D_a], Nyquist kept (zeroed in-kernel)
    double* dWx[SLDG_MAX_DIM];      // per-axis quadrature weights h_a w_j  [D_a]
    ABPoly* dPoly;                  // device copy of `poly` (v-sweep table kernel); per context: the layout depends on k
    double* dScalar;                // 1 double result of mass / energy
    unsigned long long* dCounter;   // [2] work counter of the persistent axis-0 kernel (self-resetting)
    int* hS; double* hAB;           // pinned host staging for table uploads
    long long hcap;

    // caller-owned workspace
    char* ws; size_t ws_bytes;
    double* f2;                     // second f buffer
    int* vS; double* vAB;           // v-sweep tables [X], [2 K1^2][X]
    int* vS2; double* vAB2;         // second v-sweep table (the fused v_1+v_2 pass needs both at once)
    int* vS3; double* vAB3;         // third one (fused v_1+v_2+v_3 pass, dim_x = 3)
    double* Wv;                     // [V]
    double* rho; double* E;         // [X], [dx][X]
    double* part; long long part_cap;   // rho partial sums
    double* cplx[6];                // complex scratch, X doubles each
    double* red;                    // reduction partials [4096]
    double* phi;                    // [X] potential of the CGdG solver (warm start of the next solve)
    double* cg_info;                // [4] iterations, relative residual of the last CGdG solve
    int poisson_solver;             // 0 = FFT route (reading P1), 1 = CGdG
    double cg_tol, cg_sigma; int cg_maxiter;
    bool ws_ready;

    // dry run (sldg_plan_query): the planning code runs unchanged, every launch site only counts what it would launch
    bool dry; int dry_safe;
    long long dry_x, dry_v, dry_rho, dry_field, dry_copies;   // passes over f by kind, field solves, device copies

    // instrumentation
    bool timing;
    std::vector<EventRec> ev;       // recorded since last read
    std::vector<EventRec> ev_free;
    long long launches;
    long long t_launch[SLDG_NKINDS]; double t_ms[SLDG_NKINDS];
    long long a_launch[SLDG_MAX_DIM]; double a_ms[SLDG_MAX_DIM];

    // CUDA graph of one Strang step (small problems)
    cudaStream_t cap_stream;        // capture stream of the context (used when the caller's stream is a default stream)
    cudaGraphExec_t graph_exec; const double* graph_f; double graph_dt; long long graph_launches;
    int opt_graph;                  // 0 = never, 1 = problems up to 256 MB (default), 2 = always

    // tuning
    int opt_tile_bytes;             // axis-0 kernels: bytes per chunk (per warp) / per tile (block-wide kernel)
    int opt_tile_stages;            // axis-0 line kernel: input ring depth per warp (1..4)
    int opt_axis0_impl;             // 0 = auto, 1 = per-warp pipelines, 2 = block-wide tiles, 3 = register walk
    int opt_walk_block;             // slow-axis kernel block size
    int opt_walk_vec;               // 0 = auto, 1, 2
    int opt_fuse_x;                 // 1: x_1 and x_2 sweeps in one pass when the shape allows
    int opt_fused_threads;          // fused kernel: threads per block (<= 256) = planes per block * D_0
    int opt_inplace_walk;           // 1: slow-axis x sweeps may run in place when their table allows
    int opt_fused_impl;             // 0 = auto (cell kernel, else node kernel), 1 = cell-per-thread TMA kernel, 2 = node-per-thread kernel
    int opt_fuse3;                  // 1: x_1, x_2 and x_3 sweeps in one pass (dim_x = 3, degree <= 1)
    int opt_f3_threads;             // fused3 kernel: threads per block (<= 256) = N_0 * strip cells
    int opt_f3_stages;              // fused3 kernel: input stages (2..4)
    int opt_f3d_threads;            // double x_1x_2x_3 pass: compute threads per block (<= 256) = N_0 * (strip cells + 1)
    int opt_x_copy;                 // 1: sldg_advect_x runs the plan that ends in the workspace, then copies back (tests)
    int opt_cell_threads;           // fused cell kernel: threads per block (<= 128) = planes per block * N_0
    int opt_cell_rows;              // fused cell kernel: x_2 cells per chunk (0 = from opt_cell_bytes)
    int opt_cell_bytes;             // fused cell kernel: target bytes of one input stage (all planes of the block)
    int opt_cell_stages;            // fused cell kernel: input stages (2..6)
    int opt_x_double;               // 1: sldg_steps merges the x half steps of consecutive Strang steps into one pass (dim_x = 2: degree <= 2; dim_x = 3: degree <= 1)
    int opt_fuse_v;                 // v_1 and v_2 sweeps in one pass (sldg_sweep_fusedv.cu): 0 never, 1 when the shape allows and the walks fill the GPU, 2 whenever the shape allows
    int opt_fv_wx;                  // fused v kernel: x nodes per tile (0 = auto: 128-byte rows if the threads allow)
    int opt_fv_stages;              // fused v kernel: ring depth (0 = from opt_fv_inflight)
    int opt_fv_inflight;            // fused v kernel: bytes in flight per SM to aim for
    int opt_fv_ppb;                 // fused v kernel: planes per block (0 = auto)
    int opt_fv_cps;                 // fused v kernel, degree <= 1: v_2 cells per tensor copy
    int opt_fv_l2;                  // fused v kernel: L2 promotion of the tensor map (0 none, 1 64 B, 2 128 B, 3 256 B)
    int opt_decline;                // test knob, bit mask: the launcher of a fused pass answers cudaErrorNotSupported (1 fused v_1v_2, 2 fused v_1v_2v_3, 4 fused x_1x_2x_3, 8 fused x_1x_2, 16 double x pass): the planned pass then falls back to separate sweeps
    int opt_fuse_v3;                // v_1, v_2 and v_3 sweeps in one pass (sldg_sweep_fusedv3.cu; dim_x = 3, degree <= 1): 0 never, 1 auto, 2 whenever the shape allows
    int opt_fv3_wx;                 // fused v_1v_2v_3 kernel: x nodes per tile (0 = auto)
    int opt_fv3_strip;              // fused v_1v_2v_3 kernel: v_2 donor pairs per strip (0 = auto: 4)
    int opt_fv3_pw;                 // fused v_1v_2v_3 kernel: 1 = dedicated producer warp (an extra warp per block)
    int opt_fv3_slots;              // fused v_1v_2v_3 kernel: ring slots (0 = as many as shared memory holds)
    int opt_poisson_small;          // 1: x grids of up to 1024 nodes are solved by one single-block launch (FFT route)
    int opt_rho_tma;                // 1: large problems read f through TMA tensor copies (rho_tma_kernel), 0: plain loads only
    int opt_rho_vec;                // 0 = auto (2 when aligned), 1
    int opt_rho_blocks;             // rho kernel: 128-thread blocks per SM to aim for
};

// ---- host tables (sldg_tables.cpp)
void sldg_gl_rule(int n, double* xi, double* w);
void sldg_build_poly(int k, const double* xi, const double* w, ABPoly* out, ABPolyLD* outld);
void sldg_eval_AB_host(const ABPolyLD* p, int k, double alpha, double* A, double* B);
// forward: G = F (I (x) P), inverse: H = (I (x) P^-1) F^-1 / D ; transposed storage [n][m], re block then im block
void sldg_build_dft(int k, const double* xi, int ncell, double* fwdT, double* invT);

// ---- kernel launchers (each returns cudaError_t of the launch)
// walk / line / fused-cell kernels exist in both precisions (sldg_real.h): _f64 and _f32 launchers; fin/fout are
// arrays of that type.  The un-suffixed names (sldg_api.cu) dispatch on ctx->prec.
#define SLDG_DECL_SWEEPS(sfx)                                                                                       \
    cudaError_t sldg_launch_sweep_walk##sfx(sldg_ctx* c, const void* fin, void* fout, const SweepGeom& g,           \
                                            const ShiftTable& t);                                                   \
    cudaError_t sldg_launch_sweep_line##sfx(sldg_ctx* c, const void* fin, void* fout, const SweepGeom& g,           \
                                            const ShiftTable& t);                                                   \
    cudaError_t sldg_launch_sweep_fused_cell##sfx(sldg_ctx* c, const void* fin, void* fout, const SweepGeom& g0,    \
                                                  const SweepGeom& g1, const ShiftTable& t0, const ShiftTable& t1, int any_copy); \
    cudaError_t sldg_launch_sweep_fused_cell2##sfx(sldg_ctx* c, const void* fin, void* fout, const SweepGeom& g0,   \
                                                   const SweepGeom& g1, const ShiftTable& t0, const ShiftTable& t1, int any_copy);
cudaError_t sldg_launch_sweep_fused3_f64(sldg_ctx* c, const void* fin, void* fout, const SweepGeom* g, const ShiftTable* t, int any_copy);
cudaError_t sldg_launch_sweep_fused3_f32(sldg_ctx* c, const void* fin, void* fout, const SweepGeom* g, const ShiftTable* t, int any_copy);
bool sldg_fusedv_shape_f64(const sldg_ctx* c, int* wx_out, int* threads_out);
bool sldg_fusedv_shape_f32(const sldg_ctx* c, int* wx_out, int* threads_out);
cudaError_t sldg_launch_sweep_fusedv_f64(sldg_ctx* c, const void* fin, void* fout, const ShiftTable& t1, const ShiftTable& t2);
cudaError_t sldg_launch_sweep_fusedv_f32(sldg_ctx* c, const void* fin, void* fout, const ShiftTable& t1, const ShiftTable& t2);
bool sldg_fused3d_shape_f64(const sldg_ctx* c);
bool sldg_fused3d_shape_f32(const sldg_ctx* c);
cudaError_t sldg_launch_sweep_fused3d_f64(sldg_ctx* c, const void* fin, void* fout, const SweepGeom* g, const ShiftTable* t, int any_copy);
cudaError_t sldg_launch_sweep_fused3d_f32(sldg_ctx* c, const void* fin, void* fout, const SweepGeom* g, const ShiftTable* t, int any_copy);
bool sldg_fusedv3_shape_f64(const sldg_ctx* c);
bool sldg_fusedv3_shape_f32(const sldg_ctx* c);
cudaError_t sldg_launch_sweep_fusedv3_f64(sldg_ctx* c, const void* fin, void* fout, const ShiftTable& t1, const ShiftTable& t2, const ShiftTable& t3);
cudaError_t sldg_launch_sweep_fusedv3_f32(sldg_ctx* c, const void* fin, void* fout, const ShiftTable& t1, const ShiftTable& t2, const ShiftTable& t3);
SLDG_DECL_SWEEPS(_f64)
SLDG_DECL_SWEEPS(_f32)
cudaError_t sldg_launch_sweep_walk(sldg_ctx* c, const double* fin, double* fout, const SweepGeom& g,
                                   const ShiftTable& t);
cudaError_t sldg_launch_sweep_line(sldg_ctx* c, const double* fin, double* fout, const SweepGeom& g,
                                   const ShiftTable& t);
cudaError_t sldg_launch_sweep_tma(sldg_ctx* c, const double* fin, double* fout, const SweepGeom& g,
                                  const ShiftTable& t);
cudaError_t sldg_launch_sweep_fused(sldg_ctx* c, const double* fin, double* fout, const SweepGeom& g0,
                                    const SweepGeom& g1, const ShiftTable& t0, const ShiftTable& t1);
cudaError_t sldg_launch_sweep_fused_cell(sldg_ctx* c, const double* fin, double* fout, const SweepGeom& g0,
                                         const SweepGeom& g1, const ShiftTable& t0, const ShiftTable& t1, int any_copy);
cudaError_t sldg_upload_poly(sldg_ctx* c);         // device copy of c->poly, owned by the context (c->dPoly)
cudaError_t sldg_launch_vtable(sldg_ctx* c, const double* Ed, double tau, double hv, int N, int* S, double* AB);
cudaError_t sldg_launch_wv(sldg_ctx* c);
cudaError_t sldg_launch_density(sldg_ctx* c, const double* f, double* rho);
cudaError_t sldg_launch_poisson(sldg_ctx* c, const double* rho, double* E);
cudaError_t sldg_launch_poisson_cg(sldg_ctx* c, const double* rho, double* E, double tol, int maxiter, double sigma);
double sldg_sipg_sigma_default(int k);
void sldg_sipg_tables(int k, const double* xi, const double* w, double sigma, double* M, double* B, double* Dm);
cudaError_t sldg_launch_energy(sldg_ctx* c, const double* E, double* out1);
cudaError_t sldg_launch_mass(sldg_ctx* c, const double* f, double* out1);

void sldg_graph_drop(sldg_ctx* c);          // forget the captured Strang-step graph (any state change)
// instrumentation helpers (sldg_api.cu)
void sldg_ev_begin(sldg_ctx* c, int kind, int axis);
void sldg_ev_end(sldg_ctx* c);
