/*
 * sldg.h -- C-ABI of the B200-native (sm_100a) hot path of the split-step semi-Lagrangian
 * discontinuous Galerkin (SLDG) Vlasov-Poisson solver of Einkemmer & Moriggl,
 * arXiv 2110.14557.  Citations "P:line" are lines of the paper text;
 * "reading X" refers to the table of readings in DESIGN.md section 3.
 *
 * Problem (eq. (1),(2)):  d_t f + v.grad_x f - E.grad_v f = 0,  E = -grad phi,
 * -Laplace phi = 1 - rho,  rho = int f dv,  on a periodic box in d_x + d_v dimensions.
 *
 * Discretisation: per axis, N_a cells of k+1 Gauss-Legendre nodes; f holds the
 * VALUES of the piecewise polynomial at the tensor-product nodes.
 *
 * LAYOUT OF f (reading E).  One flat fp64 array of |f| = prod_a D_a values, D_a = N_a (k+1):
 *     flat index  n = n_0 + D_0 (n_1 + D_1 (n_2 + ...)),   axes ordered x_1..x_dx, v_1..v_dv
 *     (x_1 fastest);  per-axis node index n_a = i_a (k+1) + j_a (cell i_a, node j_a);
 *     value stored = f at coordinate lo_a + (i_a + xi_{j_a}) h_a,  h_a = (hi_a - lo_a)/N_a.
 * rho is [X] with X = prod_{a<dx} D_a (same order); E is [dx][X], component-major.
 *
 * POINTERS are DEVICE pointers unless the argument is marked "host".  f, rho, E and the
 * workspace are owned by the caller, must be 16-byte aligned (256 recommended) and must not
 * alias each other.  The library never allocates O(|f|) memory itself.
 *
 * STREAM / SYNC.  All device work is enqueued on the stream given to sldg_set_stream (default:
 * the legacy default stream).  No call synchronises, except those marked "synchronises".  One conditional case:
 * the x-sweep shift tables are built on the host per time increment and cached (two increments per axis, least
 * recently used evicted: a Strang run with its dt/2 plus one more increment never rebuilds).  A call that needs
 * a table that is not cached -- sldg_advect_x, sldg_step, sldg_steps, sldg_step_host with a new dt -- rebuilds
 * it, which SYNCHRONISES the stream once (the pinned staging buffer is reused) and therefore must not happen
 * inside a caller's stream capture; sldg_advect_axis (test hook) always uploads its table and synchronises.
 * Non-finite dt or shift-table entries are rejected with SLDG_EINVAL before anything is enqueued.
 *
 * ERRORS.  Every int-returning call returns SLDG_OK (0) or a negative code; nothing throws,
 * aborts or prints.  A context is not thread-safe.  There is NO CPU fallback: without a CUDA
 * device every compute call returns SLDG_ECUDA.
 */
#ifndef SLDG_H
#define SLDG_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define SLDG_OK 0
#define SLDG_EINVAL (-1)        /* bad argument (NULL, dimension, degree, alignment, ...) */
#define SLDG_ENOMEM (-2)        /* host or small device allocation failed                  */
#define SLDG_ECUDA (-3)         /* a CUDA runtime call failed; see sldg_last_cuda_error    */
#define SLDG_ENOWORKSPACE (-4)  /* sldg_set_workspace not called or too small              */
#define SLDG_ETOOLARGE (-5)     /* sldg_density_static: x grid larger than its fixed scratch */

#define SLDG_MAX_DIM 6
#define SLDG_MAX_DEGREE 4

typedef struct sldg_ctx sldg_ctx;

/* ABI version.  Bumped whenever the signature of an existing symbol changes (round 2 inserted `fuse_v3` in the middle of
 * sldg_plan_query's argument list: a caller built against the older header passes x_double in its place without any
 * diagnostic).  From version 3 on, new parameters are only ever appended or the symbol gets a new name; a C caller should
 * compare sldg_abi_version() with the SLDG_ABI_VERSION it was compiled against before its first call. */
#define SLDG_ABI_VERSION 3
int sldg_abi_version(void);

/* ---- lifetime --------------------------------------------------------------------------
 * sldg_create: problem statement of P:50-58.  dim_x in 1..3, dim_x <= dim_v <= 3 (the paper
 * uses 2x2v, 2x3v, 3x3v; 1x1v and 1x2v are accepted as cheap test vehicles).
 *   cells  (host) [dim_x+dim_v]   cells per axis, x axes first, each >= 1
 *   degree k in 0..SLDG_MAX_DEGREE, the same on every axis (order k+1)
 *   domain (host) [2(dim_x+dim_v)] lo_a, hi_a per axis, hi_a > lo_a; every axis is periodic
 *                                  (reading C)
 * Builds host tables (GL nodes/weights, polynomial coefficients of A(alpha), B(alpha)) and
 * small device tables (O(sum_a D_a) bytes).  *out is written only on success. */
int sldg_create(sldg_ctx** out, int dim_x, int dim_v, const int* cells, int degree,
                const double* domain);
int sldg_destroy(sldg_ctx* ctx);

/* ---- single precision mode (NEXT row; Tables 3-4) ---------------------------------
 * "Running simulations with the semi-Lagrangian discontinuous Galerkin scheme in single precision is
 * a viable option. This reduces memory consumption by a factor of two".  Reading W: in an
 * SLDG_F32 context f is STORED as float and the sweep arithmetic of eq. (3) runs in fp32 (A, B
 * evaluated in fp64, rounded to fp32); the shift delta, s = floor(delta), alpha, rho (fp64 sum of the
 * fp32 values), the field solve and E stay fp64, so integer decisions are those of the fp64 path.
 * sldg_create == sldg_create_prec(..., SLDG_F64).  In an SLDG_F32 context every `f` / `f_host` /
 * `f_dev` argument of the calls below points to |f| FLOAT values (pass the float pointer cast to
 * double*); rho, E and delta tables stay double.  The workspace holds a float second buffer. */
#define SLDG_F64 0
#define SLDG_F32 1
int sldg_create_prec(sldg_ctx** out, int dim_x, int dim_v, const int* cells, int degree,
                     const double* domain, int precision);
int sldg_precision(const sldg_ctx* ctx);                          /* SLDG_F64 / SLDG_F32 */

/* stream = a cudaStream_t passed as void*; NULL selects the legacy default stream. */
int sldg_set_stream(sldg_ctx* ctx, void* stream);

/* Workspace: the second f buffer (|f| values), per-x-node shift tables, rho/E and DFT scratch.
 * Caller-owned device memory, >= sldg_workspace_bytes(ctx) bytes, 256-byte aligned. */
size_t sldg_workspace_bytes(const sldg_ctx* ctx);
int sldg_set_workspace(sldg_ctx* ctx, void* dev, size_t bytes);

/* ---- the hot path ------------------------------------ */

/* a1+a2, steps 1a-1c: for d = 1..dim_x, in that order, f(x_d - v_d dt) by the 1-D
 * SLDG update, eq. (3)
 *     u_i <- A(alpha) u_{(i-s) mod N} + B(alpha) u_{(i-s-1) mod N},
 *     delta = (v_d * dt) / h_{x_d},  s = floor(delta),  alpha = delta - s   (reading B)
 * on every line along x_d; v_d is the coordinate of the line's v_d node.  `dt` is the actual
 * time increment (a Strang half step passes Delta t / 2; reading J).  Result in f. */
int sldg_advect_x(sldg_ctx* ctx, double* f, double dt);

/* a5+a6, steps 3a-3c: for d = 1..dim_x, f(x, v_d + E_d(x) dt), i.e. the same update
 * along v_d with delta = ((-E_d(x)) * dt) / h_{v_d} per x node (sign from eq. (1), reading H).
 * Velocity axes beyond dim_x are not advected (reading D).  E is [dim_x][X].  Result in f.
 * E is the same for all sweeps, so the v_1 and v_2 sweeps (option fuse_v), or for dim_x = 3 all three
 * (option fuse_v3), may run as one pass over f: same arithmetic in the same order, bit-identical to separate sweeps. */
int sldg_advect_v(sldg_ctx* ctx, double* f, const double* E, double dt);

/* a3: rho[x] = sum_v (prod_d h_{v_d} w_{j_d}) f[x,v]. */
int sldg_density(sldg_ctx* ctx, const double* f, double* rho);

/* a4 (reading P1): -Laplace phi = 1 - rho periodic, E = -grad phi at the x
 * nodes, by interpolation to the equidistant grid, a spectral solve, and interpolation back. */
int sldg_poisson(sldg_ctx* ctx, const double* rho, double* E);

/* a7, Strang splitting: advect_x(dt/2); density; poisson; advect_v(dt);
 * advect_x(dt/2).  rho and E of the step stay in the workspace (sldg_last_rho / sldg_last_E). */
int sldg_step(sldg_ctx* ctx, double* f, double dt);
/* a7 out of place: the same Strang step with the result in f_out.  f_in (|f| values, the state at t_n) is used as
 * scratch and holds no meaningful data afterwards; f_out must not alias f_in or the workspace.  Why: sldg_step has to end in
 * the buffer it was given, which forces an even number of buffer flips -- for dim_x = 3 the v advection then runs as two
 * passes instead of one, for dim_x = 2 the fused v pass is not used.  A caller who needs f(t_n) after EVERY step (per-step
 * diagnostics) and owns two buffers anyway ping-pongs between them with this call and gets the pass budget of sldg_steps
 * (3 passes + rho for dim_x = 3).  Same 1-D sweeps in the same order as sldg_step: bit-identical result.
 * end_of_step_field = 1 additionally evaluates rho and E of f(t_{n+1}) (the paper's second density/field evaluation per
 * step, "This is done twice"): sldg_last_rho / sldg_last_E then belong to t_{n+1} instead of the half step.
 * Always enqueues plain launches (no graph replay).  sldg_workspace_field returns the |f|-value buffer inside the workspace
 * (NULL before sldg_set_workspace): it may serve as f_out / f_in of this call, so that f and the workspace ping-pong without
 * a third buffer; every other sweep or step call overwrites it. */
int sldg_step_to(sldg_ctx* ctx, double* f_in, double* f_out, double dt, int end_of_step_field);
double* sldg_workspace_field(const sldg_ctx* ctx);
/* Small problems (|f| <= 256 MB; option graph) replay a CUDA graph of the step, captured at the first call with a
 * given (f, dt).  1 if such a graph is instantiated right now (the next sldg_step with the same f, dt replays it). */
int sldg_graph_active(const sldg_ctx* ctx);

/* ---- CGdG Poisson solver (NEXT row, Appendix) --------------------------------
 * Alternative to sldg_poisson: symmetric interior penalty (SIPG) dG discretisation of
 * -Laplace phi = 1 - rho in the advection's own polynomial space (eq. (4); block-tridiagonal
 * matrix from the small matrices M, B; tensor form P:541-545; readings I, T), solved
 * matrix-free by the mean-preserving conjugate gradient method of Algorithm 1 starting
 * from the potential of the previous solve, then E = -grad phi cell-wise at the nodes
 * (reading U).  Stops when ||r||_2 < tol ||b||_2 (the paper uses tol 1e-3) or after maxiter
 * iterations (0 = the paper's bound (prod_l N_l (k+1))^(1/dim_x) times a safety factor).
 * One cooperative launch, no host synchronisation.  degree >= 1 (SLDG_EINVAL for degree 0).
 * rho [X], E [dim_x][X] device. */
int sldg_poisson_cg(sldg_ctx* ctx, const double* rho, double* E, double tol, int maxiter);
/* Which solver sldg_step uses: 0 = sldg_poisson (default), 1 = sldg_poisson_cg with these
 * parameters; sigma <= 0 selects the default penalty (k^2, 2 for k = 1; reading T). */
int sldg_set_poisson_solver(sldg_ctx* ctx, int solver, double tol, int maxiter, double sigma);
/* Zero the stored potential (cold start of the next CG solve). */
int sldg_cg_reset(sldg_ctx* ctx);
/* Iterations and relative residual ||r||_2/||b||_2 of the last CG solve (host outputs, may be NULL).
 * Synchronises. */
int sldg_cg_info(sldg_ctx* ctx, int* iters_host, double* relres_host);
/* device pointer [X] to the potential of the last CG solve (mean 0), valid until the workspace changes */
const double* sldg_last_phi(const sldg_ctx* ctx);
/* M, B of the SIPG matrix as the library builds them, row-major (k+1)x(k+1), (A_hat u)_i = M u_i +
 * B u_{i-1} + B^T u_{i+1}; sigma <= 0: default.  Host-only, needs no context or device. */
int sldg_sipg_matrices(int degree, double sigma, double* hostM, double* hostB);

/* nsteps Strang steps; the result is in f and equals nsteps calls of sldg_step bit for bit (the same 1-D
 * sweeps in the same order).  What changes is the number of passes over f: consecutive steps may keep their
 * intermediate result in the workspace buffer, and for dim_x = 2 the second x half step of a step and the
 * first x half step of the next one (same time increment, nothing in between) run as ONE pass
 * (option x_double; for dim_x = 3 only when forced with x_double = 2: that pass is slower than two on B200).  f at the intermediate integer times is then not written out: call sldg_step when a
 * per-step diagnostic needs it.  sldg_plan_query reports the pass budget of either call. */
int sldg_steps(sldg_ctx* ctx, double* f, double dt, int nsteps);

/* Same path driven from HOST memory: copies f_host (|f| doubles, pinned memory recommended) to
 * the device buffer f_dev, runs nsteps Strang steps, copies the result back into f_host and the
 * last E ([dim_x][X]) into E_host if it is not NULL.  Synchronises. */
int sldg_step_host(sldg_ctx* ctx, double* f_host, double* f_dev, double* E_host, double dt,
                   int nsteps);

/* ---- helpers ---------------------------------------------------------------------------- */
long long sldg_field_elems(const sldg_ctx* ctx);                 /* |f|                     */
long long sldg_rho_elems(const sldg_ctx* ctx);                   /* X                       */
int sldg_nodes(const sldg_ctx* ctx, int axis);                   /* D_axis, or SLDG_EINVAL  */
/* host_out (host) [D_axis]: coordinates lo + (i + xi_j) h of the nodes of `axis`. */
int sldg_node_coords(const sldg_ctx* ctx, int axis, double* host_out);
/* device pointers into the workspace, valid after sldg_step / until the workspace changes */
const double* sldg_last_rho(const sldg_ctx* ctx);
const double* sldg_last_E(const sldg_ctx* ctx);
/* 1/2 sum_x W_x |E(x)|^2 and sum_n W_n f_n; host_out is one host double.  Synchronise. */
int sldg_electric_energy(sldg_ctx* ctx, const double* E, double* host_out);
int sldg_mass(sldg_ctx* ctx, const double* f, double* host_out);
const char* sldg_strerror(int code);
int sldg_last_cuda_error(const sldg_ctx* ctx);                   /* cudaError_t as int      */

/* A(alpha), B(alpha) of eq. (3) (reading A) as the library evaluates them, row-major
 * (k+1)x(k+1), 0 <= alpha <= 1, degree in 0..SLDG_MAX_DEGREE.  Host-only, needs no context or device.
 *   device_arith = 0: the host route of the x-sweep tables (Horner in long double, rounded to fp64);
 *   device_arith = 1: the exact arithmetic of the device-side v-sweep table kernel (fp64 Horner with
 *                     fused multiply-add on the fp64 coefficients), reproduced on the host. */
int sldg_AB(int degree, double alpha, int device_arith, double* hostA, double* hostB);
/* (degree+1)-point Gauss-Legendre nodes and weights on [0,1] as the library uses them. Host-only. */
int sldg_gauss_legendre(int degree, double* host_xi, double* host_w);

/* Test hook: one sweep along `axis` with a caller-given shift table (in cells), through the
 * production kernels.  delta_host (host): for an x axis, D_{v axis dim_x+axis} entries indexed
 * by that axis' node; for a v axis, X entries indexed by flat x node.  Result in f. */
int sldg_advect_axis(sldg_ctx* ctx, double* f, int axis, const double* delta_host);

/* ---- instrumentation --------------------------------------------------------------------
 * With timing on, every kernel launch is bracketed by CUDA events on the context's stream.
 * Kinds: 0 = sweep along axis 0 (TMA/SMEM kernel), 1 = sweep along a slow axis, 2 = rho,
 * 3 = Poisson/E, 4 = shift tables (device-side v-table kernel), 5 = whole-array device copies of f (|f| read + |f| written
 * each; only fallback plans make any), 6 = fused x pass (x_1+x_2, or x_1+x_2+x_3 for dim_x = 3, in one
 * launch), 7 = fused v_1+v_2 pass (one launch), 8 = double x half step (x_1+x_2 applied twice in one launch, inside
 * sldg_steps), 9 = fused v_1+v_2+v_3 pass (one launch, dim_x = 3), 10 = double x half step for dim_x = 3
 * (x_1+x_2+x_3 applied twice in one launch, inside sldg_steps), 11 = host-to-device uploads of rebuilt x-sweep shift tables
 * (O(D) bytes; until ABI version 2 these were booked under kind 5); the per-axis figures of sldg_timing_axis book an equal share of a
 * fused launch's time on each of its axes.  sldg_timing_read synchronises, adds the elapsed
 * times of all events recorded since the last read, and returns per kind the number of launches
 * and the total milliseconds (arrays of SLDG_NKINDS entries, host). */
#define SLDG_NKINDS 12
int sldg_timing_enable(sldg_ctx* ctx, int on);
/* SLDG_ECUDA (and no figures) if an event could not be created since the last read: launches went unrecorded. */
int sldg_timing_read(sldg_ctx* ctx, long long* launches, double* ms);
/* total kernel launches enqueued by this context since creation */
long long sldg_launch_count(const sldg_ctx* ctx);
/* Per-axis sweep time (ms) and launches accumulated since the last sldg_timing_read; arrays of
 * SLDG_MAX_DIM entries (host).  Filled by sldg_timing_read; this call does not synchronise. */
int sldg_timing_axis(const sldg_ctx* ctx, long long* launches, double* ms);

/* Host-only (no CUDA device needed): the plan of one sldg_step (nsteps == 0) or of sldg_steps(nsteps) for a problem
 * of this shape, obtained by running the library's planning code with every launch replaced by a counter.
 * shifts_below_one: 1 = every x shift is 0 or -1 cell (|v| dt/2 < h_x: slow-axis x sweeps may then run in place),
 * fuse_v / fuse_v3 / x_double: the options of the same names (sldg_set_option).  counts (host, 6 entries) = passes over f of
 * the x sweeps, passes of the v sweeps, rho passes, field solves, whole-array device copies, kernel launches counted
 * by sldg_launch_count.  A fused or merged launch is ONE pass.  Returns 0 or a negative code. */
int sldg_plan_query(int dim_x, int dim_v, const int* cells, int degree, int precision, int nsteps,
                    int shifts_below_one, int fuse_v, int fuse_v3, int x_double, long long* counts);

/* Host-only: the plan of one sldg_step_to call (same arguments and counts as sldg_plan_query; end_of_step_field as in the call). */
int sldg_plan_query_step_to(int dim_x, int dim_v, const int* cells, int degree, int precision, int end_of_step_field,
                            int shifts_below_one, int fuse_v, int fuse_v3, int x_double, long long* counts);

/* ---- rho for callers that cannot allocate device memory -----------------------------------
 * Same operation as sldg_density (a3): rho[x] = sum_v Wv[v] f[v][x], f seen as a row-major [V][X]
 * array (x contiguous: exactly the layout above with X = prod of the x extents, V = prod of the v extents).
 *
 * Why it exists.  sldg_density needs a context (sldg_create calls cudaMalloc for its small tables) and a workspace
 * for the partial sums of its two-stage reduction.  Not every caller can provide those where rho is needed: a host
 * application that has already given all of HBM to its own memory pool (a new cudaMalloc fails, or makes the pool
 * shrink); a loop that shares the GPU with other streams and cannot afford the device-wide synchronisation that
 * cudaMalloc/cudaFree imply; a plug-in that receives pointers and a stream from its host and is not allowed to own
 * device memory.  This call needs NO context and NO workspace and never calls cudaMalloc, cudaFree or any allocating
 * routine: its partial sums live in a fixed 8 MiB array inside the library image.  That array occupies 8 MiB on every
 * GPU onto which the library's device code is loaded, until the process exits.
 *
 *   f          device, [V][X] values, double (precision SLDG_F64) or float (SLDG_F32); 16-byte alignment (8 for
 *              float) and even X select the 2-wide loads, anything else still works
 *   Wv         device, [V] doubles: the velocity quadrature weight of row v, prod_d h_{v_d} w_{j_d} with v_1 fastest
 *              (w from sldg_gauss_legendre; the caller builds and uploads it once, at a time when it may allocate)
 *   rho        device, [X] doubles, written completely; must not alias f or Wv
 *   stream     a cudaStream_t as void*, NULL = legacy default stream; the call enqueues two kernels and returns
 *   cuda_error_host  host, may be NULL: receives the cudaError_t when SLDG_ECUDA is returned, 0 otherwise
 * All pointers must belong to the device that is current in the calling thread.
 *
 * LIMIT.  X <= SLDG_DENSITY_STATIC_MAX_X (= sldg_density_static_max_x(), 1 048 576 x nodes; the largest BASELINE config
 * has 110 592).  A larger X returns SLDG_ETOOLARGE before anything is enqueued; V is not limited by the scratch.
 * Other errors: SLDG_EINVAL (NULL pointer, X or V < 1, unknown precision), SLDG_ECUDA.
 *
 * FIRST CALL PER DEVICE.  The first call on each device looks up the device address of the fixed array
 * (cudaGetSymbolAddress) and the SM count, under a lock, and keeps them.  Make that first call during start-up,
 * before any stream capture begins on that device; later calls only launch.
 *
 * SHARED STATE.  Every call in the process on the same device uses the same array.  Calls enqueued on one stream run
 * one after the other and are safe.  Two calls that can overlap on the GPU (different streams without an event
 * between them, or two host threads on different streams) overwrite each other's partial sums: ordering them is the
 * caller's job.  The array keeps whatever the last call left in it; that is harmless, because stage one rewrites every
 * partial sum that stage two reads, so nothing has to start at zero.  Results are bitwise reproducible from call to
 * call on the same device; they agree with sldg_density to rounding (the chunking of the v sum differs). */
#define SLDG_DENSITY_STATIC_MAX_X (1 << 20)
int sldg_density_static(const void* f, const double* Wv, long long X, long long V, int precision, double* rho,
                        void* stream, int* cuda_error_host);
long long sldg_density_static_max_x(void);

/* Tuning knob (affects speed only, never results): see DESIGN.md section 5.  A fused pass whose launcher declines
 * a shape that the planner accepted is replaced by the separate sweeps (plus one device copy when the buffer
 * parity differs): same bits, never an error. */
int sldg_set_option(sldg_ctx* ctx, const char* name, long long value);

#ifdef __cplusplus
}
#endif
#endif /* SLDG_H */
