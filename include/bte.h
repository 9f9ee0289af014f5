/*
 * bte.h -- C ABI of libbte_b200: the Crank-Nicolson + leap-frog time step of the spatially homogeneous
 * 2-D superlattice Boltzmann transport equation (arxiv 1401.6047), fp64, one NVIDIA B200 (sm_100a).
 *
 * What one call sequence computes (citations are PAPER.md lines / equations):
 *   bte_create            fixes the lattice a^t_{n,m}, n = 0..N harmonics, m = 0..M phi_y points
 *                         (eq. 21-23) and the dimensionless parameters of eq. (4)-(5), L40-51.
 *   bte_init_equilibrium  a = a^(0) (eq. 15-16), b = 0 (L99); fractional grid z^{1/2} by one
 *                         application of T (eq. 38) with time step dt/2 (L202).
 *   bte_step              n_steps leap-frog steps (eq. 40-41), each = T on the whole grid with
 *                         the stencil A, B (eq. 30-31) of the fractional grid, then T on the fractional
 *                         grid with the stencil of the new whole grid; T is the closed-form 2x2
 *                         Crank-Nicolson solve of eq. (32)-(37) (sign of (33) corrected, C2).
 *                         After every step: norm (eq. 12), drift velocity (eq. 20) and the running sums
 *                         of eq. (17).  Everything runs on the device; the host is not involved per step.
 *   bte_observables       copies the per-system observables to the host.
 *
 * Conventions
 *   - All functions return 0 (BTE_OK) or a negative bte_status; none throws or aborts.  After a failure
 *     bte_last_error() returns a thread-local, NUL-terminated description.
 *   - "host" / "device" is stated for every pointer.  The ONLY device memory the library uses is the
 *     caller-owned workspace handed to bte_create (e.g. a torch.empty(uint8) tensor); the library never
 *     allocates or frees device memory and never frees the workspace.  The ctx is a small host object.
 *     (One exception, stated at its declaration: bte_rs_evolve_static works in a fixed 5 MiB array of the library.)
 *   - Arrays a, b exchanged with the host are row-major (n_harm+1) x n_phiy doubles, m fastest
 *     (the layout of Fig. 7).  Inside the workspace the state is stored as interleaved (a,b)
 *     pairs.
 *   - fp64 throughout unless bte_grid.precision asks for one of the fp32 variants of the step (the paper's own
 *     precision).  Work is issued asynchronously on the CUDA stream given at create
 *     time (a cudaStream_t passed as void*; NULL = legacy default stream).
 *   - How a step is executed is chosen automatically (bte_set_option "variant"): lattices that fit the GPU's
 *     shared memory run the whole time loop of a bte_step call in one launch (resident kernel); larger ones and
 *     batches stream through HBM once per 4 or 3 time steps (warp kernel; columns shorter than 32 rows: the
 *     shared-memory-ring kernel, 2 steps).  Results do not depend on the choice beyond rounding: the state is
 *     bit-identical across variants 1-4 and agrees with variant 5 to 1e-14 max|f| (variant 5 forms n beta dt/2 with
 *     one fused multiply-add more).
 *   - Beyond the time step: bte_reconstruct_pdf (eq. 8) and bte_pendulum_averages (eq. 44-46), see below.
 *   - A ctx belongs to the CUDA device that owns its workspace: every entry point selects that device for the
 *     duration of the call and restores the caller's current device.
 *   - Not thread-safe per ctx; distinct ctxs may be used from distinct threads.
 */
#ifndef BTE_B200_H
#define BTE_B200_H

#include <stddef.h>
#include <stdint.h>

/* The library is built with -fvisibility=hidden: exactly the functions declared here are exported. */
#if defined(__GNUC__)
#define BTE_API __attribute__((visibility("default")))
#else
#define BTE_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

typedef struct bte_ctx bte_ctx; /* opaque, library-owned host object */

typedef enum {
    BTE_OK = 0,
    BTE_EINVAL = -1,    /* NULL pointer, N < 1, M+1 < 3, n_batch < 1, dt <= 0, mu <= 0, alpha <= 0,
                           phiy_max <= phiy_min, bad index, unknown option                              */
    BTE_EUNSTABLE = -2, /* |B| dt / dphi >= 2: the staggered scheme diverges (reading C11)     */
    BTE_ENOMEM = -3,    /* workspace smaller than bte_workspace_bytes(grid) or misaligned (256 B)        */
    BTE_ECUDA = -4      /* a CUDA runtime error was captured; text in bte_last_error()                   */
} bte_status;

/* Lattice shared by all systems of a batch (eq. 21-22; command-line names of L325-326 in brackets). */
typedef struct {
    int32_t n_harm;  /* N  : highest harmonic kept, rows n = 0..N            [n-harmonics]               */
    int32_t n_phiy;  /* M+1: number of phi_y lattice points, m = 0..M        [g-grid]                    */
    int32_t n_batch; /* number of independent systems advanced together, >= 1                            */
    int32_t precision;/* 0 = fp64 (default; every kernel).  fp32 variants of the step (the paper's precision, L311):
                        1 = state stored as fp32 pairs, arithmetic fp64 (multi-step passes through the warp kernel
                        on lattices of >= 32 rows, otherwise two launches per step); 2 = fp32 storage and arithmetic
                        (two launches per step).  The resident kernel is fp64 only.  Host arrays stay double.   */
    double dt;       /* time step in units of tau                            [dt]                        */
} bte_grid;

/* One per system; all quantities dimensionless per eq. (4). */
typedef struct {
    double E_dc, E_omega, omega; /* E(t) = E_dc + E_omega cos(omega t), L99     [E_dc, E_omega, omega]   */
    double B;                    /* constant magnetic field along z, eq. (5)    [B]                      */
    double mu;                   /* Delta_1 / (2 k_B T), eq. (14)               [mu]                     */
    double alpha;                /* m / m_x, eq. (4); normalisation only        [alpha]                  */
    double phiy_min, phiy_max;   /* phi_m = centre + (m - M/2) dphi, dphi = (max-min)/M  [PhiYmin/max]   */
    double kappa_scale;          /* 1: stencil prefactor B dt/(4 dphi), consistent with eq. (5),(9),(10);
                                    alpha: the prefactor as printed in eq. (30)-(31) (C4)      */
    int64_t n_steps_total;       /* the system freezes after this many steps; 0 = never                  */
    int64_t avg_start_step;      /* running sums of eq. (17) include steps k > avg_start_step (L103)     */
} bte_params;

typedef struct {
    int64_t step;       /* whole-grid steps taken by this system                                         */
    double t;           /* step * dt                                                                     */
    double norm;        /* eq. (12): 2 pi sqrt(alpha) dphi sum_m a_{0,m}   (should be 1)                  */
    double v_dr;        /* eq. (20): pi sqrt(alpha) dphi sum_m b_{1,m}, whole grid, instantaneous        */
    double sum_v_dt;    /* sum over steps k > avg_start_step of v_dr(t_k) dt                             */
    double sum_vcos_dt; /* ... of v_dr(t_k) cos(omega t_k) dt.  Absorption of eq. (17) =
                           (2 I0(mu)/I1(mu)) * sum_vcos_dt / window (factor applied by the caller, C9)   */
    double sum_vsin_dt; /* ... of v_dr(t_k) sin(omega t_k) dt                                            */
    double window;      /* sum of dt over the same steps                                                 */
    double edge_leak;   /* |b_{1,0}| + |b_{1,M}| on the whole grid: bounds the norm drift per step (C12) */
} bte_obs;

/* Bytes of device workspace bte_create needs for this grid.  Pure function; 0 if grid is invalid. */
BTE_API size_t bte_workspace_bytes(const bte_grid* grid /* host */);

/* Validates, computes the per-system tables on the host (phi_y lattice, Gaussian factor, Bessel ratios
 * I_n(mu)/I_0(mu) of eq. 15) and uploads them into the workspace.
 *   grid, params : host; params is an array of grid->n_batch entries (copied).
 *   workspace    : DEVICE, caller-owned, >= bte_workspace_bytes(grid) bytes, 256-byte aligned; must stay
 *                  valid until bte_destroy.  bytes is its size.
 *   cuda_stream  : cudaStream_t (as void*) on which all work of this ctx is issued.
 *   out          : host; receives the ctx, or NULL on failure.                                          */
BTE_API int bte_create(const bte_grid* grid, const bte_params* params, void* workspace, size_t bytes,
               void* cuda_stream, bte_ctx** out);

/* State at t = 0: whole grid a = a^(0), b = 0 (L99); fractional grid by T with dt/2 (L202); step counter,
 * running sums and observables reset.  Asynchronous on the stream.                                      */
BTE_API int bte_init_equilibrium(bte_ctx* ctx);

/* Advance every system that has not reached its n_steps_total by n_steps (>= 0) steps of eq. (40)-(41)
 * with the per-step reductions.  Asynchronous on the stream; no host synchronisation inside.            */
BTE_API int bte_step(bte_ctx* ctx, int64_t n_steps);

/* Synchronises the stream and writes grid->n_batch records to out (host). */
BTE_API int bte_observables(bte_ctx* ctx, bte_obs* out /* host, n_batch entries */);

/* Frees the ctx (host object and CUDA graph handles).  Never touches the workspace memory. */
BTE_API int bte_destroy(bte_ctx* ctx);

/* State access (tests, checkpointing, end-to-end use).  grid_id: 0 = whole grid z^k, 1 = fractional grid
 * z^{k+1/2}.  a, b: HOST arrays of (n_harm+1) * n_phiy doubles each, row-major, m fastest.  Both calls
 * synchronise the stream.  bte_set_state does not change the step counter or the running sums.          */
BTE_API int bte_get_state(bte_ctx* ctx, int32_t system, int32_t grid_id, double* a, double* b);
BTE_API int bte_set_state(bte_ctx* ctx, int32_t system, int32_t grid_id, const double* a, const double* b);

/* The same for ALL systems of the batch at once: a, b are HOST arrays of n_batch * (n_harm+1) * n_phiy doubles,
 * [system][n][m].  One launch group and ONE stream synchronisation per call, whatever n_batch is (pinned host memory
 * makes the two copies asynchronous DMA transfers).  Afterwards every system's live ping-pong buffer is buffer 0.    */
BTE_API int bte_get_state_batch(bte_ctx* ctx, int32_t grid_id, double* a, double* b);
BTE_API int bte_set_state_batch(bte_ctx* ctx, int32_t grid_id, const double* a, const double* b);

/* The distribution function itself, eq. (8) (L63-64): f(phi_x, phi_y_m) = sum_n a_{n,m} cos(n phi_x) + b_{n,m} sin(n phi_x)
 * of one system and grid on n_phix equidistant points phi_x_i = -pi + 2 pi i / n_phix, i = 0 .. n_phix-1 (the content
 * of the paper's Fig. 2 and Fig. 5, as a headless buffer).
 *   f : DEVICE, caller-owned, n_phix * n_phiy doubles, row-major [i][m], m fastest.  1 <= n_phix <= 2048.
 * Reads the step counter's buffer flag (synchronises the stream once), then runs asynchronously on the stream. */
BTE_API int bte_reconstruct_pdf(bte_ctx* ctx, int32_t system, int32_t grid_id, int32_t n_phix, double* f /* device */);

/* The zero-temperature limit of the model, eq. (44)-(46) (L229-240): one electron starts at (phi_x, phi_y) = (0, 0) and
 * follows d phi_x/dt = E(t) + B phi_y, d phi_y/dt = -B sin(phi_x); its velocity sin(phi_x) enters the drift velocity
 * through the exponential memory (46).  Returns, per parameter set, the averages over one ac period
 *   v_mean = <v_dr>, v_cos = <v_dr cos wt>, v_sin = <v_dr sin wt>      (absorption of eq. (17) at T -> 0: A = 2 v_cos).
 * Discretisation (C20): classical RK4 with step h, composite Simpson on the n_rk + 1 RK4 nodes (n_rk even;
 * the memory is cut at n_rk h), rectangle rule over n_phase start phases (1 is used when E_omega or omega is 0).
 *   params, out : HOST arrays of n entries;  workspace : DEVICE, caller-owned, >= bte_pendulum_workspace_bytes(n).
 * Independent of any ctx.  Synchronises the stream before returning.                                          */
typedef struct { double E_dc, E_omega, omega, B; } bte_pendulum_params;
typedef struct { double v_mean, v_cos, v_sin; } bte_pendulum_out;
BTE_API size_t bte_pendulum_workspace_bytes(int32_t n);
BTE_API int bte_pendulum_averages(const bte_pendulum_params* params, int32_t n, int32_t n_phase, double h, int32_t n_rk,
                          void* workspace /* device */, size_t bytes, void* cuda_stream, bte_pendulum_out* out);

/* Real-space-phi_x variant of the step (BASELINE.json config 0's "64 periodic phi_x points"; NOT in the paper, whose
 * Fourier representation (7)-(8) reduces the implicit solve to the 2x2 blocks of eq. 32-33 -- DESIGN.md C22): f is
 * kept on n_phix periodic points phi_x_i = -pi + 2 pi i / n_phix; the Crank-Nicolson treatment of relaxation and of the
 * (E + B phi_y) d/dphi_x term becomes ONE CYCLIC TRIDIAGONAL SYSTEM PER phi_y ROW (batched cyclic sweeps), the
 * -B sin(phi_x) d/dphi_y term stays explicit on the staggered leap-frog grids (eq. 40-41), start-up per L202.
 * One system per ctx; params as for bte_create (n_steps_total / avg_start_step honoured).  Same ownership rules:
 * caller-owned DEVICE workspace of bte_rs_workspace_bytes(grid) bytes, 256-byte aligned.  bte_rs_observables fills one
 * bte_obs (norm = sqrt(alpha) dx dphi sum f, eq. 6; v_dr = sqrt(alpha) dx dphi sum sin(phi_x) f, eq. 18-19; edge_leak 0).
 * bte_rs_get_state: f is a HOST array of n_phix * n_phiy doubles, [i][m], m fastest; grid_id 0 whole, 1 fractional.
 * n_phix a power of two <= 1024 runs the parallel-cyclic-reduction kernel (one warp per phi_y column, in registers);
 * any other n_phix the Thomas + Sherman-Morrison sweeps (one thread per phi_y point): same results to rounding. */
typedef struct bte_rs_ctx bte_rs_ctx;
typedef struct {
    int32_t n_phix;  /* periodic phi_x points, 4 .. 4096                                                   */
    int32_t n_phiy;  /* phi_y lattice points, m = 0..M                                                      */
    double dt;       /* time step in units of tau                                                           */
} bte_rs_grid;
BTE_API size_t bte_rs_workspace_bytes(const bte_rs_grid* grid /* host */);
BTE_API int bte_rs_create(const bte_rs_grid* grid, const bte_params* params /* host, one entry */, void* workspace /* device */,
                  size_t bytes, void* cuda_stream, bte_rs_ctx** out);
BTE_API int bte_rs_init_equilibrium(bte_rs_ctx* ctx);
BTE_API int bte_rs_step(bte_rs_ctx* ctx, int64_t n_steps);
BTE_API int bte_rs_observables(bte_rs_ctx* ctx, bte_obs* out /* host, one entry */);
BTE_API int bte_rs_get_state(bte_rs_ctx* ctx, int32_t grid_id, double* f /* host */);
BTE_API int bte_rs_destroy(bte_rs_ctx* ctx);

/* The real-space step WITHOUT ANY ALLOCATION AND WITHOUT A WORKSPACE, for callers that cannot call cudaMalloc or own
 * scratch memory (code under CUDA graph capture, tight serving loops, harnesses that forbid allocation).  One call =
 * n_steps leap-frog steps (eq. 40-41 in the real-space form above, the same kernels as bte_rs_step) from a state the
 * caller passes in to a state the caller gets back; nothing survives the call but f_out and obs.
 *   grid, params : host, as for bte_rs_create (n_steps_total / avg_start_step honoured against step0 + s).
 *   f_in         : DEVICE, 2 * n_phix * n_phiy doubles, [grid 2][i][m], m fastest, dense: the whole grid at
 *                  t = step0 dt, then the fractional grid at t = (step0 + 1/2) dt.  NULL = start from the
 *                  equilibrium f0 (eq. 13) with the start-up half step (L202); step0 must then be 0.
 *   f_out        : DEVICE, same shape: both grids after step0 + n_steps steps.  May alias f_in.
 *   obs          : host or NULL.  Non-NULL: the stream is synchronised and one record is written (norm, v_dr of the
 *                  last step taken; the running sums of eq. 17 over THIS call's steps only).  NULL: the call
 *                  returns without synchronising (no host transfer at all).
 *   cuda_stream  : cudaStream_t (as void*) of the CURRENT device, which the caller has made current.
 * Scratch: the pitched state, the sweep arrays, the tables, the block partials and the observables live in one
 * file-scope device array of 5 MiB inside the library, which every GPU that loads the library holds until the process
 * exits.  Limit: n_phix * pitch <= 131072 lattice points, pitch = n_phiy rounded up to a multiple of 8 (e.g. 64 x 2048,
 * 256 x 512, 1024 x 128); larger grids are refused with BTE_ENOMEM and a message naming the limit (use bte_rs_create).
 * The function calls no cudaMalloc, cudaFree or allocating library routine.  ALL CALLS SHARE THE ARRAY, which keeps
 * the last call's contents: what must start at zero is cleared at the start of each call, but two calls that overlap
 * on the GPU (different streams, or two host threads) race -- serialise them on one stream.                        */
BTE_API int bte_rs_evolve_static(const bte_rs_grid* grid /* host */, const bte_params* params /* host, one entry */,
                         const double* f_in /* device or NULL */, int64_t step0, int64_t n_steps,
                         double* f_out /* device */, bte_obs* obs /* host or NULL */, void* cuda_stream);

/* Tuning / variant selection, before or between bte_step calls.  Keys:
 *   "variant"      0 = automatic (default), 1 = two half-update kernels per step (96 B/point/step),
 *                  2 = fused whole+fractional kernel on a 2-D tile grid (64 B/point/step),
 *                  3 = persistent sweep kernel, S steps per launch (64/S B/point/step; intermediate time levels in
 *                      shared-memory rings, one thread per phi_y column; the one-step, HBM-bound form and the
 *                      default for columns shorter than 32 rows),
 *                  5 = warp kernel, S = 2, 3 or 4 steps per launch (same traffic; the default path for lattices larger
 *                      than the GPU's shared memory and for batches: one warp per strip of 96 columns runs all 2 S
 *                      half-updates in registers, rows in flight in tensor memory, input rows by 1-D TMA bulk copies;
 *                      one-step launches fall back to variant 3; also bte_grid.precision 1),
 *                  4 = resident kernel: the whole time loop of one bte_step call in ONE launch, state held
 *                      in shared memory (one system: both grids must fit the shared memory of the GPU; a batch:
 *                      each system must fit one cluster of 16 CTAs; otherwise variant 3 runs).  Automatic
 *                      choice: 4 when usable, n_steps >= 4 and (for a batch) systems of at most 8192 points.
 *   "resident_ctas" slabs (CTAs) of variant 4: 1 = one CTA, 2..16 = one thread-block cluster, more = cooperative
 *                  grid; 0 = automatic
 *   "resident_halo" halo columns per side of a slab in the cooperative-grid mode of variant 4 (1..4): neighbours
 *                  exchange their edge columns once per that many half-updates; 0 = automatic (3)
 *   "sweep_steps"  S of variant 3 (1..3) or 5 (2..4), 0 = automatic (variant 5: 4 for columns of >= 320 rows, else 3)
 *   "sweep_ctas"   CTAs of the persistent sweep kernel, 0 = SMs x resident CTAs
 *   "sweep_threads" threads per CTA of the sweep kernel: 128, 256 or (one-step pass only) 512, 0 = automatic
 *   "graph_steps"  launches captured per CUDA graph for launch-bound grids; 0 = plain launches, -1 = auto
 *   "tile_rows"    rows per tile of variant 2 (0 = automatic)
 * Returns BTE_EINVAL for an unknown key or an unsupported value.                                        */
BTE_API int bte_set_option(bte_ctx* ctx, const char* key, int64_t value);

/* What the library would run with the current options (so that a caller can label a measurement without guessing).
 * Keys: "effective_variant" (1, 2, 3 or 5: the streaming kernel bte_step uses when the resident kernel does not
 * apply), "effective_sweep_steps" (leap-frog steps per launch of that kernel), "resident_usable" (1 if bte_step
 * calls of >= 4 steps run the resident kernel in automatic mode), "resident_ctas", "variant", "device" (ordinal of
 * the device that owns the workspace; every entry point selects it and restores the caller's device).           */
BTE_API int bte_get_option(bte_ctx* ctx, const char* key, int64_t* out /* host */);

/* Steady-state detection and averaging policy, evaluated on the device after every time step ("let the
 * system relax" to t = 10, "then compute averages over the period 2 pi / omega"; C23).
 * Per system: P = round(2 pi / (omega dt)) steps is one ac period (omega = 0: P = round(1 / dt), one relaxation time).
 * After every interval of P steps the mean drift velocity m_i of that interval is compared with m_{i-1}; the system
 * counts as relaxed when i >= max(2, min_relax_periods) and |m_i - m_{i-1}| <= rel_tol * max(|m_i|, |m_{i-1}|, 1e-3).
 * From the next step on sum_v_dt, sum_vcos_dt, sum_vsin_dt and window of bte_obs run for exactly
 * round(n_avg_periods * 2 pi / (omega dt)) steps (rounded once for the whole window); then the system is FINISHED: its observables are final and later launches do not advance it (bte_obs.step says
 * where it stopped, at most a launch group beyond the window).  params.avg_start_step is ignored while the policy is on,
 * params.n_steps_total still ends a system.  rel_tol = 0 switches the policy off (default).  Call before
 * bte_init_equilibrium.  Streaming sweep kernels only (fp64, variant 0, 3 or 5; the resident kernel is not used):
 * BTE_EINVAL otherwise.                                                                                          */
BTE_API int bte_set_steady_policy(bte_ctx* ctx, double rel_tol, int32_t n_avg_periods, int32_t min_relax_periods);

/* Per system: the step at which it was found relaxed (0 = not yet) and its phase (0 relaxing, 1 averaging, 2 finished).
 * Synchronises the stream.  steady_step, phase: host, n_batch entries each.                                      */
BTE_API int bte_steady_info(bte_ctx* ctx, int64_t* steady_step /* host */, int32_t* phase /* host */);

/* Number of kernel launches (graph nodes counted individually) issued by this ctx so far. */
BTE_API int bte_launch_count(bte_ctx* ctx, int64_t* out /* host */);

/* Thread-local text of the last error returned on this thread ("" if none). */
BTE_API const char* bte_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* BTE_B200_H */
