/* dg.h -- C-ABI of the B200-native modal DG hot path of arXiv:2208.11131.
 *
 * One handle = one uniform periodic Cartesian mesh with tensor-product Legendre modes per cell
 * (Eq. 6, 121-139 Eq. 13-16; mode set per DESIGN.md reading A1).  The hot path behind
 * dg_step() is the per-Runge-Kutta-stage right-hand side of PAPER.md:175-190 (Eq. 20-21): modal -> Gauss
 * points, volume flux integral (Euler flux Eq. 4, Navier-Stokes flux Eq. 37-39, artificial viscosity
 * Eq. 24, 43-46), face reconstruction + HLLC + recovery-based viscous face flux
 * (Eq. 27-36), lifting, the SSP-RK stage combine and the global CFL
 * reduction (Eq. 23).  Every step runs in hand-written CUDA kernels for sm_100a; there is
 * no CPU fallback: every entry point returns DG_ECUDA when no CUDA device / kernel image is usable.
 *
 * Conventions
 *  - All functions return 0 (DG_OK) or a negative error code; nothing throws or aborts across the ABI.
 *    dg_last_error() returns a static thread-local text for the last failing call.
 *  - Pointers named `w`, `alpha`, `totals`, `out` may be HOST or DEVICE pointers (detected with
 *    cudaPointerGetAttributes); they are caller-owned and only accessed during the call.  All device
 *    state is library-owned and released by dg_free().
 *  - State layout of every caller buffer (the library keeps the same layout internally, except in 3D with
 *    order >= 6, where cells are stored in blocks of 2 or 4 so that the rows of a tile are adjacent in memory; the
 *    conversion happens inside dg_set_state / dg_get_state / dg_eval_rhs / dg_set_alpha / dg_get_alpha):
 *        w[(mode*Vc + var)*Ncells + cell],  Vc = dim+2 (dim+3 with the passive tracer: var dim+2 = c*rho, Eq. 40),
 *        cell = (iz*Ny + iy)*Nx + ix,  mode = (lz*m + ly)*m + lx,  m = order,
 *        var  = rho, rho v_x, rho v_y, (rho v_z), e      (Eq. 1-3).
 *    The artificial-viscosity field alpha is one more modal field, layout
 *        alpha[mode*Ncells + cell].
 *  - `order` is the paper's p = n+1: n = highest Legendre degree per axis, m = n+1
 *    Gauss points per axis.  1 <= order <= 8.
 */
#ifndef DG_B200_H
#define DG_B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

#define DG_OK            0
#define DG_EINVAL       -1   /* bad mesh / order / count / option / null pointer */
#define DG_ENOMEM       -2   /* device allocation failed */
#define DG_EUNPHYSICAL  -3   /* rho <= 0 or p <= 0 met at an evaluation point during dg_step */
#define DG_ECUDA        -4   /* CUDA runtime error, no device, or no sm_100a kernel image */

typedef struct dg_solver dg_solver;   /* opaque, library-owned */

/* Uniform Cartesian mesh of cubes (equal fixed cells of edge h). */
typedef struct dg_mesh {
    int    dim;          /* 2 or 3 */
    int    ncell[3];     /* cells per axis x, y, z (ncell[2] ignored for dim = 2) */
    double origin[3];    /* lower corner (informational: the operator is translation invariant) */
    double h;            /* cell edge */
    int    periodic[3];  /* must be 1 on every used axis (the five workloads are periodic) */
} dg_mesh;

/* Runtime options; defaults are the paper's. */
typedef struct dg_options {
    double f_cfl;        /* Courant factor of Eq. 23; default 0.5 */
    int    rk_stages;    /* 1, 2, 3: SSP-RK in Shu-Osher form, default 3; 5: the five-stage fourth-order
                          * SSP scheme the paper uses for order >= 4 (two more state buffers) */
    int    av_enable;    /* 1: carry the artificial-viscosity field alpha; default 0 */
    double f_v;          /* shock source factor, Eq. 43; default 2.5 */
    double f_tau;        /* decay time factor, Eq. 44; default 0.5 */
    double f_w;          /* wiggle source factor, Eq. 45; default 0.2 */
    double s_onset0;     /* S_onset = s_onset0 / order^2; default 1e-4 */
    double alpha_max;    /* clamp of the point-wise alpha used in Eq. 46; default 1 */
    double fixed_dt;     /* > 0: use this dt instead of Eq. 23; default 0 */
    int    use_graph;    /* 1: replay each time step as a CUDA graph (default); 0: plain launches */
    int    limiter_enable; /* 1: positivity limiter (Eq. 47) on the output of every RK stage; default 0 */
    int    basis;        /* 0 (default): all (n+1)^dim tensor products (BASELINE.json mode counts); 1: the paper's
                          * total-degree set, products with l_x+l_y(+l_z) > n are discarded (Eq. 17-18):
                          * same storage layout, the discarded rows are zeroed by dg_set_state / dg_set_alpha and stay
                          * zero; the sensor of Eq. 42 then uses the modes with l_x+l_y(+l_z) = n */
    int    tracer_enable; /* 1: carry a passive tracer (Eq. 40): one more conserved row c*rho behind
                          * the energy, i.e. Vc = dim+3 in every state count and layout below; default 0 */
    double eta;          /* tracer diffusivity of Eq. 40 (>= 0); default 0 */
} dg_options;

/* Fill *opt with the defaults above. */
int dg_default_options(dg_options *opt);

/* Run-time diagnostics of a solver (dg_get_diagnostics). */
typedef struct dg_diagnostics {
    double    t;               /* simulation time */
    double    last_dt;         /* timestep of the last step (Eq. 23, or fixed_dt) */
    double    c_max, v_max;    /* the two maxima of Eq. 23 that last_dt was computed from (reading A18) */
    double    alpha_max_seen;  /* largest point value of alpha at a volume Gauss point over the states at the start of
                                * every step since dg_set_state (alpha should stay below ~1); 0 without AV */
    long long steps;           /* full RK steps since dg_set_state */
    int       unphysical;      /* device flag, 0 = clean; bits: 1 volume point, 2 face point, 4 wave-speed pass,
                                * 8 limiter cell mean saw rho <= 0 or p <= 0 */
} dg_diagnostics;

/* Create a solver (PAPER.md:175-190 operator on `mesh`; gamma of Eq. 5; nu, chi of Eq. 37-39; nu = chi = 0
 * selects the Euler path).  Allocates all device state; the state is zero until dg_set_state.
 * opt may be NULL (defaults).  Errors: DG_EINVAL, DG_ENOMEM, DG_ECUDA. */
int dg_init(dg_solver **out, const dg_mesh *mesh, int order, double gamma, double nu, double chi,
            const dg_options *opt);

/* Same as dg_init, but all device state lives in a caller-provided device buffer (e.g. a torch tensor):
 * dg_workspace_bytes() gives the size needed; `device_workspace` must be 256-byte aligned, stay alive
 * until dg_free() and is never freed by the library. */
int dg_workspace_bytes(const dg_mesh *mesh, int order, const dg_options *opt, size_t *bytes);
int dg_init_workspace(dg_solver **out, const dg_mesh *mesh, int order, double gamma, double nu, double chi,
                      const dg_options *opt, void *device_workspace, size_t bytes);

/* Change the run-time options of an existing solver: f_cfl, fixed_dt, the AV factors of Eq. 43-46 (f_v, f_tau, f_w,
 * s_onset0), alpha_max, use_graph, limiter_enable, and eta within the limits below.  Fixed at dg_init (the call returns
 * DG_EINVAL and changes nothing if *opt differs from the solver in one of them):
 *   rk_stages, av_enable   they size the device buffers;
 *   tracer_enable          it changes the state layout (Vc);
 *   basis                  the mode set cannot change under a loaded state;
 *   eta == 0  <->  eta > 0 when nu = chi = 0: that switches between the inviscid and the viscous kernel variant
 *                          (with nu or chi > 0 any eta >= 0 is accepted).
 * Every value is validated as in dg_init.  Takes effect at the next dg_step. */
int dg_set_options(dg_solver *s, const dg_options *opt);

/* Run all later work of this solver on `cuda_stream` (a cudaStream_t passed as void*; NULL = default
 * stream).  The Python binding passes torch's current stream. */
int dg_set_stream(dg_solver *s, void *cuda_stream);

/* Upload the modal state (layout above).  count must equal Vc*M*Ncells.  Resets alpha := 0, the sensor
 * scalars := 0 and t := 0, and evaluates the wave speeds of Eq. 23 for the first step. */
int dg_set_state(dg_solver *s, const double *w, size_t count);

/* Overwrite the alpha field (count = M*Ncells); only valid with av_enable. */
int dg_set_alpha(dg_solver *s, const double *alpha, size_t count);

/* Advance nsteps full SSP-RK steps, each with its own Eq.-23 timestep (or fixed_dt).  All stages run on
 * the device without host synchronisation; the call returns after the last step has finished.
 * Returns DG_EUNPHYSICAL if any evaluation point saw rho <= 0 or p <= 0 (state then unspecified). */
int dg_step(dg_solver *s, int nsteps);

/* As dg_step but without the final synchronisation / flag read (for back-to-back timing);
 * errors surface at the next dg_step / dg_sync / dg_get_state. */
int dg_step_async(dg_solver *s, int nsteps);

/* Wait for all queued work; returns DG_EUNPHYSICAL if the device flag is set. */
int dg_sync(dg_solver *s);

/* Download the modal state / alpha field. */
int dg_get_state(dg_solver *s, double *w, size_t count);
int dg_get_alpha(dg_solver *s, double *alpha, size_t count);

/* |K| * sum_cells w_0 per conserved variable (mode 0 is the cell mean):
 * totals[0] = mass, totals[1..dim] = momentum, totals[dim+1] = energy; unused entries are 0.
 * `totals` is a HOST pointer to 5 doubles.  Deterministic fixed-shape reduction. */
int dg_conserved_totals(dg_solver *s, double totals[5]);
/* |K| * sum_cells of the cell means of the tracer row c*rho (conserved by Eq. 40 on a periodic mesh); DG_EINVAL
 * without tracer_enable.  `total` is a HOST pointer. */
int dg_tracer_total(dg_solver *s, double *total);

/* Evaluate dw/dt = L(w) (Eq. 20) of the current state without advancing it, for term-wise parity tests:
 * out has the layout of the state (count = Vc*M*Ncells); alpha_out (may be NULL) that of alpha. */
int dg_eval_rhs(dg_solver *s, double *out, size_t count, double *alpha_out, size_t alpha_count);

/* Apply the positivity limiter (Eq. 47) once to the current state, whatever `limiter_enable` says
 * (term-level parity tests; dg_step applies it after every RK stage when the option is on).  Returns
 * DG_EUNPHYSICAL if a cell mean has rho <= 0 or p <= 0. */
int dg_apply_limiter(dg_solver *s);

/* Simulation time and the last timestep used (host pointers, either may be NULL). */
int dg_get_time(dg_solver *s, double *t, double *last_dt);

/* Time, last timestep, the Eq.-23 wave-speed maxima, the running maximum of alpha, step count and the
 * unphysical-state flag in one call (`d` is a HOST pointer).  Synchronises the solver's stream. */
int dg_get_diagnostics(dg_solver *s, dg_diagnostics *d);

/* Checkpoint / restart of the lagged shock sensor ("two scalar quantities per cell"; reading
 * A15): sg[0..N) = S^K, sg[N..2N) = G^K = d ln S / dt of the previous step; count = 2*Ncells; HOST or DEVICE pointer.
 * A run is resumed bit-identically by dg_set_state + dg_set_alpha + dg_set_sensor + dg_set_time with the values read
 * from dg_get_state / dg_get_alpha / dg_get_sensor / dg_get_time (dg_set_state zeroes alpha, sensor and t). */
int dg_get_sensor(dg_solver *s, double *sg, size_t count);
int dg_set_sensor(dg_solver *s, const double *sg, size_t count);
int dg_set_time(dg_solver *s, double t);

/* Launch geometry of the stage kernel of this solver (for bench.py / DESIGN.md): cells per block, threads
 * per block, dynamic shared memory bytes per block, number of blocks.  Any pointer may be NULL. */
int dg_kernel_info(dg_solver *s, int *cells_per_block, int *threads, int *smem_bytes, int *blocks);

/* Device time of the two kernels of one RK stage, measured with CUDA events on the solver's stream around each
 * launch, averaged over `reps` repetitions (after one warm-up pass), in milliseconds.  face_ms / stage_ms are HOST
 * pointers (either may be NULL).  With rk_stages >= 3 the stage timed is the MIDDLE stage of SSP-RK3 with its real
 * combine (reads u^n and a copy of the state as u^(1), writes u^(2) = 3/4 u^n + 1/4 (u^(1) + dt L(u^(1))) into a stage
 * buffer; no sensor refresh, no wave-speed pass); with fewer stages it is the dg_eval_rhs form (dw/dt only).  The
 * state itself is not advanced; the stage buffers are overwritten.  Used by bench.py for the per-kernel roofline. */
int dg_profile_stage(dg_solver *s, int reps, double *face_ms, double *stage_ms);

/* Number of kernel launches issued by this solver since dg_init (graph replays count their nodes). */
int dg_launch_count(dg_solver *s, long long *count);

/* Sustained fp64 FMA throughput of the device in FLOP/s, measured with a register-resident DFMA loop of
 * `iters` iterations on every SM (roofline denominator for the ALU-bound configs). */
int dg_measure_fp64_peak(int iters, double *flops_per_s, void *cuda_stream);

/* Conserved totals for callers that must not allocate device memory.
 *
 * Who this is for: code that runs where every byte of the GPU is already spoken for or where an allocation is simply
 * not allowed at that point -- an in-situ diagnostics hook called from inside somebody else's time loop on a device
 * the simulation has filled, a plug-in living inside a framework whose memory pool owns the whole card (a raw
 * cudaMalloc beside the pool fails or fragments it), a job started under a hard per-process memory cap, or a
 * latency-bound monitoring thread that cannot afford the device-wide stall cudaMalloc / cudaFree imply.  Such callers
 * cannot create a dg_solver (dg_init allocates, dg_init_workspace needs a workspace somebody allocated) just to ask
 * "how much mass, momentum and energy is in this state?".
 *
 * What it computes: the same quantity as dg_conserved_totals -- cell_volume * sum over cells of the mode-0 weight
 * (the cell mean) of each of the first `nvars` variables -- by a compensated, fixed-shape and
 * therefore run-to-run reproducible reduction (4096 cells per block, block partials combined in block order).
 *
 *   w            DEVICE pointer (on the current device) to a modal state in the layout at the top of this file; only
 *                the rows of mode 0 are read, i.e. w[var*ncells + cell] for var < nvars.  Caller-owned, read only.
 *   nvars        how many leading variables to total, 1 .. DG_NOALLOC_MAX_VARS (dim+2, or dim+3 with the tracer row).
 *   ncells       cells of the mesh, 1 .. DG_NOALLOC_MAX_CELLS.  Larger meshes are refused with DG_EINVAL and a text
 *                that names the limit; nothing is launched in that case.
 *   cell_volume  h^dim.
 *   totals       `nvars` doubles, HOST or DEVICE pointer, caller-owned.  DEVICE: the result is written in stream
 *                order and the call returns without waiting.  HOST: the call copies the result out and waits for
 *                `cuda_stream` before it returns.
 *   cuda_stream  cudaStream_t passed as void* (NULL = default stream).
 *
 * Scratch memory: the block partials live in ONE array compiled into the library (static __device__, 131 136 bytes =
 * (2*8*1024 + 8) doubles).  Every GPU that loads the library carries that array until the process exits, whether or
 * not this function is ever called.  The function itself calls no cudaMalloc / cudaFree / allocating library routine.
 *   - First call on each device: looks up the device address of that array (cudaGetSymbolAddress, with the calling
 *     thread's current device) and remembers it; this may make the CUDA runtime load the library's kernels on that
 *     device.  Make this first call outside any stream capture and with the device you mean to use current.
 *   - All calls on a device share the array and it keeps whatever the previous call left.  Nothing in it has to start
 *     at zero: each call first writes every slot it later reads.  But two calls that overlap on the GPU (different
 *     streams, or two host threads) race on it and return garbage -- serialise them on one stream.
 * Errors: DG_EINVAL (NULL pointer, nvars / ncells out of range, w not device memory of the current device),
 * DG_ECUDA (no device, or a CUDA call failed). */
#define DG_NOALLOC_MAX_CELLS 4194304   /* 2^22 cells = 1024 blocks of 4096 cells; a 128^3 mesh is half of this */
#define DG_NOALLOC_MAX_VARS  8
int dg_totals_noalloc(const double *w, int nvars, long long ncells, double cell_volume, double *totals,
                      void *cuda_stream);

/* Free all device state.  NULL is allowed. */
int dg_free(dg_solver *s);

/* Text of the last error on this thread ("" if none). */
const char *dg_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* DG_B200_H */
