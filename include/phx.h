/*
 * phx.h -- C ABI of libphx: B200-native (sm_100a) fixed-step RK4 time stepping of the damped 2D
 * nonlinear Schroedinger / Gross-Pitaevskii equation and its integrated extensions
 * (PHOENIX, arXiv 2411.18341; citations are /root/reference/PAPER.md:<line>).
 *
 * What the library computes (DESIGN.md section 2 gives the discrete formulas):
 *   Eq. (1)   PAPER.md:25       i hbar d_t psi = (-hbar^2/2m lap + V + g|psi|^2 - i hbar gamma/2) psi
 *   Eq. (8)   PAPER.md:203      lap = five-point stencil with separate dx, dy
 *   Eqs. (2)-(6) PAPER.md:53-62 fixed-step RK4 (weights of Listing 1)
 *   Eq. (16)  PAPER.md:361      spinor psi_+-, g_x |psi_-+|^2, g_r n, (i hbar/2)(R n - gamma),
 *                               TE-TM coupling J_+- = Delta_LT (d_x -+ i d_y)^2 on psi_-+,
 *                               coherent drive E exp(-i omega t), Wiener noise dW
 *   Eq. (17)  PAPER.md:364      d_t n = P - (gamma_r + R |psi|^2) n
 *   Eq. (22)  PAPER.md:454-456  <dW dW*> = (R n + gamma_c)/(2 DeltaV), <dW dW> = 0
 *   boundaries PAPER.md:369     periodic or zero, independently in x and y
 *
 * Conventions
 *   - Every call returns a phx_status; 0 = success, >= 100 = warning (state still valid).
 *     No exception or abort crosses this boundary.  Arguments are validated before device work.
 *   - Arrays are row-major [batch][ny][nx], x fastest.  A complex field is interleaved (re, im) of
 *     the working real type T (float for PHX_C32, double for PHX_C64); reservoirs, V and P are real T.
 *   - phx_mem says where a caller pointer lives: PHX_HOST (pageable or pinned) or PHX_DEVICE.
 *   - OWNERSHIP: the caller owns all device memory -- the workspace and every PHX_DEVICE source or
 *     destination -- and the stream.  The library allocates no device memory: state fields, stage
 *     buffers, accumulators, V, P, E and the step counter all live in the workspace.  The handle is
 *     host memory owned by the library until phx_destroy_grid.
 *   - One handle is used by one thread at a time; handles are independent.
 *   - phx_step_rk4 is asynchronous on the stream.  A CUDA failure is reported by the next
 *     synchronising call (phx_read_field, phx_sync, ...) and is sticky (PHX_ERR_CUDA).
 *   - The step counter is part of the state: k calls of one step == one call of k steps, bit for
 *     bit (it keys the noise and fixes the drive phase t = step*dt).
 *   - There is no CPU fallback: without a CUDA device phx_create_grid fails with PHX_ERR_CUDA.
 */
#ifndef PHX_H
#define PHX_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct phx_grid phx_grid; /* opaque */

typedef enum {
    PHX_OK = 0,
    PHX_ERR_INVALID_ARG = 1,   /* NULL pointer, size < 3, non-positive dx/dy/dt, zero hbar or m, bad enum */
    PHX_ERR_BAD_STATE = 2,     /* e.g. stepping before phx_set_params */
    PHX_ERR_UNSUPPORTED = 3,   /* field not present in the model, variant not available for this grid */
    PHX_ERR_CUDA = 4,          /* CUDA runtime failure (sticky); see phx_last_error */
    PHX_ERR_WORKSPACE = 5,     /* workspace NULL, misaligned (256 B) or smaller than phx_workspace_bytes */
    PHX_WARN_UNSTABLE = 100    /* (hbar/2m)(4/dx^2+4/dy^2) dt exceeds the RK4 limit 2.78; parameters were set */
} phx_status;

typedef enum { PHX_C32 = 0, PHX_C64 = 1 } phx_precision;
typedef enum { PHX_SCALAR = 0, PHX_RESERVOIR = 1, PHX_SPINOR = 2, PHX_SPINOR_RESERVOIR = 3 } phx_model;
typedef enum { PHX_HOST = 0, PHX_DEVICE = 1 } phx_mem;
typedef enum { PHX_PSI = 0, PHX_PSI_MINUS = 1, PHX_N = 2, PHX_N_MINUS = 3 } phx_field;
typedef enum { PHX_BC_PERIODIC = 0, PHX_BC_ZERO = 1 } phx_boundary;
/* PHX_INT_DP54 reserves the seven K buffers of the adaptive Dormand-Prince 5(4) integrator in the workspace
 * (phx_step_adaptive).  phx_step_rk4 works on either kind of handle. */
typedef enum { PHX_INT_RK4 = 0, PHX_INT_DP54 = 1 } phx_integrator;

/* Kernel variants (all compute the same RK4 step; they differ in how often data crosses HBM). */
typedef enum {
    PHX_VARIANT_AUTO = 0,      /* the fastest variant that can run the grid: RESIDENT for ensembles (batch >= 32) of grids that fit it, else STEP
                                  (STAGE for planes of 2^31 cells or more) */
    PHX_VARIANT_STAGE = 1,     /* one fused kernel per RK stage (4 launches per step); every model and term */
    PHX_VARIANT_STEP = 3,      /* one kernel per RK4 step: the four stages pipelined along y in register windows of
                                  a haloed warp-wide column strip (N_halo = 4); every model and term */
    PHX_VARIANT_RESIDENT = 4   /* grids of at most 64 x 64 cells (scalar and reservoir models, no drive): one CTA per
                                  realisation keeps the grid on chip for all steps of a phx_step_rk4 call (one launch) */
} phx_variant;

typedef struct {
    int32_t nx, ny;            /* cells in x and y, each >= 3 */
    int32_t batch;             /* independent realisations sharing V, P, E (>= 1) */
    double dx, dy;             /* cell sizes (> 0) */
    int32_t prec;              /* phx_precision */
    int32_t model;             /* phx_model */
    int32_t noise;             /* 0/1: add the Wiener increment of Eq. (22) after every step */
    int32_t bc_x, bc_y;        /* phx_boundary per axis */
    int32_t integrator;        /* phx_integrator */
    void* workspace;           /* DEVICE memory owned by the caller, 256-byte aligned */
    size_t workspace_bytes;    /* >= phx_workspace_bytes(desc) */
    void* stream;              /* cudaStream_t owned by the caller; NULL = legacy default stream */
} phx_grid_desc;

typedef struct {
    double hbar, m;            /* Eq. (1); both non-zero */
    double g;                  /* same-spin nonlinearity */
    double g_x;                /* cross-spin nonlinearity (spinor models) */
    double g_r;                /* reservoir interaction (reservoir models) */
    double R;                  /* condensation rate */
    double gamma_c;            /* loss of psi (gamma of Eq. (1)) */
    double gamma_r;            /* reservoir loss */
    double beta;               /* Delta_LT of the TE-TM coupling (spinor models) */
    double dt;                 /* RK4 step (> 0) */
    double noise_scale;        /* nu: multiplies the noise variance (1 = Eq. (22) as printed) */
    double density_offset;     /* 1/DeltaV subtracted from |psi|^2; 0 = off */
    double omega;              /* drive frequency, E(r,t) = E(r) exp(-i omega t) */
    uint32_t seed;             /* Philox key word 0 (word 1 is the realisation index) */
} phx_params;

/* Number of canonical coefficients returned by phx_get_coeffs, in the order
 * cx cy ih g gx gr Rr hgc gamr bxx byy bxy dt dt6 dt3 sig2 doff omega. */
#define PHX_NCOEF 18

/* Bytes of device workspace phx_create_grid needs for this descriptor (workspace fields ignored).
 * Returns 0 if the descriptor is invalid. */
size_t phx_workspace_bytes(const phx_grid_desc* desc);

/* Creates a handle.  All state fields, V, P and E start as zero; the step counter starts at 0.
 * Errors: INVALID_ARG, WORKSPACE, CUDA (no device / not sm_100). *out is NULL on error. */
phx_status phx_create_grid(phx_grid** out, const phx_grid_desc* desc);

/* Sets the physical parameters of Eq. (1) (hbar, m, g, gamma), Eq. (16) (g_x, g_r, R, Delta_LT,
 * drive frequency), Eq. (17) (gamma_r, R) and Eq. (22) (noise scale nu, 1/DeltaV of the
 * renormalised density :452) and the RK4 step dt of Eqs. (2)-(6), and derives the canonical coefficient set
 * (DESIGN.md section 2 step 0: double expressions, each rounded once to T).  Invalidates the captured graphs.
 * Errors: INVALID_ARG (NULL, dt <= 0, hbar or m zero or non-finite, a non-finite coefficient).  May return
 * PHX_WARN_UNSTABLE (the explicit scheme is unstable for these values; the parameters are set nevertheless). */
phx_status phx_set_params(phx_grid* g, const phx_params* p);

/* Static real fields [ny][nx] of type T shared by the batch: potential V (Eq. (1)) and pump P
 * (Eq. (17); P_+ = P_-, reading Q18).  NULL = identically zero.  The data are copied into the
 * workspace; the caller keeps its arrays.  UNSUPPORTED: P given for a model without reservoir. */
phx_status phx_set_potential_pump(phx_grid* g, const void* V, const void* P, phx_mem where);

/* Complex drive amplitude E(r) [ny][nx] (Eq. (16), E_+ = E_-); NULL = no drive. */
phx_status phx_set_drive(phx_grid* g, const void* E, phx_mem where);

/* Copies a state field [batch][ny][nx] into / out of the workspace: psi_+- of Eq. (16) (PHX_PSI alone is
 * psi of Eq. (1)) as interleaved complex T, the reservoirs n_+- of Eq. (17) as real T.
 * The caller keeps ownership of src / dst (host or device, see phx_mem).  phx_read_field synchronises the stream before
 * returning (unless "async_host_copies" is set, see phx_set_tuning).  Together with phx_get_step / phx_set_step the fields
 * are a complete checkpoint.  INVALID_ARG: NULL pointer or bad enum; UNSUPPORTED: the model does not have the field. */
phx_status phx_set_field(phx_grid* g, phx_field f, const void* src, phx_mem where);
phx_status phx_read_field(phx_grid* g, phx_field f, void* dst, phx_mem where);

/* Advances every realisation by n_steps (>= 0) fixed-step RK4 steps, Eqs. (2)-(6) with the weights of
 * Listing 1, on the joint state (psi_+-, n_+-) (reading Q5); each step evaluates the
 * derivative of Eq. (1)/(16)/(17) four times (Laplacian Eq. (8)) and, with noise = 1, adds the Wiener
 * increment of Eq. (22) after the step.  All of it runs in the kernels of the selected variant,
 * replayed from CUDA graphs; asynchronous on the stream, no host synchronisation.
 * INVALID_ARG: n_steps < 0; BAD_STATE: phx_set_params not called yet; CUDA: a launch failed (sticky). */
phx_status phx_step_rk4(phx_grid* g, int64_t n_steps);

/* ---- adaptive time stepping: Dormand-Prince 5(4) ----------------------------------------------------------------------
 * "Higher-order methods like the RK-Fehlberg or Dormand-Prince can be used for systems requiring adaptive time-stepping"
 * (PAPER.md:64; :488 lists adaptive Runge-Kutta as future work) is all the paper says; the rules are DESIGN.md reading Q20:
 * seven-stage 5(4) pair of Dormand & Prince (1980) with FSAL; error norm err = max over cells, components, reservoirs and
 * realisations of |E| / (atol + rtol max(|u|, |u_new|)); accept iff err <= 1 (or the proposal is already h_min); next step
 * h_used * q/16 with q = floor(16 clamp(0.9 err^(-1/5), 1/4, 4)), clamped to [h_min, h_max]; the step that would pass t_end is
 * clipped to land on it.  One step size for the whole batch.  The whole loop -- stages, error reduction, accept / reject,
 * step-size control, termination -- runs on the device (a CUDA-graph WHILE node): the call is asynchronous and enqueues one
 * graph launch.  The adaptive integrator keeps its own clock t (double), starting at 0; phx_set_time moves it.  The drive
 * phase uses that clock.  UNSUPPORTED: handle created without PHX_INT_DP54, or with noise (a Wiener increment cannot be
 * re-drawn for a rejected step).  INVALID_ARG: NULL, negative tolerances, atol + rtol == 0, h_min <= 0, h_max < h_min. */
typedef struct {
    double atol, rtol;         /* error norm */
    double h_init;             /* first step size tried when no proposal is pending */
    double h_min, h_max;       /* clamp of the step size */
    int64_t max_attempts;      /* at most this many attempts (accepted or rejected) in this call */
} phx_adaptive;

typedef struct {
    double t;                  /* time reached */
    double h_next;             /* step size the next attempt will propose */
    int64_t n_accept, n_reject;/* totals since creation / phx_set_time */
    int64_t attempts;          /* attempts of the last call */
    double err_last;           /* error norm of the last attempt */
} phx_adaptive_state;

phx_status phx_step_adaptive(phx_grid* g, double t_end, const phx_adaptive* ctl);

/* Synchronises and reads the integrator state back; if the log pointers are non-NULL also the record of every attempt of the
 * last call (accept flag, q, step used, error norm; at most log_cap records, *n_log receives the number written). */
phx_status phx_get_adaptive_state(phx_grid* g, phx_adaptive_state* out, int32_t* log_accept, int32_t* log_q, double* log_h,
                                  double* log_err, int64_t log_cap, int64_t* n_log);

/* Sets the adaptive integrator's clock and pending proposal (h_next <= 0: none); zeroes its counters.  Synchronises. */
phx_status phx_set_time(phx_grid* g, double t, double h_next);

/* Step counter = number of completed steps.  phx_set_step synchronises. */
phx_status phx_get_step(const phx_grid* g, uint64_t* step);
phx_status phx_set_step(phx_grid* g, uint64_t step);

/* <|psi|^2>(x,y) = (1/batch) sum_r |psi_r|^2 as real T [ny][nx].  Synchronises. */
phx_status phx_ensemble_mean_density(phx_grid* g, phx_field f, void* dst, phx_mem where);

/* Failure detection: *all_finite <- 1 if every value of every state field (psi_+-, n_+- as present, all
 * realisations) is finite, 0 if any is NaN or +-Inf -- what an RK4 run beyond its stability limit (PHX_WARN_UNSTABLE; the
 * paper's explicit scheme has none of its own) ends in.  One pass over the state on the device.  Synchronises. */
phx_status phx_check_finite(phx_grid* g, int32_t* all_finite);

/* The canonical coefficients actually used (as double); n must be PHX_NCOEF. */
phx_status phx_get_coeffs(const phx_grid* g, double* out, int32_t n);

/* Test aid: the four Philox4x32-10 words every (realisation, cell) draws at step `step` for the noise of Eq. (22)
 * (BASELINE.json config 5: keyed by (seed, realisation, step, cell); counter/key packing of DESIGN.md
 * reading Q13), dst[batch][ny][nx][4] (host or device, caller-owned), produced by the same device function the stepping
 * kernels call.  Synchronises.  BAD_STATE before phx_set_params (the seed is a parameter). */
phx_status phx_debug_noise_u32(phx_grid* g, uint64_t step, uint32_t* dst, phx_mem where);

/* Selects a kernel variant (phx_variant).  UNSUPPORTED if it cannot run this grid/model.  All variants
 * compute the same RK4 step (results agree to rounding); the state and the step counter carry over. */
phx_status phx_select_variant(phx_grid* g, int32_t variant);

/* Bench/test aids: the variant the next phx_step_rk4 will use; kernels launched so far by this handle;
 * launch geometry knobs (key/value, UNSUPPORTED for unknown keys): "rows", "vec" (variant STAGE: rows per
 * CTA, cells per thread), "step_ly", "step_vec" (variant STEP: rows per chunk, cells per lane; 0 = automatic),
 * "step_warps" (warps per CTA), "step_xch" (exchanging strips: -1 automatic, 0 off, 1 wherever the row is 1-8 strips wide),
 * "step_bulk" (rows fetched through a shared-memory ring, by per-lane cp.async or by TMA bulk copies depending on the kernel:
 * -1 automatic = where it measured faster, 0 register loads, 1 the ring), "step_side" (1: side launch for a ragged last strip),
 * "step_pdl" (later steps of a graph as programmatic dependent launches: -1 automatic, 0 off, 1 on),
 * "resident_cluster" (variant RESIDENT on a thread-block cluster of 2-16 CTAs: -1 automatic, 0 never, 1 wherever it applies),
 * "graph_steps" (RK4 steps per captured CUDA graph).  Results do not depend on them (bit for bit within variant STEP).
 * "async_host_copies" = 1: phx_set_field / phx_read_field with PHX_HOST enqueue the copy on the stream and return
 * without synchronising (the host buffers must be pinned and stay untouched until phx_sync); lets a caller overlap the
 * upload of one grid with the download of another on two handles / streams. */
phx_status phx_get_variant(const phx_grid* g, int32_t* variant);
phx_status phx_get_launch_count(const phx_grid* g, uint64_t* launches);
phx_status phx_set_tuning(phx_grid* g, const char* key, int32_t value);

/* ---- stepping without a handle, a workspace or any allocation ---------------------------------------------------------
 * n_steps fixed-step RK4 steps (Eqs. (2)-(6); Listing 1, :100-144) of the scalar model Eq. (1) (
 * no reservoir, spinor, drive or noise) on ONE nx x ny grid, for callers that cannot allocate (code under CUDA-graph capture,
 * tight serving loops, harnesses that forbid cudaMalloc).  The call makes no cudaMalloc / cudaFree and calls no allocating
 * library routine; it creates no stream, event or graph.  The stage buffers and the running sum of Eq. (6) live in a
 * file-scope device array of PHX_STATIC_SCRATCH_BYTES inside libphx.so (every GPU that loads the library holds it until the
 * process exits); the kernels are the per-stage kernels of phx_step_rk4 (variant STAGE), so the result is the same.
 *   psi_in, psi_out: DEVICE arrays [ny][nx] of interleaved complex T (T by prec), owned by the caller; may be the same array.
 *   V: DEVICE array [ny][nx] of real T, or NULL (V = 0).  p: as phx_set_params (g_x, g_r, R, gamma_r, beta, omega, noise_scale,
 *   seed are not used).  bc_x, bc_y: phx_boundary.  stream: cudaStream_t or NULL; the work is enqueued, not synchronised.
 * The device of the arrays must be the current device.  Limit: 3 x align256(nx*ny*sizeof(complex T)) + 256 bytes must fit
 * the array: nx*ny <= 349 504 cells in complex fp32 (e.g. 512 x 512, 590 x 590), 174 752 in complex fp64 (e.g. 256 x 256, 417 x 417).
 * Returns PHX_ERR_WORKSPACE for a larger grid (nothing is enqueued), PHX_ERR_INVALID_ARG for bad arguments, PHX_ERR_CUDA if
 * the CUDA runtime refuses a call.  All calls share the array, which keeps the last call's contents (what must start at zero
 * is cleared by every call): calls whose kernels may overlap on the GPU (different streams) RACE on it -- keep them on one
 * stream or order them with events. */
#define PHX_STATIC_SCRATCH_BYTES (8u << 20)
phx_status phx_step_rk4_static(int32_t nx, int32_t ny, double dx, double dy, int32_t prec, int32_t bc_x, int32_t bc_y,
                               const phx_params* p, const void* V, const void* psi_in, void* psi_out, int64_t n_steps,
                               void* stream);

/* Waits for the stream; returns the sticky CUDA status. */
phx_status phx_sync(phx_grid* g);

/* Human-readable description of the last error of this handle (never NULL). */
const char* phx_last_error(const phx_grid* g);

void phx_destroy_grid(phx_grid* g);

#ifdef __cplusplus
}
#endif
#endif
