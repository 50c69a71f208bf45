/* rgrmhd.h -- C-ABI of the B200-native resistive GRMHD IMEX-RK2 step.
 *
 * What it is: one full IMEX-SSP2(2,2,2) step (Eq. 35-37) of the resistive
 * GRMHD conserved system (Eq. 22-29) on one uniform 3D Cartesian block with
 * ghost zones and a fixed, externally supplied 3+1 metric (Eq. 1-5).  All
 * arithmetic is FP64 and runs in hand-written sm_100a CUDA kernels; there is no CPU fallback.
 *
 * Field layout (every array argument): a padded structure-of-arrays field of
 *     nxp * nyp * nzp doubles,   n?p = n? + 2*ng if n? > 1 else 1,   x fastest,
 *     index(i,j,k) = (i+gx) + nxp*((j+gy) + nyp*(k+gz)),  g? = ng if n? > 1 else 0.
 * Vector components are coordinate components: v^i, E^i, B^i, beta^i contravariant; S_i
 * covariant; gamma_ij, K_ij covariant, stored xx,xy,xz,yy,yz,zz.
 *
 * Pointers: every field pointer may be a DEVICE pointer on params.device or a HOST pointer
 * (pageable or pinned); the library copies with cudaMemcpyAsync(..., cudaMemcpyDefault) on its
 * stream, so unified addressing classifies the pointer.  Pointer tables (the `const double* const x[14]`
 * arguments) are HOST arrays of such pointers.  Host scalars/structs are written
 * synchronously.
 *
 * Ownership: the handle owns all internal device memory.  Caller arrays are read (set_*) or
 * written (get_*) by work enqueued during the call and are never retained.
 *
 * Ordering: all calls enqueue on the handle's stream (default: the legacy default stream;
 * rgrmhd_set_stream changes it) and return without host synchronisation, except
 * rgrmhd_max_speed and rgrmhd_get_stats (host scalars: they synchronise the stream), rgrmhd_set_metric and
 * copies from/to pageable host memory (synchronous by CUDA's rules).
 *
 * Errors: every function returns 0 on success or a negative rgrmhd_status.  No exceptions
 * cross the ABI, there is no global state, and handles are not thread-safe.  A cell whose
 * root solve does not converge is NOT an error: it keeps its last iterate (or the floor
 * values) and is counted in rgrmhd_stats.
 */
#ifndef RGRMHD_H
#define RGRMHD_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct rgrmhd_s* rgrmhd_t;

enum rgrmhd_status {
  RGRMHD_OK        =  0,
  RGRMHD_E_INVALID = -1, /* null pointer, ng != 3, n < 1, dx <= 0, Gamma <= 1, unknown enum     */
  RGRMHD_E_STATE   = -2, /* step/get before set_metric + set_prims; set_sigma w/o ARRAY model;
                            any call but set_prims/destroy after a launch inside rgrmhd_step failed
                            (the state is half advanced: the handle refuses to hand it out)      */
  RGRMHD_E_CUDA    = -3, /* a CUDA call failed; rgrmhd_last_cuda_error() returns its string    */
  RGRMHD_E_NOMEM   = -4, /* device allocation failed                                            */
  RGRMHD_E_TOO_LARGE = -5 /* rgrmhd_max_speed_static only: more cells than its fixed scratch array allows */
};

/* boundary conditions ("Neumann": copy nearest interior cell; PAPER.md:359 periodic) */
enum { RGRMHD_BC_PERIODIC = 0, RGRMHD_BC_OUTFLOW = 1,
       /* the ghost layers of this direction belong to the CALLER (the block is a slab of a larger grid, PAPER.md:169
        * "boxes"): the library never writes them; the caller fills them through
        * rgrmhd_halo_unpack at the two exchange points of a split step (rgrmhd_step_begin / rgrmhd_step_continue).
        * Needs n >= 3 in that direction; not available with charge mode DIV_E or the general tableau driver. */
       RGRMHD_BC_EXTERNAL = 2 };

/* conductivity models: uniform; per-cell array (BASELINE config 4); sigma0*(D/Dref)^exp
 * (Eq. 52; D undensitised, exp a non-negative integer);
 * sigma0*max(1 - D_atmo/D, 0)^2 (Eq. 61; sigma_dref = D_atmo). */
enum { RGRMHD_SIGMA_UNIFORM = 0, RGRMHD_SIGMA_ARRAY = 1, RGRMHD_SIGMA_POWER_D = 2, RGRMHD_SIGMA_ATMO = 3 };

/* how the conduction current in the charge flux (last row of Eq. 27) is evaluated at faces;
 * the paper is silent (reading R3):
 *   FACE_OHM     Ohm's law (Eq. 29) on the reconstructed left/right states, sigma_L/R = cell sigma
 *   CELL_CURRENT (default) the cell-centred conduction current fixed by the implicit solve of the
 *                same stage, J_c = (calE* - calE)/(a_ii dt alpha), reconstructed like a primitive
 *   DIV_E        the charge is not evolved: q = nabla_i E^i of each stage's electric field,
 *                second-order centred differences of sqrt(gamma) E^i (reading R15); the
 *                new state's q and calQ are computed when the state is read. */
enum { RGRMHD_CHARGE_FACE_OHM = 0, RGRMHD_CHARGE_CELL_CURRENT = 1, RGRMHD_CHARGE_DIV_E = 2 };

/* characteristic speeds of HLLE and of the CFL reduction:
 *   LIGHT       lambda+- = +-alpha sqrt(gamma^kk) - beta^k everywhere (Eq. 30; default)
 *   MHD_INSIDE  the paper's alternative: the ideal-GRMHD value inside the star, the speed
 *               of light outside.  Ideal-GRMHD value = the fast-magnetosonic bound a^2 = cs^2 + vA^2 - cs^2 vA^2
 *               boosted to the coordinate frame (reading R16), envelope of the two face states;
 *               "inside" = both face states have rho > wave_rho_switch. */
enum { RGRMHD_WAVE_LIGHT = 0, RGRMHD_WAVE_MHD_INSIDE = 1 };

/* `scheme` argument of rgrmhd_step = reconstruction | time scheme */
enum { RGRMHD_RECON_MINMOD = 0, RGRMHD_RECON_MC = 1, RGRMHD_RECON_WENO5 = 2, RGRMHD_RECON_MASK = 0xff };
/* time schemes: the IMEX-RK SSP schemes the paper incorporates.  SSP2_222 (Eq. 35-37, Table I) is the
 * paper's production scheme and this library's tuned path (6 launches per step, deferred final recovery); the others
 * run through the general double-Butcher-tableau driver of Eq. 32-34 (one point-wise kernel per stage plus one for the
 * new state, one flux kernel per stage whose F is used); SSP2_222_GENERAL is the production scheme through that
 * driver (a cross-check: same result to round-off). */
enum { RGRMHD_TIME_IMEX_SSP2_222 = 0 << 8, RGRMHD_TIME_IMEX_SSP2_332 = 1 << 8, RGRMHD_TIME_IMEX_SSP3_332 = 2 << 8,
       RGRMHD_TIME_IMEX_SSP3_433 = 3 << 8, RGRMHD_TIME_IMEX_SSP2_222_GENERAL = 4 << 8, RGRMHD_TIME_MASK = 0xff00 };

typedef struct {
  int    n[3];        /* interior cells per direction; n = 1 marks an inactive direction          */
  double dx[3];       /* cell sizes (> 0; ignored for inactive directions)                        */
  int    ng;          /* ghost zones per side of an active direction; must be 3                   */
  int    bc[3];       /* RGRMHD_BC_* per direction                                                */
  double gamma_eos;   /* ideal-gas Gamma, p = (Gamma-1) rho eps (Eq. 49)            */
  int    sigma_model; /* RGRMHD_SIGMA_*                                                           */
  double sigma0, sigma_exp, sigma_dref;
  double kappa;       /* divergence-cleaning damping (1)                            */
  double rho_floor;   /* atmosphere density; 0 disables the floor                  */
  double k_atmo;      /* polytropic K of the atmosphere, p = K rho^Gamma           */
  double c2p_tol;     /* relative tolerance of the root solve; <= 0 selects 8*2^-52               */
  int    c2p_max_iter;/* cap on residual evaluations per cell and solve; <= 0 selects 100         */
  int    charge_mode; /* RGRMHD_CHARGE_*                                                          */
  double weno_eps;    /* WENO5 regulariser; <= 0 selects 1e-26 (reading R5)             */
  int    device;      /* CUDA device ordinal                                                      */
  int    wave_speed_mode;  /* RGRMHD_WAVE_*: characteristic speeds of the HLLE solver                     */
  double wave_rho_switch;  /* MHD_INSIDE: "inside the star" = both face states denser than this           */
} rgrmhd_params;

typedef struct {
  long long c2p_solves;     /* cell solves performed since create/reset                           */
  long long c2p_evals;      /* residual evaluations summed over those solves                      */
  long long c2p_failures;   /* solves that hit the cap or had no physical bracket                 */
  long long floor_resets;   /* cells reset to the atmosphere                                      */
  int       c2p_max_evals;  /* largest evaluation count of any single solve                       */
  int       reserved;
} rgrmhd_stats;

/* Fill *p with the defaults documented above (kappa = 1, charge_mode = CELL_CURRENT, ...). */
int rgrmhd_params_default(rgrmhd_params* p);

/* Allocate a handle and all device state for the block. */
int rgrmhd_create(rgrmhd_t* out, const rgrmhd_params* p);
int rgrmhd_destroy(rgrmhd_t h);

/* Use `cuda_stream` (a cudaStream_t, e.g. torch's current stream) for all later work.  Work already enqueued
 * on the previous stream (copies of set_*, kernels, a pending final recovery -- which is flushed there first) is
 * ordered BEFORE anything enqueued later on the new stream (event on the old stream, wait on the new one), so the
 * switch is safe between any two calls, also with non-blocking streams. */
int rgrmhd_set_stream(rgrmhd_t h, void* cuda_stream);

/* Fixed 3+1 metric: lapse, shift beta^i, gamma_ij, K_ij as padded
 * fields INCLUDING ghost zones (the library never extrapolates a metric).  Also computes the metric-only
 * coefficients of the geometric sources (derivatives, G^i, tr K) and allocates one field for each of them that is
 * not identically zero on the grid (up to 34; 9 for a static conformally flat metric without shift): this call
 * therefore synchronises the stream once and may return RGRMHD_E_NOMEM. */
int rgrmhd_set_metric(rgrmhd_t h, const double* alpha, const double* const beta[3],
                      const double* const gam[6], const double* const K[6]);

/* Per-cell conductivity (SIGMA_ARRAY model only), padded field. */
int rgrmhd_set_sigma(rgrmhd_t h, const double* sigma);

/* Primitive state: rho,p,vx,vy,vz,Ex,Ey,Ez,Bx,By,Bz,psi,phi,q.  Also computes
 * the conserved state (Eq. 22-24, 28).  Requires set_metric first. */
int rgrmhd_set_prims(rgrmhd_t h, const double* const prims[14]);

/* One IMEX-RK step of size dt.  scheme = RGRMHD_RECON_* | RGRMHD_TIME_*.  SSP2(2,2,2) (Eq. 35-37): implicit-E +
 * recovery (+ the point-wise explicit sources and stage-combine terms of that stage), ghost fill, reconstruction +
 * HLLE + flux divergence (an increment the next recovery adds to its stage vector); twice; final recovery.  The
 * other schemes: the same kernels stage by stage (Eq. 32); the first 3-/4-stage step allocates 28 more fields. */
int rgrmhd_step(rgrmhd_t h, double dt, int scheme);

/* The same SSP2(2,2,2) step in three parts, for blocks with a RGRMHD_BC_EXTERNAL direction.  rgrmhd_step_begin
 * enqueues the recovery of stage 1 and its ghost fill; each rgrmhd_step_continue enqueues the flux divergence of the
 * current stage and, after the first one, the recovery + ghost fill of stage 2 (*more = 1: one more exchange and one
 * more continue are due; *more = 0: the step is complete).  Between the parts the caller moves the halo layers:
 * rgrmhd_halo_pack copies the three INTERIOR layers next to `side` (0 = lower, 1 = upper) of direction `dir`, over the
 * full padded extent of the other two directions, of the 14 stage primitives and the 3 conduction-current fields into
 * dev_buf[field][layer][plane] (rgrmhd_halo_doubles doubles, DEVICE memory); rgrmhd_halo_unpack writes such a buffer
 * into the three GHOST layers of that side.  All on the handle's stream, no synchronisation.  Every other call that
 * reads or replaces the state returns RGRMHD_E_STATE while a split step is in flight. */
int rgrmhd_step_begin(rgrmhd_t h, double dt, int scheme);
int rgrmhd_step_continue(rgrmhd_t h, int* more);
int rgrmhd_halo_doubles(rgrmhd_t h, int dir, long long* host_out);
int rgrmhd_halo_pack(rgrmhd_t h, int dir, int side, double* dev_buf);
int rgrmhd_halo_unpack(rgrmhd_t h, int dir, int side, const double* dev_buf);

/* rgrmhd_step enqueues everything of its step except the final recovery P^{n+1} = recovery(U^{n+1}) (Eq. 37,
 * PAPER.md:209, 242).  That launch is deferred: the next rgrmhd_step runs it inside its first recovery kernel
 * (same arithmetic, the new state goes from one solve to the next in registers), and every entry point that reads
 * or replaces the state or the statistics (get_*, set_*, reset_stats, this call) enqueues it first.  rgrmhd_flush
 * enqueues it explicitly, e.g. before the end of a timed region; it does not synchronise and is a no-op when nothing
 * is pending.  With and without deferral the same expressions are evaluated; the two compilations may contract
 * products differently, so results agree to round-off (each call sequence on its own is deterministic). */
int rgrmhd_flush(rgrmhd_t h);

/* max over interior cells and active directions of (alpha sqrt(gamma^kk) + |beta^k|)/dx^k
 * (Eq. 30); dt = CFL / that.  With wave_speed_mode MHD_INSIDE a cell with rho > wave_rho_switch contributes
 * max(|lambda-|, |lambda+|)/dx^k of its own state instead (needs set_prims; a per-step reduction).  Synchronises;
 * in mode LIGHT the value depends on the metric only, so calls after the first one per set_metric return the cached
 * result of that reduction without a launch. */
int rgrmhd_max_speed(rgrmhd_t h, double* host_out);

/* The same reduction for callers that may not allocate (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): STATELESS -- no handle, rgrmhd_create allocates -- and with its scratch memory
 * in a fixed __device__ array of the library (65,792 bytes per GPU that loads the library, held until exit).  Calls
 * no cudaMalloc, cudaFree or allocating library routine; enqueues one 256-byte cudaMemsetAsync and one kernel on
 * `stream` (a cudaStream_t; NULL = the legacy default stream) of `device` and returns without synchronising.
 *   n, dx            HOST arrays: interior cells and spacings; ghost width 3 in every direction with n > 1 (the
 *                    field layout at the top of this file)
 *   metric_dev       HOST array of 10 DEVICE pointers: alpha, beta^x y z, gamma_xx xy xz yy yz zz (padded fields)
 *   prims_dev        HOST array of 14 DEVICE pointers (padded fields; rho, p, v^i, B^i are read); used in mode
 *                    RGRMHD_WAVE_MHD_INSIDE only, may be NULL in mode RGRMHD_WAVE_LIGHT
 *   max_speed_dev    DEVICE pointer to one double: the result, written by the kernel (valid once the stream has
 *                    reached that point; nothing is retained)
 * Unlike the other entry points every field pointer must be a device pointer on `device`: nothing is copied.
 * Limit: n[0]*n[1]*n[2] <= RGRMHD_STATIC_MAX_CELLS (= 256^3: one partial maximum per 2048 cells, 8192 slots);
 * beyond it the call returns RGRMHD_E_TOO_LARGE and touches nothing.  Otherwise RGRMHD_E_INVALID (null pointer,
 * n < 1, dx <= 0, unknown mode, Gamma <= 1 in mode MHD_INSIDE, device outside 0..63) or RGRMHD_E_CUDA.
 * Every call on a GPU shares the ONE scratch array, which keeps the last call's contents (the call clears the part
 * that has to start at zero): calls whose kernels can overlap on the GPU -- different streams, different host
 * threads, two captured graphs run concurrently -- RACE; calls on one stream are ordered and safe.  The first call
 * per device looks up the array's device address (cudaGetSymbolAddress; this may load the library's device code):
 * make it once outside a capture.  Result: the same per-cell arithmetic as rgrmhd_max_speed and an exact maximum,
 * so the two agree. */
#define RGRMHD_STATIC_MAX_CELLS 16777216LL
int rgrmhd_max_speed_static(const int n[3], const double dx[3], const double* const metric_dev[10],
                            const double* const prims_dev[14], double gamma_eos, int wave_speed_mode,
                            double wave_rho_switch, int device, void* stream, double* max_speed_dev);

/* Current primitives (ghost zones filled by the boundary rule) / conserved variables
 * D,Sx,Sy,Sz,tau,calE(3),calB(3),Psi,Phi,calQ (interior valid; ghosts unspecified). */
int rgrmhd_get_prims(rgrmhd_t h, double* const prims[14]);
int rgrmhd_get_cons(rgrmhd_t h, double* const cons[14]);

int rgrmhd_get_stats(rgrmhd_t h, rgrmhd_stats* host_out);   /* synchronises */
int rgrmhd_reset_stats(rgrmhd_t h);

/* Which flux-divergence kernel rgrmhd_step uses: 0 (default) = the TMA-staged tiled kernel (stencils
 * staged in shared memory by bulk tensor copies, each cell reconstructed once per direction, every face
 * solved once, face states and fluxes exchanged on chip; needs three active directions and an even row
 * pitch, otherwise falls back to 2); 1 = the simple one-thread-per-cell kernel that recomputes its six
 * faces from global memory (the in-library cross-check; also used for block shapes with an inactive
 * direction); 2 = the pencil-tiled kernel that reads its stencils straight from global memory.  All
 * implement the same arithmetic and agree to rounding. */
int rgrmhd_set_rhs_variant(rgrmhd_t h, int variant);
/* The variant the last rgrmhd_step actually launched (before any step: the one the next step would launch), which
 * differs from the requested one when the block shape forces a fallback. */
int rgrmhd_get_rhs_variant(rgrmhd_t h, int* host_out);

/* Kernel launches enqueued by this handle since create (bench.py's "gpu_launches"). */
int rgrmhd_launch_count(rgrmhd_t h, long long* host_out);

/* Per-kernel device timing (bench.py's roofline object).  While enabled, rgrmhd_step brackets every
 * kernel it launches with CUDA events on the handle's stream; rgrmhd_get_timing synchronises, adds the
 * elapsed milliseconds and launch counts since the last call into ms[k] / launches[k] (OVERWRITING
 * them) for the kernel classes below, and forgets the events. */
enum { RGRMHD_K_C2P = 0, RGRMHD_K_GHOST = 1, RGRMHD_K_RHS = 2, RGRMHD_K_COUNT = 3 };
int rgrmhd_set_timing(rgrmhd_t h, int enable);
int rgrmhd_get_timing(rgrmhd_t h, double ms[RGRMHD_K_COUNT], long long launches[RGRMHD_K_COUNT]);

/* Measurement aid for the FP64 roofline denominator: runs a register-resident
 * DFMA kernel (8 independent chains per thread, every SM full) on `device` and writes the best of
 * `repeats` timings as TFLOP/s (FMA = 2 flops) to *tflops_out.  Synchronises the device. */
int rgrmhd_measure_fp64_peak(int device, int repeats, double* tflops_out);

const char* rgrmhd_strerror(int code);
const char* rgrmhd_last_cuda_error(rgrmhd_t h);

#ifdef __cplusplus
}
#endif
#endif /* RGRMHD_H */
