/*
 * include/mc_tvd.h -- C ABI of libmc_tvd.so, the B200 (sm_100a) MacCormack-TVD step of
 * arXiv 2411.10372 ("Compressible turbulent convection at very high Rayleigh numbers").
 *
 * The library advances the conserved state X = (rho, rho u_x, [rho u_y,] rho u_z, E) of the fully
 * compressible Navier-Stokes + energy equations with gravity (Eqs. 13-18; vector
 * form PAPER.md:255-263, Eqs. 27-28) by the operator-split MacCormack predictor-corrector scheme with
 * a TVD correction (Eqs. 29-39), chooses the time step by an acoustic CFL rule
 * (reading R12; the paper is silent) and evaluates the Nusselt / Reynolds diagnostics
 * (Eqs. 22-26).  Around that path: the paper's non-uniform z grid (mc_tvd_grid.z_nodes,
 * PAPER.md:249), device-resident time averages (mc_tvd_stats_*), the flow statistics of
 * Sec. 5-6 (mc_tvd_flow_stats: Eqs. 40-43, the ratio K_e / I_e), and hooks for running one box as slabs over
 * several GPUs (mc_tvd_slab_*).  Every step of all of it runs in CUDA kernels; there is no CPU fallback.  All
 * arithmetic is fp64.
 *
 * Conventions
 *   - Plain C: POD structs, raw pointers, sizes.  No torch / C++ types.  "d_" = DEVICE pointer,
 *     "h_" / unmarked = HOST pointer.
 *   - Field layout (device): nf = 4 (2-D: rho, rho u_x, rho u_z, E) or 5 (3-D: rho, rho u_x,
 *     rho u_y, rho u_z, E) arrays of N = nx*ny*nz doubles, one after the other (SoA); node (i,j,k)
 *     at (k*ny + j)*nx + i; x fastest.  x_i = i lx/nx and y_j = j ly/ny are periodic; z_k = k lz/(nz-1)
 *     with k = 0 and k = nz-1 ON the plates (z_k = k lz/nz when bc_z = 1), or the caller's node heights.
 *   - Ownership: the caller owns every device buffer (d_fields, d_workspace) and the stream; the
 *     library owns only the host-side handle.  d_fields and d_workspace must stay valid and must
 *     not be touched by the caller between a call and the next stream synchronisation.
 *   - Errors: every int-returning call returns MC_TVD_OK (0) or a negative mc_tvd_status; it never
 *     throws, aborts or prints.  mc_tvd_last_error() returns a thread-local message.
 *   - Threading: a handle is not thread-safe; distinct handles are independent.
 */
#ifndef MC_TVD_H
#define MC_TVD_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    MC_TVD_OK = 0,
    MC_TVD_EINVAL = -1,       /* bad argument (NULL, size, unsupported switch value) */
    MC_TVD_ECUDA = -2,        /* a CUDA runtime call or kernel launch failed */
    MC_TVD_ENOMEM = -3,       /* workspace too small / host allocation failed */
    MC_TVD_ENONFINITE = -4,   /* state holds a non-finite value or non-positive rho or T */
    MC_TVD_EUNSUPPORTED = -5  /* valid request this build does not implement (e.g. 2^32 or more nodes per field) */
} mc_tvd_status;

/* The box (Sec. 2; aspect ratio 4). */
typedef struct {
    int ndim;                 /* 2 or 3 */
    int nx, ny, nz;           /* ny = 1 in 2-D; nx, ny = distinct periodic nodes; nz counts both plate nodes */
    double lx, ly, lz;        /* box size: 4, 4, 1 for the paper's runs */
    const double *z_nodes;    /* NULL = uniform z, z_k = k lz / (nz - 1).  Else HOST array of nz strictly increasing node
                                 heights, plates at the first and last (bc_z = 0 only): the paper's "non-uniform
                                 tangent-hyperbolic grid in the z-direction".  The paper prints no formula
                                 for it; R19 / R20: outer differences, central differences, Co and trapezoid weights
                                 use the height of the cell a node owns, (z_{k+1} - z_{k-1})/2 (half the adjacent spacing
                                 at a plate), inner one-sided differences the spacing across the face, the TVD interface
                                 flux carries the face spacing.  Read during mc_tvd_init only; any node spacing is
                                 accepted, so no stretching parameter appears in this interface.  MC_TVD_EINVAL if not
                                 increasing or bc_z != 0. */
} mc_tvd_grid;

/* The paper's dimensionless numbers and the switches of DESIGN.md's readings. */
typedef struct {
    double gamma, Pr, Ra, eps, D;   /* PAPER.md:153-167 Eqs. 9-12; closures PAPER.md:189-193 Eqs. 16-18 */
    double cfl, fixed_dt;           /* dt = cfl / max (|u_a| + c_s)/dx_a (R12); fixed_dt > 0 overrides */
    double T_bot, T_top;            /* plate temperatures; paper: 1 and 1 - eps - D */
    double lambda_coef;             /* dilatation coefficient in tau_ij: -2/3 (Stokes) or +2/3 (Eq. 18 as printed) */
    double g_override, mu_override, K_override; /* < 0: derive from the paper's numbers; >= 0: use as is */
    int bc_z;                       /* 0 = no-slip isothermal plates (paper); 1 = periodic z (test problems) */
    int tvd_form;                   /* 0 = Eq. 34 as printed; 1 = Davis/Yee sum of two G's (R4) */
    int dir_mode;                   /* 0 = backward predictor always (paper); 1 = alternate per half step (R9) */
    int tvd_off;                    /* 1 = drop the TVD term (tests) */
    int co_mode;                    /* the "local Courant number" of Eq. 39, which PAPER.md:307 does not define (R5):
                                       0 = (|u_alpha| + c_s) tau / dx_alpha, 1 = |u_alpha| tau / dx_alpha */
} mc_tvd_params;

/* Result of mc_tvd_diagnostics (host POD).  Instantaneous values; Eqs. 22-26. */
typedef struct {
    double time, dt; long long step;       /* simulated time, dt the NEXT step will use, steps taken */
    double nu_bottom, nu_top, nu_bar;      /* Eqs. 23-24: -(1/eps) d<T_sa>_A/dz at the plates, and their mean */
    double nu_bulk, nu_conv, nu_K;         /* Eq. 22 */
    double re, u_rms;                      /* Eq. 26 */
    double mass, mom_x, mom_y, mom_z, energy; /* trapezoid-weighted volume totals of X */
    double max_mach, min_rho, min_T;
} mc_tvd_diag;

/* Running time averages <.>_t of the diagnostics (the paper reports Nu, Nu_conv, Nu_K of Eq. 22 as <.>_{V,t},
 * Nu_{z=0,1} of Eq. 23 from <T_sa>_{A,t}, Re of Eq. 26 as <sqrt(<u^2>_V)>_t, and averages them over 50 time units
 * of the steady state).  Sample k is the instantaneous diagnostic of the state at
 * time t_k weighted with w_k = t_k - t_{k-1} (the time since the previous sample, or since the reset for the first
 * one): <f>_t = sum_k w_k f_k / sum_k w_k.  The plate Nusselt numbers are LINEAR in the plane means of T, so their
 * averages equal Eq. 23 applied to <T_sa>_{A,t}. */
typedef struct {
    double t_begin, t_end;                 /* averaged time span: reset time, time of the last sample */
    double weight; long long samples;      /* sum of the weights (= t_end - t_begin) and number of samples */
    double nu_bottom, nu_top, nu_bar;      /* Eqs. 23-24, time averaged */
    double nu_bulk, nu_conv, nu_K;         /* Eq. 22, <.>_{V,t} */
    double re, u_rms;                      /* Eq. 26 */
    double nu_bar_sq, re_sq;               /* <Nu_bar^2>_t, <Re^2>_t: the +- the paper quotes is sqrt(<f^2> - <f>^2) */
} mc_tvd_stats;

typedef struct mc_tvd_state mc_tvd_state;  /* opaque host-side handle */

/* Bytes of device workspace mc_tvd_init needs for this problem: the second (ping-pong) state
 * buffer, reduction partials and device scalars.  0 on invalid arguments. */
size_t mc_tvd_workspace_bytes(const mc_tvd_grid *grid, const mc_tvd_params *params);

/* Create a handle.  d_fields (DEVICE, nf*N doubles, 16-byte aligned) holds the initial state and
 * receives every later state; d_workspace (DEVICE, >= mc_tvd_workspace_bytes, 256-byte aligned) is
 * scratch; cuda_stream is a cudaStream_t (NULL = the legacy default stream) on which ALL work of
 * this handle is enqueued.  Enqueues the max-speed reduction of the initial state so that dt is
 * defined (R12).  Does not synchronise. */
int mc_tvd_init(const mc_tvd_grid *grid, const mc_tvd_params *params, double *d_fields,
                void *d_workspace, size_t workspace_bytes, void *cuda_stream, mc_tvd_state **out);

/* Advance n_steps steps of Eq. 30: X <- Lx Ly Lz Lx Ly Lz X, each operator with
 * dt/2 (operators act right to left; no Ly in 2-D); dt from the CFL rule on the step's input state,
 * kept on the device.  Asynchronous on the handle's stream; never synchronises.  The result is
 * always back in d_fields. */
int mc_tvd_step(mc_tvd_state *s, int n_steps);

/* One operator L_alpha(tau) (Eqs. 31-39) applied to d_fields in place (through the workspace):
 * alpha = 0,1,2 for x,y,z; dir = +1 backward predictor / forward corrector,
 * -1 the mirrored pair.  Exposed for per-operator parity tests.  Time and the step count do not advance;
 * dt is recomputed from the swept state (as mc_tvd_init does), so a following mc_tvd_step is CFL-safe. */
int mc_tvd_sweep(mc_tvd_state *s, int alpha, int dir, double tau);

/* Test hook: marching levels per thread block of later operator launches (the kernels march along one
 * axis and cut it into chunks, each repeating a short warm-up).  0 = automatic (default).
 * Results do not depend on it; the parity tests use it to start blocks in the middle of a column. */
int mc_tvd_debug_set_chunk(mc_tvd_state *s, int levels);

/* Test hook: the tiling of operator alpha's most recent launch on this handle (all 0 before the first one):
 * output nodes per thread-block tile along x (*tile_x) and along the tile's second direction (*tile_b; 1 in
 * 2-D; y for L_z and L_x, z for L_y) and marching levels per block (*chunk).  The full-size parity tests place
 * their sample windows across these boundaries. */
int mc_tvd_debug_geometry(const mc_tvd_state *s, int alpha, int *tile_x, int *tile_b, int *chunk);

/* The end-to-end call for callers whose state lives in HOST memory (pinned memory makes the copies
 * asynchronous, pageable memory works too): copies h_in (HOST, nf*N doubles, same layout) into
 * d_fields, recomputes dt from it (as mc_tvd_init does) and resets time and step count to zero, runs
 * n_steps steps, copies the result into h_out (HOST, nf*N doubles; may alias h_in) and synchronises
 * the stream.  Every arithmetic step still runs in the kernels; this call only adds the two copies. */
int mc_tvd_step_host(mc_tvd_state *s, const double *h_in, double *h_out, int n_steps);

/* dt the next step will use (host double).  Synchronises the stream.  MC_TVD_ENONFINITE if the
 * state holds a non-finite value or a non-positive rho or T. */
int mc_tvd_dt(mc_tvd_state *s, double *dt_host);

/* Diagnostics of the current state (Eqs. 22-26) into a HOST struct, and the
 * horizontal means <T>_A, <rho>_A, <p>_A into HOST arrays of nz doubles (each may be NULL).
 * Synchronises the stream. */
int mc_tvd_diagnostics(mc_tvd_state *s, mc_tvd_diag *out, double *T_prof, double *rho_prof,
                       double *p_prof);

/* Time averages.  mc_tvd_stats_reset zeroes the device-resident accumulators and starts the averaging
 * span at the current simulated time.  mc_tvd_step_stats advances n_steps steps like mc_tvd_step and, after every
 * `every`-th of them (counted since the reset), evaluates the diagnostics of Eqs. 22-26 on the device and adds them
 * to the accumulators with the weight stated at mc_tvd_stats; asynchronous, never synchronises.  mc_tvd_stats_read
 * forms the averages on the device, copies them into a HOST struct and the time-averaged horizontal means <T>_{A,t},
 * <rho>_{A,t}, <p>_{A,t} into HOST arrays of nz doubles (each may be NULL), and synchronises the stream.  With no
 * sample yet it returns MC_TVD_EINVAL. */
int mc_tvd_stats_reset(mc_tvd_state *s);
int mc_tvd_step_stats(mc_tvd_state *s, int n_steps, int every);
int mc_tvd_stats_read(mc_tvd_state *s, mc_tvd_stats *out, double *T_prof, double *rho_prof, double *p_prof);

/* Flow statistics of the paper's Sec. 5-6, one extra pass over the state:
 *   - the terms of the z-momentum balance, Eqs. 40-43: F_n = rho (u . grad) u_z, F_p = -d_z p,
 *     F_b = rho g, F_v = d_i tau_iz with tau_ij of Eq. 18, as volume means and root-mean-squares over the interior
 *     cells ("the volume averages of the above four terms, along with <F_b> - <F_p>");
 *   - r = K_e / I_e = (rho u^2 / 2) / (rho C_v T) "at every grid point": its largest value, the largest
 *     local Mach number, and its histogram over all nodes (Fig. 5) in MC_TVD_HIST_BINS quarter-octave bins from 2^-32
 *     to 1: bin = 4 (floor(log2 r) + 32) + (top two mantissa bits), clamped to [0, 127]; r = 0 in bin 0.
 *   - the normalised correlation C(Ra) of Eq. 49 between the vertical mass flux rho u_z and the
 *     superadiabatic temperature T_sa = T - (1 - D z) (Eq. 19), with its three averages; these are <.>_V over the WHOLE
 *     layer with the weights of Eq. 22 (half cells at the plates), so Nu_conv = sqrt(Ra Pr) / eps * flux_mean; the time
 *     average forms C from the time-averaged three (the paper's <.> is <.>_{V,t}).
 * The paper does not say how it differences these quantities; R21: second-order central differences on the
 * 3 x 3 x 3 neighbourhood, cell-height weights.
 * mc_tvd_flow_stats: instantaneous values of the current state into HOST memory (hist_r: MC_TVD_HIST_BINS counts, may
 * be NULL); synchronises the stream.  mc_tvd_stats_flow(enable = 1): every sample mc_tvd_step_stats takes from now on
 * also accumulates these numbers on the device (same weights as mc_tvd_stats).  mc_tvd_stats_read_flow: the time
 * averages since the last mc_tvd_stats_reset -- means as they are, the rms fields as the root of the time-averaged
 * mean square, max_mach / max_r as the time average of the instantaneous maxima ("the time average of maximum
 * turbulent Mach number"), `volume` = the simulated time averaged over -- and the histogram summed over
 * the samples; synchronises; MC_TVD_EINVAL with no sample yet. */
#define MC_TVD_HIST_BINS 128
typedef struct {
    double Fn_mean, Fp_mean, Fb_mean, Fv_mean;   /* volume averages of Eqs. 40-43 */
    double Fn_rms, Fp_rms, Fb_rms, Fv_rms;       /* square roots of the volume averages of their squares */
    double FbFp_mean;                            /* <F_b> - <F_p> */
    double max_mach, max_r;                      /* largest local Mach number and ratio r = K_e / I_e */
    double volume;                               /* the volume averaged over (interior cells) */
    double corr_C;                               /* Eq. 49: <rho u_z T_sa> / sqrt(<(rho u_z)^2> <T_sa^2>); NaN at rest */
    double flux_mean, rhouz_sq_mean, Tsa_sq_mean; /* its three averages <.>_V over the whole layer (weights of Eq. 22) */
} mc_tvd_forces;
int mc_tvd_flow_stats(mc_tvd_state *s, mc_tvd_forces *out, long long *hist_r);
int mc_tvd_stats_flow(mc_tvd_state *s, int enable);
int mc_tvd_stats_read_flow(mc_tvd_state *s, mc_tvd_forces *avg, long long *hist_r);

/* Slab decomposition: the hooks a multi-GPU driver needs to run one box as slabs along a periodic
 * horizontal direction, one handle per GPU, as the paper's multi-GPU runs do (App. A :573-577).  A
 * rank's handle is an ordinary handle on its LOCAL box: the rows it owns plus H >= 2 halo rows on either side, treated
 * as periodic (the wrap only corrupts the outermost 2 rows per operator, which are halo rows).  Every operator has
 * radius 2 across and along the slab axis, so the driver refreshes the halo rows from the neighbours after every
 * operator (paper_2411_10372_b200/slab.py does this with NCCL send/recv, or with device copies when several slabs
 * live on one GPU):
 *   mc_tvd_slab_op(s, op)       enqueue operator number op = 0 .. 2 ndim - 1 of the current step (Eq. 30 order: L_z,
 *                               [L_y,] L_x with dir +1, then again with dir -1), without the fused CFL reduction;
 *                               operators must come in order;
 *   mc_tvd_slab_pointers        device addresses the driver exchanges / all-reduces: the buffer that holds the state
 *                               right now (it alternates between d_fields and the workspace after every operator),
 *                               the bit pattern of the running maximum of (|u_a| + c_s)/dx_a, the per-plane sums
 *                               (nz x 11 doubles) and extrema (nz x 3: max Mach^2, min rho, min T) of the diagnostics;
 *   mc_tvd_slab_reduce(s)       after the last halo exchange of a step (or of the initial state): max-speed reduction
 *                               over the local box into the running maximum; the driver then all-reduces it (MAX);
 *   mc_tvd_slab_commit(s, adv)  dt from the maximum (R12); adv = 1 also advances time and the step count;
 *   mc_tvd_slab_diag_partial    per-plane sums of Eqs. 22-26 over the nodes whose index along axis (0 x, 1 y) lies in
 *                               [lo, hi) -- the owned rows; the driver all-reduces sums (SUM) and extrema (MAX, MIN);
 *   mc_tvd_slab_diag_finish     the diagnostics from the all-reduced plane sums; nplane_global = nodes per z plane of
 *                               the whole box.  Synchronises.
 * All asynchronous on the handle's stream except the last.  mc_tvd_step on such a handle would use stale halos.
 *
 * Fused halo push (3-D box between plates, even nx, uniform z; MC_TVD_EUNSUPPORTED otherwise): after
 *   mc_tvd_slab_buffers(s, &X, &Y)    the handle's two state buffers (d_fields and its copy in the workspace), and
 *   mc_tvd_slab_peers(s, lo_X, lo_Y, hi_X, hi_Y, own_lo, own_hi, halo)
 * with the same two buffers of the ranks that own the rows below (lo) and above (hi) this slab -- device addresses this
 * GPU can store to: another slab on the same GPU, or peer-mapped memory of another GPU -- every operator stores only the
 * owned rows [own_lo, own_hi) of the slab axis y and writes its first / last `halo` owned rows straight into the
 * neighbours' halo rows from inside the sweep kernel; no exchange between the launches, only a barrier across the ranks
 * (every rank must have finished operator k before any starts k + 1).  The last operator then carries the CFL
 * reduction over the owned rows, so mc_tvd_slab_reduce is not needed: all-reduce the maximum and commit.  Four NULLs
 * switch back to plain operators. */
int mc_tvd_slab_buffers(mc_tvd_state *s, double **d_fields, double **d_second);
int mc_tvd_slab_peers(mc_tvd_state *s, double *lo_fields, double *lo_second, double *hi_fields, double *hi_second,
                      int own_lo, int own_hi, int halo);
int mc_tvd_slab_op(mc_tvd_state *s, int op);
int mc_tvd_slab_reduce(mc_tvd_state *s);
int mc_tvd_slab_commit(mc_tvd_state *s, int advance);
int mc_tvd_slab_pointers(mc_tvd_state *s, double **fields_now, unsigned long long **smax_bits, double **plane_sums,
                         double **plane_ext);
int mc_tvd_slab_diag_partial(mc_tvd_state *s, int axis, int lo, int hi);
int mc_tvd_slab_diag_finish(mc_tvd_state *s, double nplane_global, mc_tvd_diag *out, double *T_prof, double *rho_prof,
                            double *p_prof);

/* The CFL reduction without a handle, a workspace or any allocation (R12; the "local Courant number" of
 * PAPER.md:304-307): for callers that cannot call cudaMalloc -- code under CUDA graph capture, serving loops,
 * harnesses that forbid it.  Enqueues on `cuda_stream` the same max-reduction kernel mc_tvd_init and the slab driver
 * use, over the state `d_fields` (DEVICE, layout as in mc_tvd_init, read only), and writes to `d_out` (DEVICE, 2 doubles,
 * caller-owned):  d_out[0] = s = max over nodes and directions of (|u_a| + c_s) / dx_a  (NaN if rho or T is not
 * positive anywhere),  d_out[1] = the dt the next step would use, fixed_dt if > 0 else cfl / s -- bit for bit the dt of a
 * handle initialised on the same state.  Asynchronous: read d_out after synchronising the stream.
 *
 * Scratch: the running maximum and, for a non-uniform z grid, the node heights and the metric tables built from them
 * on the device live in ONE fixed array inside the library, MC_TVD_NOALLOC_SCRATCH_BYTES (128.25 KiB) of device memory on
 * every GPU that loads the library, held until the process exits.  Hence the limit: nz <= MC_TVD_NOALLOC_MAX_NZ on any
 * grid (more levels: MC_TVD_EUNSUPPORTED, nothing is enqueued); nx, ny are limited as in mc_tvd_init only.
 * The call allocates nothing on the host or the device (no cudaMalloc / cudaFree / allocating library routine); its
 * first use on a device looks up the array's address (cudaGetSymbolAddress), at most 64 devices per process.
 * grid->z_nodes (HOST) is uploaded with cudaMemcpyAsync on the stream: keep it valid and unchanged until the stream has
 * passed the call (pageable memory is already staged when the call returns).  Make the first call on a device outside
 * stream capture (the address look-up may load the module).
 * All calls share the array: it is cleared at the start of every call and left cleared, but two calls whose kernels
 * OVERLAP on the GPU (different streams without ordering, several host threads) race on it and return rubbish -- order
 * them on one stream or with events.  Calls on different GPUs do not interact.  Handles (mc_tvd_init) never touch it.
 * Errors: MC_TVD_EINVAL (bad problem, NULL pointer), MC_TVD_EUNSUPPORTED (nz too large), MC_TVD_ECUDA. */
#define MC_TVD_NOALLOC_MAX_NZ 4096
#define MC_TVD_NOALLOC_SCRATCH_BYTES (256 + 4 * MC_TVD_NOALLOC_MAX_NZ * 8)
int mc_tvd_cfl_noalloc(const mc_tvd_grid *grid, const mc_tvd_params *params, const double *d_fields, double *d_out,
                       void *cuda_stream);

/* Number of kernel launches this handle has enqueued so far (for bench.py's gpu_launches). */
long long mc_tvd_launch_count(const mc_tvd_state *s);

/* Per-kernel device timing (for the roofline figure of bench.py).  enable = 1: every
 * operator launch of later mc_tvd_step / mc_tvd_step_host calls is bracketed by CUDA events on the
 * handle's stream (at most MC_TVD_MAX_TIMED launches are recorded, later ones run untimed);
 * enable = 0 stops recording.  mc_tvd_timing_read synchronises the stream, adds the recorded
 * durations into ms_sum[6] and count[6] (HOST arrays, overwritten), indexed by
 * kind = alpha + (dir < 0 ? 3 : 0) with alpha = 0,1,2 for L_x, L_y, L_z, and clears the records. */
#define MC_TVD_MAX_TIMED 4096
int mc_tvd_timing_enable(mc_tvd_state *s, int enable);
int mc_tvd_timing_read(mc_tvd_state *s, double *ms_sum, long long *count);

/* Free the handle (host memory only).  Synchronises the stream first. */
int mc_tvd_destroy(mc_tvd_state *s);

/* Thread-local message of the last failing call on this thread ("" if none). */
const char *mc_tvd_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* MC_TVD_H */
