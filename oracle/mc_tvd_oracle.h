/*
 * oracle/mc_tvd_oracle.h -- CPU ORACLE. TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, single-threaded C99/fp64 restatement of the operator-split
 * MacCormack-TVD step of arXiv 2411.10372 (Sec. 3.1,
 * Eqs. 27-39), the CFL time step and the Nusselt/Reynolds diagnostics
 * (Eqs. 22-26).  It follows the paper's algorithm step by
 * step, in the paper's order and notation: whole-array passes, no blocking,
 * no fusion, no reordering.  Where the paper is silent or garbled it takes
 * the readings listed in DESIGN.md ("Readings of the paper", R1..R22).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may call this.  It shares no code, header, table or
 * helper with the CUDA path (paper_2411_10372_b200/csrc, include/mc_tvd.h).
 *
 * Parity pins (tests/test_oracle_*.py): uniform state, conservation, Sod tube
 * vs exact Riemann solution, 2nd-order convergence, mirror identity, viscous
 * shear-wave decay, thermal diffusion, viscous heating pattern, acoustic
 * attenuation, hydrostatic conduction state, closed-form diagnostics,
 * axis-permutation identities, stationary contact (Eqs. 34-39 in closed form),
 * one-operator Taylor expansion with gravity (S^P of Eq. 32), compact viscous
 * stencil rate (R7), operator sequence of Eq. 30; the non-uniform z grid (R19:
 * uniform heights give the uniform scheme, mass to round-off, second-order
 * hydrostatic drift / viscous decay / mixed stress derivative, exact plate
 * gradients for a quadratic, dt rule); the flow statistics (R21: second-order
 * convergence to the symbolically differentiated Eqs. 40-43, histogram bins;
 * R22: the correlation of Eq. 49 in closed form, C = cos(phase), its numerator
 * against Nu_conv of Eq. 22, bound, scale invariance, sign).
 * Parity unpinned: R11 (TVD flux dropped on plate-adjacent interfaces) and the
 * interface weight of R20 (TVD term on the non-uniform grid): the paper is
 * silent on both and no mathematical criterion decides; each has a test that
 * records its closed form -- see DESIGN.md.
 *
 * Field layout (all calls): nf = 4 (2-D: rho, rho*u_x, rho*u_z, E) or
 * nf = 5 (3-D: rho, rho*u_x, rho*u_y, rho*u_z, E) arrays of N = nx*ny*nz
 * doubles each, one after the other (SoA); node (i,j,k) at (k*ny + j)*nx + i.
 */
#ifndef MC_TVD_ORACLE_H
#define MC_TVD_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct {
    int ndim;            /* 2 or 3 */
    int nx, ny, nz;      /* ny = 1 in 2-D; nz counts both wall nodes */
    double lx, ly, lz;   /* box size; 4,4,1 for the paper's aspect ratio 4 */
    const double *z_nodes; /* NULL: uniform z.  Else nz strictly increasing node heights, plates at the first and
                              last (bc_z = 0 only): the paper's non-uniform z grid, readings R19-R20 */
} orc_grid;

typedef struct {
    double gamma, Pr, Ra, eps, D;  /* PAPER.md:153-167 Eqs. 9-12; :189-193 Eqs. 16-18 */
    double cfl, fixed_dt;          /* fixed_dt > 0 overrides the CFL rule */
    double T_bot, T_top;           /* plate temperatures; paper: 1 and 1-eps-D */
    double lambda_coef;            /* dilatation coefficient in tau_ij; -2/3 Stokes, +2/3 = Eq. 18 as printed */
    double g_override, mu_override, K_override; /* < 0: derive from the paper's numbers; >= 0: use this value */
    int bc_z;                      /* 0 = walls (paper), 1 = periodic in z (test problems only) */
    int tvd_form;                  /* 0 = Eq. 34 as printed, 1 = Davis/Yee sum of two G's */
    int dir_mode;                  /* 0 = backward predictor always (paper), 1 = alternate per half step */
    int tvd_off;                   /* 1 = drop the TVD term T (tests only) */
    int co_mode;                   /* local Courant number of Eq. 39 (PAPER.md:307 does not define it; R5):
                                      0 = (|u_alpha| + c_s) tau / dx_alpha, 1 = |u_alpha| tau / dx_alpha */
} orc_params;

typedef struct {
    double time, dt; long long step;
    double nu_bottom, nu_top, nu_bar;    /* Eqs. 23-24 */
    double nu_bulk, nu_conv, nu_K;       /* Eq. 22 */
    double re, u_rms;                    /* Eq. 26 */
    double mass, mom_x, mom_y, mom_z, energy; /* trapezoid-weighted volume totals */
    double max_mach, min_rho, min_T;
} orc_diag;

/* One 1-D operator L_alpha(tau) (Eqs. 31-39): alpha = 0,1,2 for x,y,z;
 * dir = +1 backward predictor / forward corrector, -1 the mirror pair.
 * X_in and X_out are nf*N doubles and must not alias.  Returns 0, or -1 on bad arguments. */
int orc_sweep(const orc_grid *g, const orc_params *p, const double *X_in, double *X_out,
              int alpha, double tau, int dir);

/* max over nodes and directions of (|u_alpha| + c_s)/dx_alpha (R12).  NaN if any
 * rho or T is non-positive or non-finite. */
double orc_max_speed(const orc_grid *g, const orc_params *p, const double *X);

/* Time step the CFL rule gives for state X: fixed_dt if > 0, else cfl / orc_max_speed. */
double orc_dt(const orc_grid *g, const orc_params *p, const double *X);

/* n_steps full steps of Eq. 30 in place.  dt_in (may be NULL): prescribed dt per step, overrides
 * the rule; dt_out (may be NULL): receives the dt used by each step; *time (may be NULL) is advanced. */
int orc_step(const orc_grid *g, const orc_params *p, double *X, int n_steps,
             const double *dt_in, double *dt_out, double *time);

/* Instantaneous diagnostics (Eqs. 22-26) and horizontal-mean profiles (nz doubles each, may be NULL). */
int orc_diagnostics(const orc_grid *g, const orc_params *p, const double *X, orc_diag *out,
                    double *T_prof, double *rho_prof, double *p_prof);

/* Time averages of the diagnostics (twin of mc_tvd_step_stats / mc_tvd_stats_read; the paper averages Nu and Re
 * over 50 time units of the steady state): n_steps steps of Eq. 30; after every `every`-th
 * step the instantaneous diagnostics f_k of the state at time t_k enter with the weight w_k = t_k - t_{k-1} (time
 * since the previous sample, or since the start for the first one); <f>_t = sum w_k f_k / sum w_k.  X is advanced
 * in place.  dt_in as in orc_step.  Profiles: nz doubles each, may be NULL. */
typedef struct {
    double t_begin, t_end, weight; long long samples;
    double nu_bottom, nu_top, nu_bar, nu_bulk, nu_conv, nu_K, re, u_rms;
    double nu_bar_sq, re_sq;                 /* <Nu_bar^2>_t, <Re^2>_t */
} orc_stats;
int orc_step_stats(const orc_grid *g, const orc_params *p, double *X, int n_steps, int every,
                   const double *dt_in, orc_stats *out, double *T_prof, double *rho_prof, double *p_prof);

/* Flow statistics of Sec. 5-6, instantaneous: volume averages (means and root-mean-squares) of the z-momentum balance
 * terms of Eqs. 40-43 over the interior nodes, the largest local Mach number and ratio
 * r = K_e / I_e, and the histogram of r over all nodes in ORC_HIST_BINS quarter-octave bins from 2^-32
 * to 1 (bin = 4 (floor(log2 r) + 32) + top two mantissa bits, clamped; r = 0 in bin 0).  hist_r may be NULL.
 * Reading R21 (the paper does not say how it differences them): see the comment in the .c file. */
#define ORC_HIST_BINS 128
typedef struct {
    double Fn_mean, Fp_mean, Fb_mean, Fv_mean;
    double Fn_rms, Fp_rms, Fb_rms, Fv_rms;
    double FbFp_mean;                        /* <F_b> - <F_p> */
    double max_mach, max_r;
    double volume;                           /* the volume the averages run over (interior cells) */
    /* Eq. 49: C = <rho u_z T_sa> / sqrt(<(rho u_z)^2> <T_sa^2>), the normalised correlation of the
     * vertical mass flux and the superadiabatic temperature T_sa = T - T_A(z) (Eq. 19), and its three volume averages --
     * <.>_V over the whole layer with the weights of Eq. 22's Nu_conv (orc_diagnostics), so that
     * nu_conv = sqrt(Ra Pr) / eps * flux_mean. */
    double corr_C, flux_mean, rhouz_sq_mean, Tsa_sq_mean;
} orc_forces;
int orc_flow_stats(const orc_grid *g, const orc_params *p, const double *X, orc_forces *out, long long *hist_r);

/* Derived coefficients, in this order: R, c_v, g, mu, K, lambda, dx, dy, dz (9 doubles). */
int orc_coefficients(const orc_grid *g, const orc_params *p, double *out9);

#ifdef __cplusplus
}
#endif
#endif
