/*
 * oracle/mc_tvd_oracle.c -- CPU ORACLE. TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 * See mc_tvd_oracle.h for scope, layout and the list of parity pins.
 *
 * Every function cites the passage of /root/reference/PAPER.md it restates
 * (arXiv 2411.10372) or the DESIGN.md reading (R1..R18) it takes where the
 * paper is silent.  Plain C99, fp64, single thread, whole-array passes in the
 * paper's order; build with -O2 -ffp-contract=off (no FMA contraction).
 *
 * Internally a 2-D problem is the 3-D one with ny = 1 and rho*u_y = 0: every
 * y-difference is then an exact zero, so the 4-field result is bit-identical
 * to carrying five fields (tests/test_oracle_pins.py::test_2d_is_3d_with_ny1).
 */
#include "mc_tvd_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>

enum { Q_RHO = 0, Q_MX = 1, Q_MY = 2, Q_MZ = 3, Q_E = 4 };   /* X of Eq. 27 */
enum { W_UX = 0, W_UY = 1, W_UZ = 2, W_T = 3, W_P = 4 };     /* primitive variables */

typedef struct {
    int ndim, nx, ny, nz, nf;
    size_t N;
    double d[3];                 /* dx, dy, dz */
    const double *z;             /* NULL: uniform z; else the nz node heights z_k (R19) */
    double gamma, R, cv, icv, g, mu, K, lam;
    double Tw[2];                /* T at the bottom (k = 0) and top (k = nz-1) plates */
    int walls;                   /* 1: no-slip isothermal plates at k = 0, nz-1; 0: periodic in z */
    int tvd_form, tvd_off, dir_mode, co_mode;
    double cfl, fixed_dt;
} ctx;

/* Coefficients from the paper's dimensionless numbers (DESIGN.md table "Parameters -> coefficients"):
 * p = R rho T with R = (gamma-1)/(gamma eps D)            Eq. 16
 * internal energy rho c_v T with c_v = 1/(gamma eps D)    Eq. 17
 * gravity g = 1/eps                                        Eq. 14
 * mu = sqrt(Pr/Ra)                                         Eq. 18
 * K = 1/(eps D sqrt(Ra Pr))                                Eq. 15
 * Grid (R17): x_i = i lx/nx, y_j = j ly/ny periodic; z_k = k lz/(nz-1) with nodes on the plates
 * (z_k = k lz/nz when z is periodic). */
static int ctx_init(ctx *c, const orc_grid *g, const orc_params *p)
{
    if (!g || !p) return -1;
    if (g->ndim != 2 && g->ndim != 3) return -1;
    if (g->nx < 1 || g->ny < 1 || g->nz < 1) return -1;
    if (g->ndim == 2 && g->ny != 1) return -1;
    c->ndim = g->ndim; c->nx = g->nx; c->ny = g->ny; c->nz = g->nz;
    c->nf = (g->ndim == 2) ? 4 : 5;
    c->N = (size_t)g->nx * (size_t)g->ny * (size_t)g->nz;
    c->walls = (p->bc_z == 0);
    c->d[0] = g->lx / g->nx;
    c->d[1] = (g->ndim == 3) ? g->ly / g->ny : 1.0;
    c->d[2] = c->walls ? g->lz / (g->nz - 1) : g->lz / g->nz;
    c->z = g->z_nodes;
    if (c->z) {                                      /* R19: plates at the first and last node, strictly increasing */
        if (!c->walls || g->nz < 5) return -1;
        for (int k = 0; k + 1 < g->nz; ++k) if (!(c->z[k + 1] > c->z[k])) return -1;
    }
    c->gamma = p->gamma;
    c->icv = p->gamma * p->eps * p->D;               /* gamma eps D: T = icv*(E/rho - u^2/2 - z/eps), Eq. 17 */
    c->cv = 1.0 / c->icv;
    c->R = (p->gamma - 1.0) / c->icv;
    c->g = (p->g_override >= 0.0) ? p->g_override : 1.0 / p->eps;
    c->mu = (p->mu_override >= 0.0) ? p->mu_override : sqrt(p->Pr / p->Ra);
    c->K = (p->K_override >= 0.0) ? p->K_override : 1.0 / (p->eps * p->D * sqrt(p->Ra * p->Pr));
    c->lam = p->lambda_coef;
    c->Tw[0] = p->T_bot; c->Tw[1] = p->T_top;
    c->tvd_form = p->tvd_form; c->tvd_off = p->tvd_off; c->dir_mode = p->dir_mode; c->co_mode = p->co_mode;
    c->cfl = p->cfl; c->fixed_dt = p->fixed_dt;
    return 0;
}

static size_t at(const ctx *c, int i, int j, int k)
{
    return ((size_t)k * (size_t)c->ny + (size_t)j) * (size_t)c->nx + (size_t)i;
}

/* Node reached from (i,j,k) by `off` steps along `axis`: periodic wrap in x and y ("periodic
 * boundary condition for the vertical sideways walls") and in z when z is periodic;
 * -1 if the step leaves the box through a plate. */
static long nb(const ctx *c, int i, int j, int k, int axis, int off)
{
    if (axis == 0) { i = ((i + off) % c->nx + c->nx) % c->nx; }
    else if (axis == 1) { j = ((j + off) % c->ny + c->ny) % c->ny; }
    else {
        k += off;
        if (c->walls) { if (k < 0 || k >= c->nz) return -1; }
        else k = (k % c->nz + c->nz) % c->nz;
    }
    return (long)at(c, i, j, k);
}

static double z_of(const ctx *c, int k) { return c->z ? c->z[k] : (double)k * c->d[2]; }

/* Non-uniform z grid ("non-uniform tangent-hyperbolic grid in the z-direction"; the paper
 * gives no formulas for it: reading R19).  The scheme is written in the computational
 * coordinate zeta = k with the metric taken from the node heights themselves:
 *   h_{k+1/2} = z_{k+1} - z_k                         spacing across a face (inner one-sided differences);
 *   dzc_k = (z_{k+1} - z_{k-1})/2, half of the adjacent spacing at a plate node (the height of the cell
 *           a node owns: outer MacCormack differences, central differences, Co, trapezoid weights);
 * so that sum_k dzc_k X_k telescopes exactly as on the uniform grid.  Both reduce to dz when z_k = k dz. */
static double hface(const ctx *c, int k) { return c->z ? c->z[k + 1] - c->z[k] : c->d[2]; }
static double dzc(const ctx *c, int k)
{
    if (!c->z) return c->d[2];
    if (k == 0) return 0.5 * (c->z[1] - c->z[0]);
    if (k == c->nz - 1) return 0.5 * (c->z[k] - c->z[k - 1]);
    return 0.5 * (c->z[k + 1] - c->z[k - 1]);
}

/* Primitive variables from X (Eqs. 16-17):
 * u = (rho u)/rho;  T = gamma eps D (E/rho - u^2/2 - z/eps);  p = (gamma-1)/(gamma eps D) rho T. */
static void primitives(const ctx *c, double *const q[5], double *w[5])
{
    for (int k = 0; k < c->nz; ++k)
        for (int j = 0; j < c->ny; ++j)
            for (int i = 0; i < c->nx; ++i) {
                size_t n = at(c, i, j, k);
                double inv = 1.0 / q[Q_RHO][n];
                double ux = q[Q_MX][n] * inv, uy = q[Q_MY][n] * inv, uz = q[Q_MZ][n] * inv;
                double ke = 0.5 * (ux * ux + uy * uy + uz * uz);
                double T = (q[Q_E][n] * inv - ke - c->g * z_of(c, k)) * c->icv;
                w[W_UX][n] = ux; w[W_UY][n] = uy; w[W_UZ][n] = uz;
                w[W_T][n] = T;
                w[W_P][n] = c->R * q[Q_RHO][n] * T;
            }
}

/* Finite difference of a node array along `axis`: mode 0 = 2nd-order central, +1 = forward,
 * -1 = backward one-sided (first order).  NaN when a needed neighbour lies outside a plate
 * (such values are never used; a NaN that leaks into a result fails every test). */
static double deriv(const ctx *c, const double *f, int i, int j, int k, int axis, int mode)
{
    long n0 = (long)at(c, i, j, k);
    long np = nb(c, i, j, k, axis, +1), nm = nb(c, i, j, k, axis, -1);
    if (axis == 2 && c->z) {                         /* R19: divide by the distance between the nodes differenced */
        if (mode == 0) { if (np < 0 || nm < 0) return NAN; return (f[np] - f[nm]) / (c->z[k + 1] - c->z[k - 1]); }
        if (mode > 0)  { if (np < 0) return NAN; return (f[np] - f[n0]) / hface(c, k); }
        if (nm < 0) return NAN;
        return (f[n0] - f[nm]) / hface(c, k - 1);
    }
    if (mode == 0) { if (np < 0 || nm < 0) return NAN; return (f[np] - f[nm]) / (2.0 * c->d[axis]); }
    if (mode > 0)  { if (np < 0) return NAN; return (f[np] - f[n0]) / c->d[axis]; }
    if (nm < 0) return NAN;
    return (f[n0] - f[nm]) / c->d[axis];
}

/* Flux F_alpha at one node (Eq. 28, with the pressure in the rho*u_alpha row as
 * Eq. 14 has it, R2) and the stress tensor of Eq. 18:
 *   tau_{i alpha} = mu (d_alpha u_i + d_i u_alpha + lambda delta_{i alpha} d_m u_m).
 * Inner derivatives (R7): along alpha the one-sided difference of sign s (the caller passes the
 * sign opposite to the stage's outer difference); across alpha the central difference. */
static void flux_node(const ctx *c, int a, int s, double *const q[5], double *const w[5],
                      int i, int j, int k, double F[5])
{
    double G[3][3];                               /* G[ax][b] = d u_b / d x_ax */
    for (int ax = 0; ax < 3; ++ax)
        for (int b = 0; b < 3; ++b)
            G[ax][b] = deriv(c, w[b], i, j, k, ax, ax == a ? s : 0);
    double dT = deriv(c, w[W_T], i, j, k, a, s);
    double div = G[0][0] + G[1][1] + G[2][2];
    double tau[3];
    for (int b = 0; b < 3; ++b)
        tau[b] = c->mu * (G[a][b] + G[b][a] + (b == a ? c->lam * div : 0.0));
    size_t n = at(c, i, j, k);
    double ua = w[a][n], p = w[W_P][n];
    F[Q_RHO] = q[Q_MX + a][n];
    for (int b = 0; b < 3; ++b)
        F[Q_MX + b] = q[Q_MX + b][n] * ua + (b == a ? p : 0.0) - tau[b];
    F[Q_E] = ua * (q[Q_E][n] + p) - c->K * dT
             - (w[W_UX][n] * tau[0] + w[W_UY][n] * tau[1] + w[W_UZ][n] * tau[2]);
}

static int is_wall_row(const ctx *c, int k) { return c->walls && (k == 0 || k == c->nz - 1); }

/* Flux at every node where the sweep uses it.  x- and y-sweeps leave plate rows untouched (R10),
 * so no flux is formed there.  In a z-sweep a plate node whose one-sided neighbour is missing
 * keeps only its mass flux rho*u_z (all the wall closure needs); the other rows are NaN. */
static void flux_field(const ctx *c, int a, int s, double *const q[5], double *const w[5], double *F[5])
{
    for (int k = 0; k < c->nz; ++k)
        for (int j = 0; j < c->ny; ++j)
            for (int i = 0; i < c->nx; ++i) {
                size_t n = at(c, i, j, k);
                double Fn[5];
                if (a != 2 && is_wall_row(c, k)) {
                    for (int f = 0; f < 5; ++f) Fn[f] = NAN;
                } else {
                    flux_node(c, a, s, q, w, i, j, k, Fn);
                    if (a == 2 && c->walls && nb(c, i, j, k, 2, s) < 0) {
                        Fn[Q_RHO] = q[Q_MZ][n];
                        for (int f = 1; f < 5; ++f) Fn[f] = NAN;
                    }
                }
                for (int f = 0; f < 5; ++f) F[f][n] = Fn[f];
            }
}

/* Plate node (i,j,kw) in a z-sweep: no-slip (rho u = 0) and isothermal (T = T_w) conditions
 * fix every unknown except rho, which follows the conservative
 * half-cell closure (R10): the plate node owns a cell of height dz/2 whose outer face carries the
 * plate's own mass flux.  `o` is the stage's outer difference (-1 backward, +1 forward). */
static void wall_node(const ctx *c, double *const X[5], double *const Fl[5], double *Xs[5],
                      int i, int j, int kw, int o, double tau)
{
    size_t n = at(c, i, j, kw);
    double rho = X[Q_RHO][n];
    if (kw == 0 && o > 0) {
        size_t n1 = at(c, i, j, 1);
        rho = rho - (c->z ? tau / dzc(c, kw) : 2.0 * tau / c->d[2]) * (Fl[Q_RHO][n1] - Fl[Q_RHO][n]);
    } else if (kw == c->nz - 1 && o < 0) {
        size_t n1 = at(c, i, j, c->nz - 2);
        rho = rho - (c->z ? tau / dzc(c, kw) : 2.0 * tau / c->d[2]) * (Fl[Q_RHO][n] - Fl[Q_RHO][n1]);
    }
    double Tw = c->Tw[kw == 0 ? 0 : 1];
    Xs[Q_RHO][n] = rho;
    Xs[Q_MX][n] = 0.0; Xs[Q_MY][n] = 0.0; Xs[Q_MZ][n] = 0.0;
    Xs[Q_E][n] = rho * (c->cv * Tw + c->g * z_of(c, kw));     /* Eq. 17 with u = 0, T = T_w */
}

/* One MacCormack stage (Eq. 31 when o = -1, Eq. 32 when o = +1; R1: the
 * corrector differences the flux of the predicted state at both nodes):
 *   Xs_k = X_k - (tau/dx_alpha)(Fl_k - Fl_{k-1}) + tau S_k        (o = -1, backward)
 *   Xs_k = X_k - (tau/dx_alpha)(Fl_{k+1} - Fl_k) + tau S_k        (o = +1, forward)
 * S = (0,0,0,-g rho,0) in the z-sweep only (f_3 = -rho g), evaluated on `Ssrc`. */
static void stage(const ctx *c, int a, int o, double tau, double *const X[5], double *const Fl[5],
                  double *const Ssrc[5], double *Xs[5])
{
    double cdt = tau / c->d[a];
    for (int k = 0; k < c->nz; ++k)
        for (int j = 0; j < c->ny; ++j)
            for (int i = 0; i < c->nx; ++i) {
                size_t n = at(c, i, j, k);
                if (a == 2 && c->z) cdt = tau / dzc(c, k);       /* R19: the cell height of node k */
                if (is_wall_row(c, k)) {
                    if (a == 2) wall_node(c, X, Fl, Xs, i, j, k, o, tau);
                    else for (int f = 0; f < 5; ++f) Xs[f][n] = X[f][n];
                    continue;
                }
                long hi = (o > 0) ? nb(c, i, j, k, a, +1) : (long)n;
                long lo = (o > 0) ? (long)n : nb(c, i, j, k, a, -1);
                for (int f = 0; f < 5; ++f)
                    Xs[f][n] = X[f][n] - cdt * (Fl[f][hi] - Fl[f][lo]);
                if (a == 2) Xs[Q_MZ][n] = Xs[Q_MZ][n] + tau * (-c->g * Ssrc[Q_RHO][n]);
            }
}

static double phi_minmod(double x) { return fmax(0.0, fmin(2.0 * x, 1.0)); }

/* TVD term (Eqs. 34-39), all from the sweep input X, along alpha:
 *   dX_{k+1/2} = X_{k+1} - X_k                                        Eqs. 35-36
 *   r+_k = (dX_{k-1/2}, dX_{k+1/2}) / (dX_{k+1/2}, dX_{k+1/2}),
 *   r-_k = (dX_{k-1/2}, dX_{k+1/2}) / (dX_{k-1/2}, dX_{k-1/2})        Eq. 37 (dot product over the fields)
 *   G(x) = 0.5 C (1 - phi(x)), phi(x) = max(0, min(2x, 1))            Eq. 38
 *   C = Co(1-Co) if Co <= 0.5 else 0.25                               Eq. 39
 *   T_k = Dh_{k+1/2} - Dh_{k-1/2}                                     Eq. 34
 * with Dh_{k+1/2} = G(r+_k + r-_{k+1}) dX_{k+1/2} (tvd_form 0, as printed; C = mean of the two
 * nodes' C, R6) or [G_k(r+_k) + G_{k+1}(r-_{k+1})] dX_{k+1/2} (tvd_form 1, Davis/Yee, R4).
 * Co_k = (|u_alpha| + c_s)_k tau/dx_alpha (R5); r := 1 when its denominator is 0 (R15);
 * Dh := 0 on the two plate-adjacent interfaces of a z-sweep (R11).  Dh_{k+1/2} is stored at node k. */
static void tvd_interface_flux(const ctx *c, int a, double tau, double *const X[5], double *const w[5],
                               double *Dh[5])
{
    double *Cn = (double *)malloc(c->N * sizeof(double));
    for (int k = 0; k < c->nz; ++k)
        for (int j = 0; j < c->ny; ++j)
            for (int i = 0; i < c->nx; ++i) {
                size_t n = at(c, i, j, k);
                double cs = sqrt(c->gamma * c->R * w[W_T][n]);
                double speed = c->co_mode ? fabs(w[a][n]) : fabs(w[a][n]) + cs;      /* R5: the two readings of "local Courant number" */
                double Co = speed * tau / ((a == 2) ? dzc(c, k) : c->d[a]);
                Cn[n] = (Co <= 0.5) ? Co * (1.0 - Co) : 0.25;
            }
    for (int k = 0; k < c->nz; ++k)
        for (int j = 0; j < c->ny; ++j)
            for (int i = 0; i < c->nx; ++i) {
                size_t n = at(c, i, j, k);
                long nm = nb(c, i, j, k, a, -1), np = nb(c, i, j, k, a, +1), npp = nb(c, i, j, k, a, +2);
                int zero = (a != 2 && is_wall_row(c, k)) || nm < 0 || np < 0 || npp < 0;
                if (zero) { for (int f = 0; f < 5; ++f) Dh[f][n] = 0.0; continue; }
                double dm[5], d0[5], dp[5], b0 = 0.0, ak = 0.0, akp = 0.0;
                for (int f = 0; f < 5; ++f) {
                    dm[f] = X[f][n] - X[f][nm];
                    d0[f] = X[f][np] - X[f][n];
                    dp[f] = X[f][npp] - X[f][np];
                }
                for (int f = 0; f < 5; ++f) { b0 += d0[f] * d0[f]; ak += dm[f] * d0[f]; akp += d0[f] * dp[f]; }
                double rplus_k = (b0 == 0.0) ? 1.0 : ak / b0;      /* r+ at node k   */
                double rminus_kp = (b0 == 0.0) ? 1.0 : akp / b0;   /* r- at node k+1 */
                double coef;
                if (c->tvd_form == 0)
                    coef = 0.5 * (0.5 * (Cn[n] + Cn[np])) * (1.0 - phi_minmod(rplus_k + rminus_kp));
                else
                    coef = 0.5 * Cn[n] * (1.0 - phi_minmod(rplus_k))
                         + 0.5 * Cn[np] * (1.0 - phi_minmod(rminus_kp));
                /* R20 (non-uniform z only): in the computational coordinate the dissipation acts on dzc_k X_k, so the
                 * interface flux carries the face spacing h_{k+1/2} and sweep5 divides the difference by dzc_k; the sum
                 * of dzc_k T_k over a column then telescopes (conservation) and a uniform grid gives Eq. 34 back. */
                double hw = (a == 2 && c->z) ? hface(c, k) : 1.0;
                for (int f = 0; f < 5; ++f) Dh[f][n] = hw * (coef * d0[f]);
            }
    free(Cn);
}

static double *arr(size_t n) { return (double *)calloc(n, sizeof(double)); }

/* L_alpha(tau) on five internal fields: predictor, boundary values, corrector, TVD term, average
 * (Eqs. 31-39 in the order of PAPER.md:273-309; dir = -1 swaps the two one-sided differences, R9). */
static void sweep5(const ctx *c, int a, double tau, int dir, double *const X[5], double *Xo[5])
{
    double *w[5], *F[5], *XP[5], *XC[5], *Dh[5];
    for (int f = 0; f < 5; ++f) {
        w[f] = arr(c->N); F[f] = arr(c->N); XP[f] = arr(c->N); XC[f] = arr(c->N); Dh[f] = arr(c->N);
    }
    /* predictor, Eq. 31: outer difference backward (dir=+1), inner derivatives forward */
    primitives(c, X, w);
    flux_field(c, a, +dir, X, w, F);
    stage(c, a, -dir, tau, X, F, X, XP);
    /* TVD term from X^n while its primitives are at hand */
    if (!c->tvd_off) tvd_interface_flux(c, a, tau, X, w, Dh);
    /* corrector, Eq. 32: flux and source of the predicted state, opposite differences */
    primitives(c, XP, w);
    flux_field(c, a, -dir, XP, w, F);
    stage(c, a, +dir, tau, X, F, XP, XC);
    /* Eq. 33: X = (X^P + X^C)/2 + T, then the plate values again */
    for (int k = 0; k < c->nz; ++k)
        for (int j = 0; j < c->ny; ++j)
            for (int i = 0; i < c->nx; ++i) {
                size_t n = at(c, i, j, k);
                if (is_wall_row(c, k)) {
                    if (a != 2) { for (int f = 0; f < 5; ++f) Xo[f][n] = X[f][n]; continue; }
                    double rho = 0.5 * (XP[Q_RHO][n] + XC[Q_RHO][n]);
                    double Tw = c->Tw[k == 0 ? 0 : 1];
                    Xo[Q_RHO][n] = rho;
                    Xo[Q_MX][n] = 0.0; Xo[Q_MY][n] = 0.0; Xo[Q_MZ][n] = 0.0;
                    Xo[Q_E][n] = rho * (c->cv * Tw + c->g * z_of(c, k));
                    continue;
                }
                long nm = nb(c, i, j, k, a, -1);
                for (int f = 0; f < 5; ++f) {
                    double T = Dh[f][n] - Dh[f][nm];               /* Eq. 34 */
                    if (a == 2 && c->z) T = T / dzc(c, k);         /* R20 */
                    Xo[f][n] = 0.5 * (XP[f][n] + XC[f][n]) + T;    /* Eq. 33 */
                }
            }
    for (int f = 0; f < 5; ++f) { free(w[f]); free(F[f]); free(XP[f]); free(XC[f]); free(Dh[f]); }
}

/* Map the caller's nf-field SoA block onto five internal field pointers (2-D: rho u_y = zeros). */
static void map_fields(const ctx *c, double *X, double *zeros, double *q[5])
{
    if (c->ndim == 3) { for (int f = 0; f < 5; ++f) q[f] = X + (size_t)f * c->N; }
    else { q[Q_RHO] = X; q[Q_MX] = X + c->N; q[Q_MY] = zeros; q[Q_MZ] = X + 2 * c->N; q[Q_E] = X + 3 * c->N; }
}

int orc_sweep(const orc_grid *g, const orc_params *p, const double *X_in, double *X_out,
              int alpha, double tau, int dir)
{
    ctx c;
    if (ctx_init(&c, g, p) || alpha < 0 || alpha > 2 || (dir != 1 && dir != -1)) return -1;
    if (c.ndim == 2 && alpha == 1) return -1;
    if (c.walls && c.nz < 5) return -1;
    double *zin = arr(c.N), *zout = arr(c.N), *qi[5], *qo[5];
    map_fields(&c, (double *)X_in, zin, qi);
    map_fields(&c, X_out, zout, qo);
    sweep5(&c, alpha, tau, dir, qi, qo);
    free(zin); free(zout);
    return 0;
}

/* R12: s = max over nodes and directions of (|u_alpha| + c_s)/dx_alpha, c_s = sqrt(gamma R T). */
double orc_max_speed(const orc_grid *g, const orc_params *p, const double *X)
{
    ctx c;
    if (ctx_init(&c, g, p)) return NAN;
    double *zeros = arr(c.N), *q[5];
    map_fields(&c, (double *)X, zeros, q);
    double s = 0.0;
    int bad = 0;
    for (int k = 0; k < c.nz; ++k)
        for (int j = 0; j < c.ny; ++j)
            for (int i = 0; i < c.nx; ++i) {
                size_t n = at(&c, i, j, k);
                double rho = q[Q_RHO][n];
                double inv = 1.0 / rho;
                double u[3] = { q[Q_MX][n] * inv, q[Q_MY][n] * inv, q[Q_MZ][n] * inv };
                double ke = 0.5 * (u[0] * u[0] + u[1] * u[1] + u[2] * u[2]);
                double T = (q[Q_E][n] * inv - ke - c.g * z_of(&c, k)) * c.icv;
                if (!(rho > 0.0) || !(T > 0.0) || !isfinite(rho) || !isfinite(T)) { bad = 1; continue; }
                double cs = sqrt(c.gamma * c.R * T);
                for (int a = 0; a < 3; ++a) {
                    if (c.ndim == 2 && a == 1) continue;
                    /* z: the height of the node's cell (R19); a plate node, whose cell is a half cell, takes the
                     * full adjacent spacing, as on the uniform grid */
                    double da = c.d[a];
                    if (a == 2 && c.z) da = (k == 0 || k == c.nz - 1) ? 2.0 * dzc(&c, k) : dzc(&c, k);
                    double v = (fabs(u[a]) + cs) / da;
                    if (!isfinite(v)) bad = 1;
                    if (v > s) s = v;
                }
            }
    free(zeros);
    return bad ? NAN : s;
}

double orc_dt(const orc_grid *g, const orc_params *p, const double *X)
{
    if (p->fixed_dt > 0.0) return p->fixed_dt;
    return p->cfl / orc_max_speed(g, p, X);
}

/* Eq. 30: X^(n+1) = Lx Ly Lz Lx Ly Lz X^(n), each with dt/2, operators acting
 * right to left; the y operator is absent in 2-D.  dir_mode 1 (R9): dir = +1 in the first triple,
 * -1 in the second. */
int orc_step(const orc_grid *g, const orc_params *p, double *X, int n_steps,
             const double *dt_in, double *dt_out, double *time)
{
    ctx c;
    if (ctx_init(&c, g, p) || n_steps < 0) return -1;
    if (c.walls && c.nz < 5) return -1;
    double *za = arr(c.N), *zb = arr(c.N), *Y = arr((size_t)c.nf * c.N), *qa[5], *qb[5];
    map_fields(&c, X, za, qa);
    map_fields(&c, Y, zb, qb);
    for (int s = 0; s < n_steps; ++s) {
        double dt = dt_in ? dt_in[s] : orc_dt(g, p, X);
        if (!(dt > 0.0) || !isfinite(dt)) { free(za); free(zb); free(Y); return -4; }
        double tau = 0.5 * dt;
        double **src = qa, **dst = qb;
        for (int half = 0; half < 2; ++half) {
            int dir = (half == 1 && c.dir_mode == 1) ? -1 : +1;
            for (int a = 2; a >= 0; --a) {            /* L_z, then L_y, then L_x */
                if (c.ndim == 2 && a == 1) continue;
                sweep5(&c, a, tau, dir, src, dst);
                double **t = src; src = dst; dst = t;
            }
        }
        /* 4 (2-D) or 6 (3-D) sweeps: an even count, so the result is back in X */
        if (dt_out) dt_out[s] = dt;
        if (time) *time += dt;
    }
    free(za); free(zb); free(Y);
    return 0;
}

/* Diagnostics, instantaneous (the paper also averages in time):
 *   <f>_A(k): plane mean; <f>_V: trapezoid in z (R16);  T_A = 1 - D z (Eq. 19); T_sa = T - T_A
 *   Nu_conv = sqrt(Ra Pr)/eps <rho u_z T_sa>_V,  Nu_K = D sqrt(Ra Pr)/2 <rho u_z u^2>_V,
 *   Nu_bulk = 1 + Nu_conv + Nu_K                                       Eq. 22
 *   Nu_{z=0,1} = -(1/eps) d<T_sa>_A/dz with 2nd-order one-sided differences at the plates
 *                                                                      Eq. 23
 *   Nu_bar = (Nu_0 + Nu_1)/2                                           Eq. 24
 *   Re = sqrt(Ra/Pr) sqrt(<u^2>_V)                                     Eq. 26
 * Sums: serial along each row, rows into planes, planes into the trapezoid rule. */
int orc_diagnostics(const orc_grid *g, const orc_params *p, const double *X, orc_diag *out,
                    double *T_prof, double *rho_prof, double *p_prof)
{
    ctx c;
    if (ctx_init(&c, g, p) || !out) return -1;
    double *zeros = arr(c.N), *q[5];
    map_fields(&c, (double *)X, zeros, q);
    memset(out, 0, sizeof(*out));
    int nz = c.nz;
    double *sT = arr(nz), *sTsa = arr(nz);
    double vol_w = 0.0, v_conv = 0.0, v_K = 0.0, v_u2 = 0.0;
    double tot[5] = { 0, 0, 0, 0, 0 };
    double max_mach = 0.0, min_rho = INFINITY, min_T = INFINITY;
    double nplane = (double)c.nx * (double)c.ny;
    for (int k = 0; k < nz; ++k) {
        double z = z_of(&c, k), TA = 1.0 - p->D * z;
        double pT = 0, prho = 0, pp = 0, pconv = 0, pK = 0, pu2 = 0, pq[5] = { 0, 0, 0, 0, 0 };
        for (int j = 0; j < c.ny; ++j) {
            double rT = 0, rrho = 0, rp = 0, rconv = 0, rK = 0, ru2 = 0, rq[5] = { 0, 0, 0, 0, 0 };
            for (int i = 0; i < c.nx; ++i) {
                size_t n = at(&c, i, j, k);
                double rho = q[Q_RHO][n], inv = 1.0 / rho;
                double ux = q[Q_MX][n] * inv, uy = q[Q_MY][n] * inv, uz = q[Q_MZ][n] * inv;
                double u2 = ux * ux + uy * uy + uz * uz;
                double T = (q[Q_E][n] * inv - 0.5 * u2 - c.g * z) * c.icv;
                double pr = c.R * rho * T;
                rT += T; rrho += rho; rp += pr;
                rconv += rho * uz * (T - TA);
                rK += rho * uz * u2;
                ru2 += u2;
                for (int f = 0; f < 5; ++f) rq[f] += q[f][n];
                double mach = sqrt(u2) / sqrt(c.gamma * c.R * T);
                if (mach > max_mach) max_mach = mach;
                if (rho < min_rho) min_rho = rho;
                if (T < min_T) min_T = T;
            }
            pT += rT; prho += rrho; pp += rp; pconv += rconv; pK += rK; pu2 += ru2;
            for (int f = 0; f < 5; ++f) pq[f] += rq[f];
        }
        double wk = c.z ? dzc(&c, k) : c.d[2] * ((c.walls && (k == 0 || k == nz - 1)) ? 0.5 : 1.0);
        sT[k] = pT / nplane;
        sTsa[k] = sT[k] - TA;
        if (T_prof) T_prof[k] = sT[k];
        if (rho_prof) rho_prof[k] = prho / nplane;
        if (p_prof) p_prof[k] = pp / nplane;
        vol_w += wk;
        v_conv += wk * (pconv / nplane);
        v_K += wk * (pK / nplane);
        v_u2 += wk * (pu2 / nplane);
        for (int f = 0; f < 5; ++f) tot[f] += wk * c.d[0] * c.d[1] * pq[f];
    }
    double sRaPr = sqrt(p->Ra * p->Pr);
    out->nu_conv = sRaPr / p->eps * (v_conv / vol_w);
    out->nu_K = p->D * sRaPr / 2.0 * (v_K / vol_w);
    out->nu_bulk = 1.0 + out->nu_conv + out->nu_K;
    out->u_rms = sqrt(v_u2 / vol_w);
    out->re = sqrt(p->Ra / p->Pr) * out->u_rms;
    if (nz >= 3) {
        double dz = c.d[2];
        double g0 = (-3.0 * sTsa[0] + 4.0 * sTsa[1] - sTsa[2]) / (2.0 * dz);
        double g1 = (3.0 * sTsa[nz - 1] - 4.0 * sTsa[nz - 2] + sTsa[nz - 3]) / (2.0 * dz);
        if (c.z) {
            /* second-order one-sided differences through the plate node and its two neighbours at distances h1 < h2
             * (the derivative of the quadratic through the three points; (-3, 4, -1)/(2 dz) when h2 = 2 h1) */
            double h1 = c.z[1] - c.z[0], h2 = c.z[2] - c.z[0];
            double b = h2 / (h1 * (h2 - h1)), cc = -h1 / (h2 * (h2 - h1));
            g0 = -(b + cc) * sTsa[0] + b * sTsa[1] + cc * sTsa[2];
            h1 = c.z[nz - 1] - c.z[nz - 2]; h2 = c.z[nz - 1] - c.z[nz - 3];
            b = h2 / (h1 * (h2 - h1)); cc = -h1 / (h2 * (h2 - h1));
            g1 = (b + cc) * sTsa[nz - 1] - b * sTsa[nz - 2] - cc * sTsa[nz - 3];
        }
        out->nu_bottom = -g0 / p->eps;
        out->nu_top = -g1 / p->eps;
        out->nu_bar = 0.5 * (out->nu_bottom + out->nu_top);
    }
    out->mass = tot[Q_RHO]; out->mom_x = tot[Q_MX]; out->mom_y = tot[Q_MY]; out->mom_z = tot[Q_MZ];
    out->energy = tot[Q_E];
    out->max_mach = max_mach; out->min_rho = min_rho; out->min_T = min_T;
    out->dt = orc_dt(g, p, X);
    free(sT); free(sTsa); free(zeros);
    return 0;
}

/* Time averages (PAPER.md:218 "<.>_{V,t}", :222 "<.>_{A,t}", :236, :355): step, sample, weight with the time
 * elapsed since the previous sample, divide by the total weight at the end.  A composition of orc_step and
 * orc_diagnostics; no new arithmetic of the scheme. */
int orc_step_stats(const orc_grid *g, const orc_params *p, double *X, int n_steps, int every,
                   const double *dt_in, orc_stats *out, double *T_prof, double *rho_prof, double *p_prof)
{
    if (!g || !p || !X || !out || n_steps < 0 || every < 1) return -1;
    int nz = g->nz;
    double *aT = arr(nz), *ar = arr(nz), *ap = arr(nz), *iT = arr(nz), *ir = arr(nz), *ip = arr(nz);
    double sum[10] = { 0 }, weight = 0.0, t = 0.0, t_last = 0.0;
    long long samples = 0;
    for (int s = 0; s < n_steps; ++s) {
        int rc = orc_step(g, p, X, 1, dt_in ? dt_in + s : NULL, NULL, &t);
        if (rc) return rc;
        if ((s + 1) % every) continue;
        orc_diag d;
        orc_diagnostics(g, p, X, &d, iT, ir, ip);
        double w = t - t_last;
        double f[10] = { d.nu_bottom, d.nu_top, d.nu_bar, d.nu_bulk, d.nu_conv, d.nu_K, d.re, d.u_rms,
                         d.nu_bar * d.nu_bar, d.re * d.re };
        for (int i = 0; i < 10; ++i) sum[i] += w * f[i];
        for (int k = 0; k < nz; ++k) { aT[k] += w * iT[k]; ar[k] += w * ir[k]; ap[k] += w * ip[k]; }
        weight += w; t_last = t; samples += 1;
    }
    memset(out, 0, sizeof(*out));
    out->t_begin = 0.0; out->t_end = t_last; out->weight = weight; out->samples = samples;
    if (samples > 0) {
        double *o = &out->nu_bottom;
        for (int i = 0; i < 10; ++i) o[i] = sum[i] / weight;
        for (int k = 0; k < nz; ++k) {
            if (T_prof) T_prof[k] = aT[k] / weight;
            if (rho_prof) rho_prof[k] = ar[k] / weight;
            if (p_prof) p_prof[k] = ap[k] / weight;
        }
    }
    free(aT); free(ar); free(ap); free(iT); free(ir); free(ip);
    return 0;
}

/* Flow statistics of Sec. 5-6 (instantaneous; the paper averages them over the steady state):
 *  - the z-momentum balance terms (Eqs. 40-43)
 *        F_n = rho (u . grad) u_z,  F_p = -d_z p,  F_b = rho g,  F_v = d_i tau_iz
 *    with tau_ij of Eq. 18 (dilatation coefficient lambda, R3), so for constant mu
 *        F_v = mu [ lap u_z + (1 + lambda) d_z (div u) ];
 *    "we compute the volume averages of the above four terms, along with <F_b> - <F_p>";
 *  - the ratio r = K_e / I_e = (rho u^2/2)/(rho C_v T) "at every grid point" and its distribution (PAPER.md:395,
 *    Fig. 5); the local Mach number, of which the paper quotes the maximum, is the same number up
 *    to a constant: Mach^2 = u^2/(gamma R T) = 2 r / (gamma (gamma - 1)).
 * The paper does not say how it differences these post-processing quantities (reading R21): second-order central
 * differences on the node's 3x3x3 neighbourhood (first derivatives over the distance between the two neighbours,
 * second derivatives and mixed derivatives compact), evaluated at the INTERIOR nodes k = 1 .. nz-2 (all nodes when z
 * is periodic) and averaged with the cell heights of R16 / R19; the means and the root-mean-squares are both given
 * (the signed mean of F_n and F_v nearly cancels).  Histogram: r > 0 falls into bin 4 (floor(log2 r) + 32) +
 * (top two mantissa bits), clamped to [0, 127] -- quarter-octave bins from 2^-32 to 1, read off the bit pattern of
 * the double so that both implementations take the decision on the same number; r = 0 goes to bin 0. */
static int hist_bin(double r)
{
    if (!(r > 0.0)) return 0;
    unsigned long long bits;
    memcpy(&bits, &r, sizeof(bits));
    long b = (long)(bits >> 50) - 4L * (1023 - 32);      /* 11 exponent bits and 2 mantissa bits */
    return b < 0 ? 0 : (b > ORC_HIST_BINS - 1 ? ORC_HIST_BINS - 1 : (int)b);
}

int orc_flow_stats(const orc_grid *g, const orc_params *p, const double *X, orc_forces *out, long long *hist_r)
{
    ctx c;
    if (ctx_init(&c, g, p) || !out) return -1;
    if (c.nx < 3 || c.nz < 3 || (c.ndim == 3 && c.ny < 3)) return -1;
    double *zeros = arr(c.N), *q[5], *w[5];
    map_fields(&c, (double *)X, zeros, q);
    for (int f = 0; f < 5; ++f) w[f] = arr(c.N);
    primitives(&c, q, w);
    memset(out, 0, sizeof(*out));
    if (hist_r) memset(hist_r, 0, ORC_HIST_BINS * sizeof(long long));
    double sum[4] = { 0, 0, 0, 0 }, sq[4] = { 0, 0, 0, 0 }, vol = 0.0, max_r = 0.0;
    double cor[3] = { 0, 0, 0 }, vol_all = 0.0;      /* Eq. 49: <rho u_z T_sa>_V, <(rho u_z)^2>_V, <T_sa^2>_V */
    double dx2 = c.d[0] * c.d[0], dy2 = c.d[1] * c.d[1];
    int k0 = c.walls ? 1 : 0, k1 = c.walls ? c.nz - 1 : c.nz;
    for (int k = 0; k < c.nz; ++k) {
        double ps[4] = { 0, 0, 0, 0 }, pq[4] = { 0, 0, 0, 0 }, pc[3] = { 0, 0, 0 };
        double TA = 1.0 - p->D * z_of(&c, k);        /* Eq. 19 */
        for (int j = 0; j < c.ny; ++j)
            for (int i = 0; i < c.nx; ++i) {
                size_t n = at(&c, i, j, k);
                double u2 = w[W_UX][n] * w[W_UX][n] + w[W_UY][n] * w[W_UY][n] + w[W_UZ][n] * w[W_UZ][n];
                double r = (0.5 * u2) / (c.cv * w[W_T][n]);
                if (r > max_r) max_r = r;
                if (hist_r) hist_r[hist_bin(r)] += 1;
                /* the two factors of the correlation C of Eq. 49, at every node: <.>_V of Eq. 22 */
                double mz = q[Q_RHO][n] * w[W_UZ][n], Tsa = w[W_T][n] - TA;
                pc[0] += mz * Tsa; pc[1] += mz * mz; pc[2] += Tsa * Tsa;
                if (k < k0 || k >= k1) continue;
                /* spacings along z around level k (face spacings below and above) */
                double hm = c.z ? hface(&c, k - 1) : c.d[2], hp = c.z ? hface(&c, k) : c.d[2];
                size_t xm = (size_t)nb(&c, i, j, k, 0, -1), xp = (size_t)nb(&c, i, j, k, 0, +1);
                size_t ym = (size_t)nb(&c, i, j, k, 1, -1), yp = (size_t)nb(&c, i, j, k, 1, +1);
                size_t zm = (size_t)nb(&c, i, j, k, 2, -1), zp = (size_t)nb(&c, i, j, k, 2, +1);
                const double *uz = w[W_UZ];
                double Fn = q[Q_RHO][n] * (w[W_UX][n] * deriv(&c, uz, i, j, k, 0, 0)
                                           + w[W_UY][n] * deriv(&c, uz, i, j, k, 1, 0)
                                           + w[W_UZ][n] * deriv(&c, uz, i, j, k, 2, 0));
                double Fp = -deriv(&c, w[W_P], i, j, k, 2, 0);
                double Fb = q[Q_RHO][n] * c.g;
                double lap = (uz[xp] - 2.0 * uz[n] + uz[xm]) / dx2;
                if (c.ndim == 3) lap += (uz[yp] - 2.0 * uz[n] + uz[ym]) / dy2;
                double dzz = 2.0 * ((uz[zp] - uz[n]) / hp - (uz[n] - uz[zm]) / hm) / (hp + hm);
                /* mixed derivatives d_z d_x u_x, d_z d_y u_y: central difference along z of the central differences */
                int kp = (k + 1) % c.nz, km = (k - 1 + c.nz) % c.nz;    /* the levels of zp and zm (never wrapped between plates) */
                double dzx = (deriv(&c, w[W_UX], i, j, kp, 0, 0) - deriv(&c, w[W_UX], i, j, km, 0, 0)) / (hp + hm);
                double dzy = (c.ndim == 3)
                           ? (deriv(&c, w[W_UY], i, j, kp, 1, 0) - deriv(&c, w[W_UY], i, j, km, 1, 0)) / (hp + hm) : 0.0;
                double Fv = c.mu * (lap + dzz + (1.0 + c.lam) * (dzx + dzy + dzz));
                double F[4] = { Fn, Fp, Fb, Fv };
                for (int t = 0; t < 4; ++t) { ps[t] += F[t]; pq[t] += F[t] * F[t]; }
            }
        {   /* <.>_V as in orc_diagnostics: cell heights, half cells at the plates (R16 / R19) */
            double wa = c.z ? dzc(&c, k) : c.d[2] * ((c.walls && (k == 0 || k == c.nz - 1)) ? 0.5 : 1.0);
            vol_all += wa;
            for (int t = 0; t < 3; ++t) cor[t] += wa * (pc[t] / ((double)c.nx * (double)c.ny));
        }
        if (k < k0 || k >= k1) continue;
        double wk = dzc(&c, k) / ((double)c.nx * (double)c.ny);
        vol += dzc(&c, k);
        for (int t = 0; t < 4; ++t) { sum[t] += wk * ps[t]; sq[t] += wk * pq[t]; }
    }
    double *m = &out->Fn_mean, *r = &out->Fn_rms;
    for (int t = 0; t < 4; ++t) { m[t] = sum[t] / vol; r[t] = sqrt(sq[t] / vol); }
    out->FbFp_mean = out->Fb_mean - out->Fp_mean;
    out->max_r = max_r;
    out->max_mach = sqrt(2.0 * max_r / (c.gamma * (c.gamma - 1.0)));
    out->volume = vol;
    out->flux_mean = cor[0] / vol_all;
    out->rhouz_sq_mean = cor[1] / vol_all;
    out->Tsa_sq_mean = cor[2] / vol_all;
    out->corr_C = out->flux_mean / sqrt(out->rhouz_sq_mean * out->Tsa_sq_mean);     /* Eq. 49; 0/0 = NaN for a fluid at rest */
    for (int f = 0; f < 5; ++f) free(w[f]);
    free(zeros);
    return 0;
}

int orc_coefficients(const orc_grid *g, const orc_params *p, double *o)
{
    ctx c;
    if (ctx_init(&c, g, p) || !o) return -1;
    o[0] = c.R; o[1] = c.cv; o[2] = c.g; o[3] = c.mu; o[4] = c.K; o[5] = c.lam;
    o[6] = c.d[0]; o[7] = c.d[1]; o[8] = c.d[2];
    return 0;
}
