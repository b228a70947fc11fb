// sweep_march.cuh -- kernel k_march: one operator L_alpha(tau) of Eqs. 31-39
// for a sweep axis alpha that is NOT the fastest (x) axis: the z-sweep (2-D, 3-D) and the y-sweep (3-D).
//
// Design: one thread owns one grid column along alpha and MARCHES along it,
// keeping every along-alpha neighbour (predictor flux F_{k-1}, corrector flux F^P_{k+1}, the five-node
// TVD stencil) in registers; consecutive threads own consecutive x, so every global access is a
// coalesced row segment.  Only the velocities needed by the cross derivatives inside the viscous
// flux (d_x, d_b of u, central, R7) travel through shared memory, one plane per level, double
// buffered, ONE __syncthreads per level.  A block owns a (x, b) tile with a 2-node halo ring that is
// recomputed (ring 2: primitives; ring 1: predictor) and a chunk of levels with a 4-level warm-up.
// dir = -1 (R9) is the same code marching from the other end with a negated spacing: the mirror
// identity of the scheme (tests/test_oracle_pins.py::test_mirror_identity) makes it bit-equivalent.
//
// Pipeline of iteration j (output level j):  W(j+2) -> F(j+1) -> P(j+1) | barrier | F^P(j+1) -> out(j)
#pragma once
#include "mc_common.cuh"

namespace mc {

// CA: velocity component of alpha; CB: velocity component of the tile's second direction b (-1 in 2-D).
template <int ND, int CA, int CB>
MC_KERNEL void k_march(SweepArgs A)
{
    constexpr int NF = ND + 2;
    constexpr bool HAS_B = (CB >= 0);
    constexpr bool Z_IS_ALPHA = (CA == ND - 1);      // z is the last velocity component
    MC_SHARED_DECL(double, smem);

    const int tx = threadIdx.x, Wx = blockDim.x;
    const int ty = HAS_B ? (int)threadIdx.y : 0, Wb = HAS_B ? (int)blockDim.y : 1;
    const int tile_n = Wx * Wb, tidx = ty * Wx + tx;
    double *slotU = smem;                             // [2][ND][tile_n]  velocities of X     (levels j+1, j+2)
    double *slotP = smem + 2 * ND * tile_n;           // [2][ND][tile_n]  velocities of X^P   (level j+1)

    // ---- tile geometry --------------------------------------------------------------------
    const int gx = (int)blockIdx.x * (Wx - 4) + tx - 2;
    const int ix = wrap(gx, A.nx);
    const int rx = min(tx, Wx - 1 - tx);
    int gb = 0, rb = 99, gb_raw = 0;
    bool row_exists = true, wallrow = false;
    long long col = ix;
    if (HAS_B) {
        gb = (int)blockIdx.y * (Wb - 4) + ty - 2;
        gb_raw = gb;
        rb = min(ty, Wb - 1 - ty);
        if (A.wall_b) {
            row_exists = (gb >= 0 && gb < A.n_b);
            wallrow = (gb == 0 || gb == A.n_b - 1);
            col += (long long)(row_exists ? gb : 0) * A.s_b;
        } else {
            gb = wrap(gb, A.n_b);                     // periodic b: the node's own index (z_k of Eq. 17)
            col += (long long)gb * A.s_b;
        }
    }
    const bool needP = row_exists && !wallrow && rx >= 1 && rb >= 1 && (rx >= 2 || rb >= 2);
    const bool owner = row_exists && rx >= 2 && rb >= 2 && gx < A.nx && (!HAS_B || gb_raw < A.n_b);

    // ---- sweep constants ------------------------------------------------------------------
    const double tau = A.dt_ptr ? 0.5 * (*A.dt_ptr) : A.tau_fixed;
    const double h = (A.dir > 0) ? A.d_a : -A.d_a;    // signed spacing in marching coordinates
    const double inv_h = 1.0 / h;
    const double cdt = tau / h;                       // tau / dx_alpha of Eqs. 31-32
    const double tau_over_d = tau / A.d_a;            // for Co (R5)
    const double src_c = A.src ? -A.g : 0.0;          // S = -g rho in the rho u_z row
    const int n = A.n_m;
    const int l0 = (int)blockIdx.z * A.chunk;
    const int l1 = min(n, l0 + A.chunk);

    auto exists = [&](int l) { return A.wall_m ? (l >= 0 && l < n) : true; };
    auto phys = [&](int l) { int w = wrap(l, n); return (A.dir > 0) ? w : n - 1 - w; };
    auto gz_of = [&](int l) {                         // g z_k of Eq. 17 for this thread's node at level l
        int kz = Z_IS_ALPHA ? phys(l) : gb;
        return A.g * ((double)kz * A.dz);
    };
    auto load = [&](int l, double (&X)[NF]) {
        const double *p = A.in + col + (long long)phys(l) * A.s_m;
#pragma unroll
        for (int f = 0; f < NF; ++f) X[f] = p[(long long)f * A.N];
    };
    auto publish = [&](double *slot, int parity, const double (&u)[ND]) {
#pragma unroll
        for (int c = 0; c < ND; ++c) slot[(parity * ND + c) * tile_n + tidx] = u[c];
    };
    // central cross derivatives of the velocities published in `slot` (R7)
    auto cross = [&](const double *slot, int parity, double (&dcu_a)[ND], double (&dcu_c)[ND]) {
        const double *s = slot + parity * ND * tile_n + tidx;
#pragma unroll
        for (int c = 0; c < ND; ++c) { dcu_a[c] = 0.0; dcu_c[c] = 0.0; }
        dcu_a[0] = (s[CA * tile_n + 1] - s[CA * tile_n - 1]) * A.inv2d_x;
        dcu_c[0] = (s[0 * tile_n + 1] - s[0 * tile_n - 1]) * A.inv2d_x;
        if (HAS_B) {
            constexpr int cb = HAS_B ? CB : 0;
            dcu_a[cb] = (s[CA * tile_n + Wx] - s[CA * tile_n - Wx]) * A.inv2d_b;
            dcu_c[cb] = (s[cb * tile_n + Wx] - s[cb * tile_n - Wx]) * A.inv2d_b;
        }
    };
    // plate values of a node on a plate of the marching direction: no slip,
    // T = T_w; only rho is free (R10)
    auto plate = [&](int l, double rho, double (&X)[NF]) {
        int k = phys(l);
        double Tw = (k == 0) ? A.Tw0 : A.Tw1;
        X[0] = rho;
#pragma unroll
        for (int c = 0; c < ND; ++c) X[1 + c] = 0.0;
        X[NF - 1] = rho * (A.cv * Tw + A.g * ((double)k * A.dz));
    };

    // ---- carried state ----------------------------------------------------------------------
    double Xc[NF], F0[NF], FP0[NF], H0[NF], d0[NF];
    double uP0[ND], TP0 = 0.0, a0 = 0.0, b0 = 0.0, C0 = 0.0, C1 = 0.0;
    Prim<ND> w1;
#pragma unroll
    for (int f = 0; f < NF; ++f) { Xc[f] = 0.0; F0[f] = 0.0; FP0[f] = 0.0; H0[f] = 0.0; d0[f] = 0.0; }
#pragma unroll
    for (int c = 0; c < ND; ++c) { uP0[c] = 0.0; w1.u[c] = 0.0; }
    w1.T = 1.0; w1.p = 0.0;

    for (int j = l0 - 4; j < l1; ++j) {
        const int p1 = (j + 1) & 1, p2 = (j + 2) & 1;
        const bool ex1 = exists(j + 1), ex2 = exists(j + 2);
        const bool ld1 = ex1 && (j + 1 >= l0 - 2);              // level j+1 is loaded (Xc, w1 valid)
        const bool ld2 = ex2;                                   // level j+2 is loaded this iteration
        const bool start_wall1 = A.wall_m && (j + 1 == 0);      // level j+1 is the plate the march starts on
        const bool end_wall1 = A.wall_m && (j + 1 == n - 1);    // level j+1 is the plate the march ends on

        // (1) W(j+2): load, primitives, Courant coefficient, publish velocities
        double Xn[NF];
        Prim<ND> w2;
        double C2 = 0.0;
#pragma unroll
        for (int f = 0; f < NF; ++f) Xn[f] = 0.0;
#pragma unroll
        for (int c = 0; c < ND; ++c) w2.u[c] = 0.0;
        w2.T = 1.0; w2.p = 0.0;
        if (ld2 && row_exists) {
            load(j + 2, Xn);
            w2 = primitives<ND>(Xn, gz_of(j + 2), A);
            C2 = courant_coef(w2.u[CA], w2.T, tau_over_d, A);
            publish(slotU, p2, w2.u);
        }

        // (2) TVD (Eqs. 34-39): Dh_{j+1/2} from dX_{j-1/2}, dX_{j+1/2}, dX_{j+3/2}
        double d1[NF], a1 = 0.0, b1 = 0.0, Dh[NF];
#pragma unroll
        for (int f = 0; f < NF; ++f) { d1[f] = (ld1 && ld2) ? Xn[f] - Xc[f] : 0.0; Dh[f] = 0.0; }
#pragma unroll
        for (int f = 0; f < NF; ++f) { b1 += d1[f] * d1[f]; a1 += d0[f] * d1[f]; }
        {
            bool have = (j >= l0 - 1) && exists(j - 1) && exists(j) && ex1 && ex2 && !A.tvd_off;   // R11 at plates
            if (have && owner && !wallrow) {
                double coef = tvd_coef(a0, a1, b0, C0, C1, A.tvd_form);
#pragma unroll
                for (int f = 0; f < NF; ++f) { Dh[f] = coef * d0[f]; H0[f] += Dh[f]; }
            }
        }

        // (3) F(j+1): flux of X at level j+1 (inner derivative forward in marching coordinates)
        double F1[NF], XP[NF], H1[NF];
        Prim<ND> wP1;
#pragma unroll
        for (int f = 0; f < NF; ++f) { F1[f] = 0.0; XP[f] = Xc[f]; H1[f] = Xc[f]; }
        wP1 = w1;
        const bool doF = ld1 && needP;
        if (doF) {
            if (end_wall1) {
                F1[0] = Xc[1 + CA];                   // only the mass flux is defined and needed (R10)
            } else {
                double dau[ND], daT, dcu_a[ND], dcu_c[ND];
#pragma unroll
                for (int c = 0; c < ND; ++c) dau[c] = (w2.u[c] - w1.u[c]) * inv_h;
                daT = (w2.T - w1.T) * inv_h;
                cross(slotU, p1, dcu_a, dcu_c);
                flux<ND, CA>(Xc, w1, dau, daT, dcu_a, dcu_c, A, F1);
            }
        }
        // (4) P(j+1): predictor (Eq. 31), plate values, primitives of X^P, publish
        const bool doP = doF && (j + 1 >= l0 - 1);
        if (doP) {
            if (start_wall1) {
                plate(j + 1, Xc[0], XP);                                      // rho unchanged
            } else if (end_wall1) {
                plate(j + 1, Xc[0] - 2.0 * cdt * (F1[0] - F0[0]), XP);       // half-cell closure (R10)
            } else {
#pragma unroll
                for (int f = 0; f < NF; ++f) XP[f] = Xc[f] - cdt * (F1[f] - F0[f]);
                XP[1 + CA] += tau * (src_c * Xc[0]);
            }
            wP1 = primitives<ND>(XP, gz_of(j + 1), A);
#pragma unroll
            for (int f = 0; f < NF; ++f) H1[f] = 0.5 * (XP[f] + Xc[f]) - Dh[f];
            H1[1 + CA] += 0.5 * (tau * (src_c * XP[0]));
        }
        if (ld1 && row_exists) publish(slotP, p1, wP1.u);      // plate rows of b publish u^P = u (X^P = X there)

        __syncthreads();

        // (5) F^P(j+1): flux of X^P at level j+1 (inner derivative backward in marching coordinates)
        double FP1[NF];
#pragma unroll
        for (int f = 0; f < NF; ++f) FP1[f] = 0.0;
        const bool doFP = doP && owner && (j + 1 >= l0);
        if (doFP) {
            if (start_wall1) {
                FP1[0] = XP[1 + CA];
            } else {
                double dau[ND], daT, dcu_a[ND], dcu_c[ND];
#pragma unroll
                for (int c = 0; c < ND; ++c) dau[c] = (wP1.u[c] - uP0[c]) * inv_h;
                daT = (wP1.T - TP0) * inv_h;
                cross(slotP, p1, dcu_a, dcu_c);
                flux<ND, CA>(XP, wP1, dau, daT, dcu_a, dcu_c, A, FP1);
            }
        }
        // (6) out(j): corrector (Eq. 32), average and TVD term (Eq. 33), plate values
        if (j >= l0 && owner && exists(j)) {
            double o[NF];
            if (wallrow) {
#pragma unroll
                for (int f = 0; f < NF; ++f) o[f] = H0[f];            // plate rows of b: unchanged (R10)
            } else if (A.wall_m && j == 0) {
                plate(j, H0[0] - cdt * (FP1[0] - FP0[0]), o);        // 0.5 * (2 tau/dz) * dF
            } else if (A.wall_m && j == n - 1) {
                plate(j, H0[0], o);
            } else {
#pragma unroll
                for (int f = 0; f < NF; ++f) o[f] = H0[f] - 0.5 * cdt * (FP1[f] - FP0[f]);
            }
            double *q = A.out + col + (long long)phys(j) * A.s_m;
#pragma unroll
            for (int f = 0; f < NF; ++f) q[(long long)f * A.N] = o[f];
        }
        // (7) rotate the pipeline
#pragma unroll
        for (int f = 0; f < NF; ++f) { Xc[f] = Xn[f]; F0[f] = F1[f]; FP0[f] = FP1[f]; H0[f] = H1[f]; d0[f] = d1[f]; }
#pragma unroll
        for (int c = 0; c < ND; ++c) uP0[c] = wP1.u[c];
        TP0 = wP1.T; w1 = w2; C0 = C1; C1 = C2; a0 = a1; b0 = b1;
    }
}

}  // namespace mc
