// sweep_lane.cuh -- kernel k_lane: the operator L_x(tau) of Eqs. 31-39, i.e. the
// sweep along the fastest (x) axis, in 2-D and 3-D.
//
// Design: a warp owns 32 consecutive x columns (28 outputs + a 2-node halo on
// each side), so every along-alpha neighbour -- the predictor flux F_{i-1}, the corrector flux
// F^P_{i+1}, the five-node TVD stencil -- is a warp shuffle and every global access is one coalesced
// 256-byte row segment.  The warp marches along a cross direction m (z), keeping the central cross
// derivative's neighbours (levels j-1, j+1) in registers.  In 3-D the block stacks warps along the
// other cross direction b (y); the two velocity components the b-derivatives need go through shared
// memory, double buffered, one __syncthreads per level.  dir = -1 (R9) maps lanes to x in reverse
// order with a negated spacing (still coalesced).
//
// Pipeline of iteration j (output level j):  W(j+2) -> F(j+1) -> P(j+1) -> F^P(j) -> out(j)
#pragma once
#include "mc_common.cuh"

namespace mc {

constexpr int LANE_OUT = 28;      // outputs per warp: 32 lanes minus the 2+2 halo

template <int NF>
MC_DEV void shfl_up_vec(const double (&v)[NF], double (&r)[NF])
{
#pragma unroll
    for (int f = 0; f < NF; ++f) r[f] = __shfl_up_sync(0xffffffffu, v[f], 1);
}
template <int NF>
MC_DEV void shfl_down_vec(const double (&v)[NF], double (&r)[NF])
{
#pragma unroll
    for (int f = 0; f < NF; ++f) r[f] = __shfl_down_sync(0xffffffffu, v[f], 1);
}

// CB: velocity component of the tile's second direction b (y; -1 in 2-D); CM: component of the
// marching direction m (z).  alpha is x, component 0.
template <int ND, int CB, int CM>
MC_KERNEL void k_lane(SweepArgs A)
{
    constexpr int NF = ND + 2;
    constexpr bool HAS_B = (CB >= 0);
    constexpr int CA = 0;
    MC_SHARED_DECL(double, smem);

    const int xi = threadIdx.x;                        // lane coordinate along alpha (always "dir = +1")
    const int ty = threadIdx.y, Wy = blockDim.y;
    const int tile_n = 32 * Wy, tidx = ty * 32 + xi;
    double *slotU = smem;                              // [2][2][tile_n]: (u_x, u_b) of X
    double *slotP = smem + 4 * tile_n;                 // [2][2][tile_n]: (u_x, u_b) of X^P

    // ---- tile geometry --------------------------------------------------------------------
    const int xtile = HAS_B ? (int)blockIdx.x : (int)blockIdx.x * Wy + ty;
    const int gx0 = xtile * LANE_OUT;
    const int gx = (A.dir > 0) ? gx0 - 2 + xi : gx0 + (LANE_OUT + 1) - xi;
    const int ix = wrap(gx, A.nx);
    const bool warp_on = gx0 < A.nx;
    int rb = 99, gb = 0;
    long long col = ix;
    if (HAS_B) {
        gb = (int)blockIdx.y * (Wy - 4) + ty - 2;
        rb = min(ty, Wy - 1 - ty);
        col += (long long)wrap(gb, A.n_b) * A.s_b;
    }
    const bool needP = warp_on && rb >= 1;
    const bool rowout = warp_on && rb >= 2 && (!HAS_B || gb < A.n_b);
    const bool owner = rowout && xi >= 2 && xi < 2 + LANE_OUT && gx >= 0 && gx < A.nx;

    // ---- sweep constants ------------------------------------------------------------------
    const double tau = A.dt_ptr ? 0.5 * (*A.dt_ptr) : A.tau_fixed;
    const double h = (A.dir > 0) ? A.d_a : -A.d_a;
    const double inv_h = 1.0 / h;
    const double cdt = tau / h;
    const double tau_over_d = tau / A.d_a;
    const int n = A.n_m;
    const int l0 = (int)blockIdx.z * A.chunk;
    const int l1 = min(n, l0 + A.chunk);

    auto exists = [&](int l) { return A.wall_m ? (l >= 0 && l < n) : true; };
    auto is_plate = [&](int l) { return A.wall_m && (l == 0 || l == n - 1); };
    auto load = [&](int l, double (&X)[NF]) {
        const double *p = A.in + col + (long long)wrap(l, n) * A.s_m;
#pragma unroll
        for (int f = 0; f < NF; ++f) X[f] = p[(long long)f * A.N];
    };
    auto gz_of = [&](int l) { return A.g * ((double)wrap(l, n) * A.dz); };   // m is z
    auto publish = [&](double *slot, int parity, const double (&u)[ND]) {
        if (HAS_B) {
            constexpr int cb = HAS_B ? CB : 0;
            slot[(parity * 2 + 0) * tile_n + tidx] = u[0];
            slot[(parity * 2 + 1) * tile_n + tidx] = u[cb];
        }
    };
    // central b-derivatives of (u_x, u_b) published in `slot`
    auto cross_b = [&](const double *slot, int parity, double (&dcu_a)[ND], double (&dcu_c)[ND]) {
        if (HAS_B) {
            constexpr int cb = HAS_B ? CB : 0;
            const double *s = slot + parity * 2 * tile_n + tidx;
            dcu_a[cb] = (s[32] - s[-32]) * A.inv2d_b;
            dcu_c[cb] = (s[tile_n + 32] - s[tile_n - 32]) * A.inv2d_b;
        }
    };

    // ---- carried state ----------------------------------------------------------------------
    double X0[NF], X1[NF], XP0[NF];
    Prim<ND> w1, wP0;
    double um0[2] = {0.0, 0.0}, uPm[2] = {0.0, 0.0}, C0 = 0.0, C1 = 0.0;
#pragma unroll
    for (int f = 0; f < NF; ++f) { X0[f] = 0.0; X1[f] = 0.0; XP0[f] = 0.0; }
#pragma unroll
    for (int c = 0; c < ND; ++c) { w1.u[c] = 0.0; wP0.u[c] = 0.0; }
    w1.T = 1.0; w1.p = 0.0; wP0.T = 1.0; wP0.p = 0.0;
    double smax = 0.0;

    for (int j = l0 - 4; j < l1; ++j) {
        const int p0 = j & 1, p1 = (j + 1) & 1;
        const bool ex1 = exists(j + 1), ex2 = exists(j + 2);
        const bool ld1 = ex1 && (j + 1 >= l0 - 2);

        if (HAS_B) __syncthreads();

        // (1) W(j+2)
        double X2[NF];
        Prim<ND> w2;
        double C2 = 0.0;
#pragma unroll
        for (int f = 0; f < NF; ++f) X2[f] = 0.0;
#pragma unroll
        for (int c = 0; c < ND; ++c) w2.u[c] = 0.0;
        w2.T = 1.0; w2.p = 0.0;
        if (ex2 && warp_on) {
            load(j + 2, X2);
            w2 = primitives<ND>(X2, gz_of(j + 2), A);
            C2 = courant_coef(w2.u[CA], w2.T, tau_over_d, A);
            publish(slotU, p0, w2.u);                   // parity of level j+2
        }

        // (2) F(j+1) and (3) P(j+1): Eq. 31 with the inner derivative forward along the lanes
        double XP1[NF];
        Prim<ND> wP1 = w1;
#pragma unroll
        for (int f = 0; f < NF; ++f) XP1[f] = X1[f];
        const bool doP = ld1 && needP && (j + 1 >= l0 - 1) && !is_plate(j + 1);
        if (doP) {                                       // warp-uniform
            double F1[NF], Fm[NF], dau[ND], daT, dcu_a[ND], dcu_c[ND];
#pragma unroll
            for (int c = 0; c < ND; ++c) {
                dau[c] = (__shfl_down_sync(0xffffffffu, w1.u[c], 1) - w1.u[c]) * inv_h;
                dcu_a[c] = 0.0; dcu_c[c] = 0.0;
            }
            daT = (__shfl_down_sync(0xffffffffu, w1.T, 1) - w1.T) * inv_h;
            dcu_a[CM] = (w2.u[CA] - um0[0]) * A.inv2d_m;
            dcu_c[CM] = (w2.u[CM] - um0[1]) * A.inv2d_m;
            cross_b(slotU, p1, dcu_a, dcu_c);
            flux<ND, CA>(X1, w1, dau, daT, dcu_a, dcu_c, A, F1);
            shfl_up_vec<NF>(F1, Fm);
#pragma unroll
            for (int f = 0; f < NF; ++f) XP1[f] = X1[f] - cdt * (F1[f] - Fm[f]);
            wP1 = primitives<ND>(XP1, gz_of(j + 1), A);
        }
        if (ld1 && warp_on) publish(slotP, p1, wP1.u);   // plate levels publish u^P = u (X^P = X there, R10)

        // (4) F^P(j), (5) corrector, TVD, out(j)
        const bool doOut = (j >= l0) && rowout && exists(j);
        if (doOut) {                                     // warp-uniform
            double o[NF];
            if (is_plate(j)) {
#pragma unroll
                for (int f = 0; f < NF; ++f) o[f] = X0[f];            // x-sweeps leave the plate rows unchanged
            } else {
                double FP0[NF], FPp[NF], dau[ND], daT, dcu_a[ND], dcu_c[ND];
#pragma unroll
                for (int c = 0; c < ND; ++c) {
                    dau[c] = (wP0.u[c] - __shfl_up_sync(0xffffffffu, wP0.u[c], 1)) * inv_h;
                    dcu_a[c] = 0.0; dcu_c[c] = 0.0;
                }
                daT = (wP0.T - __shfl_up_sync(0xffffffffu, wP0.T, 1)) * inv_h;
                dcu_a[CM] = (wP1.u[CA] - uPm[0]) * A.inv2d_m;
                dcu_c[CM] = (wP1.u[CM] - uPm[1]) * A.inv2d_m;
                cross_b(slotP, p0, dcu_a, dcu_c);
                flux<ND, CA>(XP0, wP0, dau, daT, dcu_a, dcu_c, A, FP0);
                shfl_down_vec<NF>(FP0, FPp);
                // TVD term along the lanes (Eqs. 34-39)
                double Tt[NF];
#pragma unroll
                for (int f = 0; f < NF; ++f) Tt[f] = 0.0;
                if (!A.tvd_off) {
                    double Xr[NF], d0[NF], dm[NF], Dh[NF], Dhm[NF], b0 = 0.0, a0 = 0.0;
                    shfl_down_vec<NF>(X0, Xr);
#pragma unroll
                    for (int f = 0; f < NF; ++f) { d0[f] = Xr[f] - X0[f]; b0 += d0[f] * d0[f]; }
                    shfl_up_vec<NF>(d0, dm);
#pragma unroll
                    for (int f = 0; f < NF; ++f) a0 += dm[f] * d0[f];
                    double a1 = __shfl_down_sync(0xffffffffu, a0, 1);
                    double Cr = __shfl_down_sync(0xffffffffu, C0, 1);
                    double coef = tvd_coef(a0, a1, b0, C0, Cr, A.tvd_form);
#pragma unroll
                    for (int f = 0; f < NF; ++f) Dh[f] = coef * d0[f];
                    shfl_up_vec<NF>(Dh, Dhm);
#pragma unroll
                    for (int f = 0; f < NF; ++f) Tt[f] = Dh[f] - Dhm[f];
                }
#pragma unroll
                for (int f = 0; f < NF; ++f) {
                    double XC = X0[f] - cdt * (FPp[f] - FP0[f]);     // Eq. 32 (R1)
                    o[f] = 0.5 * (XP0[f] + XC) + Tt[f];              // Eq. 33
                }
            }
            if (owner) {
                double *q = A.out + col + (long long)j * A.s_m;
#pragma unroll
                for (int f = 0; f < NF; ++f) q[(long long)f * A.N] = o[f];
                if (A.reduce) {                                      // CFL max-reduction of the new state (R12)
                    Prim<ND> wo = primitives<ND>(o, gz_of(j), A);
                    double s = 0.0;
                    if (!(o[0] > 0.0) || !(wo.T > 0.0)) s = NAN;
                    double cs = sqrt(A.gamma * A.R * wo.T);
#pragma unroll
                    for (int c = 0; c < ND; ++c) s = fmax_nan(s, (fabs(wo.u[c]) + cs) * A.inv_d[c]);
                    smax = fmax_nan(smax, s);
                }
            }
        }
        // (6) rotate the pipeline
#pragma unroll
        for (int f = 0; f < NF; ++f) { X0[f] = X1[f]; X1[f] = X2[f]; XP0[f] = XP1[f]; }
        um0[0] = w1.u[CA]; um0[1] = w1.u[CM];
        uPm[0] = wP0.u[CA]; uPm[1] = wP0.u[CM];
        w1 = w2; wP0 = wP1; C0 = C1; C1 = C2;
    }

    if (A.reduce) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) smax = fmax_nan(smax, __shfl_xor_sync(0xffffffffu, smax, o));
        if (xi == 0 && warp_on) atomic_max_bits(A.smax_bits, smax);
    }
}

}  // namespace mc
