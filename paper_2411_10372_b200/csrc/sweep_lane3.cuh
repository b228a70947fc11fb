// sweep_lane3.cuh -- kernel k_lane3: the operator L_x(tau) of Eqs. 31-39 in 3-D, i.e.
// the sweep along the fastest (x) axis.
//
// Design: as k_lane (sweep_lane.cuh, which serves the 2-D x-sweep) a warp owns 32
// consecutive x columns (28 outputs + a 2-node halo on each side), every along-alpha neighbour is a
// warp shuffle and every global access one coalesced 256-byte row segment; the warp marches along z
// with the z-neighbours of the central cross derivative in registers.  The block stacks WB warps along
// y: rows 1 .. WB-2 are OUTPUT rows (the whole operator), rows 0 and WB-1 the ring-1 halo (predictor
// only); a ring-1 warp also publishes the two velocity components of its outer (ring-2) neighbour row,
// which only the y-derivatives of its own predictor need, so no warp is parked on the ring-2 rows.
// (u_x, u_y) of X and X^P travel through shared memory, double buffered, one barrier per level.
//
// Pipeline of iteration j (output level j):
//   prefetch X(j+3) | barrier | W(j+2) -> F(j+1) -> P(j+1) -> F^P(j) -> out(j)
#pragma once
#include <type_traits>

#include "mc_common.cuh"
#include "sweep_lane.cuh"

namespace mc {

#ifndef MC_LANE3_L2PF
#define MC_LANE3_L2PF 4
#endif
// CB: velocity component of the tile's second direction b (y); CM: component of the marching
// direction m (z); WB: warps (rows) per block; WALL_M: m is z with plates; TVD: -1 / 0 / 1 as in
// k_march; REDUCE: fold the CFL max-reduction of the output into the epilogue (R12).  alpha is x.
// ZS: non-uniform z grid (R19; SweepArgs::zt): z is the marching direction, a cross direction of this sweep.
// SL: this box is one slab of a larger one (y is the slab axis): store the owned rows only, push the boundary rows into
// the neighbours' halos (SweepArgs::peer_*), and reduce the CFL maximum over the owned rows only.
template <int CB, int CM, int WB, bool WALL_M, int TVD, bool REDUCE, bool ZS = false, bool SL = false>
MC_KERNEL void __maxnreg__(((65536 / (32 * WB)) / 8 * 8) > 248 ? 248 : ((65536 / (32 * WB)) / 8 * 8)) k_lane3(SweepArgs A)
{
    constexpr int ND = 3, NF = 5;
    constexpr bool HAS_B = true;
    constexpr int CA = 0;
    constexpr int OB = WB - 2;                         // output rows per tile
    constexpr int TILE = 32 * (WB + 2);                // shared-memory plane: tile rows plus the ring-2 rows
    constexpr int cb = CB;
    MC_SHARED_DECL(double, smem);
    double *const slotU = smem;                        // [2][2][TILE]: (u_x, u_b) of X
    double *const slotP = smem + 4 * TILE;             // [2][2][TILE]: (u_x, u_b) of X^P

    const int xi = threadIdx.x;                        // lane coordinate along alpha (always "dir = +1")
    const int ty = threadIdx.y;
    const int tidx = (ty + 1) * 32 + xi;

    // ---- tile geometry --------------------------------------------------------------------
    const int xtile = (int)blockIdx.x;
    const int gx0 = xtile * LANE_OUT;
    const int gx = (A.dir > 0) ? gx0 - 2 + xi : gx0 + (LANE_OUT + 1) - xi;
    const int ix = wrap(gx, A.nx);
    const bool warp_on = gx0 < A.nx;
    const bool edge = (ty == 0 || ty == WB - 1);
    const int gb = (int)blockIdx.y * OB + ty - 1;
    const int go = gb + (ty == 0 ? -1 : 1);             // the ring-2 row beyond an edge row
    const unsigned off_base = (unsigned)(ix + (long long)wrap(gb, A.n_b) * A.s_b);
    const unsigned off_base_o = (unsigned)(ix + (long long)wrap(go, A.n_b) * A.s_b);
    const int tidx_o = tidx + (ty == 0 ? -32 : 32);
    const SlabRows srow = SL ? slab_rows(A, gb) : SlabRows{true, false, false};
    const bool owner = warp_on && !edge && gb < A.n_b && xi >= 2 && xi < 2 + LANE_OUT && gx >= 0 && gx < A.nx && srow.mine;

    // ---- sweep constants ------------------------------------------------------------------
    const double tau = A.dt_ptr ? 0.5 * (*A.dt_ptr) : A.tau_fixed;
    const double cdt = tau * A.inv_h;
    const double half_tod = 0.5 * tau / A.d_a;
    const int n = A.n_m;
    const int l0 = (int)blockIdx.z * A.chunk;
    const int l1 = min(n, l0 + A.chunk);
    const unsigned sm = (unsigned)A.s_m;              // node offsets are 32-bit (N < 2^32, mc_tvd_init)
    const int pf_last = min(l1 + 1, n - 1) - MC_LANE3_L2PF;   // last j + 3 whose L2 prefetch is issued
    const double *inb[NF];
    double *outb[NF];
#pragma unroll
    for (int f = 0; f < NF; ++f) { inb[f] = A.in + (long long)f * A.N; outb[f] = A.out + (long long)f * A.N; }

    auto exists = [&](int l) MC_INL { return WALL_M ? (l >= 0 && l < n) : true; };
    auto is_plate = [&](int l) MC_INL { return WALL_M && (l == 0 || l == n - 1); };
    auto lev = [&](int l) MC_INL { return WALL_M ? l : wrap1(l, n); };
    auto gz_of = [&](int l) MC_INL { return ZS ? zt_gz(A, clampk(l, n)) : A.g * ((double)lev(l) * A.dz); };       // m is z
    auto load_at = [&](unsigned o, double (&X)[NF]) MC_INL {
#pragma unroll
        for (int f = 0; f < NF; ++f) X[f] = inb[f][o];
    };
    auto load = [&](int l, double (&X)[NF]) MC_INL { load_at(off_base + (unsigned)lev(l) * sm, X); };
    auto load_outer_at = [&](unsigned o, double (&X)[3]) MC_INL {   // rho, m_x, m_b of the ring-2 row
        X[0] = inb[0][o]; X[1] = inb[1][o]; X[2] = inb[1 + cb][o];
    };
    auto load_outer = [&](int l, double (&X)[3]) MC_INL { load_outer_at(off_base_o + (unsigned)lev(l) * sm, X); };
    auto prefetch_l2 = [&](unsigned o) MC_INL {
#pragma unroll
        for (int f = 0; f < NF; ++f) asm volatile("prefetch.global.L2 [%0];" ::"l"(inb[f] + o));
    };
    auto publish = [&](double *slot, int parity, const double (&u)[ND]) MC_INL {
        slot[(parity * 2 + 0) * TILE + tidx] = u[0];
        slot[(parity * 2 + 1) * TILE + tidx] = u[cb];
    };
    // central b-differences of (u_x, u_b) published in `slot`
    auto cross_b = [&](const double *slot, int parity, double (&dxa)[ND], double (&dxc)[ND]) MC_INL {
        if (HAS_B) {
            const double *s = slot + parity * 2 * TILE + tidx;
            dxa[cb] = s[32] - s[-32];
            dxc[cb] = s[TILE + 32] - s[TILE - 32];
        }
    };

    // ---- carried state ----------------------------------------------------------------------
    double Xn[NF];                 // X(j+2), prefetched
    double Xon[3] = {1.0, 0.0, 0.0};   // rho, m_x, m_b of the ring-2 row at level j+2 (ring-1 rows only)
    double X0[NF], X1[NF];         // X(j), X(j+1)
    double XP0[NF];                // X^P(j)
    Prim<ND> w1, wP0;              // primitives of X(j+1), X^P(j)
    double um0[2] = {0.0, 0.0};    // (u_x, u_m) of X(j)
    double uPm[2] = {0.0, 0.0};    // (u_x, u_m) of X^P(j-1)
    double hC0 = 0.0, hC1 = 0.0;   // C/2 of Eq. 39 at levels j, j+1
    double gz1 = 0.0, gz0 = 0.0;   // g z of levels j+1, j
    // fast levels only: node offsets of level j+3 (next load) and level j (next store), z index of level j+2
    unsigned o3c = 0, o0c = 0;
    double kd2c = 0.0;
    double smax = 0.0, smax2 = 0.0;   // running CFL maximum and smax^2 (1 - 1e-6) for the filter
    if (REDUCE) {
        // start the filter from the maximum other blocks have already recorded (the bottom, hottest chunks
        // are scheduled first): a node below a recorded value cannot be the maximum
        const double g0 = __longlong_as_double((long long)*(volatile unsigned long long *)A.smax_bits);
        smax2 = (g0 * g0) * (1.0 - 1e-6);
    }
#pragma unroll
    for (int f = 0; f < NF; ++f) { Xn[f] = 0.0; X0[f] = 0.0; X1[f] = 0.0; XP0[f] = 0.0; }
    Xn[0] = 1.0; X0[0] = 1.0; X1[0] = 1.0; XP0[0] = 1.0;
#pragma unroll
    for (int c = 0; c < ND; ++c) { w1.u[c] = 0.0; wP0.u[c] = 0.0; }
    w1.T = 1.0; w1.p = 0.0; wP0.T = 1.0; wP0.p = 0.0;

    auto body = [&](auto role_tag, auto fast_tag, auto par_tag, const int j) MC_INL {
        constexpr int ROLE = decltype(role_tag)::value;
        constexpr bool FAST = decltype(fast_tag)::value;
        constexpr int PAR = decltype(par_tag)::value;
        const int p0 = (PAR >= 0) ? PAR : (j & 1), p1 = p0 ^ 1;
        const bool ex1 = FAST || exists(j + 1), ex2 = FAST || exists(j + 2);
        const bool ld1 = FAST || (ex1 && (j + 1 >= l0 - 2));

        // (0) prefetch X(j+3)
        double Xq[NF];
#pragma unroll
        for (int f = 0; f < NF; ++f) Xq[f] = Xn[f];
        const bool ld3 = FAST || (exists(j + 3) && j + 3 <= l1 + 1);
        const unsigned o3 = FAST ? o3c : off_base + (unsigned)lev(j + 3) * sm;
        if (ld3) load_at(o3, Xq);
        double Xoq[3] = {Xon[0], Xon[1], Xon[2]};
        if (ROLE == LROLE_R1 && ld3) load_outer_at(o3 - off_base + off_base_o, Xoq);
#if MC_LANE3_L2PF > 0
        if (FAST) { if (j + 3 <= pf_last) prefetch_l2(o3 + (unsigned)MC_LANE3_L2PF * sm); }
        else if (j + 3 + MC_LANE3_L2PF <= l1 + 1 && exists(j + 3 + MC_LANE3_L2PF))
            prefetch_l2(off_base + (unsigned)lev(j + 3 + MC_LANE3_L2PF) * sm);
#endif

        if (HAS_B) __syncthreads();

        // (1) W(j+2)
        Prim<ND> w2 = w1;
        double hC2 = 0.0, gz2 = 0.0;
        if (ex2) {
            gz2 = (FAST && !ZS) ? A.g * (kd2c * A.dz) : gz_of(j + 2);
            w2 = primitives<ND>(Xn, gz2, A);
            if (ROLE == LROLE_IN && TVD >= 0) hC2 = half_courant_coef(w2.u[CA], w2.T, half_tod, A);
            publish(slotU, p0, w2.u);                   // parity of level j+2
            if (ROLE == LROLE_R1) {                     // side job: (u_x, u_b) of the ring-2 row
                const double inv = rcp_fast(Xon[0]);
                slotU[(p0 * 2 + 0) * TILE + tidx_o] = Xon[1] * inv;
                slotU[(p0 * 2 + 1) * TILE + tidx_o] = Xon[2] * inv;
            }
        }

        // (2) F(j+1) and (3) P(j+1): Eq. 31 with the inner derivative forward along the lanes
        double XP1[NF];
        Prim<ND> wP1 = w1;
#pragma unroll
        for (int f = 0; f < NF; ++f) XP1[f] = X1[f];
        const bool doP = FAST || (ld1 && (j + 1 >= l0 - 1) && !is_plate(j + 1));
        if (doP) {                                       // warp-uniform
            double F1[NF], Fm[NF], du[ND], dxa[ND], dxc[ND];
#pragma unroll
            for (int c = 0; c < ND; ++c) {
                du[c] = __shfl_down_sync(0xffffffffu, w1.u[c], 1) - w1.u[c];
                dxa[c] = 0.0; dxc[c] = 0.0;
            }
            const double dT = __shfl_down_sync(0xffffffffu, w1.T, 1) - w1.T;
            dxa[CM] = w2.u[CA] - um0[0];
            dxc[CM] = w2.u[CM] - um0[1];
            if (ZS) { const double sz = zt_icz(A, clampk(j + 1, n)); dxa[CM] *= sz; dxc[CM] *= sz; }   // / (z_{k+1} - z_{k-1})
            cross_b(slotU, p1, dxa, dxc);
            flux<ND, CA>(X1, w1, du, dT, dxa, dxc, A, F1);
            shfl_up_vec<NF>(F1, Fm);
#pragma unroll
            for (int f = 0; f < NF; ++f) XP1[f] = fma(-cdt, F1[f] - Fm[f], X1[f]);
            wP1 = primitives<ND>(XP1, gz1, A);
        }
        if (ld1) publish(slotP, p1, wP1.u);              // plate levels publish u^P = u (X^P = X there, R10)

        // (4) F^P(j), (5) corrector, TVD, out(j)
        if (ROLE == LROLE_IN) {
            const bool doOut = FAST || ((j >= l0) && exists(j));
            if (doOut) {                                 // warp-uniform
                double o[NF];
                if (!FAST && is_plate(j)) {
#pragma unroll
                    for (int f = 0; f < NF; ++f) o[f] = X0[f];        // x-sweeps leave the plate rows unchanged
                } else {
                    double FP0[NF], FPp[NF], du[ND], dxa[ND], dxc[ND];
#pragma unroll
                    for (int c = 0; c < ND; ++c) {               // backward along the lanes: node minus lane-1
                        du[c] = wP0.u[c] - __shfl_up_sync(0xffffffffu, wP0.u[c], 1);
                        dxa[c] = 0.0; dxc[c] = 0.0;
                    }
                    const double dT = wP0.T - __shfl_up_sync(0xffffffffu, wP0.T, 1);
                    dxa[CM] = wP1.u[CA] - uPm[0];
                    dxc[CM] = wP1.u[CM] - uPm[1];
                    if (ZS) { const double sz = zt_icz(A, clampk(j, n)); dxa[CM] *= sz; dxc[CM] *= sz; }
                    cross_b(slotP, p0, dxa, dxc);
                    flux<ND, CA>(XP0, wP0, du, dT, dxa, dxc, A, FP0);
                    shfl_down_vec<NF>(FP0, FPp);
                    // TVD term along the lanes (Eqs. 34-39)
                    double Tt[NF];
#pragma unroll
                    for (int f = 0; f < NF; ++f) Tt[f] = 0.0;
                    if (TVD >= 0) {
                        double Xr[NF], d0[NF], dm[NF], Dh[NF], Dhm[NF], b0 = 0.0, a0 = 0.0;
                        shfl_down_vec<NF>(X0, Xr);
#pragma unroll
                        for (int f = 0; f < NF; ++f) { d0[f] = Xr[f] - X0[f]; b0 = fma(d0[f], d0[f], b0); }
                        shfl_up_vec<NF>(d0, dm);
#pragma unroll
                        for (int f = 0; f < NF; ++f) a0 = fma(dm[f], d0[f], a0);
                        const double a1 = __shfl_down_sync(0xffffffffu, a0, 1);
                        const double hCr = __shfl_down_sync(0xffffffffu, hC0, 1);
                        const double coef = tvd_coef<(TVD >= 0 ? TVD : 0)>(a0, a1, b0, hC0, hCr);
#pragma unroll
                        for (int f = 0; f < NF; ++f) Dh[f] = coef * d0[f];
                        shfl_up_vec<NF>(Dh, Dhm);
#pragma unroll
                        for (int f = 0; f < NF; ++f) Tt[f] = Dh[f] - Dhm[f];
                    }
#pragma unroll
                    for (int f = 0; f < NF; ++f) {
                        const double XC = fma(-cdt, FPp[f] - FP0[f], X0[f]);     // Eq. 32 (R1)
                        o[f] = fma(0.5, XP0[f] + XC, Tt[f]);                     // Eq. 33
                    }
                }
                if (owner) {
                    const unsigned oo = FAST ? o0c : off_base + (unsigned)lev(j) * sm;
#pragma unroll
                    for (int f = 0; f < NF; ++f) outb[f][oo] = o[f];
                    if (SL) slab_push<NF>(A, srow, oo, o);
                }
                if (REDUCE) {                                        // CFL max-reduction of the new state (R12)
                    const double gzj = gz0;
                    const bool need = owner && !cfl_can_skip<ND>(o, gzj, smax2, A);
                    if (__any_sync(0xffffffffu, need)) {             // rare once the running maximum has settled
                        const double s = cfl_speed<ND>(o, gzj, A, ZS ? zt_icfl(A, clampk(j, n)) : -1.0);
                        if (owner) { smax = fmax_nan(smax, s); smax2 = fmax_nan(smax2, (smax * smax) * (1.0 - 1e-6)); }
                    }
                }
            }
        }
        // (6) rotate the pipeline
#pragma unroll
        for (int f = 0; f < NF; ++f) { X0[f] = X1[f]; X1[f] = Xn[f]; Xn[f] = Xq[f]; XP0[f] = XP1[f]; }
        Xon[0] = Xoq[0]; Xon[1] = Xoq[1]; Xon[2] = Xoq[2];
        um0[0] = w1.u[CA]; um0[1] = w1.u[CM];
        uPm[0] = wP0.u[CA]; uPm[1] = wP0.u[CM];
        w1 = w2; wP0 = wP1; hC0 = hC1; hC1 = hC2; gz0 = gz1; gz1 = gz2;
        if (FAST) { o3c += sm; o0c += sm; kd2c += 1.0; }
    };

    auto march = [&](auto role_tag) MC_INL {
        using std::integral_constant;
        integral_constant<bool, false> slow;
        integral_constant<bool, true> fast;
        integral_constant<int, -1> par_any;
        int j = (WALL_M && l0 == 0) ? -2 : l0 - 4;      // below a plate there is nothing to warm up
        if (exists(j + 2)) {
            load(j + 2, Xn);
            if (decltype(role_tag)::value == LROLE_R1) load_outer(j + 2, Xon);
        }
        // fast levels: every level j-1 .. j+3 exists, none is a plate, none wraps around
        const int jf0 = max(l0, 1);
        const int jf1 = min(l1, n - 3);
        for (; j < l1 && (j < jf0 || (j & 1)); ++j) body(role_tag, slow, par_any, j);
        if (j + 1 < jf1) { o3c = off_base + (unsigned)(j + 3) * sm; o0c = off_base + (unsigned)j * sm; kd2c = (double)(j + 2); }
        for (; j + 1 < jf1; j += 2) {
            body(role_tag, fast, integral_constant<int, 0>(), j);
            body(role_tag, fast, integral_constant<int, 1>(), j + 1);
        }
        for (; j < l1; ++j) body(role_tag, slow, par_any, j);
    };
    if (edge) {
        march(std::integral_constant<int, LROLE_R1>());
    } else {
        march(std::integral_constant<int, LROLE_IN>());
    }

    if (REDUCE) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) smax = fmax_nan(smax, __shfl_xor_sync(0xffffffffu, smax, o));
        if (xi == 0 && !edge) atomic_max_bits(A.smax_bits, smax);
    }
}

}  // namespace mc
