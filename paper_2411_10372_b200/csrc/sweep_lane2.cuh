// sweep_lane2.cuh -- kernel k_lane2: the operator L_x(tau) of Eqs. 31-39 in 2-D with
// TWO x nodes per thread (boxes with an even nx; k_lane of sweep_lane.cuh serves the others).
//
// Design.  As in k_lane a warp owns a run of consecutive x columns and marches along
// z with the z-neighbours of the central cross derivative in registers; warps are independent (no shared
// memory, no barrier).  Here lane l owns the node pair (2l, 2l+1) of a 64-node run, so
//   * every global access is one double2 per field and lane (a coalesced 512-byte row segment);
//   * half of the along-alpha neighbours are the thread's own other node: a "right" neighbour is
//     {own B, shuffle-down of A}, a "left" one {shuffle-up of B, own A}: 28 instead of 56 shuffled
//     doubles per two nodes;
//   * the 2-node halo on each side is ONE lane (lanes 0 and 31): 60 of 64 nodes are outputs (28 of 32 in
//     k_lane);
//   * each thread carries two independent dependency chains, which is what the fp64 issue stalls need.
// dir = -1 (R9) maps nodes to x in reverse order with a negated spacing: a pair is then loaded and stored
// with its two halves swapped.
//
// Pipeline of iteration j (output level j):
//   prefetch X(j+3) | W(j+2) -> F(j+1) -> P(j+1) -> F^P(j) -> TVD(j) -> out(j)
#pragma once
#include <type_traits>

#include "mc_common.cuh"
#include "sweep_lane.cuh"

namespace mc {

constexpr int LANE2_OUT = 60;      // outputs per warp: 64 nodes minus the 2 + 2 halo

// the value of the right / left neighbour node of each of the thread's two nodes (A = 2l, B = 2l + 1)
MC_DEV void nbr_right(double vA, double vB, double &rA, double &rB)
{
    rA = vB;
    rB = __shfl_down_sync(0xffffffffu, vA, 1);
}
MC_DEV void nbr_left(double vA, double vB, double &lA, double &lB)
{
    lA = __shfl_up_sync(0xffffffffu, vB, 1);
    lB = vA;
}

// WARPS: independent warps per block; WALL_M: z has plates; TVD: -1 / 0 / 1 as in k_march; REDUCE: fold the
// CFL max-reduction of the output into the epilogue (R12); MINB: resident blocks per SM (register budget).
#ifndef MC_LANE2_UNROLL
#define MC_LANE2_UNROLL 2
#endif
// FWD: dir = +1 (compile time: the pair's halves are swapped for dir = -1).  The fast loop is unrolled by
// MC_LANE2_UNROLL so that most of the register pipeline's rotation needs no moves (6 = lcm of the rotation
// periods removes them all, but measured 2 < 3 < 6 in time: 0.83 / 0.87 / 0.88 ms on C3).
// ZS: non-uniform z grid (R19; SweepArgs::zt): z is the marching direction, i.e. the cross direction of this sweep.
template <int WARPS, bool WALL_M, int TVD, bool REDUCE, int MINB, bool FWD, bool ZS = false>
MC_KERNEL void __launch_bounds__(32 * WARPS, MINB) k_lane2(SweepArgs A)
{
    constexpr int ND = 2, NF = 4, CA = 0, CM = 1;
    static_assert(!ZS || WALL_M, "the non-uniform z grid lies between plates");
    const int lane = threadIdx.x;
    const int xtile = (int)blockIdx.x * WARPS + (int)threadIdx.y;
    const int gx0 = xtile * LANE2_OUT;
    if (gx0 >= A.nx) return;                           // warps are independent

    // node n = 2 lane + P sits at x = gx0 - 2 + n (dir +1) or gx0 + 61 - n (dir -1); the pair's lower x is even
    constexpr bool fwd = FWD;
    const int xlo_raw = fwd ? gx0 - 2 + 2 * lane : gx0 + 60 - 2 * lane;
    const int xlo = wrap(xlo_raw, A.nx);               // nx even: a pair never straddles the seam
    const bool owner = lane >= 1 && lane <= 30 && xlo_raw >= 0 && xlo_raw < A.nx;

    const double tau = A.dt_ptr ? 0.5 * (*A.dt_ptr) : A.tau_fixed;
    const double cdt = tau * A.inv_h;
    const double half_tod = 0.5 * tau / A.d_a;
    const int n = A.n_m;
    const int l0 = (int)blockIdx.z * A.chunk;
    const int l1 = min(n, l0 + A.chunk);
    const unsigned sm = (unsigned)A.s_m;               // node offsets are 32-bit (N < 2^32, mc_tvd_init)
    const unsigned off_base = (unsigned)xlo;
    const int pf_last = min(l1 + 1, n - 1) - MC_SWEEP_L2PF;
    const double *inb[NF];
    double *outb[NF];
#pragma unroll
    for (int f = 0; f < NF; ++f) { inb[f] = A.in + (long long)f * A.N; outb[f] = A.out + (long long)f * A.N; }

    auto exists = [&](int l) MC_INL { return WALL_M ? (l >= 0 && l < n) : true; };
    auto is_plate = [&](int l) MC_INL { return WALL_M && (l == 0 || l == n - 1); };
    auto lev = [&](int l) MC_INL { return WALL_M ? l : wrap1(l, n); };
    auto gz_of = [&](int l) MC_INL { return ZS ? zt_gz(A, clampk(l, n)) : A.g * ((double)lev(l) * A.dz); };
    auto off_of = [&](int l) MC_INL { return off_base + (unsigned)lev(l) * sm; };
    auto load_at = [&](unsigned o, double (&X)[2][NF]) MC_INL {
#pragma unroll
        for (int f = 0; f < NF; ++f) {
            const double2 v = *reinterpret_cast<const double2 *>(inb[f] + o);
            X[0][f] = fwd ? v.x : v.y;
            X[1][f] = fwd ? v.y : v.x;
        }
    };

    // ---- carried state: [P] = the thread's node A (0) or B (1) ----------------------------------------
    double Xn[2][NF];              // X(j+2), prefetched
    double X0[2][NF], X1[2][NF];   // X(j), X(j+1)
    double XP0[2][NF];             // X^P(j)
    Prim<ND> w1[2], wP0[2];        // primitives of X(j+1), X^P(j)
    double um0[2][2];              // (u_x, u_z) of X(j)
    double uPm[2][2];              // (u_x, u_z) of X^P(j-1)
    double hC0[2] = {0.0, 0.0}, hC1[2] = {0.0, 0.0};   // C/2 of Eq. 39 at levels j, j+1
    double gz1 = 0.0, gz0 = 0.0;   // g z of levels j+1, j
    // fast levels only: node offsets of level j+3 (next load) and level j (next store), z index of level j+2
    unsigned o3c = 0, o0c = 0;
    double kd2c = 0.0;
    double smax = 0.0, smax2 = 0.0;   // running CFL maximum and smax^2 (1 - 1e-6) for the filter
    if (REDUCE) {
        // start the filter from the maximum other blocks have already recorded (cfl_can_skip)
        const double g0 = __longlong_as_double((long long)*(volatile unsigned long long *)A.smax_bits);
        smax2 = (g0 * g0) * (1.0 - 1e-6);
    }
#pragma unroll
    for (int P = 0; P < 2; ++P) {
#pragma unroll
        for (int f = 0; f < NF; ++f) { Xn[P][f] = 0.0; X0[P][f] = 0.0; X1[P][f] = 0.0; XP0[P][f] = 0.0; }
        Xn[P][0] = 1.0; X0[P][0] = 1.0; X1[P][0] = 1.0; XP0[P][0] = 1.0;
#pragma unroll
        for (int c = 0; c < ND; ++c) { w1[P].u[c] = 0.0; wP0[P].u[c] = 0.0; um0[P][c] = 0.0; uPm[P][c] = 0.0; }
        w1[P].T = 1.0; w1[P].p = 0.0; wP0[P].T = 1.0; wP0[P].p = 0.0;
    }

    auto body = [&](auto fast_tag, const int j) MC_INL {
        constexpr bool FAST = decltype(fast_tag)::value;
        const bool ex1 = FAST || exists(j + 1), ex2 = FAST || exists(j + 2);
        const bool ld1 = FAST || (ex1 && (j + 1 >= l0 - 2));

        // (0) prefetch X(j+3) into registers, X(j+3+MC_SWEEP_L2PF) into L2
        double Xq[2][NF];
#pragma unroll
        for (int P = 0; P < 2; ++P)
#pragma unroll
            for (int f = 0; f < NF; ++f) Xq[P][f] = Xn[P][f];
        const unsigned o3 = FAST ? o3c : off_of(j + 3);
        if (FAST || (exists(j + 3) && j + 3 <= l1 + 1)) load_at(o3, Xq);
#if MC_SWEEP_L2PF > 0
        if (FAST ? (j + 3 <= pf_last) : (j + 3 + MC_SWEEP_L2PF <= l1 + 1 && exists(j + 3 + MC_SWEEP_L2PF))) {
            const unsigned op = FAST ? o3 + (unsigned)MC_SWEEP_L2PF * sm : off_of(j + 3 + MC_SWEEP_L2PF);
#pragma unroll
            for (int f = 0; f < NF; ++f) asm volatile("prefetch.global.L2 [%0];" ::"l"(inb[f] + op));
        }
#endif

        // (1) W(j+2)
        Prim<ND> w2[2] = {w1[0], w1[1]};
        double hC2[2] = {0.0, 0.0}, gz2 = 0.0;
        if (ex2) {
            gz2 = (FAST && !ZS) ? A.g * (kd2c * A.dz) : gz_of(j + 2);
#pragma unroll
            for (int P = 0; P < 2; ++P) {
                w2[P] = primitives<ND>(Xn[P], gz2, A);
                if (TVD >= 0) hC2[P] = half_courant_coef(w2[P].u[CA], w2[P].T, half_tod, A);
            }
        }

        // (2) F(j+1) and (3) P(j+1): Eq. 31 with the inner derivative forward along the nodes
        double XP1[2][NF];
        Prim<ND> wP1[2] = {w1[0], w1[1]};
#pragma unroll
        for (int P = 0; P < 2; ++P)
#pragma unroll
            for (int f = 0; f < NF; ++f) XP1[P][f] = X1[P][f];
        const bool doP = FAST || (ld1 && (j + 1 >= l0 - 1) && !is_plate(j + 1));
        if (doP) {                                       // warp-uniform
            double F1[2][NF], Fm[2][NF], uR[2][ND], TR[2];
#pragma unroll
            for (int c = 0; c < ND; ++c) nbr_right(w1[0].u[c], w1[1].u[c], uR[0][c], uR[1][c]);
            nbr_right(w1[0].T, w1[1].T, TR[0], TR[1]);
#pragma unroll
            for (int P = 0; P < 2; ++P) {
                double du[ND], dxa[ND], dxc[ND];
#pragma unroll
                for (int c = 0; c < ND; ++c) { du[c] = uR[P][c] - w1[P].u[c]; dxa[c] = 0.0; dxc[c] = 0.0; }
                dxa[CM] = w2[P].u[CA] - um0[P][0];
                dxc[CM] = w2[P].u[CM] - um0[P][1];
                if (ZS) { const double sz = zt_icz(A, clampk(j + 1, n)); dxa[CM] *= sz; dxc[CM] *= sz; }   // / (z_{k+1} - z_{k-1})
                flux<ND, CA>(X1[P], w1[P], du, TR[P] - w1[P].T, dxa, dxc, A, F1[P]);
            }
#pragma unroll
            for (int f = 0; f < NF; ++f) nbr_left(F1[0][f], F1[1][f], Fm[0][f], Fm[1][f]);
#pragma unroll
            for (int P = 0; P < 2; ++P) {
#pragma unroll
                for (int f = 0; f < NF; ++f) XP1[P][f] = fma(-cdt, F1[P][f] - Fm[P][f], X1[P][f]);
                wP1[P] = primitives<ND>(XP1[P], gz1, A);
            }
        }

        // (4) F^P(j), (5) corrector, TVD, out(j)
        const bool doOut = FAST || ((j >= l0) && exists(j));
        if (doOut) {                                     // warp-uniform
            double o[2][NF];
            if (!FAST && is_plate(j)) {
#pragma unroll
                for (int P = 0; P < 2; ++P)
#pragma unroll
                    for (int f = 0; f < NF; ++f) o[P][f] = X0[P][f];  // x-sweeps leave the plate rows unchanged
            } else {
                double FP0[2][NF], FPp[2][NF], uL[2][ND], TL[2];
#pragma unroll
                for (int c = 0; c < ND; ++c) nbr_left(wP0[0].u[c], wP0[1].u[c], uL[0][c], uL[1][c]);
                nbr_left(wP0[0].T, wP0[1].T, TL[0], TL[1]);
#pragma unroll
                for (int P = 0; P < 2; ++P) {                  // backward along the nodes: node minus its left one
                    double du[ND], dxa[ND], dxc[ND];
#pragma unroll
                    for (int c = 0; c < ND; ++c) { du[c] = wP0[P].u[c] - uL[P][c]; dxa[c] = 0.0; dxc[c] = 0.0; }
                    dxa[CM] = wP1[P].u[CA] - uPm[P][0];
                    dxc[CM] = wP1[P].u[CM] - uPm[P][1];
                    if (ZS) { const double sz = zt_icz(A, clampk(j, n)); dxa[CM] *= sz; dxc[CM] *= sz; }
                    flux<ND, CA>(XP0[P], wP0[P], du, wP0[P].T - TL[P], dxa, dxc, A, FP0[P]);
                }
#pragma unroll
                for (int f = 0; f < NF; ++f) nbr_right(FP0[0][f], FP0[1][f], FPp[0][f], FPp[1][f]);
                // TVD term along the nodes (Eqs. 34-39)
                double Tt[2][NF];
#pragma unroll
                for (int P = 0; P < 2; ++P)
#pragma unroll
                    for (int f = 0; f < NF; ++f) Tt[P][f] = 0.0;
                if (TVD >= 0) {
                    double Xr[2][NF], d0[2][NF], dm[2][NF], Dh[2][NF], Dhm[2][NF];
                    double b0[2] = {0.0, 0.0}, a0[2] = {0.0, 0.0}, a1[2], hCr[2];
#pragma unroll
                    for (int f = 0; f < NF; ++f) nbr_right(X0[0][f], X0[1][f], Xr[0][f], Xr[1][f]);
#pragma unroll
                    for (int P = 0; P < 2; ++P)
#pragma unroll
                        for (int f = 0; f < NF; ++f) { d0[P][f] = Xr[P][f] - X0[P][f]; b0[P] = fma(d0[P][f], d0[P][f], b0[P]); }
#pragma unroll
                    for (int f = 0; f < NF; ++f) nbr_left(d0[0][f], d0[1][f], dm[0][f], dm[1][f]);
#pragma unroll
                    for (int P = 0; P < 2; ++P)
#pragma unroll
                        for (int f = 0; f < NF; ++f) a0[P] = fma(dm[P][f], d0[P][f], a0[P]);
                    nbr_right(a0[0], a0[1], a1[0], a1[1]);
                    nbr_right(hC0[0], hC0[1], hCr[0], hCr[1]);
#pragma unroll
                    for (int P = 0; P < 2; ++P) {
                        const double coef = tvd_coef<(TVD >= 0 ? TVD : 0)>(a0[P], a1[P], b0[P], hC0[P], hCr[P]);
#pragma unroll
                        for (int f = 0; f < NF; ++f) Dh[P][f] = coef * d0[P][f];
                    }
#pragma unroll
                    for (int f = 0; f < NF; ++f) nbr_left(Dh[0][f], Dh[1][f], Dhm[0][f], Dhm[1][f]);
#pragma unroll
                    for (int P = 0; P < 2; ++P)
#pragma unroll
                        for (int f = 0; f < NF; ++f) Tt[P][f] = Dh[P][f] - Dhm[P][f];
                }
#pragma unroll
                for (int P = 0; P < 2; ++P)
#pragma unroll
                    for (int f = 0; f < NF; ++f) {
                        const double XC = fma(-cdt, FPp[P][f] - FP0[P][f], X0[P][f]);   // Eq. 32 (R1)
                        o[P][f] = fma(0.5, XP0[P][f] + XC, Tt[P][f]);                   // Eq. 33
                    }
            }
            if (owner) {
                const unsigned oo = FAST ? o0c : off_of(j);
#pragma unroll
                for (int f = 0; f < NF; ++f)
                    *reinterpret_cast<double2 *>(outb[f] + oo) = fwd ? make_double2(o[0][f], o[1][f]) : make_double2(o[1][f], o[0][f]);
            }
            if (REDUCE) {                                        // CFL max-reduction of the new state (R12)
                const bool need = owner && !(cfl_can_skip<ND>(o[0], gz0, smax2, A) && cfl_can_skip<ND>(o[1], gz0, smax2, A));
                if (__any_sync(0xffffffffu, need)) {             // rare once the running maximum has settled
                    const double idz = ZS ? zt_icfl(A, clampk(j, n)) : -1.0;
                    const double s = fmax_nan(cfl_speed<ND>(o[0], gz0, A, idz), cfl_speed<ND>(o[1], gz0, A, idz));
                    if (owner) { smax = fmax_nan(smax, s); smax2 = fmax_nan(smax2, (smax * smax) * (1.0 - 1e-6)); }
                }
            }
        }
        // (6) rotate the pipeline
#pragma unroll
        for (int P = 0; P < 2; ++P) {
#pragma unroll
            for (int f = 0; f < NF; ++f) { X0[P][f] = X1[P][f]; X1[P][f] = Xn[P][f]; Xn[P][f] = Xq[P][f]; XP0[P][f] = XP1[P][f]; }
            um0[P][0] = w1[P].u[CA]; um0[P][1] = w1[P].u[CM];
            uPm[P][0] = wP0[P].u[CA]; uPm[P][1] = wP0[P].u[CM];
            w1[P] = w2[P]; wP0[P] = wP1[P]; hC0[P] = hC1[P]; hC1[P] = hC2[P];
        }
        gz0 = gz1; gz1 = gz2;
        if (FAST) { o3c += sm; o0c += sm; kd2c += 1.0; }
    };

    // ---- the march -------------------------------------------------------------------------------
    std::integral_constant<bool, false> slow;
    std::integral_constant<bool, true> fast;
    int j = (WALL_M && l0 == 0) ? -2 : l0 - 4;      // below a plate there is nothing to warm up
    if (exists(j + 2)) load_at(off_of(j + 2), Xn);
    // fast levels: every level j-1 .. j+3 exists, none is a plate, none wraps around
    const int jf0 = max(l0, 1);
    const int jf1 = min(l1, n - 3);
    for (; j < l1 && j < jf0; ++j) body(slow, j);
    if (j < jf1) { o3c = off_of(j + 3); o0c = off_of(j); kd2c = (double)(j + 2); }
    for (; j + MC_LANE2_UNROLL <= jf1; j += MC_LANE2_UNROLL) {
#pragma unroll
        for (int q = 0; q < MC_LANE2_UNROLL; ++q) body(fast, j + q);
    }
    for (; j < l1; ++j) body(slow, j);

    if (REDUCE) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) smax = fmax_nan(smax, __shfl_xor_sync(0xffffffffu, smax, o));
        if (lane == 0) atomic_max_bits(A.smax_bits, smax);
    }
}

}  // namespace mc
