// sweep_march.cuh -- kernel k_march: one operator L_alpha(tau) of Eqs. 31-39
// for a sweep axis alpha that is NOT the fastest (x) axis.  The library launches it for the 2-D z-sweep
// (blocks of 128 columns, 124 outputs); the 3-D box has its own kernel (k_march3, sweep_march3.cuh), so
// the (x, b) tile roles below (HAS_B) are instantiated only by developer builds.
//
// Design: one thread owns one grid column along alpha and MARCHES along it,
// keeping every along-alpha neighbour (predictor flux F_{k-1}, corrector flux F^P_{k+1}, the five-node
// TVD stencil) in registers; consecutive threads own consecutive x, so every global access is a
// coalesced row segment.  Only the velocities needed by the cross derivatives inside the viscous
// flux (d_x, d_b of u, central, R7) travel through shared memory, one plane per level, double
// buffered, ONE __syncthreads per level.  A block owns a (x, b) tile with a 2-node halo ring that is
// recomputed (ring 2: primitives; ring 1: predictor) and a chunk of levels with a 4-level warm-up.
// In 3-D a tile row is one warp, so the role of a row (ring 2 / ring 1 / plate row / interior) is warp
// uniform and each role runs its own loop; the x-halo lanes of a row simply compute along (their
// results are never stored), which keeps every warp free of divergence.
// dir = -1 (R9) is the same code marching from the other end with a negated spacing: the mirror
// identity of the scheme (tests/test_oracle_pins.py::test_mirror_identity) makes it bit-equivalent.
//
// The loop body exists in two instantiations: FAST (every level j-1 .. j+3 exists, no plate among them,
// pipeline full: no predicates at all, unrolled by two so that the register pipeline needs no moves) and
// the general one (warm-up levels, plates of the marching direction, the tail).
//
// Pipeline of iteration j (output level j):
//   prefetch X(j+3) | W(j+2) -> TVD(j+1/2) -> F(j+1) -> P(j+1) | barrier | F^P(j+1) -> out(j)
#pragma once
#include <type_traits>

#include "mc_common.cuh"

#ifndef MC_SWEEP_L2PF
#define MC_SWEEP_L2PF 4
#endif

namespace mc {

enum { ROLE_NONE = 0, ROLE_R2 = 1, ROLE_WALLROW = 2, ROLE_R1 = 3, ROLE_IN = 4 };

// CA: velocity component of alpha; CB: velocity component of the tile's second direction b (-1 in 2-D);
// WX x WB: threads of a block (WB = 1 in 2-D); WALL_M / WALL_B: the marching / second direction is z
// with plates; TVD: -1 no TVD term, 0 Eq. 34 as printed, 1 Davis/Yee (R4).
// ZS: non-uniform z grid (R19 / R20; SweepArgs::zt), z being the sweep axis.
template <int ND, int CA, int CB, int WX, int WB, bool WALL_M, bool WALL_B, int TVD, int MINB = 1, bool ZS = false>
MC_KERNEL void __launch_bounds__(WX * WB, MINB) k_march(SweepArgs A)
{
    constexpr int NF = ND + 2;
    constexpr bool HAS_B = (CB >= 0);
    constexpr bool Z_IS_ALPHA = (CA == ND - 1);      // z is the last velocity component
    static_assert(!ZS || (Z_IS_ALPHA && WALL_M && !HAS_B), "k_march serves the non-uniform grid as the 2-D z-sweep between plates");
    constexpr int TILE = WX * WB;
    constexpr int cb = HAS_B ? CB : 0;
    MC_SHARED_DECL(double, smem_raw);
    double *const smem = smem_raw + 2;                // two pad doubles in front: lane 0 may read [-1]
    double *const slotU = smem;                       // [2][ND][TILE]  velocities of X     (levels j+1, j+2)
    double *const slotP = smem + 2 * ND * TILE;       // [2][ND][TILE]  velocities of X^P   (level j+1)

    const int tx = threadIdx.x;
    const int ty = HAS_B ? (int)threadIdx.y : 0;
    const int tidx = ty * WX + tx;

    // ---- tile geometry --------------------------------------------------------------------
    const int gx = (int)blockIdx.x * (WX - 4) + tx - 2;
    const int ix = wrap(gx, A.nx);                    // any nx >= 4: a tile may wrap the seam more than once
    const int rx = min(tx, WX - 1 - tx);
    int gb = 0, rb = 99;
    bool row_exists = true, wallrow = false, row_in_range = true;
    long long col = ix;
    if (HAS_B) {
        const int gb_raw = (int)blockIdx.y * (WB - 4) + ty - 2;
        rb = min(ty, WB - 1 - ty);
        row_in_range = gb_raw < A.n_b;
        if (WALL_B) {
            row_exists = (gb_raw >= 0 && gb_raw < A.n_b);
            wallrow = (gb_raw == 0 || gb_raw == A.n_b - 1);
            gb = row_exists ? gb_raw : 0;
        } else {
            gb = wrap(gb_raw, A.n_b);                 // periodic b: the node's own index
        }
        col += (long long)gb * A.s_b;
    }
    const bool owner = row_exists && rx >= 2 && rb >= 2 && gx < A.nx && row_in_range;
    int role = ROLE_IN;
    if (HAS_B) {
        if (!row_exists) role = ROLE_NONE;
        else if (wallrow) role = ROLE_WALLROW;
        else if (rb == 0) role = ROLE_R2;
        else if (rb == 1) role = ROLE_R1;
    }

    // ---- sweep constants ------------------------------------------------------------------
    const double tau = A.dt_ptr ? 0.5 * (*A.dt_ptr) : A.tau_fixed;
    const double cdt = tau * A.inv_h;                 // tau / dx_alpha of Eqs. 31-32, signed
    const double hcdt = 0.5 * cdt;
    const double half_tod = 0.5 * tau / A.d_a;        // for Co (R5)
    const double tsrc = A.src ? -(tau * A.g) : 0.0;   // tau S: S = -g rho in the rho u_z row
    const int n = A.n_m;
    const int l0 = (int)blockIdx.z * A.chunk;
    const int l1 = min(n, l0 + A.chunk);
    // Node offsets inside a field are 32-bit element counts (N < 2^32, mc_tvd_init) in modular arithmetic.
    const unsigned sms = (unsigned)(int)((A.dir > 0) ? A.s_m : -A.s_m);
    const unsigned off_base = (unsigned)(col + ((A.dir > 0) ? 0 : (long long)(n - 1) * A.s_m));
    const double dsgn = (A.dir > 0) ? 1.0 : -1.0;
    const int pf_last = min(l1 + 1, n - 1) - MC_SWEEP_L2PF;                  // last j + 3 whose L2 prefetch is issued
    const double *inb[NF];
    double *outb[NF];
#pragma unroll
    for (int f = 0; f < NF; ++f) { inb[f] = A.in + (long long)f * A.N; outb[f] = A.out + (long long)f * A.N; }
    const double gz_fixed = A.g * ((double)gb * A.dz);                       // used when b is z

    auto exists = [&](int l) MC_INL { return WALL_M ? (l >= 0 && l < n) : true; };
    auto lev = [&](int l) MC_INL { return WALL_M ? l : wrap1(l, n); };              // l in [-n, 2n)
    auto off_of = [&](int l) MC_INL { return off_base + (unsigned)lev(l) * sms; };
    auto phys_k = [&](int l) MC_INL { const int w = lev(l); return (A.dir > 0) ? w : n - 1 - w; };
    auto kz = [&](int l) MC_INL { return clampk((A.dir > 0) ? l : n - 1 - l, n); }; // ZS: z index of level l (clamped: values beyond a plate are unused)
    auto gz_of = [&](int l) MC_INL {                         // g z_k of Eq. 17 for this thread's node at level l
        if (!Z_IS_ALPHA) return gz_fixed;
        if (ZS) return zt_gz(A, kz(l));
        return A.g * ((double)phys_k(l) * A.dz);
    };
    auto load_at = [&](unsigned o, double (&X)[NF]) MC_INL {
#pragma unroll
        for (int f = 0; f < NF; ++f) X[f] = inb[f][o];
    };
    auto load = [&](int l, double (&X)[NF]) MC_INL { load_at(off_of(l), X); };
    auto store_at = [&](unsigned o, const double (&v)[NF]) MC_INL {
#pragma unroll
        for (int f = 0; f < NF; ++f) outb[f][o] = v[f];
    };
    auto publish = [&](double *slot, int parity, const double (&u)[ND]) MC_INL {
#pragma unroll
        for (int c = 0; c < ND; ++c) slot[(parity * ND + c) * TILE + tidx] = u[c];
    };
    // central cross DIFFERENCES of the velocities published in `slot` (R7)
    auto cross = [&](const double *slot, int parity, double (&dxa)[ND], double (&dxc)[ND]) MC_INL {
        const double *s = slot + parity * ND * TILE + tidx;
#pragma unroll
        for (int c = 0; c < ND; ++c) { dxa[c] = 0.0; dxc[c] = 0.0; }
        dxa[0] = s[CA * TILE + 1] - s[CA * TILE - 1];
        dxc[0] = s[1] - s[-1];
        if (HAS_B) {
            dxa[cb] = s[CA * TILE + WX] - s[CA * TILE - WX];
            dxc[cb] = s[cb * TILE + WX] - s[cb * TILE - WX];
        }
    };
    // plate values of a node on a plate of the marching direction: no slip,
    // T = T_w; only rho is free (R10)
    auto plate = [&](int l, double rho, double (&X)[NF]) MC_INL {
        const int k = (A.dir > 0) ? l : n - 1 - l;
        const double Tw = (k == 0) ? A.Tw0 : A.Tw1;
        X[0] = rho;
#pragma unroll
        for (int c = 0; c < ND; ++c) X[1 + c] = 0.0;
        X[NF - 1] = rho * (A.cv * Tw + (ZS ? zt_gz(A, k) : A.g * ((double)k * A.dz)));
    };

    // ---- carried state (levels relative to the current output level j) -------------------------
    double Xn[NF];                 // X(j+2), prefetched during the previous iteration
    double Xc[NF];                 // X(j+1)
    double F0[NF], FP0[NF];        // F(j), F^P(j)
    double H0[NF];                 // (X^P + X)/2 + tau S^P/2 - Dh_{j-1/2} of level j
    double d0[NF];                 // dX_{j+1/2}
    double uP0[ND], TP0 = 1.0;     // u, T of X^P(j)
    double a0 = 0.0, b0 = 0.0;     // (dX_{j-1/2}, dX_{j+1/2}), |dX_{j+1/2}|^2
    double hC0 = 0.0, hC1 = 0.0;   // C/2 of Eq. 39 at levels j, j+1
    double gz1 = 0.0;              // g z of level j+1
    Prim<ND> w1;                   // primitives of X(j+1)
    // fast levels only: node offsets of level j+3 (next load) and level j (next store), and the
    // z index of level j+2 as a double (exact; saves the int-to-double conversions of g z_k)
    unsigned o3c = 0, o0c = 0;
    double kd2c = 0.0;
#pragma unroll
    for (int f = 0; f < NF; ++f) { Xn[f] = 0.0; Xc[f] = 0.0; F0[f] = 0.0; FP0[f] = 0.0; H0[f] = 0.0; d0[f] = 0.0; }
    Xn[0] = 1.0; Xc[0] = 1.0;
#pragma unroll
    for (int c = 0; c < ND; ++c) { uP0[c] = 0.0; w1.u[c] = 0.0; }
    w1.T = 1.0; w1.p = 0.0;

    // One iteration.  ROLE and FAST are compile-time tags; PAR is the compile-time parity of j in the
    // unrolled FAST pair (-1: take it from j).
    auto body = [&](auto role_tag, auto fast_tag, auto par_tag, const int j) MC_INL {
        constexpr int ROLE = decltype(role_tag)::value;
        constexpr bool FAST = decltype(fast_tag)::value;
        constexpr int PAR = decltype(par_tag)::value;
        const int p1 = (PAR >= 0) ? (PAR ^ 1) : ((j + 1) & 1);   // parity of level j+1
        const int p2 = p1 ^ 1;                                   // parity of level j+2
        const bool ex1 = FAST || exists(j + 1), ex2 = FAST || exists(j + 2);
        const bool ld1 = FAST || (ex1 && (j + 1 >= l0 - 2));     // level j+1 is loaded (Xc, w1 valid)
        const bool ld2 = ex2;
        const bool start_wall1 = !FAST && WALL_M && (j + 1 == 0);     // level j+1 is the plate the march starts on
        const bool end_wall1 = !FAST && WALL_M && (j + 1 == n - 1);   // level j+1 is the plate the march ends on

        if (ROLE == ROLE_NONE) { __syncthreads(); if (FAST) { o3c += sms; o0c += sms; kd2c += dsgn; } return; }

        // (0) prefetch X(j+3) for the next iteration
        double Xq[NF];
#pragma unroll
        for (int f = 0; f < NF; ++f) Xq[f] = Xn[f];
        const unsigned o3 = FAST ? o3c : off_of(j + 3);
        const unsigned o0 = FAST ? o0c : off_of(j);
        if (FAST || (exists(j + 3) && j + 3 <= l1 + 1)) load_at(o3, Xq);
#if MC_SWEEP_L2PF > 0
        // far-ahead L2 prefetch: the one-level register prefetch alone leaves the HBM latency exposed
        if (FAST ? (j + 3 <= pf_last) : (j + 3 + MC_SWEEP_L2PF <= l1 + 1 && exists(j + 3 + MC_SWEEP_L2PF))) {
            const unsigned op = FAST ? o3 + (unsigned)MC_SWEEP_L2PF * sms : off_of(j + 3 + MC_SWEEP_L2PF);
#pragma unroll
            for (int f = 0; f < NF; ++f) asm volatile("prefetch.global.L2 [%0];" ::"l"(inb[f] + op));
        }
#endif
        auto advance = [&]() MC_INL { if (FAST) { o3c += sms; o0c += sms; kd2c += dsgn; } };
        // ZS (R19): the outer differences of levels j and j+1 use the height of the node's cell (a plate's half cell
        // carries the factor 2 of R10), the inner one-sided differences the spacing across the face, the TVD flux of
        // face (j, j+1) is weighted by h / dzc (R20).  Uniform grid: the launch constants.
        double cdt1 = cdt, hcdt1 = hcdt, hcdt0 = hcdt, cw1 = 2.0 * cdt, cw0 = cdt, htod2 = half_tod;
        double sF = 1.0, sB = 1.0, tw0 = 1.0, tw1 = 1.0;
        if (ZS) {
            const int k0 = kz(j), k1 = kz(j + 1), k2 = kz(j + 2);
            const double idc0 = zt_idc(A, k0), idc1 = zt_idc(A, k1), hf01 = zt_hf(A, min(k0, k1));
            cdt1 = (tau * dsgn) * idc1; hcdt1 = 0.5 * cdt1; hcdt0 = (0.5 * tau * dsgn) * idc0;
            cw1 = cdt1; cw0 = hcdt0;
            htod2 = (0.5 * tau) * zt_idc(A, k2);
            sF = zt_ihf(A, min(k1, k2)); sB = zt_ihf(A, min(k0, k1));
            tw0 = hf01 * idc0; tw1 = hf01 * idc1;
        }

        // (1) W(j+2): primitives, Courant coefficient, publish velocities
        Prim<ND> w2 = w1;
        double hC2 = 0.0, gz2 = 0.0;
        if (ld2) {
            gz2 = (FAST && Z_IS_ALPHA && !ZS) ? A.g * (kd2c * A.dz) : gz_of(j + 2);
            w2 = primitives<ND>(Xn, gz2, A);
            if (ROLE == ROLE_IN && TVD >= 0) hC2 = half_courant_coef(w2.u[CA], w2.T, htod2, A);
            publish(slotU, p2, w2.u);
        }
        if (ROLE == ROLE_R2) {
            __syncthreads();
#pragma unroll
            for (int f = 0; f < NF; ++f) Xn[f] = Xq[f];
            advance();
            return;
        }
        if (ROLE == ROLE_WALLROW) {
            // a plate row of b (y-sweep): X^P = X and the output is X (R10); publish u^P = u of level j+1
            if (ld1) publish(slotP, p1, w1.u);
            __syncthreads();
            if (j >= l0 && owner) store_at(o0, H0);
#pragma unroll
            for (int f = 0; f < NF; ++f) { H0[f] = Xc[f]; Xc[f] = Xn[f]; Xn[f] = Xq[f]; }
            w1 = w2;
            advance();
            return;
        }

        // (2) TVD (Eqs. 34-39): Dh_{j+1/2} from dX_{j-1/2}, dX_{j+1/2}, dX_{j+3/2}
        double d1[NF], a1 = 0.0, b1 = 0.0;
        double cD1 = 0.0;                                          // coefficient of Dh_{j+1/2} = cD1 dX_{j+1/2} as level j+1 sees it
#pragma unroll
        for (int f = 0; f < NF; ++f) d1[f] = 0.0;
        if (ROLE == ROLE_IN && TVD >= 0) {
#pragma unroll
            for (int f = 0; f < NF; ++f) d1[f] = (ld1 && ld2) ? Xn[f] - Xc[f] : 0.0;
#pragma unroll
            for (int f = 0; f < NF; ++f) { b1 = fma(d1[f], d1[f], b1); a1 = fma(d0[f], d1[f], a1); }
            const bool have = FAST || ((j >= l0 - 1) && exists(j - 1) && exists(j) && ex1 && ex2);   // R11 at plates
            if (have) {
                const double coef = tvd_coef<(TVD >= 0 ? TVD : 0)>(a0, a1, b0, hC0, hC1);
#pragma unroll
                const double cD0 = ZS ? coef * tw0 : coef;           // (ZS: the R20 weights of levels j and j+1)
                cD1 = ZS ? coef * tw1 : coef;
#pragma unroll
                for (int f = 0; f < NF; ++f) H0[f] = fma(cD0, d0[f], H0[f]);
            }
        }

        // (3) F(j+1): flux of X at level j+1 (inner derivative forward in marching coordinates)
        double F1[NF], XP[NF], H1[NF];
        Prim<ND> wP1 = w1;
#pragma unroll
        for (int f = 0; f < NF; ++f) { F1[f] = 0.0; XP[f] = Xc[f]; H1[f] = Xc[f]; }
        const bool doF = ld1;
        if (doF) {
            if (end_wall1) {
                F1[0] = Xc[1 + CA];                   // only the mass flux is defined and needed (R10)
            } else {
                double du[ND], dxa[ND], dxc[ND];
#pragma unroll
                for (int c = 0; c < ND; ++c) du[c] = ZS ? (w2.u[c] - w1.u[c]) * sF : w2.u[c] - w1.u[c];
                cross(slotU, p1, dxa, dxc);
                flux<ND, CA>(Xc, w1, du, ZS ? (w2.T - w1.T) * sF : w2.T - w1.T, dxa, dxc, A, F1);
            }
        }
        // (4) P(j+1): predictor (Eq. 31), plate values, primitives of X^P, publish
        const bool doP = FAST || (doF && (j + 1 >= l0 - 1));
        if (doP) {
            if (start_wall1) {
                plate(j + 1, Xc[0], XP);                                      // rho unchanged
            } else if (end_wall1) {
                plate(j + 1, Xc[0] - cw1 * (F1[0] - F0[0]), XP);             // half-cell closure (R10): 2 tau / dz
            } else {
#pragma unroll
                for (int f = 0; f < NF; ++f) {
                    const double dF = F1[f] - F0[f];
                    XP[f] = fma(-cdt1, dF, Xc[f]);
                    H1[f] = fma(-cD1, d0[f], fma(-hcdt1, dF, Xc[f]));         // (X^P + X)/2 - Dh_{j+1/2}
                }
                XP[1 + CA] = fma(tsrc, Xc[0], XP[1 + CA]);
                H1[1 + CA] = fma(0.5 * tsrc, Xc[0], H1[1 + CA]);
            }
            wP1 = primitives<ND>(XP, gz1, A);
            if (start_wall1 || end_wall1) {
#pragma unroll
                for (int f = 0; f < NF; ++f) H1[f] = 0.5 * (XP[f] + Xc[f]);
            } else {
                H1[1 + CA] = fma(0.5 * tsrc, XP[0], H1[1 + CA]);             // + tau S(X^P)/2
            }
        }
        if (ld1) publish(slotP, p1, wP1.u);

        __syncthreads();

        if (ROLE == ROLE_IN) {
            // (5) F^P(j+1): flux of X^P at level j+1 (inner derivative backward in marching coordinates)
            double FP1[NF];
#pragma unroll
            for (int f = 0; f < NF; ++f) FP1[f] = 0.0;
            const bool doFP = FAST || (doP && (j + 1 >= l0));
            if (doFP) {
                if (start_wall1) {
                    FP1[0] = XP[1 + CA];
                } else {
                    double du[ND], dxa[ND], dxc[ND];
#pragma unroll
                    for (int c = 0; c < ND; ++c) du[c] = ZS ? (wP1.u[c] - uP0[c]) * sB : wP1.u[c] - uP0[c];
                    cross(slotP, p1, dxa, dxc);
                    flux<ND, CA>(XP, wP1, du, ZS ? (wP1.T - TP0) * sB : wP1.T - TP0, dxa, dxc, A, FP1);
                }
            }
            // (6) out(j): corrector (Eq. 32), average and TVD term (Eq. 33), plate values
            if (FAST || (j >= l0 && exists(j))) {
                double o[NF];
                if (!FAST && WALL_M && j == 0) {
                    plate(j, H0[0] - cw0 * (FP1[0] - FP0[0]), o);            // 0.5 * (2 tau/dz) * dF
                } else if (!FAST && WALL_M && j == n - 1) {
                    plate(j, H0[0], o);
                } else {
#pragma unroll
                    for (int f = 0; f < NF; ++f) o[f] = fma(-hcdt0, FP1[f] - FP0[f], H0[f]);
                }
                if (owner) store_at(o0, o);
            }
#pragma unroll
            for (int f = 0; f < NF; ++f) { FP0[f] = FP1[f]; d0[f] = d1[f]; }
            a0 = a1; b0 = b1; hC0 = hC1; hC1 = hC2;
#pragma unroll
            for (int c = 0; c < ND; ++c) uP0[c] = wP1.u[c];
            TP0 = wP1.T;
        }
        // (7) rotate the pipeline
#pragma unroll
        for (int f = 0; f < NF; ++f) { Xc[f] = Xn[f]; Xn[f] = Xq[f]; F0[f] = F1[f]; H0[f] = H1[f]; }
        w1 = w2; gz1 = gz2;
        advance();
    };

    // ---- the march -------------------------------------------------------------------------------
    auto march = [&](auto role_tag) MC_INL {
        using std::integral_constant;
        integral_constant<bool, false> slow;
        integral_constant<bool, true> fast;
        integral_constant<int, -1> par_any;
        int j = (WALL_M && l0 == 0) ? -2 : l0 - 4;      // below a plate there is nothing to warm up
        if (exists(j + 2)) load(j + 2, Xn);
        // fast levels: every level j-1 .. j+3 exists, none is a plate, none wraps around
        const int jf0 = max(l0, 1);
        const int jf1 = min(l1, n - 3);
        for (; j < l1 && (j < jf0 || (j & 1)); ++j) body(role_tag, slow, par_any, j);
        if (j + 1 < jf1) { o3c = off_of(j + 3); o0c = off_of(j); kd2c = (double)phys_k(j + 2); }
        for (; j + 1 < jf1; j += 2) {
            body(role_tag, fast, integral_constant<int, 0>(), j);
            body(role_tag, fast, integral_constant<int, 1>(), j + 1);
        }
        for (; j < l1; ++j) body(role_tag, slow, par_any, j);
    };
    if (!HAS_B) {
        march(std::integral_constant<int, ROLE_IN>());
    } else {
        switch (role) {
        case ROLE_NONE: march(std::integral_constant<int, ROLE_NONE>()); break;
        case ROLE_R2: march(std::integral_constant<int, ROLE_R2>()); break;
        case ROLE_WALLROW: march(std::integral_constant<int, WALL_B ? ROLE_WALLROW : ROLE_NONE>()); break;
        case ROLE_R1: march(std::integral_constant<int, ROLE_R1>()); break;
        default: march(std::integral_constant<int, ROLE_IN>()); break;
        }
    }
}

}  // namespace mc
