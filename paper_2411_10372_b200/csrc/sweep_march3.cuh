// sweep_march3.cuh -- kernel k_march3: one operator L_alpha(tau) of Eqs. 31-39 in
// 3-D for a sweep axis alpha that is NOT the fastest (x) axis: the z-sweep and the y-sweep.
//
// Design.  As in k_march (sweep_march.cuh, which serves the 2-D z-sweep) one
// thread owns one grid column along alpha and MARCHES along it with every along-alpha neighbour in
// registers; consecutive threads own consecutive x, so each global access is a coalesced row segment.
// A block owns a tile of 32 x WB columns in (x, b): tile row = one warp, so a row's role is warp
// uniform.  Rows 1 .. WB-2 are OUTPUT rows (role IN: the whole operator); rows 0 and WB-1 are the
// ring-1 halo (role R1: predictor only, because the corrector flux of an output row differentiates
// u^P across b, R7).  The ring-2 halo (the predictor of a ring-1 row differentiates u across b) needs
// only the velocities of X, so the ring-1 warp computes them for its outer neighbour row as a side
// job instead of parking two more warps on it: 10 of 12 warps do full work (28 x 10 outputs per 384
// threads; the SM allocates warps in fours, and 16 rows at 128 registers spill -- measured slower).
// In x, lanes 0, 1, 30, 31 are the halo: they compute along and never store.
// Velocities travel through shared memory, one plane per level, double buffered, ONE barrier per level.
//
// Pipeline of iteration j (output level j), identical to k_march:
//   prefetch X(j+3) | W(j+2) -> TVD(j+1/2) -> F(j+1) -> P(j+1) | barrier | F^P(j+1) -> out(j)
//
// AS = true (the default path, even nx): ASYNCHRONOUS STAGING.  The X tile of every level -- 32 columns x
// (WB + 2) rows x 5 fields, ring-2 rows included -- is brought in by ONE cp.async.bulk.tensor (TMA, 4-D tensor
// map (x, y, z, field)) per level into a ring of MARCH3_STAGES shared-memory stages, MARCH3_STAGES - 1 levels
// ahead, completing on a "full" mbarrier; a thread reads its own column's X(j+2) from the stage (conflict-free
// LDS), its warp then arrives on the stage's "empty" mbarrier, and one elected lane refills it.  So no
// register prefetch (X(j+3) and the ring-2 row: 9 doubles less carried), no L2 prefetch instructions, no
// per-thread load addresses, and no exposed HBM latency.  Nodes the box cannot deliver -- columns or rows that
// wrap around the periodic seam -- are zero-filled by the TMA unit and loaded by their thread directly.
// The per-level __syncthreads is replaced by DATAFLOW between neighbouring rows: once a row (warp) has published
// u(j+2) and u^P(j+1) it meets row r-1 and then row r+1 at a hardware named barrier of 64 threads (one barrier per
// pair of adjacent rows, ids 1 .. WB-1; every row takes its lower pair first, so the chain of rendezvous cannot
// deadlock).  Neighbouring rows thus stay within one level of each other (which is all the double buffered
// velocity planes need), but rows far apart -- and with them the three warps sharing an SM sub-partition -- drift
// by several levels, so one warp's dependent chain overlaps another's instead of all warps draining into one
// barrier together.  (Measured on C5: block barrier L_z 6.52 / L_y 6.44 ms, an mbarrier pair per row polled with
// try_wait 6.59 / 6.22, named pair barriers 6.15 / 6.03.)
#pragma once
#include <type_traits>

#include "mc_async.cuh"
#include "mc_common.cuh"
#include "sweep_march.cuh"

namespace mc {

// CA: velocity component of alpha; CB: velocity component of the tile's second direction b;
// WB: tile rows (warps) per block; WALL_M / WALL_B: the marching / second direction is z with plates;
// TVD: -1 no TVD term, 0 Eq. 34 as printed, 1 Davis/Yee (R4).
// Register budget: MINB blocks per SM, 65536 / (32 WB MINB) registers per thread rounded down to a multiple
// of 8 (__maxnreg__, because __launch_bounds__ rounds the block size up to a multiple of 128 threads).
// MC_MARCH3_L2PF: levels between the register prefetch and the L2 prefetch (4 measured best of 2..8).
#ifndef MC_MARCH3_L2PF
#define MC_MARCH3_L2PF 4
#endif
#ifndef MC_MARCH3_REGS
#define MC_MARCH3_REGS (((65536 / (32 * WB * MINB)) / 8 * 8) > 248 ? 248 : ((65536 / (32 * WB * MINB)) / 8 * 8))
#endif
#ifndef MC_MARCH3_STAGES
#define MC_MARCH3_STAGES 4
#endif
constexpr int MARCH3_STAGES = MC_MARCH3_STAGES;      // power of two
// dynamic shared memory of k_march3 / k_lane3 with asynchronous staging: stage ring (128-byte aligned) +
// mbarriers + velocity planes
__host__ __device__ constexpr size_t tile3_stage_bytes(int WB) { return (size_t)5 * 32 * (WB + 2) * sizeof(double); }
__host__ __device__ constexpr size_t tile3_async_bytes(int WB) { return MARCH3_STAGES * tile3_stage_bytes(WB) + 8 * (2 * MARCH3_STAGES); }

// ZS: non-uniform z grid (R19 / R20; SweepArgs::zt): z is the sweep axis (L_z) or the tile's second direction (L_y).
// SL: this box is one slab of a larger one (y is the slab axis: the tile's b for L_z, the march itself for L_y): store the
// owned rows only and push the boundary rows into the neighbours' halos (SweepArgs::peer_*).
template <int CA, int CB, int WB, bool WALL_M, bool WALL_B, int TVD, int MINB = 1, bool AS = false, bool ZS = false, bool SL = false>
MC_KERNEL void __maxnreg__(MC_MARCH3_REGS) k_march3(SweepArgs A, const __grid_constant__ CUtensorMap tmap)
{
    constexpr int ND = 3, NF = 5;
    constexpr bool Z_IS_ALPHA = (CA == ND - 1);
    constexpr bool ZA = ZS && Z_IS_ALPHA;             // the metric varies along the march
    static_assert(!ZS || (Z_IS_ALPHA ? WALL_M : (WALL_B && CB == ND - 1)), "the non-uniform z grid lies between plates");
    constexpr int OB = WB - 2;                        // output rows per tile
    static_assert(WB >= 3 && WB % 4 == 0 && WB <= 16, "the SM allocates warps in fours; named barriers 1 .. WB-1 pair the rows");
    constexpr int TILE = 32 * (WB + 2);               // shared-memory plane: tile rows plus the ring-2 rows
    constexpr int S = MARCH3_STAGES;
    static_assert((S & (S - 1)) == 0, "stage count must be a power of two");
    MC_SHARED_DECL(double, smem_raw);
    // AS: [stage ring (the dynamic shared memory is 128-byte aligned)][full[S], empty[S]][velocity planes]
    constexpr int RING_DOUBLES = AS ? S * (int)(tile3_stage_bytes(WB) / sizeof(double)) : 0;
    constexpr int BAR_DOUBLES = AS ? 2 * S : 0;
    const double *const ring = smem_raw;
    double *const bars = smem_raw + RING_DOUBLES;
    double *const smem = smem_raw + RING_DOUBLES + BAR_DOUBLES + 2;   // two pad doubles in front
    double *const slotU = smem;                       // [2][ND][TILE]  velocities of X     (levels j+1, j+2)
    double *const slotP = smem + 2 * ND * TILE;       // [2][ND][TILE]  velocities of X^P   (level j+1)

    const int tx = threadIdx.x;
    const int ty = threadIdx.y;
    const int tidx = (ty + 1) * 32 + tx;

    // ---- tile geometry --------------------------------------------------------------------
    const int gx = (int)blockIdx.x * 28 + tx - 2;
    const int ix = wrap(gx, A.nx);                    // any nx >= 4: a tile may wrap the seam more than once
    const int rx = min(tx, 31 - tx);
    const bool edge = (ty == 0 || ty == WB - 1);
    const int gb_raw = (int)blockIdx.y * OB + ty - 1;
    const int go_raw = gb_raw + (ty == 0 ? -1 : 1);   // the ring-2 row beyond an edge row
    bool row_exists = true, wallrow = false, has_outer = edge;
    int gb, go;
    if (WALL_B) {
        row_exists = (gb_raw >= 0 && gb_raw < A.n_b);
        wallrow = (gb_raw == 0 || gb_raw == A.n_b - 1);
        gb = row_exists ? gb_raw : 0;
        has_outer = edge && row_exists && !wallrow && go_raw >= 0 && go_raw < A.n_b;
        go = has_outer ? go_raw : 0;
    } else {
        gb = wrap(gb_raw, A.n_b);                     // periodic b: the node's own index
        go = wrap(go_raw, A.n_b);
    }
    const long long col = ix + (long long)gb * A.s_b;
    const long long col_o = ix + (long long)go * A.s_b;
    const int tidx_o = tidx + (ty == 0 ? -32 : 32);
    constexpr bool SL_B = SL && CB == 1, SL_M = SL && CA == 1;        // the slab axis y is b (L_z) or the march (L_y)
    const SlabRows srow_b = SL_B ? slab_rows(A, gb_raw) : SlabRows{true, false, false};
    const bool owner = row_exists && rx >= 2 && !edge && gx < A.nx && gb_raw < A.n_b && srow_b.mine;
    int role = ROLE_IN;
    if (!row_exists) role = ROLE_NONE;
    else if (wallrow) role = ROLE_WALLROW;
    else if (edge) role = ROLE_R1;
    // AS: can the TMA box deliver this thread's node (and its ring-2 neighbour)?  Not across the periodic seam.
    const bool in_box = gx >= 0 && gx < A.nx && gb_raw >= 0 && gb_raw < A.n_b;
    const bool in_box_o = gx >= 0 && gx < A.nx && go_raw >= 0 && go_raw < A.n_b;
    // AS: rows (warps) that take part: with plates across b the rows outside the box do nothing and leave
    const int b_first = (int)blockIdx.y * OB - 1;                      // gb_raw of row 0
    const int ty_lo = WALL_B ? max(0, -b_first) : 0;                   // first and last existing row
    const int ty_hi = WALL_B ? min(WB - 1, A.n_b - 1 - b_first) : WB - 1;

    // ---- sweep constants ------------------------------------------------------------------
    const double tau = A.dt_ptr ? 0.5 * (*A.dt_ptr) : A.tau_fixed;
    const double cdt = tau * A.inv_h;                 // tau / dx_alpha of Eqs. 31-32, signed
    const double hcdt = 0.5 * cdt;
    const double half_tod = 0.5 * tau / A.d_a;        // for Co (R5)
    const double tsrc = -(tau * A.g);                 // tau S: S = -g rho in the rho u_z row of the z-sweep only
    const int n = A.n_m;
    const int l0 = (int)blockIdx.z * A.chunk;
    const int l1 = min(n, l0 + A.chunk);
    // Node offsets inside a field are 32-bit element counts (N < 2^32, mc_tvd_init) in modular arithmetic;
    // the field bases A.in + f N are block uniform, so an address costs one IMAD.WIDE.
    const unsigned sms = (unsigned)(int)((A.dir > 0) ? A.s_m : -A.s_m);
    const long long org = (A.dir > 0) ? 0 : (long long)(n - 1) * A.s_m;
    const unsigned off_base = (unsigned)(col + org);
    const unsigned off_base_o = (unsigned)(col_o + org);
    const double dsgn = (A.dir > 0) ? 1.0 : -1.0;
    const int pf_last = min(l1 + 1, n - 1) - MC_MARCH3_L2PF;                // last j + 3 whose L2 prefetch is issued
    const double gz_fixed = (ZS && !Z_IS_ALPHA) ? zt_gz(A, gb) : A.g * ((double)gb * A.dz);   // used when b is z
    const double szb = (ZS && !Z_IS_ALPHA) ? zt_icz(A, gb) : 1.0;            // 1 / (z_{k+1} - z_{k-1}) of this thread's row

    auto exists = [&](int l) MC_INL { return WALL_M ? (l >= 0 && l < n) : true; };
    auto lev = [&](int l) MC_INL { return WALL_M ? l : wrap1(l, n); };              // l in [-n, 2n)
    const double *inb[NF];
    double *outb[NF];
#pragma unroll
    for (int f = 0; f < NF; ++f) { inb[f] = A.in + (long long)f * A.N; outb[f] = A.out + (long long)f * A.N; }
    auto off_of = [&](int l) MC_INL { return off_base + (unsigned)lev(l) * sms; };
    auto phys_k = [&](int l) MC_INL { const int w = lev(l); return (A.dir > 0) ? w : n - 1 - w; };
    auto load_at = [&](unsigned o, double (&X)[NF]) MC_INL {
#pragma unroll
        for (int f = 0; f < NF; ++f) X[f] = inb[f][o];
    };
    auto load = [&](int l, double (&X)[NF]) MC_INL { load_at(off_of(l), X); };
    auto kz = [&](int l) MC_INL { return clampk((A.dir > 0) ? l : n - 1 - l, n); }; // ZA: z index of level l (clamped: values beyond a plate are unused)
    auto gz_of = [&](int l) MC_INL {                         // g z_k of Eq. 17 for this thread's node at level l
        if (!Z_IS_ALPHA) return gz_fixed;
        if (ZA) return zt_gz(A, kz(l));
        return A.g * ((double)phys_k(l) * A.dz);
    };
    // L2 prefetch of the thread's node at level l (no register, no scoreboard): hides the HBM latency
    // the one-level register prefetch cannot cover with 12 warps per SM
    auto prefetch_l2 = [&](unsigned o) MC_INL {
#pragma unroll
        for (int f = 0; f < NF; ++f) asm volatile("prefetch.global.L2 [%0];" ::"l"(inb[f] + o));
    };
    auto load_outer = [&](unsigned o, double (&X)[ND + 1]) MC_INL {                 // rho and the momenta only
#pragma unroll
        for (int f = 0; f <= ND; ++f) X[f] = inb[f][o];
    };
    // (SL: `l` is the marching level of the node, which is its y index in L_y)
    auto store_at = [&](unsigned o, const double (&v)[NF], int l) MC_INL {
        const SlabRows r = SL_M ? slab_rows(A, phys_k(l)) : srow_b;
        if (!SL || r.mine) {
#pragma unroll
            for (int f = 0; f < NF; ++f) outb[f][o] = v[f];
        }
        if (SL) slab_push<NF>(A, r, o, v);
    };
    auto publish = [&](double *slot, int parity, int at, const double (&u)[ND]) MC_INL {
#pragma unroll
        for (int c = 0; c < ND; ++c) slot[(parity * ND + c) * TILE + at] = u[c];
    };
    // central cross DIFFERENCES of the velocities published in `slot` (R7)
    auto cross = [&](const double *slot, int parity, double (&dxa)[ND], double (&dxc)[ND]) MC_INL {
        const double *s = slot + parity * ND * TILE + tidx;
#pragma unroll
        for (int c = 0; c < ND; ++c) { dxa[c] = 0.0; dxc[c] = 0.0; }
        dxa[0] = s[CA * TILE + 1] - s[CA * TILE - 1];
        dxc[0] = s[1] - s[-1];
        dxa[CB] = s[CA * TILE + 32] - s[CA * TILE - 32];
        dxc[CB] = s[CB * TILE + 32] - s[CB * TILE - 32];
        if (ZS && !Z_IS_ALPHA) { dxa[CB] *= szb; dxc[CB] *= szb; }
    };
    // plate values of a node on a plate of the marching direction: no slip,
    // T = T_w; only rho is free (R10)
    auto plate = [&](int l, double rho, double (&X)[NF]) MC_INL {
        const int k = (A.dir > 0) ? l : n - 1 - l;
        const double Tw = (k == 0) ? A.Tw0 : A.Tw1;
        X[0] = rho;
#pragma unroll
        for (int c = 0; c < ND; ++c) X[1 + c] = 0.0;
        X[NF - 1] = rho * (A.cv * Tw + (ZA ? zt_gz(A, k) : A.g * ((double)k * A.dz)));
    };


    // ---- AS: stage ring, barriers ----------------------------------------------------------------
    const unsigned bar0 = AS ? smem_addr(bars) : 0u;                   // full[S], empty[S]
    const unsigned ring0 = AS ? smem_addr(ring) : 0u;
    const int j_start = (WALL_M && l0 == 0) ? -2 : l0 - 4;             // below a plate there is nothing to warm up
    const int n_lev = l1 + 2 - (j_start + 2);                          // levels j_start+2 .. l1+1 are staged, one per iteration
    const bool prod_warp = AS && ty == ty_lo;                          // the warp whose lane 0 feeds the ring
    // whole tile inside the box: no thread needs the direct-load path (true for all but the seam tiles)
    const bool tile_in_box = (int)blockIdx.x * 28 - 2 >= 0 && (int)blockIdx.x * 28 + 30 <= A.nx && b_first - 1 >= 0 &&
                             b_first + WB + 1 <= A.n_b;
    // issue the TMA load of staged level number q (march level j_start + 2 + q) into stage q % S (lane 0 only)
    auto issue = [&](int q) MC_INL {
        const int l = j_start + 2 + q;
        const int pk = (WALL_M && (l < 0 || l >= n)) ? -1 : phys_k(l);  // a level beyond a plate: all zero fill
        const unsigned full = bar0 + 8u * (unsigned)(q & (S - 1));
        const int x0 = (int)blockIdx.x * 28 - 2, b0 = b_first - 1;
        tma_issue_4d_if(tx == 0, ring0 + (unsigned)(q & (S - 1)) * (unsigned)tile3_stage_bytes(WB), &tmap, full,
                        (unsigned)tile3_stage_bytes(WB), x0, CB == 1 ? b0 : pk, CB == 1 ? pk : b0, 0);
    };
    if (AS) {
        if (threadIdx.x == 0 && threadIdx.y == 0) {
            for (int i = 0; i < S; ++i) { mbar_init(bar0 + 8u * i, 1); mbar_init(bar0 + 8u * (S + i), (unsigned)(ty_hi - ty_lo + 1)); }
            mbar_init_fence();
        }
        __syncthreads();
        if (role == ROLE_NONE) return;
        if (prod_warp) {
            if (tx == 0) tma_prefetch_descriptor(&tmap);
            for (int q = 0; q < S - 1 && q < n_lev; ++q) issue(q);
        }
    }
    int it = 0;                                                         // AS: iteration number = staged level number read
    // AS: take X(j+2) (and the ring-2 row's rho, m for a ring-1 row) of this iteration out of its stage
    auto stage_read = [&](auto role_tag, bool want, int l, double (&X)[NF], double (&Xo)[ND + 1]) MC_INL {
        constexpr int ROLE = decltype(role_tag)::value;
        const unsigned st = (unsigned)it & (S - 1), ph = ((unsigned)it / S) & 1u;
        mbar_wait(bar0 + 8u * st, ph);
        if (want) {
            const double *sp = ring + (size_t)st * (tile3_stage_bytes(WB) / sizeof(double));
            if (tile_in_box) {                                           // block uniform
#pragma unroll
                for (int f = 0; f < NF; ++f) X[f] = sp[f * TILE + tidx];
                if (ROLE == ROLE_R1 && has_outer) {
#pragma unroll
                    for (int f = 0; f <= ND; ++f) Xo[f] = sp[f * TILE + tidx_o];
                }
            } else {
                if (in_box) {
#pragma unroll
                    for (int f = 0; f < NF; ++f) X[f] = sp[f * TILE + tidx];
                } else {
                    load_at(off_of(l), X);
                }
                if (ROLE == ROLE_R1 && has_outer) {
                    if (in_box_o) {
#pragma unroll
                        for (int f = 0; f <= ND; ++f) Xo[f] = sp[f * TILE + tidx_o];
                    } else {
                        load_outer(off_of(l) - off_base + off_base_o, Xo);
                    }
                }
            }
        }
        __syncwarp();
        mbar_arrive_if(bar0 + 8u * (S + st), tx == 0);                   // this warp is done with the stage
        if (prod_warp && it + S - 1 < n_lev) {                           // warp uniform: refill the stage of the PREVIOUS iteration
            if (it > 0) mbar_wait(bar0 + 8u * (S + (((unsigned)it - 1) & (S - 1))), (((unsigned)it - 1) / S) & 1u);
            issue(it + S - 1);
        }
    };
    // AS: the row has published u(j+2), u^P(j+1): rendezvous with the existing neighbour rows, the lower one first
    const bool wait_lo = ty > ty_lo, wait_hi = ty < ty_hi;
    auto level_sync = [&]() MC_INL {
        if (!AS) { __syncthreads(); return; }
        if (wait_lo) asm volatile("barrier.sync.aligned %0, 64;" ::"r"(ty) : "memory");          // pair (ty - 1, ty)
        if (wait_hi) asm volatile("barrier.sync.aligned %0, 64;" ::"r"(ty + 1) : "memory");      // pair (ty, ty + 1)
    };

    // ---- carried state (levels relative to the current output level j) -------------------------
    double Xn[NF];                 // X(j+2)
    double Xc[NF];                 // X(j+1)
    double Xon[ND + 1];            // rho, m of the outer (ring-2) row at the level W works on next (ring-1 rows only)
    double F0[NF];                 // F(j)
    double H0[NF];                 // (X^P + X)/2 + tau S^P/2 - Dh_{j-1/2} + (tau/2dx) F^P(j) of level j
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
    for (int f = 0; f < NF; ++f) { Xn[f] = 0.0; Xc[f] = 0.0; F0[f] = 0.0; H0[f] = 0.0; d0[f] = 0.0; }
    Xn[0] = 1.0; Xc[0] = 1.0;
#pragma unroll
    for (int f = 0; f <= ND; ++f) Xon[f] = (f == 0) ? 1.0 : 0.0;
#pragma unroll
    for (int c = 0; c < ND; ++c) { uP0[c] = 0.0; w1.u[c] = 0.0; }
    w1.T = 1.0; w1.p = 0.0;

    // W(L): primitives of X(L) (in `X`), Courant coefficient, velocities published into slot uslot(L);
    // a ring-1 row also publishes the velocities of its ring-2 neighbour row (from `Xo`).
    auto stage_W = [&](auto role_tag, int par, double gz, double htod, const double (&X)[NF], const double (&Xo)[ND + 1],
                       Prim<ND> &w, double &hC) MC_INL {
        constexpr int ROLE = decltype(role_tag)::value;
        w = primitives<ND>(X, gz, A);
        if (ROLE == ROLE_IN && TVD >= 0) hC = half_courant_coef(w.u[CA], w.T, htod, A);
        publish(slotU, par, tidx, w.u);
        if (ROLE == ROLE_R1) {
            const double inv = rcp_fast(Xo[0]);
            double uo[ND];
#pragma unroll
            for (int c = 0; c < ND; ++c) uo[c] = Xo[1 + c] * inv;
            publish(slotU, par, tidx_o, uo);
        }
    };

    // One iteration.  ROLE and FAST are compile-time tags; PAR is the compile-time parity of j in the
    // unrolled FAST pair (-1: take it from j).
    auto body = [&](auto role_tag, auto fast_tag, auto par_tag, const int j) MC_INL {
        constexpr int ROLE = decltype(role_tag)::value;
        constexpr bool FAST = decltype(fast_tag)::value;
        constexpr int PAR = decltype(par_tag)::value;
        const int p1 = (PAR >= 0) ? (PAR ^ 1) : ((j + 1) & 1);   // parity of level j+1
        const int p2 = p1 ^ 1;                                   // parity of level j+2
        const unsigned o3 = FAST ? o3c : off_of(j + 3);
        const unsigned o0 = FAST ? o0c : off_of(j);
        const bool ex1 = FAST || exists(j + 1), ex2 = FAST || exists(j + 2), ex3 = FAST || exists(j + 3);
        const bool ld1 = FAST || (ex1 && (j + 1 >= l0 - 2));     // level j+1 is loaded (Xc, w1 valid)
        const bool ld2 = ex2;
        const bool start_wall1 = !FAST && WALL_M && (j + 1 == 0);     // level j+1 is the plate the march starts on
        const bool end_wall1 = !FAST && WALL_M && (j + 1 == n - 1);   // level j+1 is the plate the march ends on

        if (ROLE == ROLE_NONE) { level_sync(); return; }          // (AS: such rows have left already)

        // ZA (R19): the outer differences of levels j and j+1 use the height of the node's cell (a plate's half cell
        // carries the factor 2 of R10), the inner one-sided differences the spacing across the face, the TVD flux of
        // face (j, j+1) is weighted by h / dzc (R20).  Uniform grid: the launch constants.
        double cdt1 = cdt, hcdt1 = hcdt, hcdt0 = hcdt, cw1 = 2.0 * cdt, cw0 = cdt, htod2 = half_tod;
        double sF = 1.0, sB = 1.0, tw0 = 1.0, tw1 = 1.0;
        if (ZA) {
            const int k0 = kz(j), k1 = kz(j + 1), k2 = kz(j + 2);
            const double idc0 = zt_idc(A, k0), idc1 = zt_idc(A, k1), hf01 = zt_hf(A, min(k0, k1));
            cdt1 = (tau * dsgn) * idc1; hcdt1 = 0.5 * cdt1; hcdt0 = (0.5 * tau * dsgn) * idc0;
            cw1 = cdt1; cw0 = hcdt0;
            htod2 = (0.5 * tau) * zt_idc(A, k2);
            sF = zt_ihf(A, min(k1, k2)); sB = zt_ihf(A, min(k0, k1));
            tw0 = hf01 * idc0; tw1 = hf01 * idc1;
        }

        // (0) not AS: prefetch X(j+3) into registers and X(j+3+MC_MARCH3_L2PF) into L2;  AS: take X(j+2) out of its stage
        const bool ld3 = FAST || (ex3 && j + 3 <= l1 + 1);
        double Xq[NF], Xoq[ND + 1];
        if (AS) {
            stage_read(role_tag, ex2, j + 2, Xn, Xon);
        } else {
#if MC_MARCH3_L2PF > 0
            if (FAST) { if (j + 3 <= pf_last) prefetch_l2(o3 + (unsigned)MC_MARCH3_L2PF * sms); }
            else if (j + 3 + MC_MARCH3_L2PF <= l1 + 1 && exists(j + 3 + MC_MARCH3_L2PF)) prefetch_l2(off_of(j + 3 + MC_MARCH3_L2PF));
#endif
#pragma unroll
            for (int f = 0; f < NF; ++f) Xq[f] = Xn[f];
            if (ld3) load_at(o3, Xq);
#pragma unroll
            for (int f = 0; f <= ND; ++f) Xoq[f] = Xon[f];
            if (ROLE == ROLE_R1 && ld3 && has_outer) load_outer(o3 - off_base + off_base_o, Xoq);
        }

        // (1) W(j+2)
        Prim<ND> w2 = w1;
        double hC2 = 0.0, gz2 = 0.0;
        if (ld2) {
            gz2 = (FAST && Z_IS_ALPHA && !ZS) ? A.g * (kd2c * A.dz) : gz_of(j + 2);
            stage_W(role_tag, p2, gz2, htod2, Xn, Xon, w2, hC2);
        }

        if (ROLE == ROLE_WALLROW) {
            // a plate row of b (y-sweep): X^P = X and the output is X (R10); publish u^P = u of level j+1
            if (ld1) publish(slotP, p1, tidx, w1.u);
            level_sync();
            if (j >= l0 && owner) store_at(o0, H0, j);
#pragma unroll
            for (int f = 0; f < NF; ++f) { H0[f] = Xc[f]; Xc[f] = Xn[f]; if (!AS) Xn[f] = Xq[f]; }
            w1 = w2;
            if (FAST) { o3c += sms; o0c += sms; kd2c += dsgn; }
            it += 1;
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
                const double cD0 = ZA ? coef * tw0 : coef;           // (ZA: the R20 weights of levels j and j+1)
                cD1 = ZA ? coef * tw1 : coef;
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
                for (int c = 0; c < ND; ++c) du[c] = ZA ? (w2.u[c] - w1.u[c]) * sF : w2.u[c] - w1.u[c];
                cross(slotU, p1, dxa, dxc);
                flux<ND, CA>(Xc, w1, du, ZA ? (w2.T - w1.T) * sF : w2.T - w1.T, dxa, dxc, A, F1);
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
                if (Z_IS_ALPHA) {
                    XP[1 + CA] = fma(tsrc, Xc[0], XP[1 + CA]);
                    H1[1 + CA] = fma(0.5 * tsrc, Xc[0], H1[1 + CA]);
                }
            }
            wP1 = primitives<ND>(XP, gz1, A);
            if (start_wall1 || end_wall1) {
#pragma unroll
                for (int f = 0; f < NF; ++f) H1[f] = 0.5 * (XP[f] + Xc[f]);
            } else {
                if (Z_IS_ALPHA) H1[1 + CA] = fma(0.5 * tsrc, XP[0], H1[1 + CA]);   // + tau S(X^P)/2
            }
        }
        if (ld1) publish(slotP, p1, tidx, wP1.u);

        level_sync();

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
                    for (int c = 0; c < ND; ++c) du[c] = ZA ? (wP1.u[c] - uP0[c]) * sB : wP1.u[c] - uP0[c];
                    cross(slotP, p1, dxa, dxc);
                    flux<ND, CA>(XP, wP1, du, ZA ? (wP1.T - TP0) * sB : wP1.T - TP0, dxa, dxc, A, FP1);
                }
            }
            // (6) out(j): corrector (Eq. 32), average and TVD term (Eq. 33), plate values.  H0 already
            // holds + (tau/2dx) F^P(j), folded in when F^P(j) was computed.
            if (FAST || (j >= l0 && exists(j))) {
                double o[NF];
                if (!FAST && WALL_M && j == 0) {
                    plate(j, H0[0] - cw0 * FP1[0], o);    // 0.5 (2 tau/dz) (F^P(1) - F^P(0)); the plate's own mass flux is 0
                } else if (!FAST && WALL_M && j == n - 1) {
                    plate(j, H0[0], o);
                } else {
#pragma unroll
                    for (int f = 0; f < NF; ++f) o[f] = fma(-hcdt0, FP1[f], H0[f]);
                }
                if (owner) store_at(o0, o, j);
            }
#pragma unroll
            for (int f = 0; f < NF; ++f) { H1[f] = fma(hcdt1, FP1[f], H1[f]); d0[f] = d1[f]; }
            a0 = a1; b0 = b1; hC0 = hC1; hC1 = hC2;
#pragma unroll
            for (int c = 0; c < ND; ++c) uP0[c] = wP1.u[c];
            TP0 = wP1.T;
        }
        // (7) rotate the pipeline
#pragma unroll
        for (int f = 0; f < NF; ++f) { Xc[f] = Xn[f]; if (!AS) Xn[f] = Xq[f]; F0[f] = F1[f]; H0[f] = H1[f]; }
        if (!AS) {
#pragma unroll
            for (int f = 0; f <= ND; ++f) Xon[f] = Xoq[f];
        }
        w1 = w2; gz1 = gz2;
        if (FAST) { o3c += sms; o0c += sms; kd2c += dsgn; }
        it += 1;
    };

    // ---- the march -------------------------------------------------------------------------------
    auto march = [&](auto role_tag) MC_INL {
        using std::integral_constant;
        constexpr int ROLE = decltype(role_tag)::value;
        integral_constant<bool, false> slow;
        integral_constant<bool, true> fast;
        integral_constant<int, -1> par_any;
        int j = j_start;
        if (!AS && exists(j + 2)) {
            load(j + 2, Xn);
            if (ROLE == ROLE_R1 && has_outer) load_outer(off_of(j + 2) - off_base + off_base_o, Xon);
        }
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
    switch (role) {
    case ROLE_NONE: march(std::integral_constant<int, ROLE_NONE>()); break;
    case ROLE_WALLROW: march(std::integral_constant<int, WALL_B ? ROLE_WALLROW : ROLE_IN>()); break;
    case ROLE_R1: march(std::integral_constant<int, ROLE_R1>()); break;
    default: march(std::integral_constant<int, ROLE_IN>()); break;
    }
}

}  // namespace mc
