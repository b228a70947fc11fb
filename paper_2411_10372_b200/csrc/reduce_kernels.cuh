// reduce_kernels.cuh -- the reductions of the hot path: the CFL max-reduction (R12; the
// paper names only a "local Courant number") and the Nusselt / Reynolds / profile
// diagnostics (Eqs. 22-26).  Warp shuffles, then one shared-memory stage per block.
#pragma once
#include "mc_common.cuh"

namespace mc {

// Device-resident scalars of a handle (first 64 bytes of the scalar block in the workspace).
struct Scalars {
    double dt;                       // dt the next step uses
    double time;                     // simulated time
    unsigned long long smax_bits;    // running max of (|u_a| + c_s)/dx_a, as a bit pattern
    long long step;                  // steps taken
    double cfl, fixed_dt;
};

struct PointArgs {                   // what a pointwise pass over the state needs
    const double *X;
    long long N, plane;              // nodes per field, nodes per z-plane
    int nz;
    double dz, g, icv, R, gamma, D;
    double inv_d[3];
    const double *zt;                // non-uniform z grid: the tables of SweepArgs::zt, or null
    // slab decomposition (diagnostics only): sum the nodes whose index along own_axis (0: x, 1: y; -1: all) lies in
    // [own_lo, own_hi) -- the rows a rank owns, without its halo copies
    int own_axis, own_lo, own_hi, nx;
};

MC_DEV double point_z(const PointArgs &P, int k) { return P.zt ? P.zt[k] : (double)k * P.dz; }
MC_DEV double point_gz(const PointArgs &P, int k) { return P.zt ? P.zt[P.nz + k] : P.g * ((double)k * P.dz); }

template <int ND>
MC_DEV void node_primitives(const PointArgs &P, long long n, int k, double (&X)[ND + 2], double (&u)[ND],
                            double &T)
{
#pragma unroll
    for (int f = 0; f < ND + 2; ++f) X[f] = P.X[(long long)f * P.N + n];
    // the same sequence of roundings as cfl_speed (mc_common.cuh), so that this reduction and the one fused into the
    // step's last operator give the same dt bit for bit (the slab driver uses this one every step)
    double inv = rcp(X[0]), ke = 0.0;
#pragma unroll
    for (int c = 0; c < ND; ++c) { u[c] = X[1 + c] * inv; ke = fma(u[c], u[c], ke); }
    T = (fma(-0.5, ke, X[ND + 1] * inv) - point_gz(P, k)) * P.icv;             // Eq. 17
}

// s = max over nodes and directions of (|u_a| + c_s)/dx_a (R12); NaN if rho or T is not positive.
template <int ND>
MC_KERNEL void k_max_speed(PointArgs P, unsigned long long *smax_bits)
{
    double smax = 0.0;
    for (long long n = (long long)blockIdx.x * blockDim.x + threadIdx.x; n < P.N;
         n += (long long)gridDim.x * blockDim.x) {
        int k = (int)(n / P.plane);
        double X[ND + 2], u[ND], T;
        node_primitives<ND>(P, n, k, X, u, T);
        double s = 0.0;
        if (!(X[0] > 0.0) || !(T > 0.0)) s = NAN;
        double cs = sqrt_pos((P.gamma * P.R) * T);
        // non-uniform z (R19): the cell height; a plate node takes the full adjacent spacing
        const double idz = P.zt ? P.zt[2 * P.nz + k] * ((k == 0 || k == P.nz - 1) ? 0.5 : 1.0) : P.inv_d[ND - 1];
#pragma unroll
        for (int c = 0; c < ND; ++c) s = fmax_nan(s, (fabs(u[c]) + cs) * (c == ND - 1 ? idz : P.inv_d[c]));
        smax = fmax_nan(smax, s);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) smax = fmax_nan(smax, __shfl_xor_sync(0xffffffffu, smax, o));
    if ((threadIdx.x & 31) == 0) atomic_max_bits(smax_bits, smax);
}

// After a step (advance = 1) or at init (advance = 0): time += dt, step += 1; dt = fixed_dt or
// cfl / s; reset the running max.
MC_KERNEL void k_dt_update(Scalars *S, int advance)
{
    if (threadIdx.x == 0 && blockIdx.x == 0) {
        if (advance) { S->time += S->dt; S->step += 1; }
        double s = __longlong_as_double((long long)S->smax_bits);
        S->dt = (S->fixed_dt > 0.0) ? S->fixed_dt : S->cfl / s;
        S->smax_bits = 0ull;
    }
}

// ---------------------------------------------------------------------------------------------
// diagnostics
// ---------------------------------------------------------------------------------------------
// Compensated (two-sum) accumulator: the plane means of T enter Nu through a one-sided difference
// divided by dz (Eq. 23), which amplifies their rounding error by ~1/(eps dz); DESIGN.md "Tolerances".
struct Acc {
    double s, c;
    MC_DEV void add(double x)
    {
        double t = s + x;
        c += (fabs(s) >= fabs(x)) ? ((s - t) + x) : ((x - t) + s);
        s = t;
    }
    MC_DEV void merge(double s2, double c2) { add(s2); c += c2; }
};

constexpr int DQ_T = 0, DQ_RHO = 1, DQ_P = 2, DQ_CONV = 3, DQ_K = 4, DQ_U2 = 5, DQ_X0 = 6;  // then nf conserved sums
constexpr int DQ_MAXQ = 11;            // 6 + nf (nf <= 5)
constexpr int DIAG_THREADS = 256;

// Per-plane partial sums: grid (blocks_per_plane, nz).  partial[(k*gridDim.x + b)*2*DQ_MAXQ + 2*q] = (s, c);
// ext[(k*gridDim.x + b)*3] = (max Mach^2, min rho, min T).
// Only the sum of T is compensated (two-sum): its plane means enter Nu through a one-sided difference divided
// by eps dz (Eq. 23), which amplifies their rounding error by ~1/(eps dz) (4e4 on C3).  The other sums are
// plain: a thread adds <= a few hundred terms and the rest is a tree, far inside their 1e-12 / 1e-13 tolerances;
// their `c` slots are written as 0.  The pass is then HBM-bound instead of fp64-bound.
template <int ND>
MC_KERNEL void k_plane_partials(PointArgs P, double *partial, double *ext)
{
    constexpr int NF = ND + 2, NQ = 6 + NF;
    const int k = blockIdx.y;
    const double TA = 1.0 - P.D * point_z(P, k);               // adiabatic profile, Eq. 19
    const double gz = point_gz(P, k);
    const double igR = 1.0 / (P.gamma * P.R);
    Acc accT; accT.s = 0.0; accT.c = 0.0;
    double acc[NQ];
#pragma unroll
    for (int q = 0; q < NQ; ++q) acc[q] = 0.0;
    double mach2 = 0.0, rmin = INFINITY, tmin = INFINITY;
    const double *base = P.X + (long long)k * P.plane;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < P.plane;
         i += (long long)gridDim.x * blockDim.x) {
        if (P.own_axis >= 0) {
            const int idx = (P.own_axis == 0) ? (int)(i % P.nx) : (int)(i / P.nx);
            if (idx < P.own_lo || idx >= P.own_hi) continue;
        }
        double X[NF], u[ND];
#pragma unroll
        for (int f = 0; f < NF; ++f) X[f] = base[(long long)f * P.N + i];
        const double rho = X[0], inv = rcp(rho);
        double u2 = 0.0;
#pragma unroll
        for (int c = 0; c < ND; ++c) { u[c] = X[1 + c] * inv; u2 = fma(u[c], u[c], u2); }
        const double T = (X[NF - 1] * inv - 0.5 * u2 - gz) * P.icv;          // Eq. 17
        const double muz = X[NF - 2];                                        // rho u_z
        accT.add(T);
        acc[DQ_RHO] += rho;
        acc[DQ_P] += P.R * rho * T;
        acc[DQ_CONV] += muz * (T - TA);                                      // rho u_z T_sa, Eq. 22
        acc[DQ_K] += muz * u2;                                               // rho u_z u^2, Eq. 22
        acc[DQ_U2] += u2;                                                    // Eq. 26
#pragma unroll
        for (int f = 0; f < NF; ++f) acc[DQ_X0 + f] += X[f];
        mach2 = fmax(mach2, (u2 * igR) * rcp(T));                            // Mach^2 = u^2 / (gamma R T)
        rmin = fmin(rmin, rho);
        tmin = fmin(tmin, T);
    }
    // warp stage
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        const double s2 = __shfl_xor_sync(0xffffffffu, accT.s, o);
        const double c2 = __shfl_xor_sync(0xffffffffu, accT.c, o);
        accT.merge(s2, c2);
#pragma unroll
        for (int q = 1; q < NQ; ++q) acc[q] += __shfl_xor_sync(0xffffffffu, acc[q], o);
        mach2 = fmax(mach2, __shfl_xor_sync(0xffffffffu, mach2, o));
        rmin = fmin(rmin, __shfl_xor_sync(0xffffffffu, rmin, o));
        tmin = fmin(tmin, __shfl_xor_sync(0xffffffffu, tmin, o));
    }
    // block stage
    __shared__ double sh[DIAG_THREADS / 32][DQ_MAXQ + 4];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nwarp = blockDim.x >> 5;
    if (lane == 0) {
        sh[warp][0] = accT.s; sh[warp][DQ_MAXQ] = accT.c;
#pragma unroll
        for (int q = 1; q < NQ; ++q) sh[warp][q] = acc[q];
        sh[warp][DQ_MAXQ + 1] = mach2; sh[warp][DQ_MAXQ + 2] = rmin; sh[warp][DQ_MAXQ + 3] = tmin;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        const long long slot = (long long)k * gridDim.x + blockIdx.x;
        Acc a; a.s = 0.0; a.c = 0.0;
        for (int w = 0; w < nwarp; ++w) a.merge(sh[w][0], sh[w][DQ_MAXQ]);
        partial[slot * 2 * DQ_MAXQ] = a.s;
        partial[slot * 2 * DQ_MAXQ + 1] = a.c;
        for (int q = 1; q < NQ; ++q) {
            double t = 0.0;
            for (int w = 0; w < nwarp; ++w) t += sh[w][q];
            partial[slot * 2 * DQ_MAXQ + 2 * q] = t;
            partial[slot * 2 * DQ_MAXQ + 2 * q + 1] = 0.0;
        }
        for (int w = 1; w < nwarp; ++w) {
            mach2 = fmax(mach2, sh[w][DQ_MAXQ + 1]);
            rmin = fmin(rmin, sh[w][DQ_MAXQ + 2]);
            tmin = fmin(tmin, sh[w][DQ_MAXQ + 3]);
        }
        ext[slot * 3] = mach2; ext[slot * 3 + 1] = rmin; ext[slot * 3 + 2] = tmin;
    }
}

struct DiagArgs {
    const double *partial, *ext;
    double *plane_sums;              // scratch nz * DQ_MAXQ
    double *out;                     // device: 19 doubles (layout of mc_tvd_diag) then T, rho, p profiles (3*nz)
    const Scalars *S;
    int nz, nblk, nq, walls;
    double nplane, dz, dxdy, eps, D, Ra, Pr;
    const double *zt;                // non-uniform z grid: the tables of SweepArgs::zt, or null
};

// Stage 2: the partial sums of one z plane -> plane_sums[k][q] (one warp per plane, lane q walks the plane's
// blocks in order) and the plane's extrema -> plane_ext[k][3].
MC_KERNEL void k_diag_planes(DiagArgs G, double *plane_ext)
{
    const int k = (int)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (k >= G.nz) return;
    if (lane < G.nq) {
        Acc a; a.s = 0.0; a.c = 0.0;
        for (int b = 0; b < G.nblk; ++b) {
            const double *p = G.partial + ((long long)k * G.nblk + b) * 2 * DQ_MAXQ + 2 * lane;
            a.merge(p[0], p[1]);
        }
        G.plane_sums[(long long)k * DQ_MAXQ + lane] = a.s + a.c;
    } else if (lane < G.nq + 3) {
        const int e = lane - G.nq;                       // 0: max Mach^2, 1: min rho, 2: min T
        double v = (e == 0) ? 0.0 : INFINITY;
        for (int b = 0; b < G.nblk; ++b) {
            const double x = G.ext[((long long)k * G.nblk + b) * 3 + e];
            v = (e == 0) ? fmax(v, x) : fmin(v, x);
        }
        plane_ext[(long long)k * 3 + e] = v;
    }
}

// Stage 3: plane sums -> means, trapezoid rule in z (R16), one-sided plate gradients,
// Eqs. 22-26.  One block; the z sums are a strided per-thread sum followed by a shared-memory tree.
MC_KERNEL void k_diag_finish(DiagArgs G, const double *plane_ext)
{
    constexpr int NV = 9;                                // vol_w, conv, K, u2, totals[5]
    __shared__ double sh[NV + 3][DIAG_THREADS];
    const int nz = G.nz, nf = G.nq - 6;
    double *Tp = G.out + 19, *rp = Tp + nz, *pp = rp + nz;
    double v[NV], mach2 = 0.0, rmin = INFINITY, tmin = INFINITY;
#pragma unroll
    for (int i = 0; i < NV; ++i) v[i] = 0.0;
    for (int k = threadIdx.x; k < nz; k += blockDim.x) {
        const double *ps = G.plane_sums + (long long)k * DQ_MAXQ;
        // trapezoid weight = the height of the cell the node owns (R16; R19 on the non-uniform grid)
        const double wk = G.zt ? 1.0 / G.zt[2 * nz + k] : G.dz * ((G.walls && (k == 0 || k == nz - 1)) ? 0.5 : 1.0);
        Tp[k] = ps[DQ_T] / G.nplane; rp[k] = ps[DQ_RHO] / G.nplane; pp[k] = ps[DQ_P] / G.nplane;
        v[0] += wk;
        v[1] += wk * (ps[DQ_CONV] / G.nplane);
        v[2] += wk * (ps[DQ_K] / G.nplane);
        v[3] += wk * (ps[DQ_U2] / G.nplane);
        for (int f = 0; f < nf; ++f) v[4 + f] += wk * G.dxdy * ps[DQ_X0 + f];
        mach2 = fmax(mach2, plane_ext[(long long)k * 3]);
        rmin = fmin(rmin, plane_ext[(long long)k * 3 + 1]);
        tmin = fmin(tmin, plane_ext[(long long)k * 3 + 2]);
    }
#pragma unroll
    for (int i = 0; i < NV; ++i) sh[i][threadIdx.x] = v[i];
    sh[NV][threadIdx.x] = mach2; sh[NV + 1][threadIdx.x] = rmin; sh[NV + 2][threadIdx.x] = tmin;
    __syncthreads();
    for (int o = blockDim.x >> 1; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) {
#pragma unroll
            for (int i = 0; i < NV; ++i) sh[i][threadIdx.x] += sh[i][threadIdx.x + o];
            sh[NV][threadIdx.x] = fmax(sh[NV][threadIdx.x], sh[NV][threadIdx.x + o]);
            sh[NV + 1][threadIdx.x] = fmin(sh[NV + 1][threadIdx.x], sh[NV + 1][threadIdx.x + o]);
            sh[NV + 2][threadIdx.x] = fmin(sh[NV + 2][threadIdx.x], sh[NV + 2][threadIdx.x + o]);
        }
        __syncthreads();
    }
    if (threadIdx.x != 0) return;
    const double vol_w = sh[0][0], v_conv = sh[1][0], v_K = sh[2][0], v_u2 = sh[3][0];
    double tot[5];
    for (int f = 0; f < 5; ++f) tot[f] = sh[4 + f][0];
    double *o = G.out;
    const double sRaPr = sqrt(G.Ra * G.Pr);
    o[0] = G.S->time; o[1] = G.S->dt; o[2] = __longlong_as_double(G.S->step);
    double nu_conv = sRaPr / G.eps * (v_conv / vol_w);                 // Eq. 22
    double nu_K = G.D * sRaPr / 2.0 * (v_K / vol_w);
    double nu0 = 0.0, nu1 = 0.0;
    if (nz >= 3) {                                                     // Eq. 23 with PAPER.md:309
        // (Tp[0..2] and Tp[nz-3..nz-1] were written by other threads of this block before the barriers above)
        auto zk = [&](int k) { return G.zt ? G.zt[k] : (double)k * G.dz; };
        auto tsa = [&](int k) { return Tp[k] - (1.0 - G.D * zk(k)); };
        double g0 = (-3.0 * tsa(0) + 4.0 * tsa(1) - tsa(2)) / (2.0 * G.dz);
        double g1 = (3.0 * tsa(nz - 1) - 4.0 * tsa(nz - 2) + tsa(nz - 3)) / (2.0 * G.dz);
        if (G.zt) {
            // derivative at the plate of the quadratic through the plate node and its two neighbours at distances
            // h1 < h2: weights (-(b + c), b, c), b = h2 / (h1 (h2 - h1)), c = -h1 / (h2 (h2 - h1))
            double h1 = zk(1) - zk(0), h2 = zk(2) - zk(0);
            double b = h2 / (h1 * (h2 - h1)), c = -h1 / (h2 * (h2 - h1));
            g0 = -(b + c) * tsa(0) + b * tsa(1) + c * tsa(2);
            h1 = zk(nz - 1) - zk(nz - 2); h2 = zk(nz - 1) - zk(nz - 3);
            b = h2 / (h1 * (h2 - h1)); c = -h1 / (h2 * (h2 - h1));
            g1 = (b + c) * tsa(nz - 1) - b * tsa(nz - 2) - c * tsa(nz - 3);
        }
        nu0 = -g0 / G.eps; nu1 = -g1 / G.eps;
    }
    o[3] = nu0; o[4] = nu1; o[5] = 0.5 * (nu0 + nu1);                  // Eq. 24
    o[6] = 1.0 + nu_conv + nu_K; o[7] = nu_conv; o[8] = nu_K;
    double urms = sqrt(v_u2 / vol_w);
    o[9] = sqrt(G.Ra / G.Pr) * urms; o[10] = urms;                     // Eq. 26
    o[11] = tot[0]; o[12] = tot[1];
    o[13] = (nf == 5) ? tot[2] : 0.0;
    o[14] = tot[nf - 2]; o[15] = tot[nf - 1];
    o[16] = sqrt(sh[NV][0]); o[17] = sh[NV + 1][0]; o[18] = sh[NV + 2][0];   // the partials carry Mach^2
}

// ---------------------------------------------------------------------------------------------
// running time averages of the diagnostics (include/mc_tvd.h mc_tvd_stats)
// ---------------------------------------------------------------------------------------------
// Device block: [0] t_begin, [1] t_last, [2] weight, [3] samples, [4..13] weighted sums in the order of
// mc_tvd_stats from nu_bottom on, [16 .. 16 + 3 nz) weighted profile sums (T, rho, p).
constexpr int ST_HEAD = 16, ST_NSUM = 10;

MC_KERNEL void k_stats_reset(double *st, const Scalars *S, int nz)
{
    for (int i = threadIdx.x; i < ST_HEAD + 3 * nz; i += blockDim.x) st[i] = 0.0;
    __syncthreads();
    if (threadIdx.x == 0) { st[0] = S->time; st[1] = S->time; }
}

// Add the diagnostics block `diag` (layout of k_diag_finish: 19 scalars, then the T, rho, p profiles) with the weight
// w = time - t_last.
MC_KERNEL void k_stats_accumulate(double *st, const double *diag, const Scalars *S, int nz)
{
    const double w = S->time - st[1];
    // mc_tvd_diag order: 3 nu_bottom, 4 nu_top, 5 nu_bar, 6 nu_bulk, 7 nu_conv, 8 nu_K, 9 re, 10 u_rms
    if (threadIdx.x < 8) st[4 + threadIdx.x] += w * diag[3 + threadIdx.x];
    if (threadIdx.x == 8) st[12] += w * (diag[5] * diag[5]);
    if (threadIdx.x == 9) st[13] += w * (diag[9] * diag[9]);
    for (int i = threadIdx.x; i < 3 * nz; i += blockDim.x) st[ST_HEAD + i] += w * diag[19 + i];
    __syncthreads();
    if (threadIdx.x == 0) { st[2] += w; st[3] += 1.0; st[1] = S->time; }
}

// out: 4 header values (t_begin, t_end, weight, samples), the 10 averages, then the 3 nz averaged profile values
MC_KERNEL void k_stats_finish(const double *st, double *out, int nz)
{
    const double iw = 1.0 / st[2];
    if (threadIdx.x == 0) { out[0] = st[0]; out[1] = st[1]; out[2] = st[2]; out[3] = st[3]; }
    if (threadIdx.x < ST_NSUM) out[4 + threadIdx.x] = st[4 + threadIdx.x] * iw;
    for (int i = threadIdx.x; i < 3 * nz; i += blockDim.x) out[4 + ST_NSUM + i] = st[ST_HEAD + i] * iw;
}

}  // namespace mc
