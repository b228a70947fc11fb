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
};

template <int ND>
MC_DEV void node_primitives(const PointArgs &P, long long n, int k, double (&X)[ND + 2], double (&u)[ND],
                            double &T)
{
#pragma unroll
    for (int f = 0; f < ND + 2; ++f) X[f] = P.X[(long long)f * P.N + n];
    double inv = 1.0 / X[0], ke = 0.0;
#pragma unroll
    for (int c = 0; c < ND; ++c) { u[c] = X[1 + c] * inv; ke += u[c] * u[c]; }
    T = (X[ND + 1] * inv - 0.5 * ke - P.g * ((double)k * P.dz)) * P.icv;       // Eq. 17
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
        double cs = sqrt(P.gamma * P.R * T);
#pragma unroll
        for (int c = 0; c < ND; ++c) s = fmax_nan(s, (fabs(u[c]) + cs) * P.inv_d[c]);
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
// ext[(k*gridDim.x + b)*3] = (max Mach, min rho, min T).
template <int ND>
MC_KERNEL void k_plane_partials(PointArgs P, double *partial, double *ext)
{
    constexpr int NF = ND + 2, NQ = 6 + NF;
    const int k = blockIdx.y;
    const double TA = 1.0 - P.D * ((double)k * P.dz);          // adiabatic profile, Eq. 19
    Acc acc[NQ];
#pragma unroll
    for (int q = 0; q < NQ; ++q) { acc[q].s = 0.0; acc[q].c = 0.0; }
    double mach = 0.0, rmin = INFINITY, tmin = INFINITY;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < P.plane;
         i += (long long)gridDim.x * blockDim.x) {
        long long n = (long long)k * P.plane + i;
        double X[NF], u[ND], T;
        node_primitives<ND>(P, n, k, X, u, T);
        double u2 = 0.0;
#pragma unroll
        for (int c = 0; c < ND; ++c) u2 += u[c] * u[c];
        double uz = u[ND - 1], rho = X[0];
        acc[DQ_T].add(T);
        acc[DQ_RHO].add(rho);
        acc[DQ_P].add(P.R * rho * T);
        acc[DQ_CONV].add(rho * uz * (T - TA));                  // rho u_z T_sa, Eq. 22
        acc[DQ_K].add(rho * uz * u2);                           // rho u_z u^2, Eq. 22
        acc[DQ_U2].add(u2);                                     // Eq. 26
#pragma unroll
        for (int f = 0; f < NF; ++f) acc[DQ_X0 + f].add(X[f]);
        mach = fmax(mach, sqrt(u2) / sqrt(P.gamma * P.R * T));
        rmin = fmin(rmin, rho);
        tmin = fmin(tmin, T);
    }
    // warp stage
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
        for (int q = 0; q < NQ; ++q) {
            double s2 = __shfl_xor_sync(0xffffffffu, acc[q].s, o);
            double c2 = __shfl_xor_sync(0xffffffffu, acc[q].c, o);
            acc[q].merge(s2, c2);
        }
        mach = fmax(mach, __shfl_xor_sync(0xffffffffu, mach, o));
        rmin = fmin(rmin, __shfl_xor_sync(0xffffffffu, rmin, o));
        tmin = fmin(tmin, __shfl_xor_sync(0xffffffffu, tmin, o));
    }
    // block stage
    __shared__ double sh[DIAG_THREADS / 32][2 * DQ_MAXQ + 3];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nwarp = blockDim.x >> 5;
    if (lane == 0) {
#pragma unroll
        for (int q = 0; q < NQ; ++q) { sh[warp][2 * q] = acc[q].s; sh[warp][2 * q + 1] = acc[q].c; }
        sh[warp][2 * DQ_MAXQ] = mach; sh[warp][2 * DQ_MAXQ + 1] = rmin; sh[warp][2 * DQ_MAXQ + 2] = tmin;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        const long long slot = (long long)k * gridDim.x + blockIdx.x;
        for (int q = 0; q < NQ; ++q) {
            Acc a; a.s = 0.0; a.c = 0.0;
            for (int w = 0; w < nwarp; ++w) a.merge(sh[w][2 * q], sh[w][2 * q + 1]);
            partial[slot * 2 * DQ_MAXQ + 2 * q] = a.s;
            partial[slot * 2 * DQ_MAXQ + 2 * q + 1] = a.c;
        }
        for (int w = 1; w < nwarp; ++w) {
            mach = fmax(mach, sh[w][2 * DQ_MAXQ]);
            rmin = fmin(rmin, sh[w][2 * DQ_MAXQ + 1]);
            tmin = fmin(tmin, sh[w][2 * DQ_MAXQ + 2]);
        }
        ext[slot * 3] = mach; ext[slot * 3 + 1] = rmin; ext[slot * 3 + 2] = tmin;
    }
}

struct DiagArgs {
    const double *partial, *ext;
    double *plane_sums;              // scratch nz * DQ_MAXQ
    double *out;                     // device: 19 doubles (layout of mc_tvd_diag) then T, rho, p profiles (3*nz)
    const Scalars *S;
    int nz, nblk, nq, walls;
    double nplane, dz, dxdy, eps, D, Ra, Pr;
};

// Plane sums -> means, trapezoid rule in z (R16), one-sided plate gradients, Eqs. 22-26.
MC_KERNEL void k_diag_finish(DiagArgs G)
{
    __shared__ double sh_ext[3][DIAG_THREADS];
    double mach = 0.0, rmin = INFINITY, tmin = INFINITY;
    for (int k = threadIdx.x; k < G.nz; k += blockDim.x) {
        for (int q = 0; q < G.nq; ++q) {
            Acc a; a.s = 0.0; a.c = 0.0;
            for (int b = 0; b < G.nblk; ++b) {
                const double *p = G.partial + ((long long)k * G.nblk + b) * 2 * DQ_MAXQ + 2 * q;
                a.merge(p[0], p[1]);
            }
            G.plane_sums[(long long)k * DQ_MAXQ + q] = a.s + a.c;
        }
        for (int b = 0; b < G.nblk; ++b) {
            const double *e = G.ext + ((long long)k * G.nblk + b) * 3;
            mach = fmax(mach, e[0]); rmin = fmin(rmin, e[1]); tmin = fmin(tmin, e[2]);
        }
    }
    sh_ext[0][threadIdx.x] = mach; sh_ext[1][threadIdx.x] = rmin; sh_ext[2][threadIdx.x] = tmin;
    __syncthreads();
    if (threadIdx.x != 0) return;
    for (int t = 1; t < (int)blockDim.x; ++t) {
        mach = fmax(mach, sh_ext[0][t]); rmin = fmin(rmin, sh_ext[1][t]); tmin = fmin(tmin, sh_ext[2][t]);
    }
    const int nz = G.nz, nf = G.nq - 6;
    double *Tp = G.out + 19, *rp = Tp + nz, *pp = rp + nz;
    double vol_w = 0.0, v_conv = 0.0, v_K = 0.0, v_u2 = 0.0, tot[5] = {0, 0, 0, 0, 0};
    for (int k = 0; k < nz; ++k) {
        const double *ps = G.plane_sums + (long long)k * DQ_MAXQ;
        double wk = G.dz * ((G.walls && (k == 0 || k == nz - 1)) ? 0.5 : 1.0);
        Tp[k] = ps[DQ_T] / G.nplane; rp[k] = ps[DQ_RHO] / G.nplane; pp[k] = ps[DQ_P] / G.nplane;
        vol_w += wk;
        v_conv += wk * (ps[DQ_CONV] / G.nplane);
        v_K += wk * (ps[DQ_K] / G.nplane);
        v_u2 += wk * (ps[DQ_U2] / G.nplane);
        for (int f = 0; f < nf; ++f) tot[f] += wk * G.dxdy * ps[DQ_X0 + f];
    }
    double *o = G.out;
    const double sRaPr = sqrt(G.Ra * G.Pr);
    o[0] = G.S->time; o[1] = G.S->dt; o[2] = __longlong_as_double(G.S->step);
    double nu_conv = sRaPr / G.eps * (v_conv / vol_w);                 // Eq. 22
    double nu_K = G.D * sRaPr / 2.0 * (v_K / vol_w);
    double nu0 = 0.0, nu1 = 0.0;
    if (nz >= 3) {                                                     // Eq. 23 with PAPER.md:309
        auto tsa = [&](int k) { return Tp[k] - (1.0 - G.D * ((double)k * G.dz)); };
        double g0 = (-3.0 * tsa(0) + 4.0 * tsa(1) - tsa(2)) / (2.0 * G.dz);
        double g1 = (3.0 * tsa(nz - 1) - 4.0 * tsa(nz - 2) + tsa(nz - 3)) / (2.0 * G.dz);
        nu0 = -g0 / G.eps; nu1 = -g1 / G.eps;
    }
    o[3] = nu0; o[4] = nu1; o[5] = 0.5 * (nu0 + nu1);                  // Eq. 24
    o[6] = 1.0 + nu_conv + nu_K; o[7] = nu_conv; o[8] = nu_K;
    double urms = sqrt(v_u2 / vol_w);
    o[9] = sqrt(G.Ra / G.Pr) * urms; o[10] = urms;                     // Eq. 26
    o[11] = tot[0]; o[12] = tot[1];
    o[13] = (nf == 5) ? tot[2] : 0.0;
    o[14] = tot[nf - 2]; o[15] = tot[nf - 1];
    o[16] = mach; o[17] = rmin; o[18] = tmin;
}

}  // namespace mc
