// flow_stats.cuh -- the flow statistics of the paper's Sec. 5-6 as reductions over the state:
//   * the z-momentum balance terms (Eqs. 40-43)
//         F_n = rho (u . grad) u_z,   F_p = -d_z p,   F_b = rho g,   F_v = d_i tau_iz = mu [lap u_z + (1 + lambda) d_z div u]
//     (tau_ij of Eq. 18) as volume means and root-mean-squares, and <F_b> - <F_p>;
//   * r = K_e / I_e = (rho u^2 / 2) / (rho C_v T) at every node: its largest value, the largest local
//     Mach number (Mach^2 = 2 r / (gamma (gamma - 1))) and its histogram (Fig. 5);
//   * the normalised correlation C = <rho u_z T_sa> / sqrt(<(rho u_z)^2> <T_sa^2>) of Eq. 49 with
//     T_sa = T - (1 - D z) (Eq. 19): three more sums over EVERY node, weighted as the <.>_V of Eq. 22 (cell heights,
//     half cells at the plates: R16 / R19), so that Nu_conv = sqrt(Ra Pr) / eps <rho u_z T_sa>.
// Reading R21 (the paper does not say how it differences its post-processing quantities): second-order
// central differences on the node's 3 x 3 x 3 neighbourhood -- first derivatives over the distance between the two
// neighbours, second and mixed derivatives compact -- at the interior nodes k = 1 .. nz-2 (every node when z is
// periodic), averaged with the cell heights (R16 / R19).  Histogram bin of r > 0: 4 (floor(log2 r) + 32) + (top two
// mantissa bits), clamped to [0, 127], read off the bit pattern; r = 0 in bin 0.
// Not on the step's hot path: one pass over the state per sample, neighbours read through L1 / L2.
#pragma once
#include "mc_common.cuh"
#include "reduce_kernels.cuh"

namespace mc {

constexpr int FLOW_BINS = 128;
constexpr int FLOW_NQ = 11;            // sums of F_n, F_p, F_b, F_v and of their squares; of m_z T_sa, m_z^2, T_sa^2 (Eq. 49)
constexpr int FLOW_NF = 8;             // the first FLOW_NF run over the interior cells, the rest over every node
constexpr int FLOW_NOUT = 16;          // layout of mc_tvd_forces

struct FlowArgs {
    PointArgs P;
    int nx, ny, walls;
    double mu, lam, cv;
    double inv_2dx, inv_2dy, inv_dx2, inv_dy2;
};

MC_DEV int flow_hist_bin(double r)
{
    if (!(r > 0.0)) return 0;
    const long long b = (long long)((unsigned long long)__double_as_longlong(r) >> 50) - 4ll * (1023 - 32);
    return b < 0 ? 0 : (b > FLOW_BINS - 1 ? FLOW_BINS - 1 : (int)b);
}

// grid (blocks per plane, nz).  partial[(k * gridDim.x + b) * FLOW_NQ + q]; ext[k * gridDim.x + b] = max r;
// hist[FLOW_BINS] accumulates with integer atomics (exact in any order).
template <int ND>
MC_KERNEL void k_flow_partials(FlowArgs G, double *partial, double *ext, unsigned long long *hist)
{
    constexpr int NF = ND + 2;
    const PointArgs &P = G.P;
    __shared__ unsigned int sh_hist[FLOW_BINS];
    __shared__ double sh[DIAG_THREADS / 32][FLOW_NQ + 1];
    for (int i = threadIdx.x; i < FLOW_BINS; i += blockDim.x) sh_hist[i] = 0u;
    __syncthreads();
    const int k = blockIdx.y, nz = P.nz;
    const bool interior = G.walls ? (k >= 1 && k <= nz - 2) : true;
    const int kp = (k + 1 < nz) ? k + 1 : (G.walls ? k : 0), km = (k >= 1) ? k - 1 : (G.walls ? k : nz - 1);
    // spacings along z around level k: faces below and above
    const double hm = P.zt ? P.zt[4 * nz + (k >= 1 ? k - 1 : 0)] : P.dz, hp = P.zt ? P.zt[4 * nz + (k + 1 < nz ? k : nz - 2)] : P.dz;
    const double inv_2h = 1.0 / (hp + hm);
    const double gz = point_gz(P, k), gzp = point_gz(P, kp), gzm = point_gz(P, km);
    const double TA = 1.0 - P.D * point_z(P, k);                               // Eq. 19
    auto fld = [&](int f, long long n) MC_INL { return P.X[(long long)f * P.N + n]; };
    auto vel = [&](int c, long long n) MC_INL { return fld(1 + c, n) / fld(0, n); };
    auto pres = [&](long long n, double gzn) MC_INL {
        const double rho = fld(0, n), inv = 1.0 / rho;
        double ke = 0.0;
#pragma unroll
        for (int c = 0; c < ND; ++c) { const double u = fld(1 + c, n) * inv; ke += u * u; }
        return P.R * rho * ((fld(NF - 1, n) * inv - 0.5 * ke - gzn) * P.icv);
    };
    double acc[FLOW_NQ];
#pragma unroll
    for (int q = 0; q < FLOW_NQ; ++q) acc[q] = 0.0;
    double rmax = 0.0;
    constexpr int CZ = ND - 1;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < P.plane; i += (long long)gridDim.x * blockDim.x) {
        const int ix = (int)(i % G.nx), iy = (int)(i / G.nx);
        const long long n = (long long)k * P.plane + i;
        const double rho = fld(0, n), inv = 1.0 / rho;
        double u[ND], u2 = 0.0;
#pragma unroll
        for (int c = 0; c < ND; ++c) { u[c] = fld(1 + c, n) * inv; u2 += u[c] * u[c]; }
        const double T = (fld(NF - 1, n) * inv - 0.5 * u2 - gz) * P.icv;
        const double r = (0.5 * u2) / (G.cv * T);
        rmax = fmax(rmax, r);
        atomicAdd(&sh_hist[flow_hist_bin(r)], 1u);
        {
            const double mz = fld(1 + CZ, n), Tsa = T - TA;                    // Eq. 49: rho u_z is the conserved momentum
            acc[8] += mz * Tsa; acc[9] += mz * mz; acc[10] += Tsa * Tsa;
        }
        if (!interior) continue;
        const long long row = (long long)k * P.plane + (long long)iy * G.nx;
        const int ixp = (ix + 1 < G.nx) ? ix + 1 : 0, ixm = (ix >= 1) ? ix - 1 : G.nx - 1;
        const long long xp = row + ixp, xm = row + ixm;
        const long long dzp = (long long)(kp - k) * P.plane, dzm = (long long)(km - k) * P.plane;
        const double uz0 = u[CZ], uzxp = vel(CZ, xp), uzxm = vel(CZ, xm), uzzp = vel(CZ, n + dzp), uzzm = vel(CZ, n + dzm);
        double adv = u[0] * ((uzxp - uzxm) * G.inv_2dx) + uz0 * ((uzzp - uzzm) * inv_2h);
        double lap = (uzxp - 2.0 * uz0 + uzxm) * G.inv_dx2;
        // mixed derivative d_z d_x u_x: central difference along z of the central x-differences
        double mixed = ((vel(0, xp + dzp) - vel(0, xm + dzp)) * G.inv_2dx - (vel(0, xp + dzm) - vel(0, xm + dzm)) * G.inv_2dx) * inv_2h;
        if (ND == 3) {
            const int iyp = (iy + 1 < G.ny) ? iy + 1 : 0, iym = (iy >= 1) ? iy - 1 : G.ny - 1;
            const long long yp = (long long)k * P.plane + (long long)iyp * G.nx + ix, ym = (long long)k * P.plane + (long long)iym * G.nx + ix;
            const double uzyp = vel(CZ, yp), uzym = vel(CZ, ym);
            adv += u[ND == 3 ? 1 : 0] * ((uzyp - uzym) * G.inv_2dy);
            lap += (uzyp - 2.0 * uz0 + uzym) * G.inv_dy2;
            mixed += ((vel(1, yp + dzp) - vel(1, ym + dzp)) * G.inv_2dy - (vel(1, yp + dzm) - vel(1, ym + dzm)) * G.inv_2dy) * inv_2h;
        }
        const double dzz = 2.0 * ((uzzp - uz0) / hp - (uz0 - uzzm) / hm) * inv_2h;
        double F[4];
        F[0] = rho * adv;                                                    // Eq. 40
        F[1] = -(pres(n + dzp, gzp) - pres(n + dzm, gzm)) * inv_2h;          // Eq. 41
        F[2] = rho * P.g;                                                    // Eq. 42
        F[3] = G.mu * (lap + dzz + (1.0 + G.lam) * (mixed + dzz));           // Eq. 43 with Eq. 18
#pragma unroll
        for (int t = 0; t < 4; ++t) { acc[t] += F[t]; acc[4 + t] += F[t] * F[t]; }
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
        for (int q = 0; q < FLOW_NQ; ++q) acc[q] += __shfl_xor_sync(0xffffffffu, acc[q], o);
        rmax = fmax(rmax, __shfl_xor_sync(0xffffffffu, rmax, o));
    }
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31, nwarp = blockDim.x >> 5;
    if (lane == 0) {
#pragma unroll
        for (int q = 0; q < FLOW_NQ; ++q) sh[warp][q] = acc[q];
        sh[warp][FLOW_NQ] = rmax;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        const long long slot = (long long)k * gridDim.x + blockIdx.x;
        for (int q = 0; q < FLOW_NQ; ++q) {
            double t = 0.0;
            for (int w = 0; w < nwarp; ++w) t += sh[w][q];
            partial[slot * FLOW_NQ + q] = t;
        }
        for (int w = 1; w < nwarp; ++w) rmax = fmax(rmax, sh[w][FLOW_NQ]);
        ext[slot] = rmax;
    }
    for (int i = threadIdx.x; i < FLOW_BINS; i += blockDim.x)
        if (sh_hist[i]) atomicAdd(&hist[i], (unsigned long long)sh_hist[i]);
}

// plane partials -> the 16 numbers of mc_tvd_forces in out[0..16) (one block)
MC_KERNEL void k_flow_finish(FlowArgs G, const double *partial, const double *ext, int nblk, double gamma, double *out)
{
    __shared__ double sh[FLOW_NQ + 3][DIAG_THREADS];
    const PointArgs &P = G.P;
    const int nz = P.nz;
    double v[FLOW_NQ + 2], rmax = 0.0;            // [FLOW_NQ]: interior volume, [FLOW_NQ + 1]: whole volume
#pragma unroll
    for (int q = 0; q <= FLOW_NQ + 1; ++q) v[q] = 0.0;
    const double nplane = (double)G.nx * (double)G.ny;
    for (int k = threadIdx.x; k < nz; k += blockDim.x) {
        for (int b = 0; b < nblk; ++b) rmax = fmax(rmax, ext[(long long)k * nblk + b]);
        const bool plate = G.walls && (k == 0 || k == nz - 1);
        // cell height; a plate node owns half the adjacent spacing (the table holds that already)
        const double dzc = P.zt ? 1.0 / P.zt[2 * nz + k] : (plate ? 0.5 * P.dz : P.dz);
        const double wk = dzc / nplane;
#pragma unroll
        for (int q = 0; q < FLOW_NQ; ++q) {
            if (plate && q < FLOW_NF) continue;                     // the force balance runs over the interior cells
            double t = 0.0;
            for (int b = 0; b < nblk; ++b) t += partial[((long long)k * nblk + b) * FLOW_NQ + q];
            v[q] += wk * t;
        }
        if (!plate) v[FLOW_NQ] += dzc;
        v[FLOW_NQ + 1] += dzc;
    }
#pragma unroll
    for (int q = 0; q <= FLOW_NQ + 1; ++q) sh[q][threadIdx.x] = v[q];
    sh[FLOW_NQ + 2][threadIdx.x] = rmax;
    __syncthreads();
    for (int o = blockDim.x >> 1; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) {
#pragma unroll
            for (int q = 0; q <= FLOW_NQ + 1; ++q) sh[q][threadIdx.x] += sh[q][threadIdx.x + o];
            sh[FLOW_NQ + 2][threadIdx.x] = fmax(sh[FLOW_NQ + 2][threadIdx.x], sh[FLOW_NQ + 2][threadIdx.x + o]);
        }
        __syncthreads();
    }
    if (threadIdx.x != 0) return;
    const double vol = sh[FLOW_NQ][0];
    for (int t = 0; t < 4; ++t) { out[t] = sh[t][0] / vol; out[4 + t] = sqrt(sh[4 + t][0] / vol); }
    out[8] = out[2] - out[1];                                       // <F_b> - <F_p>
    out[10] = sh[FLOW_NQ + 2][0];
    out[9] = sqrt(2.0 * out[10] / (gamma * (gamma - 1.0)));
    out[11] = vol;
    const double vol_all = sh[FLOW_NQ + 1][0];
    for (int t = 0; t < 3; ++t) out[13 + t] = sh[FLOW_NF + t][0] / vol_all;
    out[12] = out[13] / sqrt(out[14] * out[15]);                    // Eq. 49 (NaN for a fluid at rest: 0 / 0)
}

// Running time averages of the flow statistics (weights as in k_stats_accumulate: time since the previous sample).
// acc: [0..4) weighted means, [4..8) weighted mean SQUARES (of the rms values), [8] <F_b - F_p>, [9] max Mach, [10] max r,
// [11] weight, [13..16) the three averages of Eq. 49 (C itself is formed from their time averages when they are read:
// the paper's <.> there is <.>_{V,t}).  hist_acc += hist (counts of every sample), then hist is cleared for the next sample.
MC_KERNEL void k_flow_accumulate(double *acc, const double *cur, const double *st, const Scalars *S,
                                 unsigned long long *hist_acc, unsigned long long *hist)
{
    const double w = S->time - st[1];              // st[1] = time of the previous sample (updated by k_stats_accumulate afterwards)
    const int t = threadIdx.x;
    if (t < 4) acc[t] += w * cur[t];
    else if (t < 8) acc[t] += w * (cur[t] * cur[t]);
    else if (t < 11) acc[t] += w * cur[t];
    else if (t == 11) acc[11] += w;
    else if (t >= 13 && t < 16) acc[t] += w * cur[t];
    for (int i = t; i < FLOW_BINS; i += blockDim.x) { hist_acc[i] += hist[i]; hist[i] = 0ull; }
}

}  // namespace mc
