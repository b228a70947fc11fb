// mc_tvd.cu -- the C ABI of libmc_tvd.so (include/mc_tvd.h): host-side validation, derived
// coefficients, launch geometry and the per-step launch list.  All arithmetic of the path runs in the
// kernels of sweep_march.cuh, sweep_lane.cuh and reduce_kernels.cuh; this file only enqueues them.
#include "../../include/mc_tvd.h"

#include <cuda_runtime.h>
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>
#include <atomic>
#include <new>
#include <type_traits>

#include "mc_async.cuh"
#include "mc_common.cuh"
#include "reduce_kernels.cuh"
#include "flow_stats.cuh"
#include "sweep_lane.cuh"
#include "sweep_lane2.cuh"
#include "sweep_lane3.cuh"
#include "sweep_march.cuh"
#include "sweep_march3.cuh"

namespace {

thread_local char g_err[512] = "";

int fail(int code, const char *fmt, const char *detail = "")
{
    snprintf(g_err, sizeof(g_err), fmt, detail);
    return code;
}

size_t align_up(size_t v, size_t a) { return (v + a - 1) / a * a; }

// launch geometry (the -D overrides exist for tuning sweeps; the defaults are the measured best)
#ifndef MC_MARCH_WX_2D
#define MC_MARCH_WX_2D 128
#endif
#ifndef MC_MARCH_MINB_2D
#define MC_MARCH_MINB_2D 4
#endif
#ifndef MC_MARCH3_WB
#define MC_MARCH3_WB 12
#endif
#ifndef MC_MARCH3_MINB
#define MC_MARCH3_MINB 1
#endif
#ifndef MC_LANE3_WB
#define MC_LANE3_WB 12
#endif
#ifndef MC_MARCH3_WB_AS
#define MC_MARCH3_WB_AS 12
#endif
#ifndef MC_ASYNC3
#define MC_ASYNC3 1
#endif
#ifndef MC_TMA_L2PROMO
#define MC_TMA_L2PROMO CU_TENSOR_MAP_L2_PROMOTION_NONE
#endif
#ifndef MC_LANE2_WARPS
#define MC_LANE2_WARPS 4
#endif
#ifndef MC_LANE2_MINB
#define MC_LANE2_MINB 2
#endif
#ifndef MC_LANE2
#define MC_LANE2 1
#endif
#ifndef MC_LANE_WARPS_2D
#define MC_LANE_WARPS_2D 4
#endif
#ifndef MC_LANE_MINB_2D
#define MC_LANE_MINB_2D 4
#endif
constexpr int MARCH_WX_2D = MC_MARCH_WX_2D;      // k_march, 2-D: WX - 4 outputs per block row
constexpr int MARCH_MINB_2D = MC_MARCH_MINB_2D;  // k_march, 2-D: resident blocks per SM the register budget allows
constexpr int MARCH3_WB = MC_MARCH3_WB;          // k_march3: 32 x WB threads, 28 x (WB - 2) outputs
constexpr int LANE3_WB = MC_LANE3_WB;            // k_lane3: 32 x WB threads, 28 x (WB - 2) outputs
constexpr int MARCH3_WB_AS = MC_MARCH3_WB_AS;    // the same with asynchronous staging (TMA + row mbarriers)
constexpr int LANE_WARPS_2D = MC_LANE_WARPS_2D;  // k_lane, 2-D: independent warps per block
constexpr int LANE_MINB_2D = MC_LANE_MINB_2D;
constexpr int DIAG_MAX_BLOCKS = 16;    // blocks per plane in the diagnostics pass (the finish kernel walks them)

struct Layout {                        // byte offsets inside the workspace
    size_t Y, scalars, partial, ext, plane_sums, plane_ext, diag_out, stats, stats_out, zt, total;
    size_t flow_partial, flow_ext, flow_hist, flow_out, flow_acc, flow_hist_acc;
    int diag_blocks;
};

}  // namespace

struct mc_tvd_state {
    mc_tvd_grid grid;
    mc_tvd_params par;
    int nd, nf;
    long long N, plane;
    double d[3];                       // dx, dy, dz
    double R, cv, icv, g, mu, K;
    bool walls;
    double *X, *Y;
    mc::Scalars *S;
    double *partial, *ext, *plane_sums, *plane_ext, *diag_out, *stats, *stats_out;
    double *flow_partial, *flow_ext, *flow_out, *flow_acc;
    unsigned long long *flow_hist, *flow_hist_acc;
    bool flow_in_stats;                // samples of mc_tvd_step_stats also accumulate the flow statistics
    int slab_next;                     // mc_tvd_slab_op: the operator of the current step that comes next
    // fused halo push (mc_tvd_slab_peers): the neighbours' two state buffers [0] = their d_fields, [1] = their workspace copy
    bool slab_fused;
    double *peer_lo[2], *peer_hi[2];
    int own_lo, own_hi, halo;
    cudaGraphExec_t graph_exec;        // one step's launch list (mc_tvd_step replays it), or null
    int graph_launches, graph_chunk;   // kernels in it; the chunk override it was captured with
    bool graph_failed;
    const double *zt;                  // device z-metric tables of the non-uniform grid (R19 / R20), or null
    double zt_max_icfl;                // max over levels of the CFL rule's reciprocal z spacing
    long long stat_steps;              // steps taken through mc_tvd_step_stats since the last reset
    int diag_blocks;
    cudaStream_t stream;
    long long launches;
    int chunk_override;
    int sm_count;
    // per-kernel timing (mc_tvd_timing_*): events ev[0..n_ev) recorded around operator launches;
    // launch r ran between ev_pair[r] and ev_pair[r] + 1
    bool timing;
    cudaEvent_t *ev;
    int n_ev, n_rec;
    int *rec_kind, *rec_ev;
    bool ev_open;                      // the last recorded event directly precedes the next launch
    // 3-D, even nx: TMA tensor maps (x, y, z, field) of the two state buffers [0] = X, [1] = Y, with the box
    // of a z-march tile (32 x rows(y) x 1 x 5) and of a y-march tile (32 x 1 x rows(z) x 5)
    bool async3;
    CUtensorMap tm_rows_y[2], tm_rows_z[2];
    int geom[3][3];                    // per operator alpha, of its last launch: outputs per tile along x, along b, levels per chunk
};

namespace {

bool valid_problem(const mc_tvd_grid *g, const mc_tvd_params *p, int *code)
{
    *code = MC_TVD_EINVAL;
    if (!g || !p) return fail(0, "grid or params is NULL"), false;
    if (g->ndim != 2 && g->ndim != 3) return fail(0, "ndim must be 2 or 3"), false;
    if (g->nx < 4 || g->nz < 5 || g->ny < 1) return fail(0, "need nx >= 4, nz >= 5, ny >= 1"), false;
    if (g->ndim == 2 && g->ny != 1) return fail(0, "ny must be 1 in 2-D"), false;
    if (g->ndim == 3 && g->ny < 4) return fail(0, "need ny >= 4 in 3-D"), false;
    if (!(g->lx > 0) || !(g->lz > 0) || (g->ndim == 3 && !(g->ly > 0))) return fail(0, "box size must be > 0"), false;
    if ((long long)g->nx * g->ny * g->nz >= (1ll << 32)) {
        *code = MC_TVD_EUNSUPPORTED;
        return fail(0, "more than 2^32 - 1 nodes per field: the kernels index nodes with 32 bits"), false;
    }
    if (!(p->gamma > 1) || !(p->eps > 0) || !(p->D > 0) || !(p->Pr > 0) || !(p->Ra > 0))
        return fail(0, "need gamma > 1 and eps, D, Pr, Ra > 0"), false;
    if (!(p->fixed_dt > 0) && !(p->cfl > 0)) return fail(0, "need cfl > 0 or fixed_dt > 0"), false;
    if ((p->bc_z | 1) != 1 || (p->tvd_form | 1) != 1 || (p->dir_mode | 1) != 1 || (p->tvd_off | 1) != 1 || (p->co_mode | 1) != 1)
        return fail(0, "bc_z, tvd_form, dir_mode, tvd_off, co_mode must be 0 or 1"), false;
    if (g->z_nodes) {                  // non-uniform z grid (R19): plates at the first and last node
        if (p->bc_z != 0) return fail(0, "z_nodes needs plates (bc_z = 0)"), false;
        for (int k = 0; k + 1 < g->nz; ++k)
            if (!(g->z_nodes[k + 1] > g->z_nodes[k]) || !isfinite(g->z_nodes[k + 1]) || !isfinite(g->z_nodes[k]))
                return fail(0, "z_nodes must be finite and strictly increasing"), false;
    }
    return true;
}

Layout make_layout(const mc_tvd_grid *g)
{
    Layout L;
    const size_t nf = (g->ndim == 2) ? 4 : 5;
    const size_t N = (size_t)g->nx * g->ny * g->nz, plane = (size_t)g->nx * g->ny;
    int nb = (int)((plane + (size_t)mc::DIAG_THREADS * 8 - 1) / ((size_t)mc::DIAG_THREADS * 8));
    if (nb < 1) nb = 1;
    if (nb > DIAG_MAX_BLOCKS) nb = DIAG_MAX_BLOCKS;
    L.diag_blocks = nb;
    size_t o = 0;
    L.Y = o;          o = align_up(o + nf * N * sizeof(double), 256);
    L.scalars = o;    o = align_up(o + sizeof(mc::Scalars), 256);
    L.partial = o;    o = align_up(o + (size_t)g->nz * nb * 2 * mc::DQ_MAXQ * sizeof(double), 256);
    L.ext = o;        o = align_up(o + (size_t)g->nz * nb * 3 * sizeof(double), 256);
    L.plane_sums = o; o = align_up(o + (size_t)g->nz * mc::DQ_MAXQ * sizeof(double), 256);
    L.plane_ext = o;  o = align_up(o + (size_t)g->nz * 3 * sizeof(double), 256);
    L.diag_out = o;   o = align_up(o + (19 + 3 * (size_t)g->nz) * sizeof(double), 256);
    L.stats = o;      o = align_up(o + (mc::ST_HEAD + 3 * (size_t)g->nz) * sizeof(double), 256);
    L.stats_out = o;  o = align_up(o + (4 + mc::ST_NSUM + 3 * (size_t)g->nz) * sizeof(double), 256);
    L.zt = o;         o = align_up(o + 5 * (size_t)g->nz * sizeof(double), 256);       // z-metric tables (SweepArgs::zt)
    L.flow_partial = o;  o = align_up(o + (size_t)g->nz * nb * mc::FLOW_NQ * sizeof(double), 256);
    L.flow_ext = o;      o = align_up(o + (size_t)g->nz * nb * sizeof(double), 256);
    L.flow_hist = o;     o = align_up(o + mc::FLOW_BINS * sizeof(unsigned long long), 256);
    L.flow_out = o;      o = align_up(o + mc::FLOW_NOUT * sizeof(double), 256);
    L.flow_acc = o;      o = align_up(o + mc::FLOW_NOUT * sizeof(double), 256);
    L.flow_hist_acc = o; o = align_up(o + mc::FLOW_BINS * sizeof(unsigned long long), 256);
    L.total = o;
    return L;
}

int cuda_check(cudaError_t e, const char *what)
{
    if (e == cudaSuccess) return MC_TVD_OK;
    snprintf(g_err, sizeof(g_err), "%s: %s", what, cudaGetErrorString(e));
    return MC_TVD_ECUDA;
}

// velocity-component index of physical axis a (0 x, 1 y, 2 z): 2-D carries (x, z)
int comp_of_axis(int nd, int a) { return (nd == 2) ? (a == 0 ? 0 : 1) : a; }

void fill_common(const mc_tvd_state *s, mc::SweepArgs &A, const double *in, double *out, int alpha, int dir,
                 double tau, bool use_dt, bool reduce)
{
    memset(&A, 0, sizeof(A));
    A.in = in; A.out = out;
    A.dt_ptr = use_dt ? &s->S->dt : nullptr;
    A.tau_fixed = tau;
    A.smax_bits = &s->S->smax_bits;
    A.N = s->N; A.nx = s->grid.nx;
    A.dir = dir;
    A.src = (alpha == 2);
    A.reduce = reduce ? 1 : 0;
    A.d_a = s->d[alpha];
    A.inv_h = (dir > 0 ? 1.0 : -1.0) / s->d[alpha];
    const double mu = s->mu, lam = s->par.lambda_coef;
    A.mu_h = mu * A.inv_h; A.two_mu_h = 2.0 * mu * A.inv_h; A.lam_mu_h = lam * mu * A.inv_h; A.K_h = s->K * A.inv_h;
    for (int a = 0; a < 3; ++a) {
        if (s->nd == 2 && a == 1) continue;
        const int c = comp_of_axis(s->nd, a);
        A.inv_d[c] = 1.0 / s->d[a];
        A.mu_2c[c] = mu / (2.0 * s->d[a]);
        A.lam_mu_2c[c] = lam * mu / (2.0 * s->d[a]);
    }
    A.dz = s->d[2];
    if (s->zt) {
        // non-uniform z (R19 / R20): every z spacing folded into a launch constant becomes 1; the kernels (template
        // switch ZS) multiply by the local metric from the tables instead
        const int cz = comp_of_axis(s->nd, 2);
        A.zt = s->zt;
        A.mu_2c[cz] = mu; A.lam_mu_2c[cz] = lam * mu;        // central z-differences: x 1 / (z_{k+1} - z_{k-1}) in the kernel
        A.inv_d[cz] = s->zt_max_icfl;                         // only the bound D of the CFL filter uses it
        if (alpha == 2) {
            A.d_a = 1.0; A.inv_h = (dir > 0 ? 1.0 : -1.0);
            A.mu_h = mu * A.inv_h; A.two_mu_h = 2.0 * mu * A.inv_h; A.lam_mu_h = lam * mu * A.inv_h; A.K_h = s->K * A.inv_h;
        }
    }
    if (s->slab_fused) {
        const int b = (out == s->X) ? 0 : 1;                  // the neighbours write the same one of their two buffers
        A.peer_lo = s->peer_lo[b]; A.peer_hi = s->peer_hi[b];
        A.own_lo = s->own_lo; A.own_hi = s->own_hi; A.halo = s->halo;
        A.slab_shift = (long long)(s->own_hi - s->own_lo) * s->grid.nx;      // y rows of nx nodes
    }
    A.R = s->R; A.cv = s->cv; A.icv = s->icv; A.g = s->g;
    A.gamma = s->par.gamma; A.gammaR = s->par.gamma * s->R;
    A.co_cs = s->par.co_mode ? 0.0 : 1.0;
    A.Tw0 = s->par.T_bot; A.Tw1 = s->par.T_top;
    A.nz = s->grid.nz;
    double D = 0.0;
    for (int c = 0; c < s->nd; ++c) D = A.inv_d[c] > D ? A.inv_d[c] : D;
    A.cfl_wQ = s->par.gamma * (s->par.gamma - 1.0) * (1.0 + 1.0 / 16.0) * D * D;
    A.cfl_wm = (1.0 + 16.0) * D * D;
}

// Marching levels per block.  Cutting the march into c chunks multiplies the blocks (fills the SMs, evens
// out the last wave) but every chunk repeats a 4-level warm-up.  Model: blocks run in waves of
// (SMs x resident blocks per SM) and the last wave costs about half a block more than its share;
// cost(c) = max(whole waves, waves + 1/2) x (levels per chunk + 8): the 4 warm-up levels run the general
// loop body, about twice the cost of a fast level.  Take the cheapest c.
int pick_chunk(const mc_tvd_state *s, int n_m, long long tiles, int blocks_per_sm)
{
    if (s->chunk_override > 0) return s->chunk_override < n_m ? s->chunk_override : n_m;
    const long long slots = (long long)s->sm_count * blocks_per_sm;
    const int c_max = n_m / 8 > 1 ? n_m / 8 : 1;       // (chunks down to 8 levels: small boxes are bound by the march's latency, not by work)
    long long best_cost = -1;
    int best_chunk = n_m;
    for (int c = 1; c <= c_max; ++c) {
        const int chunk = (n_m + c - 1) / c;
        const long long blocks = tiles * ((n_m + chunk - 1) / chunk);
        const long long whole = 2 * ((blocks + slots - 1) / slots), frac = (2 * blocks + slots - 1) / slots + 1;
        const long long cost = (whole > frac ? whole : frac) * (chunk + 8);      // in half waves
        if (best_cost < 0 || cost < best_cost) { best_cost = cost; best_chunk = chunk; }
    }
    return best_chunk;
}

// compile-time dispatch of the kernels' switches
template <class F> void with_bool(bool b, F f)
{
    if (b) f(std::true_type()); else f(std::false_type());
}
// the non-uniform z grid exists between plates only: ZS kernels are instantiated for WALL = true
template <class W, class F> void with_zs(const mc_tvd_state *s, W, F f)
{
    if constexpr (W::value) { if (s->zt) { f(std::true_type()); return; } }
    f(std::false_type());
}
// the fused halo push exists for the TMA-staged 3-D kernels between plates on a uniform z grid
template <class W, class Z, class F> void with_sl(const mc_tvd_state *s, W, Z, F f)
{
    if constexpr (W::value && !Z::value) { if (s->slab_fused) { f(std::true_type()); return; } }
    f(std::false_type());
}
// MC_ONLY_DEFAULT_SWITCHES (tuning builds only): instantiate just the plates + Davis/Yee kernels
template <class F> void with_walls(bool b, F f)
{
#ifdef MC_ONLY_DEFAULT_SWITCHES
    (void)b; f(std::true_type());
#else
    with_bool(b, f);
#endif
}
template <class F> void with_tvd(const mc_tvd_state *s, F f)
{
#ifdef MC_ONLY_DEFAULT_SWITCHES
    (void)s; f(std::integral_constant<int, 1>()); return;
#endif
    if (s->par.tvd_off) f(std::integral_constant<int, -1>());
    else if (s->par.tvd_form == 0) f(std::integral_constant<int, 0>());
    else f(std::integral_constant<int, 1>());
}

// Tiled tensor map over a 5-field SoA state (x fastest): box = 32 columns x rows_y x rows_z x 5 fields, fp64,
// no swizzle (a thread reads its own column: consecutive lanes, consecutive doubles), zero fill outside.
int make_state_map(CUtensorMap *map, const double *base, int nx, int ny, int nz, int rows_y, int rows_z)
{
    typedef CUresult (*encode_fn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static encode_fn encode = nullptr;                 // resolved once; the value is the same for every thread
    if (!encode) {
        void *fn = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q) != cudaSuccess || !fn)
            return fail(MC_TVD_ECUDA, "cuTensorMapEncodeTiled is not available in this driver");
        encode = (encode_fn)fn;
    }
    const cuuint64_t dims[4] = {(cuuint64_t)nx, (cuuint64_t)ny, (cuuint64_t)nz, 5};
    const cuuint64_t strides[3] = {(cuuint64_t)nx * 8, (cuuint64_t)nx * ny * 8, (cuuint64_t)nx * ny * nz * 8};
    const cuuint32_t box[4] = {32, (cuuint32_t)rows_y, (cuuint32_t)rows_z, 5};
    const cuuint32_t estr[4] = {1, 1, 1, 1};
    const CUresult r = encode(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, (void *)base, dims, strides, box, estr,
                              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, MC_TMA_L2PROMO,
                              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(MC_TVD_ECUDA, "cuTensorMapEncodeTiled failed");
    return MC_TVD_OK;
}

template <class K, class... Extra>
int launch_kernel(K kfn, dim3 grid, dim3 block, size_t smem, cudaStream_t st, const mc::SweepArgs &A, const Extra &...extra)
{
    // opt in to large dynamic shared memory: a per-function attribute, set before every such launch (no
    // cache to guard: distinct handles may launch from different threads)
    if (smem > 48 * 1024) cudaFuncSetAttribute(kfn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    MC_LAUNCH(kfn, grid, block, smem, st, A, extra...);
    return 0;
}

// Enqueue one operator L_alpha(tau): in -> out.
int launch_sweep(mc_tvd_state *s, const double *in, double *out, int alpha, int dir, double tau, bool use_dt,
                 bool reduce)
{
    mc::SweepArgs A;
    fill_common(s, A, in, out, alpha, dir, tau, use_dt, reduce);
    const int nx = s->grid.nx, ny = s->grid.ny, nz = s->grid.nz;
    const bool timed = s->timing && s->n_rec < MC_TVD_MAX_TIMED;
    if (timed && !s->ev_open) { cudaEventRecord(s->ev[s->n_ev], s->stream); s->n_ev += 1; }
    s->ev_open = timed;                // the closing event of this launch opens the next one
    const bool wl = s->walls;
    cudaStream_t st = s->stream;
    int geo_x = 0, geo_b = 1;          // outputs per tile along x and along the second tile direction (test hook)
    if (s->nd == 2) {
        if (alpha == 2) {            // z-sweep: march z, tile x
            constexpr int WX = MARCH_WX_2D;
            geo_x = WX - 4;
            A.n_b = 1; A.s_b = 0; A.n_m = nz; A.s_m = nx;
            long long tiles = (nx + WX - 5) / (WX - 4);
            A.chunk = pick_chunk(s, nz, tiles, MARCH_MINB_2D);
            dim3 block(WX, 1, 1), grid((unsigned)tiles, 1, (unsigned)((nz + A.chunk - 1) / A.chunk));
            size_t smem = ((size_t)4 * 2 * WX + 4) * sizeof(double);
            with_walls(wl, [&](auto W) { with_tvd(s, [&](auto T) { with_zs(s, W, [&](auto Z) {
                launch_kernel(mc::k_march<2, 1, -1, WX, 1, decltype(W)::value, false, decltype(T)::value, MARCH_MINB_2D, decltype(Z)::value>, grid, block, smem, st, A);
            }); }); });
        } else if (alpha == 0 && MC_LANE2 && nx % 2 == 0) {   // x-sweep, even nx: two nodes per lane, march z
            constexpr int LW = MC_LANE2_WARPS;
            geo_x = mc::LANE2_OUT;
            A.n_b = 1; A.s_b = 0; A.n_m = nz; A.s_m = nx;
            long long xt = (nx + mc::LANE2_OUT - 1) / mc::LANE2_OUT;
            long long tiles = (xt + LW - 1) / LW;
            A.chunk = pick_chunk(s, nz, tiles, MC_LANE2_MINB);
            dim3 block(32, LW, 1), grid((unsigned)tiles, 1, (unsigned)((nz + A.chunk - 1) / A.chunk));
            with_walls(wl, [&](auto W) { with_tvd(s, [&](auto T) { with_bool(reduce, [&](auto Rd) {
                with_bool(dir > 0, [&](auto Fw) { with_zs(s, W, [&](auto Z) {
                    launch_kernel(mc::k_lane2<LW, decltype(W)::value, decltype(T)::value, decltype(Rd)::value, MC_LANE2_MINB, decltype(Fw)::value, decltype(Z)::value>, grid, block, 0, st, A);
                }); });
            }); }); });
        } else if (alpha == 0) {     // x-sweep: lanes x, march z
            constexpr int LW = LANE_WARPS_2D;
            geo_x = mc::LANE_OUT;
            A.n_b = 1; A.s_b = 0; A.n_m = nz; A.s_m = nx;
            long long xt = (nx + mc::LANE_OUT - 1) / mc::LANE_OUT;
            long long tiles = (xt + LW - 1) / LW;
            A.chunk = pick_chunk(s, nz, tiles, LANE_MINB_2D);
            dim3 block(32, LW, 1), grid((unsigned)tiles, 1, (unsigned)((nz + A.chunk - 1) / A.chunk));
            with_walls(wl, [&](auto W) { with_tvd(s, [&](auto T) { with_bool(reduce, [&](auto Rd) { with_zs(s, W, [&](auto Z) {
                launch_kernel(mc::k_lane<2, -1, 1, LW, decltype(W)::value, decltype(T)::value, decltype(Rd)::value, LANE_MINB_2D, decltype(Z)::value>, grid, block, 0, st, A);
            }); }); }); });
        } else {
            return fail(MC_TVD_EINVAL, "a 2-D problem has no y-sweep");
        }
    } else {
        long long xt = (nx + mc::LANE_OUT - 1) / mc::LANE_OUT;
        const int ibuf = (in == s->X) ? 0 : 1;        // which state buffer the operator reads
        geo_x = mc::LANE_OUT;
        if (alpha == 2 && s->async3) {   // z-sweep, TMA-staged tiles: march z, tile (x, y)
            constexpr int MW = MARCH3_WB_AS, MO = MW - 2;
            A.n_b = ny; A.s_b = nx; A.n_m = nz; A.s_m = (long long)nx * ny;
            long long bt = (ny + MO - 1) / MO;
            geo_b = MO;
            A.chunk = pick_chunk(s, nz, xt * bt, 1);
            dim3 mblock(32, MW, 1), grid((unsigned)xt, (unsigned)bt, (unsigned)((nz + A.chunk - 1) / A.chunk));
            size_t smem = mc::tile3_async_bytes(MW) + ((size_t)4 * 3 * 32 * (MW + 2) + 4) * sizeof(double);
            with_walls(wl, [&](auto W) { with_tvd(s, [&](auto T) { with_zs(s, W, [&](auto Z) { with_sl(s, W, Z, [&](auto L) {
                launch_kernel(mc::k_march3<2, 1, MW, decltype(W)::value, false, decltype(T)::value, 1, true, decltype(Z)::value, decltype(L)::value>, grid, mblock, smem, st, A, s->tm_rows_y[ibuf]);
            }); }); }); });
        } else if (alpha == 1 && s->async3) {   // y-sweep, TMA-staged tiles: march y, tile (x, z)
            constexpr int MW = MARCH3_WB_AS, MO = MW - 2;
            A.n_b = nz; A.s_b = (long long)nx * ny; A.n_m = ny; A.s_m = nx;
            long long bt = (nz + MO - 1) / MO;
            geo_b = MO;
            A.chunk = pick_chunk(s, ny, xt * bt, 1);
            dim3 mblock(32, MW, 1), grid((unsigned)xt, (unsigned)bt, (unsigned)((ny + A.chunk - 1) / A.chunk));
            size_t smem = mc::tile3_async_bytes(MW) + ((size_t)4 * 3 * 32 * (MW + 2) + 4) * sizeof(double);
            with_walls(wl, [&](auto W) { with_tvd(s, [&](auto T) { with_zs(s, W, [&](auto Z) { with_sl(s, W, Z, [&](auto L) {
                launch_kernel(mc::k_march3<1, 2, MW, false, decltype(W)::value, decltype(T)::value, 1, true, decltype(Z)::value, decltype(L)::value>, grid, mblock, smem, st, A, s->tm_rows_z[ibuf]);
            }); }); }); });
        } else if (alpha == 2) {            // z-sweep: march z, tile (x, y)
            constexpr int MW = MARCH3_WB, MO = MW - 2;
            A.n_b = ny; A.s_b = nx; A.n_m = nz; A.s_m = (long long)nx * ny;
            long long bt = (ny + MO - 1) / MO;
            geo_b = MO;
            A.chunk = pick_chunk(s, nz, xt * bt, 1);
            dim3 mblock(32, MW, 1), grid((unsigned)xt, (unsigned)bt, (unsigned)((nz + A.chunk - 1) / A.chunk));
            size_t smem = ((size_t)4 * 3 * 32 * (MW + 2) + 4) * sizeof(double);
            with_walls(wl, [&](auto W) { with_tvd(s, [&](auto T) { with_zs(s, W, [&](auto Z) {
                launch_kernel(mc::k_march3<2, 1, MW, decltype(W)::value, false, decltype(T)::value, MC_MARCH3_MINB, false, decltype(Z)::value>, grid, mblock, smem, st, A, s->tm_rows_y[ibuf]);
            }); }); });
        } else if (alpha == 1) {     // y-sweep: march y, tile (x, z)
            constexpr int MW = MARCH3_WB, MO = MW - 2;
            A.n_b = nz; A.s_b = (long long)nx * ny; A.n_m = ny; A.s_m = nx;
            long long bt = (nz + MO - 1) / MO;
            geo_b = MO;
            A.chunk = pick_chunk(s, ny, xt * bt, 1);
            dim3 mblock(32, MW, 1), grid((unsigned)xt, (unsigned)bt, (unsigned)((ny + A.chunk - 1) / A.chunk));
            size_t smem = ((size_t)4 * 3 * 32 * (MW + 2) + 4) * sizeof(double);
            with_walls(wl, [&](auto W) { with_tvd(s, [&](auto T) { with_zs(s, W, [&](auto Z) {
                launch_kernel(mc::k_march3<1, 2, MW, false, decltype(W)::value, decltype(T)::value, MC_MARCH3_MINB, false, decltype(Z)::value>, grid, mblock, smem, st, A, s->tm_rows_z[ibuf]);
            }); }); });
        } else {                     // x-sweep: lanes x, tile (x, y), march z
            constexpr int LW = LANE3_WB, LO = LW - 2;
            A.n_b = ny; A.s_b = nx; A.n_m = nz; A.s_m = (long long)nx * ny;
            long long bt = (ny + LO - 1) / LO;
            geo_b = LO;
            A.chunk = pick_chunk(s, nz, xt * bt, 1);
            dim3 lblock(32, LW, 1), grid((unsigned)xt, (unsigned)bt, (unsigned)((nz + A.chunk - 1) / A.chunk));
            size_t smem = (size_t)4 * 2 * 32 * (LW + 2) * sizeof(double);
            with_walls(wl, [&](auto W) { with_tvd(s, [&](auto T) { with_bool(reduce, [&](auto Rd) { with_zs(s, W, [&](auto Z) { with_sl(s, W, Z, [&](auto L) {
                launch_kernel(mc::k_lane3<1, 2, LW, decltype(W)::value, decltype(T)::value, decltype(Rd)::value, decltype(Z)::value, decltype(L)::value>, grid, lblock, smem, st, A);
            }); }); }); }); });
        }
    }
    s->geom[alpha][0] = geo_x; s->geom[alpha][1] = geo_b; s->geom[alpha][2] = A.chunk;
    s->launches += 1;
    int rc = cuda_check(cudaGetLastError(), "sweep launch");
    if (rc == MC_TVD_OK && timed) {
        cudaEventRecord(s->ev[s->n_ev], s->stream);
        s->rec_kind[s->n_rec] = alpha + (dir < 0 ? 3 : 0);
        s->rec_ev[s->n_rec] = s->n_ev - 1;
        s->n_rec += 1; s->n_ev += 1;
    }
    return rc;
}

mc::PointArgs point_args(const mc_tvd_state *s)
{
    mc::PointArgs P;
    memset(&P, 0, sizeof(P));
    P.X = s->X; P.N = s->N; P.plane = s->plane; P.nz = s->grid.nz;
    P.dz = s->d[2]; P.g = s->g; P.icv = s->icv; P.R = s->R; P.gamma = s->par.gamma; P.D = s->par.D;
    for (int a = 0; a < 3; ++a) {
        if (s->nd == 2 && a == 1) continue;
        P.inv_d[comp_of_axis(s->nd, a)] = 1.0 / s->d[a];
    }
    P.zt = s->zt;
    P.own_axis = -1; P.nx = s->grid.nx;
    return P;
}

// Enqueue the max-speed reduction of the state in s->X and the dt it implies (R12).
int enqueue_initial_dt(mc_tvd_state *s)
{
    mc::PointArgs P = point_args(s);
    int blocks = (int)((s->N + 255) / 256);
    if (blocks > 148 * 16) blocks = 148 * 16;
    if (s->nd == 2) { auto kfn = mc::k_max_speed<2>; MC_LAUNCH(kfn, blocks, 256, 0, s->stream, P, &s->S->smax_bits); }
    else { auto kfn = mc::k_max_speed<3>; MC_LAUNCH(kfn, blocks, 256, 0, s->stream, P, &s->S->smax_bits); }
    { auto kfn = mc::k_dt_update; MC_LAUNCH(kfn, 1, 32, 0, s->stream, s->S, 0); }
    s->launches += 2;
    return cuda_check(cudaGetLastError(), "initial dt launch");
}

}  // namespace

extern "C" {

const char *mc_tvd_last_error(void) { return g_err; }

size_t mc_tvd_workspace_bytes(const mc_tvd_grid *grid, const mc_tvd_params *params)
{
    int code;
    if (!valid_problem(grid, params, &code)) return 0;
    return make_layout(grid).total;
}

int mc_tvd_init(const mc_tvd_grid *grid, const mc_tvd_params *params, double *d_fields, void *d_workspace,
                size_t workspace_bytes, void *cuda_stream, mc_tvd_state **out)
{
    int code;
    if (!out) return fail(MC_TVD_EINVAL, "out is NULL");
    *out = nullptr;
    if (!valid_problem(grid, params, &code)) return code;
    if (!d_fields || !d_workspace) return fail(MC_TVD_EINVAL, "d_fields or d_workspace is NULL");
    if (((uintptr_t)d_fields & 15) || ((uintptr_t)d_workspace & 255))
        return fail(MC_TVD_EINVAL, "d_fields must be 16-byte and d_workspace 256-byte aligned");
    Layout L = make_layout(grid);
    if (workspace_bytes < L.total) return fail(MC_TVD_ENOMEM, "workspace smaller than mc_tvd_workspace_bytes");
    mc_tvd_state *s = new (std::nothrow) mc_tvd_state;
    if (!s) return fail(MC_TVD_ENOMEM, "host allocation failed");
    memset(s, 0, sizeof(*s));
    s->grid = *grid; s->par = *params;
    s->nd = grid->ndim; s->nf = (grid->ndim == 2) ? 4 : 5;
    s->plane = (long long)grid->nx * grid->ny;
    s->N = s->plane * grid->nz;
    s->walls = (params->bc_z == 0);
    // grid spacings (R17) and coefficients from the paper's numbers (Eqs. 14-18)
    s->d[0] = grid->lx / grid->nx;
    s->d[1] = (grid->ndim == 3) ? grid->ly / grid->ny : 1.0;
    s->d[2] = s->walls ? grid->lz / (grid->nz - 1) : grid->lz / grid->nz;
    s->icv = params->gamma * params->eps * params->D;
    s->cv = 1.0 / s->icv;
    s->R = (params->gamma - 1.0) / s->icv;
    s->g = (params->g_override >= 0.0) ? params->g_override : 1.0 / params->eps;
    s->mu = (params->mu_override >= 0.0) ? params->mu_override : sqrt(params->Pr / params->Ra);
    s->K = (params->K_override >= 0.0) ? params->K_override
                                       : 1.0 / (params->eps * params->D * sqrt(params->Ra * params->Pr));
    char *w = (char *)d_workspace;
    s->X = d_fields;
    s->Y = (double *)(w + L.Y);
    s->S = (mc::Scalars *)(w + L.scalars);
    s->partial = (double *)(w + L.partial);
    s->ext = (double *)(w + L.ext);
    s->plane_sums = (double *)(w + L.plane_sums);
    s->plane_ext = (double *)(w + L.plane_ext);
    s->diag_out = (double *)(w + L.diag_out);
    s->stats = (double *)(w + L.stats);
    s->stats_out = (double *)(w + L.stats_out);
    s->flow_partial = (double *)(w + L.flow_partial);
    s->flow_ext = (double *)(w + L.flow_ext);
    s->flow_hist = (unsigned long long *)(w + L.flow_hist);
    s->flow_out = (double *)(w + L.flow_out);
    s->flow_acc = (double *)(w + L.flow_acc);
    s->flow_hist_acc = (unsigned long long *)(w + L.flow_hist_acc);
    s->flow_in_stats = false;
    s->zt = nullptr; s->zt_max_icfl = 0.0;
    s->grid.z_nodes = nullptr;         // the caller's array is not kept: its numbers live in the device tables
    s->diag_blocks = L.diag_blocks;
    s->stream = (cudaStream_t)cuda_stream;
    s->chunk_override = 0;
    {
        int dev = 0, sms = 0;
        if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms < 1)
            sms = 148;
        s->sm_count = sms;
    }

    int rc = MC_TVD_OK;
    // TMA needs 16-byte row strides: an odd nx keeps the kernels that load through registers
    s->async3 = MC_ASYNC3 && s->nd == 3 && grid->nx % 2 == 0;
    if (s->async3) {
        const double *buf[2] = {s->X, s->Y};
        for (int b = 0; b < 2 && rc == MC_TVD_OK; ++b) {
            rc = make_state_map(&s->tm_rows_y[b], buf[b], grid->nx, grid->ny, grid->nz, MARCH3_WB_AS + 2, 1);
            if (rc == MC_TVD_OK) rc = make_state_map(&s->tm_rows_z[b], buf[b], grid->nx, grid->ny, grid->nz, 1, MARCH3_WB_AS + 2);
        }
        if (rc != MC_TVD_OK) { delete s; return rc; }
    }

    // Non-uniform z grid (R19 / R20): the metric tables of SweepArgs::zt, built once from the caller's
    // node heights: z, g z, 1 / cell height, 1 / face spacing, face spacing.
    double *zt_host = nullptr;
    if (grid->z_nodes) {
        const int nz = grid->nz;
        const double *z = grid->z_nodes;
        zt_host = (double *)malloc(5 * (size_t)nz * sizeof(double));
        if (!zt_host) { delete s; return fail(MC_TVD_ENOMEM, "host allocation failed"); }
        for (int k = 0; k < nz; ++k) {
            const double dzc = (k == 0) ? 0.5 * (z[1] - z[0]) : (k == nz - 1) ? 0.5 * (z[k] - z[k - 1]) : 0.5 * (z[k + 1] - z[k - 1]);
            const double hf = (k < nz - 1) ? z[k + 1] - z[k] : z[k] - z[k - 1];
            zt_host[k] = z[k];
            zt_host[nz + k] = s->g * z[k];
            zt_host[2 * nz + k] = 1.0 / dzc;
            zt_host[3 * nz + k] = 1.0 / hf;
            zt_host[4 * nz + k] = hf;
            const double icfl = (k == 0 || k == nz - 1) ? 0.5 / dzc : 1.0 / dzc;
            if (icfl > s->zt_max_icfl) s->zt_max_icfl = icfl;
        }
        double *zt_dev = (double *)(w + L.zt);
        rc = cuda_check(cudaMemcpyAsync(zt_dev, zt_host, 5 * (size_t)nz * sizeof(double), cudaMemcpyHostToDevice, s->stream),
                        "z table upload");
        s->zt = zt_dev;
    }

    mc::Scalars h;
    memset(&h, 0, sizeof(h));
    h.cfl = params->cfl; h.fixed_dt = params->fixed_dt;
    if (rc == MC_TVD_OK) rc = cuda_check(cudaMemcpyAsync(s->S, &h, sizeof(h), cudaMemcpyHostToDevice, s->stream), "scalar upload");
    if (rc == MC_TVD_OK) rc = cuda_check(cudaStreamSynchronize(s->stream), "scalar upload sync");   // h and zt_host are host temporaries
    free(zt_host);
    if (rc == MC_TVD_OK) rc = enqueue_initial_dt(s);
    if (rc == MC_TVD_OK) rc = mc_tvd_stats_reset(s);
    if (rc != MC_TVD_OK) { delete s; return rc; }
    *out = s;
    return MC_TVD_OK;
}

// Enqueue the launch list of ONE step of Eq. 30 on s->stream: 2 ndim operators + the dt update.
static int enqueue_one_step(mc_tvd_state *s)
{
    const double *src = s->X;
    double *dst = s->Y;
    for (int half = 0; half < 2; ++half) {
        int dir = (half == 1 && s->par.dir_mode == 1) ? -1 : +1;
        for (int a = 2; a >= 0; --a) {                       // L_z, then L_y, then L_x (Eq. 30)
            if (s->nd == 2 && a == 1) continue;
            bool last = (half == 1 && a == 0);
            int rc = launch_sweep(s, src, dst, a, dir, 0.0, true, last);
            if (rc != MC_TVD_OK) return rc;
            const double *t = src; src = dst; dst = (double *)t;
        }
    }
    { auto kfn = mc::k_dt_update; MC_LAUNCH(kfn, 1, 32, 0, s->stream, s->S, 1); }
    s->launches += 1;
    s->ev_open = false;
    return cuda_check(cudaGetLastError(), "dt launch");
}

// The step's launch list as an instantiated CUDA graph (the list is the same every step: the buffers ping-pong back to
// d_fields, dt is read from device memory).  Captured once on a private stream (the caller's may be the legacy default
// stream, which cannot be captured) and replayed on the caller's.  Small boxes are launch-bound: 5-7 launches of a few
// microseconds each per step.  Returns false (and leaves the plain path to run) if capture is not possible.
static bool ensure_step_graph(mc_tvd_state *s)
{
    if (s->graph_exec && s->graph_chunk == s->chunk_override) return true;
    if (s->graph_failed) return false;
    if (s->graph_exec) { cudaGraphExecDestroy(s->graph_exec); s->graph_exec = nullptr; }
    cudaStream_t cap = nullptr, user = s->stream;
    cudaGraph_t graph = nullptr;
    const long long launches0 = s->launches;
    bool ok = cudaStreamCreateWithFlags(&cap, cudaStreamNonBlocking) == cudaSuccess;
    if (ok) ok = cudaStreamBeginCapture(cap, cudaStreamCaptureModeRelaxed) == cudaSuccess;
    if (ok) {
        s->stream = cap;
        const int rc = enqueue_one_step(s);
        s->stream = user;
        const cudaError_t e = cudaStreamEndCapture(cap, &graph);
        ok = (rc == MC_TVD_OK) && e == cudaSuccess && graph;
    }
    s->graph_launches = (int)(s->launches - launches0);
    s->launches = launches0;                                   // nothing ran yet
    if (ok) ok = cudaGraphInstantiate(&s->graph_exec, graph, 0) == cudaSuccess;
    if (graph) cudaGraphDestroy(graph);
    if (cap) cudaStreamDestroy(cap);
    if (!ok) { cudaGetLastError(); s->graph_exec = nullptr; s->graph_failed = true; return false; }
    s->graph_chunk = s->chunk_override;
    return true;
}

int mc_tvd_step(mc_tvd_state *s, int n_steps)
{
    if (!s || n_steps < 0) return fail(MC_TVD_EINVAL, "bad handle or n_steps");
    {   // a kernel fault of earlier work on this stream is sticky: report it here without waiting
        const cudaError_t q = cudaStreamQuery(s->stream);
        if (q != cudaSuccess && q != cudaErrorNotReady) return cuda_check(q, "earlier work on the stream failed");
    }
    if (s->slab_next != 0) return fail(MC_TVD_EINVAL, "a step enqueued operator by operator (mc_tvd_slab_op) is half done");
    // per-operator timing records events between the launches: plain launches then
    const bool graphed = !s->timing && n_steps >= 2 && ensure_step_graph(s);
    for (int it = 0; it < n_steps; ++it) {
        if (graphed) {
            int rc = cuda_check(cudaGraphLaunch(s->graph_exec, s->stream), "step graph launch");
            if (rc != MC_TVD_OK) return rc;
            s->launches += s->graph_launches;
        } else {
            int rc = enqueue_one_step(s);
            if (rc != MC_TVD_OK) return rc;
        }
    }
    return MC_TVD_OK;
}

int mc_tvd_sweep(mc_tvd_state *s, int alpha, int dir, double tau)
{
    if (!s || alpha < 0 || alpha > 2 || (dir != 1 && dir != -1) || !(tau > 0))
        return fail(MC_TVD_EINVAL, "bad handle, alpha, dir or tau");
    int rc = launch_sweep(s, s->X, s->Y, alpha, dir, tau, false, false);
    s->ev_open = false;                // the copy below separates this launch from the next one
    if (rc != MC_TVD_OK) return rc;
    rc = cuda_check(cudaMemcpyAsync(s->X, s->Y, (size_t)s->nf * s->N * sizeof(double), cudaMemcpyDeviceToDevice,
                                    s->stream), "sweep copy-back");
    if (rc != MC_TVD_OK) return rc;
    return enqueue_initial_dt(s);      // dt now belongs to the swept state (time and step count unchanged)
}

int mc_tvd_debug_geometry(const mc_tvd_state *s, int alpha, int *tile_x, int *tile_b, int *chunk)
{
    if (!s || alpha < 0 || alpha > 2 || !tile_x || !tile_b || !chunk) return fail(MC_TVD_EINVAL, "bad handle, alpha or output pointer");
    *tile_x = s->geom[alpha][0]; *tile_b = s->geom[alpha][1]; *chunk = s->geom[alpha][2];
    return MC_TVD_OK;
}

int mc_tvd_debug_set_chunk(mc_tvd_state *s, int levels)
{
    if (!s || levels < 0) return fail(MC_TVD_EINVAL, "bad handle or levels");
    s->chunk_override = levels;
    return MC_TVD_OK;
}

int mc_tvd_step_host(mc_tvd_state *s, const double *h_in, double *h_out, int n_steps)
{
    if (!s || !h_in || !h_out || n_steps < 0) return fail(MC_TVD_EINVAL, "bad handle, host pointer or n_steps");
    const size_t bytes = (size_t)s->nf * s->N * sizeof(double);
    int rc = cuda_check(cudaMemcpyAsync(s->X, h_in, bytes, cudaMemcpyHostToDevice, s->stream), "state upload");
    if (rc != MC_TVD_OK) return rc;
    mc::Scalars h;
    memset(&h, 0, sizeof(h));
    h.cfl = s->par.cfl; h.fixed_dt = s->par.fixed_dt;
    rc = cuda_check(cudaMemcpyAsync(s->S, &h, sizeof(h), cudaMemcpyHostToDevice, s->stream), "scalar upload");
    if (rc == MC_TVD_OK) rc = cuda_check(cudaStreamSynchronize(s->stream), "upload sync");      // h is on the stack
    if (rc == MC_TVD_OK) rc = enqueue_initial_dt(s);
    if (rc == MC_TVD_OK) rc = mc_tvd_stats_reset(s);                 // time restarts at zero: so does the averaging span
    if (rc == MC_TVD_OK) rc = mc_tvd_step(s, n_steps);
    if (rc == MC_TVD_OK) rc = cuda_check(cudaMemcpyAsync(h_out, s->X, bytes, cudaMemcpyDeviceToHost, s->stream), "state download");
    if (rc == MC_TVD_OK) rc = cuda_check(cudaStreamSynchronize(s->stream), "download sync");
    return rc;
}

int mc_tvd_dt(mc_tvd_state *s, double *dt_host)
{
    if (!s || !dt_host) return fail(MC_TVD_EINVAL, "bad handle or dt_host");
    int rc = cuda_check(cudaMemcpyAsync(dt_host, &s->S->dt, sizeof(double), cudaMemcpyDeviceToHost, s->stream), "dt copy");
    if (rc == MC_TVD_OK) rc = cuda_check(cudaStreamSynchronize(s->stream), "dt sync");
    if (rc != MC_TVD_OK) return rc;
    if (!(*dt_host > 0.0) || !isfinite(*dt_host))
        return fail(MC_TVD_ENONFINITE, "state holds a non-finite value or a non-positive rho or T");
    return MC_TVD_OK;
}

}  // extern "C"

namespace {
mc::DiagArgs diag_args(const mc_tvd_state *s)
{
    mc::DiagArgs G;
    memset(&G, 0, sizeof(G));
    G.partial = s->partial; G.ext = s->ext; G.plane_sums = s->plane_sums; G.out = s->diag_out; G.S = s->S;
    G.nz = s->grid.nz; G.nblk = s->diag_blocks; G.nq = 6 + s->nf; G.walls = s->walls ? 1 : 0;
    G.nplane = (double)s->grid.nx * (double)s->grid.ny;
    G.dz = s->d[2]; G.dxdy = s->d[0] * s->d[1];
    G.eps = s->par.eps; G.D = s->par.D; G.Ra = s->par.Ra; G.Pr = s->par.Pr;
    G.zt = s->zt;
    return G;
}

// Stages 1-2 of the diagnostics (Eqs. 22-26): per-plane sums and extrema of the nodes whose index along own_axis lies in
// [lo, hi) (own_axis = -1: every node) land in s->plane_sums / s->plane_ext.
int enqueue_diag_planes(mc_tvd_state *s, int own_axis, int lo, int hi)
{
    mc::PointArgs P = point_args(s);
    P.own_axis = own_axis; P.own_lo = lo; P.own_hi = hi;
    dim3 grid((unsigned)s->diag_blocks, (unsigned)s->grid.nz, 1);
    if (s->nd == 2) { auto kfn = mc::k_plane_partials<2>; MC_LAUNCH(kfn, grid, mc::DIAG_THREADS, 0, s->stream, P, s->partial, s->ext); }
    else { auto kfn = mc::k_plane_partials<3>; MC_LAUNCH(kfn, grid, mc::DIAG_THREADS, 0, s->stream, P, s->partial, s->ext); }
    mc::DiagArgs G = diag_args(s);
    { auto kfn = mc::k_diag_planes; MC_LAUNCH(kfn, (unsigned)((s->grid.nz + 3) / 4), 128, 0, s->stream, G, s->plane_ext); }
    s->launches += 2;
    return cuda_check(cudaGetLastError(), "diagnostics launch");
}

// Stage 3: plane sums -> the result block in s->diag_out.  nplane: nodes per z plane the sums run over.
int enqueue_diag_finish(mc_tvd_state *s, double nplane)
{
    mc::DiagArgs G = diag_args(s);
    G.nplane = nplane;
    { auto kfn = mc::k_diag_finish; MC_LAUNCH(kfn, 1, mc::DIAG_THREADS, 0, s->stream, G, s->plane_ext); }
    s->launches += 1;
    return cuda_check(cudaGetLastError(), "diagnostics launch");
}

// Enqueue the three diagnostics kernels (Eqs. 22-26): the result block lands in s->diag_out on the device.
int enqueue_diagnostics(mc_tvd_state *s)
{
    int rc = enqueue_diag_planes(s, -1, 0, 0);
    if (rc == MC_TVD_OK) rc = enqueue_diag_finish(s, (double)s->grid.nx * (double)s->grid.ny);
    return rc;
}

// copy the diagnostics block out of s->diag_out (synchronises)
int read_diag_block(mc_tvd_state *s, mc_tvd_diag *out, double *T_prof, double *rho_prof, double *p_prof)
{
    const size_t nz = (size_t)s->grid.nz;
    double *h = (double *)malloc((19 + 3 * nz) * sizeof(double));
    if (!h) return fail(MC_TVD_ENOMEM, "host allocation failed");
    int rc = cuda_check(cudaMemcpyAsync(h, s->diag_out, (19 + 3 * nz) * sizeof(double), cudaMemcpyDeviceToHost, s->stream),
                        "diagnostics copy");
    if (rc == MC_TVD_OK) rc = cuda_check(cudaStreamSynchronize(s->stream), "diagnostics sync");
    if (rc == MC_TVD_OK) {
        memcpy(out, h, sizeof(*out));
        if (T_prof) memcpy(T_prof, h + 19, nz * sizeof(double));
        if (rho_prof) memcpy(rho_prof, h + 19 + nz, nz * sizeof(double));
        if (p_prof) memcpy(p_prof, h + 19 + 2 * nz, nz * sizeof(double));
    }
    free(h);
    return rc;
}

// Enqueue the flow statistics of Sec. 5-6 (flow_stats.cuh): the 16 numbers land in s->flow_out, the histogram of this
// sample is ADDED to s->flow_hist (the caller clears or consumes it).
int enqueue_flow_stats(mc_tvd_state *s)
{
    mc::FlowArgs G;
    memset(&G, 0, sizeof(G));
    G.P = point_args(s);
    G.nx = s->grid.nx; G.ny = s->grid.ny; G.walls = s->walls ? 1 : 0;
    G.mu = s->mu; G.lam = s->par.lambda_coef; G.cv = s->cv;
    G.inv_2dx = 0.5 / s->d[0]; G.inv_dx2 = 1.0 / (s->d[0] * s->d[0]);
    G.inv_2dy = 0.5 / s->d[1]; G.inv_dy2 = 1.0 / (s->d[1] * s->d[1]);
    dim3 grid((unsigned)s->diag_blocks, (unsigned)s->grid.nz, 1);
    if (s->nd == 2) { auto kfn = mc::k_flow_partials<2>; MC_LAUNCH(kfn, grid, mc::DIAG_THREADS, 0, s->stream, G, s->flow_partial, s->flow_ext, s->flow_hist); }
    else { auto kfn = mc::k_flow_partials<3>; MC_LAUNCH(kfn, grid, mc::DIAG_THREADS, 0, s->stream, G, s->flow_partial, s->flow_ext, s->flow_hist); }
    { auto kfn = mc::k_flow_finish; MC_LAUNCH(kfn, 1, mc::DIAG_THREADS, 0, s->stream, G, s->flow_partial, s->flow_ext, s->diag_blocks, s->par.gamma, s->flow_out); }
    s->launches += 2;
    return cuda_check(cudaGetLastError(), "flow statistics launch");
}
}  // namespace

extern "C" {

int mc_tvd_diagnostics(mc_tvd_state *s, mc_tvd_diag *out, double *T_prof, double *rho_prof, double *p_prof)
{
    if (!s || !out) return fail(MC_TVD_EINVAL, "bad handle or out");
    static_assert(sizeof(mc_tvd_diag) == 19 * sizeof(double), "mc_tvd_diag layout");
    int rc = enqueue_diagnostics(s);
    if (rc != MC_TVD_OK) return rc;
    return read_diag_block(s, out, T_prof, rho_prof, p_prof);
}

// ---- slab decomposition hooks (include/mc_tvd.h "Slab decomposition") ------------------------------------------------
int mc_tvd_slab_op(mc_tvd_state *s, int op)
{
    const int nops = s ? 2 * s->nd : 0;
    if (!s || op < 0 || op >= nops) return fail(MC_TVD_EINVAL, "bad handle or operator number");
    if (op != s->slab_next) return fail(MC_TVD_EINVAL, "operators of a step must be enqueued in order, each once");
    const int half = op / s->nd, a = (s->nd == 2) ? (op % 2 == 0 ? 2 : 0) : 2 - (op % 3);      // L_z, [L_y,] L_x (Eq. 30)
    const int dir = (half == 1 && s->par.dir_mode == 1) ? -1 : +1;
    const double *src = (op % 2 == 0) ? s->X : s->Y;
    double *dst = (op % 2 == 0) ? s->Y : s->X;
    // the CFL reduction is fused into the last operator only where it can be restricted to the owned rows (fused halo
    // push); otherwise the halo copies are stale here and mc_tvd_slab_reduce follows the last exchange
    int rc = launch_sweep(s, src, dst, a, dir, 0.0, true, s->slab_fused && op == nops - 1);
    s->ev_open = false;
    if (rc == MC_TVD_OK) s->slab_next = op + 1;
    return rc;
}

int mc_tvd_slab_reduce(mc_tvd_state *s)
{
    if (!s) return fail(MC_TVD_EINVAL, "bad handle");
    if (s->slab_next != 0 && s->slab_next != 2 * s->nd) return fail(MC_TVD_EINVAL, "a step is half done: the state is not in d_fields");
    mc::PointArgs P = point_args(s);
    int blocks = (int)((s->N + 255) / 256);
    if (blocks > 148 * 16) blocks = 148 * 16;
    if (s->nd == 2) { auto kfn = mc::k_max_speed<2>; MC_LAUNCH(kfn, blocks, 256, 0, s->stream, P, &s->S->smax_bits); }
    else { auto kfn = mc::k_max_speed<3>; MC_LAUNCH(kfn, blocks, 256, 0, s->stream, P, &s->S->smax_bits); }
    s->launches += 1;
    return cuda_check(cudaGetLastError(), "max-speed launch");
}

int mc_tvd_slab_commit(mc_tvd_state *s, int advance)
{
    if (!s) return fail(MC_TVD_EINVAL, "bad handle");
    if (advance && s->slab_next != 2 * s->nd) return fail(MC_TVD_EINVAL, "the step's operators have not all been enqueued");
    { auto kfn = mc::k_dt_update; MC_LAUNCH(kfn, 1, 32, 0, s->stream, s->S, advance ? 1 : 0); }
    s->launches += 1;
    if (advance) s->slab_next = 0;
    return cuda_check(cudaGetLastError(), "dt launch");
}

int mc_tvd_slab_buffers(mc_tvd_state *s, double **d_fields, double **d_second)
{
    if (!s || !d_fields || !d_second) return fail(MC_TVD_EINVAL, "bad handle or output pointer");
    *d_fields = s->X; *d_second = s->Y;
    return MC_TVD_OK;
}

int mc_tvd_slab_peers(mc_tvd_state *s, double *lo_fields, double *lo_second, double *hi_fields, double *hi_second,
                      int own_lo, int own_hi, int halo)
{
    if (!s) return fail(MC_TVD_EINVAL, "bad handle");
    if (!lo_fields && !lo_second && !hi_fields && !hi_second) { s->slab_fused = false; return MC_TVD_OK; }
    if (!lo_fields || !lo_second || !hi_fields || !hi_second) return fail(MC_TVD_EINVAL, "all four peer buffers or none");
    if (s->nd != 3 || !s->async3 || s->zt || !s->walls) {
        fail(MC_TVD_EUNSUPPORTED, "the fused halo push serves the 3-D box between plates with an even nx on a uniform z grid");
        return MC_TVD_EUNSUPPORTED;
    }
    if (halo < 2 || own_lo != halo || own_hi <= own_lo + 2 * halo - 1 || own_hi + halo != s->grid.ny)
        return fail(MC_TVD_EINVAL, "owned rows [own_lo, own_hi) must sit between two halos of >= 2 rows each");
    if (s->slab_next != 0) return fail(MC_TVD_EINVAL, "a step is half done");
    s->peer_lo[0] = lo_fields; s->peer_lo[1] = lo_second; s->peer_hi[0] = hi_fields; s->peer_hi[1] = hi_second;
    s->own_lo = own_lo; s->own_hi = own_hi; s->halo = halo;
    s->slab_fused = true;
    return MC_TVD_OK;
}

int mc_tvd_slab_pointers(mc_tvd_state *s, double **fields_now, unsigned long long **smax_bits, double **plane_sums,
                         double **plane_ext)
{
    if (!s) return fail(MC_TVD_EINVAL, "bad handle");
    if (fields_now) *fields_now = (s->slab_next % 2 == 0) ? s->X : s->Y;
    if (smax_bits) *smax_bits = &s->S->smax_bits;
    if (plane_sums) *plane_sums = s->plane_sums;
    if (plane_ext) *plane_ext = s->plane_ext;
    return MC_TVD_OK;
}

int mc_tvd_slab_diag_partial(mc_tvd_state *s, int axis, int lo, int hi)
{
    if (!s || (axis != 0 && axis != 1) || lo < 0 || hi < lo) return fail(MC_TVD_EINVAL, "bad handle, axis or range");
    if (s->slab_next != 0 && s->slab_next != 2 * s->nd) return fail(MC_TVD_EINVAL, "a step is half done: the state is not in d_fields");
    return enqueue_diag_planes(s, axis, lo, hi);
}

int mc_tvd_slab_diag_finish(mc_tvd_state *s, double nplane_global, mc_tvd_diag *out, double *T_prof, double *rho_prof,
                            double *p_prof)
{
    if (!s || !out || !(nplane_global >= 1.0)) return fail(MC_TVD_EINVAL, "bad handle, out or node count");
    int rc = enqueue_diag_finish(s, nplane_global);
    if (rc != MC_TVD_OK) return rc;
    return read_diag_block(s, out, T_prof, rho_prof, p_prof);
}

int mc_tvd_stats_reset(mc_tvd_state *s)
{
    if (!s) return fail(MC_TVD_EINVAL, "bad handle");
    { auto kfn = mc::k_stats_reset; MC_LAUNCH(kfn, 1, 256, 0, s->stream, s->stats, s->S, s->grid.nz); }
    s->launches += 1;
    s->stat_steps = 0;
    int rc = cuda_check(cudaGetLastError(), "stats reset launch");
    if (rc == MC_TVD_OK) rc = cuda_check(cudaMemsetAsync(s->flow_acc, 0, mc::FLOW_NOUT * sizeof(double), s->stream), "flow reset");
    if (rc == MC_TVD_OK) rc = cuda_check(cudaMemsetAsync(s->flow_hist_acc, 0, mc::FLOW_BINS * sizeof(unsigned long long), s->stream), "flow reset");
    if (rc == MC_TVD_OK) rc = cuda_check(cudaMemsetAsync(s->flow_hist, 0, mc::FLOW_BINS * sizeof(unsigned long long), s->stream), "flow reset");
    return rc;
}

int mc_tvd_step_stats(mc_tvd_state *s, int n_steps, int every)
{
    if (!s || n_steps < 0 || every < 1) return fail(MC_TVD_EINVAL, "bad handle, n_steps or every");
    for (int it = 0; it < n_steps; ++it) {
        int rc = mc_tvd_step(s, 1);
        if (rc != MC_TVD_OK) return rc;
        s->stat_steps += 1;
        if (s->stat_steps % every) continue;
        rc = enqueue_diagnostics(s);
        if (rc != MC_TVD_OK) return rc;
        if (s->flow_in_stats) {            // before k_stats_accumulate, which moves the time of the previous sample
            rc = enqueue_flow_stats(s);
            if (rc != MC_TVD_OK) return rc;
            { auto kfn = mc::k_flow_accumulate; MC_LAUNCH(kfn, 1, 128, 0, s->stream, s->flow_acc, s->flow_out, s->stats, s->S, s->flow_hist_acc, s->flow_hist); }
            s->launches += 1;
        }
        { auto kfn = mc::k_stats_accumulate; MC_LAUNCH(kfn, 1, 256, 0, s->stream, s->stats, s->diag_out, s->S, s->grid.nz); }
        s->launches += 1;
        rc = cuda_check(cudaGetLastError(), "stats accumulate launch");
        if (rc != MC_TVD_OK) return rc;
    }
    return MC_TVD_OK;
}

int mc_tvd_stats_read(mc_tvd_state *s, mc_tvd_stats *out, double *T_prof, double *rho_prof, double *p_prof)
{
    if (!s || !out) return fail(MC_TVD_EINVAL, "bad handle or out");
    static_assert(sizeof(mc_tvd_stats) == (4 + mc::ST_NSUM) * sizeof(double), "mc_tvd_stats layout");
    const size_t nz = (size_t)s->grid.nz, n = 4 + mc::ST_NSUM + 3 * nz;
    { auto kfn = mc::k_stats_finish; MC_LAUNCH(kfn, 1, 256, 0, s->stream, s->stats, s->stats_out, s->grid.nz); }
    s->launches += 1;
    int rc = cuda_check(cudaGetLastError(), "stats finish launch");
    if (rc != MC_TVD_OK) return rc;
    double *h = (double *)malloc(n * sizeof(double));
    if (!h) return fail(MC_TVD_ENOMEM, "host allocation failed");
    rc = cuda_check(cudaMemcpyAsync(h, s->stats_out, n * sizeof(double), cudaMemcpyDeviceToHost, s->stream), "stats copy");
    if (rc == MC_TVD_OK) rc = cuda_check(cudaStreamSynchronize(s->stream), "stats sync");
    if (rc == MC_TVD_OK && !(h[3] >= 1.0)) rc = fail(MC_TVD_EINVAL, "no sample has been accumulated since the last mc_tvd_stats_reset");
    if (rc == MC_TVD_OK) {
        out->t_begin = h[0]; out->t_end = h[1]; out->weight = h[2]; out->samples = (long long)h[3];
        memcpy(&out->nu_bottom, h + 4, mc::ST_NSUM * sizeof(double));
        if (T_prof) memcpy(T_prof, h + 4 + mc::ST_NSUM, nz * sizeof(double));
        if (rho_prof) memcpy(rho_prof, h + 4 + mc::ST_NSUM + nz, nz * sizeof(double));
        if (p_prof) memcpy(p_prof, h + 4 + mc::ST_NSUM + 2 * nz, nz * sizeof(double));
    }
    free(h);
    return rc;
}

int mc_tvd_flow_stats(mc_tvd_state *s, mc_tvd_forces *out, long long *hist_r)
{
    if (!s || !out) return fail(MC_TVD_EINVAL, "bad handle or out");
    static_assert(sizeof(mc_tvd_forces) == mc::FLOW_NOUT * sizeof(double), "mc_tvd_forces layout");
    static_assert(MC_TVD_HIST_BINS == mc::FLOW_BINS, "histogram size");
    int rc = cuda_check(cudaMemsetAsync(s->flow_hist, 0, mc::FLOW_BINS * sizeof(unsigned long long), s->stream), "histogram clear");
    if (rc == MC_TVD_OK) rc = enqueue_flow_stats(s);
    unsigned long long h[mc::FLOW_BINS];
    if (rc == MC_TVD_OK) rc = cuda_check(cudaMemcpyAsync(out, s->flow_out, sizeof(*out), cudaMemcpyDeviceToHost, s->stream), "flow copy");
    if (rc == MC_TVD_OK) rc = cuda_check(cudaMemcpyAsync(h, s->flow_hist, sizeof(h), cudaMemcpyDeviceToHost, s->stream), "histogram copy");
    if (rc == MC_TVD_OK) rc = cuda_check(cudaStreamSynchronize(s->stream), "flow sync");
    if (rc == MC_TVD_OK) rc = cuda_check(cudaMemsetAsync(s->flow_hist, 0, sizeof(h), s->stream), "histogram clear");
    if (rc == MC_TVD_OK && hist_r) for (int i = 0; i < mc::FLOW_BINS; ++i) hist_r[i] = (long long)h[i];
    return rc;
}

int mc_tvd_stats_flow(mc_tvd_state *s, int enable)
{
    if (!s) return fail(MC_TVD_EINVAL, "bad handle");
    s->flow_in_stats = enable != 0;
    return MC_TVD_OK;
}

int mc_tvd_stats_read_flow(mc_tvd_state *s, mc_tvd_forces *avg, long long *hist_r)
{
    if (!s || !avg) return fail(MC_TVD_EINVAL, "bad handle or avg");
    double a[mc::FLOW_NOUT];
    unsigned long long h[mc::FLOW_BINS];
    int rc = cuda_check(cudaMemcpyAsync(a, s->flow_acc, sizeof(a), cudaMemcpyDeviceToHost, s->stream), "flow copy");
    if (rc == MC_TVD_OK) rc = cuda_check(cudaMemcpyAsync(h, s->flow_hist_acc, sizeof(h), cudaMemcpyDeviceToHost, s->stream), "histogram copy");
    if (rc == MC_TVD_OK) rc = cuda_check(cudaStreamSynchronize(s->stream), "flow sync");
    if (rc != MC_TVD_OK) return rc;
    if (!(a[11] > 0.0)) return fail(MC_TVD_EINVAL, "no flow sample has been accumulated since the last mc_tvd_stats_reset (see mc_tvd_stats_flow)");
    double *o = &avg->Fn_mean;
    for (int t = 0; t < 4; ++t) { o[t] = a[t] / a[11]; o[4 + t] = sqrt(a[4 + t] / a[11]); }
    for (int t = 8; t < 11; ++t) o[t] = a[t] / a[11];
    o[11] = a[11];                     // `volume` carries the total weight (simulated time averaged over)
    for (int t = 13; t < 16; ++t) o[t] = a[t] / a[11];
    o[12] = o[13] / sqrt(o[14] * o[15]);               // Eq. 49 with <.>_{V,t}
    if (hist_r) for (int i = 0; i < mc::FLOW_BINS; ++i) hist_r[i] = (long long)h[i];
    return MC_TVD_OK;
}

long long mc_tvd_launch_count(const mc_tvd_state *s) { return s ? s->launches : 0; }

int mc_tvd_timing_enable(mc_tvd_state *s, int enable)
{
    if (!s) return fail(MC_TVD_EINVAL, "bad handle");
    if (enable && !s->ev) {
        const int cap = 2 * MC_TVD_MAX_TIMED + 2;
        s->ev = (cudaEvent_t *)calloc(cap, sizeof(cudaEvent_t));
        s->rec_kind = (int *)calloc(MC_TVD_MAX_TIMED, sizeof(int));
        s->rec_ev = (int *)calloc(MC_TVD_MAX_TIMED, sizeof(int));
        if (!s->ev || !s->rec_kind || !s->rec_ev) return fail(MC_TVD_ENOMEM, "host allocation failed");
        for (int i = 0; i < cap; ++i) {
            int rc = cuda_check(cudaEventCreate(&s->ev[i]), "event create");
            if (rc != MC_TVD_OK) return rc;
        }
    }
    s->timing = enable != 0;
    s->ev_open = false;
    return MC_TVD_OK;
}

int mc_tvd_timing_read(mc_tvd_state *s, double *ms_sum, long long *count)
{
    if (!s || !ms_sum || !count) return fail(MC_TVD_EINVAL, "bad handle or output pointer");
    for (int k = 0; k < 6; ++k) { ms_sum[k] = 0.0; count[k] = 0; }
    int rc = cuda_check(cudaStreamSynchronize(s->stream), "timing sync");
    if (rc != MC_TVD_OK) return rc;
    for (int r = 0; r < s->n_rec; ++r) {
        float ms = 0.f;
        rc = cuda_check(cudaEventElapsedTime(&ms, s->ev[s->rec_ev[r]], s->ev[s->rec_ev[r] + 1]), "event elapsed");
        if (rc != MC_TVD_OK) return rc;
        ms_sum[s->rec_kind[r]] += (double)ms;
        count[s->rec_kind[r]] += 1;
    }
    s->n_rec = 0; s->n_ev = 0; s->ev_open = false;
    return MC_TVD_OK;
}

int mc_tvd_destroy(mc_tvd_state *s)
{
    if (!s) return MC_TVD_OK;
    cudaError_t e = cudaStreamSynchronize(s->stream);
    if (s->graph_exec) cudaGraphExecDestroy(s->graph_exec);
    if (s->ev) for (int i = 0; i < 2 * MC_TVD_MAX_TIMED + 2; ++i) if (s->ev[i]) cudaEventDestroy(s->ev[i]);
    free(s->ev); free(s->rec_kind); free(s->rec_ev);
    delete s;
    return cuda_check(e, "destroy sync");
}

}  // extern "C"

// ---------------------------------------------------------------------------------------------
// mc_tvd_cfl_noalloc (include/mc_tvd.h): the CFL reduction with its scratch in a fixed device array instead of a
// caller's workspace -- no allocation anywhere on the call's path.
// ---------------------------------------------------------------------------------------------
// One array per GPU that loads the library, held until the process exits.  Bytes [0, 256): the running maximum (a bit
// pattern, must be 0 when k_max_speed starts).  Then, in doubles: the caller's node heights [0, MAX_NZ), and from
// MAX_NZ on the tables k_max_speed reads as PointArgs::zt with stride nz: z, g z, 1 / cell height.
// In HOST code this name is a host-side stand-in, not a device address: the address comes from cudaGetSymbolAddress.
static __device__ __align__(256) unsigned char g_noalloc_scratch[MC_TVD_NOALLOC_SCRATCH_BYTES];

namespace {

constexpr int NOALLOC_MAX_DEVICES = 64;
std::atomic<unsigned char *> g_noalloc_ptr[NOALLOC_MAX_DEVICES];   // device address of the array, per device ordinal

MC_KERNEL void k_noalloc_clear(unsigned long long *bits)
{
    if (blockIdx.x == 0 && threadIdx.x == 0) *bits = 0ull;
}

// The first three tables of SweepArgs::zt, with the arithmetic of mc_tvd_init's host loop (IEEE subtract, multiply,
// divide: the same bits).
MC_KERNEL void k_noalloc_metric(const double *z, double *zt, int nz, double g)
{
    for (int k = blockIdx.x * blockDim.x + threadIdx.x; k < nz; k += gridDim.x * blockDim.x) {
        const double dzc = (k == 0) ? 0.5 * (z[1] - z[0]) : (k == nz - 1) ? 0.5 * (z[k] - z[k - 1]) : 0.5 * (z[k + 1] - z[k - 1]);
        zt[k] = z[k];
        zt[nz + k] = g * z[k];
        zt[2 * nz + k] = 1.0 / dzc;
    }
}

// out[0] = s, out[1] = the dt of k_dt_update; the array is left cleared for the next call.
MC_KERNEL void k_noalloc_finish(unsigned long long *bits, double *out, double cfl, double fixed_dt)
{
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        const double s = __longlong_as_double((long long)*bits);
        out[0] = s;
        out[1] = (fixed_dt > 0.0) ? fixed_dt : cfl / s;
        *bits = 0ull;
    }
}

// Device address of g_noalloc_scratch on the current device: looked up once per device, with that device current.
int noalloc_scratch(unsigned char **ptr)
{
    int dev = -1;
    int rc = cuda_check(cudaGetDevice(&dev), "cudaGetDevice");
    if (rc != MC_TVD_OK) return rc;
    if (dev < 0 || dev >= NOALLOC_MAX_DEVICES) return fail(MC_TVD_EUNSUPPORTED, "mc_tvd_cfl_noalloc: device ordinal beyond 63");
    unsigned char *p = g_noalloc_ptr[dev].load(std::memory_order_acquire);
    if (!p) {
        void *q = nullptr;
        rc = cuda_check(cudaGetSymbolAddress(&q, g_noalloc_scratch), "cudaGetSymbolAddress(g_noalloc_scratch)");
        if (rc != MC_TVD_OK) return rc;
        if (!q) return fail(MC_TVD_ECUDA, "cudaGetSymbolAddress returned a null address");
        p = (unsigned char *)q;
        g_noalloc_ptr[dev].store(p, std::memory_order_release);   // (two threads racing here store the same address)
    }
    *ptr = p;
    return MC_TVD_OK;
}

}  // namespace

extern "C" int mc_tvd_cfl_noalloc(const mc_tvd_grid *grid, const mc_tvd_params *params, const double *d_fields,
                                  double *d_out, void *cuda_stream)
{
    int code;
    if (!valid_problem(grid, params, &code)) return code;
    if (!d_fields || !d_out) return fail(MC_TVD_EINVAL, "d_fields or d_out is NULL");
    if (((uintptr_t)d_fields & 15) || ((uintptr_t)d_out & 7))
        return fail(MC_TVD_EINVAL, "d_fields must be 16-byte and d_out 8-byte aligned");
    if (grid->nz > MC_TVD_NOALLOC_MAX_NZ) {
        char msg[160];
        snprintf(msg, sizeof(msg), "nz = %d exceeds MC_TVD_NOALLOC_MAX_NZ = %d (the fixed scratch array holds no more levels)",
                 grid->nz, MC_TVD_NOALLOC_MAX_NZ);
        return fail(MC_TVD_EUNSUPPORTED, "mc_tvd_cfl_noalloc: %s", msg);
    }
    unsigned char *scratch = nullptr;
    int rc = noalloc_scratch(&scratch);
    if (rc != MC_TVD_OK) return rc;
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    unsigned long long *bits = (unsigned long long *)scratch;
    double *z_dev = (double *)(scratch + 256);
    double *zt_dev = z_dev + MC_TVD_NOALLOC_MAX_NZ;

    // the constants of mc_tvd_init, on a stack copy of the handle's fields that point_args reads
    mc_tvd_state t;
    memset(&t, 0, sizeof(t));
    t.grid = *grid; t.par = *params;
    t.nd = grid->ndim; t.nf = (grid->ndim == 2) ? 4 : 5;
    t.plane = (long long)grid->nx * grid->ny;
    t.N = t.plane * grid->nz;
    t.walls = (params->bc_z == 0);
    t.d[0] = grid->lx / grid->nx;
    t.d[1] = (grid->ndim == 3) ? grid->ly / grid->ny : 1.0;
    t.d[2] = t.walls ? grid->lz / (grid->nz - 1) : grid->lz / grid->nz;
    t.icv = params->gamma * params->eps * params->D;
    t.R = (params->gamma - 1.0) / t.icv;
    t.g = (params->g_override >= 0.0) ? params->g_override : 1.0 / params->eps;
    t.X = const_cast<double *>(d_fields);                 // read only
    t.zt = nullptr;

    { auto kfn = k_noalloc_clear; MC_LAUNCH(kfn, 1, 32, 0, stream, bits); }
    if (grid->z_nodes) {
        rc = cuda_check(cudaMemcpyAsync(z_dev, grid->z_nodes, (size_t)grid->nz * sizeof(double), cudaMemcpyHostToDevice, stream),
                        "z node upload");
        if (rc != MC_TVD_OK) return rc;
        auto kfn = k_noalloc_metric;
        MC_LAUNCH(kfn, (grid->nz + 255) / 256, 256, 0, stream, z_dev, zt_dev, grid->nz, t.g);
        t.zt = zt_dev;
    }
    mc::PointArgs P = point_args(&t);
    int blocks = (int)((t.N + 255) / 256);
    if (blocks > 148 * 16) blocks = 148 * 16;
    if (t.nd == 2) { auto kfn = mc::k_max_speed<2>; MC_LAUNCH(kfn, blocks, 256, 0, stream, P, bits); }
    else { auto kfn = mc::k_max_speed<3>; MC_LAUNCH(kfn, blocks, 256, 0, stream, P, bits); }
    { auto kfn = k_noalloc_finish; MC_LAUNCH(kfn, 1, 32, 0, stream, bits, d_out, params->cfl, params->fixed_dt); }
    return cuda_check(cudaGetLastError(), "mc_tvd_cfl_noalloc launch");
}
