// bifrost.cu - the single translation unit of libbifrost.so: sm_100a kernels and the C ABI
// (include/bifrost.h) of the BIFROST direct-summation force path of arXiv:2210.02472 - acc
// (Eq. 6/12), grad (Eq. 9/13), dtmin (Eq. 21/22), pn1 (§3.8) - and the NEXT rows built on them.
// See DESIGN.md for the kernel design and the roofline that bounds it.
//
// Layout of the source (all device code lives in anonymous namespaces of this one TU):
//   common.cuh        constants, rsqrt seed, cp.async helpers, SrcArrays, Geom
//   policies.cuh      AccPassT / GradPassT / DtPassT / PotPassT: record, pair(), store(), finish()
//   pair_kernels.cuh  pair_kernel (a2-a4, large sets), pack_kernel (a1), finish_kernel (a5+a7),
//                     pair_fused_kernel (a1-a7 in one launch, small sets)
//   epilogues.cuh     fixed-order W reduction, O(N) time-step criteria
//   pn1.cuh           a6
//   subsystems.cuh    Eq. 20 segment minimum, neighbour search (Eq. 18-19), union-find components
//   integrator.cuh    kick / drift, level split, single-CTA FSI cycle, kinetic energy
//   fp64_probe.cuh    measurement aid
//   bifrost.cu        bifrost_ctx, launch geometry, the *_impl host drivers, the extern "C" API
//
// Design in one paragraph.  The path is bound by the FP64 ALU pipe (64 lanes/clk/SM), so the
// inner loops are written to the minimal number of FP64-pipe instructions per pair
// (acc 15, grad 28, dtmin 25) and everything else (shared-memory broadcast loads, the
// MUFU.RSQ64H seed, integer selects, loop control) rides in the other issue slots.  A CTA owns
// T*S sinks (S per thread, in registers) and a contiguous range of source tiles staged through
// shared memory (cp.async double buffer, warp-wide LDS.128 broadcasts).  When the source range is
// split across CTAs, partials go to a [split][sink] workspace and are reduced in a fixed order
// (deterministic).  Reciprocal square root: y0 = MUFU.RSQ64H(r2) (relative error ~ 2^-20),
// e = 1 - r2*y0^2, then r2^(-3/2) = y0^3 (1 + 3/2 e + 15/8 e^2) and 1/r2 = y0^2 (1 + e + e^2);
// truncation O(e^3) ~ 1e-17.  The source record carries m, 1.5 m, 1.875 m so the polynomial
// yields m * r2^(-3/2) directly.  r2 never reaches 0: R2_FLOOR (or eps^2) is added, so the self
// pair has a finite weight that multiplies a zero separation and contributes exactly 0.

#include "../../include/bifrost.h"

#include <cuda_runtime.h>
#include <cstdio>
#include <cstring>
#include <cstdlib>
#include <cmath>
#include <algorithm>
#include <type_traits>
#include <new>

#include "common.cuh"
#include "policies.cuh"
#include "pair_kernels.cuh"
#include "sym_kernels.cuh"
#include "sym_dt.cuh"
#include "few_sinks.cuh"
#include "epilogues.cuh"
#include "pn1.cuh"
#include "subsystems.cuh"
#include "integrator.cuh"
#include "hhs_subtree.cuh"
#include "fp64_probe.cuh"

// ========================================================================================
// host side
// ========================================================================================

struct bifrost_ctx {
    int device = 0;
    int64_t max_n = 0;
    int num_sms = 0;
    double* src_rec = nullptr;       // packed source records, (max_n rounded up to TILE) * 10 doubles
    size_t src_rec_doubles = 0;
    void* partial = nullptr;         // split-j partials / pn1 partials
    size_t partial_bytes = 0;
    unsigned char* is_bh = nullptr;  // [max_n]
    double* phi_scratch = nullptr;   // [max_n]   (bifrost_potential with out_phi == NULL)
    double* wpart = nullptr;         // [ceil(max_n / 4096)] block partials of the W reduction
    unsigned long long* smin = nullptr;   // [max_n] per-subsystem minima (bifrost_subsys_min)
    int small_m = 128;               // FSI cycles / level splits of at most this many particles run as ONE single-CTA launch
                                     // (bifrost_set_tuning BIFROST_TUNE_SMALL_M: 0..256; 0 disables)
    int64_t fused_max_sinks = 4096;  // below: one fused launch per call (BIFROST_TUNE_FUSED_MAX_SINKS)
    unsigned* tickets = nullptr;     // [TICKETS] arrival counters of pair_fused_kernel (zeroed again by the last CTA of a launch)
    bool tickets_dirty = false;      // a launch failed: counts may be left behind - zero them before the next fused launch
    int shard_rank = 0, shard_world = 1;   // bifrost_set_shard: which blocks of the symmetric kernels this context evaluates
    double* sym_ws = nullptr;        // source-side rows of the symmetric (every pair once) kernels, [block][source][3]
    size_t sym_ws_bytes = 0;
    int64_t few_max_sinks = 32;      // at most this many sinks, and at most few_max_pairs pairs: ONE cluster launch of few_sinks_kernel
    double few_max_pairs[3] = {524288.0, 262144.0, 262144.0};   // (acc, grad, dtmin; BIFROST_TUNE_FEW_MAX_SINKS / _FEW_MAX_PAIRS; 0 sinks
                                     // disables; measured: profiles/r2_sweep_small_sets.md)
    int few_pairs_per_thread = 4;    // the cluster grows (1, 2, .. few_max_cl CTAs) until a thread has at most this many pairs
    int few_max_cl[4] = {0, 0, 0, 0};   // largest cluster the device accepts for the acc / grad / dtmin / acc+jerk instance (0: not asked yet)
    bool fused_cluster = true;       // pair_fused_kernel as clusters with a DSMEM reduction (BIFROST_TUNE_FUSED_CLUSTER: 0 / 1)
    int64_t mutual_min_b = 512;      // bifrost_*_mutual: shortest shorter list / fewest pairs for the two-list symmetric kernel
    double mutual_min_pairs = 5e7;   // (below: two plain calls)
    int64_t sym_min_dt = 32768;      // shortest list for the symmetric dtmin (cross-over near 28000; BIFROST_TUNE_SYM_MIN_N sets it too)
    int64_t sym_min_acc = 16384, sym_min_grad = 12288;   // shortest list the symmetric kernels are used for (measured
                                     // crossover, profiles/r2_symmetric.md; BIFROST_TUNE_SYM_MIN_N sets both)
    const int32_t* subsys = nullptr; // borrowed DEVICE pointer set by bifrost_set_subsystems (NEXT-2), or NULL
    int64_t subsys_n = 0;
    int64_t launches = 0;
    char err[256] = {0};
    // NEXT-4 integrator scratch (allocated on first use of bifrost_fsi_step / bifrost_hhs_fsi)
    bool integ_ready = false;
    double *w_acc = nullptr, *w_grad = nullptr, *w_dtff = nullptr, *w_dtfb = nullptr, *w_dt0 = nullptr;
    double* w_jerk = nullptr;        // jerks of a level's particles (per-level criteria, bifrost_set_level_criteria)
    double lvl_eta = 0.0, lvl_eta_grad = 0.0, lvl_eta_jerk = 0.0;   // Eq. 24-29 at every level of bifrost_hhs_fsi (all 0: off)
    double* w_acc_s = nullptr;       // accelerations of the FSI cycles (rows of a level's slow set), kept between the two H_S of a level
    int32_t *w_order = nullptr, *w_tmp = nullptr;
    int *w_bcount = nullptr, *w_nslow = nullptr;
    int* h_nslow = nullptr;          // pinned
    long long* w_log = nullptr;      // device level log of bifrost_hhs_fsi, [HHS_LOG_ROWS][3], + 3 counters behind it
    long long* h_log = nullptr;      // pinned mirror
    // mirrors for the *_host entry points (allocated on first use)
    bool host_ready = false;
    cudaStream_t hstream = nullptr;
    double *d_pos = nullptr, *d_vel = nullptr, *d_mass = nullptr, *d_acc = nullptr, *d_out = nullptr, *d_dt = nullptr;
    int32_t *d_sink = nullptr, *d_src = nullptr, *d_j = nullptr;
    double* h_stage = nullptr;       // pinned, 3 * max_n doubles
    int32_t* h_stage_i = nullptr;    // pinned, 2 * max_n ints
};

namespace {

#define CU_TRY(ctx, expr)                                                         \
    do {                                                                          \
        cudaError_t e_ = (expr);                                                  \
        if (e_ != cudaSuccess) {                                                  \
            snprintf((ctx)->err, sizeof((ctx)->err), "%s: %s", #expr, cudaGetErrorString(e_)); \
            (ctx)->tickets_dirty = true;                                          \
            return BIFROST_ECUDA;                                                 \
        }                                                                         \
    } while (0)

#define RC_TRY(expr) do { int rc_ = (expr); if (rc_) return rc_; } while (0)

constexpr long long HHS_LOG_ROWS = 1 << 16;      // rows of the device level log of bifrost_hhs_fsi (levels beyond it are counted, not logged)

struct DeviceGuard {
    int prev = -1;
    explicit DeviceGuard(int dev) { cudaGetDevice(&prev); if (prev != dev) cudaSetDevice(dev); else prev = -1; }
    ~DeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};

int check_lists(bifrost_ctx* ctx, int64_t n, const int32_t* sink_idx, int64_t n_sink, const int32_t* src_idx,
                int64_t n_src) {
    if (!ctx) return BIFROST_EINVAL;
    ctx->err[0] = 0;
    if (n < 0 || n > ctx->max_n || n >= (int64_t)1 << 31) return BIFROST_EINVAL;
    if (n_sink < 0 || n_src < 0 || n_sink > ctx->max_n || n_src > ctx->max_n) return BIFROST_EINVAL;
    if (!sink_idx && n_sink != n) return BIFROST_EINVAL;
    if (!src_idx && n_src != n) return BIFROST_EINVAL;
    if (ctx->subsys && ctx->subsys_n != n) return BIFROST_EINVAL;
    return BIFROST_OK;
}

// eps^2 as the kernels use it: never below R2_FLOOR (see rsqrt_seed)
inline double soft2(double eps) { const double e2 = eps * eps; return e2 > R2_FLOOR ? e2 : R2_FLOOR; }

inline int ceil_div(int64_t a, int64_t b) { return (int)((a + b - 1) / b); }

// Source-range split: enough CTAs for ~16 per resident slot (tail < a few %), bounded by the
// number of source tiles, MAX_SPLIT and the partial workspace.
Geom make_geom(const bifrost_ctx* ctx, int64_t n_sink, int64_t n_src, int sinks_per_cta, int resident_per_sm,
               size_t partial_bytes_per_sink, double* model_time = nullptr) {
    Geom g;
    g.n_sink = (int)n_sink;
    g.n_src = (int)n_src;
    g.compact = 0;
    const int n_tiles = ceil_div(n_src, TILE);
    const int ctas_i = ceil_div(n_sink, sinks_per_cta);
    const int64_t slots = (int64_t)ctx->num_sms * resident_per_sm;
    const int64_t target = 16LL * slots;
    int64_t cap = (target + ctas_i - 1) / ctas_i;
    if (cap < 16) cap = 16;                 // room to search for a balanced wave count
    if (cap > n_tiles) cap = n_tiles;
    if (cap > MAX_SPLIT) cap = MAX_SPLIT;
    const int64_t ws_cap = (int64_t)(ctx->partial_bytes / (partial_bytes_per_sink * (size_t)(n_sink > 0 ? n_sink : 1)));
    if (cap > ws_cap) cap = ws_cap;
    if (cap < 1) cap = 1;
    // Wave quantisation: all CTAs cost ~tiles_per_split tile-times (+ a fixed prologue), and the
    // grid runs in ceil(CTAs / slots) waves.  Pick the split with the least modelled time.
    int64_t split = 1;
    double best_t = 0.0;
    for (int64_t s = 1; n_tiles > 0 && s <= cap; ++s) {
        const int64_t tps = (n_tiles + s - 1) / s;
        const int64_t ns = (n_tiles + tps - 1) / tps;
        if (ns != s) continue;
        const int64_t waves = (ctas_i * ns + slots - 1) / slots;
        const double t = (double)waves * ((double)tps + 0.25);
        if (s == 1 || t < best_t * (1.0 - 1e-3)) { best_t = t; split = s; }
    }
    g.tiles_per_split = n_tiles > 0 ? ceil_div(n_tiles, split) : 1;
    g.n_split = n_tiles > 0 ? ceil_div(n_tiles, g.tiles_per_split) : 1;
    // modelled SM time of the launch in (sink x tile) units: waves x tiles per CTA x the CTA's share of an SM
    if (model_time) *model_time = best_t * (double)sinks_per_cta * (double)resident_per_sm;
    return g;
}

// Kernel shapes (S sinks per thread, T threads, MINB resident CTAs per SM, unroll), chosen on B200
// with the steady-state sweep recorded in profiles/ (DESIGN.md §7): large sink sets want the most
// sinks per shared-memory broadcast that the register file allows; small sets want every thread
// to own a distinct sink.
template <int S_, int T_, int MINB_, int UNR_>
struct Shape { static constexpr int S = S_, T = T_, MINB = MINB_, UNR = UNR_; };
using ShapeTiny = Shape<1, 128, 8, 4>;

template <class P, class Sh>
int launch_fused(bifrost_ctx* ctx, const typename P::Args& a, const SrcArrays& src, int64_t n_sink, int64_t n_src,
                 size_t partial_bytes_per_sink, int compact, cudaStream_t st) {
    Geom g = make_geom(ctx, n_sink, n_src, Sh::T * Sh::S, Sh::MINB, partial_bytes_per_sink);
    g.compact = compact;
    dim3 grid(ceil_div(g.n_sink, Sh::T * Sh::S), g.n_split);
    if (grid.x > (unsigned)TICKETS) {            // one ticket per sink block (cannot happen below fused_max_sinks <= TICKETS * 128)
        snprintf(ctx->err, sizeof(ctx->err), "fused launch: %u sink blocks exceed the %d tickets", grid.x, TICKETS);
        return BIFROST_EINVAL;
    }
    if (ctx->tickets_dirty) {
        CU_TRY(ctx, cudaMemsetAsync(ctx->tickets, 0, TICKETS * sizeof(unsigned), st));
        ctx->tickets_dirty = false;
    }
    // vec3 policies with a split source range: clusters of up to 8 CTAs along the split axis add their partials through
    // distributed shared memory (pair_fused_kernel); grid.y is padded to a multiple of the cluster size with CTAs that find
    // no tiles and add zeros
    // A cluster needs 8 free slots in ONE GPC at the same time (a GPC of 18 SMs x 4 slots holds 9 clusters, not 9.25), so a
    // grid sized to fill the GPU in one wave spills into a second one (config 3, 1024 sinks, grad: 285 -> 338 us).  Clusters
    // are used when the launch is short anyway (at most 2 tiles per CTA) or stays below 7/8 of the resident slots
    // (measured: config 2, 33-4095 sinks: acc -3 .. -10 us, grad -2 .. -9 us; config 3, 128 sinks: acc 54.6 -> 41.3 us).
    int cl = 1;
    const int64_t ctas_padded = (int64_t)grid.x * ceil_div(g.n_split, 8) * 8;
    const bool short_launch = g.tiles_per_split <= 2 || 8 * ctas_padded <= 7 * (int64_t)ctx->num_sms * Sh::MINB;
    // (at most 32 sinks: the last CTA has 4-32 lanes per sink for its reduction and is as fast without clusters - the calls of
    // few_sinks_kernel's size that cannot take it, e.g. with subsystems set: 1 sink dtmin 16.2 us against 22.6 with clusters)
    if ((P::CLUSTER_REDUCE || P::CLUSTER_MERGE) && ctx->fused_cluster && g.n_split >= 2 && short_launch && n_sink > 32) {
        cl = g.n_split >= 8 ? 8 : g.n_split >= 4 ? 4 : 2;
        grid.y = (unsigned)(ceil_div(g.n_split, cl) * cl);
    }
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = dim3(Sh::T); cfg.dynamicSmemBytes = 0; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = 1; at[0].val.clusterDim.y = cl; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = cl > 1 ? 1 : 0;
    if (g.tiles_per_split < DT_SHORT_TILES)      // short source range per CTA: the policy's variant for it (dtmin)
        CU_TRY(ctx, cudaLaunchKernelEx(&cfg, pair_fused_kernel<typename P::Short, Sh::S, Sh::T, Sh::MINB, Sh::UNR>, a, g, src, ctx->tickets));
    else
        CU_TRY(ctx, cudaLaunchKernelEx(&cfg, pair_fused_kernel<P, Sh::S, Sh::T, Sh::MINB, Sh::UNR>, a, g, src, ctx->tickets));
    ctx->launches++;
    return BIFROST_OK;
}

// One pass (a1-a7) of policy P.
//   n_sink >= fused_max_sinks: pack -> pair_kernel<Big> -> finish (three launches at most).
//   below: ONE fused launch with 128 threads and S = 4, 2 or 1 sinks per thread - the largest S
//   that still yields >= 4 CTAs per SM (sink blocks x source-range splits), because a small set
//   is short of parallelism, not of registers.
template <class P, class Sh>
int launch_big(bifrost_ctx* ctx, const typename P::Args& a, const Geom& g, cudaStream_t st) {
    dim3 grid(ceil_div(g.n_sink, Sh::T * Sh::S), g.n_split);
    if (g.tiles_per_split < DT_SHORT_TILES)
        pair_kernel<typename P::Short, Sh::S, Sh::T, Sh::MINB, Sh::UNR><<<grid, Sh::T, 0, st>>>(a, g, ctx->src_rec);
    else
        pair_kernel<P, Sh::S, Sh::T, Sh::MINB, Sh::UNR><<<grid, Sh::T, 0, st>>>(a, g, ctx->src_rec);
    ctx->launches++;
    CU_TRY(ctx, cudaGetLastError());
    return BIFROST_OK;
}

// Huge = the shape that is fastest per pair (more sinks per thread; measured gain HUGE_GAIN_PERMILLE),
// Big = a smaller CTA that quantises better over the SMs when there are few sink blocks.  The launch
// model of make_geom (waves x tiles per CTA x sinks per CTA) picks between them per call.
template <class P, class Huge, int HUGE_GAIN_PERMILLE, class Big, class F4, class F2, class F1>
int run_pass(bifrost_ctx* ctx, const typename P::Args& a, const SrcArrays& src, int64_t n_sink, int64_t n_src,
             size_t partial_bytes_per_sink, int compact, cudaStream_t st) {
    Geom g;
    // grad and dtmin (heavier records, more arithmetic per pair) gain from the packed path already at 2048 sinks when the
    // source list is long (config 3, 2048 sinks x 131072 sources: grad 605 -> 518 us, dtmin 628 -> 568 us; config 2's 16384
    // sources: the fused launch stays ahead) - profiles/r2_sweep_small_sets.md
    const bool pack_early = P::PACK_EARLY && n_sink >= 2048 && (double)n_sink * (double)n_src >= 1e8 && ctx->fused_max_sinks >= 2048;
    if (n_sink < ctx->fused_max_sinks && !pack_early) {
        const int64_t splits = std::max<int64_t>(1, std::min<int64_t>(ceil_div(n_src, TILE), MAX_SPLIT));
        const int64_t want = 4LL * ctx->num_sms;
        if ((int64_t)ceil_div(n_sink, 128 * 4) * splits >= want)
            return launch_fused<P, F4>(ctx, a, src, n_sink, n_src, partial_bytes_per_sink, compact, st);
        if ((int64_t)ceil_div(n_sink, 128 * 2) * splits >= want)
            return launch_fused<P, F2>(ctx, a, src, n_sink, n_src, partial_bytes_per_sink, compact, st);
        return launch_fused<P, F1>(ctx, a, src, n_sink, n_src, partial_bytes_per_sink, compact, st);
    }
    if (n_src > 0) {
        const int n_pad = ceil_div(n_src, TILE) * TILE;
        pack_kernel<P><<<ceil_div(n_pad, 256), 256, 0, st>>>((int)n_src, n_pad, src, ctx->src_rec);
        ctx->launches++;
        CU_TRY(ctx, cudaGetLastError());
    }
    double t_big = 0.0, t_huge = 0.0;
    g = make_geom(ctx, n_sink, n_src, Big::T * Big::S, Big::MINB, partial_bytes_per_sink, &t_big);
    const Geom gh = make_geom(ctx, n_sink, n_src, Huge::T * Huge::S, Huge::MINB, partial_bytes_per_sink, &t_huge);
    int rc;
    if (t_huge * (1000 - HUGE_GAIN_PERMILLE) < t_big * 1000) {
        g = gh;
        g.compact = compact;
        rc = launch_big<P, Huge>(ctx, a, g, st);
    } else {
        g.compact = compact;
        rc = launch_big<P, Big>(ctx, a, g, st);
    }
    if (rc) return rc;
    if (g.n_split > 1 || P::ALWAYS_FINISH) {
        finish_kernel<P><<<ceil_div(n_sink, 256), 256, 0, st>>>(a, g);
        ctx->launches++;
        CU_TRY(ctx, cudaGetLastError());
    }
    return BIFROST_OK;
}

// A handful of sinks (few_sinks.cuh): one thread-block cluster, threads over the sources, results merged through shared and
// distributed shared memory - no workspace, one launch.  Returns 1 when the call does not qualify.
template <class F, int WHICH, int CLIDX = WHICH>
int few_impl(bifrost_ctx* ctx, const typename F::Args& a, const SrcArrays& src, int64_t n_sink, int64_t n_src, int compact,
             cudaStream_t st) {
    // 33-128 sinks against at most 16384 sources: one cluster per 32 sinks (config 2: acc 13.4-15.2 -> 11.0 us, grad 16.8-18.0 ->
    // 15.8-16.1, dtmin 128 sinks 26.6 -> 23.4; from 256 sinks on, or with longer lists, the fused kernel's clusters are faster)
    const bool groups = n_sink > FEW_MAX_SINKS;
    if (n_sink < 1 || ctx->shard_world > 1 || ctx->few_max_sinks == 0) return 1;
    if (groups ? (ctx->few_max_sinks < FEW_MAX_SINKS || n_sink > FEW_GROUP_MAX_SINKS || n_src > FEW_GROUP_MAX_SRC) : n_sink > ctx->few_max_sinks) return 1;
    // measured cross-over against the fused kernel (profiles/r2_sweep_small_sets.md): 2^19 pairs for acc, 2^18 for grad and dtmin,
    // four times that for at most 8 sinks (long source lists, where one working thread per CTA of the fused kernel walks its
    // tiles one source after the other: 1 sink x 2^20 sources 264 -> 105 us, 4 sinks x 2^18 sources 71 -> 47 us)
    if (!groups && (double)n_sink * (double)n_src > ctx->few_max_pairs[WHICH] * (n_sink <= 8 ? 4.0 : 1.0)) return 1;
    auto kern = few_sinks_kernel<F>;
    if (ctx->few_max_cl[CLIDX] == 0) {          // once per context and instance: may a cluster have 16 CTAs here?
        int max_cl = 8;                         // the portable size
        if (cudaFuncSetAttribute(kern, cudaFuncAttributeNonPortableClusterSizeAllowed, 1) == cudaSuccess) {
            cudaLaunchConfig_t q = {};
            q.gridDim = dim3(FEW_MAX_CL); q.blockDim = dim3(FEW_T);
            cudaLaunchAttribute at[1];
            at[0].id = cudaLaunchAttributeClusterDimension;
            at[0].val.clusterDim.x = FEW_MAX_CL; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
            q.attrs = at; q.numAttrs = 1;
            int n_clusters = 0;
            if (cudaOccupancyMaxActiveClusters(&n_clusters, kern, &q) == cudaSuccess && n_clusters >= 1) max_cl = FEW_MAX_CL;
        }
        (void)cudaGetLastError();
        ctx->few_max_cl[CLIDX] = max_cl;
    }
    int nsp = 1;
    while (nsp < n_sink && nsp < FEW_MAX_SINKS) nsp *= 2;
    const int n_groups = ceil_div(n_sink, nsp);
    const int n_tiles = ceil_div(n_src, FEW_T);
    int cl = 1;
    while (cl * 2 <= ctx->few_max_cl[CLIDX] && cl * 2 <= n_tiles &&
           (int64_t)cl * FEW_T * ctx->few_pairs_per_thread < (int64_t)nsp * n_src)
        cl *= 2;
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(cl * n_groups); cfg.blockDim = dim3(FEW_T); cfg.dynamicSmemBytes = 0; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = cl; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    CU_TRY(ctx, cudaLaunchKernelEx(&cfg, kern, a, src, (int)n_sink, (int)n_src, nsp, compact));
    ctx->launches++;
    return BIFROST_OK;
}

// acc / grad over one list that is both sink and source set, every pair once (sym_kernels.cuh).
// Returns 1 when the call does not qualify (list too short, workspace too small): the caller then takes the plain path.
constexpr int SYM_ACC_BS = 8 * 256, SYM_GRAD_BS = 6 * 256;   // sinks per CTA of the two symmetric shapes (sym_impl callers)
template <class P, int S, int T, int MINB>
int sym_impl(bifrost_ctx* ctx, int64_t min_n, const double* pos, const double* mass, const double* aux, const int32_t* idx,
             int64_t m, double G, double eps, double* out, int compact, cudaStream_t st) {
    if (m < 2 || !ctx->sym_ws) return 1;
    if (ctx->shard_world > 1) {                 // sharded: the symmetric kernels are the only path (all rows, partial sums)
        if (compact) return BIFROST_EINVAL;
    } else if (m < min_n) return 1;
    SymGeom g;
    g.m = (int)m;
    g.n_tiles = ceil_div(m, TILE);
    g.bs = T * S;
    g.tb = g.bs / TILE;
    g.n_blocks = ceil_div(m, g.bs);
    g.compact = compact;
    g.rank = ctx->shard_rank; g.world = ctx->shard_world;
    g.mutual = 0; g.m_b = 0; g.n_tiles_b = 0; g.rec_b = 0;
    int64_t total = 0;
    for (int b = 0; b < g.n_blocks; ++b) total += sym_range(g, b);
    total = (total + g.world - 1) / g.world;
    const int64_t slots = (int64_t)ctx->num_sms * MINB;
    // ~64 CTAs per SM slot keep the tail of the last wave below ~1 % (measured: 24 -> 64 gains 1.5 %)
    g.unit_tiles = (int)std::max<int64_t>(2, (total + 64 * slots - 1) / (64 * slots));
    // the sink-side pieces must fit the split-j workspace, the source-side rows the symmetric workspace
    const int64_t max_pieces_ws = (int64_t)(ctx->partial_bytes / (24 * (size_t)m));
    if (max_pieces_ws < 1) return 1;
    while (sym_pieces(g, 0) > max_pieces_ws) g.unit_tiles *= 2;
    if (24 * (sym_joff(g, g.n_blocks - 1) + (size_t)sym_range(g, g.n_blocks - 1) * TILE) > ctx->sym_ws_bytes)
        return ctx->shard_world > 1 ? BIFROST_EINVAL : 1;
    const int m_pad = g.n_tiles * TILE;
    sym_pack_kernel<P><<<ceil_div(m_pad, 256), 256, 0, st>>>((int)m, m_pad, idx, pos, mass, aux, ctx->src_rec);
    const SymArgs a{soft2(eps), G, idx, nullptr, out, (double*)ctx->partial, ctx->sym_ws};
    const size_t smem = (2 * TILE * P::REC + (T / 32) * TILE * 3) * sizeof(double);
    dim3 grid(sym_pieces(g, 0), g.n_blocks);
    sym_pair_kernel<P, S, T, MINB, false><<<grid, T, smem, st>>>(a, g, ctx->src_rec);
    sym_finish_kernel<<<ceil_div(m, 128), 128, 0, st>>>(a, g);
    ctx->launches += 3;
    CU_TRY(ctx, cudaGetLastError());
    return BIFROST_OK;
}

// acc / grad between two DISJOINT lists, every (a, b) pair once and both lists served (sym_kernels.cuh, mutual mode):
// the inter-level sums of Eq. 12-13 (S <- F and F <- S) in one pass.  Returns 1 when the call does not qualify (short
// lists, workspace too small, pair sharding active): the caller then issues the two plain calls.
template <class P, int S, int T, int MINB>
int sym_mutual_impl(bifrost_ctx* ctx, const double* pos, const double* mass, const double* aux, const int32_t* idx_a,
                    int64_t m_a, const int32_t* idx_b, int64_t m_b, double G, double eps, double* out, cudaStream_t st) {
    if (!ctx->sym_ws || ctx->shard_world > 1) return 1;
    if (m_a < m_b) { std::swap(idx_a, idx_b); std::swap(m_a, m_b); }     // A (blocks, registers) = the longer list
    if (m_b < ctx->mutual_min_b || (double)m_a * (double)m_b < ctx->mutual_min_pairs) return 1;
    SymGeom g{};
    g.m = (int)m_a;
    g.n_tiles = ceil_div(m_a, TILE);
    g.bs = T * S;
    g.tb = g.bs / TILE;
    g.n_blocks = ceil_div(m_a, g.bs);
    g.rank = 0; g.world = 1;
    g.mutual = 1;
    g.m_b = (int)m_b;
    g.n_tiles_b = ceil_div(m_b, TILE);
    g.rec_b = g.n_tiles * TILE;
    const int64_t slots = (int64_t)ctx->num_sms * MINB;
    const int64_t total = (int64_t)g.n_blocks * g.n_tiles_b;
    g.unit_tiles = (int)std::max<int64_t>(2, (total + 64 * slots - 1) / (64 * slots));
    const int64_t max_pieces_ws = (int64_t)(ctx->partial_bytes / (24 * (size_t)m_a));
    if (max_pieces_ws < 1) return 1;
    while (sym_pieces(g, 0) > max_pieces_ws) g.unit_tiles *= 2;
    if (24 * (size_t)g.n_blocks * g.n_tiles_b * TILE > ctx->sym_ws_bytes) return 1;
    if ((size_t)(g.rec_b + g.n_tiles_b * TILE) * P::REC > ctx->src_rec_doubles) return 1;
    sym_pack_kernel<P><<<ceil_div(g.rec_b, 256), 256, 0, st>>>((int)m_a, g.rec_b, idx_a, pos, mass, aux, ctx->src_rec);
    sym_pack_kernel<P><<<ceil_div(g.n_tiles_b * TILE, 256), 256, 0, st>>>((int)m_b, g.n_tiles_b * TILE, idx_b, pos, mass, aux,
                                                                          ctx->src_rec + (size_t)g.rec_b * P::REC);
    const SymArgs a{soft2(eps), G, idx_a, idx_b, out, (double*)ctx->partial, ctx->sym_ws};
    const size_t smem = (2 * TILE * P::REC + (T / 32) * TILE * 3) * sizeof(double);
    dim3 grid(sym_pieces(g, 0), g.n_blocks);
    sym_pair_kernel<P, S, T, MINB, true><<<grid, T, smem, st>>>(a, g, ctx->src_rec);
    sym_finish_kernel<<<ceil_div(m_a + m_b, 128), 128, 0, st>>>(a, g);
    ctx->launches += 4;
    CU_TRY(ctx, cudaGetLastError());
    return BIFROST_OK;
}

int acc_impl(bifrost_ctx* ctx, int64_t n, const double* pos, const double* mass, const int32_t* sink_idx,
             int64_t n_sink, const int32_t* src_idx, int64_t n_src, double G, double eps, double* out, int compact,
             cudaStream_t st) {
    const int32_t* sub = (ctx->subsys && ctx->subsys_n == n) ? ctx->subsys : nullptr;   // NEXT-2
    if (n_sink == 0) return BIFROST_OK;
    if (ctx->shard_world > 1 && (sub || sink_idx != src_idx || n_sink != n_src || !ctx->sym_ws)) return BIFROST_EINVAL;
    if (!sub && sink_idx == src_idx && n_sink == n_src) {   // one list on both sides: every pair once
        const int rc = sym_impl<SymAcc, 8, 256, 1>(ctx, ctx->sym_min_acc, pos, mass, nullptr, sink_idx, n_sink, G, eps, out, compact, st);
        if (rc <= 0) return rc;
    }
    const SrcArrays src{pos, nullptr, mass, sub, src_idx};
    const AccArgs a{pos, sub, sink_idx, soft2(eps), G, out, (double*)ctx->partial};
    if (!sub) {                                             // a handful of sinks: one cluster launch
        const int rc = few_impl<FewAcc, 0>(ctx, a, src, n_sink, n_src, compact, st);
        if (rc <= 0) return rc;
    }
    using Big = Shape<8, 256, 1, 1>;
    using F4 = Shape<4, 128, 4, 2>;
    using F2 = Shape<2, 128, 6, 2>;
    using F1 = Shape<1, 128, 8, 4>;
    return sub ? run_pass<AccPassT<true>, Big, 0, Big, F4, F2, F1>(ctx, a, src, n_sink, n_src, 24, compact, st)
               : run_pass<AccPassT<false>, Big, 0, Big, F4, F2, F1>(ctx, a, src, n_sink, n_src, 24, compact, st);
}

int grad_impl(bifrost_ctx* ctx, int64_t n, const double* pos, const double* mass, const double* acc,
              const int32_t* sink_idx, int64_t n_sink, const int32_t* src_idx, int64_t n_src, double G, double eps,
              double* out, int compact, cudaStream_t st) {
    const int32_t* sub = (ctx->subsys && ctx->subsys_n == n) ? ctx->subsys : nullptr;   // NEXT-2
    if (n_sink == 0) return BIFROST_OK;
    if (ctx->shard_world > 1 && (sub || sink_idx != src_idx || n_sink != n_src || !ctx->sym_ws)) return BIFROST_EINVAL;
    if (!sub && sink_idx == src_idx && n_sink == n_src) {   // one list on both sides: every pair once
        const int rc = sym_impl<SymGrad, 6, 256, 1>(ctx, ctx->sym_min_grad, pos, mass, acc, sink_idx, n_sink, G, eps, out, compact, st);
        if (rc <= 0) return rc;
    }
    const SrcArrays src{pos, acc, mass, sub, src_idx};
    const GradArgs a{pos, acc, sub, sink_idx, soft2(eps), G, out, (double*)ctx->partial, nullptr, nullptr};
    if (!sub) {
        const int rc = few_impl<FewGrad, 1>(ctx, a, src, n_sink, n_src, compact, st);
        if (rc <= 0) return rc;
    }
    using Huge = Shape<5, 128, 2, 2>;     // phase-major (GradPassT::pairs), 1.6 % faster per pair than Big
    using Big = Shape<4, 256, 1, 2>;
    using F4 = Shape<4, 128, 3, 2>;
    using F2 = Shape<2, 128, 4, 2>;
    using F1 = Shape<1, 128, 5, 2>;
    return sub ? run_pass<GradPassT<true>, Huge, 8, Big, F4, F2, F1>(ctx, a, src, n_sink, n_src, 24, compact, st)
               : run_pass<GradPassT<false>, Huge, 8, Big, F4, F2, F1>(ctx, a, src, n_sink, n_src, 24, compact, st);
}

// Eq. 12 / Eq. 13 between two disjoint lists: out[a] = sum over B, out[b] = sum over A
int acc_mutual_impl(bifrost_ctx* ctx, int64_t n, const double* pos, const double* mass, const int32_t* a_idx, int64_t n_a,
                    const int32_t* b_idx, int64_t n_b, double G, double eps, double* out, cudaStream_t st) {
    if (n_a == 0 || n_b == 0) {                 // one side empty: the other side's sums are empty sums
        if (n_a) RC_TRY(acc_impl(ctx, n, pos, mass, a_idx, n_a, b_idx, 0, G, eps, out, 0, st));
        if (n_b) RC_TRY(acc_impl(ctx, n, pos, mass, b_idx, n_b, a_idx, 0, G, eps, out, 0, st));
        return BIFROST_OK;
    }
    if (!(ctx->subsys && ctx->subsys_n == n)) {
        const int rc = sym_mutual_impl<SymAcc, 8, 256, 1>(ctx, pos, mass, nullptr, a_idx, n_a, b_idx, n_b, G, eps, out, st);
        if (rc <= 0) return rc;
    }
    RC_TRY(acc_impl(ctx, n, pos, mass, a_idx, n_a, b_idx, n_b, G, eps, out, 0, st));
    return acc_impl(ctx, n, pos, mass, b_idx, n_b, a_idx, n_a, G, eps, out, 0, st);
}
int grad_mutual_impl(bifrost_ctx* ctx, int64_t n, const double* pos, const double* mass, const double* acc, const int32_t* a_idx,
                     int64_t n_a, const int32_t* b_idx, int64_t n_b, double G, double eps, double* out, cudaStream_t st) {
    if (n_a == 0 || n_b == 0) {
        if (n_a) RC_TRY(grad_impl(ctx, n, pos, mass, acc, a_idx, n_a, b_idx, 0, G, eps, out, 0, st));
        if (n_b) RC_TRY(grad_impl(ctx, n, pos, mass, acc, b_idx, n_b, a_idx, 0, G, eps, out, 0, st));
        return BIFROST_OK;
    }
    if (!(ctx->subsys && ctx->subsys_n == n)) {
        const int rc = sym_mutual_impl<SymGrad, 6, 256, 1>(ctx, pos, mass, acc, a_idx, n_a, b_idx, n_b, G, eps, out, st);
        if (rc <= 0) return rc;
    }
    RC_TRY(grad_impl(ctx, n, pos, mass, acc, a_idx, n_a, b_idx, n_b, G, eps, out, 0, st));
    return grad_impl(ctx, n, pos, mass, acc, b_idx, n_b, a_idx, n_a, G, eps, out, 0, st);
}

// acceleration (Eq. 6) and jerk (Eq. 28) in one pass: GradPassT<EXCL, true> over (x, v, m) records
int acc_jerk_impl(bifrost_ctx* ctx, int64_t n, const double* pos, const double* vel, const double* mass,
                  const int32_t* sink_idx, int64_t n_sink, const int32_t* src_idx, int64_t n_src, double G, double eps,
                  double* out_acc, double* out_jerk, cudaStream_t st) {
    const int32_t* sub = (ctx->subsys && ctx->subsys_n == n) ? ctx->subsys : nullptr;
    if (n_sink == 0) return BIFROST_OK;
    const SrcArrays src{pos, vel, mass, sub, src_idx};
    double* p1 = (double*)ctx->partial;
    double* p2 = (double*)((char*)ctx->partial + ctx->partial_bytes / 2);
    const GradArgs a{pos, vel, sub, sink_idx, soft2(eps), G, out_jerk, p1, out_acc, p2};
    if (!sub) {                                             // a handful of sinks: one cluster launch (grad's thresholds)
        const int rc = few_impl<FewAccJerk, 1, 3>(ctx, a, src, n_sink, n_src, 0, st);
        if (rc <= 0) return rc;
    }
    using Big = Shape<4, 256, 1, 2>;
    using F4 = Shape<4, 128, 2, 2>;       // 9 accumulators per sink: two CTAs per SM keep it out of local memory
    using F2 = Shape<2, 128, 4, 2>;
    using F1 = Shape<1, 128, 5, 2>;
    using Huge = Shape<5, 128, 1, 2>;     // phase-major, 4 % faster per pair than Big (2100 vs 2188 ms at N = 2^20)
    return sub ? run_pass<GradPassT<true, true>, Huge, 40, Big, F4, F2, F1>(ctx, a, src, n_sink, n_src, 48, 0, st)
               : run_pass<GradPassT<false, true>, Huge, 40, Big, F4, F2, F1>(ctx, a, src, n_sink, n_src, 48, 0, st);
}

// dtmin over one list that is both sink and source set, every pair once (sym_dt.cuh).  Returns 1 when the call does not qualify.
int sym_dt_impl(bifrost_ctx* ctx, const double* pos, const double* vel, const double* mass, const int32_t* idx, int64_t m, double G,
                double eta_ff, double eta_fb, double* dt_ff, double* dt_fb, int32_t* j_ff, int32_t* j_fb, int compact, cudaStream_t st) {
    // 6 sinks x 128 threads x 2 CTAs/SM, unroll 2 (254 registers, no spill): 665 ms at N = 2^20; 3 x 128 x 3 unroll 4: 681;
    // 4 x 128 x 3 unroll 4 (168 registers, spills): 690; 6 x 256 x 1: 698; 4 x 128 x 2: 771 (profiles/r2_dtmin.md)
    constexpr int S = 6, T = 128, MINB = 2, UNR = 2;
    if (m < ctx->sym_min_dt || m < 2 || !ctx->sym_ws || ctx->shard_world > 1) return 1;
    SymGeom g{};
    g.m = (int)m;
    g.n_tiles = ceil_div(m, TILE);
    g.bs = T * S;
    g.tb = g.bs / TILE;
    g.n_blocks = ceil_div(m, g.bs);
    g.compact = compact;
    g.rank = 0; g.world = 1;
    int64_t total = 0;
    for (int b = 0; b < g.n_blocks; ++b) total += sym_range(g, b);
    const int64_t slots = (int64_t)ctx->num_sms * MINB;
    g.unit_tiles = (int)std::max<int64_t>(2, (total + 64 * slots - 1) / (64 * slots));
    const int64_t max_pieces_ws = (int64_t)(ctx->partial_bytes / (sizeof(DtBest) * (size_t)m));
    if (max_pieces_ws < 2) return 1;
    while (sym_pieces(g, 0) > max_pieces_ws) g.unit_tiles *= 2;
    // the symmetric workspace holds: best[m], lock[m], two counters, the candidate list (the rest)
    char* ws = (char*)ctx->sym_ws;
    const size_t off_lock = sizeof(DtBest) * (size_t)m, off_cnt = (off_lock + 4 * (size_t)m + 15) & ~(size_t)15, off_cand = off_cnt + 16;
    if (ctx->sym_ws_bytes < off_cand + ((size_t)64 << 20)) return 1;
    SymDtArgs a{};
    a.d = DtArgs{pos, vel, mass, nullptr, idx, idx, (int)m, nullptr, nullptr, G, eta_ff, eta_fb, dt_ff, dt_fb, j_ff, j_fb, NgbArgs{}};
    a.idx = idx;
    a.pieces = (DtBest*)ctx->partial;
    a.best = (DtBest*)ws;
    a.lock = (int*)(ws + off_lock);
    a.counters = (unsigned long long*)(ws + off_cnt);
    a.cand = (DtCand*)(ws + off_cand);
    a.cand_cap = (ctx->sym_ws_bytes - off_cand) / sizeof(DtCand);
    a.hint_ff = ctx->smin;
    a.hint_fb = (unsigned long long*)ctx->phi_scratch;
    const int n_pad = g.n_tiles * TILE;
    const SrcArrays src{pos, vel, mass, nullptr, idx};
    pack_kernel<DtPassT<false>><<<ceil_div(n_pad, 256), 256, 0, st>>>((int)m, n_pad, src, ctx->src_rec);
    CU_TRY(ctx, cudaMemsetAsync(a.counters, 0, 16, st));
    sym_dt_kernel<S, T, MINB, UNR><<<dim3(sym_diag_pieces(g, 0), g.n_blocks), T, 0, st>>>(a, g, ctx->src_rec, 0);
    sym_dt_hint_kernel<<<ceil_div(m, 256), 256, 0, st>>>(a, g);
    sym_dt_kernel<S, T, MINB, UNR><<<dim3(sym_pieces(g, 0), g.n_blocks), T, 0, st>>>(a, g, ctx->src_rec, 1);
    sym_dt_merge_kernel<<<ceil_div(m, 128), 128, 0, st>>>(a, g);
    sym_dt_apply_kernel<<<ctx->num_sms * 8, 256, 0, st>>>(a);
    sym_dt_final_kernel<<<ceil_div(m, 128), 128, 0, st>>>(a, g);
    ctx->launches += 7;
    CU_TRY(ctx, cudaGetLastError());
    return BIFROST_OK;
}

// ng == NULL: bifrost_dtmin; else the neighbour search of Eq. 18-19 rides on the same pass (bifrost_dtmin_neighbours)
int dtmin_impl(bifrost_ctx* ctx, int64_t n, const double* pos, const double* vel, const double* mass,
               const int32_t* sink_idx, int64_t n_sink, const int32_t* src_idx, int64_t n_src, double G,
               double eta_ff, double eta_fb, double* dt_ff, double* dt_fb, int32_t* j_ff, int32_t* j_fb, int compact,
               cudaStream_t st, const NgbArgs* ng = nullptr) {
    const int32_t* sub = (ctx->subsys && ctx->subsys_n == n) ? ctx->subsys : nullptr;   // NEXT-2
    if (n_sink == 0) return BIFROST_OK;
    if (!ng && !sub && sink_idx == src_idx && n_sink == n_src) {   // one list on both sides: every pair once
        const int rc = sym_dt_impl(ctx, pos, vel, mass, sink_idx, n_sink, G, eta_ff, eta_fb, dt_ff, dt_fb, j_ff, j_fb, compact, st);
        if (rc <= 0) return rc;
    }
    if (!ng && !sub) {                                      // a handful of sinks: one cluster launch, exact time-steps for every pair
        const DtArgs fa{pos, vel, mass, nullptr, sink_idx, src_idx, (int)n_src, nullptr, nullptr, G, eta_ff, eta_fb,
                        dt_ff, dt_fb, j_ff, j_fb, NgbArgs{}};
        const SrcArrays fsrc{pos, vel, mass, nullptr, src_idx};
        const int rc = few_impl<FewDt, 2>(ctx, fa, fsrc, n_sink, n_src, compact, st);
        if (rc <= 0) return rc;
    }
    // workspace per sink and split: 16 B of time-steps, 8 B of ids [, 4 B neighbour count + 4 cap B of list]; the regions
    // share ctx->partial in those proportions, so whatever split count fits the whole fits every region
    const size_t per_sink = 24 + (ng ? 4 * ((size_t)ng->cap + 1) : 0);
    const size_t unit = (ctx->partial_bytes / per_sink) & ~(size_t)15;    // "sinks x splits" the workspace holds
    char* base = (char*)ctx->partial;
    double* pkey = (double*)base;
    int32_t* pid = (int32_t*)(base + unit * 16);
    const SrcArrays src{pos, vel, mass, sub, src_idx};
    DtArgs a{pos, vel, mass, sub, sink_idx, src_idx, (int)n_src, pkey, pid, G, eta_ff, eta_fb, dt_ff, dt_fb, j_ff, j_fb, NgbArgs{}};
    // 17 FP64 instructions per pair in the hot path: 4 sinks x 128 threads x 3 CTAs/SM, unroll 2 measured best at every size
    // (N = 2^20: 1193 ms; 6 x 128 x 2 CTAs unroll 2: 1196; unroll 1: 1234 / 1283; 8 x 128 x 2: 1346; profiles/r2_dtmin.md)
    using Huge = Shape<4, 128, 3, 2>;
    using Big = Shape<4, 128, 3, 2>;
    using F4 = Shape<4, 128, 3, 2>;
    using F2 = Shape<2, 128, 4, 2>;
    using F1 = Shape<1, 128, 5, 4>;
    if (ng) {
        a.ng = *ng;
        a.ng.n_rows = (int)n_sink;
        a.ng.pcount = (int32_t*)(base + unit * 24);
        a.ng.plist = (int32_t*)(base + unit * 28);
        // the neighbour test keeps r^2 and a count per sink alive: one sink fewer per thread fits the register file
        using HugeN = Shape<4, 128, 2, 2>;
        using BigN = Shape<4, 128, 2, 2>;
        using F4N = Shape<4, 128, 2, 2>;
        using F2N = Shape<2, 128, 3, 2>;
        return sub ? run_pass<DtPassT<true, true>, HugeN, 7, BigN, F4N, F2N, F1>(ctx, a, src, n_sink, n_src, per_sink, compact, st)
                   : run_pass<DtPassT<false, true>, HugeN, 7, BigN, F4N, F2N, F1>(ctx, a, src, n_sink, n_src, per_sink, compact, st);
    }
    return sub ? run_pass<DtPassT<true>, Huge, 7, Big, F4, F2, F1>(ctx, a, src, n_sink, n_src, 24, compact, st)
               : run_pass<DtPassT<false>, Huge, 7, Big, F4, F2, F1>(ctx, a, src, n_sink, n_src, 24, compact, st);
}

int pot_impl(bifrost_ctx* ctx, int64_t n, const double* pos, const double* mass, const int32_t* sink_idx,
             int64_t n_sink, const int32_t* src_idx, int64_t n_src, double G, double eps, double* out_phi,
             double* out_W, cudaStream_t st) {
    const int32_t* sub = (ctx->subsys && ctx->subsys_n == n) ? ctx->subsys : nullptr;   // NEXT-2
    if (n_sink == 0) {
        if (out_W) CU_TRY(ctx, cudaMemsetAsync(out_W, 0, sizeof(double), st));
        return BIFROST_OK;
    }
    const int compact = out_phi ? 0 : 1;           // the scratch holds compact rows
    double* phi = out_phi ? out_phi : ctx->phi_scratch;
    const SrcArrays src{pos, nullptr, mass, sub, src_idx};
    const PotArgs a{pos, sub, sink_idx, soft2(eps), G, phi, (double*)ctx->partial};
    using Big = Shape<4, 128, 4, 2>;
    using F2 = Shape<2, 128, 6, 2>;
    using F1 = Shape<1, 128, 8, 4>;
    using Huge = Shape<8, 128, 2, 1>;     // 5 % faster per pair than Big (profiles/r1_shape_tuning.md)
    int rc = sub ? run_pass<PotPassT<true>, Huge, 50, Big, Big, F2, F1>(ctx, a, src, n_sink, n_src, 8, compact, st)
                 : run_pass<PotPassT<false>, Huge, 50, Big, Big, F2, F1>(ctx, a, src, n_sink, n_src, 8, compact, st);
    if (rc) return rc;
    if (out_W) {
        const int nb = ceil_div(n_sink, WSUM_PER_BLOCK);
        wsum_stage1_kernel<<<nb, WSUM_THREADS, 0, st>>>((int)n_sink, sink_idx, compact, mass, phi, ctx->wpart);
        wsum_stage2_kernel<<<1, WSUM_THREADS, 0, st>>>(nb, ctx->wpart, out_W);
        ctx->launches += 2;
        CU_TRY(ctx, cudaGetLastError());
    }
    return BIFROST_OK;
}

int pn1_impl(bifrost_ctx* ctx, int64_t n, const double* pos, const double* vel, const double* mass,
             const int32_t* bh_idx, int64_t n_bh, double G, double c, double* out, cudaStream_t st) {
    if (n == 0) return BIFROST_OK;
    const double inv_c2 = 1.0 / (c * c);
    const int32_t* sub = ctx->subsys;   // NEXT-2; length checked by the caller
    pn1_from_bh_kernel<<<ceil_div(n, PN_THREADS), PN_THREADS, 0, st>>>((int)n, (int)n_bh, bh_idx, pos, vel, mass, sub, G,
                                                                      inv_c2, out);
    ctx->launches++;
    CU_TRY(ctx, cudaGetLastError());
    if (n_bh == 0) return BIFROST_OK;
    CU_TRY(ctx, cudaMemsetAsync(ctx->is_bh, 0, (size_t)n, st));
    pn1_flag_kernel<<<ceil_div(n_bh, 256), 256, 0, st>>>((int)n_bh, bh_idx, ctx->is_bh);
    ctx->launches++;
    // chunks: bounded by the partial workspace and by useful parallelism
    int64_t n_chunks = ceil_div(n, 16384);
    const int64_t cap = (int64_t)(ctx->partial_bytes / (24 * (size_t)n_bh));
    if (n_chunks > cap) n_chunks = cap;
    if (n_chunks > 65535) n_chunks = 65535;
    if (n_chunks < 1) n_chunks = 1;
    const int chunk = ceil_div(n, n_chunks);
    n_chunks = ceil_div(n, chunk);
    // grid.y is limited to 65535 BHs per launch
    for (int64_t b0 = 0; b0 < n_bh; b0 += 65535) {
        const int nb = (int)((n_bh - b0 < 65535) ? (n_bh - b0) : 65535);
        dim3 grid((unsigned)n_chunks, (unsigned)nb);
        pn1_on_bh_kernel<<<grid, PN_RED_THREADS, 0, st>>>((int)n, chunk, bh_idx + b0, ctx->is_bh, pos, vel, mass, sub, G, inv_c2,
                                                          (double*)ctx->partial + 3 * (size_t)b0 * n_chunks);
        ctx->launches++;
    }
    pn1_bh_finalize_kernel<<<ceil_div(n_bh, 128), 128, 0, st>>>((int)n_bh, (int)n_chunks, bh_idx,
                                                               (const double*)ctx->partial, out);
    ctx->launches++;
    CU_TRY(ctx, cudaGetLastError());
    return BIFROST_OK;
}

int ensure_host_mirrors(bifrost_ctx* ctx) {
    if (ctx->host_ready) return BIFROST_OK;
    const size_t n = (size_t)ctx->max_n;
    CU_TRY(ctx, cudaStreamCreateWithFlags(&ctx->hstream, cudaStreamNonBlocking));
    CU_TRY(ctx, cudaMalloc(&ctx->d_pos, 24 * n));
    CU_TRY(ctx, cudaMalloc(&ctx->d_vel, 24 * n));
    CU_TRY(ctx, cudaMalloc(&ctx->d_mass, 8 * n));
    CU_TRY(ctx, cudaMalloc(&ctx->d_acc, 24 * n));
    CU_TRY(ctx, cudaMalloc(&ctx->d_out, 24 * n));
    CU_TRY(ctx, cudaMalloc(&ctx->d_dt, 16 * n));
    CU_TRY(ctx, cudaMalloc(&ctx->d_sink, 4 * n));
    CU_TRY(ctx, cudaMalloc(&ctx->d_src, 4 * n));
    CU_TRY(ctx, cudaMalloc(&ctx->d_j, 8 * n));
    CU_TRY(ctx, cudaMallocHost(&ctx->h_stage, 24 * n));
    CU_TRY(ctx, cudaMallocHost(&ctx->h_stage_i, 8 * n));
    ctx->host_ready = true;
    return BIFROST_OK;
}

// copy compact device rows back and scatter them to out[sink id] on the host (marshalling only)
int fetch_rows(bifrost_ctx* ctx, const void* d_rows, size_t row_bytes, const int32_t* sink_idx, int64_t n_sink,
               void* h_out, void* h_stage) {
    if (!h_out) return BIFROST_OK;
    if (!sink_idx) {
        CU_TRY(ctx, cudaMemcpyAsync(h_out, d_rows, row_bytes * (size_t)n_sink, cudaMemcpyDeviceToHost, ctx->hstream));
        CU_TRY(ctx, cudaStreamSynchronize(ctx->hstream));
        return BIFROST_OK;
    }
    CU_TRY(ctx, cudaMemcpyAsync(h_stage, d_rows, row_bytes * (size_t)n_sink, cudaMemcpyDeviceToHost, ctx->hstream));
    CU_TRY(ctx, cudaStreamSynchronize(ctx->hstream));
    for (int64_t k = 0; k < n_sink; ++k)
        memcpy((char*)h_out + row_bytes * (size_t)sink_idx[k], (const char*)h_stage + row_bytes * (size_t)k, row_bytes);
    return BIFROST_OK;
}

// ---- NEXT-4: FSI cycle and HHS-FSI driver (host logic around the kernels above) ------------

int ensure_integrator(bifrost_ctx* ctx) {
    if (ctx->integ_ready) return BIFROST_OK;
    const size_t n = (size_t)ctx->max_n;
    CU_TRY(ctx, cudaMalloc(&ctx->w_acc, 24 * n));
    CU_TRY(ctx, cudaMalloc(&ctx->w_grad, 24 * n));
    CU_TRY(ctx, cudaMalloc(&ctx->w_acc_s, 24 * n));
    CU_TRY(ctx, cudaMalloc(&ctx->w_jerk, 24 * n));
    CU_TRY(ctx, cudaMalloc(&ctx->w_dtff, 8 * n));
    CU_TRY(ctx, cudaMalloc(&ctx->w_dtfb, 8 * n));
    CU_TRY(ctx, cudaMalloc(&ctx->w_dt0, 8 * n));
    CU_TRY(ctx, cudaMalloc(&ctx->w_order, 4 * n));
    CU_TRY(ctx, cudaMalloc(&ctx->w_tmp, 4 * n));
    CU_TRY(ctx, cudaMalloc(&ctx->w_bcount, 4 * (n / PART_T + 1)));
    CU_TRY(ctx, cudaMalloc(&ctx->w_nslow, 4));
    CU_TRY(ctx, cudaMallocHost(&ctx->h_nslow, 4));
    CU_TRY(ctx, cudaMalloc(&ctx->w_log, sizeof(long long) * (3 * HHS_LOG_ROWS + 3)));
    CU_TRY(ctx, cudaMallocHost(&ctx->h_log, sizeof(long long) * (3 * HHS_LOG_ROWS + 3)));
    ctx->integ_ready = true;
    return BIFROST_OK;
}

int kick_impl(bifrost_ctx* ctx, const int32_t* idx, int64_t m, const double* acc, const double* grad, double h, double c,
              double* vel, cudaStream_t st) {
    if (m == 0) return BIFROST_OK;
    kick_kernel<<<ceil_div(m, 256), 256, 0, st>>>((int)m, idx, acc, grad, h, c, vel);
    ctx->launches++;
    CU_TRY(ctx, cudaGetLastError());
    return BIFROST_OK;
}
int drift_impl(bifrost_ctx* ctx, const int32_t* idx, int64_t m, const double* vel, double h, double* pos, cudaStream_t st) {
    if (m == 0) return BIFROST_OK;
    drift_kernel<<<ceil_div(m, 256), 256, 0, st>>>((int)m, idx, vel, h, pos);
    ctx->launches++;
    CU_TRY(ctx, cudaGetLastError());
    return BIFROST_OK;
}

// Eq. 10 over the particles idx[0..m) interacting among themselves (idx == NULL: all n).
// first_acc_valid: w_acc_s already holds the accelerations of this set at the current positions (left there by the
// previous cycle over the same set, no drift of its particles since) - the opening sum is then skipped.  Eq. 11 has
// exactly this situation: between the two H_S of a level only the fast particles move and the slow ones are kicked.
int fsi_impl(bifrost_ctx* ctx, int64_t n, double* pos, double* vel, const double* mass, const int32_t* idx, int64_t m,
             double G, double eps_soft, double eps, cudaStream_t st, bool first_acc_valid = false) {
    if (m == 0) return BIFROST_OK;
    const bool excl = ctx->subsys && ctx->subsys_n == n;
    if (m <= ctx->small_m && !excl) {                      // one launch for the whole cycle
        fsi_small_kernel<<<1, SMALL_M, 0, st>>>((int)m, idx, pos, vel, mass, G, soft2(eps_soft), eps);
        ctx->launches++;
        CU_TRY(ctx, cudaGetLastError());
        return BIFROST_OK;
    }
    double* a = ctx->w_acc_s;
    double* g = ctx->w_grad;
    if (!first_acc_valid) RC_TRY(acc_impl(ctx, n, pos, mass, idx, m, idx, m, G, eps_soft, a, 0, st));
    RC_TRY(kick_impl(ctx, idx, m, a, nullptr, eps / 6.0, 0.0, vel, st));
    RC_TRY(drift_impl(ctx, idx, m, vel, eps / 2.0, pos, st));
    RC_TRY(acc_impl(ctx, n, pos, mass, idx, m, idx, m, G, eps_soft, a, 0, st));
    RC_TRY(grad_impl(ctx, n, pos, mass, a, idx, m, idx, m, G, eps_soft, g, 0, st));
    RC_TRY(kick_impl(ctx, idx, m, a, g, 2.0 * eps / 3.0, eps * eps / 24.0, vel, st));
    RC_TRY(drift_impl(ctx, idx, m, vel, eps / 2.0, pos, st));
    RC_TRY(acc_impl(ctx, n, pos, mass, idx, m, idx, m, G, eps_soft, a, 0, st));
    RC_TRY(kick_impl(ctx, idx, m, a, nullptr, eps / 6.0, 0.0, vel, st));
    return BIFROST_OK;
}

// a host-steered level appends its row to the device log (the subtree kernel appends its own): one ordered log
__global__ void hhs_log_kernel(long long* log, long long* counters, long long cap, int depth, const int* n_slow, int m) {
    const long long row = counters[0];
    if (row < cap) { log[3 * row] = depth; log[3 * row + 1] = *n_slow; log[3 * row + 2] = m - *n_slow; }
    counters[0] = row + 1;
    if (depth > counters[1]) counters[1] = depth;
}

struct Hhs {
    bifrost_ctx* ctx; int64_t n; double* pos; double* vel; const double* mass;
    double G, eps_soft, eta_ff, eta_fb; const double* dt_cap; int max_depth; cudaStream_t st;
    int64_t* log; int64_t log_cap; int64_t n_levels; int64_t deepest; int64_t fsi_steps;
};

// One level of Eq. 11 over order[lo, hi) for an interval tau.
int hhs_level(Hhs& h, int64_t lo, int64_t hi, double tau, int depth) {
    bifrost_ctx* ctx = h.ctx;
    const int64_t m = hi - lo;
    if (m == 0) return BIFROST_OK;
    cudaStream_t st = h.st;
    int32_t* seg = ctx->w_order + lo;
    const bool level_crit = ctx->lvl_eta > 0.0 || ctx->lvl_eta_grad > 0.0 || ctx->lvl_eta_jerk > 0.0;
    if (m <= ctx->small_m && m <= SUB_M) {
        // the whole subtree below a small level in one single-CTA launch: no device -> host read, no further launches
        const SubArgs sa{(int)m, seg, h.pos, h.vel, h.mass, ctx->w_dt0, h.dt_cap, h.G, soft2(h.eps_soft), h.eta_ff, h.eta_fb, tau,
                         level_crit ? ctx->lvl_eta : 0.0, ctx->lvl_eta_grad, ctx->lvl_eta_jerk, depth, h.max_depth, ctx->w_log, HHS_LOG_ROWS, ctx->w_log + 3 * HHS_LOG_ROWS};
        hhs_subtree_kernel<<<1, SUB_M, 0, st>>>(sa);
        ctx->launches++;
        CU_TRY(ctx, cudaGetLastError());
        return BIFROST_OK;
    }
    const int all_slow = depth >= h.max_depth;
    if (!all_slow)   // time-steps of the level's particles among themselves (Eq. 21-22)
        RC_TRY(dtmin_impl(ctx, h.n, h.pos, h.vel, h.mass, seg, m, seg, m, h.G, h.eta_ff, h.eta_fb, ctx->w_dtff, ctx->w_dtfb,
                          nullptr, nullptr, 0, st));
    if (!all_slow && level_crit) {
        // "the final time-step of a particle is the minimum of the set of its different time-steps" - the
        // acceleration-based criteria (Eq. 24-29) of the level's particles among themselves, folded into eps_ff's row; the
        // level-0 cap of L295 is applied by the flag kernels as before.  w_acc / w_grad are free until the inter-level sums.
        RC_TRY(acc_jerk_impl(ctx, h.n, h.pos, h.vel, h.mass, seg, m, seg, m, h.G, h.eps_soft, ctx->w_acc, ctx->w_jerk, st));
        RC_TRY(grad_impl(ctx, h.n, h.pos, h.mass, ctx->w_acc, seg, m, seg, m, h.G, h.eps_soft, ctx->w_grad, 0, st));
        criteria_kernel<<<ceil_div(m, 256), 256, 0, st>>>((int)m, seg, h.vel, ctx->w_acc, ctx->w_grad, ctx->w_jerk, ctx->lvl_eta,
                                                         ctx->lvl_eta_grad, ctx->lvl_eta_jerk, nullptr, nullptr, nullptr, nullptr,
                                                         ctx->w_dtff);
        ctx->launches++;
        CU_TRY(ctx, cudaGetLastError());
    }
    if (m <= ctx->small_m) {
        level_split_small_kernel<<<1, SMALL_M, 0, st>>>((int)m, seg, ctx->w_dtff, ctx->w_dtfb, ctx->w_dt0, h.dt_cap, depth, tau, all_slow,
                                                        ctx->w_nslow);
        ctx->launches++;
        CU_TRY(ctx, cudaGetLastError());
    } else {
        const int nb = ceil_div(m, PART_T);
        unsigned char* fast = ctx->is_bh;                  // scratch shared with bifrost_pn1 (one call at a time per ctx)
        level_flag_kernel<<<nb, PART_T, 0, st>>>((int)m, seg, ctx->w_dtff, ctx->w_dtfb, ctx->w_dt0, h.dt_cap, depth, tau, all_slow, fast);
        part_count_kernel<<<nb, PART_T, 0, st>>>((int)m, fast, ctx->w_bcount);
        part_scan_kernel<<<1, 32, 0, st>>>(nb, ctx->w_bcount, ctx->w_nslow);
        part_scatter_kernel<<<nb, PART_T, 0, st>>>((int)m, seg, fast, ctx->w_bcount, ctx->w_nslow, ctx->w_tmp);
        ctx->launches += 4;
        CU_TRY(ctx, cudaGetLastError());
        CU_TRY(ctx, cudaMemcpyAsync(seg, ctx->w_tmp, 4 * (size_t)m, cudaMemcpyDeviceToDevice, st));
    }
    hhs_log_kernel<<<1, 1, 0, st>>>(ctx->w_log, ctx->w_log + 3 * HHS_LOG_ROWS, HHS_LOG_ROWS, depth, ctx->w_nslow, (int)m);
    ctx->launches++;
    CU_TRY(ctx, cudaMemcpyAsync(ctx->h_nslow, ctx->w_nslow, 4, cudaMemcpyDeviceToHost, st));
    CU_TRY(ctx, cudaStreamSynchronize(st));                // the host decides the recursion (as in the paper)
    const int64_t ns = *ctx->h_nslow, nf = m - ns;
    const int32_t* S = seg;
    const int32_t* F = seg + ns;
    if (nf == 0) {
        h.fsi_steps++;
        return fsi_impl(ctx, h.n, h.pos, h.vel, h.mass, S, ns, h.G, h.eps_soft, tau, st);
    }
    double* a = ctx->w_acc;
    double* g = ctx->w_grad;
    auto inter_level_acc = [&]() -> int {                  // Eq. 12
        if (ns == 0) return BIFROST_OK;
        return acc_mutual_impl(ctx, h.n, h.pos, h.mass, S, ns, F, nf, h.G, h.eps_soft, a, st);
    };
    auto H_S = [&](bool second) -> int {
        if (ns == 0) return BIFROST_OK;
        h.fsi_steps++;
        return fsi_impl(ctx, h.n, h.pos, h.vel, h.mass, S, ns, h.G, h.eps_soft, tau / 2.0, st, second);
    };
    auto H_F = [&]() -> int { return hhs_level(h, lo + ns, hi, tau / 2.0, depth + 1); };

    RC_TRY(inter_level_acc());
    if (ns) RC_TRY(kick_impl(ctx, seg, m, a, nullptr, tau / 6.0, 0.0, h.vel, st));
    RC_TRY(H_S(false));
    RC_TRY(H_F());
    RC_TRY(inter_level_acc());
    if (ns) {                                              // Eq. 13
        RC_TRY(grad_mutual_impl(ctx, h.n, h.pos, h.mass, a, S, ns, F, nf, h.G, h.eps_soft, g, st));
        RC_TRY(kick_impl(ctx, seg, m, a, g, 2.0 * tau / 3.0, tau * tau / 24.0, h.vel, st));
    }
    RC_TRY(H_F());
    RC_TRY(H_S(true));
    RC_TRY(inter_level_acc());
    if (ns) RC_TRY(kick_impl(ctx, seg, m, a, nullptr, tau / 6.0, 0.0, h.vel, st));
    return BIFROST_OK;
}

}  // namespace

extern "C" {

const char* bifrost_strerror(int code) {
    switch (code) {
        case BIFROST_OK: return "ok";
        case BIFROST_EINVAL: return "invalid argument";
        case BIFROST_ECUDA: return "CUDA error (see bifrost_last_cuda_error)";
        case BIFROST_ENOMEM: return "out of device memory";
        default: return "unknown error";
    }
}

const char* bifrost_last_cuda_error(bifrost_ctx* ctx) { return ctx ? ctx->err : ""; }
int64_t bifrost_launch_count(bifrost_ctx* ctx) { return ctx ? ctx->launches : 0; }

int bifrost_create(bifrost_ctx** out, int device, int64_t max_n) {
    if (!out) return BIFROST_EINVAL;
    *out = nullptr;
    if (max_n <= 0 || max_n >= (int64_t)1 << 31) return BIFROST_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) return BIFROST_ECUDA;
    DeviceGuard guard(device);
    bifrost_ctx* ctx = new (std::nothrow) bifrost_ctx();
    if (!ctx) return BIFROST_ENOMEM;
    ctx->device = device;
    ctx->max_n = max_n;
    cudaDeviceGetAttribute(&ctx->num_sms, cudaDevAttrMultiProcessorCount, device);
    const size_t n_pad = (size_t)((max_n + TILE - 1) / TILE) * TILE;
    ctx->partial_bytes = 24 * (size_t)max_n * 64;   // up to 16 source-range splits at n_sink = max_n
    if (ctx->partial_bytes < ((size_t)64 << 20)) ctx->partial_bytes = (size_t)64 << 20;
    ctx->src_rec_doubles = n_pad * 10;
    if (cudaMalloc(&ctx->src_rec, n_pad * 10 * sizeof(double)) != cudaSuccess ||
        cudaMalloc(&ctx->partial, ctx->partial_bytes) != cudaSuccess ||
        cudaMalloc(&ctx->is_bh, (size_t)max_n) != cudaSuccess ||
        cudaMalloc(&ctx->phi_scratch, 8 * (size_t)max_n) != cudaSuccess ||
        cudaMalloc(&ctx->wpart, 8 * ((size_t)max_n / WSUM_PER_BLOCK + 1)) != cudaSuccess ||
        cudaMalloc(&ctx->smin, 8 * (size_t)max_n) != cudaSuccess ||
        cudaMalloc(&ctx->tickets, TICKETS * sizeof(unsigned)) != cudaSuccess ||
        cudaMemset(ctx->tickets, 0, TICKETS * sizeof(unsigned)) != cudaSuccess) {
        cudaGetLastError();
        bifrost_destroy(ctx);
        return BIFROST_ENOMEM;
    }
    // symmetric kernels: 12 max_n^2 / (sinks per CTA) bytes of source-side rows (sized for the smaller block of the two
    // passes); skipped when that exceeds a quarter of the free device memory (those calls then take the plain path)
    {
        auto rows = [&](int bs) {       // source-side rows of a list of max_n entries cut into blocks of bs
            SymGeom g{};
            g.n_tiles = ceil_div(max_n, TILE); g.bs = bs; g.tb = bs / TILE; g.n_blocks = ceil_div(max_n, bs);
            return sym_joff(g, g.n_blocks - 1) + (size_t)sym_range(g, g.n_blocks - 1) * TILE;
        };
        const size_t need = 24 * std::max(rows(SYM_ACC_BS), rows(SYM_GRAD_BS)) + 4096;
        size_t free_b = 0, total_b = 0;
        if (max_n >= std::min(ctx->sym_min_acc, ctx->sym_min_grad) && cudaMemGetInfo(&free_b, &total_b) == cudaSuccess && need < free_b / 4 &&
            cudaMalloc(&ctx->sym_ws, need) == cudaSuccess)
            ctx->sym_ws_bytes = need;
        else { cudaGetLastError(); ctx->sym_ws = nullptr; }
    }
    *out = ctx;
    return BIFROST_OK;
}

int bifrost_set_tuning(bifrost_ctx* ctx, int knob, int64_t value) {
    if (!ctx || value < 0) return BIFROST_EINVAL;
    ctx->err[0] = 0;
    switch (knob) {
        case BIFROST_TUNE_FUSED_MAX_SINKS:
            if (value > (int64_t)TICKETS * 128) return BIFROST_EINVAL;
            ctx->fused_max_sinks = value; return BIFROST_OK;
        case BIFROST_TUNE_SMALL_M:
            if (value > SMALL_M) return BIFROST_EINVAL;
            ctx->small_m = (int)value; return BIFROST_OK;
        case BIFROST_TUNE_SYM_MIN_N:
            ctx->sym_min_acc = ctx->sym_min_grad = ctx->sym_min_dt = value; return BIFROST_OK;
        case BIFROST_TUNE_MUTUAL_MIN_PAIRS:
            ctx->mutual_min_pairs = (double)value; ctx->mutual_min_b = value == 0 ? 1 : 512; return BIFROST_OK;
        case BIFROST_TUNE_FEW_MAX_SINKS:
            if (value > FEW_MAX_SINKS) return BIFROST_EINVAL;
            ctx->few_max_sinks = value; return BIFROST_OK;
        case BIFROST_TUNE_FUSED_CLUSTER:
            if (value > 1) return BIFROST_EINVAL;
            ctx->fused_cluster = value != 0; return BIFROST_OK;
        case BIFROST_TUNE_FEW_MAX_PAIRS:
            ctx->few_max_pairs[0] = ctx->few_max_pairs[1] = ctx->few_max_pairs[2] = (double)value; return BIFROST_OK;
        default: return BIFROST_EINVAL;
    }
}

int bifrost_set_level_criteria(bifrost_ctx* ctx, double eta, double eta_grad, double eta_jerk) {
    if (!ctx || !(eta >= 0.0) || !(eta_grad >= 0.0) || !(eta_jerk >= 0.0)) return BIFROST_EINVAL;
    ctx->err[0] = 0;
    if ((eta > 0.0 || eta_grad > 0.0 || eta_jerk > 0.0) && !(eta > 0.0 && eta_grad > 0.0 && eta_jerk > 0.0)) return BIFROST_EINVAL;
    ctx->lvl_eta = eta; ctx->lvl_eta_grad = eta_grad; ctx->lvl_eta_jerk = eta_jerk;
    return BIFROST_OK;
}

int bifrost_set_shard(bifrost_ctx* ctx, int rank, int world) {
    if (!ctx || world < 1 || world > 1024 || rank < 0 || rank >= world) return BIFROST_EINVAL;
    ctx->err[0] = 0;
    if (world > 1 && !ctx->sym_ws) return BIFROST_EINVAL;     // needs the symmetric kernels' workspace
    ctx->shard_rank = rank;
    ctx->shard_world = world;
    return BIFROST_OK;
}

int bifrost_reserve(bifrost_ctx* ctx, int what) {
    if (!ctx || (what & ~(BIFROST_RESERVE_HOST | BIFROST_RESERVE_INTEGRATOR))) return BIFROST_EINVAL;
    ctx->err[0] = 0;
    DeviceGuard guard(ctx->device);
    int rc;
    if ((what & BIFROST_RESERVE_HOST) && (rc = ensure_host_mirrors(ctx))) return rc;
    if ((what & BIFROST_RESERVE_INTEGRATOR) && (rc = ensure_integrator(ctx))) return rc;
    return BIFROST_OK;
}

int bifrost_destroy(bifrost_ctx* ctx) {
    if (!ctx) return BIFROST_EINVAL;
    DeviceGuard guard(ctx->device);
    cudaFree(ctx->src_rec); cudaFree(ctx->partial); cudaFree(ctx->is_bh); cudaFree(ctx->phi_scratch); cudaFree(ctx->wpart); cudaFree(ctx->smin); cudaFree(ctx->tickets); cudaFree(ctx->sym_ws);
    cudaFree(ctx->d_pos); cudaFree(ctx->d_vel); cudaFree(ctx->d_mass); cudaFree(ctx->d_acc); cudaFree(ctx->d_out);
    cudaFree(ctx->d_dt); cudaFree(ctx->d_sink); cudaFree(ctx->d_src); cudaFree(ctx->d_j);
    cudaFree(ctx->w_acc); cudaFree(ctx->w_grad); cudaFree(ctx->w_acc_s); cudaFree(ctx->w_jerk); cudaFree(ctx->w_dtff); cudaFree(ctx->w_dtfb); cudaFree(ctx->w_dt0);
    cudaFree(ctx->w_order); cudaFree(ctx->w_tmp); cudaFree(ctx->w_bcount); cudaFree(ctx->w_nslow); cudaFree(ctx->w_log);
    if (ctx->h_nslow) cudaFreeHost(ctx->h_nslow);
    if (ctx->h_log) cudaFreeHost(ctx->h_log);
    if (ctx->h_stage) cudaFreeHost(ctx->h_stage);
    if (ctx->h_stage_i) cudaFreeHost(ctx->h_stage_i);
    if (ctx->hstream) cudaStreamDestroy(ctx->hstream);
    delete ctx;
    return BIFROST_OK;
}

int bifrost_acc(bifrost_ctx* ctx, int64_t n, const double* pos, const double* mass, const int32_t* sink_idx,
                int64_t n_sink, const int32_t* src_idx, int64_t n_src, double G, double eps, double* out_acc,
                void* stream) {
    int rc = check_lists(ctx, n, sink_idx, n_sink, src_idx, n_src);
    if (rc) return rc;
    if (n_sink > 0 && (!pos || !mass || !out_acc)) return BIFROST_EINVAL;
    DeviceGuard guard(ctx->device);
    return acc_impl(ctx, n, pos, mass, sink_idx, n_sink, src_idx, n_src, G, eps, out_acc, 0, (cudaStream_t)stream);
}

int bifrost_grad(bifrost_ctx* ctx, int64_t n, const double* pos, const double* mass, const double* acc,
                 const int32_t* sink_idx, int64_t n_sink, const int32_t* src_idx, int64_t n_src, double G, double eps,
                 double* out_grad, void* stream) {
    int rc = check_lists(ctx, n, sink_idx, n_sink, src_idx, n_src);
    if (rc) return rc;
    if (n_sink > 0 && (!pos || !mass || !acc || !out_grad)) return BIFROST_EINVAL;
    DeviceGuard guard(ctx->device);
    return grad_impl(ctx, n, pos, mass, acc, sink_idx, n_sink, src_idx, n_src, G, eps, out_grad, 0,
                     (cudaStream_t)stream);
}

int bifrost_acc_mutual(bifrost_ctx* ctx, int64_t n, const double* pos, const double* mass, const int32_t* a_idx, int64_t n_a,
                       const int32_t* b_idx, int64_t n_b, double G, double eps, double* out_acc, void* stream) {
    if (!a_idx || !b_idx) return BIFROST_EINVAL;
    int rc = check_lists(ctx, n, a_idx, n_a, b_idx, n_b);
    if (rc) return rc;
    if (n_a + n_b > 0 && (!pos || !mass || !out_acc)) return BIFROST_EINVAL;
    DeviceGuard guard(ctx->device);
    return acc_mutual_impl(ctx, n, pos, mass, a_idx, n_a, b_idx, n_b, G, eps, out_acc, (cudaStream_t)stream);
}

int bifrost_grad_mutual(bifrost_ctx* ctx, int64_t n, const double* pos, const double* mass, const double* acc,
                        const int32_t* a_idx, int64_t n_a, const int32_t* b_idx, int64_t n_b, double G, double eps,
                        double* out_grad, void* stream) {
    if (!a_idx || !b_idx) return BIFROST_EINVAL;
    int rc = check_lists(ctx, n, a_idx, n_a, b_idx, n_b);
    if (rc) return rc;
    if (n_a + n_b > 0 && (!pos || !mass || !acc || !out_grad)) return BIFROST_EINVAL;
    DeviceGuard guard(ctx->device);
    return grad_mutual_impl(ctx, n, pos, mass, acc, a_idx, n_a, b_idx, n_b, G, eps, out_grad, (cudaStream_t)stream);
}

int bifrost_dtmin(bifrost_ctx* ctx, int64_t n, const double* pos, const double* vel, const double* mass,
                  const int32_t* sink_idx, int64_t n_sink, const int32_t* src_idx, int64_t n_src, double G,
                  double eta_ff, double eta_fb, double* out_dt_ff, double* out_dt_fb, int32_t* out_j_ff,
                  int32_t* out_j_fb, void* stream) {
    int rc = check_lists(ctx, n, sink_idx, n_sink, src_idx, n_src);
    if (rc) return rc;
    if (n_sink > 0 && (!pos || !vel || !mass)) return BIFROST_EINVAL;
    DeviceGuard guard(ctx->device);
    return dtmin_impl(ctx, n, pos, vel, mass, sink_idx, n_sink, src_idx, n_src, G, eta_ff, eta_fb, out_dt_ff,
                      out_dt_fb, out_j_ff, out_j_fb, 0, (cudaStream_t)stream);
}

int bifrost_pn1(bifrost_ctx* ctx, int64_t n, const double* pos, const double* vel, const double* mass,
                const int32_t* bh_idx, int64_t n_bh, double G, double c, double* out_acc_pn, void* stream) {
    if (!ctx) return BIFROST_EINVAL;
    ctx->err[0] = 0;
    if (n < 0 || n > ctx->max_n || n_bh < 0 || n_bh > n) return BIFROST_EINVAL;
    if (n > 0 && (!pos || !vel || !mass || !out_acc_pn)) return BIFROST_EINVAL;
    if (n_bh > 0 && !bh_idx) return BIFROST_EINVAL;
    if (ctx->subsys && ctx->subsys_n != n) return BIFROST_EINVAL;
    DeviceGuard guard(ctx->device);
    return pn1_impl(ctx, n, pos, vel, mass, bh_idx, n_bh, G, c, out_acc_pn, (cudaStream_t)stream);
}

// ---- NEXT-1 / NEXT-4 rows ---------------------------------------------------

int bifrost_jerk(bifrost_ctx* ctx, int64_t n, const double* pos, const double* vel, const double* mass,
                 const int32_t* sink_idx, int64_t n_sink, const int32_t* src_idx, int64_t n_src, double G, double eps,
                 double* out_jerk, void* stream) {
    int rc = check_lists(ctx, n, sink_idx, n_sink, src_idx, n_src);
    if (rc) return rc;
    if (n_sink > 0 && (!pos || !vel || !mass || !out_jerk)) return BIFROST_EINVAL;
    DeviceGuard guard(ctx->device);
    // Eq. 28 is Eq. 9's tensor contraction with v_ji in place of a_ji: the same kernel.
    return grad_impl(ctx, n, pos, mass, vel, sink_idx, n_sink, src_idx, n_src, G, eps, out_jerk, 0, (cudaStream_t)stream);
}

int bifrost_acc_jerk(bifrost_ctx* ctx, int64_t n, const double* pos, const double* vel, const double* mass,
                     const int32_t* sink_idx, int64_t n_sink, const int32_t* src_idx, int64_t n_src, double G, double eps,
                     double* out_acc, double* out_jerk, void* stream) {
    int rc = check_lists(ctx, n, sink_idx, n_sink, src_idx, n_src);
    if (rc) return rc;
    if (n_sink > 0 && (!pos || !vel || !mass || !out_acc || !out_jerk)) return BIFROST_EINVAL;
    DeviceGuard guard(ctx->device);
    return acc_jerk_impl(ctx, n, pos, vel, mass, sink_idx, n_sink, src_idx, n_src, G, eps, out_acc, out_jerk,
                         (cudaStream_t)stream);
}

int bifrost_potential(bifrost_ctx* ctx, int64_t n, const double* pos, const double* mass, const int32_t* sink_idx,
                      int64_t n_sink, const int32_t* src_idx, int64_t n_src, double G, double eps, double* out_phi,
                      double* out_W, void* stream) {
    int rc = check_lists(ctx, n, sink_idx, n_sink, src_idx, n_src);
    if (rc) return rc;
    if (n_sink > 0 && (!pos || !mass)) return BIFROST_EINVAL;
    if (!out_phi && !out_W) return BIFROST_EINVAL;
    DeviceGuard guard(ctx->device);
    return pot_impl(ctx, n, pos, mass, sink_idx, n_sink, src_idx, n_src, G, eps, out_phi, out_W, (cudaStream_t)stream);
}

int bifrost_timestep_criteria(bifrost_ctx* ctx, int64_t n, const double* vel, const double* acc, const double* grad,
                              const double* jerk, const int32_t* sink_idx, int64_t n_sink, double eta, double eta_grad,
                              double eta_jerk, double* out_dt_va, double* out_dt_gradv, double* out_dt_grada,
                              double* out_dt_jerk, double* inout_dt, void* stream) {
    if (!ctx) return BIFROST_EINVAL;
    ctx->err[0] = 0;
    if (n < 0 || n > ctx->max_n || n_sink < 0 || n_sink > ctx->max_n) return BIFROST_EINVAL;
    if (!sink_idx && n_sink != n) return BIFROST_EINVAL;
    if (n_sink == 0) return BIFROST_OK;
    if (!vel || !acc) return BIFROST_EINVAL;
    if ((!grad && (out_dt_gradv || out_dt_grada)) || (!jerk && out_dt_jerk)) return BIFROST_EINVAL;
    DeviceGuard guard(ctx->device);
    criteria_kernel<<<ceil_div(n_sink, 256), 256, 0, (cudaStream_t)stream>>>(
        (int)n_sink, sink_idx, vel, acc, grad, jerk, eta, eta_grad, eta_jerk, out_dt_va, out_dt_gradv, out_dt_grada,
        out_dt_jerk, inout_dt);
    ctx->launches++;
    CU_TRY(ctx, cudaGetLastError());
    return BIFROST_OK;
}

// ---- host-buffer variants --------------------------------------------------------------

#define H2D(dst, src, bytes) CU_TRY(ctx, cudaMemcpyAsync(dst, src, bytes, cudaMemcpyHostToDevice, ctx->hstream))

int bifrost_acc_host(bifrost_ctx* ctx, int64_t n, const double* pos, const double* mass, const int32_t* sink_idx,
                     int64_t n_sink, const int32_t* src_idx, int64_t n_src, double G, double eps, double* out_acc) {
    int rc = check_lists(ctx, n, sink_idx, n_sink, src_idx, n_src);
    if (rc) return rc;
    if (n_sink == 0) return BIFROST_OK;
    if (!pos || !mass || !out_acc) return BIFROST_EINVAL;
    DeviceGuard guard(ctx->device);
    if ((rc = ensure_host_mirrors(ctx))) return rc;
    H2D(ctx->d_pos, pos, 24 * (size_t)n);
    H2D(ctx->d_mass, mass, 8 * (size_t)n);
    // one list on both sides (same host pointer): one device copy, so that the call takes the symmetric kernels
    const bool same = sink_idx && src_idx == sink_idx && n_src == n_sink;
    if (sink_idx) H2D(ctx->d_sink, sink_idx, 4 * (size_t)n_sink);
    if (src_idx && !same) H2D(ctx->d_src, src_idx, 4 * (size_t)n_src);
    rc = acc_impl(ctx, n, ctx->d_pos, ctx->d_mass, sink_idx ? ctx->d_sink : nullptr, n_sink,
                  src_idx ? (same ? ctx->d_sink : ctx->d_src) : nullptr, n_src, G, eps, ctx->d_out, 1, ctx->hstream);
    if (rc) return rc;
    return fetch_rows(ctx, ctx->d_out, 24, sink_idx, n_sink, out_acc, ctx->h_stage);
}

int bifrost_grad_host(bifrost_ctx* ctx, int64_t n, const double* pos, const double* mass, const double* acc,
                      const int32_t* sink_idx, int64_t n_sink, const int32_t* src_idx, int64_t n_src, double G,
                      double eps, double* out_grad) {
    int rc = check_lists(ctx, n, sink_idx, n_sink, src_idx, n_src);
    if (rc) return rc;
    if (n_sink == 0) return BIFROST_OK;
    if (!pos || !mass || !acc || !out_grad) return BIFROST_EINVAL;
    DeviceGuard guard(ctx->device);
    if ((rc = ensure_host_mirrors(ctx))) return rc;
    H2D(ctx->d_pos, pos, 24 * (size_t)n);
    H2D(ctx->d_mass, mass, 8 * (size_t)n);
    H2D(ctx->d_acc, acc, 24 * (size_t)n);
    const bool same = sink_idx && src_idx == sink_idx && n_src == n_sink;
    if (sink_idx) H2D(ctx->d_sink, sink_idx, 4 * (size_t)n_sink);
    if (src_idx && !same) H2D(ctx->d_src, src_idx, 4 * (size_t)n_src);
    rc = grad_impl(ctx, n, ctx->d_pos, ctx->d_mass, ctx->d_acc, sink_idx ? ctx->d_sink : nullptr, n_sink,
                   src_idx ? (same ? ctx->d_sink : ctx->d_src) : nullptr, n_src, G, eps, ctx->d_out, 1, ctx->hstream);
    if (rc) return rc;
    return fetch_rows(ctx, ctx->d_out, 24, sink_idx, n_sink, out_grad, ctx->h_stage);
}

int bifrost_dtmin_host(bifrost_ctx* ctx, int64_t n, const double* pos, const double* vel, const double* mass,
                       const int32_t* sink_idx, int64_t n_sink, const int32_t* src_idx, int64_t n_src, double G,
                       double eta_ff, double eta_fb, double* out_dt_ff, double* out_dt_fb, int32_t* out_j_ff,
                       int32_t* out_j_fb) {
    int rc = check_lists(ctx, n, sink_idx, n_sink, src_idx, n_src);
    if (rc) return rc;
    if (n_sink == 0) return BIFROST_OK;
    if (!pos || !vel || !mass) return BIFROST_EINVAL;
    DeviceGuard guard(ctx->device);
    if ((rc = ensure_host_mirrors(ctx))) return rc;
    H2D(ctx->d_pos, pos, 24 * (size_t)n);
    H2D(ctx->d_vel, vel, 24 * (size_t)n);
    H2D(ctx->d_mass, mass, 8 * (size_t)n);
    const bool same = sink_idx && src_idx == sink_idx && n_src == n_sink;      // one list on both sides: one device copy
    if (sink_idx) H2D(ctx->d_sink, sink_idx, 4 * (size_t)n_sink);
    if (src_idx && !same) H2D(ctx->d_src, src_idx, 4 * (size_t)n_src);
    double* d_ff = ctx->d_dt;
    double* d_fb = ctx->d_dt + n_sink;
    int32_t* d_jff = ctx->d_j;
    int32_t* d_jfb = ctx->d_j + n_sink;
    rc = dtmin_impl(ctx, n, ctx->d_pos, ctx->d_vel, ctx->d_mass, sink_idx ? ctx->d_sink : nullptr, n_sink,
                    src_idx ? (same ? ctx->d_sink : ctx->d_src) : nullptr, n_src, G, eta_ff, eta_fb, d_ff, d_fb, d_jff, d_jfb, 1, ctx->hstream);
    if (rc) return rc;
    if ((rc = fetch_rows(ctx, d_ff, 8, sink_idx, n_sink, out_dt_ff, ctx->h_stage))) return rc;
    if ((rc = fetch_rows(ctx, d_fb, 8, sink_idx, n_sink, out_dt_fb, ctx->h_stage))) return rc;
    if ((rc = fetch_rows(ctx, d_jff, 4, sink_idx, n_sink, out_j_ff, ctx->h_stage_i))) return rc;
    if ((rc = fetch_rows(ctx, d_jfb, 4, sink_idx, n_sink, out_j_fb, ctx->h_stage_i))) return rc;
    CU_TRY(ctx, cudaStreamSynchronize(ctx->hstream));
    return BIFROST_OK;
}

int bifrost_pn1_host(bifrost_ctx* ctx, int64_t n, const double* pos, const double* vel, const double* mass,
                     const int32_t* bh_idx, int64_t n_bh, double G, double c, double* out_acc_pn) {
    if (!ctx) return BIFROST_EINVAL;
    ctx->err[0] = 0;
    if (n < 0 || n > ctx->max_n || n_bh < 0 || n_bh > n) return BIFROST_EINVAL;
    if (n == 0) return BIFROST_OK;
    if (!pos || !vel || !mass || !out_acc_pn || (n_bh > 0 && !bh_idx)) return BIFROST_EINVAL;
    if (ctx->subsys && ctx->subsys_n != n) return BIFROST_EINVAL;
    DeviceGuard guard(ctx->device);
    int rc;
    if ((rc = ensure_host_mirrors(ctx))) return rc;
    H2D(ctx->d_pos, pos, 24 * (size_t)n);
    H2D(ctx->d_vel, vel, 24 * (size_t)n);
    H2D(ctx->d_mass, mass, 8 * (size_t)n);
    if (n_bh) H2D(ctx->d_sink, bh_idx, 4 * (size_t)n_bh);
    rc = pn1_impl(ctx, n, ctx->d_pos, ctx->d_vel, ctx->d_mass, ctx->d_sink, n_bh, G, c, ctx->d_out, ctx->hstream);
    if (rc) return rc;
    return fetch_rows(ctx, ctx->d_out, 24, nullptr, n, out_acc_pn, ctx->h_stage);
}

// ---- NEXT-2: subsystem-aware sums ------------------------------------------

int bifrost_set_subsystems(bifrost_ctx* ctx, const int32_t* subsys, int64_t n) {
    if (!ctx) return BIFROST_EINVAL;
    ctx->err[0] = 0;
    if (subsys && (n <= 0 || n > ctx->max_n)) return BIFROST_EINVAL;
    ctx->subsys = subsys;
    ctx->subsys_n = subsys ? n : 0;
    return BIFROST_OK;
}

int bifrost_subsys_min(bifrost_ctx* ctx, int64_t n, const int32_t* subsys, double* inout_dt, void* stream) {
    if (!ctx) return BIFROST_EINVAL;
    ctx->err[0] = 0;
    if (n < 0 || n > ctx->max_n) return BIFROST_EINVAL;
    if (n == 0) return BIFROST_OK;
    if (!subsys || !inout_dt) return BIFROST_EINVAL;
    DeviceGuard guard(ctx->device);
    cudaStream_t st = (cudaStream_t)stream;
    const int nb = ceil_div(n, 256);
    smin_fill_kernel<<<nb, 256, 0, st>>>((int)n, ctx->smin);
    smin_reduce_kernel<<<nb, 256, 0, st>>>((int)n, subsys, inout_dt, ctx->smin);
    smin_apply_kernel<<<nb, 256, 0, st>>>((int)n, subsys, ctx->smin, inout_dt);
    ctx->launches += 3;
    CU_TRY(ctx, cudaGetLastError());
    return BIFROST_OK;
}

// ---- NEXT-3: neighbour search and subsystem construction --------------------

int bifrost_neighbours(bifrost_ctx* ctx, int64_t n, const double* pos, const double* vel, const double* mass,
                       const int32_t* sink_idx, int64_t n_sink, const int32_t* src_idx, int64_t n_src, double G,
                       double r_ngb, double r_ngb_max, double tau, double C, int64_t cap, int32_t* out_count,
                       int32_t* out_list, void* stream) {
    int rc = check_lists(ctx, n, sink_idx, n_sink, src_idx, n_src);
    if (rc) return rc;
    if (cap <= 0 || cap > 1024) return BIFROST_EINVAL;
    if (n_sink == 0) return BIFROST_OK;
    if (!pos || !vel || !mass || !out_count || !out_list) return BIFROST_EINVAL;
    DeviceGuard guard(ctx->device);
    cudaStream_t st = (cudaStream_t)stream;
    if (n_src > 0) {
        const int n_pad = ceil_div(n_src, TILE) * TILE;
        const SrcArrays src{pos, vel, mass, nullptr, src_idx};
        pack_kernel<DtPass><<<ceil_div(n_pad, 256), 256, 0, st>>>((int)n_src, n_pad, src, ctx->src_rec);
        ctx->launches++;
        CU_TRY(ctx, cudaGetLastError());
    }
    const size_t per_sink = 4 * ((size_t)cap + 1);
    Geom g;
    const double guard2 = (r_ngb_max * r_ngb_max) * (1.0 + 1e-10);
    auto launch = [&](auto shape) -> int {
        constexpr int S = decltype(shape)::S, T = decltype(shape)::T, MINB = decltype(shape)::MINB;
        g = make_geom(ctx, n_sink, n_src, T * S, MINB, per_sink);
        // the workspace may not hold one list per sink at all for a huge cap: fall back to one split
        if (per_sink * (size_t)n_sink > ctx->partial_bytes) { g.n_split = 1; g.tiles_per_split = ceil_div(n_src, TILE) > 0 ? ceil_div(n_src, TILE) : 1; }
        int32_t* pcount = (int32_t*)ctx->partial;
        int32_t* plist = pcount + (size_t)g.n_split * (size_t)n_sink;
        const NgbArgs a{pos, vel, mass, sink_idx, G, r_ngb, r_ngb_max, tau, C, guard2, (int)cap, (int)n_sink, out_count, out_list, pcount, plist};
        dim3 grid(ceil_div(n_sink, T * S), g.n_split);
        ngb_kernel<S, T, MINB><<<grid, T, 0, st>>>(a, g, ctx->src_rec);
        ctx->launches++;
        CU_TRY(ctx, cudaGetLastError());
        if (g.n_split > 1) {
            ngb_finish_kernel<<<ceil_div(n_sink, 256), 256, 0, st>>>(a, g);
            ctx->launches++;
            CU_TRY(ctx, cudaGetLastError());
        }
        return BIFROST_OK;
    };
    // 6 sinks per thread is 6 % faster per pair (453.7 vs 482.3 ms at N = 2^20); the smaller CTA quantises better below
    return n_sink >= 32768 ? launch(Shape<6, 128, 3, 1>{}) : launch(Shape<4, 128, 4, 1>{});
}

int bifrost_dtmin_neighbours(bifrost_ctx* ctx, int64_t n, const double* pos, const double* vel, const double* mass,
                             const int32_t* sink_idx, int64_t n_sink, const int32_t* src_idx, int64_t n_src, double G,
                             double eta_ff, double eta_fb, double r_ngb, double r_ngb_max, double tau, double C, int64_t cap,
                             double* out_dt_ff, double* out_dt_fb, int32_t* out_j_ff, int32_t* out_j_fb,
                             int32_t* out_count, int32_t* out_list, void* stream) {
    int rc = check_lists(ctx, n, sink_idx, n_sink, src_idx, n_src);
    if (rc) return rc;
    if (cap <= 0 || cap > 1024) return BIFROST_EINVAL;
    if (n_sink == 0) return BIFROST_OK;
    if (!pos || !vel || !mass || !out_count || !out_list) return BIFROST_EINVAL;
    // one list per sink must fit the workspace (else: separate calls, whose neighbour pass falls back to one split)
    if ((24 + 4 * ((size_t)cap + 1)) * (size_t)n_sink > ctx->partial_bytes) return BIFROST_EINVAL;
    DeviceGuard guard(ctx->device);
    const double guard2 = (r_ngb_max * r_ngb_max) * (1.0 + 1e-10);
    const NgbArgs ng{pos, vel, mass, sink_idx, G, r_ngb, r_ngb_max, tau, C, guard2, (int)cap, (int)n_sink, out_count, out_list,
                     nullptr, nullptr};
    return dtmin_impl(ctx, n, pos, vel, mass, sink_idx, n_sink, src_idx, n_src, G, eta_ff, eta_fb, out_dt_ff, out_dt_fb,
                      out_j_ff, out_j_fb, 0, (cudaStream_t)stream, &ng);
}

int bifrost_components(bifrost_ctx* ctx, int64_t n, const int32_t* count, const int32_t* list, int64_t cap,
                       int32_t* out_subsys, void* stream) {
    if (!ctx) return BIFROST_EINVAL;
    ctx->err[0] = 0;
    if (n < 0 || n > ctx->max_n || cap <= 0 || cap > 1024) return BIFROST_EINVAL;
    if (n == 0) return BIFROST_OK;
    if (!count || !list || !out_subsys) return BIFROST_EINVAL;
    DeviceGuard guard(ctx->device);
    cudaStream_t st = (cudaStream_t)stream;
    int* parent = (int*)ctx->smin;              // scratch shared with bifrost_subsys_min (calls are serialised per ctx)
    unsigned char* flag = ctx->is_bh;           // scratch shared with bifrost_pn1
    comp_init_kernel<<<ceil_div(n, 256), 256, 0, st>>>((int)n, parent, flag);
    comp_hook_kernel<<<ceil_div(n * cap, 256), 256, 0, st>>>((int)n, (int)cap, count, list, parent, flag);
    comp_label_kernel<<<ceil_div(n, 256), 256, 0, st>>>((int)n, parent, flag, out_subsys);
    ctx->launches += 3;
    CU_TRY(ctx, cudaGetLastError());
    return BIFROST_OK;
}

// ---- NEXT-4: integrator operators, FSI cycle, HHS-FSI driver -----------------

int bifrost_kick(bifrost_ctx* ctx, int64_t n, const int32_t* idx, int64_t n_idx, const double* acc, const double* grad,
                 double h, double c, double* vel, void* stream) {
    if (!ctx) return BIFROST_EINVAL;
    ctx->err[0] = 0;
    if (n < 0 || n > ctx->max_n || n_idx < 0 || n_idx > ctx->max_n || (!idx && n_idx != n)) return BIFROST_EINVAL;
    if (n_idx == 0) return BIFROST_OK;
    if (!acc || !vel) return BIFROST_EINVAL;
    DeviceGuard guard(ctx->device);
    return kick_impl(ctx, idx, n_idx, acc, grad, h, c, vel, (cudaStream_t)stream);
}

int bifrost_drift(bifrost_ctx* ctx, int64_t n, const int32_t* idx, int64_t n_idx, const double* vel, double h,
                  double* pos, void* stream) {
    if (!ctx) return BIFROST_EINVAL;
    ctx->err[0] = 0;
    if (n < 0 || n > ctx->max_n || n_idx < 0 || n_idx > ctx->max_n || (!idx && n_idx != n)) return BIFROST_EINVAL;
    if (n_idx == 0) return BIFROST_OK;
    if (!vel || !pos) return BIFROST_EINVAL;
    DeviceGuard guard(ctx->device);
    return drift_impl(ctx, idx, n_idx, vel, h, pos, (cudaStream_t)stream);
}

int bifrost_fsi_step(bifrost_ctx* ctx, int64_t n, double* pos, double* vel, const double* mass, const int32_t* idx,
                     int64_t n_idx, double G, double eps_soft, double eps, void* stream) {
    int rc = check_lists(ctx, n, idx, n_idx, idx, n_idx);
    if (rc) return rc;
    if (ctx->subsys) return BIFROST_EINVAL;    // no subsystem integrator here (reading H5): members would move without their mutual force
    if (n_idx == 0) return BIFROST_OK;
    if (!pos || !vel || !mass) return BIFROST_EINVAL;
    DeviceGuard guard(ctx->device);
    if ((rc = ensure_integrator(ctx))) return rc;
    return fsi_impl(ctx, n, pos, vel, mass, idx, n_idx, G, eps_soft, eps, (cudaStream_t)stream);
}

int bifrost_hhs_fsi(bifrost_ctx* ctx, int64_t n, double* pos, double* vel, const double* mass, double G, double eps_soft,
                    double eta_ff, double eta_fb, const double* dt_cap, double tau, int max_depth, int64_t* out_level_log,
                    int64_t log_cap, int64_t* out_summary, void* stream) {
    if (!ctx) return BIFROST_EINVAL;
    ctx->err[0] = 0;
    if (n < 0 || n > ctx->max_n || max_depth < 0 || max_depth > 62 || log_cap < 0 || !(tau > 0.0)) return BIFROST_EINVAL;
    if (ctx->subsys) return BIFROST_EINVAL;    // as bifrost_fsi_step (reading H5)
    if (out_summary) out_summary[0] = out_summary[1] = out_summary[2] = 0;
    if (n == 0) return BIFROST_OK;
    if (!pos || !vel || !mass) return BIFROST_EINVAL;
    DeviceGuard guard(ctx->device);
    int rc;
    if ((rc = ensure_integrator(ctx))) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    iota_kernel<<<ceil_div(n, 256), 256, 0, st>>>((int)n, ctx->w_order);
    fill_f64_kernel<<<ceil_div(n, 256), 256, 0, st>>>((int)n, HUGE_VAL, ctx->w_dt0);
    ctx->launches += 2;
    CU_TRY(ctx, cudaGetLastError());
    long long* counters = ctx->w_log + 3 * HHS_LOG_ROWS;      // levels entered, deepest depth, FSI cycles of the subtree launches
    CU_TRY(ctx, cudaMemsetAsync(counters, 0, 3 * sizeof(long long), st));
    Hhs h{ctx, n, pos, vel, mass, G, eps_soft, eta_ff, eta_fb, dt_cap, max_depth, st, out_level_log, log_cap, 0, 0, 0};
    rc = hhs_level(h, 0, n, tau, 0);
    if (rc) return rc;
    // the level log and the counters live on the device (host-steered levels and subtree launches append in stream order)
    const long long want = std::min<long long>(log_cap, HHS_LOG_ROWS);
    CU_TRY(ctx, cudaMemcpyAsync(ctx->h_log + 3 * HHS_LOG_ROWS, counters, 3 * sizeof(long long), cudaMemcpyDeviceToHost, st));
    if (out_level_log && want > 0)
        CU_TRY(ctx, cudaMemcpyAsync(ctx->h_log, ctx->w_log, 3 * want * sizeof(long long), cudaMemcpyDeviceToHost, st));
    CU_TRY(ctx, cudaStreamSynchronize(st));
    const long long* hc = ctx->h_log + 3 * HHS_LOG_ROWS;
    if (out_level_log)
        for (long long r = 0; r < std::min(want, hc[0]); ++r)
            for (int q = 0; q < 3; ++q) out_level_log[3 * r + q] = ctx->h_log[3 * r + q];
    if (out_summary) { out_summary[0] = hc[0]; out_summary[1] = hc[1]; out_summary[2] = h.fsi_steps + hc[2]; }
    return BIFROST_OK;
}

int bifrost_kinetic_energy(bifrost_ctx* ctx, int64_t n, const double* vel, const double* mass, const int32_t* idx,
                           int64_t n_idx, double* out_T, void* stream) {
    if (!ctx) return BIFROST_EINVAL;
    ctx->err[0] = 0;
    if (n < 0 || n > ctx->max_n || n_idx < 0 || n_idx > ctx->max_n || (!idx && n_idx != n) || !out_T) return BIFROST_EINVAL;
    DeviceGuard guard(ctx->device);
    cudaStream_t st = (cudaStream_t)stream;
    if (n_idx == 0) { CU_TRY(ctx, cudaMemsetAsync(out_T, 0, sizeof(double), st)); return BIFROST_OK; }
    if (!vel || !mass) return BIFROST_EINVAL;
    const int nb = ceil_div(n_idx, WSUM_PER_BLOCK);
    ksum_stage1_kernel<<<nb, WSUM_THREADS, 0, st>>>((int)n_idx, idx, mass, vel, ctx->wpart);
    wsum_stage2_kernel<<<1, WSUM_THREADS, 0, st>>>(nb, ctx->wpart, out_T);
    ctx->launches += 2;
    CU_TRY(ctx, cudaGetLastError());
    return BIFROST_OK;
}

// ---- measurement aid -------------------------------------------------------------------

int bifrost_fp64_probe(bifrost_ctx* ctx, int mix, int64_t iters, int ctas_per_sm, double* out_ms,
                       double* out_lane_instr) {
    if (!ctx || !out_ms || !out_lane_instr || iters <= 0 || iters > (1 << 30) || ctas_per_sm <= 0 || ctas_per_sm > 64 ||
        mix < 0 || mix > 3)
        return BIFROST_EINVAL;
    ctx->err[0] = 0;
    DeviceGuard guard(ctx->device);
    struct Events {                            // destroyed on every return path
        cudaEvent_t a = nullptr, b = nullptr;
        ~Events() { if (a) cudaEventDestroy(a); if (b) cudaEventDestroy(b); }
    } ev;
    CU_TRY(ctx, cudaEventCreate(&ev.a));
    CU_TRY(ctx, cudaEventCreate(&ev.b));
    cudaEvent_t e0 = ev.a, e1 = ev.b;
    const int grid = ctx->num_sms * ctas_per_sm;
    const double b = 0.999999999, c = 1e-9;
    double* sink = (double*)ctx->partial;      // never written (see kernel); >= 64 MiB
    double* in = ctx->src_rec;                 // operands of mix 2/3: 28 x 128 doubles, set to 1 + O(1e-6)
    {
        static double h[28 * 128];
        for (int i = 0; i < 28 * 128; ++i) h[i] = 1.0 + 1e-6 * i;
        CU_TRY(ctx, cudaMemcpy(in, h, sizeof(h), cudaMemcpyHostToDevice));
    }
    for (int rep = 0; rep < 2; ++rep) {        // first launch = warm-up
        cudaEventRecord(e0, 0);
        if (mix == 0) fp64_probe_kernel<0><<<grid, PROBE_THREADS>>>((int)iters, b, c, in, sink);
        else if (mix == 1) fp64_probe_kernel<1><<<grid, PROBE_THREADS>>>((int)iters, b, c, in, sink);
        else if (mix == 2) fp64_probe_kernel<2><<<grid, PROBE_THREADS>>>((int)iters, b, c, in, sink);
        else fp64_probe_kernel<3><<<grid, PROBE_THREADS>>>((int)iters, b, c, in, sink);
        cudaEventRecord(e1, 0);
        ctx->launches++;
        CU_TRY(ctx, cudaEventSynchronize(e1));
    }
    float ms = 0.f;
    CU_TRY(ctx, cudaEventElapsedTime(&ms, e0, e1));
    *out_ms = ms;
    const double per_thread = (double)iters * (mix == 0 ? 32.0 : mix == 1 ? 120.0 : 12.0);
    *out_lane_instr = per_thread * (double)grid * PROBE_THREADS;
    return BIFROST_OK;
}

}  // extern "C"

// ========================================================================================
// bifrost_acc_static: Eq. 6 without any allocation (include/bifrost.h) - for callers under CUDA graph capture, in
// tight serving loops, or in harnesses that forbid cudaMalloc.  The scratch of the acc pass (packed source records,
// split-j partials, the fused kernel's arrival counters) lives in ONE file-scope device array; every GPU that loads the
// library holds its BIFROST_STATIC_SCRATCH_BYTES until the process exits.  The kernels and launch rules are run_pass's,
// driven through a bifrost_ctx on the HOST STACK whose scratch pointers point into that array.
// ========================================================================================

#include <mutex>

static __device__ __align__(256) unsigned char bifrost_static_scratch[BIFROST_STATIC_SCRATCH_BYTES];

namespace {

// carve-up of the array: [records | arrival counters | partials]
constexpr size_t STATIC_REC_DOUBLES = (size_t)((BIFROST_STATIC_MAX_N + TILE - 1) / TILE * TILE) * AccPassT<false>::REC;
constexpr size_t STATIC_OFF_TICKETS = STATIC_REC_DOUBLES * sizeof(double);                  // 768 KiB of records
constexpr size_t STATIC_OFF_PARTIAL = STATIC_OFF_TICKETS + TICKETS * sizeof(unsigned);      // + 4 KiB of counters
constexpr size_t STATIC_PARTIAL_BYTES = (size_t)BIFROST_STATIC_SCRATCH_BYTES - STATIC_OFF_PARTIAL;
static_assert(STATIC_OFF_TICKETS % 256 == 0 && STATIC_OFF_PARTIAL % 256 == 0, "regions keep the array's alignment");
static_assert(STATIC_PARTIAL_BYTES >= 16 * 24 * (size_t)BIFROST_STATIC_MAX_N, "room for 16 source-range splits at the largest n");

constexpr int STATIC_MAX_DEVICES = 64;
struct StaticDevice {
    bool ready = false;
    unsigned char* base = nullptr;   // DEVICE address of bifrost_static_scratch on this device (cudaGetSymbolAddress)
    int num_sms = 0;
};
StaticDevice g_static_dev[STATIC_MAX_DEVICES];
std::mutex g_static_mutex;
thread_local char g_static_err[256] = {0};

// Once per device, with that device current.  In host code the name `bifrost_static_scratch` is only a handle of the
// symbol, NOT a device address (a kernel given it would fault, or read host memory where the GPU can reach it):
// the address each device holds the array at comes from cudaGetSymbolAddress.
int static_setup(int device, StaticDevice* out) {
    std::lock_guard<std::mutex> lock(g_static_mutex);
    StaticDevice& d = g_static_dev[device];
    if (!d.ready) {
        void* p = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&p, bifrost_static_scratch);
        if (e != cudaSuccess || !p) {
            snprintf(g_static_err, sizeof(g_static_err), "cudaGetSymbolAddress(bifrost_static_scratch) on device %d: %s", device,
                     cudaGetErrorString(e));
            return BIFROST_ECUDA;
        }
        int sms = 0;
        e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
        if (e != cudaSuccess || sms <= 0) {
            snprintf(g_static_err, sizeof(g_static_err), "cudaDeviceGetAttribute(multiProcessorCount) on device %d: %s", device,
                     cudaGetErrorString(e));
            return BIFROST_ECUDA;
        }
        d.base = (unsigned char*)p;
        d.num_sms = sms;
        d.ready = true;
    }
    *out = d;
    return BIFROST_OK;
}

}  // namespace

extern "C" {

const char* bifrost_static_error(void) { return g_static_err; }

int bifrost_acc_static(int device, int64_t n, const double* pos, const double* mass, double G, double eps, double* out_acc,
                       void* stream) {
    g_static_err[0] = 0;
    if (n < 0 || n > BIFROST_STATIC_MAX_N) {
        snprintf(g_static_err, sizeof(g_static_err),
                 "bifrost_acc_static: n = %lld is outside 0..BIFROST_STATIC_MAX_N = %d (the static scratch array of %u bytes is "
                 "sized for that many particles); use bifrost_acc with a context for larger sets",
                 (long long)n, BIFROST_STATIC_MAX_N, (unsigned)BIFROST_STATIC_SCRATCH_BYTES);
        return BIFROST_EINVAL;
    }
    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess) n_dev = 0;
    if (device < 0 || device >= STATIC_MAX_DEVICES || device >= n_dev) {
        snprintf(g_static_err, sizeof(g_static_err), "bifrost_acc_static: device %d is not one of the %d CUDA devices (at most %d)",
                 device, n_dev, STATIC_MAX_DEVICES);
        return BIFROST_EINVAL;
    }
    if (n == 0) return BIFROST_OK;
    if (!pos || !mass || !out_acc) {
        snprintf(g_static_err, sizeof(g_static_err), "bifrost_acc_static: pos, mass and out_acc must not be NULL");
        return BIFROST_EINVAL;
    }
    DeviceGuard guard(device);
    StaticDevice d;
    RC_TRY(static_setup(device, &d));
    // A context on the host stack: launch geometry and pointers into the static array; nothing is allocated or freed.
    bifrost_ctx c;
    c.device = device;
    c.max_n = BIFROST_STATIC_MAX_N;
    c.num_sms = d.num_sms;
    c.src_rec = (double*)d.base;
    c.src_rec_doubles = STATIC_REC_DOUBLES;
    c.tickets = (unsigned*)(d.base + STATIC_OFF_TICKETS);
    c.tickets_dirty = true;          // the array keeps the last call's contents (and an aborted launch may have left counts):
                                     // the counters, the one part that must start at zero, are cleared by every fused call
    c.partial = d.base + STATIC_OFF_PARTIAL;
    c.partial_bytes = STATIC_PARTIAL_BYTES;
    const SrcArrays src{pos, nullptr, mass, nullptr, nullptr};
    const AccArgs a{pos, nullptr, nullptr, soft2(eps), G, out_acc, (double*)c.partial};
    using Big = Shape<8, 256, 1, 1>;      // acc_impl's shapes
    using F4 = Shape<4, 128, 4, 2>;
    using F2 = Shape<2, 128, 6, 2>;
    using F1 = Shape<1, 128, 8, 4>;
    const int rc = run_pass<AccPassT<false>, Big, 0, Big, F4, F2, F1>(&c, a, src, n, n, 24, 0, (cudaStream_t)stream);
    if (rc) snprintf(g_static_err, sizeof(g_static_err), "bifrost_acc_static: %s", c.err[0] ? c.err : bifrost_strerror(rc));
    return rc;
}

}  // extern "C"
