// few_sinks.cuh - acc (Eq. 6/12), grad (Eq. 9/13) and dtmin (Eq. 21/22) for a HANDFUL of sinks (at most 32 per cluster; up to 128
// in all) against a source list: the fastest levels of the hierarchy, where a call is latency, not arithmetic.
// Part of the single translation unit bifrost.cu (see its header and DESIGN.md); not a public header.
//
// pair_fused_kernel gives every thread one sink and walks the sources of its CTA one after the other: with one sink, one
// thread per CTA works through 128 dependent iterations, then 128 CTAs meet at a global ticket and the last one reads 128
// partials back through L2 (12 us for 1 sink x 16384 sources, of which < 1 us is arithmetic).  Here the THREADS GO OVER THE
// SOURCES: the launch is ONE thread-block cluster of CL <= 16 CTAs of 256 threads (33-128 sinks against a short source list:
// one such cluster per 32 sinks); thread t of a CTA serves sink t mod NSP (NSP = the sink count rounded up to a power of
// two) and every (256 / NSP)-th source of the CTA's tiles, so one sink x 16384 sources is 4 pairs per thread.  The per-thread
// results are merged in a FIXED order - xor-shuffles over the lanes that share a sink, the 8 warps of the CTA through shared
// memory in warp order, the CL CTAs of the cluster through DISTRIBUTED shared memory (CTA 0 reads the other CTAs' results,
// spread over its threads, and merges them the same way) - and CTA 0 writes the outputs: no workspace in global memory, no
// ticket, no fence, no second launch; bit-reproducible.
//   acc, grad, jerk, acc + jerk : the pair arithmetic of AccPassT / GradPassT (policies.cuh), partial sums added in the order above;
//   dtmin     : DtPassT's refined keys for every pair, merged by selects (a key clear of the other by the band decides); a
//               near-tie anywhere flags the sink, and a flagged sink is settled by an exact scan: the exact (time-step, id)
//               minimum, whatever the order.
#pragma once

#include <cooperative_groups.h>

namespace {

namespace cg = cooperative_groups;

constexpr int FEW_T = 256;                 // threads per CTA = sources per tile
constexpr int FEW_WARPS = FEW_T / 32;
constexpr int FEW_MAX_SINKS = 32;            // sinks per cluster
constexpr int FEW_GROUP_MAX_SINKS = 128;     // several clusters of 32 sinks: up to this many sinks ..
constexpr int FEW_GROUP_MAX_SRC = 16384;     // .. against at most this many sources (measured cross-over, launch rule in few_impl)
constexpr int FEW_MAX_CL = 16;             // CTAs per cluster (16 = the non-portable maximum; every B200 GPC holds >= 16 SMs)

struct FewVec3 {
    double x, y, z;
    __device__ __forceinline__ FewVec3 shfl_xor(int off) const {
        return FewVec3{__shfl_xor_sync(0xffffffffu, x, off), __shfl_xor_sync(0xffffffffu, y, off), __shfl_xor_sync(0xffffffffu, z, off)};
    }
};

struct FewAcc {
    using P = AccPassT<false>;
    using Args = AccArgs;
    static constexpr int REC = P::REC;
    using Raw = P::Raw;
    using Sink = P::Sink;
    using State = P::Acc;
    using Val = FewVec3;
    __device__ __forceinline__ static void fetch(const SrcArrays& s, int j, Raw& w) { P::fetch(s, j, w); }
    __device__ __forceinline__ static void emit(const Raw& w, double2* o) { P::emit(w, o); }
    __device__ __forceinline__ static void load_sink(const Args& a, int id, Sink& s) { P::load_sink(a, id, s); }
    __device__ __forceinline__ static void init(State& c) { P::init(c); }
    __device__ __forceinline__ static void pair(const Args& a, const Sink& s, State& c, const double* __restrict__ r) { P::pair(a, s, c, r); }
    __device__ __forceinline__ static Val value(const State& c) { return Val{c.x, c.y, c.z}; }
    __device__ __forceinline__ static Val identity() { return Val{0.0, 0.0, 0.0}; }
    __device__ __forceinline__ static void merge(const Args&, int, Val& c, const Val& o) { c.x += o.x; c.y += o.y; c.z += o.z; }
    __device__ __forceinline__ static void settle(const Args&, const SrcArrays&, int, int, int, Val*, Val (*)[FEW_MAX_SINKS]) {}
    static constexpr int PARTS = 1;          // threads that share the output of one sink
    __device__ __forceinline__ static void write(const Args& a, int row, int, const Val& v, int) {
        double* o = a.out + 3 * (size_t)row;
        o[0] = a.G * v.x; o[1] = a.G * v.y; o[2] = a.G * v.z;
    }
};

struct FewGrad {
    using P = GradPassT<false, false>;
    using Args = GradArgs;
    static constexpr int REC = P::REC;
    using Raw = P::Raw;
    using Sink = P::Sink;
    using State = P::Acc;
    using Val = FewVec3;
    __device__ __forceinline__ static void fetch(const SrcArrays& s, int j, Raw& w) { P::fetch(s, j, w); }
    __device__ __forceinline__ static void emit(const Raw& w, double2* o) { P::emit(w, o); }
    __device__ __forceinline__ static void load_sink(const Args& a, int id, Sink& s) { P::load_sink(a, id, s); }
    __device__ __forceinline__ static void init(State& c) { P::init(c); }
    __device__ __forceinline__ static void pair(const Args& a, const Sink& s, State& c, const double* __restrict__ r) { P::pair(a, s, c, r); }
    // C_i = U - 3 W, formed per thread as GradPassT::store does per split
    __device__ __forceinline__ static Val value(const State& c) { return Val{fma(-3.0, c.wx, c.ux), fma(-3.0, c.wy, c.uy), fma(-3.0, c.wz, c.uz)}; }
    __device__ __forceinline__ static Val identity() { return Val{0.0, 0.0, 0.0}; }
    __device__ __forceinline__ static void merge(const Args&, int, Val& c, const Val& o) { c.x += o.x; c.y += o.y; c.z += o.z; }
    __device__ __forceinline__ static void settle(const Args&, const SrcArrays&, int, int, int, Val*, Val (*)[FEW_MAX_SINKS]) {}
    static constexpr int PARTS = 1;          // threads that share the output of one sink
    __device__ __forceinline__ static void write(const Args& a, int row, int, const Val& v, int) {
        double* o = a.out + 3 * (size_t)row;
        o[0] = a.G * v.x; o[1] = a.G * v.y; o[2] = a.G * v.z;
    }
};

// acceleration (Eq. 6) and jerk (Eq. 28) in one pass (bifrost_acc_jerk): GradPassT<false, true> over (x, v, m) records
struct FewVec6 {
    double x, y, z, u, v, w;
    __device__ __forceinline__ FewVec6 shfl_xor(int off) const {
        return FewVec6{__shfl_xor_sync(0xffffffffu, x, off), __shfl_xor_sync(0xffffffffu, y, off), __shfl_xor_sync(0xffffffffu, z, off),
                       __shfl_xor_sync(0xffffffffu, u, off), __shfl_xor_sync(0xffffffffu, v, off), __shfl_xor_sync(0xffffffffu, w, off)};
    }
};

struct FewAccJerk {
    using P = GradPassT<false, true>;
    using Args = GradArgs;
    static constexpr int REC = P::REC;
    using Raw = P::Raw;
    using Sink = P::Sink;
    using State = P::Acc;
    using Val = FewVec6;                     // jerk (x, y, z), acceleration (u, v, w)
    __device__ __forceinline__ static void fetch(const SrcArrays& s, int j, Raw& w) { P::fetch(s, j, w); }
    __device__ __forceinline__ static void emit(const Raw& w, double2* o) { P::emit(w, o); }
    __device__ __forceinline__ static void load_sink(const Args& a, int id, Sink& s) { P::load_sink(a, id, s); }
    __device__ __forceinline__ static void init(State& c) { P::init(c); }
    __device__ __forceinline__ static void pair(const Args& a, const Sink& s, State& c, const double* __restrict__ r) { P::pair(a, s, c, r); }
    __device__ __forceinline__ static Val value(const State& c) {
        return Val{fma(-3.0, c.wx, c.ux), fma(-3.0, c.wy, c.uy), fma(-3.0, c.wz, c.uz), c.ax, c.ay, c.az};
    }
    __device__ __forceinline__ static Val identity() { return Val{0.0, 0.0, 0.0, 0.0, 0.0, 0.0}; }
    __device__ __forceinline__ static void merge(const Args&, int, Val& c, const Val& o) {
        c.x += o.x; c.y += o.y; c.z += o.z; c.u += o.u; c.v += o.v; c.w += o.w;
    }
    __device__ __forceinline__ static void settle(const Args&, const SrcArrays&, int, int, int, Val*, Val (*)[FEW_MAX_SINKS]) {}
    static constexpr int PARTS = 2;          // one thread writes the jerk, one the acceleration
    __device__ __forceinline__ static void write(const Args& a, int row, int, const Val& v, int part) {
        double* o = (part == 0 ? a.out : a.out2) + 3 * (size_t)row;
        if (part == 0) { o[0] = a.G * v.x; o[1] = a.G * v.y; o[2] = a.G * v.z; }
        else { o[0] = a.G * v.u; o[1] = a.G * v.v; o[2] = a.G * v.w; }
    }
};

// the running bests of Eq. 21 and Eq. 22 as DtPassT keeps them: refined keys (m_i + m_j) / r^3 and v^2 / r^2 (maximised), the
// source ids (-1: none yet), and amb: a near-tie was met on the way (bit 0: Eq. 21, bit 1: Eq. 22)
struct FewDtVal {
    double kff, kfb;
    int jff, jfb, amb, pad;
    __device__ __forceinline__ FewDtVal shfl_xor(int off) const {
        return FewDtVal{__shfl_xor_sync(0xffffffffu, kff, off), __shfl_xor_sync(0xffffffffu, kfb, off),
                        __shfl_xor_sync(0xffffffffu, jff, off), __shfl_xor_sync(0xffffffffu, jfb, off),
                        __shfl_xor_sync(0xffffffffu, amb, off), 0};
    }
};

// dtmin: the refined keys of DtPassT for every pair (23 FP64 instructions, no tier-1 pre-selection: a thread sees only a few
// sources, so its running best changes all the time).  A contender (one pair against a thread's running best, or one
// running best against another) replaces the incumbent when its key is clear of it by the 1e-12 band, is ignored when it is
// clearly below, and otherwise - a near-tie - only raises the sticky flag: no branch anywhere (a branch to the exact
// evaluation in every merge cost 5 us for one sink, 14 us for 32).  The exact minimum is never replaced by a clear decision
// and never fails to replace one (its key is the largest to a few ulp), so without a flag the survivor IS the exact
// (time-step, id) minimum; a flagged sink (exactly tied inputs: lattices, coincident particles) is settled afterwards by
// an exact scan of the whole source list with the oracle's rule (settle).
struct FewDt {
    using P = DtPassT<false>;
    using Args = DtArgs;
    static constexpr int REC = P::REC;
    using Raw = P::Raw;
    using Sink = P::Sink;
    using State = FewDtVal;
    using Val = FewDtVal;
    __device__ __forceinline__ static void fetch(const SrcArrays& s, int j, Raw& w) { P::fetch(s, j, w); }
    __device__ __forceinline__ static void emit(const Raw& w, double2* o) { P::emit(w, o); }
    __device__ __forceinline__ static void load_sink(const Args& a, int id, Sink& s) { P::load_sink(a, id, s); }
    __device__ __forceinline__ static void init(State& c) { c = identity(); }
    // dt_exact_ids inlined: the out-of-line one takes the argument block by reference, which makes the kernel copy its 248
    // bytes of parameters to local memory on entry (0.9 us of a 10 us call)
    __device__ __forceinline__ static double exact(const Args& a, int w, int i, int j) {
        const size_t oi = 3 * (size_t)i, oj = 3 * (size_t)j;
        const double dx = a.pos[oj] - a.pos[oi], dy = a.pos[oj + 1] - a.pos[oi + 1], dz = a.pos[oj + 2] - a.pos[oi + 2];
        if (w == 0) return dt_ff_exact(dx, dy, dz, a.G, a.mass[i], a.mass[j], a.eta_ff);
        return dt_fb_exact(dx, dy, dz, a.vel[oj] - a.vel[oi], a.vel[oj + 1] - a.vel[oi + 1], a.vel[oj + 2] - a.vel[oi + 2], a.eta_fb);
    }
    // contender (key, j; j < 0: none) against the incumbent (kb, jb)
    __device__ __forceinline__ static void contend(double key, int j, double& kb, int& jb, int& amb, int bit) {
        const bool clear = (j >= 0) & ((key * KEY_SLACK > kb) | (jb < 0));
        const bool near = (j >= 0) & !clear & (key >= kb * KEY_SLACK) & (j != jb);
        amb |= near ? bit : 0;
        kb = clear ? key : kb; jb = clear ? j : jb;
    }
    __device__ __forceinline__ static void pair(const Args&, const Sink& s, State& c, const double* __restrict__ r) {
        const int jid = __double2loint(r[7]);
        double kff, kfb;
        P::keys(s, r, kff, kfb);
        const bool other = jid != s.id;                       // the self pair never contends; nor does v_ij = 0 for Eq. 22 (T3)
        contend(kff, other ? jid : -1, c.kff, c.jff, c.amb, 1);
        contend(kfb, (other && kfb > 0.0) ? jid : -1, c.kfb, c.jfb, c.amb, 2);
    }
    __device__ __forceinline__ static Val value(const State& c) { return c; }
    __device__ __forceinline__ static Val identity() { return Val{0.0, 0.0, -1, -1, 0, 0}; }
    __device__ __forceinline__ static void merge(const Args&, int, Val& c, const Val& o) {
        c.amb |= o.amb;
        contend(o.kff, o.jff, c.kff, c.jff, c.amb, 1);
        contend(o.kfb, o.jfb, c.kfb, c.jfb, c.amb, 2);
    }
    // CTA 0, all threads: every flagged sink gets the exact (time-step, id) minimum over the WHOLE source list, by the
    // oracle's rule on dt_exact_ids (smaller time-step; equal -> smaller id; +inf never wins).  Rare and slow (an exact
    // evaluation per source), but parallel: n_src / 256 evaluations per thread.
    __device__ static void settle(const Args& a, const SrcArrays& src, int k0, int n_here, int n_src, Val* cta_sm, Val (*warp_sm)[FEW_MAX_SINKS]) {
        const double inf = __longlong_as_double(0x7ff0000000000000LL);
        const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
        for (int q = 0; q < n_here; ++q) {
            const int amb = cta_sm[q].amb;                    // the same for every thread
            if (!amb) continue;
            const int i = a.sink_idx ? a.sink_idx[k0 + q] : k0 + q;
            for (int w = 0; w < 2; ++w) {
                if (!((amb >> w) & 1)) continue;
                double tb = inf;
                int jb = -1;
                for (int l = t; l < n_src; l += FEW_T) {
                    const int j = src.src_idx ? src.src_idx[l] : l;
                    if (j == i) continue;
                    const double tt = exact(a, w, i, j);
                    if (tt < tb || (tt == tb && j < jb)) { tb = tt; jb = j; }
                }
                for (int off = 16; off > 0; off >>= 1) {
                    const double to = __shfl_xor_sync(0xffffffffu, tb, off);
                    const int jo = __shfl_xor_sync(0xffffffffu, jb, off);
                    if (to < tb || (to == tb && jo >= 0 && jo < jb)) { tb = to; jb = jo; }
                }
                __syncthreads();
                if (lane == 0) { warp_sm[warp][0].kff = tb; warp_sm[warp][0].jff = jb; }
                __syncthreads();
                if (t == 0) {
                    for (int ww = 1; ww < FEW_WARPS; ++ww) {
                        const double to = warp_sm[ww][0].kff;
                        const int jo = warp_sm[ww][0].jff;
                        if (to < tb || (to == tb && jo >= 0 && jo < jb)) { tb = to; jb = jo; }
                    }
                    if (w == 0) cta_sm[q].jff = jb; else cta_sm[q].jfb = jb;
                }
                __syncthreads();
            }
        }
    }
    // Eq. 21 / Eq. 22 for the winning pairs in IEEE operations in the oracle's order (as DtPassT::finish); the two
    // time-steps of a sink by two threads
    static constexpr int PARTS = 2;
    __device__ __forceinline__ static void write(const Args& a, int row, int id, const Val& v, int part) {
        const double inf = __longlong_as_double(0x7ff0000000000000LL);
        if (part == 0) {
            if (a.dt_ff) a.dt_ff[row] = v.jff >= 0 ? exact(a, 0, id, v.jff) : inf;
            if (a.j_ff) a.j_ff[row] = v.jff;
        } else {
            if (a.dt_fb) a.dt_fb[row] = v.jfb >= 0 ? exact(a, 1, id, v.jfb) : inf;
            if (a.j_fb) a.j_fb[row] = v.jfb;
        }
    }
};

// grid = one cluster of CL CTAs of FEW_T threads per group of nsp sinks.  One group: nsp = n_sink rounded up to a power of two
// (<= 32); several groups: nsp = 32.
template <class F>
__global__ void __launch_bounds__(FEW_T, 1)
few_sinks_kernel(const typename F::Args a, const SrcArrays src, int n_sink, int n_src, int nsp, int compact) {
    constexpr int REC = F::REC;
    __shared__ __align__(16) double tile_sm[FEW_T * REC];
    __shared__ typename F::Val warp_sm[FEW_WARPS][FEW_MAX_SINKS];     // per warp, per sink
    __shared__ typename F::Val cta_sm[FEW_MAX_SINKS];                 // this CTA's result per sink (read by CTA 0 of the cluster)
    cg::cluster_group cluster = cg::this_cluster();
    const int cl = (int)cluster.num_blocks(), rank = (int)cluster.block_rank();
    const int t = threadIdx.x, lane = t & 31, warp = t >> 5;
    const int s = t & (nsp - 1), rep = t / nsp, reps = FEW_T / nsp;   // this thread: sink s, sources rep, rep + reps, .. of a tile

    const int k0 = ((int)blockIdx.x / cl) * nsp;                      // first sink of this cluster (several clusters: nsp = 32)
    const int k = k0 + s < n_sink ? k0 + s : n_sink - 1;              // a shadow thread repeats the last sink; never merged
    const int id = a.sink_idx ? a.sink_idx[k] : k;
    typename F::Sink sink;
    typename F::State st;
    F::load_sink(a, id, sink);
    F::init(st);

    // the tiles of the source list are dealt to the CTAs of the cluster round robin
    const int n_tiles = (n_src + FEW_T - 1) / FEW_T;
    typename F::Raw raw;
    auto fetch_tile = [&](int tile) {
        const int l = tile * FEW_T + t;
        F::fetch(src, l < n_src ? (src.src_idx ? src.src_idx[l] : l) : -1, raw);
    };
    if (rank < n_tiles) fetch_tile(rank);
    for (int tile = rank; tile < n_tiles; tile += cl) {
        F::emit(raw, reinterpret_cast<double2*>(tile_sm + t * REC));
        __syncthreads();
        if (tile + cl < n_tiles) fetch_tile(tile + cl);              // in flight while this tile is evaluated
        const int cnt = min(FEW_T, n_src - tile * FEW_T);
#pragma unroll 4
        for (int jj = rep; jj < cnt; jj += reps) {
            double r[REC];
#pragma unroll
            for (int q = 0; q < REC; q += 2) {
                const double2 v = *reinterpret_cast<const double2*>(tile_sm + jj * REC + q);
                r[q] = v.x; r[q + 1] = v.y;
            }
            F::pair(a, sink, st, r);
        }
        __syncthreads();                                               // everyone is done with the tile before the next emit
    }

    // Merge over the threads of the CTA that share a sink, in a fixed order: xor-butterfly over the lane bits above nsp
    // (lane = s mod nsp; every lane ends with a value formed in the same order), then the warps in warp order through
    // shared memory.  Result for sink q in cta_sm[q].
    auto cta_reduce = [&](typename F::Val v) {
        for (int off = nsp; off < 32; off <<= 1) F::merge(a, id, v, v.shfl_xor(off));
        if (lane < nsp) warp_sm[warp][lane] = v;
        __syncthreads();
        if (t < nsp) {
            typename F::Val c = warp_sm[0][t];
            for (int w = 1; w < FEW_WARPS; ++w) F::merge(a, id, c, warp_sm[w][t]);
            cta_sm[t] = c;
        }
        __syncthreads();
    };
    cta_reduce(k0 + s < n_sink ? F::value(st) : F::identity());
    cluster.sync();
    if (rank == 0) {
        // the CTAs of the cluster: thread (s, rep) of CTA 0 fetches the results of ranks rep, rep + reps, .. for its sink
        // through distributed shared memory (all reads in flight at once), then the same in-CTA merge
        typename F::Val v = F::identity();
        for (int q = rep; q < cl; q += reps) F::merge(a, id, v, *cluster.map_shared_rank(&cta_sm[s], q));
        cta_reduce(v);
        F::settle(a, src, k0, min(nsp, n_sink - k0), n_src, cta_sm, warp_sm);
        if (t < nsp * F::PARTS && k0 + s < n_sink) F::write(a, compact ? k0 + s : id, id, cta_sm[s], t / nsp);   // s = t mod nsp
    }
    cluster.sync();                             // a CTA's shared memory must outlive CTA 0's reads
}

}  // namespace
