// pair_kernels.cuh - a1-a7: pair_kernel (large sink sets), pack_kernel, finish_kernel and pair_fused_kernel (small sink sets in one launch).
// Part of the single translation unit bifrost.cu (see its header and DESIGN.md); not a public header.
#pragma once

#include <cooperative_groups.h>

namespace {

// All S sinks of a thread against one source record.  A policy may provide a phase-major
// `pairs<S>` (same arithmetic as S calls of pair(), written stage by stage over the sinks so that
// the accumulate DFMAs of one sink stay adjacent and share their weight through the operand-reuse
// cache: the register file feeds one 64-bit operand per clock per SM sub-partition).
template <class P, int S, class = void>
struct PairsOf {
    __device__ __forceinline__ static void run(const typename P::Args& a, const typename P::Sink* sink,
                                               typename P::Acc* accu, const double* __restrict__ r) {
#pragma unroll
        for (int s = 0; s < S; ++s) P::pair(a, sink[s], accu[s], r);
    }
};
template <class P, int S>
struct PairsOf<P, S, typename std::enable_if<(P::PHASED_MIN_S > 0) && (S >= P::PHASED_MIN_S)>::type> {
    __device__ __forceinline__ static void run(const typename P::Args& a, const typename P::Sink* sink,
                                               typename P::Acc* accu, const double* __restrict__ r) {
        P::template pairs<S>(a, sink, accu, r);
    }
};
template <class P, int S>
__device__ __forceinline__ void pairs_of(const typename P::Args& a, const typename P::Sink* sink, typename P::Acc* accu,
                                         const double* __restrict__ r) {
    PairsOf<P, S>::run(a, sink, accu, r);
}

// ----------------------------------------------------------------------------------------
// a2-a4: the pair kernel.  grid = (ceil(n_sink / (T*S)), n_split); T threads, S sinks per thread,
// MINB resident CTAs per SM, inner loop unrolled UNR times.
// ----------------------------------------------------------------------------------------
template <class P, int S, int T, int MINB, int UNR>
__global__ void __launch_bounds__(T, MINB)
pair_kernel(const typename P::Args a, const Geom g, const double* __restrict__ src_rec) {
    constexpr int REC = P::REC;
    constexpr int CHUNKS = TILE * REC * 8 / 16;            // 16-B chunks per tile
    __shared__ __align__(16) double sm[2][TILE * REC];

    typename P::Sink sink[S];
    typename P::Acc accu[S];
    int ids[S];
    const int kbase = blockIdx.x * (T * S) + threadIdx.x;
#pragma unroll
    for (int s = 0; s < S; ++s) {
        const int k = kbase + s * T;
        const int kk = k < g.n_sink ? k : g.n_sink - 1;      // tail threads shadow the last sink
        ids[s] = a.sink_idx ? a.sink_idx[kk] : kk;
        P::load_sink(a, ids[s], sink[s]);
        P::init(accu[s]);
    }

    const int n_tiles = (g.n_src + TILE - 1) / TILE;
    const int tile0 = blockIdx.y * g.tiles_per_split;
    const int tile1 = min(tile0 + g.tiles_per_split, n_tiles);

    auto load_tile = [&](int tile, int buf) {
        const double* gsrc = src_rec + (size_t)tile * TILE * REC;
        for (int ch = threadIdx.x; ch < CHUNKS; ch += T) cp_async16(&sm[buf][2 * ch], gsrc + 2 * ch);
        cp_async_commit();
    };

    if (tile0 < tile1) load_tile(tile0, 0);
    for (int tile = tile0; tile < tile1; ++tile) {
        const int buf = (tile - tile0) & 1;
        if (tile + 1 < tile1) { load_tile(tile + 1, buf ^ 1); cp_async_wait<1>(); }
        else cp_async_wait<0>();
        __syncthreads();
        const int cnt = min(TILE, g.n_src - tile * TILE);
        const double* __restrict__ tb = sm[buf];
#pragma unroll UNR
        for (int jj = 0; jj < cnt; ++jj) {
            double r[REC];
#pragma unroll
            for (int q = 0; q < REC; q += 2) {
                const double2 v = *reinterpret_cast<const double2*>(tb + jj * REC + q);
                r[q] = v.x; r[q + 1] = v.y;
            }
            pairs_of<P, S>(a, sink, accu, r);
        }
        __syncthreads();
    }

#pragma unroll
    for (int s = 0; s < S; ++s) {
        const int k = kbase + s * T;
        if (k < g.n_sink) P::store(a, g, blockIdx.y, k, ids[s], sink[s], accu[s]);
    }
}

// ----------------------------------------------------------------------------------------
// a1: pack kernels (gather sources through the index list into aligned records; the tail of
// the last tile is zero-filled so the cp.async stage never reads undefined memory).
// ----------------------------------------------------------------------------------------

template <class P>
__global__ void pack_kernel(int n_src, int n_pad, const SrcArrays src, double* __restrict__ rec) {
    const int l = blockIdx.x * blockDim.x + threadIdx.x;
    if (l >= n_pad) return;
    typename P::Raw w;
    P::fetch(src, l < n_src ? (src.src_idx ? src.src_idx[l] : l) : -1, w);
    P::emit(w, reinterpret_cast<double2*>(rec + (size_t)l * P::REC));
}

// ----------------------------------------------------------------------------------------
// a5 + a7 as a kernel of its own (large sink sets): P::finish for every sink.
// ----------------------------------------------------------------------------------------
template <class P>
__global__ void finish_kernel(const typename P::Args a, const Geom g) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= g.n_sink) return;
    P::finish(a, g, k, a.sink_idx ? a.sink_idx[k] : k, 0, 1, true);
}

// ----------------------------------------------------------------------------------------
// a1-a7 in ONE launch for small sink sets (the faster levels of the time-step hierarchy,
// PAPER.md:L295): each CTA gathers its source tiles straight from the caller's arrays (the next
// tile's loads are in flight while the current one is evaluated), and when the source range is
// split across blockIdx.y the CTA that arrives last at a ticket (one per blockIdx.x) reduces all
// partials in split order - so the result does not depend on which CTA that is (deterministic) and
// no second or third launch is needed.
// ----------------------------------------------------------------------------------------
// shared memory for the cluster reduction of pair_fused_kernel: 3 doubles per sink of the CTA for the policies that use it
template <class P, int S, int T>
__device__ __forceinline__ double* part_sm_of() {
    __shared__ double part_sm[(P::CLUSTER_REDUCE || P::CLUSTER_MERGE) ? 3 * T * S : 1];
    return part_sm;
}

template <class P, int S, int T, int MINB, int UNR>
__global__ void __launch_bounds__(T, MINB)
pair_fused_kernel(const typename P::Args a, const Geom g, const SrcArrays src, unsigned* __restrict__ ticket) {
    static_assert(T >= TILE, "one gathering thread per source of a tile");
    constexpr int REC = P::REC;
    __shared__ __align__(16) double sm[2][TILE * REC];
    __shared__ int s_last;

    typename P::Sink sink[S];
    typename P::Acc accu[S];
    int ids[S];
    const int kbase = blockIdx.x * (T * S) + threadIdx.x;
#pragma unroll
    for (int s = 0; s < S; ++s) {
        const int k = kbase + s * T;
        const int kk = k < g.n_sink ? k : g.n_sink - 1;
        ids[s] = a.sink_idx ? a.sink_idx[kk] : kk;
        P::load_sink(a, ids[s], sink[s]);
        P::init(accu[s]);
    }

    const int n_tiles = (g.n_src + TILE - 1) / TILE;
    const int tile0 = blockIdx.y * g.tiles_per_split;
    const int tile1 = min(tile0 + g.tiles_per_split, n_tiles);

    typename P::Raw raw;
    auto fetch_tile = [&](int tile) {
        const int l = tile * TILE + threadIdx.x;
        if (threadIdx.x < TILE) P::fetch(src, l < g.n_src ? (src.src_idx ? src.src_idx[l] : l) : -1, raw);
    };
    auto emit_tile = [&](int buf) {
        if (threadIdx.x < TILE) P::emit(raw, reinterpret_cast<double2*>(sm[buf] + threadIdx.x * REC));
    };

    if (tile0 < tile1) { fetch_tile(tile0); emit_tile(0); }
    for (int tile = tile0; tile < tile1; ++tile) {
        const int buf = (tile - tile0) & 1;
        __syncthreads();                       // sm[buf] complete; everyone is done with sm[buf ^ 1]
        const bool more = tile + 1 < tile1;
        if (more) fetch_tile(tile + 1);
        const int cnt = min(TILE, g.n_src - tile * TILE);
        const double* __restrict__ tb = sm[buf];
#pragma unroll UNR
        for (int jj = 0; jj < cnt; ++jj) {
            double r[REC];
#pragma unroll
            for (int q = 0; q < REC; q += 2) {
                const double2 v = *reinterpret_cast<const double2*>(tb + jj * REC + q);
                r[q] = v.x; r[q + 1] = v.y;
            }
            pairs_of<P, S>(a, sink, accu, r);
        }
        if (more) emit_tile(buf ^ 1);
    }

    // Launched as thread-block clusters along blockIdx.y (launch_fused, vec3 policies): the CTAs of a cluster add their
    // partials through DISTRIBUTED SHARED MEMORY in rank order - CTA r takes every cl-th double of the block's n_local x 3 -
    // and only one partial per cluster goes to global memory.  The last CTA's reduction, a chain of L2 round trips per
    // split (10 us for 128 splits), then runs over gridDim.y / cl entries; with one cluster per sink block there is no
    // global partial, no ticket and no fence at all.
    int n_part = g.n_split;                    // entries of the [.][n_sink] partial workspace the last CTA adds
    bool stored = false;
    if constexpr (P::CLUSTER_REDUCE) {
        cooperative_groups::cluster_group cluster = cooperative_groups::this_cluster();
        const int cl = (int)cluster.dim_blocks().y;
        if (cl > 1) {
            stored = true;
            double* part_sm = part_sm_of<P, S, T>();
#pragma unroll
            for (int s = 0; s < S; ++s) P::vec3(accu[s], part_sm + 3 * (threadIdx.x + s * T));
            cluster.sync();
            const int r = (int)cluster.block_rank(), base = blockIdx.x * (T * S);
            const int n_doubles = 3 * min(T * S, g.n_sink - base);
            n_part = gridDim.y / cl;
            for (int e = r + cl * threadIdx.x; e < n_doubles; e += cl * T) {
                double sum = 0.0;
                for (int q = 0; q < cl; ++q) sum += *cluster.map_shared_rank(part_sm + e, q);
                const int k = base + e / 3, c = e % 3;
                if (n_part == 1) a.out[3 * (size_t)(g.compact ? k : (a.sink_idx ? a.sink_idx[k] : k)) + c] = a.G * sum;
                else a.partial[3 * ((size_t)(blockIdx.y / cl) * g.n_sink + k) + c] = sum;
            }
            cluster.sync();                    // shared memory must outlive the other CTAs' reads
            if (n_part == 1) return;
        }
    }
    // dtmin: the same with the policy's merge (a key clear of the other by the band decides, a near-tie is decided on the exact
    // time-steps): CTA r of the cluster merges every cl-th sink of the block over the CTAs' winners and writes one entry per
    // cluster; the last CTA's finish then runs over gridDim.y / cl entries (the exact minimum whatever the order).
    if constexpr (P::CLUSTER_MERGE) {
        cooperative_groups::cluster_group cluster = cooperative_groups::this_cluster();
        const int cl = (int)cluster.dim_blocks().y;
        if (cl > 1) {
            stored = true;
            double* part_sm = part_sm_of<P, S, T>();
#pragma unroll
            for (int s = 0; s < S; ++s) {
                double kf, kb;
                int jf, jb;
                P::partial_of(a, g, blockIdx.y, ids[s], accu[s], kf, kb, jf, jb);
                double* o = part_sm + 3 * (threadIdx.x + s * T);
                o[0] = kf; o[1] = kb; o[2] = __hiloint2double(jf, jb);
            }
            cluster.sync();
            const int r = (int)cluster.block_rank(), base = blockIdx.x * (T * S);
            const int n_local = min(T * S, g.n_sink - base);
            n_part = gridDim.y / cl;
            for (int kl = r + cl * threadIdx.x; kl < n_local; kl += cl * T) {
                double v[8][3];
#pragma unroll
                for (int q = 0; q < 8; ++q) {                 // all remote reads in flight before the first merge
                    const double* p = cluster.map_shared_rank(part_sm + 3 * kl, q < cl ? q : 0);
                    v[q][0] = p[0]; v[q][1] = p[1]; v[q][2] = p[2];
                }
                const int k = base + kl, i = a.sink_idx ? a.sink_idx[k] : k;
                double kb[2] = {0.0, 0.0};
                int jb[2] = {-1, -1};
#pragma unroll
                for (int q = 0; q < 8; ++q) {
                    if (q < cl) {
                        P::merge(a, i, 0, v[q][0], __double2hiint(v[q][2]), kb[0], jb[0]);
                        P::merge(a, i, 1, v[q][1], __double2loint(v[q][2]), kb[1], jb[1]);
                    }
                }
                const size_t o = (size_t)(blockIdx.y / cl) * 2 * g.n_sink + k;
                a.pkey[o] = kb[0]; a.pkey[o + g.n_sink] = kb[1];
                a.pid[o] = jb[0];  a.pid[o + g.n_sink] = jb[1];
            }
            cluster.sync();                    // shared memory must outlive the other CTAs' reads
        }
    }
    if (!stored) {
#pragma unroll
        for (int s = 0; s < S; ++s) {
            const int k = kbase + s * T;
            if (k < g.n_sink) P::store(a, g, blockIdx.y, k, ids[s], sink[s], accu[s]);
        }
    }
    if (g.n_split == 1) {
        if (P::ALWAYS_FINISH) {                // a thread finishes the sinks it stored itself
#pragma unroll
            for (int s = 0; s < S; ++s) {
                const int k = kbase + s * T;
                if (k < g.n_sink) P::finish(a, g, k, ids[s], 0, 1, true);
            }
        }
        return;
    }
    __threadfence();
    __syncthreads();
    // one atomicAdd per CTA (a compare-and-swap loop here costs O(splits^2) retries on one address: measured 54 us instead
    // of 12 us for 1 sink x 128 splits); the last CTA zeroes the ticket again, so the next launch and CUDA-graph replays
    // start clean; after a failed launch the host zeroes all tickets before the next one (bifrost_ctx::tickets_dirty)
    if (threadIdx.x == 0) s_last = (atomicAdd(&ticket[blockIdx.x], 1u) == gridDim.y - 1);
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    // the last CTA reduces: L lanes per sink when this CTA's sinks leave threads to spare
    Geom gf = g;
    gf.n_split = n_part;
    const int base = blockIdx.x * (T * S);
    const int n_local = min(T * S, g.n_sink - base);
    int L = 1;
    while (L < 32 && n_local * (2 * L) <= T) L *= 2;
    if (L == 1) {
#pragma unroll
        for (int s = 0; s < S; ++s) {
            const int k = kbase + s * T;
            if (k < g.n_sink) P::finish(a, gf, k, ids[s], 0, 1, true);
        }
    } else {
        const int q = threadIdx.x / L;
        const bool live = q < n_local;
        const int k = base + (live ? q : 0);
        P::finish(a, gf, k, a.sink_idx ? a.sink_idx[k] : k, threadIdx.x % L, L, live);
    }
    if (threadIdx.x == 0) ticket[blockIdx.x] = 0;
}

}  // namespace
