// subsystems.cuh - NEXT-2 / NEXT-3: shared subsystem time-step (Eq. 20), neighbour search (Eq. 18-19), connected components.
// Part of the single translation unit bifrost.cu (see its header and DESIGN.md); not a public header.
#pragma once

namespace {

// NEXT-2, Eq. 20: eps_i = min_{j in S} eps_j.  Non-negative doubles order like their
// bit patterns read as unsigned integers, so the segment minimum is an integer atomicMin: exact and
// independent of the order in which members arrive (deterministic).
__global__ void smin_fill_kernel(int n, unsigned long long* __restrict__ smin) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) smin[i] = 0x7ff0000000000000ULL;     // +inf
}
__global__ void smin_reduce_kernel(int n, const int32_t* __restrict__ subsys, const double* __restrict__ dt,
                                   unsigned long long* __restrict__ smin) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int s = subsys[i];
    if (s >= 0) atomicMin(&smin[s], (unsigned long long)__double_as_longlong(dt[i]));
}
__global__ void smin_apply_kernel(int n, const int32_t* __restrict__ subsys, const unsigned long long* __restrict__ smin,
                                  double* __restrict__ dt) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int s = subsys[i];
    if (s >= 0) dt[i] = __longlong_as_double((long long)smin[s]);
}

// (NgbArgs and ngb_exact, the exact evaluation of Eq. 18-19, live in policies.cuh: the fused dtmin + neighbours pass uses them too)

template <int S, int T, int MINB>
__global__ void __launch_bounds__(T, MINB)
ngb_kernel(const NgbArgs a, const Geom g, const double* __restrict__ src_rec) {
    constexpr int REC = 8;                                  // DtPass records: x y z m vx vy vz {id}
    constexpr int CHUNKS = TILE * REC * 8 / 16;
    __shared__ __align__(16) double sm[2][TILE * REC];
    double sx[S], sy[S], sz[S];
    int ids[S], cnt[S];
    int32_t* lst[S];
    const int kbase = blockIdx.x * (T * S) + threadIdx.x;
#pragma unroll
    for (int s = 0; s < S; ++s) {
        const int k = kbase + s * T;
        const int kk = k < g.n_sink ? k : g.n_sink - 1;
        ids[s] = a.sink_idx ? a.sink_idx[kk] : kk;
        sx[s] = a.pos[3 * (size_t)ids[s]]; sy[s] = a.pos[3 * (size_t)ids[s] + 1]; sz[s] = a.pos[3 * (size_t)ids[s] + 2];
        cnt[s] = 0;
        if (k >= g.n_sink) lst[s] = nullptr;                // tail threads shadow the last sink and write nothing
        else if (g.n_split == 1) lst[s] = a.out_list + (size_t)(g.compact ? k : ids[s]) * a.cap;
        else lst[s] = a.plist + ((size_t)blockIdx.y * g.n_sink + k) * a.cap;
    }
    const int guard_hi = __double2hiint(a.r2_guard);
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
        const int cnt_t = min(TILE, g.n_src - tile * TILE);
        const double* __restrict__ tb = sm[buf];
#pragma unroll 2
        for (int jj = 0; jj < cnt_t; ++jj) {
            const double2 p0 = *reinterpret_cast<const double2*>(tb + jj * REC);
            const double pz = tb[jj * REC + 2];
            // fast path: the S distances and ONE rarely taken branch.  r^2 >= 0 and the guard >= 0, so
            // r^2 < guard implies hi(r^2) <= hi(guard): a necessary condition on the integer pipe.
            double dx[S], dy[S], dz[S], r2[S];
            bool any = false;
#pragma unroll
            for (int s = 0; s < S; ++s) {
                dx[s] = p0.x - sx[s]; dy[s] = p0.y - sy[s]; dz[s] = pz - sz[s];
                r2[s] = fma(dx[s], dx[s], fma(dy[s], dy[s], dz[s] * dz[s]));
                any |= __double2hiint(r2[s]) <= guard_hi;
            }
            if (any) {                                      // rare: candidate pairs, exact evaluation
                const int j = __double2loint(tb[jj * REC + 7]);
#pragma unroll
                for (int s = 0; s < S; ++s) {
                    if (!(r2[s] < a.r2_guard) || j == ids[s]) continue;
                    const size_t o = 3 * (size_t)ids[s];
                    const double ux = tb[jj * REC + 4] - a.vel[o], uy = tb[jj * REC + 5] - a.vel[o + 1],
                                 uz = tb[jj * REC + 6] - a.vel[o + 2];
                    if (ngb_exact(a, dx[s], dy[s], dz[s], ux, uy, uz, a.mass[ids[s]], tb[jj * REC + 3])) {
                        if (lst[s] && cnt[s] < a.cap) lst[s][cnt[s]] = j;
                        ++cnt[s];
                    }
                }
            }
        }
        __syncthreads();
    }
#pragma unroll
    for (int s = 0; s < S; ++s) {
        const int k = kbase + s * T;
        if (k >= g.n_sink) continue;
        if (g.n_split == 1) a.out_count[g.compact ? k : ids[s]] = cnt[s];
        else a.pcount[(size_t)blockIdx.y * g.n_sink + k] = cnt[s];
    }
}

// concatenate the per-split lists in split order (= source-list order); the count is never truncated
__global__ void ngb_finish_kernel(const NgbArgs a, const Geom g) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= g.n_sink) return;
    const int id = a.sink_idx ? a.sink_idx[k] : k;
    const size_t row = g.compact ? k : id;
    int total = 0;
    for (int s = 0; s < g.n_split; ++s) {
        const int c = a.pcount[(size_t)s * g.n_sink + k];
        const int32_t* l = a.plist + ((size_t)s * g.n_sink + k) * a.cap;
        for (int q = 0; q < c && q < a.cap && total + q < a.cap; ++q) a.out_list[row * a.cap + total + q] = l[q];
        total += c;
    }
    a.out_count[row] = total;
}

// Subsystems = connected components of the neighbour graph.  The paper traverses
// the graph depth-first on the host; here a lock-free union-find: every edge hooks the larger root
// under the smaller one with an integer compare-and-swap, so the root of a component ends up as its
// smallest particle id whatever the order of the edges (deterministic), then paths are flattened.
__device__ __forceinline__ int uf_find(int* parent, int x) {
    int p = parent[x];
    while (p != x) {
        const int gp = parent[p];
        if (gp != p) parent[x] = gp;            // path halving (benign race: only ever shortens)
        x = p; p = gp;
    }
    return x;
}
__global__ void comp_init_kernel(int n, int* __restrict__ parent, unsigned char* __restrict__ flag) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) { parent[i] = i; flag[i] = 0; }
}
__global__ void comp_hook_kernel(int n, int cap, const int32_t* __restrict__ count, const int32_t* __restrict__ list,
                                 int* parent, unsigned char* __restrict__ flag) {
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int i = (int)(t / cap), q = (int)(t % cap);
    if (i >= n || q >= count[i]) return;
    const int j = list[(size_t)i * cap + q];
    if (j < 0 || j >= n || j == i) return;
    flag[i] = 1; flag[j] = 1;
    int x = i, y = j;
    while (true) {
        x = uf_find(parent, x); y = uf_find(parent, y);
        if (x == y) break;
        if (x < y) { const int t2 = x; x = y; y = t2; }     // x = larger root
        const int old = atomicCAS(&parent[x], x, y);
        if (old == x) break;                                // x was still a root: hooked under the smaller root
        x = old;                                            // someone else hooked x first: retry from there
    }
}
__global__ void comp_label_kernel(int n, int* parent, const unsigned char* __restrict__ flag, int32_t* __restrict__ subsys) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    subsys[i] = flag[i] ? uf_find(parent, i) : -1;
}

}  // namespace
