// sym_kernels.cuh - acc (Eq. 6) and grad (Eq. 9) over ONE list that is both the sink and the source set, every
// unordered pair evaluated ONCE (Newton's third law: "pairwise kicks").
// Part of the single translation unit bifrost.cu (see its header and DESIGN.md); not a public header.
//
// 12 of acc's 15 and 22 of grad's 28 FP64 instructions per ordered pair are pair geometry that is identical for
// (i <- j) and (j <- i); here they are issued once and both members get their term:
//     acc : a_i += m_j s^-3 r_ji              a_j -= m_i s^-3 r_ji                         20 instructions per unordered pair
//     grad: C_i += m_j s^-3 t                 C_j -= m_i s^-3 t,   t = a_ji - 3 (a_ji.r_ji) r_ji / s^2   33
// The list is cut into blocks of BS = T*S positions.  A CTA owns one block as SINKS (S per thread, in registers)
// and a range of source tiles strictly beyond its block; for every source it also forms the source-side sum
// over its own sinks: per thread over its S sinks in registers, over the 32 lanes of a warp with a fixed
// reduce-scatter + butterfly of shuffles (4 sources at a time: 4.5 DADD per source and warp instead of 15), over
// the warps of the CTA through shared memory in warp order.  That sum goes to a [block][source] workspace; the
// tiles of the block itself (the diagonal) are evaluated the plain way (both orders, sink side only).  A finish
// kernel adds, for list position k in block b, the sink-side pieces of block b and the source-side rows written by
// blocks 0..b-1, all in a fixed order: bit-identical run to run, no floating-point atomics.
#pragma once

namespace {

struct SymGeom {
    int m;            // list length (sinks = sources)
    int n_tiles;      // ceil(m / TILE); records are zero-padded to n_tiles * TILE
    int bs;           // list positions per block = T * S
    int tb;           // tiles per block = bs / TILE
    int n_blocks;     // ceil(m / bs)
    int unit_tiles;   // target number of source tiles per CTA
    int compact;      // 1: output row = list position, 0: output row = particle id
    int rank, world;  // bifrost_set_shard: this launch evaluates the blocks owned by `rank` of `world` only
    // mutual mode (bifrost_acc_mutual / bifrost_grad_mutual, the inter-level sums of Eq. 12-13): sinks = list A (the m
    // entries above), sources = a DISJOINT list B; every (a, b) pair once, both lists get their sums.  No diagonal;
    // every block meets all tiles of B, whose records start at record row rec_b.
    int mutual;       // 0: one list on both sides (triangle), 1: two lists (rectangle)
    int m_b;          // length of list B
    int n_tiles_b;    // ceil(m_b / TILE)
    int rec_b;        // first record row of list B (= n_tiles * TILE)
};
// Owner of block b when the pair work is sharded over ranks (multi-GPU): blocks are dealt in snake order
// (0 1 .. w-1, w-1 .. 1 0, ...) - a block's work falls linearly with b, so every rank's share of the pairs is the
// same up to O(w / n_blocks^2).
__host__ __device__ inline int sym_owner(const SymGeom& g, int b) {
    const int q = b / g.world, r = b % g.world;
    return (q & 1) ? g.world - 1 - r : r;
}
// source tiles evaluated both ways by block b: the tiles strictly beyond the block (all tiles of B in mutual mode)
__host__ __device__ inline int sym_range(const SymGeom& g, int b) {
    if (g.mutual) return g.n_tiles_b;
    const int r = g.n_tiles - (b + 1) * g.tb;
    return r > 0 ? r : 0;
}
// first of those tiles (a tile index into the source records)
__host__ __device__ inline int sym_first(const SymGeom& g, int b) { return g.mutual ? 0 : (b + 1) * g.tb; }
// CTAs (pieces) that share block b: the first sym_diag_pieces do the block's own tiles (the diagonal), the others
// the tiles beyond the block, at most unit_tiles each
__host__ __device__ inline int sym_diag_tiles(const SymGeom& g, int b) {
    if (g.mutual) return 0;
    const int r = g.n_tiles - b * g.tb;
    return r < g.tb ? r : g.tb;
}
__host__ __device__ inline int sym_diag_pieces(const SymGeom& g, int b) {
    return (sym_diag_tiles(g, b) + g.unit_tiles - 1) / g.unit_tiles;
}
__host__ __device__ inline int sym_pieces(const SymGeom& g, int b) {
    return sym_diag_pieces(g, b) + (sym_range(g, b) + g.unit_tiles - 1) / g.unit_tiles;
}
// first row of block b in the source-side workspace: rows of blocks b' < b, each (n_tiles - (b'+1) tb) * TILE long
__host__ __device__ inline size_t sym_joff(const SymGeom& g, int b) {
    if (g.mutual) return (size_t)b * g.n_tiles_b * TILE;
    return ((size_t)b * g.n_tiles - (size_t)g.tb * ((size_t)b * (b + 1) / 2)) * TILE;
}

struct SymArgs {
    double eps2, G;
    const int32_t* idx;     // the list (NULL: particles 0..m-1)
    const int32_t* idx_b;   // mutual mode: list B
    double* out;            // [.][3]
    double* pi;             // sink-side pieces   [piece][m][3]
    double* pj;             // source-side rows   [sym_joff(b) + j - (b+1) bs][3]
};

// ---- policies ---------------------------------------------------------------------------------------

struct SymAcc {
    static constexpr int REC = 4;            // x y z m
    struct Sink { double x, y, z, m; };
    struct Acc { double x, y, z; };
    __device__ __forceinline__ static void load_sink(const double* __restrict__ r, bool live, Sink& s) {
        s.x = r[0]; s.y = r[1]; s.z = r[2]; s.m = live ? r[3] : 0.0;
    }
    __device__ __forceinline__ static void init(Acc& c) { c.x = c.y = c.z = 0.0; }
    // s^-3 of one pair: 3 DADD, 3 DFMA, DMUL, DFMA, 2 DFMA, 2 DMUL = 12 FP64-pipe instructions
    __device__ __forceinline__ static double inv_s3(double eps2, const Sink& s, const double* __restrict__ r, double& dx,
                                                    double& dy, double& dz) {
        dx = r[0] - s.x; dy = r[1] - s.y; dz = r[2] - s.z;
        const double r2 = fma(dx, dx, fma(dy, dy, fma(dz, dz, eps2)));
        const double y0 = rsqrt_seed(r2);
        const double t = y0 * y0;
        const double e = fma(-r2, t, 1.0);
        const double p = fma(fma(e, 1.875, 1.5), e, 1.0);
        return (y0 * t) * p;
    }
    // diagonal tiles: ordered pairs, sink side only (15 instructions)
    __device__ __forceinline__ static void pair(const SymArgs& a, const Sink& s, Acc& c, const double* __restrict__ r) {
        double dx, dy, dz;
        const double w = inv_s3(a.eps2, s, r, dx, dy, dz) * r[3];
        c.x = fma(w, dx, c.x); c.y = fma(w, dy, c.y); c.z = fma(w, dz, c.z);
    }
    // S sinks of a thread against one source, both sides (20 instructions per pair); J[0..3) = the thread's
    // source-side sum  sum_s m_s s^-3 r_js  (the finish kernel subtracts it: the force on j points to i)
    template <int S>
    __device__ __forceinline__ static void pairs(const SymArgs& a, const Sink* sk, Acc* c, const double* __restrict__ r,
                                                 double* J) {
        double jx = 0.0, jy = 0.0, jz = 0.0;
#pragma unroll
        for (int s = 0; s < S; ++s) {
            double dx, dy, dz;
            const double s3 = inv_s3(a.eps2, sk[s], r, dx, dy, dz);
            const double wi = s3 * r[3], wj = s3 * sk[s].m;
            c[s].x = fma(wi, dx, c[s].x); jx = fma(wj, dx, jx);        // neighbours share an operand (reuse cache)
            jy = fma(wj, dy, jy); c[s].y = fma(wi, dy, c[s].y);
            c[s].z = fma(wi, dz, c[s].z); jz = fma(wj, dz, jz);
        }
        J[0] = jx; J[1] = jy; J[2] = jz;
    }
    __device__ __forceinline__ static void result(const Acc& c, double* o) { o[0] = c.x; o[1] = c.y; o[2] = c.z; }
};

struct SymGrad {
    static constexpr int REC = 8;            // x y z m ax ay az -
    struct Sink { double x, y, z, m, ax, ay, az; };
    struct Acc { double x, y, z; };
    __device__ __forceinline__ static void load_sink(const double* __restrict__ r, bool live, Sink& s) {
        s.x = r[0]; s.y = r[1]; s.z = r[2]; s.m = live ? r[3] : 0.0; s.ax = r[4]; s.ay = r[5]; s.az = r[6];
    }
    __device__ __forceinline__ static void init(Acc& c) { c.x = c.y = c.z = 0.0; }
    // One pair, mass-free (25 instructions): s3 = s^-3 and the bracket of Eq. 9 times s^3,
    //     t = a_ji - 3 (a_ji . r_ji) r_ji / s^2,
    // so that the sink's term is (m_j s3) t and the source's -(m_i s3) t: one weight and three accumulate DFMAs per
    // side (the plain kernel keeps two running sums U, W per sink instead, which is cheaper for ONE side only).
    __device__ __forceinline__ static void geom(double eps2, const Sink& s, const double* __restrict__ r, double& s3, double& tx,
                                                double& ty, double& tz) {
        const double dx = r[0] - s.x, dy = r[1] - s.y, dz = r[2] - s.z;
        const double bx = r[4] - s.ax, by = r[5] - s.ay, bz = r[6] - s.az;
        const double r2 = fma(dx, dx, fma(dy, dy, fma(dz, dz, eps2)));
        const double q = fma(bx, dx, fma(by, dy, bz * dz));
        const double y0 = rsqrt_seed(r2);
        const double t = y0 * y0;
        const double e = fma(-r2, t, 1.0);
        const double p = fma(fma(e, 1.875, 1.5), e, 1.0);
        s3 = (y0 * t) * p;
        const double tn = -3.0 * t;
        const double qq = q * fma(tn, fma(e, e, e), tn);      // -3 (a_ji . r_ji) / s^2
        tx = fma(qq, dx, bx); ty = fma(qq, dy, by); tz = fma(qq, dz, bz);
    }
    __device__ __forceinline__ static void pair(const SymArgs& a, const Sink& s, Acc& c, const double* __restrict__ r) {
        double s3, tx, ty, tz;
        geom(a.eps2, s, r, s3, tx, ty, tz);
        const double wi = s3 * r[3];
        c.x = fma(wi, tx, c.x); c.y = fma(wi, ty, c.y); c.z = fma(wi, tz, c.z);
    }
    // both sides: 33 instructions per pair
    template <int S>
    __device__ __forceinline__ static void pairs(const SymArgs& a, const Sink* sk, Acc* c, const double* __restrict__ r,
                                                 double* J) {
        double jx = 0.0, jy = 0.0, jz = 0.0;
#pragma unroll
        for (int s = 0; s < S; ++s) {
            double s3, tx, ty, tz;
            geom(a.eps2, sk[s], r, s3, tx, ty, tz);
            const double wi = s3 * r[3], wj = s3 * sk[s].m;
            c[s].x = fma(wi, tx, c[s].x); jx = fma(wj, tx, jx);
            jy = fma(wj, ty, jy); c[s].y = fma(wi, ty, c[s].y);
            c[s].z = fma(wi, tz, c[s].z); jz = fma(wj, tz, jz);
        }
        J[0] = jx; J[1] = jy; J[2] = jz;
    }
    __device__ __forceinline__ static void result(const Acc& c, double* o) { o[0] = c.x; o[1] = c.y; o[2] = c.z; }
};

// ---- pack: the list's records in list order, zero-padded to a whole number of tiles -------------------
template <class P>
__global__ void sym_pack_kernel(int m, int m_pad, const int32_t* __restrict__ idx, const double* __restrict__ pos,
                                const double* __restrict__ mass, const double* __restrict__ aux, double* __restrict__ rec) {
    const int l = blockIdx.x * blockDim.x + threadIdx.x;
    if (l >= m_pad) return;
    double2* o = reinterpret_cast<double2*>(rec + (size_t)l * P::REC);
    if (l >= m) {
#pragma unroll
        for (int q = 0; q < P::REC / 2; ++q) o[q] = make_double2(0.0, 0.0);
        return;
    }
    const size_t j = idx ? idx[l] : l;
    o[0] = make_double2(pos[3 * j], pos[3 * j + 1]);
    o[1] = make_double2(pos[3 * j + 2], mass[j]);
    if (P::REC == 8) {
        o[2] = make_double2(aux[3 * j], aux[3 * j + 1]);
        o[3] = make_double2(aux[3 * j + 2], 0.0);
    }
}

// Sum over the 32 lanes of a warp of 4 sources x 3 components held per lane (L[q][c]): two reduce-scatter steps
// (lane bit 0 keeps sources {0,1} or {2,3}, lane bit 1 one of the two) and a butterfly over lane bits 2-4.
// Afterwards every lane holds, in R[0..3), the warp's sum for source q = 2 (lane & 1) + ((lane >> 1) & 1).
// 18 DADD per 4 sources; the order of the additions is fixed by the lane numbers (a + b is commutative bit for
// bit, so all lanes of a residue class agree).
__device__ __forceinline__ void warp_sum_4x3(const double (*L)[3], int lane, double* R) {
    const bool b0 = lane & 1, b1 = lane & 2;
    double M[2][3];
#pragma unroll
    for (int q = 0; q < 2; ++q)
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const double keep = b0 ? L[q + 2][c] : L[q][c];
            const double send = b0 ? L[q][c] : L[q + 2][c];
            M[q][c] = keep + __shfl_xor_sync(0xffffffffu, send, 1);
        }
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const double keep = b1 ? M[1][c] : M[0][c];
        const double send = b1 ? M[0][c] : M[1][c];
        double v = keep + __shfl_xor_sync(0xffffffffu, send, 2);
        v += __shfl_xor_sync(0xffffffffu, v, 4);
        v += __shfl_xor_sync(0xffffffffu, v, 8);
        v += __shfl_xor_sync(0xffffffffu, v, 16);
        R[c] = v;
    }
}

// ---- the pair kernel: grid = (max pieces, blocks) ---------------------------------------------------
template <class P, int S, int T, int MINB, bool MUTUAL>
__global__ void __launch_bounds__(T, MINB)
sym_pair_kernel(const SymArgs a, const SymGeom g_in, const double* __restrict__ rec) {
    SymGeom g = g_in;
    g.mutual = MUTUAL;                              // compile-time in the geometry helpers below
    constexpr int REC = P::REC;
    constexpr int NW = T / 32;
    constexpr int CHUNKS = TILE * REC * 8 / 16;
    extern __shared__ __align__(16) double sym_sm[];
    double* tile_sm = sym_sm;                       // [2][TILE * REC]
    double* wbuf = sym_sm + 2 * TILE * REC;         // [NW][TILE][3] source-side sums per warp

    const int b = blockIdx.y, piece = blockIdx.x;
    const int range = sym_range(g, b), np = sym_pieces(g, b);
    if (piece >= np || (g.world > 1 && sym_owner(g, b) != g.rank)) return;
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;

    typename P::Sink sink[S];
    typename P::Acc accu[S];
    const int kbase = b * g.bs + threadIdx.x;
#pragma unroll
    for (int s = 0; s < S; ++s) {
        const int k = kbase + s * T;
        const bool live = k < g.m;                  // tail threads shadow the last list entry with mass 0
        P::load_sink(rec + (size_t)(live ? k : g.m - 1) * REC, live, sink[s]);
        P::init(accu[s]);
    }

    const double* __restrict__ src = rec + (size_t)(g.mutual ? g.rec_b : 0) * REC;
    auto load_tile = [&](int tile, int buf) {
        const double* gsrc = src + (size_t)tile * TILE * REC;
        double* dst = tile_sm + buf * TILE * REC;
        for (int ch = threadIdx.x; ch < CHUNKS; ch += T) cp_async16(dst + 2 * ch, gsrc + 2 * ch);
        cp_async_commit();
    };

    // this piece's tiles: an equal share of the diagonal [b tb, (b+1) tb) or of the tiles beyond the block
    const int jb = sym_first(g, b);
    const int nd = sym_diag_pieces(g, b), dt = sym_diag_tiles(g, b);
    const bool diag = piece < nd;
    const int len = diag ? (dt + nd - 1) / nd : (range + (np - nd) - 1) / (np - nd);
    const int t0 = diag ? b * g.tb + piece * len : jb + (piece - nd) * len;
    const int t1 = min(t0 + len, diag ? b * g.tb + dt : jb + range);
    const int n_my = max(t1 - t0, 0);
    auto tile_of = [&](int q) { return t0 + q; };

    if (n_my > 0) load_tile(tile_of(0), 0);
    for (int q = 0; q < n_my; ++q) {
        const int buf = q & 1;
        const int tile = tile_of(q);
        if (q + 1 < n_my) { load_tile(tile_of(q + 1), buf ^ 1); cp_async_wait<1>(); }
        else cp_async_wait<0>();
        __syncthreads();
        const double* __restrict__ tb = tile_sm + buf * TILE * REC;
        if (diag) {                                 // diagonal: ordered pairs, sink side only
            const int cnt = min(TILE, g.m - tile * TILE);
            for (int jj = 0; jj < cnt; ++jj) {
                double r[REC];
#pragma unroll
                for (int w = 0; w < REC; w += 2) {
                    const double2 v = *reinterpret_cast<const double2*>(tb + jj * REC + w);
                    r[w] = v.x; r[w + 1] = v.y;
                }
#pragma unroll
                for (int s = 0; s < S; ++s) P::pair(a, sink[s], accu[s], r);
            }
            __syncthreads();
            continue;
        }
        // beyond the block: every pair once, both sides (padding records have mass 0 and get a sum nobody reads)
        for (int j4 = 0; j4 < TILE; j4 += 4) {
            double L[4][3];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                double r[REC];
#pragma unroll
                for (int w = 0; w < REC; w += 2) {
                    const double2 v = *reinterpret_cast<const double2*>(tb + (j4 + u) * REC + w);
                    r[w] = v.x; r[w + 1] = v.y;
                }
                P::template pairs<S>(a, sink, accu, r, L[u]);
            }
            double R[3];
            warp_sum_4x3(L, lane, R);
            if (lane < 4) {
                double* o = wbuf + ((size_t)warp * TILE + j4 + 2 * (lane & 1) + (lane >> 1)) * 3;
                o[0] = R[0]; o[1] = R[1]; o[2] = R[2];
            }
        }
        __syncthreads();
        // the CTA's source-side sum of this tile: warps added in warp order, rows to the workspace
        {
            double* dst = a.pj + (sym_joff(g, b) + (size_t)(tile - jb) * TILE) * 3;
            for (int e = threadIdx.x; e < TILE * 3; e += T) {
                double v = wbuf[e];
#pragma unroll
                for (int w = 1; w < NW; ++w) v += wbuf[w * TILE * 3 + e];
                dst[e] = v;
            }
        }
        __syncthreads();
    }

    // sink-side piece
#pragma unroll
    for (int s = 0; s < S; ++s) {
        const int k = kbase + s * T;
        if (k < g.m) P::result(accu[s], a.pi + 3 * ((size_t)piece * g.m + k));
    }
}

// ---- finish: fixed-order sum of the sink-side pieces of the own block and the source-side rows of the earlier blocks
// (sharded: only of the blocks this rank owns - the result is then this rank's PARTIAL sum for every row, and the
// caller adds the ranks' outputs, one all-reduce)
__global__ void sym_finish_kernel(const SymArgs a, const SymGeom g) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= g.m + (g.mutual ? g.m_b : 0)) return;
    if (k >= g.m) {                                 // mutual mode, a row of list B: the source-side rows of ALL blocks
        const int j = k - g.m;
        double jx = 0.0, jy = 0.0, jz = 0.0;
        for (int bb = 0; bb < g.n_blocks; ++bb) {
            if (g.world > 1 && sym_owner(g, bb) != g.rank) continue;
            const double* q = a.pj + 3 * (sym_joff(g, bb) + (size_t)j);
            jx += __ldcg(q); jy += __ldcg(q + 1); jz += __ldcg(q + 2);
        }
        double* o = a.out + 3 * (size_t)(a.idx_b ? a.idx_b[j] : j);
        o[0] = -a.G * jx; o[1] = -a.G * jy; o[2] = -a.G * jz;
        return;
    }
    const int b = k / g.bs;
    const int np = (g.world > 1 && sym_owner(g, b) != g.rank) ? 0 : sym_pieces(g, b);
    double sx = 0.0, sy = 0.0, sz = 0.0;
    for (int p = 0; p < np; ++p) {
        const double* q = a.pi + 3 * ((size_t)p * g.m + k);
        sx += __ldcg(q); sy += __ldcg(q + 1); sz += __ldcg(q + 2);
    }
    double jx = 0.0, jy = 0.0, jz = 0.0;
    for (int bb = 0; bb < b && !g.mutual; ++bb) {
        if (g.world > 1 && sym_owner(g, bb) != g.rank) continue;
        const double* q = a.pj + 3 * (sym_joff(g, bb) + (size_t)(k - (bb + 1) * g.bs));
        jx += __ldcg(q); jy += __ldcg(q + 1); jz += __ldcg(q + 2);
    }
    const size_t row = g.compact ? (size_t)k : (size_t)(a.idx ? a.idx[k] : k);
    double* o = a.out + 3 * row;
    o[0] = a.G * (sx - jx); o[1] = a.G * (sy - jy); o[2] = a.G * (sz - jz);
}

}  // namespace
