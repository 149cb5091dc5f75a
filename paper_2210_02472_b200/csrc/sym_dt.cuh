// sym_dt.cuh - dtmin (Eq. 21 / Eq. 22) over ONE list that is both the sink and the source set, every
// unordered pair evaluated ONCE.  Part of the single translation unit bifrost.cu (see its header and DESIGN.md).
//
// Both keys are symmetric in (i, j): (m_i + m_j) / r^3 and v^2 / r^2.  So the 17 FP64 instructions of a pair's tier-1 keys
// (policies.cuh, DtPassT) can serve both members.  The SINK side is DtPassT's: thresholds in registers, one rarely taken
// branch per source.  The SOURCE side needs, for source j, the maximum over all sinks that meet it - spread over many CTAs.
// It is made just as rare: every list position has a global HINT, the largest refined key any pair has produced for it so
// far (bit pattern of a double >= 0, raised with atomicMax).  A pair whose key is clearly below the hint of its source cannot be
// that source's minimum and is dropped by one more integer compare per key; a pair that reaches the hint (inside or above the
// 1e-12 band) is a CANDIDATE: it is appended to a global list and raises the hint.  A stale hint only lets more candidates
// through, never fewer, so the result does not depend on the order in which CTAs run.  Hints start from the block diagonal
// (every particle against the 768 members of its own block - a short last block reaches back to a full block's worth -
// evaluated one-sided by a first launch), so that even the first
// off-diagonal CTAs see few candidates.  Afterwards: the sink-side pieces are merged per particle, the candidates are applied
// under a per-particle lock with the same band rule as everywhere else (clear key decides, near-tie -> exact time-steps, ties ->
// smaller id), and Eq. 21 / 22 are evaluated once for the winners.  The winner is the exact (time-step, id) minimum over all
// pairs: unique, hence bit-reproducible although the candidate order is not.
#pragma once

namespace {

struct DtBest { double kff, kfb; int jff, jfb; };                     // 24 B: refined keys and ids of the two bests
struct DtCand { double key; int pos2; int id; };                      // candidate for list position pos2 >> 1, kind pos2 & 1

struct SymDtArgs {
    DtArgs d;                          // arrays, G, eta, outputs (DtPassT's argument block)
    const int32_t* idx;                // the list (NULL: 0..m-1)
    DtBest* pieces;                    // sink-side pieces [piece][m]
    DtBest* best;                      // merged result per list position [m]
    unsigned long long* hint_ff;       // [m_pad] bit patterns of the largest refined key seen for a position
    unsigned long long* hint_fb;
    int* lock;                         // [m]
    DtCand* cand;                      // candidate list
    unsigned long long* counters;      // [0] candidates appended, [1] overflow flag
    unsigned long long cand_cap;
};

// The diagonal of a block for dtmin.  A short last block would take its first hints from its few members only, and its
// positions then collect hundreds of candidates each (m = 16384: 256 members, 400-500 candidates per position, all fighting
// for one lock per position: 3.2 ms instead of 1.0 ms per call).  Its diagonal pieces therefore reach back over a full
// block's worth of tiles; a pair seen twice cannot change a maximum.
__host__ __device__ inline bool sym_dt_short_last(const SymGeom& g, int b) { return b > 0 && sym_diag_tiles(g, b) < g.tb; }
__host__ __device__ inline int sym_dt_diag_tiles(const SymGeom& g, int b) { return sym_dt_short_last(g, b) ? g.tb : sym_diag_tiles(g, b); }
__host__ __device__ inline int sym_dt_diag_first(const SymGeom& g, int b) { return sym_dt_short_last(g, b) ? g.n_tiles - g.tb : b * g.tb; }
__host__ __device__ inline int sym_dt_diag_pieces(const SymGeom& g, int b) { return (sym_dt_diag_tiles(g, b) + g.unit_tiles - 1) / g.unit_tiles; }
__host__ __device__ inline int sym_dt_pieces(const SymGeom& g, int b) {
    return sym_dt_diag_pieces(g, b) + (sym_range(g, b) + g.unit_tiles - 1) / g.unit_tiles;
}

// phase = 0: the diagonal pieces only (one-sided; sets the hints);  phase = 1: the pieces beyond the block (both sides)
template <int S, int T, int MINB, int UNR = 2>
__global__ void __launch_bounds__(T, MINB)
sym_dt_kernel(const SymDtArgs a, const SymGeom g_in, const double* __restrict__ rec, int phase) {
    using D = DtPassT<false>;
    constexpr int REC = D::REC;
    constexpr int CHUNKS = TILE * REC * 8 / 16;
    __shared__ __align__(16) double tile_sm[2][TILE * REC];
    __shared__ int2 hint_hi[2][TILE];                  // high words of hint * KEY_PRE (ff, fb) of the tile's sources
    __shared__ double hint_val[2][TILE][2];            // the hints themselves
    SymGeom g = g_in;
    g.mutual = 0;
    const int b = blockIdx.y, piece = blockIdx.x;
    const int range = sym_range(g, b), np = sym_dt_pieces(g, b);
    const int nd = sym_dt_diag_pieces(g, b), dt = sym_dt_diag_tiles(g, b), dfirst = sym_dt_diag_first(g, b);
    if (piece >= np) return;
    const bool diag = piece < nd;
    if (diag != (phase == 0)) return;

    D::Sink sink[S];
    D::Acc accu[S];
    bool live[S];
    const int kbase = b * g.bs + threadIdx.x;
#pragma unroll
    for (int s = 0; s < S; ++s) {
        const int k = kbase + s * T;
        live[s] = k < g.m;
        const double* r = rec + (size_t)(live[s] ? k : g.m - 1) * REC;
        sink[s] = D::Sink{r[0], r[1], r[2], r[3], r[4], r[5], r[6], __double2loint(r[7]), 0};
        D::init(accu[s]);
        // beyond the diagonal the sink side starts from the position's hint as well: a pair clearly below the best key
        // already on record for this particle cannot be its minimum, in whichever piece it turns up (id -1 = "nothing in this
        // piece reaches the record").  Without it every piece restarts its running maxima and takes the branch at most
        // sources of a short piece.
        if (!diag && live[s]) {
            accu[s].thr_ff = __longlong_as_double((long long)__ldcg(a.hint_ff + k)) * KEY_PRE;
            accu[s].thr_fb = __longlong_as_double((long long)__ldcg(a.hint_fb + k)) * KEY_PRE;
        }
    }

    const int jb = sym_first(g, b);
    const int len = diag ? (dt + nd - 1) / nd : (range + (np - nd) - 1) / (np - nd);
    const int t0 = diag ? dfirst + piece * len : jb + (piece - nd) * len;
    const int t1 = min(t0 + len, diag ? dfirst + dt : jb + range);
    const int n_my = max(t1 - t0, 0);

    auto load_tile = [&](int tile, int buf) {
        const double* gsrc = rec + (size_t)tile * TILE * REC;
        for (int ch = threadIdx.x; ch < CHUNKS; ch += T) cp_async16(&tile_sm[buf][2 * ch], gsrc + 2 * ch);
        cp_async_commit();
    };
    auto load_hints = [&](int tile, int buf) {           // (phase 1 only) fresh values: other CTAs raise them while we run
        if (threadIdx.x < TILE) {
            const size_t p = (size_t)tile * TILE + threadIdx.x;
            const double hf = p < (size_t)g.m ? __longlong_as_double((long long)__ldcg(a.hint_ff + p)) : 0.0;
            const double hb = p < (size_t)g.m ? __longlong_as_double((long long)__ldcg(a.hint_fb + p)) : 0.0;
            hint_val[buf][threadIdx.x][0] = hf; hint_val[buf][threadIdx.x][1] = hb;
            hint_hi[buf][threadIdx.x] = make_int2(__double2hiint(hf * KEY_PRE), __double2hiint(hb * KEY_PRE));
        }
    };

    if (n_my > 0) { load_tile(t0, 0); if (!diag) load_hints(t0, 0); }
    for (int q = 0; q < n_my; ++q) {
        const int buf = q & 1, tile = t0 + q;
        if (q + 1 < n_my) { load_tile(tile + 1, buf ^ 1); if (!diag) load_hints(tile + 1, buf ^ 1); cp_async_wait<1>(); }
        else cp_async_wait<0>();
        __syncthreads();
        const double* __restrict__ tb = tile_sm[buf];
        const int cnt = min(TILE, g.m - tile * TILE);
#pragma unroll UNR
        for (int jj = 0; jj < cnt; ++jj) {
            double r[REC];
#pragma unroll
            for (int w = 0; w < REC; w += 2) {
                const double2 v = *reinterpret_cast<const double2*>(tb + jj * REC + w);
                r[w] = v.x; r[w + 1] = v.y;
            }
            const int2 hh = diag ? make_int2(0x7fffffff, 0x7fffffff) : hint_hi[buf][jj];
            double kff[S], kfb[S], r2;
            bool any = false;
#pragma unroll
            for (int s = 0; s < S; ++s) {
                D::keys_fast(sink[s], r, kff[s], kfb[s], r2);
                const int hf = __double2hiint(kff[s]), hb = __double2hiint(kfb[s]);
                any |= (hf >= __double2hiint(accu[s].thr_ff)) | (hb >= __double2hiint(accu[s].thr_fb)) | (hf >= hh.x) | (hb >= hh.y);
            }
            if (__builtin_expect(any, 0)) {
                const int jid = __double2loint(r[7]);
                const double hff = diag ? 0.0 : hint_val[buf][jj][0], hfb = diag ? 0.0 : hint_val[buf][jj][1];
#pragma unroll
                for (int s = 0; s < S; ++s) {
                    if (jid == sink[s].id) continue;
                    const bool si = (kff[s] >= accu[s].thr_ff) | (kfb[s] >= accu[s].thr_fb);
                    const bool sj = !diag & live[s] & ((kff[s] >= hff * KEY_PRE) | (kfb[s] >= hfb * KEY_PRE));
                    if (!(si | sj)) continue;
                    double rff, rfb;
                    D::Sink t = sink[s];
                    asm volatile("" : "+d"(t.x), "+d"(t.y), "+d"(t.z), "+d"(t.vx), "+d"(t.vy), "+d"(t.vz));
                    D::keys(t, r, rff, rfb);
                    if (si) {
                        D::contend(a.d, 0, sink[s].id, rff, jid, accu[s].thr_ff, accu[s].jff);
                        if (rfb > 0.0) D::contend(a.d, 1, sink[s].id, rfb, jid, accu[s].thr_fb, accu[s].jfb);
                    }
                    if (sj) {                                   // the pair as seen from the source: a candidate if it reaches the hint
                        const int pos = tile * TILE + jj;
                        if (rff >= hff * KEY_SLACK) {
                            const unsigned long long at = atomicAdd(a.counters, 1ULL);
                            if (at < a.cand_cap) a.cand[at] = DtCand{rff, 2 * pos, sink[s].id}; else a.counters[1] = 1ULL;
                            if (rff > hff) atomicMax(a.hint_ff + pos, (unsigned long long)__double_as_longlong(rff));
                        }
                        if (rfb > 0.0 && rfb >= hfb * KEY_SLACK) {
                            const unsigned long long at = atomicAdd(a.counters, 1ULL);
                            if (at < a.cand_cap) a.cand[at] = DtCand{rfb, 2 * pos + 1, sink[s].id}; else a.counters[1] = 1ULL;
                            if (rfb > hfb) atomicMax(a.hint_fb + pos, (unsigned long long)__double_as_longlong(rfb));
                        }
                    }
                }
            }
        }
        __syncthreads();
    }

#pragma unroll
    for (int s = 0; s < S; ++s) {
        const int k = kbase + s * T;
        if (!live[s]) continue;
        const DtBest o{accu[s].thr_ff * KEY_PRE_INV, accu[s].thr_fb * KEY_PRE_INV, accu[s].jff, accu[s].jfb};
        a.pieces[(size_t)piece * g.m + k] = o;
        if (!diag) {                                            // what this piece found raises the particle's hints
            if (accu[s].jff >= 0) atomicMax(a.hint_ff + k, (unsigned long long)__double_as_longlong(o.kff));
            if (accu[s].jfb >= 0) atomicMax(a.hint_fb + k, (unsigned long long)__double_as_longlong(o.kfb));
        }
    }
}

// the first hints: the largest key of a position over the diagonal pieces of its block
__global__ void sym_dt_hint_kernel(const SymDtArgs a, const SymGeom g) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= g.m) return;
    const int nd = sym_dt_diag_pieces(g, k / g.bs);
    double hf = 0.0, hb = 0.0;
    for (int p = 0; p < nd; ++p) {
        const DtBest o = a.pieces[(size_t)p * g.m + k];
        if (o.jff >= 0 && o.kff > hf) hf = o.kff;
        if (o.jfb >= 0 && o.kfb > hb) hb = o.kfb;
    }
    a.hint_ff[k] = (unsigned long long)__double_as_longlong(hf);
    a.hint_fb[k] = (unsigned long long)__double_as_longlong(hb);
}

// sink-side pieces of a list position -> best[k] (same band rule as DtPassT::finish)
__global__ void sym_dt_merge_kernel(const SymDtArgs a, const SymGeom g) {
    using D = DtPassT<false>;
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= g.m) return;
    const int i = a.idx ? a.idx[k] : k;
    const int np = sym_dt_pieces(g, k / g.bs);
    double kb[2] = {0.0, 0.0};
    int jb[2] = {-1, -1};
    for (int p = 0; p < np; ++p) {
        const DtBest o = a.pieces[(size_t)p * g.m + k];
        D::merge(a.d, i, 0, o.kff, o.jff, kb[0], jb[0]);
        D::merge(a.d, i, 1, o.kfb, o.jfb, kb[1], jb[1]);
    }
    a.best[k] = DtBest{kb[0], kb[1], jb[0], jb[1]};
    a.lock[k] = 0;
}

// Every candidate into best[] under the position's lock.  Candidates of one source found by the sinks of one CTA sit next to
// each other in the list, so the lanes of a warp would fight for one lock (a ragged last block, whose diagonal hints come from
// few members, collected 400-500 candidates per position: 2.2 ms instead of 0.15 ms for 16384 entries).  The lanes of a warp
// that hold the same (position, kind) elect a leader (__match_any_sync); it merges its group with the band rule first and
// takes the lock once.
__global__ void sym_dt_apply_kernel(const SymDtArgs a) {
    using D = DtPassT<false>;
    const unsigned long long n = min(a.counters[0], a.cand_cap);
    const int lane = threadIdx.x & 31;
    const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
    for (unsigned long long base = (unsigned long long)blockIdx.x * blockDim.x + (threadIdx.x & ~31); base < n; base += stride) {
        const unsigned long long c = base + lane;
        const bool valid = c < n;
        const DtCand cd = valid ? a.cand[c] : DtCand{0.0, -1 - lane, -1};
        const unsigned peers = __match_any_sync(0xffffffffu, cd.pos2);
        const bool leader = valid && lane == __ffs(peers) - 1;
        const int pos = cd.pos2 >> 1, w = cd.pos2 & 1;
        const int i = valid ? (a.idx ? a.idx[pos] : pos) : 0;
        double kg = cd.key;                     // the group's best, formed by its leader
        int jg = cd.id;
        if (__any_sync(0xffffffffu, (peers & (peers - 1)) != 0)) {      // some group of this warp has more than one lane: only where candidates cluster
            for (int src = 0; src < 32; ++src) {
                const double ks = __shfl_sync(0xffffffffu, cd.key, src);
                const int js = __shfl_sync(0xffffffffu, cd.id, src);
                if (leader && src != lane && ((peers >> src) & 1)) D::merge(a.d, i, w, ks, js, kg, jg);
            }
        }
        if (!leader) continue;
        bool done = false;
        while (!done) {
            if (atomicCAS(a.lock + pos, 0, 1) == 0) {
                __threadfence();
                DtBest* o = a.best + pos;
                double kb = w ? ((volatile DtBest*)o)->kfb : ((volatile DtBest*)o)->kff;
                int jb = w ? ((volatile DtBest*)o)->jfb : ((volatile DtBest*)o)->jff;
                D::merge(a.d, i, w, kg, jg, kb, jb);
                if (w) { ((volatile DtBest*)o)->kfb = kb; ((volatile DtBest*)o)->jfb = jb; }
                else { ((volatile DtBest*)o)->kff = kb; ((volatile DtBest*)o)->jff = jb; }
                __threadfence();
                atomicExch(a.lock + pos, 0);
                done = true;
            }
        }
    }
}

// Eq. 21 / Eq. 22 for the winners in IEEE operations, outputs at the particle's row.  If the candidate list overflowed
// (only an adversarial list order can do that) the position is settled by an exact rescan of all sources instead.
__global__ void sym_dt_final_kernel(const SymDtArgs a, const SymGeom g) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= g.m) return;
    const int i = a.idx ? a.idx[k] : k;
    int jf = a.best[k].jff, jb = a.best[k].jfb;
    if (a.counters[1]) { jf = dt_rescan(a.d, 0, i, 0, g.m); jb = dt_rescan(a.d, 1, i, 0, g.m); }
    const double inf = __longlong_as_double(0x7ff0000000000000LL);
    const int row = g.compact ? k : i;
    if (a.d.dt_ff) a.d.dt_ff[row] = jf >= 0 ? dt_exact_ids(a.d, 0, i, jf) : inf;
    if (a.d.dt_fb) a.d.dt_fb[row] = jb >= 0 ? dt_exact_ids(a.d, 1, i, jb) : inf;
    if (a.d.j_ff) a.d.j_ff[row] = jf;
    if (a.d.j_fb) a.d.j_fb[row] = jb;
}

}  // namespace
