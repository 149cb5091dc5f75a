// policies.cuh - the pass policies (acc, grad / jerk, dtmin, potential): packed source record, per-sink state, the pair update (the FP64 inner loop), store and split-j finish of each pass.
// Part of the single translation unit bifrost.cu (see its header and DESIGN.md); not a public header.
#pragma once

namespace {

// ----------------------------------------------------------------------------------------
// Pass policies.  Each defines the packed source record, the per-sink state, the pair update
// and how a thread's result is stored.
// ----------------------------------------------------------------------------------------

// NEXT-2: with EXCL = true every record carries the subsystem code of
// its source (-1 for a single particle) and every sink its own (-2 for a single particle, so that it
// never matches); a pair with equal codes gets the seed y0 = 0, hence the weight 0 - one integer
// compare and one 32-bit select per pair, nothing on the FP64 pipe.
__device__ __forceinline__ double mask_seed(double y0, bool same) {
    return __hiloint2double(same ? 0 : __double2hiint(y0), 0);
}
__device__ __forceinline__ int sink_code(const int32_t* subsys, int id) {
    const int c = subsys[id];
    return c < 0 ? -2 : c;
}

// source-side subsystem code: -1 for a single particle (never equal to a sink's code, which is
// -2 for a single particle), the subsystem id otherwise
__device__ __forceinline__ int src_code(const int32_t* subsys, int j) {
    if (!subsys) return -1;
    const int c = subsys[j];
    return c < 0 ? -1 : c;
}

// a5 + a7: reduction of one sink's partials in a FIXED order, then scatter.  A group of L lanes
// (L = 1, 2, .. 32, a power of two; lane = index in the group) shares one sink: lane l adds the
// partials of splits l, l+L, ... in that order and a butterfly adds the lanes - an order that
// depends only on (n_split, L), never on which CTA runs it.  All 32 lanes of a warp must call
// (write = false for a group that shadows a sink).  The partials come from other CTAs: L2 loads.
__device__ __forceinline__ double group_add(double v, int L) {
    for (int off = L >> 1; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
    return v;
}
__device__ __forceinline__ void finish_vec3(const double* partial, double* out, double G, const Geom& g, int k, int id,
                                            int lane, int L, bool write) {
    double sx = 0.0, sy = 0.0, sz = 0.0;
    for (int s = lane; s < g.n_split; s += L) {
        const double* p = partial + 3 * ((size_t)s * g.n_sink + k);
        sx += __ldcg(p); sy += __ldcg(p + 1); sz += __ldcg(p + 2);
    }
    if (L > 1) { sx = group_add(sx, L); sy = group_add(sy, L); sz = group_add(sz, L); }
    if (write && lane == 0) {
        double* o = out + 3 * (size_t)(g.compact ? k : id);
        o[0] = G * sx; o[1] = G * sy; o[2] = G * sz;
    }
}

struct AccArgs {
    const double* pos;
    const int32_t* subsys;
    const int32_t* sink_idx;
    double eps2, G;
    double* out;        // final output [.][3]
    double* partial;    // [split][n_sink][3]
};

template <bool EXCL>
struct AccPassT {
    using Short = AccPassT;
    static constexpr int REC = EXCL ? 8 : 6;   // x y z m 1.5m 1.875m [subsystem code (bits), pad]
    static constexpr bool PACK_EARLY = false;  // (see run_pass)
    static constexpr int PHASED_MIN_S = EXCL ? 2 : 0;
    using Args = AccArgs;
    struct Sink { double x, y, z; int sub; };
    struct Acc { double x, y, z; };
    struct Raw { double x, y, z, m; int code; };
    // a1: gather one source (j < 0: padding record) and write its packed record
    __device__ __forceinline__ static void fetch(const SrcArrays& s, int j, Raw& w) {
        if (j >= 0) {
            w.x = s.pos[3 * (size_t)j]; w.y = s.pos[3 * (size_t)j + 1]; w.z = s.pos[3 * (size_t)j + 2];
            w.m = s.mass[j]; w.code = EXCL ? src_code(s.subsys, j) : 0;
        } else { w.x = w.y = w.z = w.m = 0.0; w.code = 0; }
    }
    __device__ __forceinline__ static void emit(const Raw& w, double2* o) {
        o[0] = make_double2(w.x, w.y);
        o[1] = make_double2(w.z, w.m);
        o[2] = make_double2(1.5 * w.m, 1.875 * w.m);
        if (EXCL) o[3] = make_double2(__hiloint2double(0, w.code), 0.0);
    }
    __device__ static void load_sink(const Args& a, int id, Sink& s) {
        s.x = a.pos[3 * (size_t)id]; s.y = a.pos[3 * (size_t)id + 1]; s.z = a.pos[3 * (size_t)id + 2];
        s.sub = EXCL ? sink_code(a.subsys, id) : 0;
    }
    __device__ static void init(Acc& c) { c.x = c.y = c.z = 0.0; }
    // 15 FP64-pipe instructions: 3 DADD, 3 DFMA (r2), DMUL t, DFMA e, 2 DFMA poly, 2 DMUL, 3 DFMA.
    __device__ __forceinline__ static void pair(const Args& a, const Sink& s, Acc& c, const double* __restrict__ r) {
        const double dx = r[0] - s.x, dy = r[1] - s.y, dz = r[2] - s.z;
        const double r2 = fma(dx, dx, fma(dy, dy, fma(dz, dz, a.eps2)));
        double y0 = rsqrt_seed(r2);
        if (EXCL) y0 = mask_seed(y0, __double2loint(r[6]) == s.sub);
        const double t = y0 * y0;
        const double e = fma(-r2, t, 1.0);
        const double pm = fma(fma(e, r[5], r[4]), e, r[3]);   // m (1 + 3/2 e + 15/8 e^2)
        const double w = (y0 * t) * pm;                       // m / s^3
        c.x = fma(w, dx, c.x); c.y = fma(w, dy, c.y); c.z = fma(w, dz, c.z);
    }
    // EXCL only: the same 15 instructions per pair for the S sinks of a thread; a same-subsystem pair is rare, so its
    // weight is zeroed in a branch taken only when the source shares a subsystem with one of the thread's sinks,
    // instead of an integer compare and a select per pair (N = 2^20: 1063 -> 1042 ms; plain acc 995 ms).
    template <int S>
    __device__ __forceinline__ static void pairs(const Args& a, const Sink* sk, Acc* c, const double* __restrict__ r) {
        double dx[S], dy[S], dz[S], w[S];
        const int jcode = __double2loint(r[6]);
        bool any = false;
#pragma unroll
        for (int s = 0; s < S; ++s) {
            dx[s] = r[0] - sk[s].x; dy[s] = r[1] - sk[s].y; dz[s] = r[2] - sk[s].z;
            const double r2 = fma(dx[s], dx[s], fma(dy[s], dy[s], fma(dz[s], dz[s], a.eps2)));
            const double y0 = rsqrt_seed(r2);
            const double t = y0 * y0;
            const double e = fma(-r2, t, 1.0);
            const double pm = fma(fma(e, r[5], r[4]), e, r[3]);
            w[s] = (y0 * t) * pm;
            any |= jcode == sk[s].sub;
        }
        if (__builtin_expect(any, 0)) {
#pragma unroll
            for (int s = 0; s < S; ++s)
                if (jcode == sk[s].sub) w[s] = 0.0;
        }
#pragma unroll
        for (int s = 0; s < S; ++s) {
            c[s].x = fma(w[s], dx[s], c[s].x); c[s].y = fma(w[s], dy[s], c[s].y); c[s].z = fma(w[s], dz[s], c[s].z);
        }
    }
    __device__ static void store(const Args& a, const Geom& g, int split, int k, int id, const Sink&, const Acc& c) {
        if (g.n_split == 1) {
            double* o = a.out + 3 * (size_t)(g.compact ? k : id);
            o[0] = a.G * c.x; o[1] = a.G * c.y; o[2] = a.G * c.z;
        } else {
            double* o = a.partial + 3 * ((size_t)split * g.n_sink + k);
            o[0] = c.x; o[1] = c.y; o[2] = c.z;
        }
    }
    static constexpr bool ALWAYS_FINISH = false;
    // the split-j partial of a sink is three doubles that add: pair_fused_kernel may add the partials of the CTAs of a
    // thread-block cluster through distributed shared memory before anything goes to global memory
    static constexpr bool CLUSTER_REDUCE = true;
    static constexpr bool CLUSTER_MERGE = false;
    __device__ __forceinline__ static void vec3(const Acc& c, double* v) { v[0] = c.x; v[1] = c.y; v[2] = c.z; }
    __device__ static void finish(const Args& a, const Geom& g, int k, int id, int lane, int L, bool write) {
        finish_vec3(a.partial, a.out, a.G, g, k, id, lane, L, write);
    }
};

using AccPass = AccPassT<false>;

struct GradArgs {
    const double* pos;
    const double* acc;
    const int32_t* subsys;
    const int32_t* sink_idx;
    double eps2, G;
    double* out;
    double* partial;
    double* out2;        // WITH_ACC only: the acceleration sum (bifrost_acc_jerk)
    double* partial2;    // WITH_ACC only: its split-j partials
};

// WITH_ACC = true (bifrost_acc_jerk): the record holds v_j for a_j and the pair also accumulates
// Eq. 6's w * r_ji - acceleration and jerk in 31 FP64 instructions instead of 15 + 28.
template <bool EXCL, bool WITH_ACC = false>
struct GradPassT {
    using Short = GradPassT;
    static constexpr int REC = 10;  // x y z ax ay az m 1.5m 1.875m [subsystem code (bits)]
    static constexpr bool PACK_EARLY = true;
    static constexpr int PHASED_MIN_S = 5;   // measured: phase-major helps at S = 5 (+1.4 %), hurts at S = 4
    using Args = GradArgs;
    struct Sink { double x, y, z, ax, ay, az; int sub; };
    struct Acc { double ux, uy, uz, wx, wy, wz, ax, ay, az; };   // U = sum w a_ji,  W = sum w (a_ji.r_ji)/s^2 r_ji,  A = sum w r_ji
    struct Raw { double x, y, z, ax, ay, az, m; int code; };
    __device__ __forceinline__ static void fetch(const SrcArrays& s, int j, Raw& w) {
        if (j >= 0) {
            const size_t b = 3 * (size_t)j;
            w.x = s.pos[b]; w.y = s.pos[b + 1]; w.z = s.pos[b + 2];
            w.ax = s.aux[b]; w.ay = s.aux[b + 1]; w.az = s.aux[b + 2];
            w.m = s.mass[j]; w.code = src_code(s.subsys, j);
        } else { w.x = w.y = w.z = w.ax = w.ay = w.az = w.m = 0.0; w.code = 0; }
    }
    __device__ __forceinline__ static void emit(const Raw& w, double2* o) {
        o[0] = make_double2(w.x, w.y);
        o[1] = make_double2(w.z, w.ax);
        o[2] = make_double2(w.ay, w.az);
        o[3] = make_double2(w.m, 1.5 * w.m);
        o[4] = make_double2(1.875 * w.m, __hiloint2double(0, w.code));
    }
    __device__ static void load_sink(const Args& a, int id, Sink& s) {
        const size_t o = 3 * (size_t)id;
        s.x = a.pos[o]; s.y = a.pos[o + 1]; s.z = a.pos[o + 2];
        s.ax = a.acc[o]; s.ay = a.acc[o + 1]; s.az = a.acc[o + 2];
        s.sub = EXCL ? sink_code(a.subsys, id) : 0;
    }
    __device__ static void init(Acc& c) { c.ux = c.uy = c.uz = c.wx = c.wy = c.wz = c.ax = c.ay = c.az = 0.0; }
    // 28 FP64-pipe instructions; C_i = U - 3 W is formed once per sink in store().
    __device__ __forceinline__ static void pair(const Args& a, const Sink& s, Acc& c, const double* __restrict__ r) {
        const double dx = r[0] - s.x, dy = r[1] - s.y, dz = r[2] - s.z;
        const double bx = r[3] - s.ax, by = r[4] - s.ay, bz = r[5] - s.az;       // a_ji
        const double r2 = fma(dx, dx, fma(dy, dy, fma(dz, dz, a.eps2)));
        const double q = fma(bx, dx, fma(by, dy, bz * dz));                       // a_ji . r_ji
        double y0 = rsqrt_seed(r2);
        if (EXCL) y0 = mask_seed(y0, __double2loint(r[9]) == s.sub);
        const double t = y0 * y0;
        const double e = fma(-r2, t, 1.0);
        const double pm = fma(fma(e, r[8], r[7]), e, r[6]);
        const double w = (y0 * t) * pm;                                           // m / s^3
        const double y2 = fma(t, fma(e, e, e), t);                                // 1 / s^2
        const double v = (w * y2) * q;                                            // m (a_ji.r_ji) / s^5
        c.ux = fma(w, bx, c.ux); c.uy = fma(w, by, c.uy); c.uz = fma(w, bz, c.uz);
        if (WITH_ACC) { c.ax = fma(w, dx, c.ax); c.ay = fma(w, dy, c.ay); c.az = fma(w, dz, c.az); }
        c.wx = fma(v, dx, c.wx); c.wy = fma(v, dy, c.wy); c.wz = fma(v, dz, c.wz);
    }
    // the same 28 instructions per pair, stage by stage over the S sinks of a thread
    template <int S>
    __device__ __forceinline__ static void pairs(const Args& a, const Sink* sk, Acc* c, const double* __restrict__ r) {
        double dx[S], dy[S], dz[S], bx[S], by[S], bz[S], r2[S], q[S], y0[S], w[S], v[S];
#pragma unroll
        for (int s = 0; s < S; ++s) { dx[s] = r[0] - sk[s].x; dy[s] = r[1] - sk[s].y; dz[s] = r[2] - sk[s].z; }
#pragma unroll
        for (int s = 0; s < S; ++s) r2[s] = fma(dx[s], dx[s], fma(dy[s], dy[s], fma(dz[s], dz[s], a.eps2)));
#pragma unroll
        for (int s = 0; s < S; ++s) {
            y0[s] = rsqrt_seed(r2[s]);
            if (EXCL) y0[s] = mask_seed(y0[s], __double2loint(r[9]) == sk[s].sub);
        }
#pragma unroll
        for (int s = 0; s < S; ++s) { bx[s] = r[3] - sk[s].ax; by[s] = r[4] - sk[s].ay; bz[s] = r[5] - sk[s].az; }
#pragma unroll
        for (int s = 0; s < S; ++s) q[s] = fma(bx[s], dx[s], fma(by[s], dy[s], bz[s] * dz[s]));
#pragma unroll
        for (int s = 0; s < S; ++s) {
            const double t = y0[s] * y0[s];
            const double e = fma(-r2[s], t, 1.0);
            const double pm = fma(fma(e, r[8], r[7]), e, r[6]);
            w[s] = (y0[s] * t) * pm;
            const double y2 = fma(t, fma(e, e, e), t);
            v[s] = (w[s] * y2) * q[s];
        }
#pragma unroll
        for (int s = 0; s < S; ++s) {
            c[s].ux = fma(w[s], bx[s], c[s].ux); c[s].uy = fma(w[s], by[s], c[s].uy); c[s].uz = fma(w[s], bz[s], c[s].uz);
            if (WITH_ACC) { c[s].ax = fma(w[s], dx[s], c[s].ax); c[s].ay = fma(w[s], dy[s], c[s].ay); c[s].az = fma(w[s], dz[s], c[s].az); }
            c[s].wx = fma(v[s], dx[s], c[s].wx); c[s].wy = fma(v[s], dy[s], c[s].wy); c[s].wz = fma(v[s], dz[s], c[s].wz);
        }
    }
    __device__ static void store(const Args& a, const Geom& g, int split, int k, int id, const Sink&, const Acc& c) {
        const double cx = fma(-3.0, c.wx, c.ux), cy = fma(-3.0, c.wy, c.uy), cz = fma(-3.0, c.wz, c.uz);
        if (g.n_split == 1) {
            double* o = a.out + 3 * (size_t)(g.compact ? k : id);
            o[0] = a.G * cx; o[1] = a.G * cy; o[2] = a.G * cz;
        } else {
            double* o = a.partial + 3 * ((size_t)split * g.n_sink + k);
            o[0] = cx; o[1] = cy; o[2] = cz;
        }
        if (WITH_ACC) {
            if (g.n_split == 1) {
                double* o = a.out2 + 3 * (size_t)(g.compact ? k : id);
                o[0] = a.G * c.ax; o[1] = a.G * c.ay; o[2] = a.G * c.az;
            } else {
                double* o = a.partial2 + 3 * ((size_t)split * g.n_sink + k);
                o[0] = c.ax; o[1] = c.ay; o[2] = c.az;
            }
        }
    }
    static constexpr bool ALWAYS_FINISH = false;
    static constexpr bool CLUSTER_REDUCE = !WITH_ACC;       // (see AccPassT; the acc + jerk pass has two partials per sink)
    static constexpr bool CLUSTER_MERGE = false;
    __device__ __forceinline__ static void vec3(const Acc& c, double* v) {
        v[0] = fma(-3.0, c.wx, c.ux); v[1] = fma(-3.0, c.wy, c.uy); v[2] = fma(-3.0, c.wz, c.uz);     // as store()
    }
    __device__ static void finish(const Args& a, const Geom& g, int k, int id, int lane, int L, bool write) {
        finish_vec3(a.partial, a.out, a.G, g, k, id, lane, L, write);
        if (WITH_ACC) finish_vec3(a.partial2, a.out2, a.G, g, k, id, lane, L, write);
    }
};

using GradPass = GradPassT<false>;

// ----------------------------------------------------------------------------------------
// NEXT-3: neighbour search, §3.4, Eq. 18-19, and subsystem construction.
// A floating-point test decides an integer result here (is j a neighbour of i), so the decision is
// taken in plain IEEE fp64 operation by operation (no contraction, correctly rounded sqrt and
// division) in the order the paper states it: r_ij < r_ngb,max first, then the two-body a, e,
// then Eq. 18 (bound) or Eq. 19 (unbound).  Only a conservative distance pre-filter runs on the
// fast path (7 FP64 instructions per pair: the contracted r^2 against r_ngb,max^2 (1 + 1e-10)).
// ----------------------------------------------------------------------------------------
struct NgbArgs {
    const double* pos; const double* vel; const double* mass;
    const int32_t* sink_idx;
    double G, r_ngb, r_ngb_max, tau, C, r2_guard;
    int cap;
    int n_rows;                                 // n_sink (row stride of the per-split scratch)
    int32_t* out_count; int32_t* out_list;     // rows at sink ids (or sink positions when compact)
    int32_t* pcount; int32_t* plist;           // [split][n_sink], [split][n_sink][cap]
};

__device__ __noinline__ bool ngb_exact(const NgbArgs& a, double dx, double dy, double dz, double ux, double uy, double uz,
                                       double mi, double mj) {
    const double r2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
    const double r = sqrt(r2);
    if (!(r < a.r_ngb_max)) return false;
    const double v2 = __dadd_rn(__dadd_rn(__dmul_rn(ux, ux), __dmul_rn(uy, uy)), __dmul_rn(uz, uz));
    const double mu = __dmul_rn(a.G, __dadd_rn(mi, mj));
    const double E = __dsub_rn(__dmul_rn(0.5, v2), mu / r);             // two-body orbital energy per reduced mass
    if (E < 0.0) {                                                       // bound: Eq. 18
        const double sma = -mu / __dmul_rn(2.0, E);
        return (sma < a.r_ngb) || (r < a.r_ngb);
    }
    const double hx = __dsub_rn(__dmul_rn(dy, uz), __dmul_rn(dz, uy));   // h = r x v
    const double hy = __dsub_rn(__dmul_rn(dz, ux), __dmul_rn(dx, uz));
    const double hz = __dsub_rn(__dmul_rn(dx, uy), __dmul_rn(dy, ux));
    const double h2 = __dadd_rn(__dadd_rn(__dmul_rn(hx, hx), __dmul_rn(hy, hy)), __dmul_rn(hz, hz));
    double e2 = __dadd_rn(1.0, __dmul_rn(__dmul_rn(2.0, E), h2) / __dmul_rn(mu, mu));
    if (e2 < 0.0) e2 = 0.0;
    const double ecc = sqrt(e2);
    const double r_peri = (h2 / mu) / __dadd_rn(1.0, ecc);               // = a (1 - e), finite for E = 0
    if (!(r_peri < a.r_ngb)) return false;                               // Eq. 19
    if (r < a.r_ngb) return true;
    return __dmul_rn(a.C, r) / sqrt(v2) < a.tau;
}


struct DtArgs {
    const double* pos;
    const double* vel;
    const double* mass;
    const int32_t* subsys;
    const int32_t* sink_idx;
    const int32_t* src_idx;   // the source list (NULL: 0..n_src-1), for the exact rescan of an ambiguous sink (SHORT variant)
    int n_src;
    double* pkey;      // [split][2][n_sink]  refined key of the best source of a split (ff, fb)
    int32_t* pid;      // [split][2][n_sink]  its id
    double G, eta_ff, eta_fb;
    double* dt_ff; double* dt_fb; int32_t* j_ff; int32_t* j_fb;   // outputs (any may be NULL)
    NgbArgs ng;        // NGB only (bifrost_dtmin_neighbours): the neighbour search riding on the same pass
};

// Eq. 21 / Eq. 22 for ONE pair in plain IEEE operations (no contraction, correctly rounded sqrt and division),
// term by term in the oracle's order: the value a time-step is reported with, and the value near-ties are decided
// on.  Never on the hot path, so they stay out of line.
__device__ __noinline__ double dt_ff_exact(double dx, double dy, double dz, double G, double mi, double mj, double eta) {
    const double r2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
    const double r = sqrt(r2);
    return __dmul_rn(eta, sqrt(__dmul_rn(r2, r) / __dmul_rn(G, __dadd_rn(mi, mj))));
}
__device__ __noinline__ double dt_fb_exact(double dx, double dy, double dz, double ux, double uy, double uz, double eta) {
    const double r2 = __dadd_rn(__dadd_rn(__dmul_rn(dx, dx), __dmul_rn(dy, dy)), __dmul_rn(dz, dz));
    const double v2 = __dadd_rn(__dadd_rn(__dmul_rn(ux, ux), __dmul_rn(uy, uy)), __dmul_rn(uz, uz));
    if (v2 == 0.0) return __longlong_as_double(0x7ff0000000000000LL);    // reading T3
    return __dmul_rn(eta, sqrt(r2)) / sqrt(v2);
}
// exact time-step of sink i against source j, both read from the caller's arrays (w = 0: Eq. 21, w = 1: Eq. 22)
__device__ __noinline__ double dt_exact_ids(const DtArgs& a, int w, int i, int j) {
    const size_t oi = 3 * (size_t)i, oj = 3 * (size_t)j;
    const double dx = a.pos[oj] - a.pos[oi], dy = a.pos[oj + 1] - a.pos[oi + 1], dz = a.pos[oj + 2] - a.pos[oi + 2];
    if (w == 0) return dt_ff_exact(dx, dy, dz, a.G, a.mass[i], a.mass[j], a.eta_ff);
    return dt_fb_exact(dx, dy, dz, a.vel[oj] - a.vel[oi], a.vel[oj + 1] - a.vel[oi + 1], a.vel[oj + 2] - a.vel[oi + 2], a.eta_fb);
}
// near-tie between the running best jb and the contender jc of sink i: the oracle's rule on the exact values
// (smaller time-step; equal time-steps -> smaller particle id, reading T4)
__device__ __noinline__ bool dt_contender_wins(const DtArgs& a, int w, int i, int jb, int jc) {
    if (jb < 0) return true;
    const double tb = dt_exact_ids(a, w, i, jb), tc = dt_exact_ids(a, w, i, jc);
    return tc < tb || (tc == tb && jc < jb);
}

// The exact (time-step, id) minimum of sink i over the sources [l0, l1) of the list, straight from the oracle's
// definition: used only when a near-tie was seen for this sink in a short source range (DtPassT<.., SHORT>), i.e. for
// exactly tied inputs such as lattices.  w = 0: Eq. 21, w = 1: Eq. 22.  Returns the id (-1: none).
__device__ __noinline__ int dt_rescan(const DtArgs& a, int w, int i, int l0, int l1) {
    double tb = __longlong_as_double(0x7ff0000000000000LL);
    int jb = -1;
    const int ci = a.subsys ? a.subsys[i] : -1;
    for (int l = l0; l < l1; ++l) {
        const int j = a.src_idx ? a.src_idx[l] : l;
        if (j == i || (ci >= 0 && a.subsys[j] == ci)) continue;
        const double t = dt_exact_ids(a, w, i, j);
        if (t < tb || (t == tb && j < jb)) { tb = t; jb = j; }      // +inf (v_ij = 0) never replaces the initial +inf
    }
    return jb;
}

// The fast path MAXIMISES the monotone keys kff = (m_i+m_j)/r^3 (= eta^2/(G dt_ff^2)) and kfb = v^2/r^2
// (= eta^2/dt_fb^2): no sqrt or division per pair.  Three tiers:
//  (1) every pair: the keys from the UNREFINED reciprocal-square-root seed (relative error <= 3 x 2^-20 in y0^3; 17
//      FP64 instructions) against a threshold kept KEY_PRE = 1 - 1e-5 below the key of the running best - one integer
//      compare of the high words per key; this only SELECTS, so the seed's accuracy is enough;
//  (2) a selected pair (rare): the keys again with the polynomial refinement (a few ulp); a refined key decides only
//      when it is clear of the running best's by KEY_SLACK = 1e-12 relative;
//  (3) inside that band (a near-tie): the contender and the running best are both evaluated with dt_*_exact and the
//      oracle's rule decides.
// Every pair that could win passes (1) and (2): a winner's exact time-step is <= the best's, so its true key is >= the
// best's up to a few ulp.  The running best is thus always the exact (time-step, id) minimum of the sources seen,
// whatever the order of the source list, and the argmin is the oracle's bit for bit.
constexpr double KEY_SLACK = 1.0 - 1e-12;
constexpr double KEY_PRE = 1.0 - 1e-5;
constexpr double KEY_PRE_INV = 1.0 / KEY_PRE;

// NGB = true (bifrost_dtmin_neighbours, "along with the time-step assignment"): the pass also runs the
// neighbour search of Eq. 18-19 on the r^2 it already holds - one more integer pre-test per pair (r^2 below the
// guarded r_ngb,max^2), candidates through ngb_exact in the rare path, lists appended in source order.
// SHORT = true: the variant for short source ranges per CTA (a few tiles: small sink sets split many ways, the
// faster levels of the hierarchy).  There the running maxima still change every few sources, so the "rare" branch
// would be taken at almost every source (measured 3-4x slower than round 1's select variant).  This variant computes
// the REFINED keys for every pair (23 instructions) and updates the running best with selects when a key is clear of
// it by the band; only a key INSIDE the band - a near-tie, which is the truly rare event - takes a branch to the
// exact evaluation.  Same decisions, same results.
constexpr int DT_SHORT_TILES = 4;      // measured: from ~4 tiles per CTA on the three-tier variant is faster (config 2, 8192 sinks: 347 vs 388 us)

template <bool EXCL, bool NGB = false, bool SHORT = false>
struct DtPassT {
    using Short = DtPassT<EXCL, NGB, true>;
    static constexpr int REC = 8;   // x y z m vx vy vz {id (low word), subsystem code (high word)}
    static constexpr bool PACK_EARLY = true;
    static constexpr int PHASED_MIN_S = 1;
    using Args = DtArgs;
    struct Sink { double x, y, z, m, vx, vy, vz; int id, sub; };
    // thr = (refined key of the running best) * KEY_PRE; j = its source id (-1: none yet); nc = neighbours found (NGB)
    // (SHORT: thr = key of the running best * KEY_SLACK; amb = a near-tie was seen: bit 0 ff, bit 1 fb)
    struct Acc { double thr_ff, thr_fb; int jff, jfb, nc, amb; };
    struct Raw { double x, y, z, m, vx, vy, vz; int j, code; };
    __device__ __forceinline__ static void fetch(const SrcArrays& s, int j, Raw& w) {
        if (j >= 0) {
            const size_t b = 3 * (size_t)j;
            w.x = s.pos[b]; w.y = s.pos[b + 1]; w.z = s.pos[b + 2];
            w.vx = s.aux[b]; w.vy = s.aux[b + 1]; w.vz = s.aux[b + 2];
            w.m = s.mass[j]; w.j = j; w.code = src_code(s.subsys, j);
        } else { w.x = w.y = w.z = w.vx = w.vy = w.vz = w.m = 0.0; w.j = 0; w.code = 0; }
    }
    __device__ __forceinline__ static void emit(const Raw& w, double2* o) {
        o[0] = make_double2(w.x, w.y);
        o[1] = make_double2(w.z, w.m);
        o[2] = make_double2(w.vx, w.vy);
        o[3] = make_double2(w.vz, __hiloint2double(w.code, w.j));
    }
    __device__ static void load_sink(const Args& a, int id, Sink& s) {
        const size_t o = 3 * (size_t)id;
        s.x = a.pos[o]; s.y = a.pos[o + 1]; s.z = a.pos[o + 2];
        s.vx = a.vel[o]; s.vy = a.vel[o + 1]; s.vz = a.vel[o + 2];
        s.m = a.mass[id]; s.id = id;
        s.sub = EXCL ? sink_code(a.subsys, id) : 0;
    }
    __device__ static void init(Acc& c) { c.thr_ff = 0.0; c.thr_fb = 0.0; c.jff = -1; c.jfb = -1; c.nc = 0; c.amb = 0; }
    // one refined key of one sink against the running best (rare path, tiers 2 and 3)
    __device__ __forceinline__ static void contend(const Args& a, int w, int i, double key, int jid, double& thr, int& jbest) {
        const double K = thr * KEY_PRE_INV;               // the running best's key (to ~2 ulp)
        if (!(key >= K * KEY_SLACK)) return;
        if (key * KEY_SLACK > K || dt_contender_wins(a, w, i, jbest, jid)) { thr = key * KEY_PRE; jbest = jid; }
    }
    // tier 1: 7 DADD, 6 DFMA (r2, v2), DMUL y0^2, DMUL y0^3, 2 DMUL keys = 17 FP64-pipe instructions
    __device__ __forceinline__ static void keys_fast(const Sink& s, const double* __restrict__ r, double& kff, double& kfb, double& r2) {
        const double dx = r[0] - s.x, dy = r[1] - s.y, dz = r[2] - s.z;
        const double ux = r[4] - s.vx, uy = r[5] - s.vy, uz = r[6] - s.vz;
        r2 = fma(dx, dx, fma(dy, dy, fma(dz, dz, R2_FLOOR)));
        const double v2 = fma(ux, ux, fma(uy, uy, uz * uz));
        const double y0 = rsqrt_seed(r2);
        const double t = y0 * y0;
        kff = (s.m + r[3]) * (y0 * t);
        kfb = v2 * t;
    }
    __device__ __forceinline__ static double dist2(const Sink& s, const double* __restrict__ r) {
        const double dx = r[0] - s.x, dy = r[1] - s.y, dz = r[2] - s.z;
        return fma(dx, dx, fma(dy, dy, fma(dz, dz, R2_FLOOR)));
    }
    // tier 2: the same keys with the seed refined (e = 1 - r2 y0^2; y0^3 (1 + 3/2 e + 15/8 e^2), y0^2 (1 + e + e^2))
    __device__ __forceinline__ static void keys(const Sink& s, const double* __restrict__ r, double& kff, double& kfb) {
        const double dx = r[0] - s.x, dy = r[1] - s.y, dz = r[2] - s.z;
        const double ux = r[4] - s.vx, uy = r[5] - s.vy, uz = r[6] - s.vz;
        const double r2 = fma(dx, dx, fma(dy, dy, fma(dz, dz, R2_FLOOR)));
        const double v2 = fma(ux, ux, fma(uy, uy, uz * uz));
        const double y0 = rsqrt_seed(r2);
        const double t = y0 * y0;
        const double e = fma(-r2, t, 1.0);
        const double p3 = fma(fma(e, 1.875, 1.5), e, 1.0);
        kff = (s.m + r[3]) * ((y0 * t) * p3);
        kfb = v2 * fma(t, fma(e, e, e), t);
    }
    // The tier-1 keys of the S sinks of a thread and ONE branch per source that is almost never taken (after the first
    // sources a key comes near the running maximum ~1/j of the time for the j-th source).  The pre-test is a
    // necessary condition on the integer pipe: keys and thresholds are >= 0, so key >= thr implies
    // hi(key) >= hi(thr).  (The self pair and same-subsystem pairs are filtered in the rare path only.)
    template <int S>
    __device__ __forceinline__ static void pairs(const Args& a, const Sink* sk, Acc* c, const double* __restrict__ r) {
        if (SHORT) { pairs_short<S>(a, sk, c, r); return; }
        double kff[S], kfb[S], r2[S];
        bool any = false;
        const int guard_hi = NGB ? __double2hiint(a.ng.r2_guard) : 0;
#pragma unroll
        for (int s = 0; s < S; ++s) {
            keys_fast(sk[s], r, kff[s], kfb[s], r2[s]);
            any |= (__double2hiint(kff[s]) >= __double2hiint(c[s].thr_ff)) | (__double2hiint(kfb[s]) >= __double2hiint(c[s].thr_fb));
            // r^2 >= 0 and the guard >= 0, so r^2 < guard implies hi(r^2) <= hi(guard)
            if (NGB) any |= __double2hiint(r2[s]) <= guard_hi;
        }
        if (__builtin_expect(any, 0)) {
            const int jid = __double2loint(r[7]);
#pragma unroll
            for (int s = 0; s < S; ++s) {
                if (jid == sk[s].id) continue;
                if (NGB && r2[s] < a.ng.r2_guard) neighbour(a, sk[s], c[s], sink_row<S>(s), r, jid);     // ignores subsystems, as bifrost_neighbours
                if (EXCL && __double2hiint(r[7]) == sk[s].sub) continue;
                if (!((kff[s] >= c[s].thr_ff) | (kfb[s] >= c[s].thr_fb))) continue;
                double rff, rfb;
                Sink t = sk[s];         // opaque copy: keeps the compiler from holding tier 1's intermediates alive for tier 2
                asm volatile("" : "+d"(t.x), "+d"(t.y), "+d"(t.z), "+d"(t.vx), "+d"(t.vy), "+d"(t.vz));
                keys(t, r, rff, rfb);
                contend(a, 0, sk[s].id, rff, jid, c[s].thr_ff, c[s].jff);
                if (rfb > 0.0) contend(a, 1, sk[s].id, rfb, jid, c[s].thr_fb, c[s].jfb);   // v_ij = 0: dt_fb = +inf, never a minimum (T3)
            }
        }
    }
    // SHORT: refined keys for every pair; a key beyond the band above the running best replaces it by selects; a key
    // INSIDE the band (a near-tie) only sets a sticky flag - no branch in the loop, so the unrolled sources overlap (a
    // branch per source, even one never taken, serialised them: 22 us instead of 13 us for one sink) - and store() then
    // settles that sink by an exact rescan of the CTA's source range.  thr = K * KEY_SLACK, K = the running best's key.
    template <int S>
    __device__ __forceinline__ static void pairs_short(const Args& a, const Sink* sk, Acc* c, const double* __restrict__ r) {
        const int jid = __double2loint(r[7]);
        const int guard_hi = NGB ? __double2hiint(a.ng.r2_guard) : 0;
        bool cand = false;
        double kff[S], kfb[S];
#pragma unroll
        for (int s = 0; s < S; ++s) {
            keys(sk[s], r, kff[s], kfb[s]);
            bool other = jid != sk[s].id;
            if (NGB) cand |= other & (__double2hiint(dist2(sk[s], r)) <= guard_hi);
            if (EXCL) other &= __double2hiint(r[7]) != sk[s].sub;
            // ks KEY_SLACK > thr  <=>  key KEY_SLACK > K: beyond the band above the best.  key >= thr: inside or above it.
            const double ksf = kff[s] * KEY_SLACK, ksb = kfb[s] * KEY_SLACK;
            const bool wf = other & (ksf * KEY_SLACK > c[s].thr_ff), wb = other & (ksb * KEY_SLACK > c[s].thr_fb);
            const bool nf = other & !wf & (kff[s] >= c[s].thr_ff) & (jid != c[s].jff);
            const bool nb = other & !wb & (kfb[s] >= c[s].thr_fb) & (jid != c[s].jfb) & (__double2hiint(kfb[s]) != 0);   // v_ij = 0: never a minimum (T3)
            c[s].amb |= (nf ? 1 : 0) | (nb ? 2 : 0);
            c[s].thr_ff = wf ? ksf : c[s].thr_ff; c[s].jff = wf ? jid : c[s].jff;
            c[s].thr_fb = wb ? ksb : c[s].thr_fb; c[s].jfb = wb ? jid : c[s].jfb;
        }
        if (NGB && __builtin_expect(cand, 0)) {
#pragma unroll
            for (int s = 0; s < S; ++s)
                if (jid != sk[s].id && dist2(sk[s], r) < a.ng.r2_guard) neighbour(a, sk[s], c[s], sink_row<S>(s), r, jid);
        }
    }
    // row of the thread's s-th sink (the kernels lay sinks out as k = blockIdx.x * T * S + threadIdx.x + s * T)
    template <int S>
    __device__ __forceinline__ static int sink_row(int s) { return blockIdx.x * (blockDim.x * S) + threadIdx.x + s * blockDim.x; }
    // NGB: Eq. 18-19 for a candidate pair in plain IEEE operations; the id is appended to this split's list of the
    // sink.  Out of line with everything passed BY VALUE, so that the thread's sinks and running state stay in registers.
    __device__ __noinline__ static int neighbour_slow(const NgbArgs& ng, double dx, double dy, double dz, double ux, double uy,
                                                      double uz, double mi, double mj, int nc, int k, int jid) {
        if (!ngb_exact(ng, dx, dy, dz, ux, uy, uz, mi, mj)) return nc;
        if (k < ng.n_rows && nc < ng.cap) ng.plist[((size_t)blockIdx.y * ng.n_rows + k) * ng.cap + nc] = jid;
        return nc + 1;
    }
    __device__ __forceinline__ static void neighbour(const Args& a, const Sink& s, Acc& c, int k, const double* __restrict__ r, int jid) {
        c.nc = neighbour_slow(a.ng, r[0] - s.x, r[1] - s.y, r[2] - s.z, r[4] - s.vx, r[5] - s.vy, r[6] - s.vz, s.m, r[3], c.nc, k, jid);
    }
    // the split's winners: refined key of the running best (recovered from the threshold, ~2 ulp) and its id
    // refined keys of sink s against particle j read from the caller's arrays (rescan only)
    __device__ __noinline__ static void key_of(const Args& a, const Sink& s, int j, double& kff, double& kfb) {
        const size_t o = 3 * (size_t)j;
        const double r[8] = {a.pos[o], a.pos[o + 1], a.pos[o + 2], a.mass[j], a.vel[o], a.vel[o + 1], a.vel[o + 2], 0.0};
        keys(s, r, kff, kfb);
    }
    // the split's winners: refined keys of the running bests (recovered from the thresholds, ~2 ulp) and their ids
    __device__ __forceinline__ static void partial_of(const Args& a, const Geom& g, int split, int id, const Acc& c, double& kf, double& kb,
                                                      int& jf, int& jb) {
        constexpr double UNSCALE = SHORT ? 1.0 / KEY_SLACK : KEY_PRE_INV;
        kf = c.thr_ff * UNSCALE; kb = c.thr_fb * UNSCALE;
        jf = c.jff; jb = c.jfb;
        if (SHORT && __builtin_expect(c.amb != 0, 0)) {      // a near-tie in this range: settle it on the exact time-steps
            const int l0 = min(split * g.tiles_per_split * TILE, g.n_src), l1 = min(l0 + g.tiles_per_split * TILE, g.n_src);
            Sink t;
            load_sink(a, id, t);
            if (c.amb & 1) { jf = dt_rescan(a, 0, id, l0, l1); if (jf >= 0) { double d0, d1; key_of(a, t, jf, d0, d1); kf = d0; } }
            if (c.amb & 2) { jb = dt_rescan(a, 1, id, l0, l1); if (jb >= 0) { double d0, d1; key_of(a, t, jb, d0, d1); kb = d1; } }
        }
    }
    __device__ static void store(const Args& a, const Geom& g, int split, int k, int id, const Sink&, const Acc& c) {
        const size_t o = (size_t)split * 2 * g.n_sink + k;
        double kf, kb;
        int jf, jb;
        partial_of(a, g, split, id, c, kf, kb, jf, jb);
        a.pkey[o] = kf; a.pkey[o + g.n_sink] = kb;
        a.pid[o] = jf;  a.pid[o + g.n_sink] = jb;
        if (NGB) a.ng.pcount[(size_t)split * g.n_sink + k] = c.nc;
    }
    // dtmin epilogue: the winner over the splits by the same rule as inside a split - a key clear of the best by the band
    // decides, a near-tie is decided on the exact time-steps - then Eq. 21 / Eq. 22 for the winning pair in IEEE operations
    // in the oracle's order.  The winner is the exact (time-step, id) minimum, so the order of the splits does not matter.
    static constexpr bool ALWAYS_FINISH = true;
    static constexpr bool CLUSTER_REDUCE = false;
    // pair_fused_kernel as clusters: the winners of the CTAs of a cluster are merged through distributed shared memory with
    // merge() below, one entry per cluster goes to the workspace (not with the neighbour lists riding along)
    static constexpr bool CLUSTER_MERGE = !NGB;
    __device__ __forceinline__ static void vec3(const Acc&, double*) {}
    __device__ __forceinline__ static void merge(const Args& a, int i, int w, double key, int j, double& kb, int& jb) {
        const bool clear = (j >= 0) & ((key * KEY_SLACK > kb) | (jb < 0));
        const bool near = (j >= 0) & !clear & (key >= kb * KEY_SLACK) & (j != jb);
        if (__builtin_expect(near, 0)) {
            if (dt_contender_wins(a, w, i, jb, j)) { kb = key; jb = j; }
        } else {
            kb = clear ? key : kb; jb = clear ? j : jb;
        }
    }
    __device__ static void finish(const Args& a, const Geom& g, int k, int i, int lane, int L, bool write) {
        const double inf = __longlong_as_double(0x7ff0000000000000LL);
        double kb[2] = {0.0, 0.0};
        int jb[2] = {-1, -1};
        // four splits per trip, all 16 loads issued before the first compare (they come from other CTAs through L2: one
        // dependent round trip per split made this loop 0.5 us per split - 65 us for 128 sinks x 128 splits)
        for (int s0 = lane; s0 < g.n_split; s0 += 4 * L) {
            double t[4][2];
            int j[4][2];
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const int s = s0 + q * L;
                const bool in = s < g.n_split;
#pragma unroll
                for (int w = 0; w < 2; ++w) {
                    const size_t o = ((size_t)(in ? s : s0) * 2 + w) * g.n_sink + k;
                    t[q][w] = __ldcg(a.pkey + o);
                    j[q][w] = in ? __ldcg(a.pid + o) : -1;
                }
            }
#pragma unroll
            for (int q = 0; q < 4; ++q)
#pragma unroll
                for (int w = 0; w < 2; ++w) merge(a, i, w, t[q][w], j[q][w], kb[w], jb[w]);
        }
        for (int off = L >> 1; off > 0; off >>= 1) {
            for (int w = 0; w < 2; ++w) {
                const double key = __shfl_xor_sync(0xffffffffu, kb[w], off);
                const int j = __shfl_xor_sync(0xffffffffu, jb[w], off);
                merge(a, i, w, key, j, kb[w], jb[w]);
            }
        }
        if (!write || lane != 0) return;
        const int row = g.compact ? k : i;
        double tb[2];
        tb[0] = jb[0] >= 0 ? dt_exact_ids(a, 0, i, jb[0]) : inf;
        tb[1] = jb[1] >= 0 ? dt_exact_ids(a, 1, i, jb[1]) : inf;
        if (a.dt_ff) a.dt_ff[row] = jb[0] >= 0 ? tb[0] : inf;
        if (a.dt_fb) a.dt_fb[row] = jb[1] >= 0 ? tb[1] : inf;
        if (a.j_ff) a.j_ff[row] = jb[0];
        if (a.j_fb) a.j_fb[row] = jb[1];
        if (NGB) {      // the per-split lists in split order (= source-list order); the count is never truncated
            int total = 0;
            for (int s = 0; s < g.n_split; ++s) {
                const int cnt = __ldcg(a.ng.pcount + (size_t)s * g.n_sink + k);
                const int32_t* l = a.ng.plist + ((size_t)s * g.n_sink + k) * a.ng.cap;
                for (int q = 0; q < cnt && q < a.ng.cap && total + q < a.ng.cap; ++q)
                    a.ng.out_list[(size_t)row * a.ng.cap + total + q] = __ldcg(l + q);
                total += cnt;
            }
            a.ng.out_count[row] = total;
        }
    }
};

using DtPass = DtPassT<false>;

struct PotArgs {
    const double* pos;
    const int32_t* subsys;
    const int32_t* sink_idx;
    double eps2, G;
    double* out;        // phi at [.]
    double* partial;    // [split][n_sink]
};

// Potential (Eq. 4 second term, Eq. 68): p_i = sum_j m_j / s_ij; phi_i = -G p_i.
// 1/s = y0 (1 + e/2 + 3/8 e^2); the record carries m, m/2, 3m/8 and the source id, because here
// the self pair does not multiply a zero separation and must be dropped by id (integer select).
template <bool EXCL>
struct PotPassT {
    using Short = PotPassT;
    static constexpr int REC = 8;   // x y z m 0.5m 0.375m {id, subsystem code}(bits) pad
    static constexpr bool PACK_EARLY = false;
    static constexpr int PHASED_MIN_S = 2;
    using Args = PotArgs;
    struct Sink { double x, y, z; int id, sub; };
    struct Acc { double p; };
    struct Raw { double x, y, z, m; int j, code; };
    __device__ __forceinline__ static void fetch(const SrcArrays& s, int j, Raw& w) {
        if (j >= 0) {
            w.x = s.pos[3 * (size_t)j]; w.y = s.pos[3 * (size_t)j + 1]; w.z = s.pos[3 * (size_t)j + 2];
            w.m = s.mass[j]; w.j = j; w.code = src_code(s.subsys, j);
        } else { w.x = w.y = w.z = w.m = 0.0; w.j = -1; w.code = 0; }
    }
    __device__ __forceinline__ static void emit(const Raw& w, double2* o) {
        o[0] = make_double2(w.x, w.y);
        o[1] = make_double2(w.z, w.m);
        o[2] = make_double2(0.5 * w.m, 0.375 * w.m);
        o[3] = make_double2(__hiloint2double(w.code, w.j), 0.0);
    }
    __device__ static void load_sink(const Args& a, int id, Sink& s) {
        s.x = a.pos[3 * (size_t)id]; s.y = a.pos[3 * (size_t)id + 1]; s.z = a.pos[3 * (size_t)id + 2]; s.id = id;
        s.sub = EXCL ? sink_code(a.subsys, id) : 0;
    }
    __device__ static void init(Acc& c) { c.p = 0.0; }
    // 12 FP64-pipe instructions: 3 DADD, 3 DFMA, DMUL, DFMA, 2 DFMA, DMUL, DADD.
    __device__ __forceinline__ static void pair(const Args& a, const Sink& s, Acc& c, const double* __restrict__ r) {
        const double dx = r[0] - s.x, dy = r[1] - s.y, dz = r[2] - s.z;
        const double r2 = fma(dx, dx, fma(dy, dy, fma(dz, dz, a.eps2)));
        const double y0 = rsqrt_seed(r2);
        const double t = y0 * y0;
        const double e = fma(-r2, t, 1.0);
        const double pm = fma(fma(e, r[5], r[4]), e, r[3]);   // m (1 + 1/2 e + 3/8 e^2)
        double w = y0 * pm;                                   // m / s
        if (__double2loint(r[6]) == s.id) w = 0.0;            // j != i
        if (EXCL && __double2hiint(r[6]) == s.sub) w = 0.0;   // same subsystem
        c.p += w;
    }
    // the same sums for the S sinks of a thread; the self pair (and a same-subsystem pair) is zeroed in a branch
    // that is taken once per sink and source list, instead of two selects per pair
    template <int S>
    __device__ __forceinline__ static void pairs(const Args& a, const Sink* sk, Acc* c, const double* __restrict__ r) {
        double w[S];
        const int jid = __double2loint(r[6]), jcode = __double2hiint(r[6]);
        bool any = false;
#pragma unroll
        for (int s = 0; s < S; ++s) {
            const double dx = r[0] - sk[s].x, dy = r[1] - sk[s].y, dz = r[2] - sk[s].z;
            const double r2 = fma(dx, dx, fma(dy, dy, fma(dz, dz, a.eps2)));
            const double y0 = rsqrt_seed(r2);
            const double t = y0 * y0;
            const double e = fma(-r2, t, 1.0);
            const double pm = fma(fma(e, r[5], r[4]), e, r[3]);
            w[s] = y0 * pm;
            any |= (jid == sk[s].id) | (EXCL && jcode == sk[s].sub);
        }
        if (__builtin_expect(any, 0)) {
#pragma unroll
            for (int s = 0; s < S; ++s)
                if ((jid == sk[s].id) | (EXCL && jcode == sk[s].sub)) w[s] = 0.0;
        }
#pragma unroll
        for (int s = 0; s < S; ++s) c[s].p += w[s];
    }
    __device__ static void store(const Args& a, const Geom& g, int split, int k, int id, const Sink&, const Acc& c) {
        if (g.n_split == 1) a.out[g.compact ? k : id] = -a.G * c.p;
        else a.partial[(size_t)split * g.n_sink + k] = c.p;
    }
    static constexpr bool ALWAYS_FINISH = false;
    static constexpr bool CLUSTER_REDUCE = false;
    static constexpr bool CLUSTER_MERGE = false;
    __device__ __forceinline__ static void vec3(const Acc&, double*) {}
    __device__ static void finish(const Args& a, const Geom& g, int k, int id, int lane, int L, bool write) {
        double s = 0.0;
        for (int q = lane; q < g.n_split; q += L) s += __ldcg(a.partial + (size_t)q * g.n_sink + k);     // fixed order
        if (L > 1) s = group_add(s, L);
        if (write && lane == 0) a.out[g.compact ? k : id] = -a.G * s;
    }
};

using PotPass = PotPassT<false>;

}  // namespace
