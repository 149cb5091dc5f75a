// hhs_subtree.cuh - NEXT-4: a whole SUBTREE of the HHS-FSI recursion (Eq. 11-13) in one single-CTA launch.
// Part of the single translation unit bifrost.cu (see its header and DESIGN.md); not a public header.
//
// The deep levels of the time-step hierarchy hold a handful of particles and are visited 2^depth times per interval (the
// Fig. 8 cluster: 454 of the 517 levels of an interval have <= 128 particles).  Steered from the host each of them costs
// a dozen launches and one device -> host read.  Here a level of m <= SUB_M particles and everything below it runs in ONE
// launch of one CTA: one thread per particle of the current level, the subtree's particles in shared memory, the
// recursion as an explicit stack of frames, a barrier between the stages.  Arithmetic and summation order are those of
// the general path (AccPass / GradPass ::pair over the level's list in list order; kicks and drifts in the same IEEE
// operations; the same stable partitions of the order list), and the time-steps are the exact Eq. 21-22 minima, so the
// state after the interval and the level log are bit-identical to the host-steered path (tested).  With
// bifrost_set_level_criteria the level's own accelerations, jerks (acc_jerk's pair arithmetic) and gradient sums are formed at
// every level as well and Eq. 24-29 enter the level's time-steps in criteria_kernel's operations.
#pragma once

namespace {

constexpr int SUB_M = 128;           // largest level handled here (one source tile: the general path would not split it)
constexpr int SUB_STACK = 72;        // frames: max_depth <= 62

struct SubArgs {
    int m;                           // particles of the subtree's root level
    int32_t* seg;                    // the root level's segment of the order list (reordered in place, as the general path does)
    double* pos; double* vel; const double* mass;
    double* dt0;                     // per-particle level-0 time-step; written when depth0 == 0
    const double* dt_cap;            // optional further criteria at level 0 (reading H4)
    double G, eps2, eta_ff, eta_fb, tau;
    double crit_eta, crit_eta_grad, crit_eta_jerk;   // Eq. 24-29 at every level (bifrost_set_level_criteria); all 0: off
    int depth0, max_depth;
    long long* log;                  // device log [log_cap][3] of (depth, |S|, |F|), in the order the levels are entered
    long long log_cap;
    long long* counters;             // device: [0] levels entered (= next log row), [1] deepest depth, [2] FSI cycles
};

struct SubState {                    // shared memory; indexed by SLOT = position in the root level's list at entry
    double x[SUB_M], y[SUB_M], z[SUB_M], vx[SUB_M], vy[SUB_M], vz[SUB_M], ms[SUB_M], dt0[SUB_M];
    double ax[SUB_M], ay[SUB_M], az[SUB_M];         // inter-level accelerations (Eq. 12), rows of the current level
    double gx[SUB_M], gy[SUB_M], gz[SUB_M];         // inter-level gradient sums (Eq. 13)
    double jx[SUB_M], jy[SUB_M], jz[SUB_M];         // jerks of the level's particles (per-level criteria only)
    double rec[SUB_M * 10];                         // packed records of the current operation, by list position
    int id[SUB_M];                                  // particle id of a slot
    int ord[SUB_M];                                 // slot at list position k (the order list, local copy)
    int tmp[SUB_M];
    int warp_cnt[SUB_M / 32];
    int f_lo[SUB_STACK], f_hi[SUB_STACK], f_ns[SUB_STACK], f_stage[SUB_STACK];
    double f_tau[SUB_STACK];
};

// exact Eq. 21 / Eq. 22 minima of slot i over the level [lo, hi) (list order), the oracle's tie rule on particle ids
__device__ __noinline__ double sub_dtmin(const SubState& s, const SubArgs& a, int i, int lo, int hi) {
    using D = DtPassT<false>;
    D::Sink sk{s.x[i], s.y[i], s.z[i], s.ms[i], s.vx[i], s.vy[i], s.vz[i], s.id[i], 0};
    double kf = 0.0, kb = 0.0;       // refined keys of the running bests
    int jf = -1, jb = -1;            // their slots
    for (int p = lo; p < hi; ++p) {
        const int j = s.ord[p];
        if (j == i) continue;
        const double r[8] = {s.x[j], s.y[j], s.z[j], s.ms[j], s.vx[j], s.vy[j], s.vz[j], 0.0};
        double ff, fb;
        D::keys(sk, r, ff, fb);
        // a key clear of the best by the band decides; inside the band the exact time-steps and the id decide (reading T4)
        if (jf < 0 || ff * KEY_SLACK > kf) { kf = ff; jf = j; }
        else if (ff >= kf * KEY_SLACK) {
            const double tb = dt_ff_exact(s.x[jf] - sk.x, s.y[jf] - sk.y, s.z[jf] - sk.z, a.G, sk.m, s.ms[jf], a.eta_ff);
            const double tc = dt_ff_exact(r[0] - sk.x, r[1] - sk.y, r[2] - sk.z, a.G, sk.m, r[3], a.eta_ff);
            if (tc < tb || (tc == tb && s.id[j] < s.id[jf])) { kf = ff; jf = j; }
        }
        if (__double2hiint(fb) != 0) {                       // v_ij = 0: dt_fb = +inf, never a minimum (T3)
            if (jb < 0 || fb * KEY_SLACK > kb) { kb = fb; jb = j; }
            else if (fb >= kb * KEY_SLACK) {
                const double tb = dt_fb_exact(s.x[jb] - sk.x, s.y[jb] - sk.y, s.z[jb] - sk.z, s.vx[jb] - sk.vx, s.vy[jb] - sk.vy,
                                              s.vz[jb] - sk.vz, a.eta_fb);
                const double tc = dt_fb_exact(r[0] - sk.x, r[1] - sk.y, r[2] - sk.z, r[4] - sk.vx, r[5] - sk.vy, r[6] - sk.vz, a.eta_fb);
                if (tc < tb || (tc == tb && s.id[j] < s.id[jb])) { kb = fb; jb = j; }
            }
        }
    }
    const double inf = __longlong_as_double(0x7ff0000000000000LL);
    const double tff = jf < 0 ? inf : dt_ff_exact(s.x[jf] - sk.x, s.y[jf] - sk.y, s.z[jf] - sk.z, a.G, sk.m, s.ms[jf], a.eta_ff);
    const double tfb = jb < 0 ? inf : dt_fb_exact(s.x[jb] - sk.x, s.y[jb] - sk.y, s.z[jb] - sk.z, s.vx[jb] - sk.vx, s.vy[jb] - sk.vy,
                                                  s.vz[jb] - sk.vz, a.eta_fb);
    return fmin(tff, tfb);
}

__global__ void __launch_bounds__(SUB_M)
hhs_subtree_kernel(const SubArgs a) {
    using PA = AccPassT<false>;
    using PG = GradPassT<false>;
    using PJ = GradPassT<false, true>;      // acceleration + jerk in one pass (bifrost_acc_jerk's policy)
    __shared__ SubState s;
    const int t = threadIdx.x;
    const int lane = t & 31, warp = t >> 5;
    if (t < a.m) {
        const int id = a.seg[t];
        const size_t o = 3 * (size_t)id;
        s.id[t] = id; s.ord[t] = t;
        s.x[t] = a.pos[o]; s.y[t] = a.pos[o + 1]; s.z[t] = a.pos[o + 2];
        s.vx[t] = a.vel[o]; s.vy[t] = a.vel[o + 1]; s.vz[t] = a.vel[o + 2];
        s.ms[t] = a.mass[id];
        s.dt0[t] = a.dt0[id];
    }
    AccArgs aa{}; aa.eps2 = a.eps2;
    GradArgs ga{}; ga.eps2 = a.eps2;
    long long n_levels = 0, deepest = 0, fsi_steps = 0;      // kept by thread 0

    // ---- building blocks; every thread of the CTA calls them (barriers inside) ---------------------------------
    // accelerations of the positions [lo, hi) among themselves into (rx, ry, rz) of their slots (Eq. 6 over the set)
    auto acc_set = [&](int lo, int hi, double* rx, double* ry, double* rz) {
        const int m = hi - lo;
        __syncthreads();
        if (t < m) { const int i = s.ord[lo + t]; PA::Raw w{s.x[i], s.y[i], s.z[i], s.ms[i], 0}; PA::emit(w, reinterpret_cast<double2*>(s.rec + t * PA::REC)); }
        __syncthreads();
        if (t < m) {
            const int i = s.ord[lo + t];
            PA::Sink sk{s.x[i], s.y[i], s.z[i], 0};
            PA::Acc c; PA::init(c);
#pragma unroll 2
            for (int j = 0; j < m; ++j) {
                double r[PA::REC];
#pragma unroll
                for (int q = 0; q < PA::REC; ++q) r[q] = s.rec[j * PA::REC + q];
                PA::pair(aa, sk, c, r);
            }
            rx[i] = a.G * c.x; ry[i] = a.G * c.y; rz[i] = a.G * c.z;
        }
    };
    // Eq. 12: S = [lo, mid) against F = [mid, hi) and F against S, into s.ax/ay/az
    auto acc_inter = [&](int lo, int mid, int hi) {
        const int m = hi - lo;
        __syncthreads();
        if (t < m) { const int i = s.ord[lo + t]; PA::Raw w{s.x[i], s.y[i], s.z[i], s.ms[i], 0}; PA::emit(w, reinterpret_cast<double2*>(s.rec + t * PA::REC)); }
        __syncthreads();
        if (t < m) {
            const int i = s.ord[lo + t];
            const bool slow = lo + t < mid;
            const int j0 = slow ? mid - lo : 0, j1 = slow ? m : mid - lo;
            PA::Sink sk{s.x[i], s.y[i], s.z[i], 0};
            PA::Acc c; PA::init(c);
            for (int j = j0; j < j1; ++j) {
                double r[PA::REC];
#pragma unroll
                for (int q = 0; q < PA::REC; ++q) r[q] = s.rec[j * PA::REC + q];
                PA::pair(aa, sk, c, r);
            }
            s.ax[i] = a.G * c.x; s.ay[i] = a.G * c.y; s.az[i] = a.G * c.z;
        }
    };
    // Eq. 9 / Eq. 13 with the accelerations (qx, qy, qz): sinks [lo, hi) against sources [j0(t), j1(t)) of the same level
    auto grad_rows = [&](int lo, int mid, int hi, bool inter, const double* qx, const double* qy, const double* qz, double* rx,
                         double* ry, double* rz) {
        const int m = hi - lo;
        __syncthreads();
        if (t < m) {
            const int i = s.ord[lo + t];
            PG::Raw w{s.x[i], s.y[i], s.z[i], qx[i], qy[i], qz[i], s.ms[i], -1};
            PG::emit(w, reinterpret_cast<double2*>(s.rec + t * PG::REC));
        }
        __syncthreads();
        if (t < m) {
            const int i = s.ord[lo + t];
            const bool slow = lo + t < mid;
            const int j0 = inter ? (slow ? mid - lo : 0) : 0, j1 = inter ? (slow ? m : mid - lo) : m;
            PG::Sink sk{s.x[i], s.y[i], s.z[i], qx[i], qy[i], qz[i], 0};
            PG::Acc c; PG::init(c);
            for (int j = j0; j < j1; ++j) {
                double r[PG::REC];
#pragma unroll
                for (int q = 0; q < PG::REC; ++q) r[q] = s.rec[j * PG::REC + q];
                PG::pair(ga, sk, c, r);
            }
            rx[i] = a.G * fma(-3.0, c.wx, c.ux); ry[i] = a.G * fma(-3.0, c.wy, c.uy); rz[i] = a.G * fma(-3.0, c.wz, c.uz);
        }
    };
    // Eq. 6 and Eq. 28 of the positions [lo, hi) among themselves in one pass (acc_jerk_impl's arithmetic): accelerations into
    // (ax, ay, az), jerks into (jx, jy, jz) of their slots
    auto acc_jerk_set = [&](int lo, int hi) {
        const int m = hi - lo;
        __syncthreads();
        if (t < m) {
            const int i = s.ord[lo + t];
            PJ::Raw w{s.x[i], s.y[i], s.z[i], s.vx[i], s.vy[i], s.vz[i], s.ms[i], -1};
            PJ::emit(w, reinterpret_cast<double2*>(s.rec + t * PJ::REC));
        }
        __syncthreads();
        if (t < m) {
            const int i = s.ord[lo + t];
            PJ::Sink sk{s.x[i], s.y[i], s.z[i], s.vx[i], s.vy[i], s.vz[i], 0};
            PJ::Acc c; PJ::init(c);
            for (int j = 0; j < m; ++j) {
                double r[PJ::REC];
#pragma unroll
                for (int q = 0; q < PJ::REC; ++q) r[q] = s.rec[j * PJ::REC + q];
                PJ::pair(ga, sk, c, r);
            }
            s.jx[i] = a.G * fma(-3.0, c.wx, c.ux); s.jy[i] = a.G * fma(-3.0, c.wy, c.uy); s.jz[i] = a.G * fma(-3.0, c.wz, c.uz);
            s.ax[i] = a.G * c.ax; s.ay[i] = a.G * c.ay; s.az[i] = a.G * c.az;
        }
    };
    // v += h (acc + c grad) for the positions [lo, hi) (kick_kernel's operations)
    auto kick = [&](int lo, int hi, const double* qx, const double* qy, const double* qz, const double* hx, const double* hy,
                    const double* hz, double h, double cc) {
        __syncthreads();
        if (t < hi - lo) {
            const int i = s.ord[lo + t];
            double tx = qx[i], ty = qy[i], tz = qz[i];
            if (hx) { tx = __dadd_rn(tx, __dmul_rn(cc, hx[i])); ty = __dadd_rn(ty, __dmul_rn(cc, hy[i])); tz = __dadd_rn(tz, __dmul_rn(cc, hz[i])); }
            s.vx[i] = __dadd_rn(s.vx[i], __dmul_rn(h, tx)); s.vy[i] = __dadd_rn(s.vy[i], __dmul_rn(h, ty)); s.vz[i] = __dadd_rn(s.vz[i], __dmul_rn(h, tz));
        }
    };
    auto drift = [&](int lo, int hi, double h) {
        __syncthreads();
        if (t < hi - lo) {
            const int i = s.ord[lo + t];
            s.x[i] = __dadd_rn(s.x[i], __dmul_rn(h, s.vx[i])); s.y[i] = __dadd_rn(s.y[i], __dmul_rn(h, s.vy[i])); s.z[i] = __dadd_rn(s.z[i], __dmul_rn(h, s.vz[i]));
        }
    };
    // one FSI cycle (Eq. 10) over the positions [lo, hi) among themselves; scratch rows: (gx, gy, gz) hold the set's own
    // accelerations, tmp rows of rec are free again after each sum
    double* const bx = s.gx; double* const by = s.gy; double* const bz = s.gz;
    auto fsi = [&](int lo, int hi, double eps, double* cx, double* cy, double* cz) {
        if (hi <= lo) return;
        acc_set(lo, hi, bx, by, bz);
        kick(lo, hi, bx, by, bz, nullptr, nullptr, nullptr, eps / 6.0, 0.0);
        drift(lo, hi, eps / 2.0);
        acc_set(lo, hi, bx, by, bz);
        grad_rows(lo, hi, hi, false, bx, by, bz, cx, cy, cz);
        kick(lo, hi, bx, by, bz, cx, cy, cz, 2.0 * eps / 3.0, eps * eps / 24.0);
        drift(lo, hi, eps / 2.0);
        acc_set(lo, hi, bx, by, bz);
        kick(lo, hi, bx, by, bz, nullptr, nullptr, nullptr, eps / 6.0, 0.0);
        if (t == 0) ++fsi_steps;
    };

    // ---- the recursion (hhs_level of bifrost.cu, as a stack machine) ------------------------------------------------
    int sp = 0;
    if (t == 0) { s.f_lo[0] = 0; s.f_hi[0] = a.m; s.f_stage[0] = 0; s.f_tau[0] = a.tau; s.f_ns[0] = 0; }
    __syncthreads();
    while (sp >= 0) {
        const int lo = s.f_lo[sp], hi = s.f_hi[sp], stage = s.f_stage[sp];
        const double tau = s.f_tau[sp];
        const int depth = a.depth0 + sp;
        const int m = hi - lo;
        if (stage == 0) {
            // time-steps of the level's particles among themselves, slow / fast split (stable, S first)
            const bool all_slow = depth >= a.max_depth;
            const bool crit = a.crit_eta > 0.0 && !all_slow;
            if (crit) {     // Eq. 24-29 over the level's own particles: (ax..), (jx..), then C into (gx..)
                acc_jerk_set(lo, hi);
                grad_rows(lo, hi, hi, false, s.ax, s.ay, s.az, bx, by, bz);
                __syncthreads();
            }
            int fast = 0, slot = 0;
            if (t < m) {
                slot = s.ord[lo + t];
                if (!all_slow) {
                    double dt = sub_dtmin(s, a, slot, lo, hi);
                    if (crit) {     // criteria_kernel's operations
                        const double inf = __longlong_as_double(0x7ff0000000000000LL);
                        auto norm = [](double p0, double p1, double p2) {
                            return sqrt(__dadd_rn(__dadd_rn(__dmul_rn(p0, p0), __dmul_rn(p1, p1)), __dmul_rn(p2, p2)));
                        };
                        const double v = norm(s.vx[slot], s.vy[slot], s.vz[slot]), ac = norm(s.ax[slot], s.ay[slot], s.az[slot]);
                        const double gp = norm(bx[slot], by[slot], bz[slot]) / 24.0, jk = norm(s.jx[slot], s.jy[slot], s.jz[slot]);
                        dt = fmin(dt, (ac == 0.0) ? inf : __dmul_rn(a.crit_eta, v) / ac);
                        dt = fmin(dt, fmin((gp == 0.0) ? inf : a.crit_eta_grad * cbrt(v / gp), (gp == 0.0) ? inf : a.crit_eta_grad * sqrt(ac / gp)));
                        dt = fmin(dt, (jk == 0.0) ? inf : __dmul_rn(a.crit_eta_jerk, ac) / jk);
                    }
                    if (depth == 0) { if (a.dt_cap) dt = fmin(dt, a.dt_cap[s.id[slot]]); s.dt0[slot] = dt; }
                    dt = fmin(dt, s.dt0[slot]);
                    fast = dt < tau ? 1 : 0;
                }
            }
            const int slow = (t < m) && !fast;
            const unsigned bal = __ballot_sync(0xffffffffu, slow);
            if (lane == 0) s.warp_cnt[warp] = __popc(bal);
            __syncthreads();                                  // also: every ord[lo + t] has been read
            int before = 0, ns = 0;
            for (int w = 0; w < SUB_M / 32; ++w) { if (w < warp) before += s.warp_cnt[w]; ns += s.warp_cnt[w]; }
            const int rank_slow = before + __popc(bal & ((1u << lane) - 1u));
            if (t < m) s.ord[lo + (slow ? rank_slow : ns + (t - rank_slow))] = slot;
            const int nf = m - ns;
            if (t == 0) {
                const long long row = a.counters[0] + n_levels;
                if (row < a.log_cap) { a.log[3 * row] = depth; a.log[3 * row + 1] = ns; a.log[3 * row + 2] = nf; }
                ++n_levels;
                if (depth > deepest) deepest = depth;
                s.f_ns[sp] = ns;
            }
            __syncthreads();
            if (nf == 0) { fsi(lo, hi, tau, s.ax, s.ay, s.az); --sp; continue; }
            if (ns) {
                acc_inter(lo, lo + ns, hi);
                kick(lo, hi, s.ax, s.ay, s.az, nullptr, nullptr, nullptr, tau / 6.0, 0.0);
                fsi(lo, lo + ns, tau / 2.0, s.ax, s.ay, s.az);      // (its scratch rows are S's: the inter-level rows are dead by now)
            }
            __syncthreads();
            if (t == 0) {
                s.f_stage[sp] = 1;
                s.f_lo[sp + 1] = lo + ns; s.f_hi[sp + 1] = hi; s.f_stage[sp + 1] = 0; s.f_tau[sp + 1] = tau / 2.0;
            }
            __syncthreads();
            ++sp;
        } else if (stage == 1) {
            const int ns = s.f_ns[sp];
            if (ns) {
                acc_inter(lo, lo + ns, hi);
                // Eq. 13 needs its own output rows: the accelerations (ax..) are its input
                __syncthreads();
                grad_rows(lo, lo + ns, hi, true, s.ax, s.ay, s.az, bx, by, bz);
                kick(lo, hi, s.ax, s.ay, s.az, bx, by, bz, 2.0 * tau / 3.0, tau * tau / 24.0);
            }
            __syncthreads();
            if (t == 0) {
                s.f_stage[sp] = 2;
                s.f_lo[sp + 1] = lo + ns; s.f_hi[sp + 1] = hi; s.f_stage[sp + 1] = 0; s.f_tau[sp + 1] = tau / 2.0;
            }
            __syncthreads();
            ++sp;
        } else {
            const int ns = s.f_ns[sp];
            if (ns) {
                fsi(lo, lo + ns, tau / 2.0, s.ax, s.ay, s.az);
                acc_inter(lo, lo + ns, hi);
                kick(lo, hi, s.ax, s.ay, s.az, nullptr, nullptr, nullptr, tau / 6.0, 0.0);
            }
            __syncthreads();
            --sp;
        }
    }
    __syncthreads();
    if (t < a.m) {
        const int id = s.id[t];
        const size_t o = 3 * (size_t)id;
        a.pos[o] = s.x[t]; a.pos[o + 1] = s.y[t]; a.pos[o + 2] = s.z[t];
        a.vel[o] = s.vx[t]; a.vel[o + 1] = s.vy[t]; a.vel[o + 2] = s.vz[t];
        if (a.depth0 == 0) a.dt0[id] = s.dt0[t];
        a.seg[t] = s.id[s.ord[t]];
    }
    if (t == 0) {
        a.counters[0] += n_levels;
        if (deepest > a.counters[1]) a.counters[1] = deepest;
        a.counters[2] += fsi_steps;
    }
}

}  // namespace
