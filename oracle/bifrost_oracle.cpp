// bifrost_oracle.cpp - the parity ORACLE for the BIFROST direct-summation force path.
//
// TEST INFRASTRUCTURE ONLY.  A plain, slow, obviously-correct CPU implementation of
// what the hot path computes, written from the paper's definitions
// (/root/reference/PAPER.md, Rantala et al., BIFROST, arXiv:2210.02472).  Only
// tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
// legs may load it.  It shares no code, header, table or constant with the CUDA
// path (paper_2210_02472_b200/csrc); neither includes or imports the other.
//
// Every function is the paper's definition written out sink by sink with a
// straight `for j` loop over the source list in list order.  Arithmetic is plain
// IEEE binary64 (compile with -O2 -ffp-contract=off, no fast-math): IEEE sqrt and
// division, no blocking, no reordering.  Sums are accumulated with Neumaier's
// compensated summation so that the oracle's own rounding error (~2u per term,
// ~u in the sum) is well below the 1e-12 parity gate and it can arbitrate.
// OpenMP parallelises over sinks only, so results do not depend on thread count.
//
// Each routine is also instantiated in `long double` (x87 80-bit) - suffix _ld -
// which the CPU tests use to bound the binary64 instance's rounding error.
//
// Pins (tests/test_oracle_*.py, all `-m "not gpu"`): two-body closed forms, a
// hand-computed collinear three-body fixture (tests/golden/), sum_i m_i a_i = 0 and
// sum_i m_i G_i = 0, central finite difference of sum_k m_k |a_k|^2 for the gradient
// term (eps = 0 and eps ~ r), Plummer potential energy -3 pi G M^2/(32 a),
// independent numpy brute force for the time-step minima, exact lattice ties,
// and for pn1: label-swap symmetry, exact c -> 2c scaling, the test-particle
// limit, the centre-of-mass relative-acceleration identity and the periapsis
// advance of PAPER.md:L534 Eq. 46.
// jerk (NEXT-1): central finite difference in time of O-acc along r + v h, two-body closed
// form, sum_i m_i j_i = 0.  phi: two-body value, W = 1/2 sum m_i phi_i against O-pot and the
// Plummer value, -m_i a_i = finite difference of W.  criteria: hand-set vectors with integer
// norms (3-4-5 triangles) evaluated by hand from Eq. 24, 26, 27, 29.
// NEXT-2 (subsystem exclusion): all-(-1) ids reproduce the plain routines bit for bit; excluded +
// intra-subsystem partial sums (index lists) = full sums; one all-embracing subsystem gives 0 / +inf;
// numpy brute force with an explicit mask for dtmin; Eq. 20 against numpy minimum.reduceat.
// NEXT-3 (neighbour search, Eq. 18-19; components): circular / eccentric binaries and hyperbolic
// fly-bys built from chosen (a, e, true anomaly) so that every branch of Eq. 18-19 is hit with a known
// answer; Fig. 1's chain F-G (shared neighbour) for the components; numpy re-derivation of a, e from
// the vis-viva and Laplace-Runge-Lenz vector; brute-force union-find.
// Parity status: acc, grad, dtmin, potential, jerk, phi, criteria, pn1 pinned.  pn1: the paper prints
// no PN1.0 formula (PAPER.md:L439, L476 cite Thorne & Hartle 1985 / Einstein et al. 1938); reading P1
// takes the two-body EIH term.  Its relative dynamics are pinned by the test-particle
// limit, the centre-of-mass identity and the periapsis advance of Eq. 46; the split
// of the velocity terms between the two bodies, which those cannot see, is pinned in a BOOSTED
// frame: the 1PN total momentum and energy (Landau & Lifshitz §106) drift as c^-4 along an orbit
// integrated with acc + pn1, and as c^-2 for any other split (tests/test_oracle_dtmin_pn1.py).
//
// Conventions: r_ji = r_j - r_i, the force on
// sink i points towards source j; a source whose particle id equals the sink's id
// is skipped (Eq. 6, "j != i"); sink_idx / src_idx == NULL means "all
// n particles in id order"; outputs are compact, row k belongs to the k-th sink.

#include <cmath>
#include <cstdint>
#include <limits>
#include <vector>

namespace {

template <class T>
struct Neumaier {  // compensated running sum (Neumaier 1974)
    T s = 0, c = 0;
    inline void add(T x) {
        T t = s + x;
        if (std::fabs(s) >= std::fabs(x)) c += (s - t) + x;
        else                              c += (x - t) + s;
        s = t;
    }
    inline T value() const { return s + c; }
};

inline int64_t pid(const int32_t* idx, int64_t k) { return idx ? (int64_t)idx[k] : k; }

// NEXT-2, subsystem-aware sums.  PAPER.md:L233 Alg. 1 "Acceleration calculations ignore
// intra-subsystem contributions"; L299 §3.5.2 "the other particles j in the same subsystem are
// excluded from the time-step assignment"; L488 §3.8 (PN kicks exclude the same subsystem).
// subsys[k] >= 0 is the subsystem particle k belongs to, -1 marks a single particle; a NULL
// array means "no subsystems".  A pair (i, j) is dropped iff both carry the same id >= 0.
inline bool same_subsystem(const int32_t* subsys, int64_t i, int64_t j) {
    return subsys && subsys[i] >= 0 && subsys[i] == subsys[j];
}

// ---------------------------------------------------------------------------
// O-acc.  PAPER.md:L75 Eq. 6 (all pairs) and PAPER.md:L115-119 Eq. 12 (inter-level:
// the same sum restricted to a source set), with Plummer softening
// ("standard Plummer (1911) softening"; reading A2):
//     a_i = G sum_{j in src, j != i} m_j r_ji / (|r_ji|^2 + eps^2)^(3/2)
// ---------------------------------------------------------------------------
template <class T>
void acc_impl(int64_t n, const double* pos, const double* mass, const int32_t* sink_idx,
              int64_t n_sink, const int32_t* src_idx, int64_t n_src, double G, double eps,
              double* out, const int32_t* subsys = nullptr) {
    (void)n;
    const T eps2 = (T)eps * (T)eps;
#pragma omp parallel for schedule(dynamic, 8) if (n_sink * n_src > 16384)
    for (int64_t k = 0; k < n_sink; ++k) {
        const int64_t i = pid(sink_idx, k);
        const T xi = pos[3 * i], yi = pos[3 * i + 1], zi = pos[3 * i + 2];
        Neumaier<T> sx, sy, sz;
        for (int64_t l = 0; l < n_src; ++l) {
            const int64_t j = pid(src_idx, l);
            if (j == i || same_subsystem(subsys, i, j)) continue;
            const T dx = (T)pos[3 * j] - xi, dy = (T)pos[3 * j + 1] - yi, dz = (T)pos[3 * j + 2] - zi;
            const T s2 = dx * dx + dy * dy + dz * dz + eps2;
            const T w = (T)mass[j] / (s2 * std::sqrt(s2));
            sx.add(w * dx); sy.add(w * dy); sz.add(w * dz);
        }
        out[3 * k]     = (double)((T)G * sx.value());
        out[3 * k + 1] = (double)((T)G * sy.value());
        out[3 * k + 2] = (double)((T)G * sz.value());
    }
}

// ---------------------------------------------------------------------------
// O-grad.  The sum in PAPER.md:L90 Eq. 9 / L123-127 Eq. 13 without the step factor
// eps_step^2/24 (reading G3: the caller applies it; Eq. 23 relates
// the three normalisations: a~_i - a_i = eps^2/24 C_i, g_i = 2 C_i, g'_i = C_i/24):
//     C_i = G sum_{j != i} m_j [ a_ji / s^3 - 3 (a_ji . r_ji) r_ji / s^5 ],
//     a_ji = a_j - a_i,  s^2 = |r_ji|^2 + eps^2.
// For eps = 0 this is literally Eq. 9's G m_j/|r|^5 (|r|^2 a_ji - 3 (a_ji.r_ji) r_ji).
// Softened form (reading G1): the Jacobian of the softened pair acceleration
// d/dr [ r / (r^2+eps^2)^(3/2) ] = I/s^3 - 3 r r^T / s^5.
// acc[] holds a_k for every particle id that appears as sink or source (reading G2).
// ---------------------------------------------------------------------------
template <class T>
void grad_impl(int64_t n, const double* pos, const double* mass, const double* acc,
               const int32_t* sink_idx, int64_t n_sink, const int32_t* src_idx, int64_t n_src,
               double G, double eps, double* out, const int32_t* subsys = nullptr) {
    (void)n;
    const T eps2 = (T)eps * (T)eps;
#pragma omp parallel for schedule(dynamic, 8) if (n_sink * n_src > 16384)
    for (int64_t k = 0; k < n_sink; ++k) {
        const int64_t i = pid(sink_idx, k);
        const T xi = pos[3 * i], yi = pos[3 * i + 1], zi = pos[3 * i + 2];
        const T axi = acc[3 * i], ayi = acc[3 * i + 1], azi = acc[3 * i + 2];
        Neumaier<T> sx, sy, sz;
        for (int64_t l = 0; l < n_src; ++l) {
            const int64_t j = pid(src_idx, l);
            if (j == i || same_subsystem(subsys, i, j)) continue;
            const T dx = (T)pos[3 * j] - xi, dy = (T)pos[3 * j + 1] - yi, dz = (T)pos[3 * j + 2] - zi;
            const T dax = (T)acc[3 * j] - axi, day = (T)acc[3 * j + 1] - ayi, daz = (T)acc[3 * j + 2] - azi;
            const T s2 = dx * dx + dy * dy + dz * dz + eps2;
            const T q = dax * dx + day * dy + daz * dz;          // a_ji . r_ji
            const T inv3 = (T)1 / (s2 * std::sqrt(s2));
            const T inv5 = inv3 / s2;
            const T m = mass[j];
            const T c = (T)3 * q * inv5;
            sx.add(m * (inv3 * dax - c * dx));
            sy.add(m * (inv3 * day - c * dy));
            sz.add(m * (inv3 * daz - c * dz));
        }
        out[3 * k]     = (double)((T)G * sx.value());
        out[3 * k + 1] = (double)((T)G * sy.value());
        out[3 * k + 2] = (double)((T)G * sz.value());
    }
}

// ---------------------------------------------------------------------------
// O-dt.  PAPER.md:L312 Eq. 21 and L317 Eq. 22, unsoftened (reading T1):
//     dt_ff_i = eta_ff min_{j != i} sqrt( |r_ij|^3 / (G (m_i + m_j)) )
//     dt_fb_i = eta_fb min_{j != i} |r_ij| / |v_ij|        (+inf if v_ij = 0, reading T3)
// with the argmin source ids; ties -> smaller particle id (reading T4); empty
// source set -> +inf and id -1.  margin_* = (second smallest / smallest) - 1, so a
// disagreement in argmin with another implementation can be diagnosed.
// ---------------------------------------------------------------------------
void dtmin_impl(int64_t n, const double* pos, const double* vel, const double* mass,
                const int32_t* sink_idx, int64_t n_sink, const int32_t* src_idx, int64_t n_src,
                double G, double eta_ff, double eta_fb, double* dt_ff, double* dt_fb,
                int32_t* j_ff, int32_t* j_fb, double* margin_ff, double* margin_fb,
                const int32_t* subsys = nullptr) {
    (void)n;
    const double inf = std::numeric_limits<double>::infinity();
#pragma omp parallel for schedule(dynamic, 8) if (n_sink * n_src > 16384)
    for (int64_t k = 0; k < n_sink; ++k) {
        const int64_t i = pid(sink_idx, k);
        double bff = inf, bfb = inf, sff = inf, sfb = inf;   // best and second best
        int64_t iff = -1, ifb = -1;
        for (int64_t l = 0; l < n_src; ++l) {
            const int64_t j = pid(src_idx, l);
            if (j == i || same_subsystem(subsys, i, j)) continue;
            const double dx = pos[3 * j] - pos[3 * i], dy = pos[3 * j + 1] - pos[3 * i + 1],
                         dz = pos[3 * j + 2] - pos[3 * i + 2];
            const double r2 = dx * dx + dy * dy + dz * dz;
            const double r = std::sqrt(r2);
            const double tff = eta_ff * std::sqrt(r2 * r / (G * (mass[i] + mass[j])));
            const double dvx = vel[3 * j] - vel[3 * i], dvy = vel[3 * j + 1] - vel[3 * i + 1],
                         dvz = vel[3 * j + 2] - vel[3 * i + 2];
            const double v2 = dvx * dvx + dvy * dvy + dvz * dvz;
            const double tfb = (v2 == 0.0) ? inf : eta_fb * r / std::sqrt(v2);
            if (tff < bff || (tff == bff && j < iff)) { sff = bff; bff = tff; iff = j; }
            else if (tff < sff) sff = tff;
            if (tfb < bfb || (tfb == bfb && j < ifb)) { sfb = bfb; bfb = tfb; ifb = j; }
            else if (tfb < sfb) sfb = tfb;
        }
        dt_ff[k] = bff; dt_fb[k] = bfb;
        j_ff[k] = (int32_t)iff; j_fb[k] = (int32_t)ifb;
        if (margin_ff) margin_ff[k] = sff / bff - 1.0;
        if (margin_fb) margin_fb[k] = sfb / bfb - 1.0;
    }
}

// ---------------------------------------------------------------------------
// O-pn1.  PAPER.md:L476-488 §3.8, Eq. 42-43: the global PN1.0 term, "applying the PN
// accelerations only for pairwise interactions when either of the particles is
// massive enough".  The paper does not print the PN1.0 pair formula (it cites
// Thorne & Hartle 1985 / Einstein et al. 1938); reading P1 takes the
// standard two-body 1PN (EIH) acceleration in harmonic coordinates, general frame.
// For sink i and source j, with r = |r_i - r_j|, n = (r_i - r_j)/r:
//   f(i<-j) = G m_j/(c^2 r^2) { n [ 5 G m_i/r + 4 G m_j/r + 3/2 (n.v_j)^2
//                                   - v_i.v_i + 4 v_i.v_j - 2 v_j.v_j ]
//                               + (4 n.v_i - 3 n.v_j)(v_i - v_j) }
// (only the 1/c^2 part; the Newtonian part belongs to a_i).  Unsoftened (P3).
// Pair selection (reading P2): every ordered pair (i, j), i != j, with i in the BH
// list or j in the BH list, each once.  out[n][3] is fully overwritten.
// ---------------------------------------------------------------------------
template <class T>
inline void pn1_pair(const double* pos, const double* vel, const double* mass, int64_t i, int64_t j,
                     T G, T c2inv, Neumaier<T>& sx, Neumaier<T>& sy, Neumaier<T>& sz) {
    const T rx = (T)pos[3 * i] - (T)pos[3 * j], ry = (T)pos[3 * i + 1] - (T)pos[3 * j + 1],
            rz = (T)pos[3 * i + 2] - (T)pos[3 * j + 2];
    const T r2 = rx * rx + ry * ry + rz * rz;
    const T r = std::sqrt(r2);
    const T nx = rx / r, ny = ry / r, nz = rz / r;
    const T vix = vel[3 * i], viy = vel[3 * i + 1], viz = vel[3 * i + 2];
    const T vjx = vel[3 * j], vjy = vel[3 * j + 1], vjz = vel[3 * j + 2];
    const T nvi = nx * vix + ny * viy + nz * viz;
    const T nvj = nx * vjx + ny * vjy + nz * vjz;
    const T vivi = vix * vix + viy * viy + viz * viz;
    const T vjvj = vjx * vjx + vjy * vjy + vjz * vjz;
    const T vivj = vix * vjx + viy * vjy + viz * vjz;
    const T mi = mass[i], mj = mass[j];
    const T A = (T)5 * G * mi / r + (T)4 * G * mj / r + (T)1.5 * nvj * nvj - vivi + (T)4 * vivj - (T)2 * vjvj;
    const T B = (T)4 * nvi - (T)3 * nvj;
    const T pref = G * mj * c2inv / r2;
    sx.add(pref * (nx * A + B * (vix - vjx)));
    sy.add(pref * (ny * A + B * (viy - vjy)));
    sz.add(pref * (nz * A + B * (viz - vjz)));
}

template <class T>
void pn1_impl(int64_t n, const double* pos, const double* vel, const double* mass,
              const int32_t* bh_idx, int64_t n_bh, double G, double c, double* out,
              const int32_t* subsys = nullptr) {
    std::vector<char> is_bh((size_t)n, 0);
    for (int64_t b = 0; b < n_bh; ++b) is_bh[(size_t)bh_idx[b]] = 1;
    const T c2inv = (T)1 / ((T)c * (T)c);
#pragma omp parallel for schedule(dynamic, 64) if (n * n_bh > 8192)
    for (int64_t i = 0; i < n; ++i) {
        Neumaier<T> sx, sy, sz;
        if (is_bh[(size_t)i]) {
            for (int64_t j = 0; j < n; ++j)
                if (j != i && !same_subsystem(subsys, i, j)) pn1_pair<T>(pos, vel, mass, i, j, (T)G, c2inv, sx, sy, sz);
        } else {
            for (int64_t b = 0; b < n_bh; ++b)
                if (!same_subsystem(subsys, i, (int64_t)bh_idx[b]))
                    pn1_pair<T>(pos, vel, mass, i, (int64_t)bh_idx[b], (T)G, c2inv, sx, sy, sz);
        }
        out[3 * i] = (double)sx.value(); out[3 * i + 1] = (double)sy.value(); out[3 * i + 2] = (double)sz.value();
    }
}

// ---------------------------------------------------------------------------
// O-jerk.  PAPER.md:L360 Eq. 28 (reading J1: the garbled lhs is j_i = da_i/dt, the
// sum runs over j != i), softened like the accelerations (exact time derivative
// of the softened pair acceleration along r_ji(t), dr_ji/dt = v_ji):
//     j_i = G sum_{j in src, j != i} m_j [ v_ji / s^3 - 3 (r_ji . v_ji) r_ji / s^5 ],
//     v_ji = v_j - v_i,  s^2 = |r_ji|^2 + eps^2.
// For eps = 0 this is literally Eq. 28's G m_j/|r|^5 (|r|^2 v_ji - 3 (r_ji.v_ji) r_ji).
// ---------------------------------------------------------------------------
template <class T>
void jerk_impl(int64_t n, const double* pos, const double* vel, const double* mass,
               const int32_t* sink_idx, int64_t n_sink, const int32_t* src_idx, int64_t n_src,
               double G, double eps, double* out, const int32_t* subsys = nullptr) {
    (void)n;
    const T eps2 = (T)eps * (T)eps;
#pragma omp parallel for schedule(dynamic, 8) if (n_sink * n_src > 16384)
    for (int64_t k = 0; k < n_sink; ++k) {
        const int64_t i = pid(sink_idx, k);
        Neumaier<T> sx, sy, sz;
        for (int64_t l = 0; l < n_src; ++l) {
            const int64_t j = pid(src_idx, l);
            if (j == i || same_subsystem(subsys, i, j)) continue;
            const T dx = (T)pos[3 * j] - (T)pos[3 * i], dy = (T)pos[3 * j + 1] - (T)pos[3 * i + 1],
                    dz = (T)pos[3 * j + 2] - (T)pos[3 * i + 2];
            const T ux = (T)vel[3 * j] - (T)vel[3 * i], uy = (T)vel[3 * j + 1] - (T)vel[3 * i + 1],
                    uz = (T)vel[3 * j + 2] - (T)vel[3 * i + 2];
            const T s2 = dx * dx + dy * dy + dz * dz + eps2;
            const T s = std::sqrt(s2);
            const T s3 = s2 * s, s5 = s3 * s2;
            const T rv = dx * ux + dy * uy + dz * uz;       // r_ji . v_ji
            const T m = mass[j];
            sx.add(m * (ux / s3 - (T)3 * rv * dx / s5));
            sy.add(m * (uy / s3 - (T)3 * rv * dy / s5));
            sz.add(m * (uz / s3 - (T)3 * rv * dz / s5));
        }
        out[3 * k]     = (double)((T)G * sx.value());
        out[3 * k + 1] = (double)((T)G * sy.value());
        out[3 * k + 2] = (double)((T)G * sz.value());
    }
}

// ---------------------------------------------------------------------------
// O-phi.  Per-sink potential of PAPER.md:L63 Eq. 4 (second term) / L724 Eq. 68, softened
// like the accelerations:  phi_i = -G sum_{j in src, j != i} m_j / sqrt(|r_ji|^2 + eps^2),
// so that W = 1/2 sum_i m_i phi_i when sinks = sources = all.
// ---------------------------------------------------------------------------
template <class T>
void phi_impl(int64_t n, const double* pos, const double* mass, const int32_t* sink_idx, int64_t n_sink,
              const int32_t* src_idx, int64_t n_src, double G, double eps, double* out,
              const int32_t* subsys = nullptr) {
    (void)n;
    const T eps2 = (T)eps * (T)eps;
#pragma omp parallel for schedule(dynamic, 8) if (n_sink * n_src > 16384)
    for (int64_t k = 0; k < n_sink; ++k) {
        const int64_t i = pid(sink_idx, k);
        Neumaier<T> s;
        for (int64_t l = 0; l < n_src; ++l) {
            const int64_t j = pid(src_idx, l);
            if (j == i || same_subsystem(subsys, i, j)) continue;
            const T dx = (T)pos[3 * j] - (T)pos[3 * i], dy = (T)pos[3 * j + 1] - (T)pos[3 * i + 1],
                    dz = (T)pos[3 * j + 2] - (T)pos[3 * i + 2];
            s.add((T)mass[j] / std::sqrt(dx * dx + dy * dy + dz * dz + eps2));
        }
        out[k] = (double)(-(T)G * s.value());
    }
}

// ---------------------------------------------------------------------------
// O-crit.  The O(N) per-particle time-step criteria of PAPER.md §3.5.4-3.5.5:
//     dt_va    = eta      |v_i| / |a_i|                 (L338 Eq. 24)
//     dt_gradv = eta_grad (|v_i| / |g'_i|)^(1/3)        (L346 Eq. 26)
//     dt_grada = eta_grad (|a_i| / |g'_i|)^(1/2)        (L350 Eq. 27)
//     dt_jerk  = eta_jerk |a_i| / |j_i|                 (L365 Eq. 29)
// with g'_i = C_i / 24 (L327-332 Eq. 23), C_i the bare gradient sum (O-grad).
// A zero denominator gives +inf (reading J2).  Inputs are indexed by particle id;
// outputs are compact rows of the sink list.
// ---------------------------------------------------------------------------
inline double norm3(const double* p) { return std::sqrt(p[0] * p[0] + p[1] * p[1] + p[2] * p[2]); }

void criteria_impl(int64_t n, const double* vel, const double* acc, const double* grad_c, const double* jerk,
                   const int32_t* sink_idx, int64_t n_sink, double eta, double eta_grad, double eta_jerk,
                   double* dt_va, double* dt_gradv, double* dt_grada, double* dt_jerk) {
    (void)n;
    const double inf = std::numeric_limits<double>::infinity();
    for (int64_t k = 0; k < n_sink; ++k) {
        const int64_t i = pid(sink_idx, k);
        const double v = norm3(vel + 3 * i), a = norm3(acc + 3 * i);
        const double gp = norm3(grad_c + 3 * i) / 24.0;
        const double j = norm3(jerk + 3 * i);
        dt_va[k]    = (a == 0.0) ? inf : eta * v / a;
        dt_gradv[k] = (gp == 0.0) ? inf : eta_grad * std::cbrt(v / gp);
        dt_grada[k] = (gp == 0.0) ? inf : eta_grad * std::sqrt(a / gp);
        dt_jerk[k]  = (j == 0.0) ? inf : eta_jerk * a / j;
    }
}

// ---------------------------------------------------------------------------
// O-pot.  PAPER.md:L63 Eq. 4 (second term), softened like the accelerations:
//     W = -G sum_{i<j} m_i m_j / sqrt(|r_ji|^2 + eps^2).   Self-check only.
// ---------------------------------------------------------------------------
template <class T>
double potential_impl(int64_t n, const double* pos, const double* mass, double G, double eps) {
    const T eps2 = (T)eps * (T)eps;
    std::vector<double> row((size_t)n, 0.0);
#pragma omp parallel for schedule(dynamic, 8) if (n > 128)
    for (int64_t i = 0; i < n; ++i) {
        Neumaier<T> s;
        for (int64_t j = i + 1; j < n; ++j) {
            const T dx = (T)pos[3 * j] - (T)pos[3 * i], dy = (T)pos[3 * j + 1] - (T)pos[3 * i + 1],
                    dz = (T)pos[3 * j + 2] - (T)pos[3 * i + 2];
            s.add((T)mass[j] / std::sqrt(dx * dx + dy * dy + dz * dz + eps2));
        }
        row[(size_t)i] = (double)((T)mass[i] * s.value());
    }
    Neumaier<T> tot;
    for (int64_t i = 0; i < n; ++i) tot.add((T)row[(size_t)i]);
    return (double)(-(T)G * tot.value());
}

// ---------------------------------------------------------------------------
// O-share.  PAPER.md:L303 Eq. 20: "Each particle in the same subsystem shares the same
// time-step": eps_i = min_{j in S} eps_j for every member i of subsystem S; single particles
// (subsys = -1) keep their own value.  Written as the definition: for each i, a loop over all j.
// ---------------------------------------------------------------------------
void subsys_min_impl(int64_t n, const int32_t* subsys, const double* dt, double* out) {
    for (int64_t i = 0; i < n; ++i) {
        double best = dt[i];
        if (subsys[i] >= 0)
            for (int64_t j = 0; j < n; ++j)
                if (subsys[j] == subsys[i] && dt[j] < best) best = dt[j];
        out[i] = best;
    }
}

// ---------------------------------------------------------------------------
// O-ngb (NEXT-3).  PAPER.md:L227-281 §3.4 "Finding subsystems", Eq. 18-19, in the paper's order:
// for each pair (i, j) with r_ij = |r_j - r_i| < r_ngb_max compute the two-body orbital elements
// a (semi-major axis) and e (eccentricity) from the relative orbit,
//     mu = G (m_i + m_j),  E = v_ij^2/2 - mu/r_ij,  a = -mu/(2E),
//     h = r_ij x v_ij,     e = sqrt(1 + 2 E h^2/mu^2),
// then
//   bound   (E <  0):  neighbours iff  a < r_ngb  or  (a >= r_ngb and r_ij < r_ngb)             (Eq. 18)
//   unbound (E >= 0):  r_peri = a (1 - e); reject if r_peri >= r_ngb; otherwise neighbours iff
//                      r_ij < r_ngb  or  (r_ij >= r_ngb and C r_ij/|v_ij| < tau)                  (Eq. 19)
// Readings (N1-N3): r_peri is evaluated as p/(1+e) with p = h^2/mu, which equals a(1-e)
// for every conic and stays finite for the parabolic case E = 0 (a infinite); 1 + 2Eh^2/mu^2 is
// clamped at 0 before the square root; a pair with v_ij = 0 is bound (E < 0).  The relation is
// exactly symmetric in floating point (every quantity is even in the pair order).
// Output: for sink k, count[k] neighbours among the sources, their ids in source-list order in
// list[k*cap .. k*cap+min(count,cap)-1] (cap = capacity per sink; count itself is never truncated).
// ---------------------------------------------------------------------------
inline bool ngb_pair(const double* pos, const double* vel, const double* mass, int64_t i, int64_t j, double G,
                     double r_ngb, double r_ngb_max, double tau, double C) {
    const double dx = pos[3 * j] - pos[3 * i], dy = pos[3 * j + 1] - pos[3 * i + 1], dz = pos[3 * j + 2] - pos[3 * i + 2];
    const double r2 = dx * dx + dy * dy + dz * dz;
    const double r = std::sqrt(r2);
    if (!(r < r_ngb_max)) return false;
    const double ux = vel[3 * j] - vel[3 * i], uy = vel[3 * j + 1] - vel[3 * i + 1], uz = vel[3 * j + 2] - vel[3 * i + 2];
    const double v2 = ux * ux + uy * uy + uz * uz;
    const double mu = G * (mass[i] + mass[j]);
    const double E = 0.5 * v2 - mu / r;
    if (E < 0.0) {
        const double a = -mu / (2.0 * E);
        return (a < r_ngb) || (r < r_ngb);
    }
    const double hx = dy * uz - dz * uy, hy = dz * ux - dx * uz, hz = dx * uy - dy * ux;
    const double h2 = hx * hx + hy * hy + hz * hz;
    double e2 = 1.0 + 2.0 * E * h2 / (mu * mu);
    if (e2 < 0.0) e2 = 0.0;
    const double e = std::sqrt(e2);
    const double r_peri = (h2 / mu) / (1.0 + e);
    if (!(r_peri < r_ngb)) return false;
    if (r < r_ngb) return true;
    return C * r / std::sqrt(v2) < tau;
}

void ngb_impl(int64_t n, const double* pos, const double* vel, const double* mass, const int32_t* sink_idx,
              int64_t n_sink, const int32_t* src_idx, int64_t n_src, double G, double r_ngb, double r_ngb_max,
              double tau, double C, int64_t cap, int32_t* count, int32_t* list) {
    (void)n;
#pragma omp parallel for schedule(dynamic, 8) if (n_sink * n_src > 16384)
    for (int64_t k = 0; k < n_sink; ++k) {
        const int64_t i = pid(sink_idx, k);
        int64_t c = 0;
        for (int64_t l = 0; l < n_src; ++l) {
            const int64_t j = pid(src_idx, l);
            if (j == i) continue;
            if (ngb_pair(pos, vel, mass, i, j, G, r_ngb, r_ngb_max, tau, C)) {
                if (c < cap) list[k * cap + c] = (int32_t)j;
                ++c;
            }
        }
        count[k] = (int32_t)c;
    }
}

// O-comp.  PAPER.md:L279: subsystems = connected components of the neighbour graph ("finding the
// components of a finite graph", depth-first search).  label = smallest particle id of the
// component; a particle without any edge is single (-1).  edges: n_edge pairs (i, j).
void components_impl(int64_t n, const int32_t* edge_i, const int32_t* edge_j, int64_t n_edge, int32_t* subsys) {
    std::vector<std::vector<int32_t>> adj((size_t)n);
    for (int64_t q = 0; q < n_edge; ++q) {
        adj[(size_t)edge_i[q]].push_back(edge_j[q]);
        adj[(size_t)edge_j[q]].push_back(edge_i[q]);
    }
    for (int64_t i = 0; i < n; ++i) subsys[i] = -1;
    std::vector<char> seen((size_t)n, 0);
    std::vector<int32_t> stack, members;
    for (int64_t s = 0; s < n; ++s) {
        if (seen[(size_t)s] || adj[(size_t)s].empty()) continue;
        stack.assign(1, (int32_t)s); members.clear(); seen[(size_t)s] = 1;
        while (!stack.empty()) {                      // depth-first traversal
            const int32_t u = stack.back(); stack.pop_back();
            members.push_back(u);
            for (int32_t v : adj[(size_t)u])
                if (!seen[(size_t)v]) { seen[(size_t)v] = 1; stack.push_back(v); }
        }
        int32_t lab = members[0];
        for (int32_t u : members) if (u < lab) lab = u;
        for (int32_t u : members) subsys[(size_t)u] = lab;
    }
}

}  // namespace

extern "C" {

int oracle_acc(int64_t n, const double* pos, const double* mass, const int32_t* sink_idx, int64_t n_sink,
               const int32_t* src_idx, int64_t n_src, double G, double eps, double* out) {
    acc_impl<double>(n, pos, mass, sink_idx, n_sink, src_idx, n_src, G, eps, out);
    return 0;
}
int oracle_acc_ld(int64_t n, const double* pos, const double* mass, const int32_t* sink_idx, int64_t n_sink,
                  const int32_t* src_idx, int64_t n_src, double G, double eps, double* out) {
    acc_impl<long double>(n, pos, mass, sink_idx, n_sink, src_idx, n_src, G, eps, out);
    return 0;
}
int oracle_grad(int64_t n, const double* pos, const double* mass, const double* acc, const int32_t* sink_idx,
                int64_t n_sink, const int32_t* src_idx, int64_t n_src, double G, double eps, double* out) {
    grad_impl<double>(n, pos, mass, acc, sink_idx, n_sink, src_idx, n_src, G, eps, out);
    return 0;
}
int oracle_grad_ld(int64_t n, const double* pos, const double* mass, const double* acc, const int32_t* sink_idx,
                   int64_t n_sink, const int32_t* src_idx, int64_t n_src, double G, double eps, double* out) {
    grad_impl<long double>(n, pos, mass, acc, sink_idx, n_sink, src_idx, n_src, G, eps, out);
    return 0;
}
int oracle_dtmin(int64_t n, const double* pos, const double* vel, const double* mass, const int32_t* sink_idx,
                 int64_t n_sink, const int32_t* src_idx, int64_t n_src, double G, double eta_ff, double eta_fb,
                 double* dt_ff, double* dt_fb, int32_t* j_ff, int32_t* j_fb, double* margin_ff,
                 double* margin_fb) {
    dtmin_impl(n, pos, vel, mass, sink_idx, n_sink, src_idx, n_src, G, eta_ff, eta_fb, dt_ff, dt_fb, j_ff, j_fb,
               margin_ff, margin_fb);
    return 0;
}
int oracle_pn1(int64_t n, const double* pos, const double* vel, const double* mass, const int32_t* bh_idx,
               int64_t n_bh, double G, double c, double* out) {
    pn1_impl<double>(n, pos, vel, mass, bh_idx, n_bh, G, c, out);
    return 0;
}
int oracle_pn1_ld(int64_t n, const double* pos, const double* vel, const double* mass, const int32_t* bh_idx,
                  int64_t n_bh, double G, double c, double* out) {
    pn1_impl<long double>(n, pos, vel, mass, bh_idx, n_bh, G, c, out);
    return 0;
}
int oracle_jerk(int64_t n, const double* pos, const double* vel, const double* mass, const int32_t* sink_idx,
                int64_t n_sink, const int32_t* src_idx, int64_t n_src, double G, double eps, double* out) {
    jerk_impl<double>(n, pos, vel, mass, sink_idx, n_sink, src_idx, n_src, G, eps, out);
    return 0;
}
int oracle_jerk_ld(int64_t n, const double* pos, const double* vel, const double* mass, const int32_t* sink_idx,
                   int64_t n_sink, const int32_t* src_idx, int64_t n_src, double G, double eps, double* out) {
    jerk_impl<long double>(n, pos, vel, mass, sink_idx, n_sink, src_idx, n_src, G, eps, out);
    return 0;
}
int oracle_phi(int64_t n, const double* pos, const double* mass, const int32_t* sink_idx, int64_t n_sink,
               const int32_t* src_idx, int64_t n_src, double G, double eps, double* out) {
    phi_impl<double>(n, pos, mass, sink_idx, n_sink, src_idx, n_src, G, eps, out);
    return 0;
}
int oracle_criteria(int64_t n, const double* vel, const double* acc, const double* grad_c, const double* jerk,
                    const int32_t* sink_idx, int64_t n_sink, double eta, double eta_grad, double eta_jerk,
                    double* dt_va, double* dt_gradv, double* dt_grada, double* dt_jerk) {
    criteria_impl(n, vel, acc, grad_c, jerk, sink_idx, n_sink, eta, eta_grad, eta_jerk, dt_va, dt_gradv, dt_grada, dt_jerk);
    return 0;
}
double oracle_potential(int64_t n, const double* pos, const double* mass, double G, double eps) {
    return potential_impl<double>(n, pos, mass, G, eps);
}
double oracle_potential_ld(int64_t n, const double* pos, const double* mass, double G, double eps) {
    return potential_impl<long double>(n, pos, mass, G, eps);
}

// ---- NEXT-2: subsystem-aware variants (same routines, pairs inside one subsystem dropped) ----
int oracle_acc_sub(int64_t n, const double* pos, const double* mass, const int32_t* sink_idx, int64_t n_sink,
                   const int32_t* src_idx, int64_t n_src, double G, double eps, const int32_t* subsys, double* out) {
    acc_impl<double>(n, pos, mass, sink_idx, n_sink, src_idx, n_src, G, eps, out, subsys);
    return 0;
}
int oracle_grad_sub(int64_t n, const double* pos, const double* mass, const double* acc, const int32_t* sink_idx,
                    int64_t n_sink, const int32_t* src_idx, int64_t n_src, double G, double eps,
                    const int32_t* subsys, double* out) {
    grad_impl<double>(n, pos, mass, acc, sink_idx, n_sink, src_idx, n_src, G, eps, out, subsys);
    return 0;
}
int oracle_jerk_sub(int64_t n, const double* pos, const double* vel, const double* mass, const int32_t* sink_idx,
                    int64_t n_sink, const int32_t* src_idx, int64_t n_src, double G, double eps,
                    const int32_t* subsys, double* out) {
    jerk_impl<double>(n, pos, vel, mass, sink_idx, n_sink, src_idx, n_src, G, eps, out, subsys);
    return 0;
}
int oracle_phi_sub(int64_t n, const double* pos, const double* mass, const int32_t* sink_idx, int64_t n_sink,
                   const int32_t* src_idx, int64_t n_src, double G, double eps, const int32_t* subsys, double* out) {
    phi_impl<double>(n, pos, mass, sink_idx, n_sink, src_idx, n_src, G, eps, out, subsys);
    return 0;
}
int oracle_dtmin_sub(int64_t n, const double* pos, const double* vel, const double* mass, const int32_t* sink_idx,
                     int64_t n_sink, const int32_t* src_idx, int64_t n_src, double G, double eta_ff, double eta_fb,
                     const int32_t* subsys, double* dt_ff, double* dt_fb, int32_t* j_ff, int32_t* j_fb,
                     double* margin_ff, double* margin_fb) {
    dtmin_impl(n, pos, vel, mass, sink_idx, n_sink, src_idx, n_src, G, eta_ff, eta_fb, dt_ff, dt_fb, j_ff, j_fb,
               margin_ff, margin_fb, subsys);
    return 0;
}
int oracle_pn1_sub(int64_t n, const double* pos, const double* vel, const double* mass, const int32_t* bh_idx,
                   int64_t n_bh, double G, double c, const int32_t* subsys, double* out) {
    pn1_impl<double>(n, pos, vel, mass, bh_idx, n_bh, G, c, out, subsys);
    return 0;
}
int oracle_subsys_min(int64_t n, const int32_t* subsys, const double* dt, double* out) {
    subsys_min_impl(n, subsys, dt, out);
    return 0;
}

// ---- NEXT-3: neighbour search and subsystem construction (§3.4) ----
int oracle_ngb(int64_t n, const double* pos, const double* vel, const double* mass, const int32_t* sink_idx,
               int64_t n_sink, const int32_t* src_idx, int64_t n_src, double G, double r_ngb, double r_ngb_max,
               double tau, double C, int64_t cap, int32_t* count, int32_t* list) {
    ngb_impl(n, pos, vel, mass, sink_idx, n_sink, src_idx, n_src, G, r_ngb, r_ngb_max, tau, C, cap, count, list);
    return 0;
}
int oracle_components(int64_t n, const int32_t* edge_i, const int32_t* edge_j, int64_t n_edge, int32_t* subsys) {
    components_impl(n, edge_i, edge_j, n_edge, subsys);
    return 0;
}

}  // extern "C"
