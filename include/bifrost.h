/* bifrost.h - C ABI of the B200 (sm_100a) direct-summation force path of BIFROST's
 * hierarchical fourth-order forward symplectic integrator (HHS-FSI).
 *
 * Paper: Rantala et al., "BIFROST: simulating compact subsystems in star clusters using a
 * hierarchical fourth-order forward symplectic integrator code", arXiv:2210.02472
 * (citations below are lines of /root/reference/PAPER.md).
 *
 * The library evaluates, for a set of active SINK particles i against a set of SOURCE
 * particles j, in binary64:
 *   bifrost_acc    softened Newtonian accelerations         (Eq. 6, Eq. 12)
 *   bifrost_grad   the FSI gradient ("extra") force sum     (Eq. 9, Eq. 13)
 *   bifrost_dtmin  free-fall / fly-by time-step minima      (Eq. 21, Eq. 22)
 *   bifrost_pn1    the global PN1.0 pair term, BH x N        (§3.8, Eq. 42-43)
 * Every step (index gather, pair kernels, fixed-order reductions, scatter) runs in
 * hand-written CUDA kernels; there is no CPU fallback.
 *
 * Common conventions
 *  - Particle arrays are indexed by particle id 0..n-1:
 *      pos, vel, acc, out_acc, out_grad, out_acc_pn : double[n][3], row-major;  mass : double[n].
 *  - sink_idx / src_idx / bh_idx : int32 particle ids in [0, n) (not range-checked).
 *    NULL means "all n particles in id order" and then the matching count must equal n.
 *  - r_ji = r_j - r_i (L65): the force on sink i points towards source j.
 *  - A source whose id equals the sink's id is skipped ("j != i", Eq. 6).
 *  - Coincident DISTINCT particles (r_ji = 0 exactly, j != i) at eps = 0 (reading A3b), where the
 *    literal formulas have 0/0: r^2 carries a floor of 2^-300, so the pair's weight is finite (m 2^450) and
 *    nothing becomes inf or NaN.  In bifrost_acc it multiplies a zero separation: the pair contributes
 *    exactly 0.  In bifrost_grad / bifrost_jerk it multiplies a_ji (v_ji): the two coincident sinks get a
 *    finite value WITHOUT meaning (0 if a_ji = 0 exactly, else rounding noise times 2^450); every OTHER
 *    sink is unaffected in all calls.
 *    bifrost_dtmin reports dt_ff = 0 (and dt_fb = 0 unless v_ij = 0 too) with that source as argmin, as
 *    Eq. 21-22 give; bifrost_potential a large finite value.  With eps > 0 such a pair is regular.
 *  - Duplicate ids in src_idx are summed twice; duplicates in sink_idx are harmless.
 *  - n_sink == 0 is a no-op.  n_src == 0 gives zeros (acc, grad) or +inf with id -1 (dtmin).
 *  - Results are written only at out[sink id]; other rows are untouched (bifrost_pn1 overwrites
 *    all n rows).  Outputs must not alias inputs.
 *  - Device entry points: every pointer is a DEVICE pointer owned by the caller; the call is
 *    asynchronous on `stream` (a cudaStream_t passed as void*, NULL = legacy default stream) and
 *    never synchronises the host.  The library owns only the scratch inside bifrost_ctx.  The scratch of
 *    the pair calls (packed records, split-j partials, the symmetric kernels' rows) is allocated in
 *    bifrost_create.  Two groups are allocated on FIRST USE - an implicit device synchronisation and a
 *    possible BIFROST_ECUDA in the middle of a run: the device mirrors + pinned staging of the *_host
 *    calls, and the integrator scratch of bifrost_fsi_step / bifrost_hhs_fsi.  bifrost_reserve
 *    allocates them ahead of time; after it no call allocates.
 *  - *_host entry points: every pointer is a HOST pointer (pinned or pageable); the call copies
 *    the inputs to device scratch owned by the context, runs the same kernels, copies the
 *    results back and returns after the stream has drained.
 *  - One context per stream; concurrent calls on one context are not allowed.
 *  - Results are bit-identical for identical inputs on the same GPU model: tiling is fixed by
 *    the argument sizes and every reduction runs in a fixed order (no floating-point atomics).
 *  - Launch shapes are chosen from the argument sizes alone: at most 32 sinks and a bounded number of pairs
 *    (128 sinks against at most 16384 sources) are one launch of thread-block clusters with the threads over the sources; below 4096 sinks a call is one
 *    fused launch (gather + pairs + last-CTA fixed-order reduction), above it is pack -> pair -> finish;
 *    bifrost_acc / bifrost_grad / bifrost_dtmin whose sink and source lists are the SAME list (same
 *    pointer, or both NULL) of >= 16384 / 12288 / 32768 entries evaluate every unordered pair once
 *    (symmetric kernels; results as before, in another summation order - dtmin's are bit-identical).
 *    The thresholds are bifrost_set_tuning knobs; no environment variable or file is read.
 *  - Return value: BIFROST_OK (0) or a negative BIFROST_E* code.  Nothing is printed, nothing
 *    aborts.  On BIFROST_ECUDA, bifrost_last_cuda_error(ctx) holds the CUDA error string.
 */
#ifndef BIFROST_H
#define BIFROST_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define BIFROST_OK      0
#define BIFROST_EINVAL (-1)  /* NULL where a pointer is required, negative count, n > max_n, n >= 2^31,
                                count/NULL-list mismatch */
#define BIFROST_ECUDA  (-2)  /* a CUDA runtime call or kernel launch failed */
#define BIFROST_ENOMEM (-3)  /* bifrost_create could not allocate its workspace */

typedef struct bifrost_ctx bifrost_ctx;

/* Create a context on CUDA device `device` able to handle up to max_n particles (ids < max_n,
 * list lengths <= max_n).  Allocates the scratch of the pair calls: packed source records (80 B x max_n),
 * split-j partials (1536 B x max_n), BH flags, and - when max_n >= 12288 and it fits in a quarter of the
 * free device memory - the source-side rows of the symmetric kernels (12 max_n^2 / 1536 bytes: 8.6 GB at
 * max_n = 2^20, 34 GB at 2^21; without them those calls take the plain kernels).  *ctx is set to NULL on failure. */
int bifrost_create(bifrost_ctx** ctx, int device, int64_t max_n);
int bifrost_destroy(bifrost_ctx* ctx);

/* Allocate now what would otherwise be allocated on first use (see "Device entry points" above):
 * what = BIFROST_RESERVE_HOST (mirrors of the *_host calls, ~30 x 8 B x max_n device + 32 B x max_n pinned)
 * and/or BIFROST_RESERVE_INTEGRATOR (scratch of bifrost_fsi_step / bifrost_hhs_fsi, ~110 B x max_n).
 * Synchronous.  BIFROST_ECUDA if an allocation fails (the context stays usable for the other calls). */
#define BIFROST_RESERVE_HOST        1
#define BIFROST_RESERVE_INTEGRATOR  2
int bifrost_reserve(bifrost_ctx* ctx, int what);

/* bifrost_set_shard - multi-GPU: shard the PAIR WORK of same-list bifrost_acc / bifrost_grad calls over `world`
 * ranks (one context, one process, one GPU each).  With world > 1 a call whose sink and source
 * lists are the same list evaluates only the blocks of the symmetric kernels owned by `rank` (dealt in snake
 * order, so every rank gets the same share of the pairs) and writes, for EVERY row of the list, this rank's partial
 * sum; the caller adds the ranks' outputs - one all-reduce (sum) of double[n][3], the path's exchange step - to
 * obtain the result.  Such calls take the symmetric kernels at any list length; calls with different sink and
 * source lists, with subsystems set, or on a context without the symmetric workspace return BIFROST_EINVAL while
 * world > 1 (shard those over sinks instead: disjoint sink lists per rank, no partial sums).  Every other entry
 * point is unaffected.  rank in [0, world); world = 1 restores the unsharded behaviour. */
int bifrost_set_shard(bifrost_ctx* ctx, int rank, int world);

/* Launch-shape knobs.  They never change a result beyond its summation order; they exist for tuning and so
 * that tests can drive every launch path at small sizes.
 *   BIFROST_TUNE_FUSED_MAX_SINKS  calls with fewer sinks run as one fused launch (default 4096, 0..131072)
 *   BIFROST_TUNE_SMALL_M          largest particle set whose FSI cycle / level split is one single-CTA launch
 *                                 (default 128, 0..256; 0 disables)
 *   BIFROST_TUNE_SYM_MIN_N        shortest same-list call that takes the symmetric kernels (default 16384 for
 *                                 acc, 12288 for grad, 32768 for dtmin; this knob sets all three; a value above
 *                                 max_n disables them) */
#define BIFROST_TUNE_FUSED_MAX_SINKS 0
#define BIFROST_TUNE_SMALL_M         1
#define BIFROST_TUNE_SYM_MIN_N       2
#define BIFROST_TUNE_MUTUAL_MIN_PAIRS 3   /* bifrost_*_mutual: fewest n_a * n_b pairs for the two-list symmetric kernel
                                             (default 5e7, and >= 512 entries in the shorter list; 0 = always) */
#define BIFROST_TUNE_FEW_MAX_SINKS 4      /* calls with at most this many sinks (default 32, 0..32; 0 disables) and at most */
#define BIFROST_TUNE_FEW_MAX_PAIRS 5      /* this many sink-source pairs (default 2^19 for acc, 2^18 for grad and dtmin; the knob sets
                                             all three; four times that for <= 8 sinks) run as ONE thread-block-cluster launch: threads
                                             over the sources, results merged through distributed shared memory, no workspace.
                                             At the default 32, calls with 33-128 sinks and at most 16384 sources take the same
                                             kernel with one cluster per 32 sinks. */
#define BIFROST_TUNE_FUSED_CLUSTER 6      /* 1 (default): the fused launch runs as clusters of up to 8 CTAs that combine their split-j
                                             partials through distributed shared memory (sums for acc / grad / jerk, the winners'
                                             merge for dtmin); 0: every CTA's partial goes through global memory (the order of
                                             the additions differs, nothing else; dtmin is bit-identical) */
int bifrost_set_tuning(bifrost_ctx* ctx, int knob, int64_t value);

const char* bifrost_strerror(int code);                 /* static string */
const char* bifrost_last_cuda_error(bifrost_ctx* ctx);  /* "" if none; valid until the next call */
/* Number of kernels this context has launched since creation (for bench.py's gpu_launches). */
int64_t bifrost_launch_count(bifrost_ctx* ctx);

/* bifrost_acc - PAPER.md:L75 Eq. 6 and L115-119 Eq. 12 with Plummer softening (L818):
 *     out_acc[i] = G * sum_{j in src, j != i} mass[j] * r_ji / (|r_ji|^2 + eps^2)^(3/2),  i in sinks.
 * eps is the softening LENGTH (eps = 0: BIFROST's unsoftened standard mode). */
int bifrost_acc(bifrost_ctx* ctx, int64_t n, const double* pos, const double* mass,
                const int32_t* sink_idx, int64_t n_sink, const int32_t* src_idx, int64_t n_src,
                double G, double eps, double* out_acc, void* stream);

/* bifrost_grad - the sum of PAPER.md:L90 Eq. 9 / L123-127 Eq. 13, second pass:
 *     out_grad[i] = G * sum_{j in src, j != i} mass[j] * [ a_ji / s^3 - 3 (a_ji . r_ji) r_ji / s^5 ],
 *     a_ji = acc[j] - acc[i],  s^2 = |r_ji|^2 + eps^2
 * i.e. the bare tidal-tensor contraction C_i; the caller forms the gradient acceleration
 * a~_i = a_i + (eps_step^2 / 24) C_i (Eq. 9; Eq. 23: g_i = 2 C_i, g'_i = C_i / 24).
 * acc[] must hold the up-to-date Newtonian acceleration of every id that appears as a sink or
 * a source (L99: "up-to-date Newtonian accelerations are required"); which accelerations
 * those are (all-active or inter-level, Eq. 12) is the caller's choice. */
int bifrost_grad(bifrost_ctx* ctx, int64_t n, const double* pos, const double* mass, const double* acc,
                 const int32_t* sink_idx, int64_t n_sink, const int32_t* src_idx, int64_t n_src,
                 double G, double eps, double* out_grad, void* stream);

/* bifrost_acc_mutual / bifrost_grad_mutual - the inter-level sums of PAPER.md:L115-127 (Eq. 12, Eq. 13) for BOTH sets
 * of a level in one call: with two DISJOINT id lists A (e.g. the slow set S) and B (the fast set F),
 *     out[a] = the bifrost_acc (bifrost_grad) sum of sink a over the sources B,   a in A,
 *     out[b] = the same sum of sink b over the sources A,                         b in B
 * - exactly what the pair of calls (sinks A, sources B) and (sinks B, sources A) writes, rounding order apart.  Eq. 12-13
 * are "pairwise kicks" (L131): each (a, b) pair's geometry serves both members, so large lists go through the
 * two-list symmetric kernel (every pair evaluated once, 20 / 33 instead of 30 / 56 FP64 instructions per pair);
 * short lists, and calls while subsystems are set, are issued as the two plain calls.  Both lists are required
 * (non-NULL); an id that appears in both gets only one of its two sums.  Other conventions as bifrost_acc /
 * bifrost_grad.  DEVICE pointers, asynchronous on stream. */
int bifrost_acc_mutual(bifrost_ctx* ctx, int64_t n, const double* pos, const double* mass,
                       const int32_t* a_idx, int64_t n_a, const int32_t* b_idx, int64_t n_b,
                       double G, double eps, double* out_acc, void* stream);
int bifrost_grad_mutual(bifrost_ctx* ctx, int64_t n, const double* pos, const double* mass, const double* acc,
                        const int32_t* a_idx, int64_t n_a, const int32_t* b_idx, int64_t n_b,
                        double G, double eps, double* out_grad, void* stream);

/* bifrost_dtmin - PAPER.md:L312 Eq. 21 and L317 Eq. 22 (unsoftened), per sink i:
 *     out_dt_ff[i] = eta_ff * min_{j in src, j != i} sqrt( |r_ij|^3 / (G (m_i + m_j)) ),  out_j_ff[i] = argmin id
 *     out_dt_fb[i] = eta_fb * min_{j in src, j != i} |r_ij| / |v_ij|,                      out_j_fb[i] = argmin id
 * Exact ties go to the smaller particle id.  A pair with v_ij = 0 has fly-by time +inf; if no
 * source gives a finite value the result is +inf with id -1.  Any of the four outputs may be
 * NULL.  The caller takes min(dt_ff, dt_fb) (L293). */
int bifrost_dtmin(bifrost_ctx* ctx, int64_t n, const double* pos, const double* vel, const double* mass,
                  const int32_t* sink_idx, int64_t n_sink, const int32_t* src_idx, int64_t n_src,
                  double G, double eta_ff, double eta_fb,
                  double* out_dt_ff, double* out_dt_fb, int32_t* out_j_ff, int32_t* out_j_fb, void* stream);

/* bifrost_pn1 - PAPER.md:L476-488 §3.8 (Eq. 42-43): the global PN1.0 term "only for pairwise
 * interactions when either of the particles is massive enough".  The caller supplies the ids of
 * the massive particles (m > m_PN) in bh_idx (distinct ids; n_bh may be 0).  For every ordered
 * pair (i, j), i != j, with i or j in bh_idx, each pair once:
 *     out_acc_pn[i] += G m_j / (c^2 r^2) { n [ 5 G m_i / r + 4 G m_j / r + 3/2 (n.v_j)^2 - v_i.v_i
 *                                              + 4 v_i.v_j - 2 v_j.v_j ] + (4 n.v_i - 3 n.v_j)(v_i - v_j) },
 *     r = |r_i - r_j|,  n = (r_i - r_j) / r
 * (standard two-body 1PN/EIH term in harmonic coordinates; the paper cites Thorne & Hartle 1985
 * without printing it - DESIGN.md reading P1).  out_acc_pn : double[n][3], fully overwritten. */
int bifrost_pn1(bifrost_ctx* ctx, int64_t n, const double* pos, const double* vel, const double* mass,
                const int32_t* bh_idx, int64_t n_bh, double G, double c, double* out_acc_pn, void* stream);

/* ---- NEXT rows, built on the same kernels.  Device pointers, asynchronous. ---- */

/* bifrost_jerk - PAPER.md:L360 Eq. 28 (lhs garbled in the extraction; reading J1: j_i = da_i/dt,
 * sum over j != i), softened like bifrost_acc so that it is the exact time derivative of it:
 *     out_jerk[i] = G * sum_{j in src, j != i} mass[j] * [ v_ji / s^3 - 3 (r_ji . v_ji) r_ji / s^5 ],
 *     v_ji = vel[j] - vel[i],  s^2 = |r_ji|^2 + eps^2.
 * Same tensor contraction as bifrost_grad with v_ji for a_ji (one kernel serves both).
 * Index-list, self-pair and output conventions as for bifrost_acc. */
int bifrost_jerk(bifrost_ctx* ctx, int64_t n, const double* pos, const double* vel, const double* mass,
                 const int32_t* sink_idx, int64_t n_sink, const int32_t* src_idx, int64_t n_src,
                 double G, double eps, double* out_jerk, void* stream);

/* bifrost_acc_jerk - NEXT-1 ("can be fused into the acc pass"): bifrost_acc's acceleration
 * (Eq. 6) and bifrost_jerk's jerk (Eq. 28) of the sinks in ONE pass over the
 * sources - the pair's separation, softened distance and reciprocal square root are shared, 31 FP64
 * instructions per pair instead of 15 + 28.  Arguments, layout and index semantics as bifrost_acc /
 * bifrost_jerk; out_acc and out_jerk (double[n][3], distinct, written at sink rows) must not alias inputs. */
int bifrost_acc_jerk(bifrost_ctx* ctx, int64_t n, const double* pos, const double* vel, const double* mass,
                     const int32_t* sink_idx, int64_t n_sink, const int32_t* src_idx, int64_t n_src,
                     double G, double eps, double* out_acc, double* out_jerk, void* stream);

/* bifrost_potential - the potential term of PAPER.md:L63 Eq. 4 (and the first two terms' potential
 * part of the energy book-keeping, L724 Eq. 68), softened like bifrost_acc:
 *     out_phi[i] = -G * sum_{j in src, j != i} mass[j] / sqrt(|r_ji|^2 + eps^2)      (i in sinks; double[n])
 *     *out_W     = 1/2 * sum_{i in sinks} mass[i] * phi_i                             (one DEVICE double)
 * With sinks = sources = all, *out_W = -sum_{i<j} G m_i m_j / s_ij.  Either output may be NULL (not
 * both).  The self pair is dropped by particle id.  The sum over sinks runs in a fixed order
 * (two-stage block reduction), so *out_W is bit-reproducible. */
int bifrost_potential(bifrost_ctx* ctx, int64_t n, const double* pos, const double* mass,
                      const int32_t* sink_idx, int64_t n_sink, const int32_t* src_idx, int64_t n_src,
                      double G, double eps, double* out_phi, double* out_W, void* stream);

/* bifrost_timestep_criteria - the O(N) per-particle criteria of PAPER.md §3.5.4-3.5.5, for i in sinks:
 *     out_dt_va[i]    = eta      * |vel_i| / |acc_i|                      (L338 Eq. 24)
 *     out_dt_gradv[i] = eta_grad * (|vel_i| / |g'_i|)^(1/3)               (L346 Eq. 26)
 *     out_dt_grada[i] = eta_grad * (|acc_i| / |g'_i|)^(1/2)               (L350 Eq. 27)
 *     out_dt_jerk[i]  = eta_jerk * |acc_i| / |jerk_i|                     (L365 Eq. 29)
 * with g'_i = grad_i / 24 (L327-332 Eq. 23), grad = the output of bifrost_grad, jerk = the output of
 * bifrost_jerk; all double[n][3] indexed by particle id.  A zero denominator gives +inf.
 * grad and/or jerk may be NULL (their criteria are skipped; the matching outputs must be NULL).
 * Any out_* may be NULL.  If inout_dt (double[n]) is not NULL, inout_dt[i] = min(inout_dt[i], every
 * criterion evaluated) - "the final time-step of a particle is the minimum of the set of its
 * different time-steps" (L293); seed it with min(dt_ff, dt_fb) from bifrost_dtmin or with +inf. */
int bifrost_timestep_criteria(bifrost_ctx* ctx, int64_t n, const double* vel, const double* acc,
                              const double* grad, const double* jerk, const int32_t* sink_idx, int64_t n_sink,
                              double eta, double eta_grad, double eta_jerk,
                              double* out_dt_va, double* out_dt_gradv, double* out_dt_grada, double* out_dt_jerk,
                              double* inout_dt, void* stream);

/* ---- NEXT-2: subsystem-aware sums ----
 * bifrost_set_subsystems - PAPER.md:L233 Alg. 1 ("Acceleration calculations ignore intra-subsystem
 * contributions"), L299 §3.5.2 (same-subsystem particles are excluded from the time-step assignment)
 * and L488 §3.8 (no PN kick between members of one subsystem).  subsys : DEVICE int32[n]; subsys[k] is
 * the subsystem particle k belongs to (0 <= id < n) or -1 for a single particle.  While set, EVERY
 * pair routine of this context (acc, grad, jerk, potential, dtmin, pn1 and their *_host variants)
 * drops each pair (i, j) whose members carry the same id >= 0, in addition to j == i; calls must then
 * use the same n (else BIFROST_EINVAL).  The pointer is BORROWED: the caller keeps the array alive and
 * unchanged until it is replaced or reset with subsys = NULL (which restores the plain sums).
 * The exclusion is decided inside the pair kernels (an integer compare and a select per pair; the
 * excluded term is never formed, so there is no cancellation against the huge intra-subsystem force). */
int bifrost_set_subsystems(bifrost_ctx* ctx, const int32_t* subsys, int64_t n);

/* bifrost_subsys_min - PAPER.md:L303 Eq. 20: every member of a subsystem shares the minimum time-step
 * of its members: inout_dt[i] = min_{j : subsys[j] == subsys[i]} inout_dt[j] for subsys[i] >= 0; single
 * particles keep their value.  DEVICE pointers, asynchronous on stream; inout_dt : double[n] >= 0.
 * Exact and order-independent (integer atomic minimum on the bit patterns). */
int bifrost_subsys_min(bifrost_ctx* ctx, int64_t n, const int32_t* subsys, double* inout_dt, void* stream);

/* bifrost_neighbours - NEXT-3, §3.4 "Finding subsystems", Eq. 18-19.  For every sink i
 * and every source j != i with r_ij = |r_j - r_i| < r_ngb_max the two-body orbital elements of the pair
 * are formed (mu = G (m_i + m_j), E = v_ij^2/2 - mu/r_ij, a = -mu/(2E), h = r_ij x v_ij,
 * e = sqrt(max(0, 1 + 2 E h^2/mu^2))) and j is a neighbour of i iff
 *   bound   (E <  0): a < r_ngb  or  r_ij < r_ngb                                              (Eq. 18)
 *   unbound (E >= 0): r_peri < r_ngb  and  ( r_ij < r_ngb  or  C r_ij/|v_ij| < tau )           (Eq. 19)
 * with r_peri = a (1 - e) evaluated as (h^2/mu)/(1 + e) (finite for the parabolic case).  tau is the
 * pivot time-step of the hierarchy level, C < 1 the safety factor.  The relation is symmetric.
 * The decision is taken in IEEE fp64, operation by operation (no contraction; correctly rounded sqrt
 * and division), so it is reproducible bit for bit; only a conservative distance pre-filter runs in
 * the fast path.  DEVICE pointers, asynchronous on stream.
 *   out_count : int32[n]        number of neighbours of sink i among the sources, at row i (never truncated)
 *   out_list  : int32[n][cap]   their ids in source-list order, the first min(count, cap) of them, at row i;
 *                               entries beyond that and rows of non-sinks are untouched.  1 <= cap <= 1024. */
int bifrost_neighbours(bifrost_ctx* ctx, int64_t n, const double* pos, const double* vel, const double* mass,
                       const int32_t* sink_idx, int64_t n_sink, const int32_t* src_idx, int64_t n_src,
                       double G, double r_ngb, double r_ngb_max, double tau, double C, int64_t cap,
                       int32_t* out_count, int32_t* out_list, void* stream);

/* bifrost_dtmin_neighbours - bifrost_dtmin and bifrost_neighbours in ONE pass over the pairs.  The paper does
 * the neighbour search "at the beginning of each integration hierarchy level along with the time-step assignment"
 * (both are among the O(N^2) loops of L747); the two need the same records (x, v, m) and the same
 * r_ij^2, so the pass of Eq. 21-22 (L312, L317) carries the distance pre-filter of Eq. 18-19 as one integer test
 * per pair and sends the rare candidates through the same exact evaluation as bifrost_neighbours.  Arguments and
 * outputs are those of the two calls; all six outputs are bit-identical to the separate calls' (out_count and
 * out_list required, the four time-step outputs may be NULL).  While bifrost_set_subsystems is active the
 * time-steps exclude same-subsystem pairs (L299) and the neighbour search does not, as in the separate calls.
 * BIFROST_EINVAL if (28 + 4 cap) * n_sink bytes exceed the split-j workspace (1536 B x max_n).
 * DEVICE pointers, asynchronous on stream. */
int bifrost_dtmin_neighbours(bifrost_ctx* ctx, int64_t n, const double* pos, const double* vel, const double* mass,
                             const int32_t* sink_idx, int64_t n_sink, const int32_t* src_idx, int64_t n_src,
                             double G, double eta_ff, double eta_fb,
                             double r_ngb, double r_ngb_max, double tau, double C, int64_t cap,
                             double* out_dt_ff, double* out_dt_fb, int32_t* out_j_ff, int32_t* out_j_fb,
                             int32_t* out_count, int32_t* out_list, void* stream);

/* bifrost_components - NEXT-3: subsystems are the connected components of the neighbour
 * graph.  count / list are bifrost_neighbours' outputs (rows of particles that were not sinks must have
 * count = 0; ids outside [0, n) and self edges are ignored; an edge listed in one direction only still
 * joins its two ends).  out_subsys[i] = smallest particle id of i's component, or -1 if no edge touches i
 * - the array bifrost_set_subsystems and bifrost_subsys_min take.  The paper traverses the graph
 * depth-first on the host; here it is a lock-free union-find on the device whose result does not
 * depend on the order of the edges.  DEVICE pointers, asynchronous on stream. */
int bifrost_components(bifrost_ctx* ctx, int64_t n, const int32_t* count, const int32_t* list, int64_t cap,
                       int32_t* out_subsys, void* stream);

/* ---- NEXT-4: the integrator built on the sums above (§2.1-2.2) -------------------------
 * Scratch for these calls (2 x double[max_n][3], 3 x double[max_n], 2 x int32[max_n]) is allocated on
 * their first use, not in bifrost_create. */

/* bifrost_kick - Eq. 5 / Eq. 8-9: vel[i] += h * (acc[i] + c * grad[i]) for i in idx
 * (grad == NULL: vel[i] += h * acc[i]).  The gradient kick of a cycle of length eps is h = 2 eps/3,
 * c = eps^2/24 with grad = bifrost_grad's output.  idx == NULL means all n (n_idx must equal n).
 * DEVICE pointers, asynchronous on stream. */
int bifrost_kick(bifrost_ctx* ctx, int64_t n, const int32_t* idx, int64_t n_idx, const double* acc,
                 const double* grad, double h, double c, double* vel, void* stream);

/* bifrost_drift - Eq. 7: pos[i] += h * vel[i] for i in idx.  As bifrost_kick. */
int bifrost_drift(bifrost_ctx* ctx, int64_t n, const int32_t* idx, int64_t n_idx, const double* vel, double h,
                  double* pos, void* stream);

/* bifrost_fsi_step - one FSI cycle, Eq. 10: kick(eps/6) drift(eps/2) gradient kick(2 eps/3)
 * drift(eps/2) kick(eps/6) over the particles idx interacting ONLY among themselves (sinks = sources = idx;
 * idx == NULL: all n): four O(N^2) sums (acc, acc, grad, acc) and five O(N) updates, all on
 * stream, no host synchronisation.  pos and vel (double[n][3]) are updated in place at the rows in idx.
 * eps_soft is the Plummer softening of the sums, eps the time-step.  BIFROST_EINVAL while
 * bifrost_set_subsystems is active: Alg. 1 drifts single particles only and hands subsystem
 * members to the regularised integrator, which is outside this library (reading H5) - integrating
 * them here would move them without their mutual force. */
int bifrost_fsi_step(bifrost_ctx* ctx, int64_t n, double* pos, double* vel, const double* mass,
                     const int32_t* idx, int64_t n_idx, double G, double eps_soft, double eps, void* stream);

/* bifrost_hhs_fsi - one HHS-FSI integration interval of length tau, Eq. 11-13, without
 * subsystem integration (the "softened FROST-like" mode of PAPER.md:L818).  At every level: time-steps
 * eps_i = min(eps_ff, eps_fb) (Eq. 21-22 with eta_ff, eta_fb) of the level's particles among themselves,
 * capped by the particle's level-0 value; fast F = {eps_i < tau}, slow S = the rest (stable
 * partition, S first); then  U_SF(tau/6) H_S(tau/2) H_F(tau/2) U~_SF(2 tau/3) H_F(tau/2) H_S(tau/2) U_SF(tau/6)
 * with the inter-level accelerations of Eq. 12, the gradient accelerations of Eq. 13, H_S = bifrost_fsi_step
 * over S and H_F = this procedure over F with tau/2.  A level without fast particles (or at depth max_depth,
 * 0 <= max_depth <= 62) is one FSI cycle of length tau.  Every sum and update runs on the device; the host
 * reads one integer (|S|) per level to steer the recursion, so the call is SYNCHRONOUS.
 *   dt_cap : DEVICE double[n] or NULL - further per-particle time-steps taken at the start of the interval
 *            (e.g. bifrost_timestep_criteria's Eq. 24-29 minimum): eps_i^{level 0} = min(eps_ff, eps_fb, dt_cap[i]),
 *            "the final time-step of a particle is the minimum of the set of its different time-steps" (L293);
 *   out_level_log : HOST int64[log_cap][3] or NULL - (depth, |S|, |F|) of the first log_cap levels, in the
 *                   order they are entered;   out_summary : HOST int64[3] or NULL - levels entered, deepest
 *                   depth, FSI cycles run.  pos, vel : DEVICE double[n][3], updated in place.
 * BIFROST_EINVAL while bifrost_set_subsystems is active (as bifrost_fsi_step). */
/* bifrost_set_level_criteria - bifrost_hhs_fsi evaluates the acceleration-based time-step criteria of Eq. 24, 26, 27, 29
 * (bifrost_timestep_criteria's formulas with eta, eta_grad, eta_jerk) at EVERY level, over the level's
 * own particles (accelerations, gradient sums and jerks of the level's particles among themselves), and takes
 * eps_i = min(eps_ff, eps_fb, those four) before the level-0 cap: "the final time-step of a particle is the minimum of
 * the set of its different time-steps" (L293), "eps_i = min(eps_i, eps_i^{level 0})" (L295).  Costs one acc+jerk pass and one
 * grad pass per level.
 * All three > 0 switches it on, all three 0 (the default) off: then only dt_cap carries such criteria, at level 0
 * (reading H4).  Anything else is BIFROST_EINVAL. */
int bifrost_set_level_criteria(bifrost_ctx* ctx, double eta, double eta_grad, double eta_jerk);

int bifrost_hhs_fsi(bifrost_ctx* ctx, int64_t n, double* pos, double* vel, const double* mass, double G,
                    double eps_soft, double eta_ff, double eta_fb, const double* dt_cap, double tau, int max_depth,
                    int64_t* out_level_log, int64_t log_cap, int64_t* out_summary, void* stream);

/* bifrost_kinetic_energy - first term of Eq. 4: *out_T = 1/2 sum_{i in idx} m_i |v_i|^2
 * (DEVICE double, fixed-order two-stage reduction: deterministic).  With bifrost_potential's out_W this
 * is the total energy of the relative-energy-error check, Eq. 72-73. */
int bifrost_kinetic_energy(bifrost_ctx* ctx, int64_t n, const double* vel, const double* mass,
                           const int32_t* idx, int64_t n_idx, double* out_T, void* stream);

/* Host-buffer variants: same semantics, HOST pointers, synchronous (see header comment).
 * Index lists may be NULL as above.  Outputs are written only at sink ids (other host rows are
 * untouched), bifrost_pn1_host overwrites all n rows. */
int bifrost_acc_host(bifrost_ctx* ctx, int64_t n, const double* pos, const double* mass,
                     const int32_t* sink_idx, int64_t n_sink, const int32_t* src_idx, int64_t n_src,
                     double G, double eps, double* out_acc);
int bifrost_grad_host(bifrost_ctx* ctx, int64_t n, const double* pos, const double* mass, const double* acc,
                      const int32_t* sink_idx, int64_t n_sink, const int32_t* src_idx, int64_t n_src,
                      double G, double eps, double* out_grad);
int bifrost_dtmin_host(bifrost_ctx* ctx, int64_t n, const double* pos, const double* vel, const double* mass,
                       const int32_t* sink_idx, int64_t n_sink, const int32_t* src_idx, int64_t n_src,
                       double G, double eta_ff, double eta_fb,
                       double* out_dt_ff, double* out_dt_fb, int32_t* out_j_ff, int32_t* out_j_fb);
int bifrost_pn1_host(bifrost_ctx* ctx, int64_t n, const double* pos, const double* vel, const double* mass,
                     const int32_t* bh_idx, int64_t n_bh, double G, double c, double* out_acc_pn);

/* Measurement aid, not part of the paper's path: runs a register-only kernel of independent FP64
 * chains (no memory traffic) on the context's device, on the legacy default stream, synchronously,
 * so that bench.py can quote a MEASURED FP64-pipe peak beside the derived one.
 *   mix = 0: pure DFMA;  mix = 1: 3 DADD + 9 DFMA + 3 DMUL per 15 instructions (the acc pair's mix);
 *   mix = 2: DFMA with three distinct register operands;  mix = 3: groups of three DFMAs sharing one
 *   operand (the pair kernels' accumulate pattern) - these two expose the register-file operand limit.
 *   iters: loop trips per thread (32 (mix 0), 120 (mix 1) or 12 (mix 2, 3) FP64 instructions each);
 *   ctas_per_sm: grid = SM count x ctas_per_sm CTAs of 128 threads (4 are resident per SM).
 * HOST outputs: *out_ms = device time of one launch (CUDA events, after a warm-up launch);
 * *out_lane_instr = FP64-pipe lane-instructions that launch executed (threads x instructions). */
int bifrost_fp64_probe(bifrost_ctx* ctx, int mix, int64_t iters, int ctas_per_sm, double* out_ms,
                       double* out_lane_instr);

/* bifrost_acc_static - bifrost_acc (Eq. 6, all n particles as sinks and as sources) for callers
 * that cannot allocate: code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.
 * It needs NO context and calls no cudaMalloc, cudaFree or allocating library routine: the packed source
 * records, the split-j partial sums and the arrival counters of the fused kernel live in ONE file-scope
 * `static __device__` array of BIFROST_STATIC_SCRATCH_BYTES (8 MiB) inside libbifrost.so, which every GPU that
 * loads the library holds until the process exits.  The kernels are those of bifrost_acc (one fused launch
 * below 4096 particles, pack -> pair -> finish from there on); only the split count, hence the summation
 * order, can differ from a context's (the workspace is smaller), so results agree with bifrost_acc to rounding.
 *   device   CUDA device ordinal (0 <= device < 64); made current for the call and restored afterwards.  The first
 *            call on a device does the set-up (the array's device address, the SM count); make one call
 *            before starting a graph capture.
 *   n        0 <= n <= BIFROST_STATIC_MAX_N (16384); beyond that the call is refused with BIFROST_EINVAL and a
 *            message that names the limit (bifrost_static_error) - use bifrost_acc with a context instead.
 *   pos [n][3], mass [n], out_acc [n][3]: DEVICE pointers on `device`, borrowed; G, eps as for bifrost_acc.
 *   stream   cudaStream_t (NULL = legacy default); asynchronous like bifrost_acc.
 * Every call on a device shares that device's array.  The array keeps the last call's contents; the one part that
 * must start at zero (the arrival counters) is cleared on the stream by every call that uses it, everything
 * else is written before it is read.  Two calls that OVERLAP on the same GPU (different streams, or different
 * host threads without ordering between their streams) race on the array and give undefined results; calls on
 * one stream, or ordered by events, are safe.
 * Returns BIFROST_OK, BIFROST_EINVAL (bad device, n out of range, NULL pointer) or BIFROST_ECUDA. */
#define BIFROST_STATIC_MAX_N 16384
#define BIFROST_STATIC_SCRATCH_BYTES (8u << 20)
int bifrost_acc_static(int device, int64_t n, const double* pos, const double* mass, double G, double eps,
                       double* out_acc, void* stream);
/* Message of the calling thread's last failed bifrost_acc_static ("" if it succeeded); static storage. */
const char* bifrost_static_error(void);

#ifdef __cplusplus
}
#endif
#endif /* BIFROST_H */
