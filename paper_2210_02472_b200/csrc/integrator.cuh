// integrator.cuh - NEXT-4: kick / drift (Eq. 5, 7, 8), the slow/fast split of a hierarchy level, single-CTA FSI cycle for small levels, kinetic energy.
// Part of the single translation unit bifrost.cu (see its header and DESIGN.md); not a public header.
#pragma once

namespace {

// ----------------------------------------------------------------------------------------
// NEXT-4: the O(N) operators of the FSI cycle (Eq. 5, 7, 8) and the slow/fast
// split of a hierarchy level.
// ----------------------------------------------------------------------------------------
__global__ void kick_kernel(int m, const int32_t* __restrict__ idx, const double* __restrict__ acc,
                            const double* __restrict__ grad, double h, double c, double* __restrict__ vel) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= m) return;
    const size_t o = 3 * (size_t)(idx ? idx[k] : k);
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        double a = acc[o + d];
        if (grad) a = __dadd_rn(a, __dmul_rn(c, grad[o + d]));        // a~ = a + (eps^2/24) C   (Eq. 9)
        vel[o + d] = __dadd_rn(vel[o + d], __dmul_rn(h, a));          // v += h a                (Eq. 5, 8)
    }
}
__global__ void drift_kernel(int m, const int32_t* __restrict__ idx, const double* __restrict__ vel, double h,
                             double* __restrict__ pos) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= m) return;
    const size_t o = 3 * (size_t)(idx ? idx[k] : k);
#pragma unroll
    for (int d = 0; d < 3; ++d) pos[o + d] = __dadd_rn(pos[o + d], __dmul_rn(h, vel[o + d]));   // r += h v (Eq. 7)
}

// eps_i = min(eps_ff, eps_fb), never above the level-0 value; fast iff eps_i < tau
__global__ void level_flag_kernel(int m, const int32_t* __restrict__ seg, const double* __restrict__ dt_ff,
                                  const double* __restrict__ dt_fb, double* __restrict__ dt0,
                                  const double* __restrict__ dt_cap, int depth, double tau,
                                  int all_slow, unsigned char* __restrict__ fast) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= m) return;
    if (all_slow) { fast[k] = 0; return; }
    const int i = seg[k];
    double dt = fmin(dt_ff[i], dt_fb[i]);
    if (depth == 0) { if (dt_cap) dt = fmin(dt, dt_cap[i]); dt0[i] = dt; }
    dt = fmin(dt, dt0[i]);
    fast[k] = dt < tau ? 1 : 0;
}

// stable partition of a segment into [slow | fast]: block counts -> scan -> scatter
constexpr int PART_T = 256;
__global__ void __launch_bounds__(PART_T)
part_count_kernel(int m, const unsigned char* __restrict__ fast, int* __restrict__ block_slow) {
    const int k = blockIdx.x * PART_T + threadIdx.x;
    const int slow = (k < m) && !fast[k];
    const int c = __syncthreads_count(slow);
    if (threadIdx.x == 0) block_slow[blockIdx.x] = c;
}
__global__ void part_scan_kernel(int nb, int* __restrict__ block_slow, int* __restrict__ n_slow) {
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    int run = 0;
    for (int b = 0; b < nb; ++b) { const int c = block_slow[b]; block_slow[b] = run; run += c; }
    *n_slow = run;
}
__global__ void __launch_bounds__(PART_T)
part_scatter_kernel(int m, const int32_t* __restrict__ seg, const unsigned char* __restrict__ fast,
                    const int* __restrict__ block_slow, const int* __restrict__ n_slow, int32_t* __restrict__ out) {
    __shared__ int warp_slow[PART_T / 32];
    const int k = blockIdx.x * PART_T + threadIdx.x;
    const int live = k < m;
    const int slow = live && !fast[k];
    const unsigned bal = __ballot_sync(0xffffffffu, slow);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane == 0) warp_slow[warp] = __popc(bal);
    __syncthreads();
    int before = 0;                                           // slow elements of this block before this warp
    for (int w = 0; w < warp; ++w) before += warp_slow[w];
    const int rank_slow = before + __popc(bal & ((1u << lane) - 1u));
    if (!live) return;
    const int slow_before_block = block_slow[blockIdx.x];
    if (slow) out[slow_before_block + rank_slow] = seg[k];
    else {
        const int fast_before = (blockIdx.x * PART_T - slow_before_block) + (threadIdx.x - rank_slow);
        out[*n_slow + fast_before] = seg[k];
    }
}
// Small levels (m <= SMALL_M particles: the deep, sparsely populated levels of the hierarchy): the
// whole FSI cycle of Eq. 10 in ONE launch of one CTA, one thread per particle, the set's records in
// shared memory, a barrier between the stages.  The pair arithmetic is AccPass / GradPass ::pair
// and the sums run over the set in list order - for m <= 128 exactly what the general path (one
// tile, no split) computes, so the two paths agree bit for bit.
constexpr int SMALL_M = 256;
__global__ void __launch_bounds__(SMALL_M)
fsi_small_kernel(int m, const int32_t* __restrict__ idx, double* __restrict__ pos, double* __restrict__ vel,
                 const double* __restrict__ mass, double G, double eps2, double eps) {
    using PA = AccPassT<false>;
    using PG = GradPassT<false>;
    __shared__ __align__(16) double rec[SMALL_M * PG::REC];
    const int k = threadIdx.x;
    const bool live = k < m;
    const int id = live ? (idx ? idx[k] : k) : 0;
    const size_t o = 3 * (size_t)id;
    double x = 0, y = 0, z = 0, vx = 0, vy = 0, vz = 0, ms = 0;
    if (live) { x = pos[o]; y = pos[o + 1]; z = pos[o + 2]; vx = vel[o]; vy = vel[o + 1]; vz = vel[o + 2]; ms = mass[id]; }
    AccArgs aa{}; aa.eps2 = eps2;
    GradArgs ga{}; ga.eps2 = eps2;
    double ax, ay, az;
    auto accel = [&]() {                                   // Eq. 6 over the set
        __syncthreads();
        if (live) { PA::Raw w{x, y, z, ms, 0}; PA::emit(w, reinterpret_cast<double2*>(rec + k * PA::REC)); }
        __syncthreads();
        PA::Sink sk{x, y, z, 0};
        PA::Acc c; PA::init(c);
#pragma unroll 2
        for (int j = 0; j < m; ++j) {
            double r[PA::REC];
#pragma unroll
            for (int q = 0; q < PA::REC; ++q) r[q] = rec[j * PA::REC + q];
            PA::pair(aa, sk, c, r);
        }
        ax = G * c.x; ay = G * c.y; az = G * c.z;
    };
    auto kick = [&](double h, double gx, double gy, double gz, double cc, bool with_grad) {
        double tx = ax, ty = ay, tz = az;
        if (with_grad) { tx = __dadd_rn(tx, __dmul_rn(cc, gx)); ty = __dadd_rn(ty, __dmul_rn(cc, gy)); tz = __dadd_rn(tz, __dmul_rn(cc, gz)); }
        vx = __dadd_rn(vx, __dmul_rn(h, tx)); vy = __dadd_rn(vy, __dmul_rn(h, ty)); vz = __dadd_rn(vz, __dmul_rn(h, tz));
    };
    auto drift = [&](double h) {
        x = __dadd_rn(x, __dmul_rn(h, vx)); y = __dadd_rn(y, __dmul_rn(h, vy)); z = __dadd_rn(z, __dmul_rn(h, vz));
    };
    accel();
    kick(eps / 6.0, 0, 0, 0, 0, false);
    drift(eps / 2.0);
    accel();
    {                                                      // Eq. 9 over the set
        __syncthreads();
        if (live) { PG::Raw w{x, y, z, ax, ay, az, ms, -1}; PG::emit(w, reinterpret_cast<double2*>(rec + k * PG::REC)); }
        __syncthreads();
        PG::Sink sk{x, y, z, ax, ay, az, 0};
        PG::Acc c; PG::init(c);
#pragma unroll 2
        for (int j = 0; j < m; ++j) {
            double r[PG::REC];
#pragma unroll
            for (int q = 0; q < PG::REC; ++q) r[q] = rec[j * PG::REC + q];
            PG::pair(ga, sk, c, r);
        }
        const double gx = G * fma(-3.0, c.wx, c.ux), gy = G * fma(-3.0, c.wy, c.uy), gz = G * fma(-3.0, c.wz, c.uz);
        kick(2.0 * eps / 3.0, gx, gy, gz, eps * eps / 24.0, true);
    }
    drift(eps / 2.0);
    accel();
    kick(eps / 6.0, 0, 0, 0, 0, false);
    if (live) { pos[o] = x; pos[o + 1] = y; pos[o + 2] = z; vel[o] = vx; vel[o + 1] = vy; vel[o + 2] = vz; }
}

// Small levels: flag + stable S|F partition + write-back of the level's segment in one CTA.
__global__ void __launch_bounds__(SMALL_M)
level_split_small_kernel(int m, int32_t* __restrict__ seg, const double* __restrict__ dt_ff, const double* __restrict__ dt_fb,
                         double* __restrict__ dt0, const double* __restrict__ dt_cap, int depth, double tau, int all_slow,
                         int* __restrict__ n_slow) {
    __shared__ int warp_slow[SMALL_M / 32];
    const int k = threadIdx.x;
    const bool live = k < m;
    int i = 0, fast = 0;
    if (live) {
        i = seg[k];
        if (!all_slow) {
            double dt = fmin(dt_ff[i], dt_fb[i]);
            if (depth == 0) { if (dt_cap) dt = fmin(dt, dt_cap[i]); dt0[i] = dt; }
            dt = fmin(dt, dt0[i]);
            fast = dt < tau ? 1 : 0;
        }
    }
    const int slow = live && !fast;
    const unsigned bal = __ballot_sync(0xffffffffu, slow);
    const int lane = k & 31, warp = k >> 5;
    if (lane == 0) warp_slow[warp] = __popc(bal);
    __syncthreads();                                       // also: every seg[k] has been read
    int before = 0, total = 0;
    for (int w = 0; w < SMALL_M / 32; ++w) { if (w < warp) before += warp_slow[w]; total += warp_slow[w]; }
    const int rank_slow = before + __popc(bal & ((1u << lane) - 1u));
    if (live) seg[slow ? rank_slow : total + (k - rank_slow)] = i;
    if (k == 0) *n_slow = total;
}

__global__ void iota_kernel(int n, int32_t* __restrict__ a) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) a[i] = i;
}
__global__ void fill_f64_kernel(int n, double v, double* __restrict__ a) {
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) a[i] = v;
}

// T = 1/2 sum m v^2 over a set, fixed order (stage 1 of the W reduction with another integrand)
__global__ void __launch_bounds__(WSUM_THREADS)
ksum_stage1_kernel(int m, const int32_t* __restrict__ idx, const double* __restrict__ mass,
                   const double* __restrict__ vel, double* __restrict__ block_part) {
    const int base = blockIdx.x * WSUM_PER_BLOCK;
    double v = 0.0;
    for (int q = threadIdx.x; q < WSUM_PER_BLOCK; q += WSUM_THREADS) {
        const int k = base + q;
        if (k < m) {
            const int id = idx ? idx[k] : k;
            const double* u = vel + 3 * (size_t)id;
            v += mass[id] * (u[0] * u[0] + u[1] * u[1] + u[2] * u[2]);
        }
    }
    const double s = block_sum_fixed(v);
    if (threadIdx.x == 0) block_part[blockIdx.x] = s;
}

}  // namespace
