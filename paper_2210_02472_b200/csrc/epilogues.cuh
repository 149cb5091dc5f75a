// epilogues.cuh - fixed-order W / T reductions (Eq. 4, 68) and the O(N) time-step criteria (Eq. 24-29).
// Part of the single translation unit bifrost.cu (see its header and DESIGN.md); not a public header.
#pragma once

namespace {

// W = 1/2 sum_{i in sinks} m_i phi_i in two fixed-order stages (deterministic; no atomics).
constexpr int WSUM_THREADS = 256;
constexpr int WSUM_PER_BLOCK = 4096;
__device__ __forceinline__ double block_sum_fixed(double v) {
    __shared__ double red[WSUM_THREADS / 32];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) v += __shfl_down_sync(0xffffffffu, v, off);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = v;
    __syncthreads();
    double s = 0.0;
    if (threadIdx.x == 0)
        for (int w = 0; w < WSUM_THREADS / 32; ++w) s += red[w];
    return s;   // valid in thread 0
}
__global__ void __launch_bounds__(WSUM_THREADS)
wsum_stage1_kernel(int n_sink, const int32_t* __restrict__ sink_idx, int compact_phi, const double* __restrict__ mass,
                   const double* __restrict__ phi, double* __restrict__ block_part) {
    const int base = blockIdx.x * WSUM_PER_BLOCK;
    double v = 0.0;
    for (int q = threadIdx.x; q < WSUM_PER_BLOCK; q += WSUM_THREADS) {
        const int k = base + q;
        if (k < n_sink) {
            const int id = sink_idx ? sink_idx[k] : k;
            v += mass[id] * phi[compact_phi ? k : id];
        }
    }
    const double s = block_sum_fixed(v);
    if (threadIdx.x == 0) block_part[blockIdx.x] = s;
}
__global__ void __launch_bounds__(WSUM_THREADS)
wsum_stage2_kernel(int n_blocks, const double* __restrict__ block_part, double* __restrict__ out_W) {
    double v = 0.0;
    for (int q = threadIdx.x; q < n_blocks; q += WSUM_THREADS) v += block_part[q];
    const double s = block_sum_fixed(v);
    if (threadIdx.x == 0) *out_W = 0.5 * s;
}

// O(N) time-step criteria, Eq. 24, 26, 27, 29; IEEE sqrt / cbrt / division.
__global__ void criteria_kernel(int n_sink, const int32_t* __restrict__ sink_idx, const double* __restrict__ vel,
                                const double* __restrict__ acc, const double* __restrict__ grad,
                                const double* __restrict__ jerk, double eta, double eta_grad, double eta_jerk,
                                double* __restrict__ dt_va, double* __restrict__ dt_gradv, double* __restrict__ dt_grada,
                                double* __restrict__ dt_jerk, double* __restrict__ inout_dt) {
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n_sink) return;
    const int i = sink_idx ? sink_idx[k] : k;
    const size_t o = 3 * (size_t)i;
    const double inf = __longlong_as_double(0x7ff0000000000000LL);
    auto norm = [](const double* p) {
        return sqrt(__dadd_rn(__dadd_rn(__dmul_rn(p[0], p[0]), __dmul_rn(p[1], p[1])), __dmul_rn(p[2], p[2])));
    };
    const double v = norm(vel + o), a = norm(acc + o);
    double best = inout_dt ? inout_dt[i] : inf;
    const double t_va = (a == 0.0) ? inf : __dmul_rn(eta, v) / a;
    if (dt_va) dt_va[i] = t_va;
    best = fmin(best, t_va);
    if (grad) {
        const double gp = norm(grad + o) / 24.0;
        const double t_gv = (gp == 0.0) ? inf : eta_grad * cbrt(v / gp);
        const double t_ga = (gp == 0.0) ? inf : eta_grad * sqrt(a / gp);
        if (dt_gradv) dt_gradv[i] = t_gv;
        if (dt_grada) dt_grada[i] = t_ga;
        best = fmin(best, fmin(t_gv, t_ga));
    }
    if (jerk) {
        const double j = norm(jerk + o);
        const double t_j = (j == 0.0) ? inf : __dmul_rn(eta_jerk, a) / j;
        if (dt_jerk) dt_jerk[i] = t_j;
        best = fmin(best, t_j);
    }
    if (inout_dt) inout_dt[i] = best;
}

}  // namespace
