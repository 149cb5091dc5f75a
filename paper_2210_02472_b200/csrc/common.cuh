// common.cuh - constants, device helpers, the source-array and launch-geometry structs shared by every kernel.
// Part of the single translation unit bifrost.cu (see its header and DESIGN.md); not a public header.
#pragma once

namespace {

constexpr int TILE = 128;         // sources per shared-memory tile
constexpr int MAX_SPLIT = 256;    // upper bound on grid.y (source-range splits)
constexpr int TICKETS = 1024;     // >= the largest grid.x of pair_fused_kernel

// ----------------------------------------------------------------------------------------
// small device helpers
// ----------------------------------------------------------------------------------------

// Seed for r2^(-1/2): MUFU.RSQ64H looks only at the high word.  Every caller adds R2_FLOOR (or a
// larger eps^2) to r2, so the argument is a positive normal number and the seed is finite even
// for the self pair (r_ji = 0 exactly), whose finite weight then multiplies a zero separation.
constexpr double R2_FLOOR = 4.909093465297727e-91;    // 2^-300: below any representable |r_ji|^2 of interest
__device__ __forceinline__ double rsqrt_seed(double r2) {
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(r2));
    return y;
}

__device__ __forceinline__ void cp_async16(void* smem, const void* gmem) {
    unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(s), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// a1 inputs: the caller's arrays a source record is gathered from (aux = acc for grad, vel for
// dtmin / jerk, unused otherwise); src_idx == NULL means sources are particles 0..n_src-1.
struct SrcArrays {
    const double* pos;
    const double* aux;
    const double* mass;
    const int32_t* subsys;
    const int32_t* src_idx;
};

struct Geom {
    int n_sink;           // number of sinks
    int n_src;            // number of sources (valid records)
    int tiles_per_split;  // source tiles handled by one blockIdx.y
    int n_split;          // gridDim.y
    int compact;          // 1: output row = sink position k, 0: output row = sink particle id
};

}  // namespace
