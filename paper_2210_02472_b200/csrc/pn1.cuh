// pn1.cuh - a6: the sparse BH x N PN1.0 pair term (§3.8).
// Part of the single translation unit bifrost.cu (see its header and DESIGN.md); not a public header.
#pragma once

namespace {

// ----------------------------------------------------------------------------------------
// a6: PN1.0 pair term (§3.8).  Standard two-body 1PN acceleration in harmonic coordinates.
// ----------------------------------------------------------------------------------------
struct Body { double x, y, z, m, vx, vy, vz; };

__device__ __forceinline__ Body load_body(const double* pos, const double* vel, const double* mass, int id) {
    Body b;
    const size_t o = 3 * (size_t)id;
    b.x = pos[o]; b.y = pos[o + 1]; b.z = pos[o + 2];
    b.vx = vel[o]; b.vy = vel[o + 1]; b.vz = vel[o + 2];
    b.m = mass[id];
    return b;
}

// acceleration of body `i` due to body `j`, 1/c^2 part only
__device__ __forceinline__ void pn1_pair(const Body& i, const Body& j, double G, double inv_c2,
                                         double& fx, double& fy, double& fz) {
    const double rx = i.x - j.x, ry = i.y - j.y, rz = i.z - j.z;
    const double r2 = rx * rx + ry * ry + rz * rz;
    const double rinv = 1.0 / sqrt(r2);
    const double nx = rx * rinv, ny = ry * rinv, nz = rz * rinv;
    const double nvi = nx * i.vx + ny * i.vy + nz * i.vz;
    const double nvj = nx * j.vx + ny * j.vy + nz * j.vz;
    const double vivi = i.vx * i.vx + i.vy * i.vy + i.vz * i.vz;
    const double vjvj = j.vx * j.vx + j.vy * j.vy + j.vz * j.vz;
    const double vivj = i.vx * j.vx + i.vy * j.vy + i.vz * j.vz;
    const double A = G * (5.0 * i.m + 4.0 * j.m) * rinv + 1.5 * nvj * nvj - vivi + 4.0 * vivj - 2.0 * vjvj;
    const double B = 4.0 * nvi - 3.0 * nvj;
    const double pref = G * j.m * inv_c2 * (rinv * rinv);
    fx += pref * (nx * A + B * (i.vx - j.vx));
    fy += pref * (ny * A + B * (i.vy - j.vy));
    fz += pref * (nz * A + B * (i.vz - j.vz));
}

__global__ void pn1_flag_kernel(int n_bh, const int32_t* __restrict__ bh_idx, unsigned char* __restrict__ is_bh) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b < n_bh) is_bh[bh_idx[b]] = 1;
}

// every particle i <- all BHs j != i (BH records staged through shared memory)
constexpr int PN_THREADS = 128;
__global__ void __launch_bounds__(PN_THREADS)
pn1_from_bh_kernel(int n, int n_bh, const int32_t* __restrict__ bh_idx, const double* __restrict__ pos,
                   const double* __restrict__ vel, const double* __restrict__ mass,
                   const int32_t* __restrict__ subsys, double G, double inv_c2, double* __restrict__ out) {
    __shared__ Body sb[PN_THREADS];
    __shared__ int sid[PN_THREADS];
    __shared__ int ssub[PN_THREADS];
    const int i = blockIdx.x * PN_THREADS + threadIdx.x;
    const int ii = i < n ? i : n - 1;
    const Body me = load_body(pos, vel, mass, ii);
    const int my_sub = subsys ? sink_code(subsys, ii) : -2;
    double fx = 0.0, fy = 0.0, fz = 0.0;
    for (int b0 = 0; b0 < n_bh; b0 += PN_THREADS) {
        const int b = b0 + threadIdx.x;
        if (b < n_bh) {
            sid[threadIdx.x] = bh_idx[b];
            sb[threadIdx.x] = load_body(pos, vel, mass, bh_idx[b]);
            ssub[threadIdx.x] = src_code(subsys, bh_idx[b]);
        }
        __syncthreads();
        const int cnt = min(PN_THREADS, n_bh - b0);
        for (int q = 0; q < cnt; ++q)
            if (sid[q] != ii && ssub[q] != my_sub) pn1_pair(me, sb[q], G, inv_c2, fx, fy, fz);
        __syncthreads();
    }
    if (i < n) { out[3 * (size_t)i] = fx; out[3 * (size_t)i + 1] = fy; out[3 * (size_t)i + 2] = fz; }
}

// each BH b <- all non-BH particles of one chunk; deterministic block reduction
constexpr int PN_RED_THREADS = 256;
__global__ void __launch_bounds__(PN_RED_THREADS)
pn1_on_bh_kernel(int n, int chunk, const int32_t* __restrict__ bh_idx, const unsigned char* __restrict__ is_bh,
                 const double* __restrict__ pos, const double* __restrict__ vel, const double* __restrict__ mass,
                 const int32_t* __restrict__ subsys, double G, double inv_c2,
                 double* __restrict__ partial /*[n_bh][n_chunks][3]*/) {
    __shared__ double red[3][PN_RED_THREADS / 32];
    const int b = blockIdx.y;
    const Body me = load_body(pos, vel, mass, bh_idx[b]);
    const int my_sub = subsys ? sink_code(subsys, bh_idx[b]) : -2;
    const int j0 = blockIdx.x * chunk, j1 = min(j0 + chunk, n);
    double fx = 0.0, fy = 0.0, fz = 0.0;
    for (int j = j0 + threadIdx.x; j < j1; j += PN_RED_THREADS) {
        if (is_bh[j] || src_code(subsys, j) == my_sub) continue;
        const Body o = load_body(pos, vel, mass, j);
        pn1_pair(me, o, G, inv_c2, fx, fy, fz);
    }
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        fx += __shfl_down_sync(0xffffffffu, fx, off);
        fy += __shfl_down_sync(0xffffffffu, fy, off);
        fz += __shfl_down_sync(0xffffffffu, fz, off);
    }
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) { red[0][warp] = fx; red[1][warp] = fy; red[2][warp] = fz; }
    __syncthreads();
    if (threadIdx.x == 0) {
        double sx = 0.0, sy = 0.0, sz = 0.0;
        for (int w = 0; w < PN_RED_THREADS / 32; ++w) { sx += red[0][w]; sy += red[1][w]; sz += red[2][w]; }
        double* o = partial + 3 * ((size_t)b * gridDim.x + blockIdx.x);
        o[0] = sx; o[1] = sy; o[2] = sz;
    }
}

__global__ void pn1_bh_finalize_kernel(int n_bh, int n_chunks, const int32_t* __restrict__ bh_idx,
                                       const double* __restrict__ partial, double* __restrict__ out) {
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= n_bh) return;
    double sx = 0.0, sy = 0.0, sz = 0.0;
    for (int c = 0; c < n_chunks; ++c) {
        const double* p = partial + 3 * ((size_t)b * n_chunks + c);
        sx += p[0]; sy += p[1]; sz += p[2];
    }
    double* o = out + 3 * (size_t)bh_idx[b];
    o[0] += sx; o[1] += sy; o[2] += sz;
}

}  // namespace
