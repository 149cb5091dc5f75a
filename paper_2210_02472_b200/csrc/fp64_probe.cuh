// fp64_probe.cuh - measurement aid: register-only FP64 chains that measure the FP64-pipe peak.
// Part of the single translation unit bifrost.cu (see its header and DESIGN.md); not a public header.
#pragma once

namespace {

// ----------------------------------------------------------------------------------------
// Measurement aid: register-only FP64 chains (no memory traffic), to MEASURE the FP64-pipe peak
// that bench.py's roofline quotes next to the derived 64 lanes/clk/SM figure.
//   MIX 0: 8 independent DFMA chains per thread (pure DFMA peak).
//   MIX 1: per 15 instructions 3 DADD + 9 DFMA + 3 DMUL (the acc pair's instruction mix).
// ----------------------------------------------------------------------------------------
constexpr int PROBE_THREADS = 128;
constexpr int PROBE_CHAINS = 8;
//   MIX 2: DFMA with three DISTINCT register operands, x = fma(y, z, x) (no reuse possible).
//   MIX 3: the pair kernels' accumulate pattern: groups of three DFMAs sharing one operand,
//          x0 = fma(w, y0, x0); x1 = fma(w, y1, x1); x2 = fma(w, y2, x2).
// MIX 2 and 3 show the register-file operand limit (one 64-bit operand per clock per SM
// sub-partition): 2/3 and 6/7 of the MIX 0 rate.
template <int MIX>
__global__ void __launch_bounds__(PROBE_THREADS, 4)
fp64_probe_kernel(int iters, double b, double c, const double* __restrict__ in, double* __restrict__ sink) {
    double a[PROBE_CHAINS];
#pragma unroll
    for (int k = 0; k < PROBE_CHAINS; ++k) a[k] = 1.0 + 1e-9 * (double)(threadIdx.x + k);
    if (MIX == 2 || MIX == 3) {
        // operands that the compiler cannot fold: loaded from memory (all 1 + O(1e-6))
        double x[12], y[12], w[4];
#pragma unroll
        for (int k = 0; k < 12; ++k) { x[k] = in[threadIdx.x + 128 * k]; y[k] = in[threadIdx.x + 128 * (k + 12)]; }
#pragma unroll
        for (int k = 0; k < 4; ++k) w[k] = in[threadIdx.x + 128 * (k + 24)];
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int g = 0; g < 4; ++g) {
                if (MIX == 2) {
                    x[3 * g] = fma(y[3 * g], w[g], x[3 * g]);
                    x[3 * g + 1] = fma(y[3 * g + 1], y[(3 * g + 5) % 12], x[3 * g + 1]);
                    x[3 * g + 2] = fma(y[3 * g + 2], y[(3 * g + 7) % 12], x[3 * g + 2]);
                } else {
                    x[3 * g] = fma(w[g], y[3 * g], x[3 * g]);
                    x[3 * g + 1] = fma(w[g], y[3 * g + 1], x[3 * g + 1]);
                    x[3 * g + 2] = fma(w[g], y[3 * g + 2], x[3 * g + 2]);
                }
            }
        }
#pragma unroll
        for (int k = 0; k < 12; ++k) a[k % PROBE_CHAINS] += x[k] + y[k];
    } else {
        for (int it = 0; it < iters; ++it) {
            if (MIX == 0) {
#pragma unroll
                for (int u = 0; u < 4; ++u)
#pragma unroll
                    for (int k = 0; k < PROBE_CHAINS; ++k) a[k] = fma(a[k], b, c);          // 32 DFMA
            } else {
#pragma unroll
                for (int k = 0; k < PROBE_CHAINS; ++k) {                                     // 8 x 15 instructions
                    double x = a[k];
                    x = x + c; x = fma(x, b, c); x = fma(x, b, c); x = x * b; x = fma(x, b, c);
                    x = x + c; x = fma(x, b, c); x = fma(x, b, c); x = x * b; x = fma(x, b, c);
                    x = x + c; x = fma(x, b, c); x = fma(x, b, c); x = x * b; x = fma(x, b, c);
                    a[k] = x;
                }
            }
        }
    }
    double s = 0.0;
#pragma unroll
    for (int k = 0; k < PROBE_CHAINS; ++k) s += a[k];
    if (s == 123.456) sink[blockIdx.x * blockDim.x + threadIdx.x] = s;   // never true; keeps the chains alive
}

}  // namespace
