/* cpu_fast.c - a plain, reasonably fast CPU restatement of acc (Eq. 6) and the grad sum
 * (Eq. 9) for bench.py's `cpu_fast` line ONLY (the parity oracle is deliberately
 * slow - compensated sums, one IEEE sqrt + division per pair at -O2 - so a GPU/oracle ratio flatters the GPU).
 *
 * NOT the parity oracle and never used for a parity decision: it is itself pinned to the oracle at 1e-12
 * (tests/test_oracle_cpu_fast.py).  Uncompensated sums, sources gathered once into SoA arrays, the inner loop
 * over sources written so that gcc vectorises it (AVX2 + FMA: vsqrtpd / vdivpd, four pairs per instruction),
 * OpenMP over sinks.  Same conventions as the oracle: r_ji = r_j - r_i, the self pair skipped by id, Plummer
 * softening, outputs compact (row k = k-th sink).  Shares no code with the CUDA path.
 * Build: gcc -O3 -mavx2 -mfma -fopenmp -fPIC -shared (no -ffast-math: sqrt and division stay IEEE). */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

static int64_t pid(const int32_t* idx, int64_t k) { return idx ? (int64_t)idx[k] : k; }

/* gather the sources into x[], y[], z[], m[] (+ ax, ay, az); ids[] keeps the particle id for the self test */
static int gather(int64_t n_src, const int32_t* src_idx, const double* pos, const double* mass, const double* aux,
                  double** buf, int64_t** ids) {
    const int nf = aux ? 7 : 4;
    *buf = (double*)malloc(sizeof(double) * (size_t)nf * (size_t)(n_src > 0 ? n_src : 1));
    *ids = (int64_t*)malloc(sizeof(int64_t) * (size_t)(n_src > 0 ? n_src : 1));
    if (!*buf || !*ids) return -1;
    for (int64_t l = 0; l < n_src; ++l) {
        const int64_t j = pid(src_idx, l);
        (*ids)[l] = j;
        (*buf)[0 * n_src + l] = pos[3 * j]; (*buf)[1 * n_src + l] = pos[3 * j + 1]; (*buf)[2 * n_src + l] = pos[3 * j + 2];
        (*buf)[3 * n_src + l] = mass[j];
        if (aux) { (*buf)[4 * n_src + l] = aux[3 * j]; (*buf)[5 * n_src + l] = aux[3 * j + 1]; (*buf)[6 * n_src + l] = aux[3 * j + 2]; }
    }
    return 0;
}

int cpu_fast_acc(int64_t n, const double* pos, const double* mass, const int32_t* sink_idx, int64_t n_sink,
                 const int32_t* src_idx, int64_t n_src, double G, double eps, double* out) {
    (void)n;
    double* b; int64_t* ids;
    if (gather(n_src, src_idx, pos, mass, 0, &b, &ids)) return -1;
    const double *x = b, *y = b + n_src, *z = b + 2 * n_src, *m = b + 3 * n_src;
    const double eps2 = eps * eps;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t k = 0; k < n_sink; ++k) {
        const int64_t i = pid(sink_idx, k);
        const double xi = pos[3 * i], yi = pos[3 * i + 1], zi = pos[3 * i + 2];
        double sx = 0.0, sy = 0.0, sz = 0.0;
#pragma omp simd reduction(+ : sx, sy, sz)
        for (int64_t l = 0; l < n_src; ++l) {
            const double dx = x[l] - xi, dy = y[l] - yi, dz = z[l] - zi;
            const double s2 = dx * dx + dy * dy + dz * dz + eps2;
            /* the self pair (and only it, by id) is dropped: weight 0 instead of 0/0 */
            const double w = ids[l] == i ? 0.0 : m[l] / (s2 * sqrt(s2));
            sx += w * dx; sy += w * dy; sz += w * dz;
        }
        out[3 * k] = G * sx; out[3 * k + 1] = G * sy; out[3 * k + 2] = G * sz;
    }
    free(b); free(ids);
    return 0;
}

int cpu_fast_grad(int64_t n, const double* pos, const double* mass, const double* acc, const int32_t* sink_idx,
                  int64_t n_sink, const int32_t* src_idx, int64_t n_src, double G, double eps, double* out) {
    (void)n;
    double* b; int64_t* ids;
    if (gather(n_src, src_idx, pos, mass, acc, &b, &ids)) return -1;
    const double *x = b, *y = b + n_src, *z = b + 2 * n_src, *m = b + 3 * n_src;
    const double *ax = b + 4 * n_src, *ay = b + 5 * n_src, *az = b + 6 * n_src;
    const double eps2 = eps * eps;
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t k = 0; k < n_sink; ++k) {
        const int64_t i = pid(sink_idx, k);
        const double xi = pos[3 * i], yi = pos[3 * i + 1], zi = pos[3 * i + 2];
        const double axi = acc[3 * i], ayi = acc[3 * i + 1], azi = acc[3 * i + 2];
        double sx = 0.0, sy = 0.0, sz = 0.0;
#pragma omp simd reduction(+ : sx, sy, sz)
        for (int64_t l = 0; l < n_src; ++l) {
            const double dx = x[l] - xi, dy = y[l] - yi, dz = z[l] - zi;
            const double bx = ax[l] - axi, by = ay[l] - ayi, bz = az[l] - azi;
            const double s2 = dx * dx + dy * dy + dz * dz + eps2;
            const double w = ids[l] == i ? 0.0 : m[l] / (s2 * sqrt(s2));        /* m_j / s^3 */
            const double q = 3.0 * (bx * dx + by * dy + bz * dz) / (ids[l] == i ? 1.0 : s2);
            sx += w * (bx - q * dx); sy += w * (by - q * dy); sz += w * (bz - q * dz);
        }
        out[3 * k] = G * sx; out[3 * k + 1] = G * sy; out[3 * k + 2] = G * sz;
    }
    free(b); free(ids);
    return 0;
}
