/*
 * pfsm_gen.c -- seeded synthetic inputs for the PFSM path.
 *
 * This module only DRAWS NUMBERS.  It holds none of the method's arithmetic
 * (no partition, no eigensolve, no iteration, no orthonormalization): it is
 * the one piece of code that both the CPU oracle's tests and the CUDA path's
 * tests/bench are allowed to share.
 *
 * Counter-based generator: entry `idx` of stream `stream` under `seed` is a
 * pure function of (seed, stream, idx), so a matrix is reproducible whatever
 * the thread count or fill order.
 *
 *   key  = seed * 0x9E3779B97F4A7C15 + stream * 0xBF58476D1CE4E5B9 + idx      (mod 2^64)
 *   h1   = mix64(key)              h2 = mix64(key ^ 0xD6E8FEB86659FD93)
 *   mix64(z): z ^= z>>30; z *= 0xBF58476D1CE4E5B9; z ^= z>>27; z *= 0x94D049BB133111EB; z ^= z>>31
 *   u1   = ((h1 >> 11) + 0.5) * 2^-53  in (0,1);  u2 likewise from h2
 *   uniform(idx) = u1
 *   normal(idx)  = sqrt(-2 ln u1) * cos(2 pi u2)          (Box-Muller)
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>

static inline uint64_t mix64(uint64_t z) {
    z ^= z >> 30; z *= 0xBF58476D1CE4E5B9ULL;
    z ^= z >> 27; z *= 0x94D049BB133111EBULL;
    z ^= z >> 31;
    return z;
}
static inline uint64_t key_of(uint64_t seed, uint64_t stream, uint64_t idx) {
    return seed * 0x9E3779B97F4A7C15ULL + stream * 0xBF58476D1CE4E5B9ULL + idx;
}
static inline double u01(uint64_t h) { return ((double)(h >> 11) + 0.5) * (1.0 / 9007199254740992.0); }

static inline double gen_uniform1(uint64_t seed, uint64_t stream, uint64_t idx) {
    return u01(mix64(key_of(seed, stream, idx)));
}
static inline double gen_normal1(uint64_t seed, uint64_t stream, uint64_t idx) {
    uint64_t k = key_of(seed, stream, idx);
    double u1 = u01(mix64(k));
    double u2 = u01(mix64(k ^ 0xD6E8FEB86659FD93ULL));
    return sqrt(-2.0 * log(u1)) * cos(6.283185307179586476925286766559 * u2);
}

/* out[k] = uniform(idx0 + k), k < n */
void pfsm_gen_uniform(uint64_t seed, uint64_t stream, uint64_t idx0, int64_t n, double* out) {
    for (int64_t k = 0; k < n; ++k) out[k] = gen_uniform1(seed, stream, idx0 + (uint64_t)k);
}
/* out[k] = normal(idx0 + k), k < n */
void pfsm_gen_normal(uint64_t seed, uint64_t stream, uint64_t idx0, int64_t n, double* out) {
    for (int64_t k = 0; k < n; ++k) out[k] = gen_normal1(seed, stream, idx0 + (uint64_t)k);
}

/*
 * out (N x N, ld = N; the matrix is exactly symmetric so row/column-major is immaterial):
 *   out[i][j] = out[j][i] = amp * normal(i*N + j) * exp(-|i-j| / width)   for i <= j
 *   out[i][i] += diag[i]                                                   (diag may be NULL)
 */
void pfsm_gen_banded_symmetric(int64_t N, const double* diag, double amp, double width,
                               uint64_t seed, uint64_t stream, double* out) {
#pragma omp parallel for schedule(dynamic, 16)
    for (int64_t i = 0; i < N; ++i) {
        for (int64_t j = i; j < N; ++j) {
            double g = gen_normal1(seed, stream, (uint64_t)(i * N + j));
            double e = amp * g * exp(-(double)(j - i) / width);
            if (i == j && diag) e += diag[i];
            out[i * N + j] = e;
            out[j * N + i] = e;
        }
    }
}
