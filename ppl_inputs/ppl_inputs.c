/*
 * ppl_inputs.c -- seeded, counter-based generators for the synthetic pp-ladder inputs.
 *
 * This module holds NONE of the method's arithmetic: it only fills host buffers that the CPU
 * oracle (oracle/) and the CUDA path (paper_2603_20912_b200/) both read, so the two sides see
 * bit-identical inputs by construction.  Neither of them shares any other code.
 *
 * Recipe (BASELINE.json "configs"; readings A9-A12 of DESIGN.md; the paper itself only says the
 * contraction benchmark used "randomly generated numbers"):
 *   L [P,a,c] = L [P,c,a]   = g * exp(-3 P / nchol),  g ~ N(0,1),   P zero-based
 *   t2[i,j,a,b] = t2[j,i,b,a] = 0.1 * g               (N(0,1e-2): variance 1e-2, sigma 0.1)
 * Symmetrisation is by MIRRORING a canonical entry (a<=c, resp. (i,a)<=(j,b)), not by averaging,
 * so every entry has exactly the stated marginal distribution.
 *
 * g is drawn from a counter-based stream: two splitmix64 outputs per canonical linear index ->
 * two uniforms in (0,1) -> Box-Muller.  Order-free, so the fill is parallel (OpenMP).
 *
 * mode: 0 = normal (the recipe above), 1 = small integers in {-2,..,2} (no decay, no 0.1 scale:
 *           every product and partial sum of the ladder is then an exact integer in binary64),
 *       2 = uniform on (0,1) (ppl_inputs_fill_vec only: index sampling for tests),
 * symmetric: 1 = mirror as above, 0 = every entry drawn from its own linear index.
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>

static inline uint64_t splitmix64(uint64_t z) {
    z += 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

static inline uint64_t stream_key(uint64_t seed, uint64_t tag) {
    return splitmix64(splitmix64(seed) ^ (tag * 0xD6E8FEB86659FD93ull));
}

static inline double u01(uint64_t h) { /* (0,1), 53 bits */
    return ((double)(h >> 11) + 0.5) * (1.0 / 9007199254740992.0);
}

static inline double draw(uint64_t key, uint64_t idx, int mode) {
    uint64_t h1 = splitmix64(key + 2 * idx);
    if (mode == 1) return (double)((int)(h1 % 5ull) - 2);
    if (mode == 2) return u01(h1);
    uint64_t h2 = splitmix64(key + 2 * idx + 1);
    double u1 = u01(h1), u2 = u01(h2);
    return sqrt(-2.0 * log(u1)) * cos(6.283185307179586476925286766559 * u2);
}

/* L[nchol][nvirt][nvirt], row-major. */
void ppl_inputs_fill_L(double *L, int nvirt, int nchol, uint64_t seed, int symmetric, int mode) {
    const uint64_t key = stream_key(seed, 1);
    const int64_t v = nvirt;
#pragma omp parallel for schedule(static)
    for (int64_t P = 0; P < nchol; ++P) {
        const double decay = (mode == 1) ? 1.0 : exp(-3.0 * (double)P / (double)nchol);
        for (int64_t a = 0; a < v; ++a)
            for (int64_t c = 0; c < v; ++c) {
                int64_t lo = a, hi = c;
                if (symmetric && lo > hi) { lo = c; hi = a; }
                uint64_t idx = (uint64_t)((P * v + lo) * v + hi);
                L[(P * v + a) * v + c] = draw(key, idx, mode) * decay;
            }
    }
}

/* t2[nocc][nocc][nvirt][nvirt], row-major. */
void ppl_inputs_fill_t2(double *t2, int nocc, int nvirt, uint64_t seed, int symmetric, int mode) {
    const uint64_t key = stream_key(seed, 2);
    const int64_t o = nocc, v = nvirt, ov = o * v;
    const double scale = (mode == 1) ? 1.0 : 0.1;
#pragma omp parallel for collapse(2) schedule(static)
    for (int64_t i = 0; i < o; ++i)
        for (int64_t j = 0; j < o; ++j)
            for (int64_t a = 0; a < v; ++a)
                for (int64_t b = 0; b < v; ++b) {
                    int64_t p = i * v + a, q = j * v + b;
                    if (symmetric && p > q) { int64_t t = p; p = q; q = t; }
                    uint64_t idx = (uint64_t)(p * ov + q);
                    t2[((i * o + j) * v + a) * v + b] = draw(key, idx, mode) * scale;
                }
}

/* plain N(0,1) / integer vector for test vectors (tag chosen by the caller, >= 16). */
void ppl_inputs_fill_vec(double *x, int64_t n, uint64_t seed, uint64_t tag, int mode) {
    const uint64_t key = stream_key(seed, tag);
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < n; ++k) x[k] = draw(key, (uint64_t)k, mode);
}
