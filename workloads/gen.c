/*
 * workloads/gen.c -- seeded, counter-based synthetic INPUT generators.
 *
 * This module serves both the CUDA path's harness and the CPU oracle's harness
 * and therefore holds NONE of the method's arithmetic (no put/get/AMO/collective
 * logic, no ordering logic): it only produces input arrays that are pure
 * functions of (seed, stream, index).  Recipes: SURVEY.md Appendix D; the
 * distributions are the ones BASELINE.json's configs name.
 *
 * Every output element depends only on its own index, so the OpenMP loops are
 * deterministic regardless of thread count.
 */
#include <math.h>
#include <stdint.h>
#include <string.h>

/* 64-bit mix of (seed, stream, i): two SplitMix64-style finaliser rounds. */
static inline uint64_t fin64(uint64_t x) {
    x ^= x >> 30; x *= 0xBF58476D1CE4E5B9ull;
    x ^= x >> 27; x *= 0x94D049BB133111EBull;
    x ^= x >> 31;
    return x;
}
static inline uint64_t mix64(uint64_t seed, uint64_t stream, uint64_t i) {
    uint64_t x = fin64(seed * 0xD1342543DE82EF95ull + stream * 0x9E3779B97F4A7C15ull + 0x2545F4914F6CDD1Dull);
    return fin64(x ^ (i * 0x9E3779B97F4A7C15ull + 0x632BE59BD9B4E019ull));
}
static inline uint64_t mulhi64(uint64_t a, uint64_t b) {
    return (uint64_t)(((unsigned __int128)a * b) >> 64);
}

uint64_t wl_mix64(uint64_t seed, uint64_t stream, uint64_t i) { return mix64(seed, stream, i); }

/* raw 64-bit words */
void wl_fill_u64(uint64_t *out, uint64_t n, uint64_t seed, uint64_t stream, uint64_t i0) {
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < (int64_t)n; ++k) out[k] = mix64(seed, stream, i0 + (uint64_t)k);
}

/* uniform integers in [lo, lo+range) by multiply-high (range >= 1) */
void wl_fill_uniform_i64(int64_t *out, uint64_t n, int64_t lo, uint64_t range,
                         uint64_t seed, uint64_t stream, uint64_t i0) {
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < (int64_t)n; ++k)
        out[k] = lo + (int64_t)mulhi64(mix64(seed, stream, i0 + (uint64_t)k), range);
}
void wl_fill_uniform_i32(int32_t *out, uint64_t n, int32_t lo, uint32_t range,
                         uint64_t seed, uint64_t stream, uint64_t i0) {
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < (int64_t)n; ++k)
        out[k] = lo + (int32_t)mulhi64(mix64(seed, stream, i0 + (uint64_t)k), (uint64_t)range);
}

/* uniform [0,1) doubles: top 53 bits * 2^-53 */
void wl_fill_uniform_f64(double *out, uint64_t n, uint64_t seed, uint64_t stream, uint64_t i0) {
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < (int64_t)n; ++k)
        out[k] = (double)(mix64(seed, stream, i0 + (uint64_t)k) >> 11) * 0x1.0p-53;
}

/* N(0,1) by Box-Muller in fp64 (host only: payload bits are inputs) */
static inline double normal01(uint64_t seed, uint64_t stream, uint64_t i) {
    double u1 = ((double)(mix64(seed, stream, 2 * i) >> 11) + 1.0) * 0x1.0p-53;   /* (0,1] */
    double u2 = (double)(mix64(seed, stream, 2 * i + 1) >> 11) * 0x1.0p-53;       /* [0,1) */
    return sqrt(-2.0 * log(u1)) * cos(6.283185307179586476925286766559 * u2);
}
void wl_fill_normal_f32(float *out, uint64_t n, uint64_t seed, uint64_t stream, uint64_t i0) {
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < (int64_t)n; ++k) out[k] = (float)normal01(seed, stream, i0 + (uint64_t)k);
}
/* bf16 bit patterns, round-to-nearest-even from the fp32 value */
void wl_fill_normal_bf16(uint16_t *out, uint64_t n, uint64_t seed, uint64_t stream, uint64_t i0) {
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < (int64_t)n; ++k) {
        float f = (float)normal01(seed, stream, i0 + (uint64_t)k);
        uint32_t b; memcpy(&b, &f, 4);
        b += 0x7FFFu + ((b >> 16) & 1u);
        out[k] = (uint16_t)(b >> 16);
    }
}

/*
 * RMAT edge list: for edge e and level l the quadrant is
 * chosen by comparing the top 32 bits of mix64(seed, l, e) with integer
 * thresholds ta = floor(a*2^32), tab = floor((a+b)*2^32), tabc = floor((a+b+c)*2^32).
 * No noise, no relabelling, duplicates and self loops kept.
 */
void wl_rmat_edges(uint32_t *u_out, uint32_t *v_out, uint64_t n_edges, int scale,
                   uint32_t ta, uint32_t tab, uint32_t tabc, uint64_t seed, uint64_t e0) {
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < (int64_t)n_edges; ++k) {
        uint64_t e = e0 + (uint64_t)k;
        uint32_t u = 0, v = 0;
        for (int l = 0; l < scale; ++l) {
            uint32_t r = (uint32_t)(mix64(seed, (uint64_t)l, e) >> 32);
            uint32_t ub, vb;
            if (r < ta)        { ub = 0; vb = 0; }
            else if (r < tab)  { ub = 0; vb = 1; }
            else if (r < tabc) { ub = 1; vb = 0; }
            else               { ub = 1; vb = 1; }
            u = (u << 1) | ub;
            v = (v << 1) | vb;
        }
        u_out[k] = u; v_out[k] = v;
    }
}
