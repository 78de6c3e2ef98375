/*
 * ibp_datagen.c -- seeded, counter-based synthetic input generators.
 *
 * This module is the ONE piece shared by the oracle tests and the CUDA path:
 * it produces the inputs both sides consume.  It holds none of the method's
 * arithmetic (no masks, no packing, no decoding) -- only value distributions
 * with the shapes of BASELINE.json `configs` (recipe in DESIGN.md section 4).
 *
 * Every element i of a stream is a pure function of (seed, i): the generators
 * are reproducible for any thread count and any chunking, so a test can
 * regenerate just the rows it samples from a multi-GB table.
 *
 *   u64 h(seed, c)   = splitmix64 finaliser of (seed * GOLDEN + c)
 *   uniform  U(0,1)  = (h >> 40 + 0.5) * 2^-24      (24-bit, never 0 or 1)
 *   normal   N(0,1)  = Box-Muller on two uniforms drawn from counters 2j, 2j+1;
 *                      elements 2j and 2j+1 take the cos and the sin branch.
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC ibp_datagen.c -o libibp_datagen.so -lm
 */
#include <math.h>
#include <stdint.h>
#include <string.h>

#define GOLDEN 0x9E3779B97F4A7C15ull

static inline uint64_t mix64(uint64_t z) {
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}
static inline uint64_t h64(uint64_t seed, uint64_t c) { return mix64(mix64(seed * GOLDEN + 0x1234567ull) + c * GOLDEN); }
static inline float u01(uint64_t seed, uint64_t c) { return ((float)(h64(seed, c) >> 40) + 0.5f) * (1.0f / 16777216.0f); }

/* one standard normal for stream element i */
static inline float normal_at(uint64_t seed, uint64_t i) {
    uint64_t j = i >> 1;
    float u1 = u01(seed, 2 * j), u2 = u01(seed, 2 * j + 1);
    float r = sqrtf(-2.0f * logf(u1));
    float a = 6.28318530717958647692f * u2;
    return (i & 1) ? r * sinf(a) : r * cosf(a);
}

static inline uint16_t f32_to_bf16_rne(float f) {
    uint32_t u;
    memcpy(&u, &f, 4);
    if ((u & 0x7fffffffu) > 0x7f800000u) return (uint16_t)((u >> 16) | 0x40u); /* NaN stays NaN */
    u += 0x7fffu + ((u >> 16) & 1u);
    return (uint16_t)(u >> 16);
}

/* N(0, sigma) -> optional snap to multiples of `step` (round-to-nearest-even via rintf)
 * -> optional clip to [-clip, clip].  step <= 0 / clip <= 0 disable the stage.
 * `first` is the index of out[0] in the stream, so sub-ranges can be regenerated. */
void ibp_gen_normal_f32(float* out, uint64_t n, uint64_t seed, uint64_t first, float sigma, float step, float clip) {
    const float inv = step > 0 ? 1.0f / step : 0.0f;
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < (int64_t)n; ++k) {
        float x = sigma * normal_at(seed, first + (uint64_t)k);
        if (step > 0) x = rintf(x * inv) * step;
        if (clip > 0) x = x > clip ? clip : (x < -clip ? -clip : x);
        out[k] = x;
    }
}

/* U(lo, hi) -> optional snap to multiples of `step`. */
void ibp_gen_uniform_f32(float* out, uint64_t n, uint64_t seed, uint64_t first, float lo, float hi, float step) {
    const float inv = step > 0 ? 1.0f / step : 0.0f;
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < (int64_t)n; ++k) {
        float x = lo + (hi - lo) * u01(seed, first + (uint64_t)k);
        if (step > 0) x = rintf(x * inv) * step;
        out[k] = x;
    }
}

/* Bernoulli(p) as 0.0f / 1.0f (sparse binary bag-of-words rows). */
void ibp_gen_bernoulli_f32(float* out, uint64_t n, uint64_t seed, uint64_t first, float p) {
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < (int64_t)n; ++k) out[k] = u01(seed, first + (uint64_t)k) < p ? 1.0f : 0.0f;
}

/* N(0, sigma) rounded to bf16 (round-to-nearest-even). */
void ibp_gen_normal_bf16(uint16_t* out, uint64_t n, uint64_t seed, uint64_t first, float sigma) {
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < (int64_t)n; ++k) out[k] = f32_to_bf16_rne(sigma * normal_at(seed, first + (uint64_t)k));
}

/* Uniformly random bytes (every bit an independent fair coin). */
void ibp_gen_random_bytes(uint8_t* out, uint64_t n, uint64_t seed, uint64_t first) {
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < (int64_t)n; ++k) {
        uint64_t i = first + (uint64_t)k;
        out[k] = (uint8_t)(h64(seed, i >> 3) >> (8 * (i & 7)));
    }
}

/* Rows for the Fig. 7-style sweep: each row is `pattern` at the
 * positions where `fixed` has a 1 bit and a fair coin elsewhere.  `fixed` and
 * `pattern` are row_bytes long and are INPUTS chosen by the caller. */
void ibp_gen_rows_with_fixed_bits(uint8_t* out, uint64_t n_rows, uint32_t row_bytes, const uint8_t* fixed,
                                  const uint8_t* pattern, uint64_t seed, uint64_t first_row) {
#pragma omp parallel for schedule(static)
    for (int64_t r = 0; r < (int64_t)n_rows; ++r) {
        uint64_t base = (first_row + (uint64_t)r) * row_bytes;
        uint8_t* o = out + (uint64_t)r * row_bytes;
        for (uint32_t b = 0; b < row_bytes; ++b) {
            uint64_t i = base + b;
            uint8_t rnd = (uint8_t)(h64(seed, i >> 3) >> (8 * (i & 7)));
            o[b] = (uint8_t)((pattern[b] & fixed[b]) | (rnd & (uint8_t)~fixed[b]));
        }
    }
}

/* u64 hash stream, for id sampling done in Python (exposed so ids are also seeded here). */
void ibp_gen_u64(uint64_t* out, uint64_t n, uint64_t seed, uint64_t first) {
#pragma omp parallel for schedule(static)
    for (int64_t k = 0; k < (int64_t)n; ++k) out[k] = h64(seed, first + (uint64_t)k);
}
