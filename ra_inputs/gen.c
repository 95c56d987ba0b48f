/*
 * ra_inputs/gen.c -- seeded synthetic input generator (host only).
 *
 * This module is the ONLY code shared by the CPU oracle side and the CUDA side
 * of the tests/bench: it fills HOST buffers that are then handed, bit for bit,
 * to both.  It holds none of the method's arithmetic (no GEMM, no reduction,
 * no permutation) -- only a counter-based PRNG and value shaping.
 *
 * Recipe:
 *   h(seed, stream, i) = splitmix64_finalise(key(seed, stream) + (i+1) * GOLDEN)
 *   - counter based: element i depends only on (seed, stream, i), so generation
 *     is order independent and parallel.
 *   normal  : Box-Muller on two 24-bit uniforms taken from one 64-bit draw,
 *             computed in double, rounded to float, then to bf16 (RNE).
 *   uniform : 24-bit integer u -> (float)u * 2^-23 - 1  in [-1, 1), exact in fp32.
 *   bits    : the raw 64-bit draw (alltoall payload: arbitrary bit patterns,
 *             NaN encodings included).
 *   smallint: integers uniform in [lo, hi] as bf16 (exact) -- the integer-exact
 *             GEMM pin.
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <string.h>

#define RA_GOLDEN 0x9E3779B97F4A7C15ull

static inline uint64_t mix64(uint64_t z) {
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

static inline uint64_t stream_key(uint64_t seed, uint64_t stream) {
    return mix64(seed + RA_GOLDEN) ^ mix64(stream * RA_GOLDEN + 0x632BE59BD9B4E019ull);
}

static inline uint64_t draw(uint64_t key, uint64_t i) {
    return mix64(key + (i + 1) * RA_GOLDEN);
}

static inline uint16_t f32_to_bf16_rne_gen(float f) {
    uint32_t u;
    memcpy(&u, &f, 4);
    if ((u & 0x7FFFFFFFu) > 0x7F800000u) return (uint16_t)((u >> 16) | 0x0040u); /* quiet NaN */
    u += 0x7FFFu + ((u >> 16) & 1u);
    return (uint16_t)(u >> 16);
}

/* raw 64-bit draws */
void ra_inputs_bits_u64(uint64_t* out, size_t n, uint64_t seed, uint64_t stream) {
    const uint64_t key = stream_key(seed, stream);
#pragma omp parallel for schedule(static)
    for (long long i = 0; i < (long long)n; ++i) out[i] = draw(key, (uint64_t)i);
}

/* U[-1, 1) fp32, 24-bit resolution */
void ra_inputs_uniform_f32(float* out, size_t n, uint64_t seed, uint64_t stream) {
    const uint64_t key = stream_key(seed, stream);
#pragma omp parallel for schedule(static)
    for (long long i = 0; i < (long long)n; ++i) {
        const uint32_t u = (uint32_t)(draw(key, (uint64_t)i) >> 40); /* 24 bits */
        out[i] = (float)u * (1.0f / 8388608.0f) - 1.0f;
    }
}

/* N(0,1) rounded to bf16 (stored as uint16 bit patterns) */
void ra_inputs_normal_bf16(uint16_t* out, size_t n, uint64_t seed, uint64_t stream) {
    const uint64_t key = stream_key(seed, stream);
    const double two_pi = 6.283185307179586476925286766559;
#pragma omp parallel for schedule(static)
    for (long long i = 0; i < (long long)n; ++i) {
        const uint64_t h = draw(key, (uint64_t)i);
        const double u1 = ((double)(h >> 40) + 1.0) * (1.0 / 16777216.0);         /* (0, 1] */
        const double u2 = (double)((h >> 16) & 0xFFFFFFull) * (1.0 / 16777216.0); /* [0, 1) */
        const double z = sqrt(-2.0 * log(u1)) * cos(two_pi * u2);
        out[i] = f32_to_bf16_rne_gen((float)z);
    }
}

/* integers uniform in [lo, hi] (|lo|,|hi| <= 128) as bf16 bit patterns */
void ra_inputs_smallint_bf16(uint16_t* out, size_t n, uint64_t seed, uint64_t stream, int lo, int hi) {
    const uint64_t key = stream_key(seed, stream);
    const uint64_t span = (uint64_t)(hi - lo + 1);
#pragma omp parallel for schedule(static)
    for (long long i = 0; i < (long long)n; ++i) {
        const uint64_t h = draw(key, (uint64_t)i);
        const int v = lo + (int)((h >> 33) % span);
        out[i] = f32_to_bf16_rne_gen((float)v);
    }
}

/* tagged alltoall payload: word w of chunk (i,j) = i<<56 | j<<48 | w  (every
 * misrouted or shifted 8-byte word is identifiable). */
void ra_inputs_tagged_chunks_u64(uint64_t* out, int P, size_t words_per_chunk) {
#pragma omp parallel for schedule(static) collapse(2)
    for (int i = 0; i < P; ++i)
        for (int j = 0; j < P; ++j) {
            uint64_t* c = out + ((size_t)i * P + j) * words_per_chunk;
            for (size_t w = 0; w < words_per_chunk; ++w)
                c[w] = ((uint64_t)i << 56) | ((uint64_t)j << 48) | (uint64_t)w;
        }
}
