// host_sha256.cpp -- production SHA-256 for the sub-frame hashes h_i.
// FIPS 180-4 compression function on the x86 SHA extensions (SHA-NI) when the CPU has them, portable
// 32-bit code otherwise; chosen at run time.  Shares nothing with oracle/.
#include "host.hpp"

#include <cstring>
#if defined(__x86_64__)
#include <immintrin.h>
#endif

namespace vh {

// FIPS 180-4 section 4.2.2: first 32 bits of the fractional parts of the cube roots of the first 64 primes.
alignas(64) static const uint32_t KT[64] = {
    0x428a2f98, 0x71374491, 0xb5c0fbcf, 0xe9b5dba5, 0x3956c25b, 0x59f111f1, 0x923f82a4, 0xab1c5ed5, 0xd807aa98,
    0x12835b01, 0x243185be, 0x550c7dc3, 0x72be5d74, 0x80deb1fe, 0x9bdc06a7, 0xc19bf174, 0xe49b69c1, 0xefbe4786,
    0x0fc19dc6, 0x240ca1cc, 0x2de92c6f, 0x4a7484aa, 0x5cb0a9dc, 0x76f988da, 0x983e5152, 0xa831c66d, 0xb00327c8,
    0xbf597fc7, 0xc6e00bf3, 0xd5a79147, 0x06ca6351, 0x14292967, 0x27b70a85, 0x2e1b2138, 0x4d2c6dfc, 0x53380d13,
    0x650a7354, 0x766a0abb, 0x81c2c92e, 0x92722c85, 0xa2bfe8a1, 0xa81a664b, 0xc24b8b70, 0xc76c51a3, 0xd192e819,
    0xd6990624, 0xf40e3585, 0x106aa070, 0x19a4c116, 0x1e376c08, 0x2748774c, 0x34b0bcb5, 0x391c0cb3, 0x4ed8aa4a,
    0x5b9cca4f, 0x682e6ff3, 0x748f82ee, 0x78a5636f, 0x84c87814, 0x8cc70208, 0x90befffa, 0xa4506ceb, 0xbef9a3f7,
    0xc67178f2};

static inline uint32_t ror(uint32_t x, int n) { return (x >> n) | (x << (32 - n)); }

static void compress_portable(uint32_t st[8], const uint8_t *p, size_t nblk) {
    for (; nblk; --nblk, p += 64) {
        uint32_t w[16];
        for (int t = 0; t < 16; ++t) {
            uint32_t v;
            std::memcpy(&v, p + 4 * t, 4);
            w[t] = __builtin_bswap32(v);
        }
        uint32_t a = st[0], b = st[1], c = st[2], d = st[3], e = st[4], f = st[5], g = st[6], h = st[7];
        for (int t = 0; t < 64; ++t) {
            if (t >= 16) {
                const uint32_t w15 = w[(t + 1) & 15], w2 = w[(t + 14) & 15];
                w[t & 15] += (ror(w15, 7) ^ ror(w15, 18) ^ (w15 >> 3)) + w[(t + 9) & 15] +
                             (ror(w2, 17) ^ ror(w2, 19) ^ (w2 >> 10));
            }
            const uint32_t t1 = h + (ror(e, 6) ^ ror(e, 11) ^ ror(e, 25)) + (g ^ (e & (f ^ g))) + KT[t] + w[t & 15];
            const uint32_t t2 = (ror(a, 2) ^ ror(a, 13) ^ ror(a, 22)) + ((a & b) | (c & (a | b)));
            h = g; g = f; f = e; e = d + t1; d = c; c = b; b = a; a = t1 + t2;
        }
        st[0] += a; st[1] += b; st[2] += c; st[3] += d; st[4] += e; st[5] += f; st[6] += g; st[7] += h;
    }
}

#if defined(__x86_64__)
// Four rounds per group g: the message quad W[4g..4g+3] is either loaded (g < 4) or produced from the previous
// four quads by SHA256MSG1 / SHA256MSG2; SHA256RNDS2 consumes W + K two rounds at a time with the state held as
// (ABEF, CDGH).
__attribute__((target("sha,sse4.1,ssse3"))) static void compress_shani(uint32_t st[8], const uint8_t *p,
                                                                       size_t nblk) {
    const __m128i bswap = _mm_set_epi64x(0x0c0d0e0f08090a0bLL, 0x0405060700010203LL);
    __m128i t = _mm_loadu_si128(reinterpret_cast<const __m128i *>(st));      // D C B A (high..low)
    __m128i s1 = _mm_loadu_si128(reinterpret_cast<const __m128i *>(st + 4));  // H G F E
    t = _mm_shuffle_epi32(t, 0xB1);                                          // C D A B
    s1 = _mm_shuffle_epi32(s1, 0x1B);                                        // E F G H
    __m128i s0 = _mm_alignr_epi8(t, s1, 8);                                  // A B E F
    s1 = _mm_blend_epi16(s1, t, 0xF0);                                       // C D G H
    for (; nblk; --nblk, p += 64) {
        const __m128i save0 = s0, save1 = s1;
        __m128i W[4];
#pragma GCC unroll 16
        for (int g = 0; g < 16; ++g) {
            if (g < 4) {
                W[g] = _mm_shuffle_epi8(_mm_loadu_si128(reinterpret_cast<const __m128i *>(p + 16 * g)), bswap);
            } else {
                __m128i x = _mm_sha256msg1_epu32(W[g & 3], W[(g + 1) & 3]);
                x = _mm_add_epi32(x, _mm_alignr_epi8(W[(g + 3) & 3], W[(g + 2) & 3], 4));
                W[g & 3] = _mm_sha256msg2_epu32(x, W[(g + 3) & 3]);
            }
            __m128i m = _mm_add_epi32(W[g & 3], _mm_load_si128(reinterpret_cast<const __m128i *>(KT + 4 * g)));
            s1 = _mm_sha256rnds2_epu32(s1, s0, m);
            m = _mm_shuffle_epi32(m, 0x0E);
            s0 = _mm_sha256rnds2_epu32(s0, s1, m);
        }
        s0 = _mm_add_epi32(s0, save0);
        s1 = _mm_add_epi32(s1, save1);
    }
    t = _mm_shuffle_epi32(s0, 0x1B);        // F E B A
    s1 = _mm_shuffle_epi32(s1, 0xB1);       // D C H G
    s0 = _mm_blend_epi16(t, s1, 0xF0);      // D C B A
    s1 = _mm_alignr_epi8(s1, t, 8);         // H G F E
    _mm_storeu_si128(reinterpret_cast<__m128i *>(st), s0);
    _mm_storeu_si128(reinterpret_cast<__m128i *>(st + 4), s1);
}
#endif

bool cpu_has_shani() {
#if defined(__x86_64__)
    static const bool v = __builtin_cpu_supports("sha") && __builtin_cpu_supports("sse4.1") &&
                          __builtin_cpu_supports("ssse3");
    return v;
#else
    return false;
#endif
}

void sha256(const uint8_t *msg, size_t len, uint8_t out[32], bool allow_simd) {
    // FIPS 180-4 section 5.3.3 initial hash value
    uint32_t st[8] = {0x6a09e667, 0xbb67ae85, 0x3c6ef372, 0xa54ff53a, 0x510e527f, 0x9b05688c, 0x1f83d9ab, 0x5be0cd19};
    void (*compress)(uint32_t *, const uint8_t *, size_t) = compress_portable;
#if defined(__x86_64__)
    if (allow_simd && cpu_has_shani()) compress = compress_shani;
#endif
    const size_t full = len / 64, rem = len % 64;
    if (full) compress(st, msg, full);
    // section 5.1.1 padding: 1 bit, zeros, 64-bit big-endian bit length
    uint8_t tail[128] = {0};
    if (rem) std::memcpy(tail, msg + 64 * full, rem);
    tail[rem] = 0x80;
    const size_t tl = rem < 56 ? 64 : 128;
    const uint64_t bits = (uint64_t)len * 8u;
    for (int i = 0; i < 8; ++i) tail[tl - 1 - i] = (uint8_t)(bits >> (8 * i));
    compress(st, tail, tl / 64);
    for (int i = 0; i < 8; ++i) {
        const uint32_t v = __builtin_bswap32(st[i]);
        std::memcpy(out + 4 * i, &v, 4);
    }
}

}  // namespace vh
