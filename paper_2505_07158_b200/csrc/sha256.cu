// sha256.cu -- device-side sub-frame hashing: h_m = SHA-256(f_m) for the n row bands of each
// frame of a batch and H = xor_m h_m, on the frames that were uploaded for the cipher kernels anyway.
//
// SHA-256 (FIPS 180-4) is serial inside a message, so the parallelism is one thread per (frame, band): n x batch
// independent message streams (256 at n = 32, batch = 8), one warp per CTA so that the warps spread over as many SMs as
// possible.  A thread walks its band 64 bytes at a time with 128-bit loads, the next block in flight while the current
// one is compressed (64 fully unrolled rounds on a 16-word rolling schedule), pads the tail as the standard says and
// xors its digest into the frame's H with eight atomicXor.
#include <cuda_runtime.h>
#include <stdint.h>

#include "kernels.cuh"

namespace vk {

namespace {

// FIPS 180-4 section 4.2.2: first 32 bits of the fractional parts of the cube roots of the first 64 primes.
__constant__ uint32_t KT[64] = {
    0x428a2f98, 0x71374491, 0xb5c0fbcf, 0xe9b5dba5, 0x3956c25b, 0x59f111f1, 0x923f82a4, 0xab1c5ed5, 0xd807aa98,
    0x12835b01, 0x243185be, 0x550c7dc3, 0x72be5d74, 0x80deb1fe, 0x9bdc06a7, 0xc19bf174, 0xe49b69c1, 0xefbe4786,
    0x0fc19dc6, 0x240ca1cc, 0x2de92c6f, 0x4a7484aa, 0x5cb0a9dc, 0x76f988da, 0x983e5152, 0xa831c66d, 0xb00327c8,
    0xbf597fc7, 0xc6e00bf3, 0xd5a79147, 0x06ca6351, 0x14292967, 0x27b70a85, 0x2e1b2138, 0x4d2c6dfc, 0x53380d13,
    0x650a7354, 0x766a0abb, 0x81c2c92e, 0x92722c85, 0xa2bfe8a1, 0xa81a664b, 0xc24b8b70, 0xc76c51a3, 0xd192e819,
    0xd6990624, 0xf40e3585, 0x106aa070, 0x19a4c116, 0x1e376c08, 0x2748774c, 0x34b0bcb5, 0x391c0cb3, 0x4ed8aa4a,
    0x5b9cca4f, 0x682e6ff3, 0x748f82ee, 0x78a5636f, 0x84c87814, 0x8cc70208, 0x90befffa, 0xa4506ceb, 0xbef9a3f7,
    0xc67178f2};

__device__ __forceinline__ uint32_t ror(uint32_t x, int n) { return __funnelshift_r(x, x, n); }
__device__ __forceinline__ uint32_t bswap(uint32_t x) { return __byte_perm(x, 0u, 0x0123); }

// One 64-byte block: w[] holds the 16 big-endian message words on entry (destroyed).
__device__ __forceinline__ void compress(uint32_t (&st)[8], uint32_t (&w)[16]) {
    uint32_t a = st[0], b = st[1], c = st[2], d = st[3], e = st[4], f = st[5], g = st[6], h = st[7];
#pragma unroll
    for (int t = 0; t < 64; ++t) {
        if (t >= 16) {
            const uint32_t w15 = w[(t + 1) & 15], w2 = w[(t + 14) & 15];
            w[t & 15] += (ror(w15, 7) ^ ror(w15, 18) ^ (w15 >> 3)) + w[(t + 9) & 15] + (ror(w2, 17) ^ ror(w2, 19) ^ (w2 >> 10));
        }
        const uint32_t t1 = h + (ror(e, 6) ^ ror(e, 11) ^ ror(e, 25)) + (g ^ (e & (f ^ g))) + KT[t] + w[t & 15];
        const uint32_t t2 = (ror(a, 2) ^ ror(a, 13) ^ ror(a, 22)) + ((a & b) | (c & (a | b)));
        h = g; g = f; f = e; e = d + t1; d = c; c = b; b = a; a = t1 + t2;
    }
    st[0] += a; st[1] += b; st[2] += c; st[3] += d; st[4] += e; st[5] += f; st[6] += g; st[7] += h;
}

}  // namespace

// frames: m x (h x 3w) bytes, 16-byte aligned, row_bytes % 16 == 0.  H: m x 8 words, zeroed by the caller; on exit
// H[f] holds the xor of the digests of bands band0 .. n-1 as big-endian words (byte-swapped to digest order by finish_hash_kernel).
__global__ void __launch_bounds__(32) sha_bands_kernel(const uint8_t *__restrict__ frames, Geom g, uint32_t n, uint32_t band0,
                                                       uint32_t m, uint32_t *H) {
    const uint32_t t = blockIdx.x * 32u + threadIdx.x, nb = n - band0;  // bands band0 .. n-1 of every frame
    if (t >= m * nb) return;
    const uint32_t f = t / nb, band = band0 + (t - f * nb);
    const uint64_t r0 = ((uint64_t)band * g.h) / n, r1 = ((uint64_t)(band + 1u) * g.h) / n;
    const uint64_t len = (r1 - r0) * g.row_bytes;
    const uint8_t *msg = frames + (size_t)f * g.frame_bytes + r0 * g.row_bytes;
    const uint4 *p = reinterpret_cast<const uint4 *>(msg);
    uint32_t st[8] = {0x6a09e667u, 0xbb67ae85u, 0x3c6ef372u, 0xa54ff53au, 0x510e527fu, 0x9b05688cu, 0x1f83d9abu, 0x5be0cd19u};
    const uint64_t nblk = len >> 6;
    uint4 nx[4];
    if (nblk) {
#pragma unroll
        for (int i = 0; i < 4; ++i) nx[i] = __ldg(p + i);
    }
    for (uint64_t b = 0; b < nblk; ++b) {
        uint32_t w[16] = {bswap(nx[0].x), bswap(nx[0].y), bswap(nx[0].z), bswap(nx[0].w), bswap(nx[1].x), bswap(nx[1].y),
                          bswap(nx[1].z), bswap(nx[1].w), bswap(nx[2].x), bswap(nx[2].y), bswap(nx[2].z), bswap(nx[2].w),
                          bswap(nx[3].x), bswap(nx[3].y), bswap(nx[3].z), bswap(nx[3].w)};
        if (b + 1 < nblk) {
#pragma unroll
            for (int i = 0; i < 4; ++i) nx[i] = __ldg(p + 4 * (b + 1) + i);
        }
        compress(st, w);
    }
    // tail: len % 64 bytes (a multiple of 16 here), 0x80, zeros, 64-bit big-endian bit length
    {
        const uint32_t rem = (uint32_t)(len & 63u);  // 0, 16, 32 or 48
        uint32_t w[16];
#pragma unroll
        for (int i = 0; i < 16; ++i) w[i] = 0u;
        const uint4 *q = p + 4 * nblk;
#pragma unroll
        for (int i = 0; i < 3; ++i)
            if ((uint32_t)(16 * (i + 1)) <= rem) {
                const uint4 v = __ldg(q + i);
                w[4 * i] = bswap(v.x); w[4 * i + 1] = bswap(v.y); w[4 * i + 2] = bswap(v.z); w[4 * i + 3] = bswap(v.w);
            }
#pragma unroll
        for (int i = 0; i < 4; ++i)
            if (rem == (uint32_t)(16 * i)) w[4 * i] = 0x80000000u;
        // rem <= 48 < 56: the length always fits in this block
        const uint64_t bits = len << 3;
        w[14] = (uint32_t)(bits >> 32);
        w[15] = (uint32_t)bits;
        compress(st, w);
    }
#pragma unroll
    for (int i = 0; i < 8; ++i) atomicXor(H + (size_t)f * 8u + i, st[i]);
}

// big-endian words -> digest byte order, in place
__global__ void finish_hash_kernel(uint32_t *H, uint32_t nwords) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < nwords) H[i] = __byte_perm(H[i], 0u, 0x0123);
}

cudaError_t hash_device(const Geom &g, const uint8_t *d_frames, uint32_t n, uint32_t band0, size_t m, uint32_t *d_H,
                        cudaStream_t st) {
    if (!m || band0 >= n) return m ? cudaMemsetAsync(d_H, 0, m * 32u, st) : cudaSuccess;
    if (g.row_bytes % 16u != 0u || (reinterpret_cast<uintptr_t>(d_frames) & 15u)) return cudaErrorInvalidValue;
    cudaError_t e = cudaMemsetAsync(d_H, 0, m * 32u, st);
    if (e != cudaSuccess) return e;
    const uint32_t total = (uint32_t)(m * (n - band0));
    sha_bands_kernel<<<(total + 31u) / 32u, 32, 0, st>>>(d_frames, g, n, band0, (uint32_t)m, d_H);
    finish_hash_kernel<<<(unsigned)((m * 8u + 127u) / 128u), 128, 0, st>>>(d_H, (uint32_t)(m * 8u));
    return cudaGetLastError();
}

}  // namespace vk
