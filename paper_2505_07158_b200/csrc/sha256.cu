// sha256.cu -- device-side sub-frame hashing: h_m = SHA-256(f_m) for the n row bands of each
// frame of a batch and H = xor_m h_m, on the frames that were uploaded for the cipher kernels anyway.
//
// SHA-256 (FIPS 180-4) is serial inside a message, so the parallelism is one message per (frame, band): n x batch
// independent message streams (256 at n = 32, batch = 8), 32 messages per CTA (two warps, see below) so that the CTAs
// spread over as many SMs as possible.  A band is walked 64 bytes at a time with 128-bit loads, the next block in flight
// while the current one is processed, the tail padded as the standard says, and the digest xor-ed into the frame's H
// with eight atomicXor.
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
__device__ __forceinline__ void bar_sync(uint32_t id, uint32_t n) { asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(n) : "memory"); }
__device__ __forceinline__ void bar_arrive(uint32_t id, uint32_t n) { asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(n) : "memory"); }

}  // namespace

// SHA-256 is serial inside a message, and a lone warp is bound by its own instruction stream (about 1 500 instructions per
// 64-byte block, 2 cycles each on the ALU pipe).  The message schedule W_t (FIPS 180-4 section 6.2.2 step 1) does not
// depend on the hash state, so a CTA is two warps working on the same 32 messages: the SCHEDULE warp loads the block,
// expands W_0..63, adds K_t and leaves the 64 words in shared memory (double-buffered); the ROUND warp runs the 64 rounds
// (step 3) reading them back.  The round warp is the longer of the two (about 960 instructions per block), the schedule warp
// (about 650) runs one block ahead.  Hand-over with named barriers: FULL[buf] schedule -> round, EMPTY[buf] round -> schedule.
//
// frames: m x (h x 3w) bytes, 16-byte aligned, row_bytes % 16 == 0.  H: m x 8 words, zeroed by the caller; on exit
// H[f] holds the xor of the digests of bands band0 .. n-1 as big-endian words (byte-swapped to digest order by finish_hash_kernel).
__global__ void __launch_bounds__(64) sha_bands_kernel(const uint8_t *__restrict__ frames, Geom g, uint32_t n, uint32_t band0,
                                                       uint32_t m, uint32_t *H) {
    __shared__ uint32_t Wb[2][64][32];  // [buffer][t][lane]: W_t + K_t of the lane's current block
    const uint32_t lane = threadIdx.x & 31u, role = threadIdx.x >> 5;  // role 0: rounds, 1: schedule
    const uint32_t nb = n - band0, total = m * nb;                    // bands band0 .. n-1 of every frame
    uint32_t t = blockIdx.x * 32u + lane;
    const bool live = t < total;
    if (!live) t = total - 1u;  // keeps both warps' loop bounds equal; a dead lane repeats the last message and writes nothing
    const uint32_t f = t / nb, band = band0 + (t - f * nb);
    const uint64_t r0 = ((uint64_t)band * g.h) / n, r1 = ((uint64_t)(band + 1u) * g.h) / n;
    const uint64_t len = (r1 - r0) * g.row_bytes;
    const uint4 *p = reinterpret_cast<const uint4 *>(frames + (size_t)f * g.frame_bytes + r0 * g.row_bytes);
    const uint32_t nblk = (uint32_t)(len >> 6);                      // whole blocks; one more block holds the tail and the padding
    const uint32_t iters = __reduce_max_sync(0xffffffffu, nblk + 1u);  // the same in both warps: lane l holds the same message
    constexpr uint32_t FULL = 1, EMPTY = 3;                           // named barriers FULL + buf, EMPTY + buf (64 threads each)

    if (role == 1u) {
        // ---------------- schedule warp ----------------
        uint4 nx[4];
#pragma unroll
        for (int i = 0; i < 4; ++i) nx[i] = make_uint4(0u, 0u, 0u, 0u);
        if (nblk) {
#pragma unroll
            for (int i = 0; i < 4; ++i) nx[i] = __ldg(p + i);
        }
        for (uint32_t b = 0; b < iters; ++b) {
            const uint32_t buf = b & 1u;
            uint32_t w[16];
            if (b < nblk) {
                w[0] = bswap(nx[0].x); w[1] = bswap(nx[0].y); w[2] = bswap(nx[0].z); w[3] = bswap(nx[0].w);
                w[4] = bswap(nx[1].x); w[5] = bswap(nx[1].y); w[6] = bswap(nx[1].z); w[7] = bswap(nx[1].w);
                w[8] = bswap(nx[2].x); w[9] = bswap(nx[2].y); w[10] = bswap(nx[2].z); w[11] = bswap(nx[2].w);
                w[12] = bswap(nx[3].x); w[13] = bswap(nx[3].y); w[14] = bswap(nx[3].z); w[15] = bswap(nx[3].w);
                if (b + 1u < nblk) {
#pragma unroll
                    for (int i = 0; i < 4; ++i) nx[i] = __ldg(p + 4u * (b + 1u) + i);
                }
            } else {
                // tail block (b == nblk): len % 64 bytes (a multiple of 16 here), 0x80, zeros, 64-bit big-endian bit length;
                // blocks past it (b > nblk, other lanes still running) are ignored by the round warp
#pragma unroll
                for (int i = 0; i < 16; ++i) w[i] = 0u;
                if (b == nblk) {
                    const uint32_t rem = (uint32_t)(len & 63u);  // 0, 16, 32 or 48
                    const uint4 *q = p + 4u * nblk;
#pragma unroll
                    for (int i = 0; i < 3; ++i)
                        if ((uint32_t)(16 * (i + 1)) <= rem) {
                            const uint4 v = __ldg(q + i);
                            w[4 * i] = bswap(v.x); w[4 * i + 1] = bswap(v.y); w[4 * i + 2] = bswap(v.z); w[4 * i + 3] = bswap(v.w);
                        }
#pragma unroll
                    for (int i = 0; i < 4; ++i)
                        if (rem == (uint32_t)(16 * i)) w[4 * i] = 0x80000000u;
                    const uint64_t bits = len << 3;  // rem <= 48 < 56: the length always fits in this block
                    w[14] = (uint32_t)(bits >> 32);
                    w[15] = (uint32_t)bits;
                }
            }
            if (b >= 2u) bar_sync(EMPTY + buf, 64);  // the round warp has finished with this buffer (block b - 2)
#pragma unroll
            for (int tt = 0; tt < 64; ++tt) {
                if (tt >= 16) {
                    const uint32_t w15 = w[(tt + 1) & 15], w2 = w[(tt + 14) & 15];
                    w[tt & 15] += (ror(w15, 7) ^ ror(w15, 18) ^ (w15 >> 3)) + w[(tt + 9) & 15] + (ror(w2, 17) ^ ror(w2, 19) ^ (w2 >> 10));
                }
                Wb[buf][tt][lane] = w[tt & 15] + KT[tt];
            }
            __threadfence_block();
            bar_arrive(FULL + buf, 64);
        }
        return;
    }

    // ---------------- round warp ----------------
    uint32_t st[8] = {0x6a09e667u, 0xbb67ae85u, 0x3c6ef372u, 0xa54ff53au, 0x510e527fu, 0x9b05688cu, 0x1f83d9abu, 0x5be0cd19u};
    for (uint32_t b = 0; b < iters; ++b) {
        const uint32_t buf = b & 1u;
        bar_sync(FULL + buf, 64);
        uint32_t a = st[0], bb = st[1], c = st[2], d = st[3], e = st[4], ff = st[5], gg = st[6], h = st[7];
#pragma unroll
        for (int tt = 0; tt < 64; ++tt) {
            const uint32_t t1 = h + (ror(e, 6) ^ ror(e, 11) ^ ror(e, 25)) + (gg ^ (e & (ff ^ gg))) + Wb[buf][tt][lane];
            const uint32_t t2 = (ror(a, 2) ^ ror(a, 13) ^ ror(a, 22)) + ((a & bb) | (c & (a | bb)));
            h = gg; gg = ff; ff = e; e = d + t1; d = c; c = bb; bb = a; a = t1 + t2;
        }
        if (b <= nblk) {  // this lane's message still has this block
            st[0] += a; st[1] += bb; st[2] += c; st[3] += d; st[4] += e; st[5] += ff; st[6] += gg; st[7] += h;
        }
        if (b + 2u < iters) bar_arrive(EMPTY + buf, 64);  // only when the schedule warp will wait for it
    }
    if (live) {
#pragma unroll
        for (int i = 0; i < 8; ++i) atomicXor(H + (size_t)f * 8u + i, st[i]);
    }
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
    sha_bands_kernel<<<(total + 31u) / 32u, 64, 0, st>>>(d_frames, g, n, band0, (uint32_t)m, d_H);
    finish_hash_kernel<<<(unsigned)((m * 8u + 127u) / 128u), 128, 0, st>>>(d_H, (uint32_t)(m * 8u));
    return cudaGetLastError();
}

}  // namespace vk
