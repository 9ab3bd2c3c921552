// membench.cu -- memory-system probes behind vcrypt_memory_probe (bench hook, include/vcrypt.h).
//
// They move the SAME bytes as one vcrypt_encrypt_device call on `frames` frames of the context's shape, with no
// cipher arithmetic, so that bench.py can print what the memory system itself allows next to what the cipher
// kernels reach:
//   probe 0  sequential copy            : read 3wh, write 3wh per frame, fully coalesced (the HBM copy rate)
//   probe 1  two-pass traffic, sequential: pass 1 reads F (DRAM) and writes T; pass 2 reads T (L2), reads B (DRAM),
//                                          writes O (DRAM) -- the 5 trips through L2 per byte of any two-pass design
//   probe 2  column strips              : read B and write O in 64-byte-wide column strips of the h x 3w matrix
//                                          (the DRAM side of the column pass: row-strided 64-byte accesses)
// Buffers rotate through > 1 GB so that nothing but T is L2-resident between repetitions.
#include <cuda_runtime.h>
#include <stdint.h>

#include "kernels.cuh"

namespace vk {

__global__ void __launch_bounds__(512) probe_copy(const uint4 *__restrict__ s, uint4 *__restrict__ d, size_t n, int stream_out) {
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const size_t st = (size_t)gridDim.x * blockDim.x;
    for (; i + 3 * st < n; i += 4 * st) {
        const uint4 a = __ldcs(s + i), b = __ldcs(s + i + st), c = __ldcs(s + i + 2 * st), e = __ldcs(s + i + 3 * st);
        if (stream_out) { __stcs(d + i, a); __stcs(d + i + st, b); __stcs(d + i + 2 * st, c); __stcs(d + i + 3 * st, e); }
        else { d[i] = a; d[i + st] = b; d[i + 2 * st] = c; d[i + 3 * st] = e; }
    }
    for (; i < n; i += st) d[i] = s[i];
}

__global__ void __launch_bounds__(512) probe_xor(const uint4 *t, const uint4 *__restrict__ b, uint4 *o, size_t n) {
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    const size_t st = (size_t)gridDim.x * blockDim.x;
    for (; i + st < n; i += 2 * st) {
        const uint4 x = t[i], y = __ldcs(b + i), x2 = t[i + st], y2 = __ldcs(b + i + st);
        __stcs(o + i, make_uint4(x.x ^ y.x, x.y ^ y.y, x.z ^ y.z, x.w ^ y.w));
        __stcs(o + i + st, make_uint4(x2.x ^ y2.x, x2.y ^ y2.y, x2.z ^ y2.z, x2.w ^ y2.w));
    }
    for (; i < n; i += st) { const uint4 x = t[i], y = b[i]; o[i] = make_uint4(x.x ^ y.x, x.y ^ y.y, x.z ^ y.z, x.w ^ y.w); }
}

// one CTA per strip of 64 byte columns x h rows; a lane owns 8 bytes of a row, a sub-warp of 8 lanes 8 consecutive rows
__global__ void __launch_bounds__(256) probe_strips(const uint8_t *__restrict__ B, uint8_t *__restrict__ O, uint32_t h, uint32_t rb,
                                                     uint32_t strips) {
    const uint32_t f = blockIdx.x / strips, x0 = (blockIdx.x - f * strips) * 64u;
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5, sub = lane >> 3, j = lane & 7u;
    if (x0 + 8u * j >= rb) return;
    const size_t base = (size_t)f * h * rb + x0 + 8u * j;
    for (uint32_t r0 = (warp * 4u + sub) * 8u; r0 < h; r0 += 8u * 4u * 8u) {
        uint2 v[8];
#pragma unroll
        for (int i = 0; i < 8; ++i) v[i] = r0 + i < h ? __ldcs(reinterpret_cast<const uint2 *>(B + base + (size_t)(r0 + i) * rb)) : make_uint2(0, 0);
#pragma unroll
        for (int i = 0; i < 8; ++i)
            if (r0 + i < h) __stcs(reinterpret_cast<uint2 *>(O + base + (size_t)(r0 + i) * rb), make_uint2(v[i].x ^ 1u, v[i].y));
    }
}

cudaError_t memory_probe(const Geom &g, int which, size_t frames, int reps, cudaStream_t st, double *us_per_call) {
    if (which < 0 || which > 2 || frames == 0 || reps < 1 || g.row_bytes % 16 != 0) return cudaErrorInvalidValue;
    const size_t batch = frames * g.frame_bytes;
    size_t nrot = ((size_t)1200 << 20) / batch;
    if (nrot < 2) nrot = 2;
    if (nrot > 64) nrot = 64;
    uint8_t *A = nullptr, *Bb = nullptr, *O = nullptr, *T = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    cudaError_t e = cudaMalloc(&A, batch * nrot);
    if (!e) e = cudaMalloc(&Bb, batch * nrot);
    if (!e) e = cudaMalloc(&O, batch * nrot);
    if (!e) e = cudaMalloc(&T, batch);
    if (!e) e = cudaMemsetAsync(A, 1, batch * nrot, st);
    if (!e) e = cudaMemsetAsync(Bb, 2, batch * nrot, st);
    if (!e) e = cudaMemsetAsync(O, 3, batch * nrot, st);
    if (!e) e = cudaMemsetAsync(T, 4, batch, st);
    if (!e) e = cudaEventCreate(&e0);
    if (!e) e = cudaEventCreate(&e1);
    int sms = 148, dev = 0;
    if (!e) e = cudaGetDevice(&dev);
    if (!e) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (!e) {
        const size_t n16 = batch / 16;
        const unsigned grid = (unsigned)sms * 8u;
        const uint32_t strips = (g.row_bytes + 63u) / 64u;
        for (int it = -3; it < reps && !e; ++it) {
            if (it == 0) e = cudaEventRecord(e0, st);
            const size_t off = (size_t)((it + 3) % (int)nrot) * batch;
            if (which == 0) {
                probe_copy<<<grid, 512, 0, st>>>((const uint4 *)(A + off), (uint4 *)(O + off), n16, 1);
            } else if (which == 1) {
                probe_copy<<<grid, 512, 0, st>>>((const uint4 *)(A + off), (uint4 *)T, n16, 0);
                probe_xor<<<grid, 512, 0, st>>>((const uint4 *)T, (const uint4 *)(Bb + off), (uint4 *)(O + off), n16);
            } else {
                probe_strips<<<(unsigned)(frames * strips), 256, 0, st>>>(Bb + off, O + off, g.h, g.row_bytes, strips);
            }
            if (!e) e = cudaGetLastError();
        }
        if (!e) e = cudaEventRecord(e1, st);
        if (!e) e = cudaEventSynchronize(e1);
        float ms = 0.f;
        if (!e) e = cudaEventElapsedTime(&ms, e0, e1);
        if (!e && us_per_call) *us_per_call = 1e3 * (double)ms / reps;
    }
    cudaStreamSynchronize(st);
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(A); cudaFree(Bb); cudaFree(O); cudaFree(T);
    return e;
}

}  // namespace vk
