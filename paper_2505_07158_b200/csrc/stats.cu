// stats.cu -- statistical evaluation of frames resident in HBM (PAPER.md sections III-IV):
// histogram variance (Eq. 4), chi^2 (Eq. 5), adjacent-pixel correlation (Eq. 6-9), information entropy (Eq. 10), local
// Shannon entropy (Eq. 11) and NPCR / UACI (Eq. 14-16).
//
// The kernels are single-pass reductions that produce EXACT integer sufficient statistics (histograms, sums of x, y, xy,
// x^2, y^2 over all adjacent pairs, counts of differing bytes, sums of absolute differences); the few floating-point
// operations that turn them into the paper's quantities are done on the host in binary64 (vcrypt.cpp), so the integer
// part is bit-exact against the oracle and the rest agrees to rounding.  Every channel of every frame is read once.
#include <cuda_runtime.h>
#include <stdint.h>

#include "kernels.cuh"

namespace vk {

namespace {

__device__ __forceinline__ uint64_t warp_sum(uint64_t v) {
#pragma unroll
    for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

}  // namespace

// Per frame f: hist[f][c][256] (u32) and pairs[f][c][d][5] (u64: sum x, sum y, sum xy, sum x^2, sum y^2) for the
// directions d = 0 horizontal (i, j)-(i, j+1), 1 vertical (i, j)-(i+1, j), 2 diagonal (i, j)-(i+1, j+1), over ALL pairs.
// One item = 4 consecutive pixels (12 bytes) of one row, so that byte b of an item always belongs to channel b % 3.
__global__ void __launch_bounds__(256) stats_kernel(const uint8_t *__restrict__ F, Geom g, uint32_t nframes, uint32_t *hist,
                                                    unsigned long long *pairs) {
    __shared__ uint32_t sh[3 * 256];
    __shared__ unsigned long long sp[45];
    const uint32_t f = blockIdx.y, w = g.w, h = g.h, rb = g.row_bytes;
    for (uint32_t i = threadIdx.x; i < 768; i += blockDim.x) sh[i] = 0;
    if (threadIdx.x < 45) sp[threadIdx.x] = 0;
    __syncthreads();
    const uint8_t *fr = F + (size_t)f * g.frame_bytes;
    const uint32_t qpr = (w + 3u) / 4u;  // items per row
    const uint64_t nitems = (uint64_t)qpr * h;
    uint32_t acc[3][3][5];  // [channel][direction][sum]: u32 partials, flushed before they can overflow
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int d = 0; d < 3; ++d)
#pragma unroll
            for (int k = 0; k < 5; ++k) acc[c][d][k] = 0;
    uint32_t since_flush = 0;
    auto flush = [&]() {
#pragma unroll
        for (int c = 0; c < 3; ++c)
#pragma unroll
            for (int d = 0; d < 3; ++d)
#pragma unroll
                for (int k = 0; k < 5; ++k) {
                    const uint64_t s = warp_sum(acc[c][d][k]);
                    if ((threadIdx.x & 31u) == 0 && s) atomicAdd(&sp[(c * 3 + d) * 5 + k], (unsigned long long)s);
                    acc[c][d][k] = 0;
                }
    };
    for (uint64_t it0 = (uint64_t)blockIdx.x * blockDim.x; it0 < nitems; it0 += (uint64_t)gridDim.x * blockDim.x) {
        const uint64_t it = it0 + threadIdx.x;
        if (it < nitems) {
            const uint32_t i = (uint32_t)(it / qpr), q = (uint32_t)(it - (uint64_t)i * qpr);
            const uint8_t *r0 = fr + (size_t)i * rb + 12u * q;
            const bool has_below = i + 1u < h;
            const uint8_t *r1 = has_below ? r0 + rb : r0;
            const uint32_t npx = w - 4u * q < 4u ? w - 4u * q : 4u;  // pixels of this item inside the row
#pragma unroll
            for (int p = 0; p < 4; ++p) {
                if ((uint32_t)p >= npx) break;
                const bool has_right = 4u * q + p + 1u < w;
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const uint32_t x = r0[3 * p + c];
                    atomicAdd(&sh[c * 256 + x], 1u);
                    if (has_right) {
                        const uint32_t y = r0[3 * p + 3 + c];
                        acc[c][0][0] += x; acc[c][0][1] += y; acc[c][0][2] += x * y; acc[c][0][3] += x * x; acc[c][0][4] += y * y;
                    }
                    if (has_below) {
                        const uint32_t y = r1[3 * p + c];
                        acc[c][1][0] += x; acc[c][1][1] += y; acc[c][1][2] += x * y; acc[c][1][3] += x * x; acc[c][1][4] += y * y;
                        if (has_right) {
                            const uint32_t z = r1[3 * p + 3 + c];
                            acc[c][2][0] += x; acc[c][2][1] += z; acc[c][2][2] += x * z; acc[c][2][3] += x * x; acc[c][2][4] += z * z;
                        }
                    }
                }
            }
        }
        // 4 pixels x 65025 per iteration: flush the u32 partials every 8192 iterations (< 2^32)
        if (++since_flush == 8192u) { flush(); since_flush = 0; }
    }
    flush();
    __syncthreads();
    for (uint32_t i = threadIdx.x; i < 768; i += blockDim.x)
        if (sh[i]) atomicAdd(hist + (size_t)f * 768u + i, sh[i]);
    if (threadIdx.x < 45 && sp[threadIdx.x]) atomicAdd(pairs + (size_t)f * 45u + threadIdx.x, sp[threadIdx.x]);
}

// NPCR / UACI (Eq. 14-16): per frame and channel, the number of differing bytes and the sum of |a - b|.
// out[f][c][2] (u64).  Words of 4 bytes; the channel of byte b of word k is (4k + b) % 3.
__global__ void __launch_bounds__(256) diff_kernel(const uint8_t *__restrict__ A, const uint8_t *__restrict__ B, size_t frame_bytes,
                                                   unsigned long long *out) {
    __shared__ unsigned long long s[6];
    if (threadIdx.x < 6) s[threadIdx.x] = 0;
    __syncthreads();
    const uint32_t f = blockIdx.y;
    const uint8_t *a = A + (size_t)f * frame_bytes, *b = B + (size_t)f * frame_bytes;
    uint32_t ne[3] = {0, 0, 0}, ad[3] = {0, 0, 0};
    // one item = 12 bytes (4 pixels): static byte -> channel mapping; frame_bytes = 3wh is a multiple of 3, tail by bytes
    const size_t nitems = frame_bytes / 12u;
    for (size_t it = (size_t)blockIdx.x * blockDim.x + threadIdx.x; it < nitems; it += (size_t)gridDim.x * blockDim.x) {
#pragma unroll
        for (int k = 0; k < 12; ++k) {
            const int x = a[12u * it + k], y = b[12u * it + k];
            ne[k % 3] += x != y;
            ad[k % 3] += (uint32_t)(x > y ? x - y : y - x);
        }
    }
    if (blockIdx.x == 0 && threadIdx.x == 0)
        for (size_t o = nitems * 12u; o < frame_bytes; ++o) {
            const int x = a[o], y = b[o];
            ne[o % 3] += x != y;
            ad[o % 3] += (uint32_t)(x > y ? x - y : y - x);
        }
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const uint64_t n1 = warp_sum(ne[c]), n2 = warp_sum(ad[c]);
        if ((threadIdx.x & 31u) == 0) { atomicAdd(&s[2 * c], (unsigned long long)n1); atomicAdd(&s[2 * c + 1], (unsigned long long)n2); }
    }
    __syncthreads();
    if (threadIdx.x < 6 && s[threadIdx.x]) atomicAdd(out + (size_t)f * 6u + threadIdx.x, s[threadIdx.x]);
}

// Local Shannon entropy (Eq. 11): histogram of each channel of each of k square blocks (side x side pixels, top-left
// corners in xy[k][2]) of every frame.  One CTA per (block, frame).  bh[f][blk][c][256] (u32), zeroed by the caller.
__global__ void __launch_bounds__(256) block_hist_kernel(const uint8_t *__restrict__ F, Geom g, const uint32_t *__restrict__ xy,
                                                         uint32_t side, uint32_t *bh) {
    __shared__ uint32_t sh[768];
    for (uint32_t i = threadIdx.x; i < 768; i += blockDim.x) sh[i] = 0;
    __syncthreads();
    const uint32_t blk = blockIdx.x, f = blockIdx.y, x0 = xy[2 * blk], y0 = xy[2 * blk + 1];
    const uint8_t *fr = F + (size_t)f * g.frame_bytes;
    const uint32_t nb = side * side * 3u;
    for (uint32_t t = threadIdx.x; t < nb; t += blockDim.x) {
        const uint32_t r = t / (side * 3u), o = t - r * side * 3u;
        const uint32_t v = fr[(size_t)(y0 + r) * g.row_bytes + 3u * x0 + o];
        atomicAdd(&sh[(o % 3u) * 256u + v], 1u);
    }
    __syncthreads();
    uint32_t *dst = bh + ((size_t)f * gridDim.x + blk) * 768u;
    for (uint32_t i = threadIdx.x; i < 768; i += blockDim.x) dst[i] = sh[i];
}

cudaError_t stats_device(const Geom &g, const uint8_t *d_frames, size_t n, uint32_t *d_hist, unsigned long long *d_pairs,
                         cudaStream_t st) {
    if (!n) return cudaSuccess;
    cudaError_t e = cudaMemsetAsync(d_hist, 0, n * 768u * sizeof(uint32_t), st);
    if (!e) e = cudaMemsetAsync(d_pairs, 0, n * 45u * sizeof(unsigned long long), st);
    if (e) return e;
    const uint64_t items = (uint64_t)((g.w + 3u) / 4u) * g.h;
    uint32_t gx = (uint32_t)((items + 256u * 8u - 1u) / (256u * 8u));
    if (gx > 592u) gx = 592u;
    if (gx < 1u) gx = 1u;
    stats_kernel<<<dim3(gx, (unsigned)n), 256, 0, st>>>(d_frames, g, (uint32_t)n, d_hist, d_pairs);
    return cudaGetLastError();
}

cudaError_t diff_device(const Geom &g, const uint8_t *d_a, const uint8_t *d_b, size_t n, unsigned long long *d_out, cudaStream_t st) {
    if (!n) return cudaSuccess;
    cudaError_t e = cudaMemsetAsync(d_out, 0, n * 6u * sizeof(unsigned long long), st);
    if (e) return e;
    uint32_t gx = (uint32_t)((g.frame_bytes / 12u + 256u * 8u - 1u) / (256u * 8u));
    if (gx > 592u) gx = 592u;
    if (gx < 1u) gx = 1u;
    diff_kernel<<<dim3(gx, (unsigned)n), 256, 0, st>>>(d_a, d_b, g.frame_bytes, d_out);
    return cudaGetLastError();
}

cudaError_t block_hist_device(const Geom &g, const uint8_t *d_frames, size_t n, const uint32_t *d_xy, uint32_t k, uint32_t side,
                              uint32_t *d_bh, cudaStream_t st) {
    if (!n || !k) return cudaSuccess;
    block_hist_kernel<<<dim3(k, (unsigned)n), 256, 0, st>>>(d_frames, g, d_xy, side, d_bh);
    return cudaGetLastError();
}

}  // namespace vk
