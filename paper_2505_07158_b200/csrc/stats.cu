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

#include <mutex>

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

// Fast path for w % 4 == 0 (rows are whole 32-bit words, an item of 4 pixels is never ragged).  Per item three words of
// row i (+ one more for the pixel to the right of the last one) and the same of row i+1; the neighbour of every byte is
// three bytes further, i.e. the same byte lane and the same channel after a 24-bit funnel shift; per byte four PRMT extract
// x and its three neighbours and four IMAD accumulate (measured: 4-way byte dot products, DP4A, are 3x slower on this part):
//   raw[f][c] = { S1 = sum x, S2 = sum x^2 over ALL pixels; XY[d] = sum x*y over the pairs of direction d;
//                 border sums (sum, sum of squares) of the first / last column and first / last row; the four corners }
// from which the host gets the per-direction sums of Eq. 7-9 exactly (a pair set is "all pixels minus a border").
constexpr int RAW_PER_CH = 2 + 3 + 8 + 4;  // 17 u64 per (frame, channel)

__global__ void __launch_bounds__(256) stats_fast_kernel(const uint8_t *__restrict__ F, Geom g, uint32_t *hist, unsigned long long *raw) {
    __shared__ uint32_t sh[8][3 * 256];  // one histogram per warp: fewer collisions on smooth frames
    __shared__ unsigned long long sp[3 * RAW_PER_CH];
    const uint32_t f = blockIdx.y, w = g.w, h = g.h, rb = g.row_bytes, warp = threadIdx.x >> 5;
    for (uint32_t i = threadIdx.x; i < 8 * 768; i += blockDim.x) (&sh[0][0])[i] = 0;
    if (threadIdx.x < 3 * RAW_PER_CH) sp[threadIdx.x] = 0;
    __syncthreads();
    const uint8_t *fr = F + (size_t)f * g.frame_bytes;
    const uint32_t qpr = w >> 2;
    const uint64_t nitems = (uint64_t)qpr * h;
    uint32_t S1[3] = {0, 0, 0}, S2[3] = {0, 0, 0}, XY[3][3] = {{0, 0, 0}, {0, 0, 0}, {0, 0, 0}};
    unsigned long long bs[3][8];  // borders: rare, straight to 64 bits
    uint32_t corner[3][4];
    bool has_corner[4] = {false, false, false, false};
#pragma unroll
    for (int c = 0; c < 3; ++c) {
#pragma unroll
        for (int k = 0; k < 8; ++k) bs[c][k] = 0;
#pragma unroll
        for (int k = 0; k < 4; ++k) corner[c][k] = 0;
    }
    uint32_t n_done = 0;
    auto flush = [&]() {
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            uint64_t v[5] = {S1[c], S2[c], XY[c][0], XY[c][1], XY[c][2]};
#pragma unroll
            for (int k = 0; k < 5; ++k) {
                const uint64_t t = warp_sum(v[k]);
                if ((threadIdx.x & 31u) == 0 && t) atomicAdd(&sp[c * RAW_PER_CH + k], (unsigned long long)t);
            }
            S1[c] = S2[c] = XY[c][0] = XY[c][1] = XY[c][2] = 0;
        }
    };
    // item loader: three words of row i (+ one for the pixel to the right of the last one), the same of row i + 1, and
    // the item's position flags.  No row below / no pixel to the right: the neighbour words are zero, so the products vanish.
    auto load_item = [&](uint64_t it, uint32_t (&X)[4], uint32_t (&Z)[4], uint32_t &flags) {
        const uint32_t i = (uint32_t)(it / qpr), q = (uint32_t)(it - (uint64_t)i * qpr);
        const uint32_t *r0 = reinterpret_cast<const uint32_t *>(fr + (size_t)i * rb) + 3u * q;
        const bool last_q = q + 1u == qpr, below = i + 1u < h;
        const uint32_t *r1 = reinterpret_cast<const uint32_t *>(reinterpret_cast<const uint8_t *>(r0) + (below ? rb : 0u));
        X[0] = __ldg(r0); X[1] = __ldg(r0 + 1); X[2] = __ldg(r0 + 2); X[3] = last_q ? 0u : __ldg(r0 + 3);
        Z[0] = below ? __ldg(r1) : 0u; Z[1] = below ? __ldg(r1 + 1) : 0u; Z[2] = below ? __ldg(r1 + 2) : 0u;
        Z[3] = (below && !last_q) ? __ldg(r1 + 3) : 0u;
        flags = (i == 0 ? 1u : 0u) | (i + 1u == h ? 2u : 0u) | (q == 0 ? 4u : 0u) | (last_q ? 8u : 0u);
    };
    const uint64_t stride = (uint64_t)gridDim.x * blockDim.x;
    uint32_t Xn[4] = {0, 0, 0, 0}, Zn[4] = {0, 0, 0, 0}, fn = 0;
    if ((uint64_t)blockIdx.x * blockDim.x + threadIdx.x < nitems) load_item((uint64_t)blockIdx.x * blockDim.x + threadIdx.x, Xn, Zn, fn);
    for (uint64_t it0 = (uint64_t)blockIdx.x * blockDim.x; it0 < nitems; it0 += stride) {
        const uint64_t it = it0 + threadIdx.x;
        if (it < nitems) {
            // software pipeline: the next item's eight loads are in flight while this one is accumulated
            uint32_t X[4], Z[4];
            const uint32_t flags = fn;
#pragma unroll
            for (int k = 0; k < 4; ++k) { X[k] = Xn[k]; Z[k] = Zn[k]; }
            if (it + stride < nitems) load_item(it + stride, Xn, Zn, fn);
#pragma unroll
            for (int k = 0; k < 3; ++k) {
                // the pixel to the right sits 3 bytes further: same byte lane, same channel after a 24-bit funnel shift
                const uint32_t yh = __funnelshift_r(X[k], X[k + 1], 24), zd = __funnelshift_r(Z[k], Z[k + 1], 24);
#pragma unroll
                for (int b = 0; b < 4; ++b) {
                    const int c = (4 * k + b) % 3;
                    const uint32_t sel = 0x4440u | (uint32_t)b;  // byte b, zero-extended (PRMT; the products go to the FMA pipe)
                    const uint32_t x = __byte_perm(X[k], 0u, sel), y0 = __byte_perm(yh, 0u, sel), y1 = __byte_perm(Z[k], 0u, sel),
                                   y2 = __byte_perm(zd, 0u, sel);
                    S1[c] += x;
                    S2[c] += x * x;
                    XY[c][0] += x * y0;
                    XY[c][1] += x * y1;
                    XY[c][2] += x * y2;
                    atomicAdd(&sh[warp][c * 256 + x], 1u);
                }
            }
            // borders (a small fraction of the items)
            const bool fr_row = flags & 1u, lr_row = flags & 2u, fc = flags & 4u, lc = flags & 8u;
            if (fr_row || lr_row || fc || lc) {
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const uint32_t p0 = (X[c >> 2] >> (8 * (c & 3))) & 0xFFu;                       // pixel 0: byte c
                    const uint32_t p3 = (X[(9 + c) >> 2] >> (8 * ((9 + c) & 3))) & 0xFFu;           // pixel 3: byte 9 + c
                    if (fc) { bs[c][0] += p0; bs[c][1] += p0 * p0; }
                    if (lc) { bs[c][2] += p3; bs[c][3] += p3 * p3; }
                    if (fr_row || lr_row) {
                        uint32_t s = 0, s2 = 0;
#pragma unroll
                        for (int p = 0; p < 4; ++p) {
                            const uint32_t v = (X[(3 * p + c) >> 2] >> (8 * ((3 * p + c) & 3))) & 0xFFu;
                            s += v; s2 += v * v;
                        }
                        if (fr_row) { bs[c][4] += s; bs[c][5] += s2; }
                        if (lr_row) { bs[c][6] += s; bs[c][7] += s2; }
                    }
                    if (fr_row && fc) { corner[c][0] = p0; has_corner[0] = true; }
                    if (fr_row && lc) { corner[c][1] = p3; has_corner[1] = true; }
                    if (lr_row && fc) { corner[c][2] = p0; has_corner[2] = true; }
                    if (lr_row && lc) { corner[c][3] = p3; has_corner[3] = true; }
                }
            }
        }
        if (++n_done == 4096u) { flush(); n_done = 0; }  // at most 4 x 65025 per item and sum: far below 2^32
    }
    flush();
#pragma unroll
    for (int c = 0; c < 3; ++c) {
#pragma unroll
        for (int k = 0; k < 8; ++k) {
            const uint64_t t = warp_sum(bs[c][k]);
            if ((threadIdx.x & 31u) == 0 && t) atomicAdd(&sp[c * RAW_PER_CH + 5 + k], (unsigned long long)t);
        }
#pragma unroll
        for (int k = 0; k < 4; ++k)
            if (has_corner[k]) sp[c * RAW_PER_CH + 13 + k] = corner[c][k];  // exactly one thread of the grid owns each corner
    }
    __syncthreads();
    for (uint32_t i = threadIdx.x; i < 768; i += blockDim.x) {
        uint32_t t = 0;
#pragma unroll
        for (int wv = 0; wv < 8; ++wv) t += sh[wv][i];
        if (t) atomicAdd(hist + (size_t)f * 768u + i, t);
    }
    if (threadIdx.x < 3 * RAW_PER_CH && sp[threadIdx.x]) atomicAdd(raw + (size_t)f * 3u * RAW_PER_CH + threadIdx.x, sp[threadIdx.x]);
}

// raw (fast path) -> pairs[f][c][d][5] = sum x, sum y, sum xy, sum x^2, sum y^2 of direction d
__global__ void raw_to_pairs_kernel(const unsigned long long *__restrict__ raw, unsigned long long *pairs, uint32_t n) {
    const uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n * 3u) return;
    const unsigned long long *r = raw + (size_t)t * RAW_PER_CH;
    unsigned long long *p = pairs + (size_t)t * 15u;
    const unsigned long long S1 = r[0], S2 = r[1];
    const unsigned long long fc = r[5], fc2 = r[6], lc = r[7], lc2 = r[8], frw = r[9], frw2 = r[10], lr = r[11], lr2 = r[12];
    const unsigned long long c00 = r[13], chw = r[16];  // corners (0, 0) and (h-1, w-1)
    // horizontal: x in all but the last column, y in all but the first column
    p[0] = S1 - lc; p[1] = S1 - fc; p[2] = r[2]; p[3] = S2 - lc2; p[4] = S2 - fc2;
    // vertical: x in all but the last row, y in all but the first row
    p[5] = S1 - lr; p[6] = S1 - frw; p[7] = r[3]; p[8] = S2 - lr2; p[9] = S2 - frw2;
    // diagonal: x in all but the last row and last column, y in all but the first row and first column
    p[10] = S1 - lr - lc + chw; p[11] = S1 - frw - fc + c00; p[12] = r[4];
    p[13] = S2 - lr2 - lc2 + chw * chw; p[14] = S2 - frw2 - fc2 + c00 * c00;
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
    // persistent grid: about four CTAs per SM over all frames (every CTA pays for zeroing and merging its histograms)
    uint32_t gx = (uint32_t)((items + 256u * 4u - 1u) / (256u * 4u));
    const uint32_t cap = (uint32_t)((592u + n - 1u) / n);
    if (gx > cap) gx = cap;
    if (gx < 1u) gx = 1u;
    const bool fast = g.w % 4u == 0 && (reinterpret_cast<uintptr_t>(d_frames) & 3u) == 0;
    if (!fast) {
        stats_kernel<<<dim3(gx, (unsigned)n), 256, 0, st>>>(d_frames, g, (uint32_t)n, d_hist, d_pairs);
        return cudaGetLastError();
    }
    unsigned long long *d_raw = nullptr;
    e = cudaMallocAsync(&d_raw, n * 3u * RAW_PER_CH * sizeof(unsigned long long), st);
    if (!e) e = cudaMemsetAsync(d_raw, 0, n * 3u * RAW_PER_CH * sizeof(unsigned long long), st);
    if (!e) {
        stats_fast_kernel<<<dim3(gx, (unsigned)n), 256, 0, st>>>(d_frames, g, d_hist, d_raw);
        raw_to_pairs_kernel<<<(unsigned)((n * 3u + 127u) / 128u), 128, 0, st>>>(d_raw, d_pairs, (uint32_t)n);
        e = cudaGetLastError();
    }
    if (d_raw) cudaFreeAsync(d_raw, st);
    return e;
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

// ---------------------------------------------------------------------------------------------------------------
// NPCR / UACI for callers that must not allocate device memory (vcrypt_npcr_uaci_device_noalloc in include/vcrypt.h).
//
// diff_kernel accumulates into 6 words per frame that have to exist somewhere in global memory and start at zero.
// diff_device gets them from its caller, who allocated them.  Here they live in the library image instead: a
// file-scope __device__ array of kDiffStaticMaxFrames x 6 words (24 KB).  Every GPU that loads libvcrypt.so carries
// its own copy from the moment the module is loaded until the process exits, whether or not this path is ever used.
//
// Two things follow from that choice and are the caller's to know:
//   * `g_diff_acc` below is a DEVICE symbol.  In host code the identifier is only a handle for the runtime; it is not
//     an address the GPU understands.  The address each device gave its copy is asked for once per device
//     (cudaGetSymbolAddress, with that device current) and kept in a small table; only that value is handed to
//     cudaMemsetAsync, to the kernel and to cudaMemcpyAsync.
//   * There is ONE array per device, shared by every context, stream and thread in the process, and it keeps what the
//     previous call left in it.  Each call clears the 6n words it is about to use, in stream order, before its kernel.
//     Two calls whose GPU work can overlap in time (different streams, or different host threads) would clear and add
//     into the same words: that is a data race with wrong results, not an error the library can detect.
// ---------------------------------------------------------------------------------------------------------------
namespace {

static __device__ __align__(256) unsigned long long g_diff_acc[kDiffStaticMaxFrames * 6u];

constexpr int kDiffStaticMaxDevices = 64;

// Device address of the current device's copy of g_diff_acc.  The first call on a device performs the lookup (which
// may also be what makes the runtime load this module onto that device); later calls read the table.
cudaError_t diff_static_address(unsigned long long **out) {
    static std::mutex mu;
    static unsigned long long *table[kDiffStaticMaxDevices] = {};
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kDiffStaticMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(mu);
    if (!table[dev]) {
        unsigned long long *ptr = nullptr;
        e = cudaGetSymbolAddress((void **)&ptr, g_diff_acc);
        if (e != cudaSuccess) return e;
        if (!ptr) return cudaErrorInvalidSymbol;
        table[dev] = ptr;
    }
    *out = table[dev];
    return cudaSuccess;
}

}  // namespace

// Same sums as diff_device, accumulated in the library's own static device array and copied to h_out (host, n x 6 words:
// per channel the number of differing bytes and the sum of |a - b|).  Calls nothing that allocates or frees device
// memory.  Waits for the stream before returning, so h_out is complete and the array is free for the next call.
// n > kDiffStaticMaxFrames: cudaErrorInvalidValue (the C entry point checks first and reports VCRYPT_E_LIMIT).
cudaError_t diff_device_static(const Geom &g, const uint8_t *d_a, const uint8_t *d_b, size_t n, unsigned long long *h_out,
                               cudaStream_t st) {
    if (!n) return cudaSuccess;
    if (n > kDiffStaticMaxFrames) return cudaErrorInvalidValue;
    unsigned long long *acc = nullptr;
    cudaError_t e = diff_static_address(&acc);
    if (e != cudaSuccess) return e;
    const size_t bytes = n * 6u * sizeof(unsigned long long);
    e = cudaMemsetAsync(acc, 0, bytes, st);  // the previous call's sums are still in there
    if (e != cudaSuccess) return e;
    uint32_t gx = (uint32_t)((g.frame_bytes / 12u + 256u * 8u - 1u) / (256u * 8u));
    if (gx > 592u) gx = 592u;
    if (gx < 1u) gx = 1u;
    diff_kernel<<<dim3(gx, (unsigned)n), 256, 0, st>>>(d_a, d_b, g.frame_bytes, acc);
    e = cudaGetLastError();
    if (e == cudaSuccess) e = cudaMemcpyAsync(h_out, acc, bytes, cudaMemcpyDeviceToHost, st);
    const cudaError_t es = cudaStreamSynchronize(st);  // also after a failure: nothing of this call may still be running
    return e != cudaSuccess ? e : es;
}

cudaError_t block_hist_device(const Geom &g, const uint8_t *d_frames, size_t n, const uint32_t *d_xy, uint32_t k, uint32_t side,
                              uint32_t *d_bh, cudaStream_t st) {
    if (!n || !k) return cudaSuccess;
    block_hist_kernel<<<dim3(k, (unsigned)n), 256, 0, st>>>(d_frames, g, d_xy, side, d_bh);
    return cudaGetLastError();
}

}  // namespace vk
