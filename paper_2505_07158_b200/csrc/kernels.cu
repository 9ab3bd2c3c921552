// kernels.cu -- hand-written sm_100a kernels for the frame cipher's GPU steps
// (Algorithms 3-7 of PAPER.md:113-156 and their inverse, :79).
//
// The paper runs five kernels over explicit 0/1 bit matrices M_t^c / M_e^c of
// size 8w x h (Algorithm 1 steps 16-20).  Those matrices are never materialised
// here.  Per channel c the five steps compose to:
//
//   hrot(i, j, c) = ( F_o(i, (j-q) mod w, c) << r  |  F_o(i, (j-q-1) mod w, c) >> (8-r) ) & 0xFF
//                   with s = d_h(i,c) mod 8w, q = s >> 3, r = s & 7          (Algo 3 + 4 + 7, Eq. 2)
//   F_e(ro, j, c) = B(ro, j, c) xor hrot((ro - d_v(j,c) mod h) mod h, j, c)   (Algo 5 + 6, Eq. 3)
//
// i.e. a per-(row, channel) bit rotation of a w-byte little-endian integer,
// followed by a per-byte-column circular shift in the interleaved H x 3W byte
// matrix, followed by a byte XOR.  Two tiled passes do exactly that with every
// global access coalesced:
//
//   row pass    : a CTA stages whole rows in shared memory, de-interleaved into
//                 three channel planes, so that the bit rotation becomes a
//                 32-bit funnel shift of two neighbouring plane words; the
//                 rotated planes are re-interleaved in registers and stored
//                 with 128-bit stores.
//   column pass : a CTA owns a strip of X byte-columns x all h rows in shared
//                 memory (row stride X = a whole number of banks, so a lane
//                 always reads its own bank: conflict-free byte gathers at
//                 data-dependent rows), then streams B in and F_e out.
//
// The intermediate between the passes lives in the output buffer (each CTA of
// the second pass reads its whole strip before it writes it), and launches are
// sized so that it stays resident in the 126 MB L2: DRAM traffic stays at the
// algorithmic read F_o + read B + write F_e.
//
// A one-thread-per-output-byte gather kernel covers every shape the tiled
// passes do not (w not a multiple of 16, or h too large for a strip).
#include "kernels.cuh"

namespace vk {

// ---------------------------------------------------------------------------------------------
// small helpers
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t pick2(uint32_t wa, int ba, uint32_t wb, int bb) {
    // byte 0 <- wa.byte[ba], byte 1 <- wb.byte[bb]
    return __byte_perm(wa, wb, (uint32_t)(ba | ((4 + bb) << 4)));
}
__device__ __forceinline__ uint32_t join2(uint32_t lo, uint32_t hi) { return __byte_perm(lo, hi, 0x5410); }

// 48 interleaved bytes (16 pixels, 12 words) -> three planes of 4 words
__device__ __forceinline__ void deinterleave16(const uint32_t (&in)[12], uint32_t (&P)[3][4]) {
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            const int i0 = 3 * (4 * m) + c, i1 = i0 + 3, i2 = i0 + 6, i3 = i0 + 9;
            P[c][m] = join2(pick2(in[i0 >> 2], i0 & 3, in[i1 >> 2], i1 & 3),
                            pick2(in[i2 >> 2], i2 & 3, in[i3 >> 2], i3 & 3));
        }
}

// three planes of 4 words -> 48 interleaved bytes
__device__ __forceinline__ void interleave16(const uint32_t (&P)[3][4], uint32_t (&out)[12]) {
#pragma unroll
    for (int n = 0; n < 12; ++n) {
        const int b0 = 4 * n, b1 = b0 + 1, b2 = b0 + 2, b3 = b0 + 3;  // byte b = 3*pixel + channel
        out[n] = join2(pick2(P[b0 % 3][(b0 / 3) >> 2], (b0 / 3) & 3, P[b1 % 3][(b1 / 3) >> 2], (b1 / 3) & 3),
                       pick2(P[b2 % 3][(b2 / 3) >> 2], (b2 / 3) & 3, P[b3 % 3][(b3 / 3) >> 2], (b3 / 3) & 3));
    }
}

__device__ __forceinline__ uint4 ld_stream(const uint4 *p) { return __ldcs(p); }
__device__ __forceinline__ void st_stream(uint4 *p, uint4 v) { __stcs(p, v); }

// ---------------------------------------------------------------------------------------------
// Row pass: horizontal bit rotation (Algorithm 4 / Eq. 2 on the rows of Algorithm 3's bit matrix,
// packed back as in Algorithm 7).  One item = 16 pixels of one row; a CTA stages `rows_per_block`
// rows.  INV = false: bit p of channel c moves to (p + d_h mod 8w) mod 8w.  INV = true: the inverse.
// Requires w % 16 == 0 and 16-byte aligned frames.  In place (dst == src) is safe: a CTA reads all
// of its rows before the barrier and writes only those rows after it.
// ---------------------------------------------------------------------------------------------
constexpr int ROW_NT = 128;

template <bool INV>
__global__ void __launch_bounds__(ROW_NT) row_pass_kernel(const uint8_t *src, uint8_t *dst,
                                                          const uint16_t *__restrict__ D, Geom g,
                                                          int rows_per_block, uint32_t total_rows) {
    extern __shared__ __align__(16) uint8_t smem[];
    const uint32_t w = g.w, W32 = w >> 2, chunks = w >> 4;
    const uint32_t plane_stride = w + 16;  // + 4 words: copy of the first 16 bytes, so a 5-word window never wraps
    const uint32_t row_stride = 3 * plane_stride;
    const uint32_t row0 = blockIdx.x * (uint32_t)rows_per_block;
    const uint32_t items = (uint32_t)rows_per_block * chunks;

    for (uint32_t item = threadIdx.x; item < items; item += ROW_NT) {
        const uint32_t rs = item / chunks, k = item - rs * chunks, grow = row0 + rs;
        if (grow >= total_rows) break;
        const uint4 *p = reinterpret_cast<const uint4 *>(src + (size_t)grow * g.row_bytes + 48u * k);
        uint4 a, b, c;
        if (INV) { a = p[0]; b = p[1]; c = p[2]; }                       // intermediate: keep L2-resident
        else { a = ld_stream(p); b = ld_stream(p + 1); c = ld_stream(p + 2); }  // plaintext: streamed once
        const uint32_t in[12] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w, c.x, c.y, c.z, c.w};
        uint32_t P[3][4];
        deinterleave16(in, P);
        uint8_t *rowbase = smem + rs * row_stride;
#pragma unroll
        for (int ch = 0; ch < 3; ++ch) {
            const uint4 v = make_uint4(P[ch][0], P[ch][1], P[ch][2], P[ch][3]);
            *reinterpret_cast<uint4 *>(rowbase + ch * plane_stride + 16u * k) = v;
            if (k == 0) *reinterpret_cast<uint4 *>(rowbase + ch * plane_stride + w) = v;
        }
    }
    __syncthreads();

    const uint32_t W8 = 8u * w;
    for (uint32_t item = threadIdx.x; item < items; item += ROW_NT) {
        const uint32_t rs = item / chunks, k = item - rs * chunks, grow = row0 + rs;
        if (grow >= total_rows) break;
        const uint32_t f = grow / g.h, i = grow - f * g.h;
        const uint16_t *Df = D + (size_t)f * g.nD;
        const uint8_t *rowbase = smem + rs * row_stride;
        uint32_t R[3][4];
#pragma unroll
        for (int ch = 0; ch < 3; ++ch) {
            const uint32_t s = (uint32_t)Df[ch * (g.h + w) + i] % W8;
            // output bit d takes source bit (d + sh) mod 8w
            const uint32_t sh = INV ? s : (s ? W8 - s : 0u);
            const uint32_t bsh = sh & 31u;
            uint32_t aw = 4u * k + (sh >> 5);
            if (aw >= W32) aw -= W32;
            const uint32_t al = aw & 3u;
            const uint4 *q = reinterpret_cast<const uint4 *>(rowbase + ch * plane_stride + 4u * (aw & ~3u));
            const uint4 q0 = q[0], q1 = q[1];
            switch (al) {  // uniform over the CTA's threads of this (row, channel)
                case 0:
                    R[ch][0] = __funnelshift_r(q0.x, q0.y, bsh); R[ch][1] = __funnelshift_r(q0.y, q0.z, bsh);
                    R[ch][2] = __funnelshift_r(q0.z, q0.w, bsh); R[ch][3] = __funnelshift_r(q0.w, q1.x, bsh);
                    break;
                case 1:
                    R[ch][0] = __funnelshift_r(q0.y, q0.z, bsh); R[ch][1] = __funnelshift_r(q0.z, q0.w, bsh);
                    R[ch][2] = __funnelshift_r(q0.w, q1.x, bsh); R[ch][3] = __funnelshift_r(q1.x, q1.y, bsh);
                    break;
                case 2:
                    R[ch][0] = __funnelshift_r(q0.z, q0.w, bsh); R[ch][1] = __funnelshift_r(q0.w, q1.x, bsh);
                    R[ch][2] = __funnelshift_r(q1.x, q1.y, bsh); R[ch][3] = __funnelshift_r(q1.y, q1.z, bsh);
                    break;
                default:
                    R[ch][0] = __funnelshift_r(q0.w, q1.x, bsh); R[ch][1] = __funnelshift_r(q1.x, q1.y, bsh);
                    R[ch][2] = __funnelshift_r(q1.y, q1.z, bsh); R[ch][3] = __funnelshift_r(q1.z, q1.w, bsh);
                    break;
            }
        }
        uint32_t o[12];
        interleave16(R, o);
        uint4 *po = reinterpret_cast<uint4 *>(dst + (size_t)grow * g.row_bytes + 48u * k);
        const uint4 o0 = make_uint4(o[0], o[1], o[2], o[3]), o1 = make_uint4(o[4], o[5], o[6], o[7]),
                    o2 = make_uint4(o[8], o[9], o[10], o[11]);
        if (INV) { st_stream(po, o0); st_stream(po + 1, o1); st_stream(po + 2, o2); }  // plaintext out: streamed
        else { po[0] = o0; po[1] = o1; po[2] = o2; }                                   // intermediate: L2-resident
    }
}

// ---------------------------------------------------------------------------------------------
// Column pass: vertical circular shift of every byte column (Algorithm 5 / Eq. 3, one d_v per pixel
// column and channel = per byte column of the interleaved matrix) fused with the XOR of Algorithm 6.
//   INV = false:  dst(ro, x) = B(ro, x) xor src((ro - t_x) mod h, x)
//   INV = true :  dst(i, x)  = (src xor B)((i + t_x) mod h, x)
// One CTA = one strip of X byte-columns of one frame, all h rows in shared memory.  Lane (sub, g) of a
// warp owns byte-columns 4g..4g+3 of the strip (one shared-memory bank, because the row stride X is a
// multiple of 128 B or divides it evenly with consecutive rows in disjoint bank groups) and row
// `sub` of the RPW = 128/X rows the warp emits per step.  In place is safe: phase A reads the whole
// strip before the barrier, phase B writes only that strip.
// ---------------------------------------------------------------------------------------------
template <int X, bool INV, int NT, int MINB, int U>
__global__ void __launch_bounds__(NT, MINB)
    col_pass_kernel(const uint8_t *src, const uint8_t *__restrict__ Bk, uint8_t *dst, const uint16_t *__restrict__ D,
                    Geom g, int strips_per_frame) {
    extern __shared__ __align__(16) uint8_t S[];
    constexpr int LPR = X / 4;     // lanes per strip row
    constexpr int RPW = 32 / LPR;  // strip rows per warp step
    constexpr int VPR = X / 16;    // 16-byte vectors per strip row
    constexpr int NW = NT / 32;
    const uint32_t f = blockIdx.x / (uint32_t)strips_per_frame;
    const uint32_t x0 = (blockIdx.x - f * (uint32_t)strips_per_frame) * X;
    const uint32_t h = g.h, rb = g.row_bytes;
    const size_t fbase = (size_t)f * g.frame_bytes + x0;
    const uint8_t *fsrc = src + fbase;
    const uint8_t *fB = Bk + fbase;
    uint8_t *fdst = dst + fbase;

    // ---- phase A: strip -> shared memory (16-byte vectors, coalesced X-byte row segments)
    {
        const uint32_t nvec = h * VPR;
        for (uint32_t v0 = threadIdx.x; v0 < nvec; v0 += NT * U) {
            uint4 val[U], kb[U];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const uint32_t v = v0 + u * NT;
                const uint32_t row = v / VPR, q = v % VPR;
                const bool ok = v < nvec && x0 + 16u * q < rb;
                val[u] = make_uint4(0, 0, 0, 0);
                kb[u] = make_uint4(0, 0, 0, 0);
                if (ok) {
                    const size_t off = (size_t)row * rb + 16u * q;
                    if (INV) {
                        val[u] = ld_stream(reinterpret_cast<const uint4 *>(fsrc + off));
                        kb[u] = ld_stream(reinterpret_cast<const uint4 *>(fB + off));
                    } else {
                        val[u] = *reinterpret_cast<const uint4 *>(fsrc + off);
                    }
                }
            }
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const uint32_t v = v0 + u * NT;
                if (v < nvec) {
                    uint4 t = val[u];
                    if (INV) { t.x ^= kb[u].x; t.y ^= kb[u].y; t.z ^= kb[u].z; t.w ^= kb[u].w; }
                    *reinterpret_cast<uint4 *>(S + (size_t)v * 16u) = t;
                }
            }
        }
    }
    __syncthreads();

    // ---- phase B: gather each byte column at its shifted row, XOR, stream out
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const uint32_t sub = lane / LPR, gc = lane % LPR;
    const uint32_t xcol = x0 + 4u * gc;
    const bool col_ok = xcol < rb;  // rb % 4 == 0 on this path, so a word is inside or outside as a whole
    const uint32_t hX = h * X;
    constexpr uint32_t STEP = NW * RPW;  // rows between two steps of one warp
    const uint32_t adv = (STEP % h) * X;
    const uint32_t r0 = warp * RPW + sub;
    uint32_t p[4];
    {
        const uint16_t *Df = D + (size_t)f * g.nD;
#pragma unroll
        for (int b = 0; b < 4; ++b) {
            uint32_t x = xcol + b;
            if (!col_ok) x = 0;
            const uint32_t j = x / 3u, c = x - 3u * j;
            const uint32_t t = (uint32_t)Df[c * (h + g.w) + h + j] % h;
            const uint32_t up = INV ? t : (t ? h - t : 0u);  // source row = (row + up) mod h
            p[b] = ((r0 + up) % h) * X + 4u * gc + b;
        }
    }
    for (uint32_t row = r0; row < h; row += STEP * U) {
        uint32_t kb[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const uint32_t rr = row + u * STEP;
            kb[u] = 0;
            if (!INV && col_ok && rr < h)
                kb[u] = __ldcs(reinterpret_cast<const uint32_t *>(fB + (size_t)rr * rb + 4u * gc));
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const uint32_t rr = row + u * STEP;
            uint32_t v = (uint32_t)S[p[0]] | ((uint32_t)S[p[1]] << 8) | ((uint32_t)S[p[2]] << 16) |
                         ((uint32_t)S[p[3]] << 24);
            v ^= kb[u];
            if (col_ok && rr < h) {
                uint32_t *po = reinterpret_cast<uint32_t *>(fdst + (size_t)rr * rb + 4u * gc);
                if (INV) *po = v;  // intermediate for the inverse row pass: L2-resident
                else __stcs(po, v);
            }
#pragma unroll
            for (int b = 0; b < 4; ++b) {
                p[b] += adv;
                if (p[b] >= hX) p[b] -= hX;
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// Any-shape kernels: the logical mapping of the paper, one thread per pixel per channel
// (PAPER.md:65), each computing its output byte from the closed form with global gathers.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
    encrypt_generic_kernel(const uint8_t *__restrict__ src, const uint16_t *__restrict__ D,
                           const uint8_t *__restrict__ Bk, uint8_t *__restrict__ dst, Geom g, size_t total) {
    const size_t idx = (size_t)blockIdx.x * 256u + threadIdx.x;
    if (idx >= total) return;
    const uint32_t w = g.w, h = g.h;
    const size_t f = idx / g.frame_bytes;
    const uint32_t rem = (uint32_t)(idx - f * g.frame_bytes);
    const uint32_t ro = rem / g.row_bytes, x = rem - ro * g.row_bytes, j = x / 3u, c = x - 3u * j;
    const uint16_t *Df = D + f * g.nD + (size_t)c * (h + w);
    const uint32_t t = (uint32_t)Df[h + j] % h;
    const uint32_t i0 = ro >= t ? ro - t : ro + h - t;
    const uint32_t s = (uint32_t)Df[i0] % (8u * w);
    const uint32_t q = (s >> 3) % w, r = s & 7u;
    const uint32_t ja = j >= q ? j - q : j + w - q;  // (j - q) mod w
    const uint32_t jb = ja ? ja - 1 : w - 1;         // (j - q - 1) mod w
    const uint8_t *row = src + f * g.frame_bytes + (size_t)i0 * g.row_bytes;
    const uint32_t a = row[3u * ja + c], b = row[3u * jb + c];
    dst[idx] = (uint8_t)((((a << 8) | b) << r) >> 8) ^ Bk[idx];
}

__global__ void __launch_bounds__(256)
    decrypt_generic_kernel(const uint8_t *__restrict__ src, const uint16_t *__restrict__ D,
                           const uint8_t *__restrict__ Bk, uint8_t *__restrict__ dst, Geom g, size_t total) {
    const size_t idx = (size_t)blockIdx.x * 256u + threadIdx.x;
    if (idx >= total) return;
    const uint32_t w = g.w, h = g.h;
    const size_t f = idx / g.frame_bytes;
    const uint32_t rem = (uint32_t)(idx - f * g.frame_bytes);
    const uint32_t i = rem / g.row_bytes, x = rem - i * g.row_bytes, j = x / 3u, c = x - 3u * j;
    const uint16_t *Df = D + f * g.nD + (size_t)c * (h + w);
    const uint32_t s = (uint32_t)Df[i] % (8u * w);
    const uint32_t q = (s >> 3) % w, r = s & 7u;
    // plaintext bit 8j+k sits at bit (8j+k+s) mod 8w of the rotated row: bytes (j+q) and (j+q+1) mod w
    uint32_t ja = j + q; if (ja >= w) ja -= w;
    uint32_t jb = ja + 1; if (jb >= w) jb -= w;
    const uint32_t ta = (uint32_t)Df[h + ja] % h, tb = (uint32_t)Df[h + jb] % h;
    uint32_t ra = i + ta; if (ra >= h) ra -= h;  // where the vertical shift put row i of column ja
    uint32_t rb2 = i + tb; if (rb2 >= h) rb2 -= h;
    const size_t fo = f * g.frame_bytes;
    const size_t oa = fo + (size_t)ra * g.row_bytes + 3u * ja + c, ob = fo + (size_t)rb2 * g.row_bytes + 3u * jb + c;
    const uint32_t a = src[oa] ^ Bk[oa], b = src[ob] ^ Bk[ob];
    dst[idx] = (uint8_t)(((b << 8) | a) >> r);
}

// ---------------------------------------------------------------------------------------------
// host side: plan + launches
// ---------------------------------------------------------------------------------------------
constexpr int COL_NT = 512;
constexpr int COL_U = 4;

template <int X, bool INV>
static cudaError_t col_set_attr(size_t smem) {
    return cudaFuncSetAttribute(col_pass_kernel<X, INV, COL_NT, 1, COL_U>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                (int)smem);
}

cudaError_t make_plan(const Geom &g, int device, Plan *out) {
    Plan p{};
    int smem_optin = 0, smem_sm = 0;
    cudaError_t e = cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, device);
    if (e != cudaSuccess) return e;
    e = cudaDeviceGetAttribute(&smem_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, device);
    if (e != cudaSuccess) return e;
    p.tiled = false;
    p.max_frames_per_launch = 1;
    if (g.w % 16 == 0) {
        // column strip: widest X whose strip leaves room for 3 CTAs per SM, else the widest that fits at all
        const int cands[4] = {128, 64, 32, 16};
        int X = 0, ctas = 0;
        for (int want = 3; want >= 1 && !X; --want)
            for (int c = 0; c < 4 && !X; ++c) {
                const size_t need = (size_t)g.h * cands[c];
                if (need <= (size_t)smem_optin && want * (need + 1024) <= (size_t)smem_sm) { X = cands[c]; ctas = want; }
            }
        p.rows_per_block = (int)(ROW_NT / (g.w / 16));
        if (p.rows_per_block < 1) p.rows_per_block = 1;
        if (p.rows_per_block > 8) p.rows_per_block = 8;
        p.smem_row = (size_t)p.rows_per_block * 3 * (g.w + 16);
        if (X && p.smem_row <= (size_t)smem_optin) {
            p.tiled = true;
            p.strip_bytes = X;
            p.strips_per_frame = (int)((g.row_bytes + X - 1) / X);
            p.smem_col = (size_t)g.h * X;
            p.col_ctas_per_sm = ctas;
            const size_t l2_budget = (size_t)48 << 20;  // intermediate kept well inside the 126 MB L2
            p.max_frames_per_launch = l2_budget / g.frame_bytes ? l2_budget / g.frame_bytes : 1;
            switch (X) {
                case 128: e = col_set_attr<128, false>(p.smem_col); if (!e) e = col_set_attr<128, true>(p.smem_col); break;
                case 64: e = col_set_attr<64, false>(p.smem_col); if (!e) e = col_set_attr<64, true>(p.smem_col); break;
                case 32: e = col_set_attr<32, false>(p.smem_col); if (!e) e = col_set_attr<32, true>(p.smem_col); break;
                default: e = col_set_attr<16, false>(p.smem_col); if (!e) e = col_set_attr<16, true>(p.smem_col); break;
            }
            if (e != cudaSuccess) return e;
            if (p.smem_row > 48 * 1024) {
                e = cudaFuncSetAttribute(row_pass_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p.smem_row);
                if (!e) e = cudaFuncSetAttribute(row_pass_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p.smem_row);
                if (e != cudaSuccess) return e;
            }
        }
    }
    *out = p;
    return cudaSuccess;
}

template <bool INV>
static cudaError_t launch_row(const Geom &g, const Plan &p, const uint8_t *src, const uint16_t *D, size_t n,
                              uint8_t *dst, cudaStream_t st) {
    const uint32_t total_rows = (uint32_t)(n * g.h);
    const uint32_t grid = (total_rows + p.rows_per_block - 1) / p.rows_per_block;
    row_pass_kernel<INV><<<grid, ROW_NT, p.smem_row, st>>>(src, dst, D, g, p.rows_per_block, total_rows);
    return cudaGetLastError();
}

template <bool INV>
static cudaError_t launch_col(const Geom &g, const Plan &p, const uint8_t *src, const uint16_t *D, const uint8_t *B,
                              size_t n, uint8_t *dst, cudaStream_t st) {
    const uint32_t grid = (uint32_t)(n * p.strips_per_frame);
    switch (p.strip_bytes) {
        case 128: col_pass_kernel<128, INV, COL_NT, 1, COL_U><<<grid, COL_NT, p.smem_col, st>>>(src, B, dst, D, g, p.strips_per_frame); break;
        case 64: col_pass_kernel<64, INV, COL_NT, 1, COL_U><<<grid, COL_NT, p.smem_col, st>>>(src, B, dst, D, g, p.strips_per_frame); break;
        case 32: col_pass_kernel<32, INV, COL_NT, 1, COL_U><<<grid, COL_NT, p.smem_col, st>>>(src, B, dst, D, g, p.strips_per_frame); break;
        default: col_pass_kernel<16, INV, COL_NT, 1, COL_U><<<grid, COL_NT, p.smem_col, st>>>(src, B, dst, D, g, p.strips_per_frame); break;
    }
    return cudaGetLastError();
}

cudaError_t encrypt_tiled(const Geom &g, const Plan &p, const uint8_t *src, const uint16_t *D, const uint8_t *B,
                          size_t n, uint8_t *dst, cudaStream_t st, int *launches) {
    for (size_t f0 = 0; f0 < n; f0 += p.max_frames_per_launch) {
        const size_t m = n - f0 < p.max_frames_per_launch ? n - f0 : p.max_frames_per_launch;
        const size_t off = f0 * g.frame_bytes;
        cudaError_t e = launch_row<false>(g, p, src + off, D + f0 * g.nD, m, dst + off, st);
        if (e != cudaSuccess) return e;
        e = launch_col<false>(g, p, dst + off, D + f0 * g.nD, B + off, m, dst + off, st);
        if (e != cudaSuccess) return e;
        *launches += 2;
    }
    return cudaSuccess;
}

cudaError_t decrypt_tiled(const Geom &g, const Plan &p, const uint8_t *src, const uint16_t *D, const uint8_t *B,
                          size_t n, uint8_t *dst, cudaStream_t st, int *launches) {
    for (size_t f0 = 0; f0 < n; f0 += p.max_frames_per_launch) {
        const size_t m = n - f0 < p.max_frames_per_launch ? n - f0 : p.max_frames_per_launch;
        const size_t off = f0 * g.frame_bytes;
        cudaError_t e = launch_col<true>(g, p, src + off, D + f0 * g.nD, B + off, m, dst + off, st);
        if (e != cudaSuccess) return e;
        e = launch_row<true>(g, p, dst + off, D + f0 * g.nD, m, dst + off, st);
        if (e != cudaSuccess) return e;
        *launches += 2;
    }
    return cudaSuccess;
}

cudaError_t encrypt_generic(const Geom &g, const uint8_t *src, const uint16_t *D, const uint8_t *B, size_t n,
                            uint8_t *dst, cudaStream_t st, int *launches) {
    const size_t total = n * g.frame_bytes;
    // keep each grid below 2^31 blocks
    const size_t per = ((size_t)1 << 30) / g.frame_bytes ? ((size_t)1 << 30) / g.frame_bytes : 1;
    for (size_t f0 = 0; f0 < n; f0 += per) {
        const size_t m = n - f0 < per ? n - f0 : per, tot = m * g.frame_bytes, off = f0 * g.frame_bytes;
        encrypt_generic_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, st>>>(src + off, D + f0 * g.nD, B + off,
                                                                               dst + off, g, tot);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
        *launches += 1;
    }
    (void)total;
    return cudaSuccess;
}

cudaError_t decrypt_generic(const Geom &g, const uint8_t *src, const uint16_t *D, const uint8_t *B, size_t n,
                            uint8_t *dst, cudaStream_t st, int *launches) {
    const size_t per = ((size_t)1 << 30) / g.frame_bytes ? ((size_t)1 << 30) / g.frame_bytes : 1;
    for (size_t f0 = 0; f0 < n; f0 += per) {
        const size_t m = n - f0 < per ? n - f0 : per, tot = m * g.frame_bytes, off = f0 * g.frame_bytes;
        decrypt_generic_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, st>>>(src + off, D + f0 * g.nD, B + off,
                                                                               dst + off, g, tot);
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) return e;
        *launches += 1;
    }
    return cudaSuccess;
}

}  // namespace vk
