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
// matrix, followed by a byte XOR.  Two tiled passes do exactly that:
//
//   row pass    : work unit = a block of 4 rows; persistent CTAs run a three-buffer ring.  The rows
//                 arrive in shared memory with one bulk async copy (TMA, cp.async.bulk), two blocks
//                 ahead of the one being computed, are de-interleaved into three channel planes so
//                 that the bit rotation becomes a 32-bit funnel shift of two neighbouring plane
//                 words, and leave with one bulk async store.  When encrypting, the block is
//                 written in the "T4" layout: the word at (row 4R + (x & 3), word column x >> 2)
//                 holds byte column x of rows 4R .. 4R+3 -- a permutation inside the block, so the
//                 intermediate still lives in the output buffer.
//   column pass : a CTA owns a strip of X byte columns x all h rows in shared memory, in the T4
//                 layout, so that ONE 32-bit shared-memory load returns four consecutive rows of a
//                 byte column: 8 output rows of a column cost 3 conflict-free loads instead of 8
//                 byte loads.  The words are byte-aligned and transposed back to row-major in
//                 registers (PRMT), XORed with the keystream and streamed out.
//
// The intermediate between the passes lives in the output buffer (every CTA of either pass reads all
// of its rows / its whole strip before it writes them), and launches are sized so that it stays
// resident in the 126 MB L2: DRAM traffic stays at the algorithmic read F_o + read B + write F_e.
//
// A one-thread-per-output-byte gather kernel covers every shape the tiled passes do not
// (w % 16 != 0, h % 4 != 0, h < 16, or a strip / row block too large for shared memory).
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

// 4 x 4 byte transpose: out[b].byte[j] = in[j].byte[b]
__device__ __forceinline__ void transpose4x4(const uint32_t (&in)[4], uint32_t (&out)[4]) {
    const uint32_t t01a = __byte_perm(in[0], in[1], 0x5140), t01b = __byte_perm(in[0], in[1], 0x7362);
    const uint32_t t23a = __byte_perm(in[2], in[3], 0x5140), t23b = __byte_perm(in[2], in[3], 0x7362);
    out[0] = __byte_perm(t01a, t23a, 0x5410);
    out[1] = __byte_perm(t01a, t23a, 0x7632);
    out[2] = __byte_perm(t01b, t23b, 0x5410);
    out[3] = __byte_perm(t01b, t23b, 0x7632);
}

// ---- async-copy / mbarrier PTX (sm_90+; SASS: UBLKCP, SYNCS) -----------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint64_t *bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t *bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t *bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
// Bounded wait: a copy that never lands must trap, not hang the GPU.
__device__ __forceinline__ void mbar_wait(uint64_t *bar, uint32_t parity) {
    for (uint32_t spin = 0; !mbar_try_wait(bar, parity); ++spin)
        if (spin > (1u << 24)) __trap();
}
// global -> shared bulk copy (16-byte aligned, size multiple of 16), completion on the mbarrier
__device__ __forceinline__ void bulk_g2s(void *smem_dst, const void *gsrc, uint32_t bytes, uint64_t *bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(smem_dst)),
                 "l"(__cvta_generic_to_global(gsrc)), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
// shared -> global bulk copy
__device__ __forceinline__ void bulk_s2g(void *gdst, const void *smem_src, uint32_t bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(__cvta_generic_to_global(gdst)),
                 "r"(smem_u32(smem_src)), "r"(bytes)
                 : "memory");
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
}
__device__ __forceinline__ void bulk_wait_read_1() { asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_all() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }
__device__ __forceinline__ void fence_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

// 16-byte cp.async (LDGSTS), L2 only
__device__ __forceinline__ void cp_async16(void *smem_dst, const void *gsrc) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(smem_u32(smem_dst)), "l"(__cvta_generic_to_global(gsrc))
                 : "memory");
}
__device__ __forceinline__ void cp_async_wait_all() {
    asm volatile("cp.async.commit_group;" ::: "memory");
    asm volatile("cp.async.wait_group 0;" ::: "memory");
}

// Gathers four bytes, each from a register of `r` (index i*) at byte position b*, into one word.
// All indices are compile-time constants after unrolling, so the selector arithmetic folds away:
// 1 PRMT for <= 2 distinct registers, 2 for 3, 3 for 4.
__device__ __forceinline__ uint32_t gather4(const uint32_t *r, int i0, int b0, int i1, int b1, int i2, int b2, int i3,
                                            int b3) {
    const int idx[4] = {i0, i1, i2, i3}, by[4] = {b0, b1, b2, b3};
    int u[4] = {i0, -1, -1, -1}, nu = 1, slot[4] = {0, 0, 0, 0};
#pragma unroll
    for (int k = 1; k < 4; ++k) {
        int found = -1;
#pragma unroll
        for (int q = 0; q < 4; ++q)
            if (q < nu && u[q] == idx[k]) found = q;
        if (found < 0) { u[nu] = idx[k]; found = nu; ++nu; }
        slot[k] = found;
    }
    if (nu <= 2) {
        uint32_t sel = 0;
#pragma unroll
        for (int k = 0; k < 4; ++k) sel |= (uint32_t)(by[k] + 4 * slot[k]) << (4 * k);
        return __byte_perm(r[u[0]], r[nu > 1 ? u[1] : u[0]], sel);
    }
    // first PRMT: bytes living in u0 / u1 land at their final position k
    uint32_t sel1 = 0, sel2 = 0;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
        if (slot[k] < 2) { sel1 |= (uint32_t)(by[k] + 4 * slot[k]) << (4 * k); sel2 |= (uint32_t)k << (4 * k); }
        else if (slot[k] == 2) sel2 |= (uint32_t)(4 + by[k]) << (4 * k);
    }
    uint32_t t = __byte_perm(__byte_perm(r[u[0]], r[u[1]], sel1), r[u[2]], sel2);
    if (nu == 4) {
        uint32_t sel3 = 0;
#pragma unroll
        for (int k = 0; k < 4; ++k) sel3 |= (uint32_t)(slot[k] == 3 ? 4 + by[k] : k) << (4 * k);
        t = __byte_perm(t, r[u[3]], sel3);
    }
    return t;
}

// ---------------------------------------------------------------------------------------------
// Row pass: horizontal bit rotation (Algorithm 4 / Eq. 2 on the rows of Algorithm 3's bit matrix,
// packed back as in Algorithm 7).  Work unit = one block of 4 consecutive rows of one frame (h % 4 == 0,
// so a block never straddles two frames); one item = 16 pixels (48 bytes) of each of the 4 rows.
//   INV = false: bit p of channel c moves to (p + d_h mod 8w) mod 8w; the block is written in T4 layout.
//   INV = true : the inverse rotation; input and output are row-major.
// Persistent CTAs walk the blocks round-robin with a three-buffer ring: while block i is being rotated,
// the bulk async load (TMA, cp.async.bulk) of blocks i+1 and i+2 and the bulk store of block i-1 are in
// flight.  A buffer is: loaded -> de-interleaved into planes -> overwritten with the rotated block ->
// stored.  A plane (one row, one channel: w/4 words) is kept as chunks of 4 words at a stride of 5 words
// (odd: thread k's chunk sits at bank 5k + i, no conflicts), plus a copy of chunk 0 at the end so that the
// 5-word window of a funnel shift never wraps.
// In place (dst == src) is safe: a block is read completely before it is written.
// ---------------------------------------------------------------------------------------------
constexpr int ROW_RB = 4;      // rows per block
constexpr int ROW_HDR = 256;   // 3 mbarriers + 2 x 12 shift parameters
constexpr int ROW_NBUF = 3;

// shift parameter of one (row, channel): bits 0-4 bit shift, 8-9 first slot, 16-31 chunk shift
__device__ __forceinline__ uint32_t row_param(const uint16_t *__restrict__ D, const Geom &g, uint32_t grow, uint32_t ch,
                                              bool inv) {
    const uint32_t f = grow / g.h, i = grow - f * g.h, W8 = 8u * g.w;
    const uint32_t s = (uint32_t)D[(size_t)f * g.nD + ch * (g.h + g.w) + i] % W8;
    const uint32_t sh = inv ? s : (s ? W8 - s : 0u);  // output bit d takes source bit (d + sh) mod 8w
    const uint32_t dw = sh >> 5;                      // source word offset
    return (sh & 31u) | ((dw & 3u) << 8) | ((dw >> 2) << 16);
}

template <bool INV>
__global__ void __launch_bounds__(256) row_pass_kernel(const uint8_t *src, uint8_t *dst, const uint16_t *__restrict__ D,
                                                       Geom g, uint32_t nblocks) {
    extern __shared__ __align__(128) uint8_t smem[];
    uint64_t *bar = reinterpret_cast<uint64_t *>(smem);           // [ROW_NBUF]
    uint32_t *par = reinterpret_cast<uint32_t *>(smem + 64);      // [2][16]
    const uint32_t w = g.w, rb = g.row_bytes, C = w >> 4;          // C items per row
    const uint32_t blk_bytes = ROW_RB * rb;
    const uint32_t plane_stride = 20u * (C + 1u);                  // bytes: (C + 1) chunks of 5 words
    uint8_t *stage0 = smem + ROW_HDR;
    uint8_t *planes = stage0 + ROW_NBUF * blk_bytes;
    const uint32_t G = gridDim.x, tid = threadIdx.x;

    uint32_t blk = blockIdx.x;
    if (blk >= nblocks) return;
    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < ROW_NBUF; ++s) mbar_init(bar + s, 1);
        mbar_expect_tx(bar + 0, blk_bytes);
        bulk_g2s(stage0, src + (size_t)blk * blk_bytes, blk_bytes, bar + 0);
        if (blk + G < nblocks) {
            mbar_expect_tx(bar + 1, blk_bytes);
            bulk_g2s(stage0 + blk_bytes, src + (size_t)(blk + G) * blk_bytes, blk_bytes, bar + 1);
        }
    }
    if (tid < 3 * ROW_RB) par[tid] = row_param(D, g, blk * ROW_RB + tid / 3u, tid % 3u, INV);
    __syncthreads();  // mbarriers initialised, parameters of the first block visible

    uint32_t s = 0;
    for (uint32_t it = 0; blk < nblocks; ++it, blk += G) {
        uint8_t *stage = stage0 + s * blk_bytes;
        const uint32_t *pc = par + (it & 1u) * 16u;
        uint32_t pnext = 0;
        if (tid < 3 * ROW_RB && blk + G < nblocks) pnext = row_param(D, g, (blk + G) * ROW_RB + tid / 3u, tid % 3u, INV);
        mbar_wait(bar + s, (it / ROW_NBUF) & 1u);

        // ---- de-interleave into planes
        for (uint32_t k = tid; k < C; k += blockDim.x) {
#pragma unroll
            for (int r = 0; r < ROW_RB; ++r) {
                const uint4 *p = reinterpret_cast<const uint4 *>(stage + r * rb + 48u * k);
                const uint4 a = p[0], b = p[1], c = p[2];
                const uint32_t in[12] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w, c.x, c.y, c.z, c.w};
#pragma unroll
                for (int ch = 0; ch < 3; ++ch) {
                    uint32_t *pb = reinterpret_cast<uint32_t *>(planes + (r * 3 + ch) * plane_stride) + 5u * k;
#pragma unroll
                    for (int m = 0; m < 4; ++m) {
                        const int o = 12 * m + ch;  // byte offsets o, o+3, o+6, o+9 of the 48
                        const uint32_t v = gather4(in, o >> 2, o & 3, (o + 3) >> 2, (o + 3) & 3, (o + 6) >> 2, (o + 6) & 3,
                                                   (o + 9) >> 2, (o + 9) & 3);
                        pb[m] = v;
                        if (k == 0) pb[5u * C + m] = v;
                    }
                }
            }
        }
        __syncthreads();  // planes complete; the raw block in `stage` may now be overwritten

        // ---- rotate, re-interleave, write the output block over the input block
        for (uint32_t k = tid; k < C; k += blockDim.x) {
            uint32_t R[ROW_RB * 3 * 4];  // [r][ch][word]
#pragma unroll
            for (int r = 0; r < ROW_RB; ++r)
#pragma unroll
                for (int ch = 0; ch < 3; ++ch) {
                    const uint32_t pv = pc[r * 3 + ch];
                    const uint32_t slot0 = (pv >> 8) & 3u;
                    uint32_t kb = k + (pv >> 16);
                    if (kb >= C) kb -= C;
                    const uint32_t *q = reinterpret_cast<const uint32_t *>(planes + (r * 3 + ch) * plane_stride) + 5u * kb + slot0;
                    const uint32_t v0 = q[0], v1 = q[1], v2 = q[2], v3 = q[3], v4 = q[4], v5 = q[5];
                    // the window skips the unused 5th word of a chunk after (4 - slot0) words
                    const uint32_t w1 = slot0 == 3u ? v2 : v1, w2 = slot0 >= 2u ? v3 : v2, w3 = slot0 >= 1u ? v4 : v3;
                    uint32_t *o = R + (r * 3 + ch) * 4;
                    o[0] = __funnelshift_r(v0, w1, pv);  // shift amount = pv & 31
                    o[1] = __funnelshift_r(w1, w2, pv);
                    o[2] = __funnelshift_r(w2, w3, pv);
                    o[3] = __funnelshift_r(w3, v5, pv);
                }
#pragma unroll
            for (int ro = 0; ro < 4; ++ro) {
                uint32_t o[12];
#pragma unroll
                for (int m = 0; m < 12; ++m) {
                    if (INV) {  // row-major: row ro, bytes 4m .. 4m+3 of the 48
                        const int x0 = 4 * m, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3;
                        o[m] = gather4(R + ro * 12, (x0 % 3) * 4 + ((x0 / 3) >> 2), (x0 / 3) & 3, (x1 % 3) * 4 + ((x1 / 3) >> 2),
                                       (x1 / 3) & 3, (x2 % 3) * 4 + ((x2 / 3) >> 2), (x2 / 3) & 3,
                                       (x3 % 3) * 4 + ((x3 / 3) >> 2), (x3 / 3) & 3);
                    } else {  // T4: block row ro, word m = byte column 4m + ro of rows 0..3
                        const int x = 4 * m + ro, ri = (x % 3) * 4 + ((x / 3) >> 2), by = (x / 3) & 3;
                        o[m] = gather4(R, ri, by, 12 + ri, by, 24 + ri, by, 36 + ri, by);
                    }
                }
                uint4 *po = reinterpret_cast<uint4 *>(stage + ro * rb + 48u * k);
                po[0] = make_uint4(o[0], o[1], o[2], o[3]);
                po[1] = make_uint4(o[4], o[5], o[6], o[7]);
                po[2] = make_uint4(o[8], o[9], o[10], o[11]);
            }
        }
        if (tid < 3 * ROW_RB) par[((it + 1u) & 1u) * 16u + tid] = pnext;
        fence_async_smem();  // generic-proxy writes to the stage -> visible to the bulk store
        __syncthreads();
        if (tid == 0) {
            bulk_s2g(dst + (size_t)blk * blk_bytes, stage, blk_bytes);
            const uint32_t nb = blk + 2u * G;
            if (nb < nblocks) {
                const uint32_t s2 = s >= 1 ? s - 1 : ROW_NBUF - 1;  // (s + 2) % 3: the buffer of block it - 1
                bulk_wait_read_1();                                 // its store has left shared memory
                mbar_expect_tx(bar + s2, blk_bytes);
                bulk_g2s(stage0 + s2 * blk_bytes, src + (size_t)nb * blk_bytes, blk_bytes, bar + s2);
            }
        }
        s = s + 1 == ROW_NBUF ? 0 : s + 1;
    }
    if (tid == 0) bulk_wait_all();
}

// ---------------------------------------------------------------------------------------------
// Column pass: vertical circular shift of every byte column (Algorithm 5 / Eq. 3, one d_v per pixel
// column and channel = per byte column of the interleaved matrix) fused with the XOR of Algorithm 6.
//   INV = false:  dst(ro, x) = B(ro, x) xor I((ro - t_x) mod h, x)      src = I in T4 layout
//   INV = true :  dst(i, x)  = (src xor B)((i + t_x) mod h, x)          src = F_e row-major; dst row-major
// One CTA = one strip of X byte columns of one frame: h + 8 strip rows of X bytes in shared memory in T4
// layout (strip row 4R + b, word l = rows 4R..4R+3 of byte column 4l + b; the last 8 strip rows repeat the
// first 8 so that a window never wraps).  A warp is split into NSUB = 128 / X sub-warps of X / 4 lanes;
// lane l of a sub-warp owns byte columns 4l .. 4l+3 of the strip and the sub-warp emits groups of 8
// consecutive output rows: per byte column 3 word loads (12 source rows), a byte alignment (PRMT) and a
// 4 x 4 byte transpose back to row-major words.  Bank of a load = (strip row * X/4 + l) mod 32 with strip
// row = 4R + b, i.e. (b * X/4 + l) mod 32: sub-warp s walks the byte columns in the order b = a xor s, so
// the sub-warps of a warp always sit in disjoint bank groups.  No conflicts for X = 128, 64, 32.
// The keystream words of the next group are fetched while the current one is gathered.
// In place is safe: phase A reads the whole strip before the barrier, phase B writes only that strip.
// ---------------------------------------------------------------------------------------------
constexpr int COL_G = 8;    // output rows per group
constexpr int COL_PAD = 8;  // repeated strip rows

template <int X, bool INV, int NT, int MINB>
__global__ void __launch_bounds__(NT, MINB)
    col_pass_kernel(const uint8_t *src, const uint8_t *__restrict__ Bk, uint8_t *dst, const uint16_t *__restrict__ D,
                    Geom g, int strips_per_frame) {
    extern __shared__ __align__(128) uint8_t S[];
    constexpr int LPR = X / 4;      // lanes per strip row
    constexpr int NSUB = 32 / LPR;  // sub-warps per warp
    constexpr int NW = NT / 32;
    const uint32_t f = blockIdx.x / (uint32_t)strips_per_frame;
    const uint32_t x0 = (blockIdx.x - f * (uint32_t)strips_per_frame) * X;
    const uint32_t h = g.h, rb = g.row_bytes;
    const size_t fbase = (size_t)f * g.frame_bytes + x0;
    const uint8_t *fsrc = src + fbase;

    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const uint32_t sub = lane / LPR, l = lane % LPR;
    const uint32_t xw = x0 + 4u * l;  // first of this lane's 4 byte columns (frame coordinates)
    const bool col_ok = xw < rb;      // rb % 4 == 0 on this path: a word is inside or outside as a whole
    constexpr uint32_t GSTEP = NW * NSUB;  // groups between two iterations of a sub-warp
    const uint32_t g0 = warp * NSUB + sub; // first group of this sub-warp
    const uint32_t ngroups = (h + COL_G - 1) / COL_G;
    // this lane's word in row r of the frame sits at word offset r * rw of these (32-bit indexing)
    const uint32_t rw = rb >> 2;
    const uint32_t *Bw = reinterpret_cast<const uint32_t *>(Bk + fbase) + l;
    uint32_t *Ow = reinterpret_cast<uint32_t *>(dst + fbase) + l;

    // keystream words of the first group: issued before the strip arrives
    uint32_t kb[COL_G];
#pragma unroll
    for (int i = 0; i < COL_G; ++i) kb[i] = 0;
    if (!INV && col_ok && g0 < ngroups) {
        const uint32_t ro = g0 * COL_G;
#pragma unroll
        for (int i = 0; i < COL_G; ++i)
            if (ro + i < h) kb[i] = __ldcs(Bw + (ro + i) * rw);
    }

    // ---- phase A: strip -> shared memory
    if (!INV) {
        constexpr int VPR = X / 16;  // 16-byte vectors per strip row
        const uint32_t nvec = (h + COL_PAD) * VPR;
        for (uint32_t v = threadIdx.x; v < nvec; v += NT) {
            const uint32_t row = v / VPR, q = v % VPR;
            const uint32_t srow = row < h ? row : row - h;
            if (x0 + 16u * q < rb) cp_async16(S + (size_t)v * 16u, fsrc + (size_t)srow * rb + 16u * q);
        }
        cp_async_wait_all();
    } else {
        // row-major F_e xor B -> T4: one item = (block of 4 rows, word column)
        const uint32_t nblk = (h + COL_PAD) >> 2, hb = h >> 2;
        const uint32_t *Sw = reinterpret_cast<const uint32_t *>(fsrc);
        const uint32_t *Bw0 = reinterpret_cast<const uint32_t *>(Bk + fbase);
        for (uint32_t it = threadIdx.x; it < nblk * LPR; it += NT) {
            const uint32_t R4 = it / LPR, ll = it % LPR;
            const uint32_t sR = R4 < hb ? R4 : R4 - hb;
            uint32_t v[4] = {0, 0, 0, 0}, o[4];
            if (x0 + 4u * ll < rb) {
                uint32_t kk[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const uint32_t off = (4u * sR + j) * rw + ll;
                    v[j] = __ldcs(Sw + off);
                    kk[j] = __ldcs(Bw0 + off);
                }
#pragma unroll
                for (int j = 0; j < 4; ++j) v[j] ^= kk[j];
            }
            transpose4x4(v, o);
#pragma unroll
            for (int b = 0; b < 4; ++b) *reinterpret_cast<uint32_t *>(S + ((size_t)(4u * R4 + b) * LPR + ll) * 4u) = o[b];
        }
    }

    // per byte column: source pointer, wrap limit, alignment selector
    const uint32_t hX = h * X;
    constexpr uint32_t ADV = GSTEP * COL_G * X;  // bytes of strip between two iterations
    uint32_t p[4], lim[4], sel[4];
    {
        const uint16_t *Df = D + (size_t)f * g.nD;
#pragma unroll
        for (int a = 0; a < 4; ++a) {
            const uint32_t b = (uint32_t)a ^ (sub & 3u);  // byte column walked at step a (NSUB <= 4)
            uint32_t x = xw + b;
            if (!col_ok) x = b;
            const uint32_t j = x / 3u, c = x - 3u * j;
            const uint32_t t = (uint32_t)Df[c * (h + g.w) + h + j] % h;
            const uint32_t up = INV ? t : (t ? h - t : 0u);  // source row = (row + up) mod h
            uint32_t s0 = (g0 * COL_G) % h + up;
            if (s0 >= h) s0 -= h;
            const uint32_t al = s0 & 3u;
            sel[a] = 0x3210u + 0x1111u * al;
            const uint32_t cst = b * X + 4u * l;
            p[a] = (s0 - al) * X + cst;
            lim[a] = hX + cst;
        }
    }
    // transpose selectors: A[0], A[1] hold byte columns (s, s^1), A[2], A[3] hold (s^2, s^3)
    const uint32_t selA = (sub & 1u) ? 0x1504u : 0x5140u, selB = (sub & 1u) ? 0x3726u : 0x7362u;
    const uint32_t selLo = (sub & 2u) ? 0x1054u : 0x5410u, selHi = (sub & 2u) ? 0x3276u : 0x7632u;
    __syncthreads();

    // ---- phase B: per byte column, 8 output rows at a time
    for (uint32_t gi = g0; gi < ngroups; gi += GSTEP) {
        const uint32_t ro = gi * COL_G;
        const bool full = ro + COL_G <= h;
        // next group's keystream
        uint32_t kn[COL_G];
#pragma unroll
        for (int i = 0; i < COL_G; ++i) kn[i] = 0;
        if (!INV && col_ok && gi + GSTEP < ngroups) {
            const uint32_t rn = ro + GSTEP * COL_G;
            if (rn + COL_G <= h) {
#pragma unroll
                for (int i = 0; i < COL_G; ++i) kn[i] = __ldcs(Bw + (rn + i) * rw);
            } else {
#pragma unroll
                for (int i = 0; i < COL_G; ++i)
                    if (rn + i < h) kn[i] = __ldcs(Bw + (rn + i) * rw);
            }
        }
        uint32_t A[4][2];
#pragma unroll
        for (int a = 0; a < 4; ++a) {
            const uint8_t *q = S + p[a];
            const uint32_t r0 = *reinterpret_cast<const uint32_t *>(q);
            const uint32_t r1 = *reinterpret_cast<const uint32_t *>(q + 4 * X);
            const uint32_t r2 = *reinterpret_cast<const uint32_t *>(q + 8 * X);
            A[a][0] = __byte_perm(r0, r1, sel[a]);
            A[a][1] = __byte_perm(r1, r2, sel[a]);
            p[a] += ADV;
            if (p[a] >= lim[a]) p[a] -= hX;
        }
        uint32_t o[COL_G];
#pragma unroll
        for (int hg = 0; hg < 2; ++hg) {
            const uint32_t t01a = __byte_perm(A[0][hg], A[1][hg], selA), t01b = __byte_perm(A[0][hg], A[1][hg], selB);
            const uint32_t t23a = __byte_perm(A[2][hg], A[3][hg], selA), t23b = __byte_perm(A[2][hg], A[3][hg], selB);
            o[4 * hg + 0] = __byte_perm(t01a, t23a, selLo) ^ kb[4 * hg + 0];
            o[4 * hg + 1] = __byte_perm(t01a, t23a, selHi) ^ kb[4 * hg + 1];
            o[4 * hg + 2] = __byte_perm(t01b, t23b, selLo) ^ kb[4 * hg + 2];
            o[4 * hg + 3] = __byte_perm(t01b, t23b, selHi) ^ kb[4 * hg + 3];
        }
        if (col_ok) {
            uint32_t *po = Ow + ro * rw;
            if (full) {
#pragma unroll
                for (int i = 0; i < COL_G; ++i) {
                    if (INV) po[i * rw] = o[i];  // intermediate for the inverse row pass: keep it L2-resident
                    else __stcs(po + i * rw, o[i]);
                }
            } else {
#pragma unroll
                for (int i = 0; i < COL_G; ++i)
                    if (ro + i < h) {
                        if (INV) po[i * rw] = o[i];
                        else __stcs(po + i * rw, o[i]);
                    }
            }
        }
#pragma unroll
        for (int i = 0; i < COL_G; ++i) kb[i] = kn[i];
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
static size_t row_smem_bytes(const Geom &g) {
    const size_t C = g.w / 16;
    return (size_t)ROW_HDR + (size_t)ROW_NBUF * ROW_RB * g.row_bytes + (size_t)ROW_RB * 3 * 20 * (C + 1);
}
static size_t col_smem_bytes(const Geom &g, int X) { return (size_t)(g.h + COL_PAD) * X; }

template <int X, int NT, int MINB>
static cudaError_t col_set_attr(size_t smem) {
    cudaError_t e = cudaFuncSetAttribute(col_pass_kernel<X, false, NT, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(col_pass_kernel<X, true, NT, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    return e;
}

cudaError_t make_plan(const Geom &g, int device, Plan *out) {
    Plan p{};
    int smem_optin = 0, smem_sm = 0, sms = 0;
    cudaError_t e = cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&smem_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
    if (e != cudaSuccess) return e;
    p.tiled = false;
    p.max_frames_per_launch = 1;
    if (g.w % 16 == 0 && g.h % 4 == 0 && g.h >= 2 * COL_PAD) {
        // column strip: the widest X that leaves room for 3 CTAs per SM (256 threads each); else the
        // widest that fits at all (one CTA of 512 threads per SM)
        const int cands[3] = {128, 64, 32};
        int X = 0, ctas = 0;
        for (int c = 0; c < 3 && !X; ++c)
            if (3 * (col_smem_bytes(g, cands[c]) + 1024) <= (size_t)smem_sm) { X = cands[c]; ctas = 3; }
        for (int c = 0; c < 3 && !X; ++c)
            if (col_smem_bytes(g, cands[c]) <= (size_t)smem_optin) { X = cands[c]; ctas = 1; }
        p.smem_row = row_smem_bytes(g);
        if (X && p.smem_row <= (size_t)smem_optin) {
            p.tiled = true;
            p.strip_bytes = X;
            p.col_ctas_per_sm = ctas;
            p.strips_per_frame = (int)((g.row_bytes + X - 1) / X);
            p.smem_col = col_smem_bytes(g, X);
            p.row_threads = g.w / 16 <= 128 ? (int)(((g.w / 16 + 31) / 32) * 32) : 256;
            int rc = (int)((size_t)smem_sm / (p.smem_row + 1024));
            if (rc > 4) rc = 4;
            if (rc < 1) rc = 1;
            p.row_grid_max = rc * sms;
            const size_t l2_budget = (size_t)56 << 20;  // intermediate kept well inside the 126 MB L2
            p.max_frames_per_launch = l2_budget / g.frame_bytes ? l2_budget / g.frame_bytes : 1;
            if (ctas == 3) {
                if (X == 128) e = col_set_attr<128, 256, 3>(p.smem_col);
                else if (X == 64) e = col_set_attr<64, 256, 3>(p.smem_col);
                else e = col_set_attr<32, 256, 3>(p.smem_col);
            } else {
                if (X == 128) e = col_set_attr<128, 512, 1>(p.smem_col);
                else if (X == 64) e = col_set_attr<64, 512, 1>(p.smem_col);
                else e = col_set_attr<32, 512, 1>(p.smem_col);
            }
            if (e != cudaSuccess) return e;
            e = cudaFuncSetAttribute(row_pass_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p.smem_row);
            if (!e) e = cudaFuncSetAttribute(row_pass_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p.smem_row);
            if (e != cudaSuccess) return e;
        }
    }
    *out = p;
    return cudaSuccess;
}

template <bool INV>
static cudaError_t launch_row(const Geom &g, const Plan &p, const uint8_t *src, const uint16_t *D, size_t n,
                              uint8_t *dst, cudaStream_t st) {
    const uint32_t nblocks = (uint32_t)(n * g.h / ROW_RB);
    const uint32_t grid = nblocks < (uint32_t)p.row_grid_max ? nblocks : (uint32_t)p.row_grid_max;
    row_pass_kernel<INV><<<grid, p.row_threads, p.smem_row, st>>>(src, dst, D, g, nblocks);
    return cudaGetLastError();
}

template <bool INV>
static cudaError_t launch_col(const Geom &g, const Plan &p, const uint8_t *src, const uint16_t *D, const uint8_t *B,
                              size_t n, uint8_t *dst, cudaStream_t st) {
    const uint32_t grid = (uint32_t)(n * p.strips_per_frame);
#define VK_COL(X, NT, MINB) col_pass_kernel<X, INV, NT, MINB><<<grid, NT, p.smem_col, st>>>(src, B, dst, D, g, p.strips_per_frame)
    if (p.col_ctas_per_sm == 3) {
        if (p.strip_bytes == 128) VK_COL(128, 256, 3);
        else if (p.strip_bytes == 64) VK_COL(64, 256, 3);
        else VK_COL(32, 256, 3);
    } else {
        if (p.strip_bytes == 128) VK_COL(128, 512, 1);
        else if (p.strip_bytes == 64) VK_COL(64, 512, 1);
        else VK_COL(32, 512, 1);
    }
#undef VK_COL
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
