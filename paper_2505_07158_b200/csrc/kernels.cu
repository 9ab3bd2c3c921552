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
//   row pass    : work unit = a block of 4 rows.  Two variants of the same two phases: row_reg_kernel (frames up to 4096
//                 pixels wide: a block lands in the threads' registers, three to four small CTAs per SM) and
//                 row_pass_kernel, described here.  Warp-specialised persistent CTAs: a copy warp brings
//                 blocks in with bulk async copies (TMA, cp.async.bulk) into a ring of stages and sends
//                 finished blocks out with bulk async stores; the compute warps de-interleave a block
//                 into three channel planes (already rotated by the whole-chunk part of the distance),
//                 so that the bit rotation becomes ONE 32-bit funnel shift of two neighbouring plane
//                 words per output word.  When encrypting, the block is written in the "T4" layout: the
//                 word at (row 4R + (x & 3), word column x >> 2) holds byte column x of rows 4R .. 4R+3
//                 -- a permutation inside the block, so the intermediate still lives in the output buffer.
//   column pass : a CTA owns a strip of 64 byte columns x all h rows in shared memory, in the T4 layout
//                 (encrypt: brought in by TMA tensor tiles; decrypt: transposed in registers on the way
//                 in), so that ONE 32-bit shared-memory load returns four consecutive rows of a byte
//                 column: 8 output rows of a column cost 3 conflict-free loads + 2 funnel shifts.  The
//                 words are transposed back to row-major in registers (PRMT), XORed with the keystream
//                 (64-bit streaming loads) and streamed out (64-bit stores).
//
// The intermediate between the passes lives in the output buffer (every CTA of either pass reads all
// of its rows / its whole strip before it writes them), and launches are sized so that it stays
// resident in the 126 MB L2: DRAM traffic stays at the algorithmic read F_o + read B + write F_e.
// The kernels of one call are chained with programmatic dependent launch (griddepcontrol); a call on a long resident clip
// is cut into launch pairs (row pass + column pass) that alternate over two streams, so that one pair's column pass
// overlaps the next pair's row pass (vcrypt.cpp: launch_cipher).
//
// A one-thread-per-output-byte gather kernel covers every shape the tiled passes do not
// (w % 16 != 0, w < 64, h % 4 != 0, h < 16, or a strip / row block too large for shared memory).
#include <cuda.h>

#include <type_traits>

#include "kernels.cuh"
#include "ptx.cuh"
#include "smem_attr.hpp"

namespace vk {

// ---------------------------------------------------------------------------------------------
// Row pass: horizontal bit rotation (Algorithm 4 / Eq. 2 on the rows of Algorithm 3's bit matrix,
// packed back as in Algorithm 7).  Work unit = one block of 4 consecutive rows of one frame (h % 4 == 0,
// so a block never straddles two frames).
//   INV = false: bit p of channel c moves to (p + d_h mod 8w) mod 8w; the block is written in T4 layout.
//   INV = true : the inverse rotation; input and output are row-major.
// Warp-specialised persistent CTAs.  The last warp is the copy warp: it computes the shift parameters of
// a block from D, brings the block into a ring of NS shared-memory stages with one bulk async copy (TMA,
// cp.async.bulk -> UBLKCP), and sends finished blocks back with one bulk async store.  The other
// NC threads are compute threads and work on a stage in two phases separated by a named barrier:
//   phase 1 (one item = 16 pixels of one row): 48 interleaved bytes -> three channel planes (PRMT network),
//            so that the per-(row, channel) bit rotation becomes a 32-bit funnel shift of two neighbouring
//            plane words; the chunk is stored already rotated by the whole-chunk part of the distance;
//   phase 2 (one item = a quad of 4 pixels, all 4 rows, all 3 channels): 12 funnel shifts, then either three
//            4 x 4 byte transposes (T4: the word at (row 4R + (x & 3), word column x >> 2) holds byte column x
//            of rows 4R .. 4R+3) or the re-interleave to row-major; the result goes to one output buffer.
// Synchronisation: full[s] (mbarrier, transaction bytes) copy warp -> compute threads; empty[s] (one arrival)
// compute threads -> copy warp once phase 1 has consumed the stage; ofull / ofree (one arrival each) hand the
// output buffer to the copy warp's bulk store and back; named barrier 1 among the compute threads.
// In place (dst == src) is safe: a block is read completely before it is written.
// ---------------------------------------------------------------------------------------------
constexpr int ROW_RB = 4;       // rows per block
constexpr int ROW_HDR = 1024;   // mbarriers + shift parameters
constexpr int ROW_MAXNS = 4;    // stages at most

// Rotation of one (row, channel): output bit d takes source bit (d + sh) mod 8w, sh = 32 * (4 * dq + fine) + sh5.
// Phase 1 writes chunk k (16 pixels) of the plane at chunk position (k - dq) mod C, so that phase 2 reads the two
// words q + fine, q + fine + 1 of the pre-rotated plane (never wrapping: two pad chunks repeat chunks 0 and 1).
//   p1 = 16 * dq                      (bytes; phase 1)
//   p2 = (plane offset + 4 * fine) << 8 | sh5   (phase 2: one LEA.HI gives the address, the funnel shift takes sh5)
__device__ __forceinline__ uint32_t row_dist(const uint16_t *__restrict__ D, const Geom &g, uint32_t grow, uint32_t ch) {
    const uint32_t f = grow / g.h, i = grow - f * g.h;
    return (uint32_t)D[(size_t)f * g.nD + ch * (g.h + g.w) + i];  // d_h of (frame f, row i, channel ch)
}
__device__ __forceinline__ uint2 row_param_of(uint32_t d, const Geom &g, bool inv, uint32_t plane_off) {
    const uint32_t W8 = 8u * g.w, s = d % W8;
    const uint32_t sh = inv ? s : (s ? W8 - s : 0u);
    const uint32_t dw = sh >> 5;
    return make_uint2((dw >> 2) << 4, ((plane_off + 4u * (dw & 3u)) << 8) | (sh & 31u));
}
__device__ __forceinline__ uint2 row_param(const uint16_t *__restrict__ D, const Geom &g, uint32_t grow, uint32_t ch,
                                           bool inv, uint32_t plane_off) {
    return row_param_of(row_dist(D, g, grow, ch), g, inv, plane_off);
}

template <bool INV, int MAXT, int MINB>
__global__ void __launch_bounds__(MAXT, MINB) row_pass_kernel(const uint8_t *src, uint8_t *dst, const uint16_t *__restrict__ D,
                                                           Geom g, uint32_t nblocks, uint32_t NS, uint32_t NC) {
    extern __shared__ __align__(128) uint8_t smem[];
    uint64_t *full = reinterpret_cast<uint64_t *>(smem);                // [ROW_MAXNS] input stage loaded
    uint64_t *empty = reinterpret_cast<uint64_t *>(smem + 32);          // [ROW_MAXNS] input stage consumed by phase 1
    uint64_t *ofull = reinterpret_cast<uint64_t *>(smem + 64);          // output buffer written by phase 2
    uint64_t *ofree = reinterpret_cast<uint64_t *>(smem + 72);          // output buffer read by the bulk store
    uint32_t *par1 = reinterpret_cast<uint32_t *>(smem + 128);          // [ROW_MAXNS][4 rows][4]  (64 B per stage)
    uint32_t *par2 = reinterpret_cast<uint32_t *>(smem + 128 + 64 * ROW_MAXNS);  // same shape
    const uint32_t w = g.w, rb = g.row_bytes, C = w >> 4, Q = w >> 2;   // items / quads per row
    const uint32_t blk_bytes = ROW_RB * rb;
    const uint32_t PS = w + 32u;                                        // plane stride (bytes): w/4 words + 2 pad chunks
    uint8_t *stage0 = smem + ROW_HDR;                                   // NS input stages
    uint8_t *obuf = stage0 + NS * blk_bytes;                            // one output buffer
    uint8_t *planes = obuf + blk_bytes;
    const uint32_t G = gridDim.x, tid = threadIdx.x;
    const uint32_t blk0 = blockIdx.x;
    if (blk0 >= nblocks) return;
    const uint32_t niter = (nblocks - blk0 + G - 1) / G;

    if (tid == 0) {
        for (uint32_t s = 0; s < NS; ++s) { mbar_init(full + s, 1); mbar_init(empty + s, 1); }
        mbar_init(ofull, 1);
        mbar_init(ofree, 1);
        mbar_init_fence();
    }
    __syncthreads();
    pdl_wait();     // everything below reads or writes global memory the previous kernel of the stream may have written
    pdl_trigger();  // only now: the column pass reads its keystream before its own wait, so it must not start before this point

    if (tid >= NC) {
        // ================= copy warp =================
        const uint32_t lane = tid - NC;
        const uint32_t pr = lane / 3u, pch = lane - 3u * pr;           // lanes 0..11: (row, channel) of the block
        const uint32_t pslot = pr * 4u + pch, poff = (pr * 3u + pch) * PS;
        const uint64_t pol_in = policy_evict_first();
        // prologue: fill every stage
        for (uint32_t it = 0; it < NS && it < niter; ++it) {
            const uint32_t blk = INV ? nblocks - 1u - (blk0 + it * G) : blk0 + it * G;
            if (lane < 3 * ROW_RB) {
                const uint2 pv = row_param(D, g, blk * ROW_RB + pr, pch, INV, poff);
                par1[it * 16u + pslot] = pv.x;
                par2[it * 16u + pslot] = pv.y;
            }
            __syncwarp();
            if (lane == 0) {
                mbar_expect_tx(full + it, blk_bytes);
                bulk_g2s_hint(stage0 + it * blk_bytes, src + (size_t)blk * blk_bytes, blk_bytes, full + it, pol_in);
            }
        }
        uint32_t s = 0, ph = 0;
        for (uint32_t it = 0; it < niter; ++it) {
            // decrypt walks the blocks last-first: the column pass wrote the last frames last, they are the likeliest in L2
            const uint32_t blk = INV ? nblocks - 1u - (blk0 + it * G) : blk0 + it * G;
            const uint32_t blk_next = INV ? blk - NS * G : blk + NS * G;  // only used when it + NS < niter
            const bool refill = it + NS < niter;
            if (refill) {
                uint2 pnext = make_uint2(0u, 0u);
                if (lane < 3 * ROW_RB) pnext = row_param(D, g, blk_next * ROW_RB + pr, pch, INV, poff);
                if (lane == 0) mbar_wait(empty + s, ph);  // phase 1 and phase 2 of block `it` no longer need stage s / its parameters
                __syncwarp();
                if (lane < 3 * ROW_RB) { par1[s * 16u + pslot] = pnext.x; par2[s * 16u + pslot] = pnext.y; }
                __syncwarp();
                if (lane == 0) {
                    mbar_expect_tx(full + s, blk_bytes);
                    bulk_g2s_hint(stage0 + s * blk_bytes, src + (size_t)blk_next * blk_bytes, blk_bytes, full + s, pol_in);
                }
            }
            if (lane == 0) {
                mbar_wait(ofull, it & 1u);  // the compute threads have written block `it` into the output buffer
                bulk_s2g(dst + (size_t)blk * blk_bytes, obuf, blk_bytes);
                bulk_wait_read_0();         // the store has left shared memory
                mbar_arrive(ofree);
            }
            __syncwarp();
            if (++s == NS) { s = 0; ph ^= 1u; }
        }
        if (lane == 0) bulk_wait_all();
        return;
    }

    // ================= compute threads =================
    // loop-invariant work assignment: phase 1 item (row r1, chunk k1) = tid (further items: + NC), phase 2 quad = tid
    const uint32_t r1 = (tid >= C) + (tid >= 2u * C) + (tid >= 3u * C), k1 = tid - r1 * C;
    uint32_t s = 0, ph = 0;
    for (uint32_t it = 0; it < niter; ++it) {
        const uint8_t *stage = stage0 + s * blk_bytes;
        const uint32_t *p1 = par1 + s * 16u, *p2 = par2 + s * 16u;
        mbar_wait(full + s, ph);

        // ---- phase 1: de-interleave into planes; item = (row r, 16 pixels k)
        for (uint32_t i = tid; i < ROW_RB * C; i += NC) {
            uint32_t r = r1, k = k1;
            if (i != tid) { r = (i >= C) + (i >= 2u * C) + (i >= 3u * C); k = i - r * C; }
            const uint4 *p = reinterpret_cast<const uint4 *>(stage + r * rb + 48u * k);
            const uint4 a = p[0], b = p[1], c = p[2];
            const uint4 dq = *reinterpret_cast<const uint4 *>(p1 + 4u * r);
            const uint32_t W[12] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w, c.x, c.y, c.z, c.w};
            uint4 v0, v1, v2;  // channel 0, 1, 2: four plane words each
#define VK_DEINT(m, X0, X1, X2)                                                     \
    X0 = __byte_perm(__byte_perm(W[3 * m], W[3 * m + 1], 0x0630), W[3 * m + 2], 0x5210); \
    X1 = __byte_perm(__byte_perm(W[3 * m], W[3 * m + 1], 0x0741), W[3 * m + 2], 0x6210); \
    X2 = __byte_perm(__byte_perm(W[3 * m], W[3 * m + 1], 0x0052), W[3 * m + 2], 0x7410);
            VK_DEINT(0, v0.x, v1.x, v2.x)
            VK_DEINT(1, v0.y, v1.y, v2.y)
            VK_DEINT(2, v0.z, v1.z, v2.z)
            VK_DEINT(3, v0.w, v1.w, v2.w)
#undef VK_DEINT
            uint8_t *pl = planes + r * 3u * PS;
            const int32_t k16 = (int32_t)(16u * k);
#define VK_PUT(V, DQ, CH)                                                      \
    {                                                                          \
        int32_t kb = k16 - (int32_t)(DQ);                                      \
        if (kb < 0) kb += (int32_t)w;                                          \
        uint8_t *d = pl + (CH) * PS + kb;                                      \
        *reinterpret_cast<uint4 *>(d) = V;                                     \
        if (kb < 32) *reinterpret_cast<uint4 *>(d + w) = V; /* pad chunks */   \
    }
            VK_PUT(v0, dq.x, 0u)
            VK_PUT(v1, dq.y, 1u)
            VK_PUT(v2, dq.z, 2u)
#undef VK_PUT
        }
        // the 12 phase-2 parameters of this block: read them before the stage (and its parameter slot) is released
        uint4 pv[ROW_RB];
#pragma unroll
        for (int r = 0; r < ROW_RB; ++r) pv[r] = *reinterpret_cast<const uint4 *>(p2 + 4 * r);
        named_bar_sync(1, NC);  // planes complete, raw block consumed
        if (tid == 0) mbar_arrive(empty + s);
        if (it > 0) mbar_wait(ofree, (it - 1u) & 1u);  // the previous block's store has left the output buffer

        // ---- phase 2: rotate; item = quad q (4 pixels) of all 4 rows and 3 channels
        for (uint32_t q = tid; q < Q; q += NC) {
            const uint8_t *qa = planes + 4u * q;
            uint32_t R[ROW_RB][3];
#pragma unroll
            for (int r = 0; r < ROW_RB; ++r) {
                const uint32_t pvv[3] = {pv[r].x, pv[r].y, pv[r].z};
#pragma unroll
                for (int ch = 0; ch < 3; ++ch) {
                    const uint32_t *P = reinterpret_cast<const uint32_t *>(qa + (pvv[ch] >> 8));
                    R[r][ch] = __funnelshift_r(P[0], P[1], pvv[ch]);  // shift amount = low 5 bits
                }
            }
            uint8_t *o = obuf + 12u * q;
            if (!INV) {
                // T4: pixel p of the quad, channel ch = byte column x = 12q + 3p + ch -> block row x & 3, word x >> 2
#pragma unroll
                for (int ch = 0; ch < 3; ++ch) {
                    const uint32_t t01a = __byte_perm(R[0][ch], R[1][ch], 0x5140), t01b = __byte_perm(R[0][ch], R[1][ch], 0x7362);
                    const uint32_t t23a = __byte_perm(R[2][ch], R[3][ch], 0x5140), t23b = __byte_perm(R[2][ch], R[3][ch], 0x7362);
                    const uint32_t T[4] = {__byte_perm(t01a, t23a, 0x5410), __byte_perm(t01a, t23a, 0x7632),
                                           __byte_perm(t01b, t23b, 0x5410), __byte_perm(t01b, t23b, 0x7632)};
#pragma unroll
                    for (int p = 0; p < 4; ++p) {
                        const int y = 3 * p + ch;
                        *reinterpret_cast<uint32_t *>(o + (y & 3) * rb + 4 * (y >> 2)) = T[p];
                    }
                }
            } else {
                // row-major: byte y = 3 * pixel + channel of the quad's 12 bytes
#pragma unroll
                for (int r = 0; r < ROW_RB; ++r) {
                    uint32_t *po = reinterpret_cast<uint32_t *>(o + r * rb);
                    po[0] = __byte_perm(__byte_perm(R[r][0], R[r][1], 0x1040), R[r][2], 0x3410);
                    po[1] = __byte_perm(__byte_perm(R[r][0], R[r][1], 0x6205), R[r][2], 0x3250);
                    po[2] = __byte_perm(__byte_perm(R[r][0], R[r][1], 0x0730), R[r][2], 0x7216);
                }
            }
        }
        fence_async_smem();     // generic-proxy writes to the output buffer -> visible to the bulk store
        named_bar_sync(1, NC);  // block complete; planes free for the next block
        if (tid == 0) mbar_arrive(ofull);
        if (++s == NS) { s = 0; ph ^= 1u; }
    }
}

// ---------------------------------------------------------------------------------------------
// Row pass, register-landing variant (frames up to 4096 pixels wide): the same two phases on the same planes and the same
// output buffer as row_pass_kernel, but a block comes in through the threads' own 128-bit streaming loads (LDG.E.128,
// evict-first) instead of a ring of shared-memory stages filled by the TMA engine: thread `tid` owns phase-1 item(s)
// tid (+ NT) of every block its CTA takes, loads the item of the NEXT block right after it has consumed the current one,
// and so keeps 48 (96) bytes in flight in registers through phase 2.  A CTA then needs the planes and one output buffer only
// (47 KB at w = 1920 instead of 93 KB), three or four CTAs share an SM -- and, under the two-stream schedule, a row CTA
// fits beside the column pass's CTAs far more often.  Measured on B200 (resident clips, two streams): FHD encrypt
// 4.33 -> 4.07 us per frame, 4K 22.9 -> 19.6; the decrypt direction takes it too, except for frames 1537 to 2048
// pixels wide, where row_pass_kernel as three small CTAs per SM is as fast or faster (make_plan).
// Synchronisation: CTA barrier A (planes complete, the previous block's bulk store has left the output buffer: thread 0
// waits for it before arriving), CTA barrier B (output buffer complete, planes free); thread 0 then issues the bulk store.
// Shift parameters: 12 threads of the last warp compute block it+1's while block it is in phase 1; four slots, so that a
// slot is rewritten three barriers after its last reader.
// ---------------------------------------------------------------------------------------------
constexpr int RR_HDR = 512;  // par1[4][16], par2[4][16]

template <bool INV, int NT, int MINB, int IPT>
__global__ void __launch_bounds__(NT, MINB) row_reg_kernel(const uint8_t *src, uint8_t *dst, const uint16_t *__restrict__ D,
                                                         Geom g, uint32_t nblocks) {
    extern __shared__ __align__(128) uint8_t smem[];
    uint32_t *par1 = reinterpret_cast<uint32_t *>(smem);
    uint32_t *par2 = reinterpret_cast<uint32_t *>(smem + 256);
    const uint32_t w = g.w, rb = g.row_bytes, C = w >> 4, Q = w >> 2;
    const uint32_t blk_bytes = ROW_RB * rb, PS = w + 32u;
    uint8_t *obuf = smem + RR_HDR;
    uint8_t *planes = obuf + blk_bytes;
    const uint32_t G = gridDim.x, tid = threadIdx.x, blk0 = blockIdx.x;
    if (blk0 >= nblocks) return;
    const uint32_t niter = (nblocks - blk0 + G - 1) / G;
    pdl_wait();     // everything below reads or writes global memory the previous kernel of the stream may have written
    pdl_trigger();  // only now (see row_pass_kernel)

    // decrypt walks the blocks last-first: the column pass wrote the last frames last, they are the likeliest in L2
    auto blk_of = [&](uint32_t it) -> uint32_t { return INV ? nblocks - 1u - (blk0 + it * G) : blk0 + it * G; };
    bool has[IPT];
    uint32_t r1[IPT], k1[IPT], item_off[IPT];
    uint4 L[IPT][3];
#pragma unroll
    for (int m = 0; m < IPT; ++m) {
        const uint32_t i = tid + (uint32_t)m * NT;  // phase-1 item (row r1, 16 pixels k1)
        has[m] = i < ROW_RB * C;
        r1[m] = (i >= C) + (i >= 2u * C) + (i >= 3u * C);
        k1[m] = i - r1[m] * C;
        item_off[m] = r1[m] * rb + 48u * k1[m];
        L[m][0] = L[m][1] = L[m][2] = make_uint4(0u, 0u, 0u, 0u);
        if (has[m]) {
            const uint4 *p = reinterpret_cast<const uint4 *>(src + (size_t)blk_of(0) * blk_bytes + item_off[m]);
            L[m][0] = __ldcs(p); L[m][1] = __ldcs(p + 1); L[m][2] = __ldcs(p + 2);
        }
    }
    const uint32_t plane_lane = tid - (NT - 32);  // parameter threads: lanes 0 .. 11 of the last warp
    const bool is_par = plane_lane < 3u * ROW_RB;
    const uint32_t pr = plane_lane / 3u, pch = plane_lane - 3u * pr;
    const uint32_t pslot = pr * 4u + pch, poff = (pr * 3u + pch) * PS;
    uint32_t dnext = 0;  // parameter threads: the distance of block it + 1, loaded one iteration before it is turned into parameters
    if (is_par) {
        const uint2 pv = row_param(D, g, blk_of(0) * ROW_RB + pr, pch, INV, poff);
        par1[pslot] = pv.x;
        par2[pslot] = pv.y;
        if (niter > 1) dnext = row_dist(D, g, blk_of(1) * ROW_RB + pr, pch);
    }
    __syncthreads();

    for (uint32_t it = 0; it < niter; ++it) {
        const uint32_t blk = blk_of(it);
        const uint32_t *p1 = par1 + (it & 3u) * 16u, *p2 = par2 + (it & 3u) * 16u;
        if (is_par && it + 1 < niter) {  // no global-memory latency between the parameter threads and barrier A
            const uint2 pv = row_param_of(dnext, g, INV, poff);
            par1[((it + 1) & 3u) * 16u + pslot] = pv.x;
            par2[((it + 1) & 3u) * 16u + pslot] = pv.y;
            if (it + 2 < niter) dnext = row_dist(D, g, blk_of(it + 2) * ROW_RB + pr, pch);
        }
        // ---- phase 1: registers -> planes (as in row_pass_kernel), then the same item of the next block -> registers
#pragma unroll
        for (int m = 0; m < IPT; ++m) {
            if (!has[m]) continue;
            const uint4 a = L[m][0], b = L[m][1], c = L[m][2];
            const uint4 dq = *reinterpret_cast<const uint4 *>(p1 + 4u * r1[m]);
            const uint32_t W[12] = {a.x, a.y, a.z, a.w, b.x, b.y, b.z, b.w, c.x, c.y, c.z, c.w};
            uint4 v0, v1, v2;
#define VK_DEINT(m_, X0, X1, X2)                                                          \
    X0 = __byte_perm(__byte_perm(W[3 * m_], W[3 * m_ + 1], 0x0630), W[3 * m_ + 2], 0x5210); \
    X1 = __byte_perm(__byte_perm(W[3 * m_], W[3 * m_ + 1], 0x0741), W[3 * m_ + 2], 0x6210); \
    X2 = __byte_perm(__byte_perm(W[3 * m_], W[3 * m_ + 1], 0x0052), W[3 * m_ + 2], 0x7410);
            VK_DEINT(0, v0.x, v1.x, v2.x)
            VK_DEINT(1, v0.y, v1.y, v2.y)
            VK_DEINT(2, v0.z, v1.z, v2.z)
            VK_DEINT(3, v0.w, v1.w, v2.w)
#undef VK_DEINT
            uint8_t *pl = planes + r1[m] * 3u * PS;
            const int32_t k16 = (int32_t)(16u * k1[m]);
#define VK_PUT(V, DQ, CH)                                                      \
    {                                                                          \
        int32_t kb = k16 - (int32_t)(DQ);                                      \
        if (kb < 0) kb += (int32_t)w;                                          \
        uint8_t *d = pl + (CH) * PS + kb;                                      \
        *reinterpret_cast<uint4 *>(d) = V;                                     \
        if (kb < 32) *reinterpret_cast<uint4 *>(d + w) = V; /* pad chunks */   \
    }
            VK_PUT(v0, dq.x, 0u)
            VK_PUT(v1, dq.y, 1u)
            VK_PUT(v2, dq.z, 2u)
#undef VK_PUT
            if (it + 1 < niter) {
                const uint4 *p = reinterpret_cast<const uint4 *>(src + (size_t)blk_of(it + 1) * blk_bytes + item_off[m]);
                L[m][0] = __ldcs(p); L[m][1] = __ldcs(p + 1); L[m][2] = __ldcs(p + 2);
            }
        }
        if (tid == 0) bulk_wait_read_0();  // the previous block's store has left the output buffer
        __syncthreads();                   // A

        // ---- phase 2: rotate; item = quad q (4 pixels) of all 4 rows and 3 channels (as in row_pass_kernel)
        for (uint32_t q = tid; q < Q; q += NT) {
            const uint8_t *qa = planes + 4u * q;
            uint32_t R[ROW_RB][3];
#pragma unroll
            for (int r = 0; r < ROW_RB; ++r) {
                const uint4 pvr = *reinterpret_cast<const uint4 *>(p2 + 4 * r);
                const uint32_t pvv[3] = {pvr.x, pvr.y, pvr.z};
#pragma unroll
                for (int ch = 0; ch < 3; ++ch) {
                    const uint32_t *P = reinterpret_cast<const uint32_t *>(qa + (pvv[ch] >> 8));
                    R[r][ch] = __funnelshift_r(P[0], P[1], pvv[ch]);  // shift amount = low 5 bits
                }
            }
            uint8_t *o = obuf + 12u * q;
            if (!INV) {
#pragma unroll
                for (int ch = 0; ch < 3; ++ch) {
                    const uint32_t t01a = __byte_perm(R[0][ch], R[1][ch], 0x5140), t01b = __byte_perm(R[0][ch], R[1][ch], 0x7362);
                    const uint32_t t23a = __byte_perm(R[2][ch], R[3][ch], 0x5140), t23b = __byte_perm(R[2][ch], R[3][ch], 0x7362);
                    const uint32_t T[4] = {__byte_perm(t01a, t23a, 0x5410), __byte_perm(t01a, t23a, 0x7632),
                                           __byte_perm(t01b, t23b, 0x5410), __byte_perm(t01b, t23b, 0x7632)};
#pragma unroll
                    for (int p = 0; p < 4; ++p) {
                        const int y = 3 * p + ch;
                        *reinterpret_cast<uint32_t *>(o + (y & 3) * rb + 4 * (y >> 2)) = T[p];
                    }
                }
            } else {
#pragma unroll
                for (int r = 0; r < ROW_RB; ++r) {
                    uint32_t *po = reinterpret_cast<uint32_t *>(o + r * rb);
                    po[0] = __byte_perm(__byte_perm(R[r][0], R[r][1], 0x1040), R[r][2], 0x3410);
                    po[1] = __byte_perm(__byte_perm(R[r][0], R[r][1], 0x6205), R[r][2], 0x3250);
                    po[2] = __byte_perm(__byte_perm(R[r][0], R[r][1], 0x0730), R[r][2], 0x7216);
                }
            }
        }
        fence_async_smem();  // generic-proxy writes to the output buffer -> visible to the bulk store
        __syncthreads();     // B
        if (tid == 0) bulk_s2g(dst + (size_t)blk * blk_bytes, obuf, blk_bytes);
    }
    if (tid == 0) bulk_wait_all();
}

// ---------------------------------------------------------------------------------------------
// Column pass, encrypt direction: vertical circular shift of every byte column (Algorithm 5 / Eq. 3, one
// d_v per pixel column and channel = per byte column of the interleaved matrix) fused with the XOR of
// Algorithm 6:   dst(ro, x) = B(ro, x) xor I((ro - t_x) mod h, x),   I = the row pass output in T4 layout.
// One CTA = one strip of X byte columns of one frame, all h rows (+ 8 repeated rows so that a window never
// wraps) in shared memory, brought in by the TMA engine as 2-D tensor tiles (cp.async.bulk.tensor ->
// UTMALDG): no thread touches the strip on its way in.  In T4 layout ONE 32-bit shared-memory load returns
// four consecutive rows of a byte column, so 8 output rows of a column cost 3 loads + 2 funnel shifts.
// A warp is split into NSUB = 256 / X sub-warps of X / 8 lanes; a lane owns 8 byte columns (two T4 word
// columns x four byte lanes) and a sub-warp emits groups of 8 consecutive output rows with 64-bit
// keystream loads and ciphertext stores.  Bank of a load = (strip row * X/4 + word column) mod 32 with strip
// row = 4R + b: sub-warp s walks its columns in the order (word column a_l ^ (s & 1), byte lane a_b ^ (s >> 1)),
// so the sub-warps of a warp always sit in disjoint banks whatever rows they read: no conflicts for
// X = 128, 64, 32.  The permutation is undone by the selectors of the 4 x 4 byte transposes and by one
// select per output word.
// Checked per instruction in round 3 (profiles/r3_source_summary.txt, from the source page of a full ncu capture):
// every LDS / STS of col_enc_kernel and col_dec_kernel issues exactly its ideal number of wavefronts ("L1 Wavefronts
// Shared Excessive" = 0 of 382 500 and of 870 300 per launch at FHD).  The hardware counter
// l1tex__data_bank_conflicts_pipe_lsu_mem_shared that the kernel-level summary shows (186 K for col_enc_kernel, 507 K
// for col_dec_kernel) is, to within 4 %, the number of shared-memory wavefronts that belong to NO instruction of the kernel
// (575 K - 382.5 K = 193 K; 1 375 K - 870 K = 505 K): the TMA engine
// writing the strip tiles (and, in the row kernels, the bulk stores reading the output buffer).  ncu counts that
// async-proxy traffic in the same pipe counter; it is not a conflict between the threads' accesses.
// In place is safe: the whole strip is in shared memory before the first store.
// ---------------------------------------------------------------------------------------------
// keystream prefetch depths (rounds of loads in flight per thread): decrypt column pass with three CTAs per SM / one CTA per
// SM, encrypt column pass with one CTA per SM (development builds may override)
#ifndef VK_KD3
#define VK_KD3 3
#endif
#ifndef VK_KD1
#define VK_KD1 3
#endif
#ifndef VK_DE1
#define VK_DE1 2
#endif
#ifndef VK_DE2
#define VK_DE2 2
#endif
constexpr int CE_PAD = 8;   // repeated strip rows
constexpr int CE_G = 8;     // output rows per group

template <int X, int NT, int MINB, int DEPTH>
__global__ void __launch_bounds__(NT, MINB)
    col_enc_kernel(const __grid_constant__ CUtensorMap tm_main, const __grid_constant__ CUtensorMap tm_pad,
                   const __grid_constant__ CUtensorMap tm_B, const uint8_t *__restrict__ Bk, uint8_t *dst, const uint16_t *__restrict__ D, Geom g,
                   uint32_t strips_per_frame, uint32_t nframes, uint32_t box_rows, uint32_t h_magic, uint32_t pf_rows) {
    extern __shared__ __align__(128) uint8_t S[];
    constexpr uint32_t LPS = X / 8;       // lanes per strip row
    constexpr uint32_t NSUB = 32 / LPS;   // sub-warps per warp
    constexpr uint32_t NW = NT / 32;
    constexpr uint32_t GSTEP = NW * NSUB;  // groups between two iterations of a sub-warp
    constexpr uint32_t CE_AHEAD = 2u * GSTEP * CE_G;  // keystream rows on their way to L2 ahead of the CTA: two iterations (measured optimum)
    const uint32_t h = g.h, rb = g.row_bytes;
    uint64_t *bar = reinterpret_cast<uint64_t *>(S + (size_t)(h + CE_PAD) * X);
    uint16_t *ups = reinterpret_cast<uint16_t *>(S + (size_t)(h + CE_PAD) * X + 16);  // [X] source row offset per byte column
    // the last frame first: its intermediate was written last and is the most likely to be in L2
    const uint32_t fr = blockIdx.x / strips_per_frame;
    const uint32_t f = nframes - 1u - fr;
    const uint32_t x0 = (blockIdx.x - fr * strips_per_frame) * X;

    pdl_trigger();
    // keystream look-ahead: thread 0 asks the TMA engine to pull the strip's keystream tiles into L2, CE_AHEAD rows
    // ahead of the row group the CTA is working on (the threads' own loads then hit L2 instead of waiting on DRAM)
    // (only where a thread has ONE round of keystream loads in flight: with two, the look-ahead costs more than it hides --
    // FHD, two CTAs per SM: 4.38 -> 4.30 us per frame without it)
    constexpr bool LOOKAHEAD = DEPTH == 1;
    uint32_t pf_row = 0;
    if (threadIdx.x == 0) {
        if (LOOKAHEAD)
            for (; pf_row < h && pf_row < CE_AHEAD + (DEPTH - 1) * GSTEP * CE_G; pf_row += pf_rows)
                tma_prefetch_2d(&tm_B, (int32_t)x0, (int32_t)(f * h + pf_row));
        mbar_init(bar, 1);
        mbar_init_fence();
        pdl_wait();  // the strip is the row pass's output
        const uint64_t pol = policy_evict_first();
        mbar_expect_tx(bar, (h + CE_PAD) * X);
        const int32_t y0 = (int32_t)(f * h);
        for (uint32_t r0 = 0; r0 < h; r0 += box_rows) tma_load_2d(S + (size_t)r0 * X, &tm_main, (int32_t)x0, y0 + (int32_t)r0, bar, pol);
        tma_load_2d(S + (size_t)h * X, &tm_pad, (int32_t)x0, y0, bar, pol);
    }
    // one thread per byte column of the strip: up = (h - d_v mod h) mod h, the row offset of the column's source
    if (threadIdx.x >= NT - X) {
        const uint32_t xs = threadIdx.x - (NT - X);
        uint32_t x = x0 + xs;
        if (x >= rb) x = 0;
        const uint32_t jj = x / 3u, c = x - 3u * jj;
        const uint32_t dv = D[(size_t)f * g.nD + c * (h + g.w) + h + jj];
        const uint32_t t = dv - __umulhi(dv, h_magic) * h;  // d_v mod h  (h_magic = ceil(2^32 / h), d_v < 2^16)
        ups[xs] = (uint16_t)(t ? h - t : 0u);
    }

    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const uint32_t sub = lane / LPS, j = lane % LPS;
    const uint32_t sl = sub & 1u, sb = sub >> 1;   // permutation of the word column / byte lane order
    const uint32_t xt = x0 + 8u * j;               // first of this lane's 8 byte columns (frame coordinates)
    const bool col_ok = xt < rb;                   // rb % 8 == 0 on this path: the 8 columns are inside or outside together
    const uint32_t g0 = warp * NSUB + sub;         // first group of this sub-warp
    const uint32_t nfull = h / CE_G;               // full groups; h % 8 == 4 leaves one half group
    const bool active = col_ok && g0 * CE_G < h;
    const size_t fbase = (size_t)f * g.frame_bytes + xt + (size_t)(g0 * CE_G) * rb;
    const uint8_t *pB = Bk + fbase;                // row g0 * 8 of this lane's columns
    uint8_t *pO = dst + fbase;
    const uint32_t rb2 = 2u * rb, rb3 = 3u * rb, rb4 = 4u * rb, rb5 = 5u * rb, rb6 = 6u * rb, rb7 = 7u * rb;
    const size_t gstep = (size_t)(GSTEP * CE_G) * rb;

#define VK_ROWPTR(T, P, OFF) reinterpret_cast<T>(mad_wide_ptr(P, OFF))
    // keystream of the first DEPTH groups: issued before the strip arrives (DEPTH = 2 where the registers are there: two
    // rounds of loads in flight per thread, and two rounds of latency hidden)
    uint2 kb[DEPTH][CE_G];
#pragma unroll
    for (int d = 0; d < DEPTH; ++d)
#pragma unroll
        for (int i = 0; i < CE_G; ++i) kb[d][i] = make_uint2(0u, 0u);
    if (active) {
        const uint32_t offs[8] = {0u, rb, rb2, rb3, rb4, rb5, rb6, rb7};
#pragma unroll
        for (int d = 0; d < DEPTH; ++d) {
            const uint32_t gd = g0 + (uint32_t)d * GSTEP;
            const uint8_t *pd = pB + (size_t)d * gstep;
            if (gd < nfull) {
#pragma unroll
                for (int i = 0; i < CE_G; ++i) kb[d][i] = ldg_once_u2(VK_ROWPTR(const uint2 *, pd, offs[i]));
            } else if (gd * CE_G < h) {
#pragma unroll
                for (int i = 0; i < CE_G / 2; ++i) kb[d][i] = ldg_once_u2(VK_ROWPTR(const uint2 *, pd, offs[i]));
            }
        }
    }
    __syncthreads();  // mbarrier initialised, ups[] complete

    // per step a = (a_l, a_b): state of byte column 4 * (2j + (a_l ^ sl)) + (a_b ^ sb) of the strip.
    // q = byte offset of the aligned source block row in the strip (a multiple of 4X) | 8j | K_s | row alignment
    // (low 2 bits); the T4 word of the column sits at (q & ~3) ^ K_a  with  K = byte lane * X + 4 * word column bit.
    const uint32_t hX = h * X;
    const uint32_t ADVX = ((GSTEP * CE_G) % h) * X;  // strip bytes between two iterations (h % 4 == 0 keeps alignment)
    const uint32_t Ks = sb * X + 4u * sl;
    uint32_t q[8];
    {
        // the lane's 8 offsets in natural order (two per word), then permuted into walking order a -> a ^ (4 sl + sb)
        const uint4 u4 = *reinterpret_cast<const uint4 *>(ups + 8u * j);
        uint32_t u[4] = {u4.x, u4.y, u4.z, u4.w};
        const uint32_t sw = (sb & 1u) ? 0x1032u : 0x3210u;
#pragma unroll
        for (int k = 0; k < 4; ++k) u[k] = __byte_perm(u[k], 0u, sw);
        if (sb & 2u) { uint32_t t0 = u[0]; u[0] = u[1]; u[1] = t0; t0 = u[2]; u[2] = u[3]; u[3] = t0; }
        if (sl) { uint32_t t0 = u[0]; u[0] = u[2]; u[2] = t0; t0 = u[1]; u[1] = u[3]; u[3] = t0; }
        const uint32_t base = (8u * j) | Ks;
        uint32_t ro0 = g0 * CE_G;
        if (ro0 >= h) ro0 = 0;
#pragma unroll
        for (int a = 0; a < 8; ++a) {
            const uint32_t up = (a & 1) ? (u[a >> 1] >> 16) : (u[a >> 1] & 0xFFFFu);
            uint32_t s0 = ro0 + up;
            if (s0 >= h) s0 -= h;
            q[a] = (s0 & ~3u) * X + (base | (s0 & 3u));
        }
    }
    // transpose selectors: in[0], in[1] hold byte lanes (sb&1, sb&1 ^ 1); in[2], in[3] the other pair
    const uint32_t selA = (sb & 1u) ? 0x1504u : 0x5140u, selB = (sb & 1u) ? 0x3726u : 0x7362u;
    const uint32_t selLo = (sb & 2u) ? 0x1054u : 0x5410u, selHi = (sb & 2u) ? 0x3276u : 0x7632u;
    const uint32_t m3 = ~3u;

    mbar_wait(bar, 0);  // strip (and its wrap rows) has landed: the previous kernel has completed (thread 0 waited for it)
    if (!active) return;

    // one round = one group of 8 output rows of this lane's columns; PD = which keystream register set it uses (compile time)
    uint32_t gi = g0;
    auto round = [&](auto PD) -> bool {
        constexpr int pd = decltype(PD)::value;
        {
            uint32_t O[CE_G][2];
#pragma unroll
            for (int al_ = 0; al_ < 2; ++al_) {
                uint32_t A[4][2];
#pragma unroll
                for (int ab = 0; ab < 4; ++ab) {
                    const int a = al_ * 4 + ab;
                    const uint32_t Ka = (uint32_t)ab * X + 4u * (uint32_t)al_;
                    const uint8_t *p = S + ((q[a] & m3) ^ Ka);
                    const uint32_t r0 = *reinterpret_cast<const uint32_t *>(p);
                    const uint32_t r1 = *reinterpret_cast<const uint32_t *>(p + 4 * X);
                    const uint32_t r2 = *reinterpret_cast<const uint32_t *>(p + 8 * X);
                    const uint32_t shamt = q[a] << 3;  // funnel shift uses the low 5 bits: 8 * alignment
                    A[ab][0] = __funnelshift_r(r0, r1, shamt);
                    A[ab][1] = __funnelshift_r(r1, r2, shamt);
                    q[a] += ADVX;
                    if (q[a] >= hX) q[a] -= hX;
                }
#pragma unroll
                for (int hg = 0; hg < 2; ++hg) {
                    const uint32_t t01a = __byte_perm(A[0][hg], A[1][hg], selA), t01b = __byte_perm(A[0][hg], A[1][hg], selB);
                    const uint32_t t23a = __byte_perm(A[2][hg], A[3][hg], selA), t23b = __byte_perm(A[2][hg], A[3][hg], selB);
                    O[4 * hg + 0][al_] = __byte_perm(t01a, t23a, selLo);
                    O[4 * hg + 1][al_] = __byte_perm(t01a, t23a, selHi);
                    O[4 * hg + 2][al_] = __byte_perm(t01b, t23b, selLo);
                    O[4 * hg + 3][al_] = __byte_perm(t01b, t23b, selHi);
                }
            }
            // undo the word column permutation, xor the keystream, store
            const uint32_t offs[8] = {0u, rb, rb2, rb3, rb4, rb5, rb6, rb7};
            if (gi < nfull) {
#pragma unroll
                for (int i = 0; i < CE_G; ++i) {
                    const uint32_t lo = sl ? O[i][1] : O[i][0], hi = sl ? O[i][0] : O[i][1];
                    stg_once_u2(VK_ROWPTR(uint2 *, pO, offs[i]), make_uint2(lo ^ kb[pd][i].x, hi ^ kb[pd][i].y));
                }
            } else {  // the half group at the bottom of a frame with h % 8 == 4: always the last one
#pragma unroll
                for (int i = 0; i < CE_G / 2; ++i) {
                    const uint32_t lo = sl ? O[i][1] : O[i][0], hi = sl ? O[i][0] : O[i][1];
                    stg_once_u2(VK_ROWPTR(uint2 *, pO, offs[i]), make_uint2(lo ^ kb[pd][i].x, hi ^ kb[pd][i].y));
                }
                return false;
            }
            const uint32_t gn = gi + GSTEP;
            if (gn * CE_G >= h) return false;
            // keystream of the group DEPTH rounds on, into the registers just used
            const uint32_t gl = gi + (uint32_t)DEPTH * GSTEP;
            if (LOOKAHEAD && threadIdx.x == 0)
                for (; pf_row < h && pf_row < gl * CE_G + CE_AHEAD; pf_row += pf_rows)
                    tma_prefetch_2d(&tm_B, (int32_t)x0, (int32_t)(f * h + pf_row));
            {
                const uint8_t *pl = pB + (size_t)DEPTH * gstep;
                if (gl < nfull) {
#pragma unroll
                    for (int i = 0; i < CE_G; ++i) kb[pd][i] = ldg_once_u2(VK_ROWPTR(const uint2 *, pl, offs[i]));
                } else if (gl * CE_G < h) {
#pragma unroll
                    for (int i = 0; i < CE_G / 2; ++i) kb[pd][i] = ldg_once_u2(VK_ROWPTR(const uint2 *, pl, offs[i]));
                }
            }
            pB += gstep;
            pO += gstep;
            gi = gn;
        }
        return true;
    };
    for (;;) {
        if (!round(std::integral_constant<int, 0>{})) break;
        if (DEPTH > 1 && !round(std::integral_constant<int, (DEPTH > 1 ? 1 : 0)>{})) break;
        if (DEPTH > 2 && !round(std::integral_constant<int, (DEPTH > 2 ? 2 : 0)>{})) break;
    }
#undef VK_ROWPTR
}

// ---------------------------------------------------------------------------------------------
// Column pass, decrypt direction: undo the XOR of Algorithm 6, then the vertical shift of
// Algorithm 5:   dst(i, x) = (src xor B)((i + t_x) mod h, x),   src = F_e row-major, dst row-major (the
// inverse row pass follows).  Same strip, same T4 layout in shared memory and the same conflict-free
// gather as the encrypt direction.  The ciphertext strip is brought in by the TMA engine (all of it in
// flight from the first cycle, no registers held); the threads then turn it into (src xor B) in T4 layout
// IN PLACE: a lane reads its 8 bytes of four rows, xors the keystream (64-bit global loads, one block ahead,
// their tiles pulled into L2 by TMA prefetches), transposes 4 x 4 bytes per word column and writes the same
// 32 bytes back (sub-warps take the rows / byte lanes in the order t ^ (s & 1), so that the two sub-warps of
// a half warp sit in disjoint banks).
// In place (dst == src) is safe: the whole strip is in shared memory (barrier) before the first store.
// ---------------------------------------------------------------------------------------------
template <int X, int NT, int MINB, int KD>
__global__ void __launch_bounds__(NT, MINB)
    col_dec_kernel(const __grid_constant__ CUtensorMap tm_src, const __grid_constant__ CUtensorMap tm_B,
                   const uint8_t *__restrict__ Bk, uint8_t *dst, const uint16_t *__restrict__ D, Geom g,
                   uint32_t strips_per_frame, uint32_t h_magic, uint32_t box_rows, uint32_t pf_rows) {
    extern __shared__ __align__(128) uint8_t S[];
    constexpr uint32_t LPS = X / 8;       // lanes per strip row
    constexpr uint32_t NSUB = 32 / LPS;   // sub-warps per warp
    constexpr uint32_t NW = NT / 32;
    constexpr uint32_t GSTEP = NW * NSUB;  // row groups / row blocks between two iterations of a sub-warp
    const uint32_t h = g.h, rb = g.row_bytes;
    uint64_t *bar = reinterpret_cast<uint64_t *>(S + (size_t)(h + CE_PAD) * X);
    uint16_t *ups = reinterpret_cast<uint16_t *>(S + (size_t)(h + CE_PAD) * X + 16);  // [X] source row offset per byte column
    const uint32_t f = blockIdx.x / strips_per_frame;
    const uint32_t x0 = (blockIdx.x - f * strips_per_frame) * X;

    // keystream look-ahead: thread 0 asks the TMA engine to pull the strip's keystream tiles into L2, CD_AHEAD rows ahead
    // of the rows the CTA is loading.  The first tiles are requested BEFORE the wait for the previous kernel (the
    // keystream is never that kernel's output), which overlaps its tail.
    constexpr uint32_t CD_AHEAD = 2u * 4u * GSTEP;  // two iterations (measured: 1 -> 6.93, 2 -> 6.78, 4 -> 6.95 us per FHD frame)
    uint32_t pf_row = 0;
    if (threadIdx.x == 0) {
        for (; pf_row < h && pf_row < CD_AHEAD + (KD - 1) * 4u * GSTEP; pf_row += pf_rows)
            tma_prefetch_2d(&tm_B, (int32_t)x0, (int32_t)(f * h + pf_row));
        mbar_init(bar, 1);
        mbar_init_fence();
        pdl_wait();  // the ciphertext may be the previous kernel's output
        const uint64_t pol = policy_evict_first();
        mbar_expect_tx(bar, h * X);
        const int32_t y0 = (int32_t)(f * h);
        for (uint32_t r0 = 0; r0 < h; r0 += box_rows) tma_load_2d(S + (size_t)r0 * X, &tm_src, (int32_t)x0, y0 + (int32_t)r0, bar, pol);
    }
    // D and the keystream are inputs too: whoever wrote them (a kernel of the caller's, launched just before on this stream)
    // must be complete before the first read -- only the L2 look-ahead above runs ahead of this wait
    pdl_wait();
    pdl_trigger();
    // one thread per byte column of the strip: t = d_v mod h, the row offset of the column's source
    if (threadIdx.x >= NT - X) {
        const uint32_t xs = threadIdx.x - (NT - X);
        uint32_t x = x0 + xs;
        if (x >= rb) x = 0;
        const uint32_t jj = x / 3u, c = x - 3u * jj;
        const uint32_t dv = D[(size_t)f * g.nD + c * (h + g.w) + h + jj];
        ups[xs] = (uint16_t)(dv - __umulhi(dv, h_magic) * h);  // d_v mod h  (h_magic = ceil(2^32 / h), d_v < 2^16)
    }

    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const uint32_t sub = lane / LPS, j = lane % LPS;
    const uint32_t sl = sub & 1u, sb = sub >> 1;   // permutation of the word column / byte lane order (gather)
    const uint32_t xt = x0 + 8u * j;               // first of this lane's 8 byte columns (frame coordinates)
    const bool col_ok = xt < rb;
    const uint32_t g0 = warp * NSUB + sub;
    const size_t fcol = (size_t)f * g.frame_bytes + xt;
    const uint32_t rb2 = 2u * rb, rb3 = 3u * rb, rb4 = 4u * rb, rb5 = 5u * rb, rb6 = 6u * rb, rb7 = 7u * rb;
#define VK_ROWPTR(T, P, OFF) reinterpret_cast<T>(mad_wide_ptr(P, OFF))

    // ---- phase A: strip -> (strip xor B) in T4 layout, in place.  Item = (block of 4 rows R, this lane's 8 byte columns);
    // step t works on row / byte lane t ^ s1.
    const uint32_t s1 = sub & 1u;
    const uint32_t nblk = h >> 2;
    const uint32_t offs4[4] = {s1 ? rb : 0u, s1 ? 0u : rb, s1 ? rb3 : rb2, s1 ? rb2 : rb3};
    const uint8_t *pB = Bk + fcol + (size_t)(4u * g0) * rb;
    // keystream of the first KD blocks of this sub-warp: issued before the strip arrives (KD blocks of loads in flight per thread)
    const size_t bstep = (size_t)(4u * GSTEP) * rb;
    uint2 kq[KD][4];
#pragma unroll
    for (int d = 0; d < KD; ++d) {
#pragma unroll
        for (int t = 0; t < 4; ++t) kq[d][t] = make_uint2(0u, 0u);
        if (col_ok && g0 + (uint32_t)d * GSTEP < nblk) {
#pragma unroll
            for (int t = 0; t < 4; ++t) kq[d][t] = ldg_once_u2(VK_ROWPTR(const uint2 *, pB + (size_t)d * bstep, offs4[t]));
        }
    }
    __syncthreads();    // mbarrier initialised, ups[] complete
    mbar_wait(bar, 0);  // the ciphertext strip has landed
    if (col_ok) {
        const uint32_t selA = s1 ? 0x1504u : 0x5140u, selB = s1 ? 0x3726u : 0x7362u;  // inputs arrive as rows (t ^ s1)
        const uint32_t selF = s1 ? 0x7632u : 0x5410u, selS = s1 ? 0x5410u : 0x7632u;  // first / second byte lane of a pair
        const int32_t d1 = s1 ? -(int32_t)X : (int32_t)X;
        uint32_t R4 = g0;
        auto block = [&](auto PD) {
            constexpr int pd = decltype(PD)::value;
            uint2 k[4];
#pragma unroll
            for (int t = 0; t < 4; ++t) k[t] = kq[pd][t];
            if (threadIdx.x == 0)
                for (; pf_row < h && pf_row < 4u * (R4 + (uint32_t)KD * GSTEP) + CD_AHEAD; pf_row += pf_rows)
                    tma_prefetch_2d(&tm_B, (int32_t)x0, (int32_t)(f * h + pf_row));
            if (R4 + (uint32_t)KD * GSTEP < nblk) {  // the block KD rounds on, into the registers just read
#pragma unroll
                for (int t = 0; t < 4; ++t) kq[pd][t] = ldg_once_u2(VK_ROWPTR(const uint2 *, pB + (size_t)KD * bstep, offs4[t]));
            }
            pB += bstep;
            uint8_t *ps = S + ((size_t)(4u * R4) * X + 8u * j) + (s1 ? X : 0u);
            uint2 v[4];
            v[0] = *reinterpret_cast<const uint2 *>(ps);
            v[1] = *reinterpret_cast<const uint2 *>(ps + d1);
            v[2] = *reinterpret_cast<const uint2 *>(ps + 2 * X);
            v[3] = *reinterpret_cast<const uint2 *>(ps + 2 * X + d1);
#pragma unroll
            for (int t = 0; t < 4; ++t) { v[t].x ^= k[t].x; v[t].y ^= k[t].y; }
            // two 4 x 4 byte transposes: word column 2j (x) and 2j + 1 (y); outputs in the order b = t ^ s1
            uint32_t lo[4], hi[4];
            {
                const uint32_t a = __byte_perm(v[0].x, v[1].x, selA), b = __byte_perm(v[0].x, v[1].x, selB);
                const uint32_t c = __byte_perm(v[2].x, v[3].x, selA), d = __byte_perm(v[2].x, v[3].x, selB);
                lo[0] = __byte_perm(a, c, selF); lo[1] = __byte_perm(a, c, selS);
                lo[2] = __byte_perm(b, d, selF); lo[3] = __byte_perm(b, d, selS);
            }
            {
                const uint32_t a = __byte_perm(v[0].y, v[1].y, selA), b = __byte_perm(v[0].y, v[1].y, selB);
                const uint32_t c = __byte_perm(v[2].y, v[3].y, selA), d = __byte_perm(v[2].y, v[3].y, selB);
                hi[0] = __byte_perm(a, c, selF); hi[1] = __byte_perm(a, c, selS);
                hi[2] = __byte_perm(b, d, selF); hi[3] = __byte_perm(b, d, selS);
            }
            // step t holds byte lane b = t ^ s1: strip row 4 R4 + b, bytes 8j .. 8j+7
            *reinterpret_cast<uint2 *>(ps) = make_uint2(lo[0], hi[0]);
            *reinterpret_cast<uint2 *>(ps + d1) = make_uint2(lo[1], hi[1]);
            *reinterpret_cast<uint2 *>(ps + 2 * X) = make_uint2(lo[2], hi[2]);
            *reinterpret_cast<uint2 *>(ps + 2 * X + d1) = make_uint2(lo[3], hi[3]);
            if (R4 < CE_PAD / 4) {  // wrap rows: strip rows h .. h+7 repeat rows 0 .. 7
                uint8_t *pw = ps + (size_t)h * X;
                *reinterpret_cast<uint2 *>(pw) = make_uint2(lo[0], hi[0]);
                *reinterpret_cast<uint2 *>(pw + d1) = make_uint2(lo[1], hi[1]);
                *reinterpret_cast<uint2 *>(pw + 2 * X) = make_uint2(lo[2], hi[2]);
                *reinterpret_cast<uint2 *>(pw + 2 * X + d1) = make_uint2(lo[3], hi[3]);
            }
            R4 += GSTEP;
        };
        while (R4 < nblk) {
            block(std::integral_constant<int, 0>{});
            if (KD > 1 && R4 < nblk) block(std::integral_constant<int, (KD > 1 ? 1 : 0)>{});
            if (KD > 2 && R4 < nblk) block(std::integral_constant<int, (KD > 2 ? 2 : 0)>{});
        }
    }
    __syncthreads();  // strip and ups[] complete

    const uint32_t nfull = h / CE_G;
    const bool active = col_ok && g0 * CE_G < h;
    if (!active) return;
    uint8_t *pO = dst + fcol + (size_t)(g0 * CE_G) * rb;
    const size_t gstep = (size_t)(GSTEP * CE_G) * rb;

    const uint32_t hX = h * X;
    const uint32_t ADVX = ((GSTEP * CE_G) % h) * X;
    const uint32_t Ks = sb * X + 4u * sl;
    uint32_t q[8];
    {
        const uint4 u4 = *reinterpret_cast<const uint4 *>(ups + 8u * j);
        uint32_t u[4] = {u4.x, u4.y, u4.z, u4.w};
        const uint32_t sw = (sb & 1u) ? 0x1032u : 0x3210u;
#pragma unroll
        for (int k = 0; k < 4; ++k) u[k] = __byte_perm(u[k], 0u, sw);
        if (sb & 2u) { uint32_t t0 = u[0]; u[0] = u[1]; u[1] = t0; t0 = u[2]; u[2] = u[3]; u[3] = t0; }
        if (sl) { uint32_t t0 = u[0]; u[0] = u[2]; u[2] = t0; t0 = u[1]; u[1] = u[3]; u[3] = t0; }
        const uint32_t base = (8u * j) | Ks;
        const uint32_t ro0 = g0 * CE_G;
#pragma unroll
        for (int a = 0; a < 8; ++a) {
            const uint32_t up = (a & 1) ? (u[a >> 1] >> 16) : (u[a >> 1] & 0xFFFFu);
            uint32_t s0 = ro0 + up;
            if (s0 >= h) s0 -= h;
            q[a] = (s0 & ~3u) * X + (base | (s0 & 3u));
        }
    }
    const uint32_t selA = (sb & 1u) ? 0x1504u : 0x5140u, selB = (sb & 1u) ? 0x3726u : 0x7362u;
    const uint32_t selLo = (sb & 2u) ? 0x1054u : 0x5410u, selHi = (sb & 2u) ? 0x3276u : 0x7632u;
    const uint32_t m3 = ~3u;

    for (uint32_t gi = g0;; gi += GSTEP) {
        uint32_t O[CE_G][2];
#pragma unroll
        for (int al_ = 0; al_ < 2; ++al_) {
            uint32_t A[4][2];
#pragma unroll
            for (int ab = 0; ab < 4; ++ab) {
                const int a = al_ * 4 + ab;
                const uint32_t Ka = (uint32_t)ab * X + 4u * (uint32_t)al_;
                const uint8_t *p = S + ((q[a] & m3) ^ Ka);
                const uint32_t r0 = *reinterpret_cast<const uint32_t *>(p);
                const uint32_t r1 = *reinterpret_cast<const uint32_t *>(p + 4 * X);
                const uint32_t r2 = *reinterpret_cast<const uint32_t *>(p + 8 * X);
                const uint32_t shamt = q[a] << 3;
                A[ab][0] = __funnelshift_r(r0, r1, shamt);
                A[ab][1] = __funnelshift_r(r1, r2, shamt);
                q[a] += ADVX;
                if (q[a] >= hX) q[a] -= hX;
            }
#pragma unroll
            for (int hg = 0; hg < 2; ++hg) {
                const uint32_t t01a = __byte_perm(A[0][hg], A[1][hg], selA), t01b = __byte_perm(A[0][hg], A[1][hg], selB);
                const uint32_t t23a = __byte_perm(A[2][hg], A[3][hg], selA), t23b = __byte_perm(A[2][hg], A[3][hg], selB);
                O[4 * hg + 0][al_] = __byte_perm(t01a, t23a, selLo);
                O[4 * hg + 1][al_] = __byte_perm(t01a, t23a, selHi);
                O[4 * hg + 2][al_] = __byte_perm(t01b, t23b, selLo);
                O[4 * hg + 3][al_] = __byte_perm(t01b, t23b, selHi);
            }
        }
        // undo the word column permutation and store (default caching: the inverse row pass reads this from L2)
        const uint32_t offs[8] = {0u, rb, rb2, rb3, rb4, rb5, rb6, rb7};
        if (gi < nfull) {
#pragma unroll
            for (int i = 0; i < CE_G; ++i)
                *VK_ROWPTR(uint2 *, pO, offs[i]) = make_uint2(sl ? O[i][1] : O[i][0], sl ? O[i][0] : O[i][1]);
        } else {
#pragma unroll
            for (int i = 0; i < CE_G / 2; ++i)
                *VK_ROWPTR(uint2 *, pO, offs[i]) = make_uint2(sl ? O[i][1] : O[i][0], sl ? O[i][0] : O[i][1]);
            break;
        }
        if ((gi + GSTEP) * CE_G >= h) break;
        pO += gstep;
    }
#undef VK_ROWPTR
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
static size_t row_smem_bytes(const Geom &g, int ns) {
    return (size_t)ROW_HDR + (size_t)(ns + 1) * ROW_RB * g.row_bytes + (size_t)ROW_RB * 3 * (g.w + 32);
}
static size_t rowreg_smem_bytes(const Geom &g) { return (size_t)RR_HDR + (size_t)ROW_RB * g.row_bytes + (size_t)ROW_RB * 3 * (g.w + 32); }
static size_t cole_smem_bytes(const Geom &g, int X) { return (size_t)(g.h + CE_PAD) * X + 16 + 2 * (size_t)X; }

template <int X, int NT, int MINB, int KD>
static cudaError_t col_set_attr(int device, size_t smem) {
    return raise_dyn_smem((const void *)col_dec_kernel<X, NT, MINB, KD>, device, smem);
}
template <int X, int NT, int MINB, int DEPTH>
static cudaError_t cole_set_attr(int device, size_t smem) {
    return raise_dyn_smem((const void *)col_enc_kernel<X, NT, MINB, DEPTH>, device, smem);
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

cudaError_t make_plan(const Geom &g, int device, bool row_tma, Plan *out) {
    Plan p{};
    int smem_optin = 0, smem_sm = 0, sms = 0;
    cudaError_t e = cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&smem_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
    if (e != cudaSuccess) return e;
    p.tiled = false;
    p.max_frames_per_launch = 1;
    const bool shape_ok = g.w % 16 == 0 && g.h % 4 == 0 && g.h >= 2 * CE_PAD && g.w >= 64 &&
                          g.frame_bytes < ((size_t)1 << 31);
    if (shape_ok) {
        // column strips: 64 byte columns (32 when 64 do not fit); 256-thread CTAs when at least two fit on an SM, else
        // one 512-thread CTA.  Measured on B200: at 4K one CTA with X = 64 beats three CTAs with X = 32 (27.4 vs 29.4 us
        // per frame); the width itself hardly matters for the row-strided DRAM side (profiles/).
        int X = 0, ctas = 0;
        if (cole_smem_bytes(g, 64) <= (size_t)smem_optin) X = 64;
        else if (cole_smem_bytes(g, 32) <= (size_t)smem_optin) X = 32;
        if (X) ctas = 2 * (cole_smem_bytes(g, X) + 1024) <= (size_t)smem_sm ? 3 : 1;
        // row pass: compute threads = one per quad of 4 pixels, at most 15 warps (+ the copy warp) when
        // several CTAs share an SM; the deepest ring of stages that still leaves 2 CTAs per SM, else what fits
        const uint32_t Q = g.w / 4;
        int nc = (int)(((Q + 31) / 32) * 32);
        if (nc > 480) nc = 480;
        int ns = 0;
        for (int cand = 3; cand >= 2 && !ns; --cand)
            if (2 * (row_smem_bytes(g, cand) + 1024) <= (size_t)smem_sm) ns = cand;
        bool row_big = false;
        if (!ns) {
            for (int cand = 3; cand >= 1 && !ns; --cand)
                if (row_smem_bytes(g, cand) <= (size_t)smem_optin) ns = cand;
            row_big = true;
            nc = (int)(((Q + 31) / 32) * 32);
            if (nc > 992) nc = 992;
        }
        void *fn = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (X && ns && cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess && fn) {
            p.tiled = true;
            p.encode_tiled = fn;
            p.strip_bytes = X;
            p.col_ctas_per_sm = ctas;
            p.strips_per_frame = (int)((g.row_bytes + X - 1) / X);
            p.smem_cole = cole_smem_bytes(g, X);
            // Encrypt direction: when three CTAs per SM would need the largest shared-memory carve-out (more than 196 KB with the
            // 1 KB the system reserves per CTA), ask for so much that only TWO fit.  Measured on B200 under the two-stream schedule,
            // ns per frame row at w = 1920: strips up to h = 1008 (three CTAs inside 196 KB) 4.13 - 4.15, h = 1024 .. 1184 (three CTAs,
            // 228 KB) 4.37 - 4.42, h >= 1200 (two CTAs) 4.12; FHD with the larger request 4.74 -> 4.49 us per frame.  The decrypt
            // direction, whose CTAs also convert their strip in shared memory, is faster with three (5.56 against 5.71).
            p.smem_cole_enc = p.smem_cole;
            if (ctas == 3 && 3 * (p.smem_cole + 1024) > (size_t)196 * 1024) {
                const size_t two_only = ((size_t)smem_sm / 3 - 1024 + 255) / 128 * 128;  // 3 x (this + 1 KB) > shared memory of an SM
                if (two_only > p.smem_cole && two_only <= (size_t)smem_optin) p.smem_cole_enc = two_only;
            }
            uint32_t br = 1;
            for (uint32_t d = 1; d <= 256 && d <= g.h; ++d)
                if (g.h % d == 0) br = d;
            p.box_rows = br;
            p.h_magic = (uint32_t)((((uint64_t)1 << 32) + g.h - 1) / g.h);
            p.row_ns = ns;
            p.row_nc = nc;
            p.row_big = row_big;
            p.smem_row = row_smem_bytes(g, ns);
            // Decrypt direction: where three CTAs with one input stage each fit an SM, the inverse row pass runs as three small
            // CTAs (160 compute threads: the pass waits on its copies, not on its arithmetic -- 128 to 480 compute threads give
            // the same time) instead of two with two stages.  Its CTAs then share an SM with the decrypt column pass's (three per
            // SM, the same 70 KB) in any mix.  Measured at FHD: decrypt 5.42 -> 5.19 us per frame (batches of 8: 6.50 -> 6.21);
            // the encrypt direction, whose column pass runs two CTAs per SM, loses with it (4.41 -> 4.60) and keeps two.
            p.row_nc_dec = nc;
            p.row_ns_dec = ns;
            p.smem_row_dec = p.smem_row;
            if (!row_big && 3 * (p.smem_row + 1024) > (size_t)smem_sm && 3 * (row_smem_bytes(g, 1) + 1024) <= (size_t)smem_sm) {
                p.row_nc_dec = nc < 160 ? nc : 160;
                p.row_ns_dec = 1;
                p.smem_row_dec = row_smem_bytes(g, 1);
            }
            // register-landing row pass: every width whose phase-1 items (w / 4 per block) fit one or two per thread
            p.row_reg = 0;
            p.row_reg_dec = false;
            p.smem_row_reg = rowreg_smem_bytes(g);
            if (!row_tma && p.smem_row_reg <= (size_t)smem_optin) {
                const uint32_t items = g.w / 4u;
                int per_sm = 0;
                if (items <= 256) { p.row_reg = 1; per_sm = 4; }
                else if (items <= 512) { p.row_reg = 2; per_sm = 3; }
                else if (items <= 1024) { p.row_reg = 3; per_sm = 2; }
                const int by_smem = (int)((size_t)smem_sm / (p.smem_row_reg + 1024));
                if (per_sm > by_smem) per_sm = by_smem;
                if (per_sm < 1) p.row_reg = 0;
                p.row_reg_grid_max = per_sm * sms;
                // inverse direction: everywhere except frames 1537 to 2048 pixels wide, where the TMA-staged pass as three small CTAs per
                // SM (row_ns_dec == 1) is as fast or faster.  Measured decrypt, TMA-staged -> register-landing, us per frame on resident
                // clips: 640 x 480 0.84 -> 0.75, 1024 x 768 1.99 -> 1.90, 1280 x 720 2.27 -> 2.21, 3840 x 2160 26.6 -> 25.2, but
                // 1760 x 992 4.30 -> 4.33, 1920 x 1080 4.95 -> 5.07, 2048 x 1080 5.40 -> 5.46.
                p.row_reg_dec = p.row_reg != 0 && !(p.row_ns_dec == 1 && g.w > 1536);
            }
            int rc = (int)((size_t)smem_sm / (p.smem_row + 1024));
            const int by_threads = 2048 / (nc + 32);
            if (rc > by_threads) rc = by_threads;
            if (rc > 3) rc = 3;
            if (rc < 1 || row_big) rc = 1;
            p.row_grid_max = rc * sms;
            {
                int rd = (int)((size_t)smem_sm / (p.smem_row_dec + 1024));
                const int bt = 2048 / (p.row_nc_dec + 32);
                if (rd > bt) rd = bt;
                if (rd > 3) rd = 3;
                if (rd < 1 || row_big) rd = 1;
                p.row_grid_max_dec = rd * sms;
            }
            // frames per launch pair: the intermediate of one pair should mostly fit the 126 MB L2.  Measured (profiles/):
            // 100 MB beats 56 MB (4K: 25.1 vs 27.4 us per frame; fewer, longer launches), and even a fully spilled
            // intermediate costs little -- the L2 trips bound the path, not the DRAM.
            const size_t l2_budget = (size_t)100 << 20;
            p.max_frames_per_launch = l2_budget / g.frame_bytes ? l2_budget / g.frame_bytes : 1;
            if (ctas == 3) {
                if (X == 64) { e = col_set_attr<64, 256, 3, VK_KD3>(device, p.smem_cole); if (!e) e = cole_set_attr<64, 256, 3, 1>(device, p.smem_cole_enc); if (!e) e = cole_set_attr<64, 256, 2, VK_DE2>(device, p.smem_cole_enc); }
                else { e = col_set_attr<32, 256, 3, VK_KD3>(device, p.smem_cole); if (!e) e = cole_set_attr<32, 256, 3, 1>(device, p.smem_cole_enc); }
            } else {
                if (X == 64) { e = col_set_attr<64, 512, 1, VK_KD1>(device, p.smem_cole); if (!e) e = cole_set_attr<64, 512, 1, VK_DE1>(device, p.smem_cole_enc); }
                else { e = col_set_attr<32, 512, 1, VK_KD1>(device, p.smem_cole); if (!e) e = cole_set_attr<32, 512, 1, VK_DE1>(device, p.smem_cole_enc); }
            }
            if (e != cudaSuccess) return e;
            e = raise_dyn_smem((const void *)row_pass_kernel<false, 512, 2>, device, p.smem_row);
            if (!e) e = raise_dyn_smem((const void *)row_pass_kernel<true, 512, 2>, device, p.smem_row);
            if (!e) e = raise_dyn_smem((const void *)row_pass_kernel<true, 256, 3>, device, p.smem_row_dec);
            if (!e) e = raise_dyn_smem((const void *)row_pass_kernel<false, 1024, 1>, device, p.smem_row);
            if (!e) e = raise_dyn_smem((const void *)row_pass_kernel<true, 1024, 1>, device, p.smem_row);
            if (!e && p.row_reg == 1) e = raise_dyn_smem((const void *)row_reg_kernel<false, 256, 4, 1>, device, p.smem_row_reg);
            if (!e && p.row_reg == 1) e = raise_dyn_smem((const void *)row_reg_kernel<true, 256, 4, 1>, device, p.smem_row_reg);
            if (!e && p.row_reg == 2) e = raise_dyn_smem((const void *)row_reg_kernel<false, 512, 3, 1>, device, p.smem_row_reg);
            if (!e && p.row_reg == 2) e = raise_dyn_smem((const void *)row_reg_kernel<true, 512, 3, 1>, device, p.smem_row_reg);
            if (!e && p.row_reg == 3) e = raise_dyn_smem((const void *)row_reg_kernel<false, 512, 2, 2>, device, p.smem_row_reg);
            if (!e && p.row_reg == 3) e = raise_dyn_smem((const void *)row_reg_kernel<true, 512, 2, 2>, device, p.smem_row_reg);
            if (e != cudaSuccess) return e;
        }
    }
    *out = p;
    return cudaSuccess;
}

// Launch with programmatic stream serialization (PDL): the kernel's prologue may overlap the tail of the previous kernel
// in the stream; every kernel launched this way calls pdl_wait() before it touches global memory that kernel may have written.
template <typename... KArgs, typename... Args>
static cudaError_t launch_pdl(void (*kernel)(KArgs...), uint32_t grid, uint32_t block, size_t smem, cudaStream_t st, Args... args) {
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3(grid);
    cfg.blockDim = dim3(block);
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, static_cast<KArgs>(args)...);
}

template <bool INV>
static cudaError_t launch_row(const Geom &g, const Plan &p, const uint8_t *src, const uint16_t *D, size_t n,
                              uint8_t *dst, cudaStream_t st) {
    const uint32_t nblocks = (uint32_t)(n * g.h / ROW_RB);
    if (p.row_reg && (!INV || p.row_reg_dec)) {
        const uint32_t gm = (uint32_t)p.row_reg_grid_max;
        const uint32_t rr = (nblocks + gm - 1u) / gm, gr = (nblocks + rr - 1u) / rr;  // balanced, as below
        if (p.row_reg == 3) return launch_pdl(row_reg_kernel<INV, 512, 2, 2>, gr, 512u, p.smem_row_reg, st, src, dst, D, g, nblocks);
        if (p.row_reg == 2) return launch_pdl(row_reg_kernel<INV, 512, 3, 1>, gr, 512u, p.smem_row_reg, st, src, dst, D, g, nblocks);
        if (p.row_reg == 1) return launch_pdl(row_reg_kernel<INV, 256, 4, 1>, gr, 256u, p.smem_row_reg, st, src, dst, D, g, nblocks);
    }
    // persistent CTAs, balanced: the fewest rounds the resident CTAs allow, then the smallest grid that needs no more rounds
    // (FHD, 5 frames: 1350 blocks = 5 rounds of 270 CTAs instead of 296 CTAs of which 166 take a 5th block; measured 4.50 ->
    // 4.44 us per frame, decrypt 5.58 -> 5.46: no CTA idles through a last round while it holds its share of the SM)
    const bool small = INV && p.row_ns_dec == 1 && p.row_nc_dec + 32 <= 256 && !p.row_big;  // three small CTAs per SM (decrypt)
    const uint32_t gmax = (uint32_t)(INV ? p.row_grid_max_dec : p.row_grid_max);
    const uint32_t rounds = (nblocks + gmax - 1u) / gmax;
    const uint32_t grid = (nblocks + rounds - 1u) / rounds;
    const uint32_t nc = (uint32_t)(INV ? p.row_nc_dec : p.row_nc), ns = (uint32_t)(INV ? p.row_ns_dec : p.row_ns);
    const size_t smem = INV ? p.smem_row_dec : p.smem_row;
    const uint32_t nt = nc + 32u;
    if (p.row_big) return launch_pdl(row_pass_kernel<INV, 1024, 1>, grid, nt, smem, st, src, dst, D, g, nblocks, ns, nc);
    if (small) return launch_pdl(row_pass_kernel<true, 256, 3>, grid, nt, smem, st, src, dst, D, g, nblocks, ns, nc);
    return launch_pdl(row_pass_kernel<INV, 512, 2>, grid, nt, smem, st, src, dst, D, g, nblocks, ns, nc);
}

// tensor map of an n*h x 3w byte matrix with tiles of X bytes x `rows` rows
static bool make_tmap(const Plan &p, const Geom &g, const void *base, size_t n, uint32_t rows, CUtensorMap *out) {
    const cuuint64_t dims[2] = {g.row_bytes, (cuuint64_t)n * g.h};
    const cuuint64_t strides[1] = {g.row_bytes};
    const cuuint32_t es[2] = {1, 1};
    const cuuint32_t box[2] = {(cuuint32_t)p.strip_bytes, rows};
    EncodeTiledFn enc = reinterpret_cast<EncodeTiledFn>(p.encode_tiled);
    return enc(out, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<void *>(base), dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// decrypt direction (row-major in and out)
static cudaError_t launch_col_dec(const Geom &g, const Plan &p, const uint8_t *src, const uint16_t *D, const uint8_t *B,
                                  size_t n, uint8_t *dst, cudaStream_t st) {
    alignas(64) CUtensorMap tm_src, tm_B;
    const uint32_t pbox = 64;  // look-ahead tile height (rows)
    if (!make_tmap(p, g, src, n, p.box_rows, &tm_src) || !make_tmap(p, g, B, n, pbox, &tm_B)) return cudaErrorInvalidValue;
    const uint32_t grid = (uint32_t)(n * p.strips_per_frame);
#define VK_COLD(X, NT, MINB, KD)                                                                                     \
    return launch_pdl(col_dec_kernel<X, NT, MINB, KD>, grid, NT, p.smem_cole, st, tm_src, tm_B, B, dst, D, g,           \
                      (uint32_t)p.strips_per_frame, p.h_magic, p.box_rows, pbox)
    if (p.col_ctas_per_sm == 3) {
        if (p.strip_bytes == 64) VK_COLD(64, 256, 3, VK_KD3);
        else VK_COLD(32, 256, 3, VK_KD3);
    } else {
        if (p.strip_bytes == 64) VK_COLD(64, 512, 1, VK_KD1);
        else VK_COLD(32, 512, 1, VK_KD1);
    }
#undef VK_COLD
    return cudaGetLastError();
}

// encrypt direction: the T4 intermediate in `io` is replaced by the ciphertext
static cudaError_t launch_col_enc(const Geom &g, const Plan &p, uint8_t *io, const uint16_t *D, const uint8_t *B, size_t n,
                                  cudaStream_t st) {
    alignas(64) CUtensorMap tm_main, tm_pad;
    const cuuint64_t dims[2] = {g.row_bytes, (cuuint64_t)n * g.h};
    const cuuint64_t strides[1] = {g.row_bytes};
    const cuuint32_t es[2] = {1, 1};
    const cuuint32_t box_main[2] = {(cuuint32_t)p.strip_bytes, p.box_rows}, box_pad[2] = {(cuuint32_t)p.strip_bytes, CE_PAD};
    EncodeTiledFn enc = reinterpret_cast<EncodeTiledFn>(p.encode_tiled);
    CUresult r = enc(&tm_main, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, io, dims, strides, box_main, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                     CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r == CUDA_SUCCESS)
        r = enc(&tm_pad, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, io, dims, strides, box_pad, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    alignas(64) CUtensorMap tm_B;
    const uint32_t pbox = 64;  // look-ahead tile height (rows)
    const cuuint32_t box_pf[2] = {(cuuint32_t)p.strip_bytes, pbox};
    if (r == CUDA_SUCCESS)
        r = enc(&tm_B, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<uint8_t *>(B), dims, strides, box_pf, es,
                CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return cudaErrorInvalidValue;
    const uint32_t grid = (uint32_t)(n * p.strips_per_frame);
#define VK_COLE(X, NT, MINB, DEPTH)                                                                                 \
    return launch_pdl(col_enc_kernel<X, NT, MINB, DEPTH>, grid, NT, p.smem_cole_enc, st, tm_main, tm_pad, tm_B, B, (uint8_t *)io, D, g, \
                      (uint32_t)p.strips_per_frame, (uint32_t)n, p.box_rows, p.h_magic, pbox)
    if (p.col_ctas_per_sm == 3) {
        // two CTAs per SM (the larger shared-memory request): registers for two rounds of keystream in flight per thread
        if (p.strip_bytes == 64 && p.smem_cole_enc != p.smem_cole) VK_COLE(64, 256, 2, VK_DE2);
        else if (p.strip_bytes == 64) VK_COLE(64, 256, 3, 1);
        else VK_COLE(32, 256, 3, 1);
    } else {
        if (p.strip_bytes == 64) VK_COLE(64, 512, 1, VK_DE1);
        else VK_COLE(32, 512, 1, VK_DE1);
    }
#undef VK_COLE
    return cudaGetLastError();
}

cudaError_t encrypt_tiled(const Geom &g, const Plan &p, const uint8_t *src, const uint16_t *D, const uint8_t *B,
                          size_t n, uint8_t *dst, cudaStream_t st, int *launches) {
    for (size_t f0 = 0; f0 < n; f0 += p.max_frames_per_launch) {
        const size_t m = n - f0 < p.max_frames_per_launch ? n - f0 : p.max_frames_per_launch;
        const size_t off = f0 * g.frame_bytes;
        cudaError_t e = launch_row<false>(g, p, src + off, D + f0 * g.nD, m, dst + off, st);
        if (e != cudaSuccess) return e;
        e = launch_col_enc(g, p, dst + off, D + f0 * g.nD, B + off, m, st);
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
        cudaError_t e = launch_col_dec(g, p, src + off, D + f0 * g.nD, B + off, m, dst + off, st);
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
