// cipher.cu -- the frame cipher's GPU steps (Algorithms 3-7 of PAPER.md:113-156 and their inverse, :79) as ONE
// persistent sm_100a kernel per call.
//
// The paper runs five kernels over explicit 0/1 bit matrices M_t^c / M_e^c of size 8w x h (Algorithm 1 steps 16-20).
// Those matrices are never materialised here.  Per channel c the five steps compose to:
//
//   hrot(i, j, c) = ( F_o(i, (j-q) mod w, c) << r  |  F_o(i, (j-q-1) mod w, c) >> (8-r) ) & 0xFF
//                   with s = d_h(i,c) mod 8w, q = s >> 3, r = s & 7          (Algo 3 + 4 + 7, Eq. 2)
//   F_e(ro, j, c) = B(ro, j, c) xor hrot((ro - d_v(j,c) mod h) mod h, j, c)   (Algo 5 + 6, Eq. 3)
//
// i.e. a per-(row, channel) bit rotation of a w-byte little-endian integer, then a per-byte-column circular shift in
// the interleaved h x 3w byte matrix, then a byte XOR.  The horizontal step needs whole rows, the vertical step whole
// columns, and a frame (6.2 MB at FHD) does not fit in shared memory: the exchange between them goes through the L2.
//
//   row blocks : 4 consecutive rows of one frame.  A load warp brings blocks into a ring of shared-memory stages with one
//                bulk async copy each (TMA, cp.async.bulk); the row team's compute warps de-interleave a block into three
//                channel planes (already rotated by the whole-chunk part of the distance), so that the bit rotation is ONE
//                32-bit funnel shift of two neighbouring plane words per output word; a store warp sends finished blocks out
//                with one bulk async store each.  When encrypting, a block is written in the "T4" layout: the word at
//                (row 4R + (x & 3), word column x >> 2) holds byte column x of rows 4R .. 4R+3 -- a permutation inside the
//                block, so the intermediate lives in the output buffer.
//   strips     : X = 64 byte columns x all h rows of one frame in shared memory, in the T4 layout (encrypt: brought in by
//                TMA tensor tiles; decrypt: converted in place after the XOR), so that ONE 32-bit shared-memory load returns
//                four consecutive rows of a byte column: 8 output rows of a column cost 3 conflict-free loads + 2 funnel
//                shifts.  The words are transposed back to row-major in registers (PRMT), XORed with the keystream
//                (64-bit streaming loads) and streamed out (64-bit stores).
//
// Round 1 ran the two as separate kernels; each alone left the DRAM and the L2 slices mostly idle (ncu: DRAM <= 31 %, lts <=
// 47 % busy): both are bound by the latency of their loads (2 - 3 us for a 23 KB block when the memory system is busy), and
// on an SM they ran in phases.  Here ONE persistent CTA per SM holds two specialised teams that run side by side for the
// whole call:
//   row team   : load warp + 8 compute warps + store warp.  The blocks are a continuous stream: the ring of stages is kept
//                full across work units (a ticket = a run of `bpi` blocks of one frame), two output buffers decouple the
//                compute warps from the stores, and the store warp -- not the compute warps -- pays for the gpu-scope release
//                that publishes finished blocks.
//   strip team : service warp + 12 compute warps (three rounds of row groups at FHD instead of five with 8 warps).
// Each team takes its work from its own ticket counter, frame after frame.  What couples them are two counters per frame:
// the following pass waits (acquire load by one lane) until the leading pass has finished the frame -- encrypt: strips wait
// for the frame's row blocks; decrypt: row blocks wait for the frame's strips -- and the leading pass stays at most `window`
// frames ahead of the following one, so that only a few frames of intermediate are alive in L2.  A team takes a ticket only
// when it runs and works its tickets in order, and everything a ticket waits for has a smaller frame number: no assumption
// on co-residency.  The launch state (tickets, exit count, per-frame counters) is zeroed by the last CTA to leave.
#include <cuda.h>

#include "kernels.cuh"
#include "ptx.cuh"
#include "smem_attr.hpp"

namespace vk {

constexpr int ROW_RB = 4;        // rows per block
constexpr int UNI_HDR = 2048;    // mbarriers, descriptors, shift parameters, column offsets
constexpr int ROW_MAXNS = 8;     // input stages at most
constexpr int ROW_MAXOB = 2;     // output buffers at most
constexpr int CE_PAD = 8;        // repeated strip rows
constexpr int CE_G = 8;          // output rows per group
#ifndef VK_NRW
#define VK_NRW 8
#endif
#ifndef VK_NSW
#define VK_NSW 12
#endif
constexpr int NRW = VK_NRW;      // row team: compute warps
constexpr int NSW = VK_NSW;      // strip team: compute warps
constexpr uint32_t DESC_TERM = 0xFFFFFFFFu, DESC_LAST = 0x80000000u;

// Per-item timeline for development builds (-DVK_TRACE; not part of the product)
#ifdef VK_TRACE
#define VK_TRACE_ITEMS 96
uint64_t *g_trace = nullptr;
#define VK_T(team, it, k) do { if (a.trace && (it) < VK_TRACE_ITEMS) a.trace[(((size_t)blockIdx.x * 2 + (team)) * VK_TRACE_ITEMS + (it)) * 8 + (k)] = global_timer_ns(); } while (0)
#else
#define VK_T(team, it, k) do { } while (0)
#endif

struct UniArgs {
#ifdef VK_TRACE
    uint64_t *trace;
#endif
    const uint8_t *src;
    uint8_t *dst;
    const uint16_t *D;
    const uint8_t *Bk;
    uint32_t *sched;        // [0] row tickets taken, [1] strip tickets taken, [2] CTAs that left, [4 + 2f] row blocks of frame f
                            // that are complete, [5 + 2f] strips of frame f that are complete
    Geom g;
    uint32_t nframes;
    uint32_t bpi;           // blocks per row ticket
    uint32_t rtpf;          // row tickets per frame
    uint32_t nblk;          // blocks per frame (h / 4)
    uint32_t strips;        // per frame
    uint32_t window;        // frames the leading pass may be ahead of the following one
    uint32_t NS, NOB;       // row team: input stages, output buffers
    uint32_t strip_off;     // byte offset of the strip inside the dynamic shared memory
    uint32_t bring_off;     // ... of the keystream ring
    uint32_t nring;         // chunks in the keystream ring (0 .. 2): the first rounds of a strip take their keystream from it
    uint32_t box_rows, h_magic, pf_rows;
};

// Waits until *p >= target (gpu-scope acquire), then orders the async proxy after it.  One lane.
__device__ __forceinline__ void wait_count(const uint32_t *p, uint32_t target) {
    uint64_t t0 = 0;
    for (uint32_t spin = 1; ld_acquire_gpu(p) < target; ++spin) {
        __nanosleep(32);
        if ((spin & 1023u) == 0) {
            const uint64_t t = global_timer_ns();
            if (t0 == 0) t0 = t;
            else if (t - t0 > kWaitLimitNs) __trap();
        }
    }
    fence_async_all();
}

struct Smem {
    uint64_t *full, *empty, *ofull, *ofree, *sitem, *sbar, *sfree, *bfull, *bfree;
    volatile uint32_t *sdesc;  // [2][2]: frame, strip (or DESC_TERM) of the strip team's current / next item
    volatile uint32_t *odesc;  // [ROW_MAXOB]: block in output buffer o (| DESC_LAST), or DESC_TERM
    volatile uint32_t *bdesc;  // [ROW_MAXNS]: block in stage s (| DESC_LAST), or DESC_TERM
    uint32_t *par1, *par2;     // [ROW_MAXNS][16]
    uint16_t *ups;             // [X]
    uint8_t *rows;             // stages, planes, output buffers
    uint8_t *strip;
    uint8_t *bring;            // keystream ring: chunks of GSTEP * 8 rows x X bytes
};
__device__ __forceinline__ Smem smem_map(uint8_t *smem, uint32_t strip_off, uint32_t bring_off) {
    Smem m;
    m.full = reinterpret_cast<uint64_t *>(smem);
    m.empty = reinterpret_cast<uint64_t *>(smem + 64);
    m.ofull = reinterpret_cast<uint64_t *>(smem + 128);
    m.ofree = reinterpret_cast<uint64_t *>(smem + 144);
    m.sitem = reinterpret_cast<uint64_t *>(smem + 160);
    m.sbar = reinterpret_cast<uint64_t *>(smem + 168);
    m.sfree = reinterpret_cast<uint64_t *>(smem + 176);
    m.bfull = reinterpret_cast<uint64_t *>(smem + 224);
    m.bfree = reinterpret_cast<uint64_t *>(smem + 240);
    m.sdesc = reinterpret_cast<volatile uint32_t *>(smem + 192);
    m.odesc = reinterpret_cast<volatile uint32_t *>(smem + 208);
    m.bdesc = reinterpret_cast<volatile uint32_t *>(smem + 256 + 128 * ROW_MAXNS + 256);
    m.par1 = reinterpret_cast<uint32_t *>(smem + 256);
    m.par2 = reinterpret_cast<uint32_t *>(smem + 256 + 64 * ROW_MAXNS);
    m.ups = reinterpret_cast<uint16_t *>(smem + 256 + 128 * ROW_MAXNS);
    m.rows = smem + UNI_HDR;
    m.strip = smem + strip_off;
    m.bring = smem + bring_off;
    return m;
}

// ---------------------------------------------------------------------------------------------
// Row team: horizontal bit rotation (Algorithm 4 / Eq. 2 on the rows of Algorithm 3's bit matrix, packed back as in
// Algorithm 7), block after block.
//   INV = false: bit p of channel c moves to (p + d_h mod 8w) mod 8w; the block is written in T4 layout.
//   INV = true : the inverse rotation; input and output are row-major.
// The compute threads work on a stage in two phases separated by a named barrier:
//   phase 1 (one item = 16 pixels of one row): 48 interleaved bytes -> three channel planes (PRMT network); the chunk is
//            stored already rotated by the whole-chunk part of the distance;
//   phase 2 (one item = a quad of 4 pixels, all 4 rows, all 3 channels): 12 funnel shifts, then either three 4 x 4 byte
//            transposes (T4) or the re-interleave to row-major; the result goes to an output buffer.
// Synchronisation: full[s] (mbarrier, two arrivals + the copy's bytes: block landed, parameters and descriptor written)
// load warp -> compute threads; empty[s] compute threads -> load warp once phase 1 has consumed the stage; ofull[o] /
// ofree[o] hand output buffer o to the store warp and back; named barrier 1 among the compute threads.
// In place (dst == src) is safe: a block is read completely before it is written.
// ---------------------------------------------------------------------------------------------

// Rotation of one (row, channel): output bit d takes source bit (d + sh) mod 8w, sh = 32 * (4 * dq + fine) + sh5.
// Phase 1 writes chunk k (16 pixels) of the plane at chunk position (k - dq) mod C, so that phase 2 reads the two
// words q + fine, q + fine + 1 of the pre-rotated plane (never wrapping: two pad chunks repeat chunks 0 and 1).
//   p1 = 16 * dq                      (bytes; phase 1)
//   p2 = (plane offset + 4 * fine) << 8 | sh5   (phase 2: one LEA.HI gives the address, the funnel shift takes sh5)
__device__ __forceinline__ uint2 row_param(const uint16_t *__restrict__ D, const Geom &g, uint32_t grow, uint32_t ch,
                                           bool inv, uint32_t plane_off) {
    const uint32_t f = grow / g.h, i = grow - f * g.h, W8 = 8u * g.w;
    const uint32_t s = (uint32_t)D[(size_t)f * g.nD + ch * (g.h + g.w) + i] % W8;
    const uint32_t sh = inv ? s : (s ? W8 - s : 0u);
    const uint32_t dw = sh >> 5;
    return make_uint2((dw >> 2) << 4, ((plane_off + 4u * (dw & 3u)) << 8) | (sh & 31u));
}

// The load warp: tickets, flow control / dependency, block copies, shift parameters.
template <bool INV>
__device__ __forceinline__ void row_load_warp(const Smem &m, const UniArgs &a, uint32_t lane) {
    const Geom &g = a.g;
    const uint32_t blk_bytes = ROW_RB * g.row_bytes, NS = a.NS, PS = g.w + 32u;
    const uint8_t *rsrc = INV ? a.dst : a.src;                      // decrypt: the strips' output, already in dst
    const uint32_t pr = lane / 3u, pch = lane - 3u * pr;            // lanes 0..11: (row, channel) of a block
    const uint32_t pslot = pr * 4u + pch, poff = (pr * 3u + pch) * PS;
    const uint64_t pol_in = policy_evict_first();
    const uint32_t total = a.nframes * a.rtpf;
    uint32_t tn = 0;
    if (lane == 0) tn = atomicAdd(a.sched + 0, 1u);
    uint32_t gi = 0;
    for (;;) {
        const uint32_t t = __shfl_sync(0xffffffffu, tn, 0);
        if (t >= total) break;
        if (lane == 0) tn = atomicAdd(a.sched + 0, 1u);            // the next ticket: its round trip hides behind this one
        const uint32_t f = t / a.rtpf, b0 = (t - f * a.rtpf) * a.bpi, nb = a.nblk - b0 < a.bpi ? a.nblk - b0 : a.bpi;
        if (lane == 0) {
            if (INV) wait_count(a.sched + 5 + 2 * f, a.strips);                                  // the frame's strips are written
            else if (f >= a.window) wait_count(a.sched + 5 + 2 * (f - a.window), a.strips);      // stay `window` frames ahead at most
        }
        __syncwarp();
        for (uint32_t k = 0; k < nb; ++k, ++gi) {
            const uint32_t s = gi % NS, blk = f * a.nblk + b0 + k;
            if (gi >= NS && lane == 0) mbar_wait(m.empty + s, ((gi / NS) - 1u) & 1u);  // the stage's previous block is consumed
            __syncwarp();
            if (lane == 0) {  // the copy first: the shift parameters need a round trip to D, the block must not wait for it
                mbar_expect_tx(m.full + s, blk_bytes);
                bulk_g2s_hint(m.rows + s * blk_bytes, rsrc + (size_t)blk * blk_bytes, blk_bytes, m.full + s, pol_in);
                m.bdesc[s] = blk | (k + 1u == nb ? DESC_LAST : 0u);
            }
            if (lane < 3 * ROW_RB) {
                const uint2 pv = row_param(a.D, g, blk * ROW_RB + pr, pch, INV, poff);
                m.par1[s * 16u + pslot] = pv.x;
                m.par2[s * 16u + pslot] = pv.y;
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(m.full + s);  // second arrival: parameters and descriptor are written
        }
    }
    if (lane == 0) {  // end of the stream
        const uint32_t s = gi % NS;
        if (gi >= NS) mbar_wait(m.empty + s, ((gi / NS) - 1u) & 1u);
        m.bdesc[s] = DESC_TERM;
        mbar_arrive(m.full + s);
        mbar_arrive(m.full + s);
    }
}

// The store warp: finished blocks out, output buffers back, and -- at the end of every ticket -- the gpu-scope release that
// tells the other pass (and the flow control) how many blocks of the frame are written.
__device__ __forceinline__ void row_store_warp(const Smem &m, const UniArgs &a, uint32_t lane) {
    if (lane != 0) return;
    const uint32_t blk_bytes = ROW_RB * a.g.row_bytes, NOB = a.NOB;
    uint8_t *obuf0 = m.rows + a.NS * blk_bytes + ROW_RB * 3u * (a.g.w + 32u);
    uint32_t npend = 0;
    for (uint32_t oi = 0;; ++oi) {
        const uint32_t o = oi % NOB;
        mbar_wait(m.ofull + o, (oi / NOB) & 1u);  // the compute threads have written a block into output buffer o
        const uint32_t d = m.odesc[o];
        if (d == DESC_TERM) break;
        const uint32_t blk = d & ~DESC_LAST;
        bulk_s2g(a.dst + (size_t)blk * blk_bytes, obuf0 + o * blk_bytes, blk_bytes);
        bulk_wait_read_0();                        // the store has left shared memory
        mbar_arrive(m.ofree + o);
        ++npend;
        if (d & DESC_LAST) {
            bulk_wait_all();                       // the ticket's blocks are written
            fence_async_all();
            red_release_gpu_add(a.sched + 4 + 2 * (blk / a.nblk), npend);
            npend = 0;
        }
    }
}

template <bool INV>
__device__ __forceinline__ void row_compute(const Smem &m, const UniArgs &a, uint32_t tid) {
    constexpr uint32_t NC = NRW * 32;
    const Geom &g = a.g;
    const uint32_t w = g.w, rb = g.row_bytes, C = w >> 4, Q = w >> 2;   // items / quads per row
    const uint32_t blk_bytes = ROW_RB * rb, NS = a.NS, NOB = a.NOB;
    const uint32_t PS = w + 32u;                                        // plane stride (bytes): w/4 words + 2 pad chunks
    uint8_t *stage0 = m.rows;
    uint8_t *planes = stage0 + NS * blk_bytes;
    uint8_t *obuf0 = planes + ROW_RB * 3u * PS;
    // loop-invariant work assignment: phase 1 item (row r1, chunk k1) = tid (further items: + NC), phase 2 quad = tid
    const uint32_t r1 = (tid >= C) + (tid >= 2u * C) + (tid >= 3u * C), k1 = tid - r1 * C;
    uint32_t gi = 0;
    for (;; ++gi) {
        const uint32_t s = gi % NS;
        const uint8_t *stage = stage0 + s * blk_bytes;
        const uint32_t *p1 = m.par1 + s * 16u, *p2 = m.par2 + s * 16u;
        mbar_wait(m.full + s, (gi / NS) & 1u);
        const uint32_t desc = m.bdesc[s];
        if (desc == DESC_TERM) break;
        if (tid == 0) VK_T(0, gi, 0);

        // ---- phase 1: de-interleave into planes; item = (row r, 16 pixels k)
        for (uint32_t i = tid; i < ROW_RB * C; i += NC) {
            uint32_t r = r1, k = k1;
            if (i != tid) { r = (i >= C) + (i >= 2u * C) + (i >= 3u * C); k = i - r * C; }
            const uint4 *p = reinterpret_cast<const uint4 *>(stage + r * rb + 48u * k);
            const uint4 va = p[0], vb = p[1], vc = p[2];
            const uint4 dq = *reinterpret_cast<const uint4 *>(p1 + 4u * r);
            const uint32_t W[12] = {va.x, va.y, va.z, va.w, vb.x, vb.y, vb.z, vb.w, vc.x, vc.y, vc.z, vc.w};
            uint4 v0, v1, v2;  // channel 0, 1, 2: four plane words each
#define VK_DEINT(mm, X0, X1, X2)                                                       \
    X0 = __byte_perm(__byte_perm(W[3 * mm], W[3 * mm + 1], 0x0630), W[3 * mm + 2], 0x5210); \
    X1 = __byte_perm(__byte_perm(W[3 * mm], W[3 * mm + 1], 0x0741), W[3 * mm + 2], 0x6210); \
    X2 = __byte_perm(__byte_perm(W[3 * mm], W[3 * mm + 1], 0x0052), W[3 * mm + 2], 0x7410);
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
        if (tid == 0) mbar_arrive(m.empty + s);
        const uint32_t o = gi % NOB;
        if (gi >= NOB) mbar_wait(m.ofree + o, ((gi / NOB) - 1u) & 1u);  // the buffer's previous block has left shared memory
        uint8_t *obuf = obuf0 + o * blk_bytes;

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
            uint8_t *op = obuf + 12u * q;
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
                        *reinterpret_cast<uint32_t *>(op + (y & 3) * rb + 4 * (y >> 2)) = T[p];
                    }
                }
            } else {
                // row-major: byte y = 3 * pixel + channel of the quad's 12 bytes
#pragma unroll
                for (int r = 0; r < ROW_RB; ++r) {
                    uint32_t *po = reinterpret_cast<uint32_t *>(op + r * rb);
                    po[0] = __byte_perm(__byte_perm(R[r][0], R[r][1], 0x1040), R[r][2], 0x3410);
                    po[1] = __byte_perm(__byte_perm(R[r][0], R[r][1], 0x6205), R[r][2], 0x3250);
                    po[2] = __byte_perm(__byte_perm(R[r][0], R[r][1], 0x0730), R[r][2], 0x7216);
                }
            }
        }
        fence_async_smem();     // generic-proxy writes to the output buffer -> visible to the bulk store
        named_bar_sync(1, NC);  // block complete; planes free for the next block
        if (tid == 0) {
            m.odesc[o] = desc;
            mbar_arrive(m.ofull + o);
            VK_T(0, gi, 1);
        }
    }
    if (tid == 0) {  // end of the stream: tell the store warp
        const uint32_t o = gi % NOB;
        if (gi >= NOB) mbar_wait(m.ofree + o, ((gi / NOB) - 1u) & 1u);
        m.odesc[o] = DESC_TERM;
        mbar_arrive(m.ofull + o);
    }
}

// ---------------------------------------------------------------------------------------------
// Strip team.  Encrypt direction: vertical circular shift of every byte column (Algorithm 5 / Eq. 3, one d_v per pixel
// column and channel = per byte column of the interleaved matrix) fused with the XOR of Algorithm 6:
//   dst(ro, x) = B(ro, x) xor I((ro - t_x) mod h, x),   I = the row team's output in T4 layout.
// One item = one strip of X byte columns of one frame, all h rows (+ 8 repeated rows so that a window never wraps) in
// shared memory, brought in by the TMA engine as 2-D tensor tiles (cp.async.bulk.tensor -> UTMALDG) once the frame's row
// blocks are complete: no thread touches the strip on its way in.  A warp is split into NSUB = 256 / X sub-warps of X / 8
// lanes; a lane owns 8 byte columns (two T4 word columns x four byte lanes) and a sub-warp emits groups of 8 consecutive
// output rows with 64-bit keystream loads and ciphertext stores.  Bank of a load = (strip row * X/4 + word column) mod 32
// with strip row = 4R + b: sub-warp s walks its columns in the order (word column a_l ^ (s & 1), byte lane a_b ^ (s >> 1)),
// so the sub-warps of a warp always sit in disjoint banks whatever rows they read: no conflicts.  The permutation is undone
// by the selectors of the 4 x 4 byte transposes and by one select per output word.  The keystream is kept two iterations of
// rows ahead on its way from DRAM to L2 with TMA tile prefetches.
// In place is safe: the whole strip is in shared memory before the first store.
// ---------------------------------------------------------------------------------------------
#define VK_ROWPTR(T, P, OFF) reinterpret_cast<T>(mad_wide_ptr(P, OFF))

// The conflict-free gather shared by both directions: emits the groups gi = g0, g0 + GSTEP, ... of 8 output rows of this
// lane's 8 byte columns.  XOR_B: xor the keystream (encrypt) and stream the result out; else plain stores (decrypt: the
// inverse row items read them from L2).
template <int X, int NT, bool XOR_B>
__device__ __forceinline__ void strip_gather(const uint8_t *S, const uint16_t *ups, const CUtensorMap *tm_B, const uint8_t *pB,
                                             uint8_t *pO, uint2 (&kb)[CE_G], uint32_t h, uint32_t rb, uint32_t g0, uint32_t j,
                                             uint32_t sub, uint32_t x0, uint32_t frow0, uint32_t pf_row, uint32_t pf_rows, bool pf_lead,
                                             const uint8_t *bring, uint64_t *bfull, uint64_t *bfree, uint32_t bpar, uint32_t nring,
                                             uint64_t *tr = nullptr) {
    constexpr uint32_t LPS = X / 8, NSUB = 32 / LPS, NW = NT / 32, GSTEP = NW * NSUB;
    constexpr uint32_t CE_AHEAD = 2u * GSTEP * CE_G;
    const uint32_t sl = sub & 1u, sb = sub >> 1;   // permutation of the word column / byte lane order
    const uint32_t nfull = h / CE_G;               // full groups; h % 8 == 4 leaves one half group
    const uint32_t rb2 = 2u * rb, rb3 = 3u * rb, rb4 = 4u * rb, rb5 = 5u * rb, rb6 = 6u * rb, rb7 = 7u * rb;
    const size_t gstep = (size_t)(GSTEP * CE_G) * rb;
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

    // keystream of a round: rounds 0 .. nring-1 from the shared-memory ring (chunk r = the GSTEP * 8 rows of round r, brought
    // in by TMA tiles long before), later rounds from registers (kb: loaded one round ahead, the first of them at item start)
    const uint8_t *bk_s = bring + (size_t)(g0 * CE_G) * X + 8u * j;
    uint32_t r = 0;
    for (uint32_t gi = g0;; gi += GSTEP, ++r) {
        const bool ring = XOR_B && r < nring;
        if (ring) mbar_wait(bfull + r, bpar);
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
        const int nrow = gi < nfull ? CE_G : CE_G / 2;  // the half group at the bottom of a frame with h % 8 == 4: always the last one
        if (ring) {
            const uint8_t *bc = bk_s + (size_t)r * (GSTEP * CE_G * X);
#pragma unroll
            for (int i = 0; i < CE_G; ++i) {
                if (i < nrow) {
                    const uint2 k = *reinterpret_cast<const uint2 *>(bc + i * X);
                    const uint32_t lo = sl ? O[i][1] : O[i][0], hi = sl ? O[i][0] : O[i][1];
                    __stcs(VK_ROWPTR(uint2 *, pO, offs[i]), make_uint2(lo ^ k.x, hi ^ k.y));
                }
            }
        } else if (gi < nfull) {
#pragma unroll
            for (int i = 0; i < CE_G; ++i) {
                const uint32_t lo = sl ? O[i][1] : O[i][0], hi = sl ? O[i][0] : O[i][1];
                if (XOR_B) __stcs(VK_ROWPTR(uint2 *, pO, offs[i]), make_uint2(lo ^ kb[i].x, hi ^ kb[i].y));
                else *VK_ROWPTR(uint2 *, pO, offs[i]) = make_uint2(lo, hi);
            }
        } else {
#pragma unroll
            for (int i = 0; i < CE_G / 2; ++i) {
                const uint32_t lo = sl ? O[i][1] : O[i][0], hi = sl ? O[i][0] : O[i][1];
                if (XOR_B) __stcs(VK_ROWPTR(uint2 *, pO, offs[i]), make_uint2(lo ^ kb[i].x, hi ^ kb[i].y));
                else *VK_ROWPTR(uint2 *, pO, offs[i]) = make_uint2(lo, hi);
            }
        }
        if (tr) tr[3 + r] = global_timer_ns();
        if (ring) mbar_arrive(bfree + r);  // this thread has read its part of chunk r (every thread of the team arrives once per chunk)
        if (nrow != CE_G) break;
        const uint32_t gn = gi + GSTEP;
        if (gn * CE_G >= h) break;
        pO += gstep;
        if (XOR_B) {
            pB += gstep;
            if (r + 1u > nring) {  // (round nring's keystream was loaded at item start)
                // keystream of the next group; the team's first thread keeps its tiles CE_AHEAD rows ahead on their way to L2
                if (pf_lead && pf_rows)
                    for (; pf_row < h && pf_row < gn * CE_G + CE_AHEAD; pf_row += pf_rows)
                        tma_prefetch_2d(tm_B, (int32_t)x0, (int32_t)(frow0 + pf_row));
                if (gn < nfull) {
#pragma unroll
                    for (int i = 0; i < CE_G; ++i) kb[i] = __ldcs(VK_ROWPTR(const uint2 *, pB, offs[i]));
                } else {
#pragma unroll
                    for (int i = 0; i < CE_G / 2; ++i) kb[i] = __ldcs(VK_ROWPTR(const uint2 *, pB, offs[i]));
                }
            }
        }
    }
    if (XOR_B)
        for (++r; r < nring; ++r) mbar_arrive(bfree + r);  // chunks of rounds this thread has no group in
}

// The service warp of the strip team: tickets, dependency / flow control, keystream look-ahead, the strip's tensor tiles,
// and the gpu-scope release for the strip the team has just finished.
template <bool INV, int X, int NT>
__device__ __forceinline__ void strip_service_warp(const Smem &m, const UniArgs &a, const CUtensorMap *tm_a, const CUtensorMap *tm_pad,
                                                   const CUtensorMap *tm_B, uint32_t lane) {
    if (lane != 0) return;
    constexpr uint32_t LPS = X / 8, NSUB = 32 / LPS, NW = NT / 32, GSTEP = NW * NSUB;
    constexpr uint32_t AHEAD = INV ? 2u * 4u * GSTEP : 2u * GSTEP * CE_G;  // keystream rows asked for before the strip
    constexpr uint32_t RPR = GSTEP * CE_G;                                 // rows of one round of the team = rows of a ring chunk
    const uint32_t h = a.g.h, total = a.nframes * a.strips;
    const uint32_t rounds = (h + RPR - 1u) / RPR, nr = INV ? 0u : (a.nring < rounds ? a.nring : rounds);
    const uint64_t pol = policy_evict_first();
    uint32_t tn = atomicAdd(a.sched + 1, 1u);
    uint32_t ci = 0, prev_f = 0;
    for (;; ++ci) {
        const uint32_t t = tn;
        if (t >= total) break;
        tn = atomicAdd(a.sched + 1, 1u);
        const uint32_t f = t / a.strips, strip = t - f * a.strips, x0 = strip * X, frow0 = f * h;
        // keystream: the chunks of the first rounds into the shared-memory ring as soon as the team has read the previous strip's
        // (TMA tiles; nothing here depends on the other pass), the L2 look-ahead for the rounds that load it themselves
        for (uint32_t c = 0; c < nr; ++c) {
            if (ci > 0) mbar_wait(m.bfree + c, (ci - 1u) & 1u);
            mbar_expect_tx(m.bfull + c, RPR * X);
            for (uint32_t r0 = 0; r0 < RPR; r0 += a.pf_rows)
                tma_load_2d(m.bring + (size_t)(c * RPR + r0) * X, tm_B, (int32_t)x0, (int32_t)(frow0 + c * RPR + r0), m.bfull + c, pol);
        }
        for (uint32_t pf_row = nr * RPR; pf_row < h && pf_row < nr * RPR + AHEAD; pf_row += a.pf_rows)
            tma_prefetch_2d(tm_B, (int32_t)x0, (int32_t)(frow0 + pf_row));
        if (ci > 0) mbar_wait(m.sfree, (ci - 1u) & 1u);  // the team is done with the previous strip: its buffer is free
        m.sdesc[2u * (ci & 1u)] = f;
        m.sdesc[2u * (ci & 1u) + 1u] = strip;
        mbar_arrive(m.sitem);                            // the team may start on the column offsets and its first keystream loads
        // what this strip waits for: encrypt -- the frame's row blocks; decrypt -- the row team `window` frames behind
        const uint32_t *wp = nullptr;
        uint32_t wt = 0;
        if (!INV) { wp = a.sched + 4 + 2 * f; wt = a.nblk; }
        else if (f >= a.window) { wp = a.sched + 4 + 2 * (f - a.window); wt = a.nblk; }
        const bool ready = !wp || ld_acquire_gpu(wp) >= wt;
        if (!ready && ci > 0) {  // publish the previous strip before blocking: somebody upstream may be waiting for it
            __threadfence();
            red_release_gpu_add(a.sched + 5 + 2 * prev_f, 1u);
        }
        if (wp) wait_count(wp, wt);
        VK_T(1, ci, 6);
        fence_async_all();       // the strip buffer was last written / read through the generic proxy
        if (!INV) {
            mbar_expect_tx(m.sbar, (h + CE_PAD) * X);
            for (uint32_t r0 = 0; r0 < h; r0 += a.box_rows) tma_load_2d(m.strip + (size_t)r0 * X, tm_a, (int32_t)x0, (int32_t)(frow0 + r0), m.sbar, pol);
            tma_load_2d(m.strip + (size_t)h * X, tm_pad, (int32_t)x0, (int32_t)frow0, m.sbar, pol);
        } else {
            mbar_expect_tx(m.sbar, h * X);
            for (uint32_t r0 = 0; r0 < h; r0 += a.box_rows) tma_load_2d(m.strip + (size_t)r0 * X, tm_a, (int32_t)x0, (int32_t)(frow0 + r0), m.sbar, pol);
        }
        if (ready && ci > 0) {   // the previous strip's release, behind this strip's loads
            __threadfence();
            red_release_gpu_add(a.sched + 5 + 2 * prev_f, 1u);
        }
        prev_f = f;
    }
    if (ci > 0) {
        mbar_wait(m.sfree, (ci - 1u) & 1u);
        __threadfence();
        red_release_gpu_add(a.sched + 5 + 2 * prev_f, 1u);
    }
    m.sdesc[2u * (ci & 1u)] = DESC_TERM;
    mbar_arrive(m.sitem);
}

template <bool INV, int X, int NT>
__device__ __forceinline__ void strip_compute(const Smem &m, const UniArgs &a, const CUtensorMap *tm_B, uint32_t tid) {
    constexpr uint32_t LPS = X / 8, NSUB = 32 / LPS, NW = NT / 32, GSTEP = NW * NSUB;
    constexpr uint32_t CE_AHEAD = 2u * GSTEP * CE_G, CD_AHEAD = 2u * 4u * GSTEP;
    const Geom &g = a.g;
    const uint32_t h = g.h, rb = g.row_bytes;
    uint8_t *S = m.strip;
    const uint32_t lane = tid & 31u, warp = tid >> 5;
    const uint32_t sub = lane / LPS, j = lane % LPS;
    const uint32_t g0 = warp * NSUB + sub;         // first row group (encrypt, gather) / first block of 4 rows (decrypt, phase A)
    const uint32_t nfull = h / CE_G;
    const uint32_t rb2 = 2u * rb, rb3 = 3u * rb;
    const uint32_t rounds = (h + GSTEP * CE_G - 1u) / (GSTEP * CE_G), nr = INV ? 0u : (a.nring < rounds ? a.nring : rounds);
    for (uint32_t ci = 0;; ++ci) {
        mbar_wait(m.sitem, ci & 1u);
        const uint32_t f = m.sdesc[2u * (ci & 1u)];
        if (f == DESC_TERM) break;
        const uint32_t strip = m.sdesc[2u * (ci & 1u) + 1u];
        const uint32_t x0 = strip * X, frow0 = f * h;
        if (tid == 0) VK_T(1, ci, 0);
        // one thread per byte column of the strip: the row offset of the column's source
        if (tid >= NT - X) {
            const uint32_t xs = tid - (NT - X);
            uint32_t x = x0 + xs;
            if (x >= rb) x = 0;
            const uint32_t jj = x / 3u, c = x - 3u * jj;
            const uint32_t dv = a.D[(size_t)f * g.nD + c * (h + g.w) + h + jj];
            const uint32_t t = dv - __umulhi(dv, a.h_magic) * h;  // d_v mod h  (h_magic = ceil(2^32 / h), d_v < 2^16)
            m.ups[xs] = (uint16_t)(INV ? t : (t ? h - t : 0u));
        }
        const uint32_t xt = x0 + 8u * j;               // first of this lane's 8 byte columns (frame coordinates)
        const bool col_ok = xt < rb;                   // rb % 8 == 0 on this path: the 8 columns are inside or outside together
        const size_t fcol = (size_t)f * g.frame_bytes + xt;
        if (!INV) {
            const bool active = col_ok && g0 * CE_G < h;
            const size_t fbase = fcol + (size_t)(g0 * CE_G) * rb;
            const uint8_t *pB = a.Bk + fbase;          // row g0 * 8 of this lane's columns
            uint8_t *pO = a.dst + fbase;
            // keystream: the first nr rounds come from the shared-memory ring; the next one is loaded here, before the strip arrives
            uint2 kb[CE_G];
#pragma unroll
            for (int i = 0; i < CE_G; ++i) kb[i] = make_uint2(0u, 0u);
            const uint32_t gk = g0 + nr * GSTEP;
            if (col_ok && gk * CE_G < h) {
                const uint8_t *pk = pB + (size_t)(nr * GSTEP * CE_G) * rb;
                const uint32_t offs[8] = {0u, rb, 2u * rb, 3u * rb, 4u * rb, 5u * rb, 6u * rb, 7u * rb};
                if (gk < nfull) {
#pragma unroll
                    for (int i = 0; i < CE_G; ++i) kb[i] = __ldcs(VK_ROWPTR(const uint2 *, pk, offs[i]));
                } else {
#pragma unroll
                    for (int i = 0; i < CE_G / 2; ++i) kb[i] = __ldcs(VK_ROWPTR(const uint2 *, pk, offs[i]));
                }
            }
            named_bar_sync(2, NT);       // ups[] complete
            mbar_wait(m.sbar, ci & 1u);  // strip (and its wrap rows) has landed
            if (tid == 0) VK_T(1, ci, 1);
            if (active) {
                uint32_t pf_row = nr * GSTEP * CE_G;     // where the service lane's look-ahead stopped
                while (pf_row < h && pf_row < nr * GSTEP * CE_G + CE_AHEAD) pf_row += a.pf_rows;
#ifdef VK_TRACE
                uint64_t *tr = (tid == 0 && a.trace && ci < VK_TRACE_ITEMS) ? a.trace + (((size_t)blockIdx.x * 2 + 1) * VK_TRACE_ITEMS + ci) * 8 : nullptr;
#else
                uint64_t *tr = nullptr;
#endif
                strip_gather<X, NT, true>(S, m.ups, tm_B, pB, pO, kb, h, rb, g0, j, sub, x0, frow0, pf_row, a.pf_rows, tid == 0, m.bring,
                                          m.bfull, m.bfree, ci & 1u, nr, tr);
            } else {
                for (uint32_t c = 0; c < nr; ++c) mbar_arrive(m.bfree + c);
            }
        } else {
            // ---- phase A: strip -> (strip xor B) in T4 layout, in place.  Item = (block of 4 rows R, this lane's 8 byte
            // columns); step t works on row / byte lane t ^ s1 (the two sub-warps of a half warp sit in disjoint banks).
            const uint32_t s1 = sub & 1u;
            const uint32_t nblk4 = h >> 2;
            const uint32_t offs4[4] = {s1 ? rb : 0u, s1 ? 0u : rb, s1 ? rb3 : rb2, s1 ? rb2 : rb3};
            const uint8_t *pB = a.Bk + fcol + (size_t)(4u * g0) * rb;
            uint2 kn[4];
#pragma unroll
            for (int t = 0; t < 4; ++t) kn[t] = make_uint2(0u, 0u);
            if (col_ok && g0 < nblk4) {  // keystream of the first block: issued before the strip arrives
#pragma unroll
                for (int t = 0; t < 4; ++t) kn[t] = __ldcs(VK_ROWPTR(const uint2 *, pB, offs4[t]));
            }
            named_bar_sync(2, NT);       // ups[] complete
            mbar_wait(m.sbar, ci & 1u);  // the ciphertext strip has landed
            if (tid == 0) VK_T(1, ci, 1);
            if (col_ok) {
                uint32_t pf_row = 0;
                while (a.pf_rows && pf_row < h && pf_row < CD_AHEAD) pf_row += a.pf_rows;
                const uint32_t selA = s1 ? 0x1504u : 0x5140u, selB = s1 ? 0x3726u : 0x7362u;  // inputs arrive as rows (t ^ s1)
                const uint32_t selF = s1 ? 0x7632u : 0x5410u, selS = s1 ? 0x5410u : 0x7632u;  // first / second byte lane of a pair
                const size_t bstep = (size_t)(4u * GSTEP) * rb;
                const int32_t d1 = s1 ? -(int32_t)X : (int32_t)X;
                for (uint32_t R4 = g0; R4 < nblk4; R4 += GSTEP) {
                    uint2 k[4];
#pragma unroll
                    for (int t = 0; t < 4; ++t) k[t] = kn[t];
                    pB += bstep;
                    if (tid == 0 && a.pf_rows)
                        for (; pf_row < h && pf_row < 4u * (R4 + GSTEP) + CD_AHEAD; pf_row += a.pf_rows)
                            tma_prefetch_2d(tm_B, (int32_t)x0, (int32_t)(frow0 + pf_row));
                    if (R4 + GSTEP < nblk4) {
#pragma unroll
                        for (int t = 0; t < 4; ++t) kn[t] = __ldcs(VK_ROWPTR(const uint2 *, pB, offs4[t]));
                    }
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
                        const uint32_t aa = __byte_perm(v[0].x, v[1].x, selA), bb = __byte_perm(v[0].x, v[1].x, selB);
                        const uint32_t cc = __byte_perm(v[2].x, v[3].x, selA), dd = __byte_perm(v[2].x, v[3].x, selB);
                        lo[0] = __byte_perm(aa, cc, selF); lo[1] = __byte_perm(aa, cc, selS);
                        lo[2] = __byte_perm(bb, dd, selF); lo[3] = __byte_perm(bb, dd, selS);
                    }
                    {
                        const uint32_t aa = __byte_perm(v[0].y, v[1].y, selA), bb = __byte_perm(v[0].y, v[1].y, selB);
                        const uint32_t cc = __byte_perm(v[2].y, v[3].y, selA), dd = __byte_perm(v[2].y, v[3].y, selB);
                        hi[0] = __byte_perm(aa, cc, selF); hi[1] = __byte_perm(aa, cc, selS);
                        hi[2] = __byte_perm(bb, dd, selF); hi[3] = __byte_perm(bb, dd, selS);
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
                }
            }
            named_bar_sync(2, NT);  // strip converted
            if (col_ok && g0 * CE_G < h) {
                uint8_t *pO = a.dst + fcol + (size_t)(g0 * CE_G) * rb;
                uint2 kb[CE_G];     // unused in this direction
                strip_gather<X, NT, false>(S, m.ups, tm_B, nullptr, pO, kb, h, rb, g0, j, sub, x0, frow0, 0u, 0u, false, nullptr, nullptr, nullptr, 0u, 0u);
            }
        }
        named_bar_sync(2, NT);      // everybody is done with the strip and has issued its stores
        if (tid == 0) {
            mbar_arrive(m.sfree);   // (release at CTA scope; the service lane adds the gpu-scope release)
            VK_T(1, ci, 2);
        }
    }
}
#undef VK_ROWPTR

// ---------------------------------------------------------------------------------------------
// The kernel: one persistent CTA per SM.  Warps 0 .. 7 row compute, 8 row load, 9 row store, 10 .. 10 + NSW - 1 strip
// compute, 10 + NSW strip service.
// ---------------------------------------------------------------------------------------------
template <bool INV, int X, int NSW_>
__global__ void __launch_bounds__((NRW + NSW_ + 3) * 32, 1)
    cipher_kernel(const __grid_constant__ CUtensorMap tm_a, const __grid_constant__ CUtensorMap tm_pad,
                  const __grid_constant__ CUtensorMap tm_B, const UniArgs a) {
    extern __shared__ __align__(1024) uint8_t smem[];
    const Smem m = smem_map(smem, a.strip_off, a.bring_off);
    const uint32_t tid = threadIdx.x, warp = tid >> 5, lane = tid & 31u;
    if (tid == 0) {
        for (uint32_t s = 0; s < ROW_MAXNS; ++s) { mbar_init(m.full + s, 2); mbar_init(m.empty + s, 1); }
        for (uint32_t o = 0; o < ROW_MAXOB; ++o) { mbar_init(m.ofull + o, 1); mbar_init(m.ofree + o, 1); }
        mbar_init(m.sitem, 1);
        mbar_init(m.sbar, 1);
        mbar_init(m.sfree, 1);
        for (uint32_t c = 0; c < 2; ++c) { mbar_init(m.bfull + c, 1); mbar_init(m.bfree + c, NSW_ * 32); }
        mbar_init_fence();
    }
    if (tid == 32) { tmap_prefetch(&tm_a); tmap_prefetch(&tm_pad); tmap_prefetch(&tm_B); }
    pdl_trigger();    // the next kernel of the stream may be scheduled as SMs free up; it waits below before it touches anything
    __syncthreads();
    pdl_wait();       // everything below reads or writes global memory (and the launch state) the previous kernel may have written

    if (warp < NRW) row_compute<INV>(m, a, tid);
    else if (warp == NRW) row_load_warp<INV>(m, a, lane);
    else if (warp == NRW + 1) row_store_warp(m, a, lane);
    else if (warp < NRW + 2 + NSW_) strip_compute<INV, X, NSW_ * 32>(m, a, &tm_B, tid - (NRW + 2) * 32);
    else strip_service_warp<INV, X, NSW_ * 32>(m, a, &tm_a, &tm_pad, &tm_B, lane);

    // the last CTA to leave restores the launch state for the next launch that uses this buffer
    __syncthreads();
    if (warp == 0) {
        uint32_t last = 0;
        if (lane == 0) {
            __threadfence();
            last = atomicAdd(a.sched + 2, 1u) == gridDim.x - 1u;
        }
        last = __shfl_sync(0xffffffffu, last, 0);
        if (last) {
            __threadfence();
            for (uint32_t i = lane; i < 2u * a.nframes; i += 32u) a.sched[4 + i] = 0u;
            if (lane == 0) { a.sched[0] = 0u; a.sched[1] = 0u; a.sched[2] = 0u; }
        }
    }
}

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
static size_t uni_row_bytes(const Geom &g, int ns, int nob) {
    const size_t b = (size_t)(ns + nob) * ROW_RB * g.row_bytes + (size_t)ROW_RB * 3 * (g.w + 32);
    return (b + 127) / 128 * 128;
}
static size_t uni_strip_bytes(const Geom &g, int X) { return (size_t)(g.h + CE_PAD) * X; }

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *, const cuuint64_t *,
                                  const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

template <bool INV, int X, int NSW_>
static cudaError_t uni_attr(int device, size_t smem) {
    return raise_dyn_smem((const void *)cipher_kernel<INV, X, NSW_>, device, smem);
}

cudaError_t make_uni_plan(const Geom &g, int device, const UniTune &tune, UniPlan *out) {
    UniPlan p{};
    int smem_optin = 0, sms = 0;
    cudaError_t e = cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, device);
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, device);
    if (e != cudaSuccess) return e;
    p.ok = false;
    const bool shape_ok = g.w % 16 == 0 && g.h % 4 == 0 && g.h >= 2 * CE_PAD && g.w >= 64 && g.frame_bytes < ((size_t)1 << 31);
    if (shape_ok) {
        // strips of 64 byte columns (32 when a 64-wide strip leaves no room for the row team); the row ring gets what is left:
        // two output buffers and up to ROW_MAXNS stages
        int X = 0;
        for (int cand = 64; cand >= 32 && !X; cand /= 2)
            if (UNI_HDR + uni_row_bytes(g, 1, 1) + uni_strip_bytes(g, cand) <= (size_t)smem_optin) X = cand;
        if (X) {
            // what is left beside the strip goes to the keystream ring (two chunks = two rounds of the strip team) and to the row
            // ring: at least two stages and one output buffer before the keystream ring gets its second chunk
            const size_t chunk = (size_t)NSW * (32 / (X / 8)) * CE_G * X;  // GSTEP * 8 rows x X bytes
            const size_t room = (size_t)smem_optin - UNI_HDR - uni_strip_bytes(g, X);
            int ns = 1, nob = 1, nring = 0;
            const int want_ring = tune.ring == 3 ? 0 : (tune.ring ? (int)tune.ring : 2);
            for (int r = want_ring; r >= 0; --r)
                if (uni_row_bytes(g, r ? 2 : 1, 1) + (size_t)r * chunk <= room) { nring = r; break; }
            const size_t rroom = room - (size_t)nring * chunk;
            while (ns < 3 && uni_row_bytes(g, ns + 1, nob) <= rroom) ++ns;
            if (uni_row_bytes(g, ns, 2) <= rroom) nob = 2;
            while (ns < 4 && uni_row_bytes(g, ns + 1, nob) <= rroom) ++ns;
            if (tune.row_stages >= 1 && tune.row_stages <= (uint32_t)ROW_MAXNS) {
                for (int o = 2; o >= 1; --o)
                    if (uni_row_bytes(g, (int)tune.row_stages, o) <= rroom) { ns = (int)tune.row_stages; nob = o; break; }
            }
            p.X = X;
            p.ns = ns;
            p.nob = nob;
            p.nring = nring;
            p.strip_off = (uint32_t)(UNI_HDR + uni_row_bytes(g, ns, nob));
            p.bring_off = (uint32_t)(p.strip_off + uni_strip_bytes(g, X));
            p.smem = p.bring_off + (size_t)nring * chunk;
            p.grid_max = sms;
            p.nblk = g.h / ROW_RB;
            p.bpi = tune.row_item_blocks ? (int)tune.row_item_blocks : 3;  // measured at FHD: 3 blocks per ticket, window 8 (4.61 us per frame; 6 / 4: 7.98)
            if (p.bpi > (int)p.nblk) p.bpi = (int)p.nblk;
            p.row_items = (p.nblk + p.bpi - 1) / p.bpi;
            p.strips = (g.row_bytes + X - 1) / X;
            p.window = tune.window ? tune.window : 8;
            uint32_t br = 1;
            for (uint32_t d = 1; d <= 256 && d <= g.h; ++d)
                if (g.h % d == 0) br = d;
            p.box_rows = br;
            p.h_magic = (uint32_t)((((uint64_t)1 << 32) + g.h - 1) / g.h);
            void *fn = nullptr;
            cudaDriverEntryPointQueryResult qres;
            if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres) == cudaSuccess &&
                qres == cudaDriverEntryPointSuccess && fn) {
                p.encode_tiled = fn;
                if (X == 64) { e = uni_attr<false, 64, NSW>(device, p.smem); if (!e) e = uni_attr<true, 64, NSW>(device, p.smem); }
                else { e = uni_attr<false, 32, NSW>(device, p.smem); if (!e) e = uni_attr<true, 32, NSW>(device, p.smem); }
                if (e != cudaSuccess) return e;
                p.ok = true;
            }
        }
    }
    *out = p;
    return cudaSuccess;
}

// tensor map of an n*h x 3w byte matrix with tiles of X bytes x `rows` rows
static bool make_tmap(const UniPlan &p, const Geom &g, const void *base, size_t n, uint32_t rows, CUtensorMap *out) {
    const cuuint64_t dims[2] = {g.row_bytes, (cuuint64_t)n * g.h};
    const cuuint64_t strides[1] = {g.row_bytes};
    const cuuint32_t es[2] = {1, 1};
    const cuuint32_t box[2] = {(cuuint32_t)p.X, rows};
    EncodeTiledFn enc = reinterpret_cast<EncodeTiledFn>(p.encode_tiled);
    return enc(out, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, const_cast<void *>(base), dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

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

cudaError_t cipher_launch(const Geom &g, const UniPlan &p, bool decrypt, const uint8_t *src, const uint16_t *D, const uint8_t *B,
                          size_t n, uint8_t *dst, uint32_t *sched, cudaStream_t st) {
    alignas(64) CUtensorMap tm_a, tm_pad, tm_B;
    const uint32_t pbox = 128;  // keystream tile height (rows): ring chunks and L2 look-ahead
    // encrypt: the strips are read from the intermediate in dst; decrypt: from the ciphertext in src
    const void *sbase = decrypt ? (const void *)src : (const void *)dst;
    if (!make_tmap(p, g, sbase, n, p.box_rows, &tm_a) || !make_tmap(p, g, sbase, n, CE_PAD, &tm_pad) || !make_tmap(p, g, B, n, pbox, &tm_B))
        return cudaErrorInvalidValue;
    UniArgs a{};
#ifdef VK_TRACE
    a.trace = g_trace;
#endif
    a.src = src; a.dst = dst; a.D = D; a.Bk = B; a.sched = sched; a.g = g;
    a.nframes = (uint32_t)n;
    a.bpi = (uint32_t)p.bpi; a.rtpf = p.row_items; a.nblk = p.nblk; a.strips = p.strips; a.window = p.window;
    a.NS = (uint32_t)p.ns; a.NOB = (uint32_t)p.nob; a.strip_off = p.strip_off; a.bring_off = p.bring_off; a.nring = (uint32_t)p.nring;
    a.box_rows = p.box_rows; a.h_magic = p.h_magic; a.pf_rows = pbox;
    const uint64_t units = (uint64_t)n * (p.row_items < p.strips ? p.row_items : p.strips);
    const uint32_t grid = units < (uint64_t)p.grid_max ? (uint32_t)(units ? units : 1) : (uint32_t)p.grid_max;
    const uint32_t block = (uint32_t)(NRW + NSW + 3) * 32u;
    if (p.X == 64)
        return decrypt ? launch_pdl(cipher_kernel<true, 64, NSW>, grid, block, p.smem, st, tm_a, tm_pad, tm_B, a)
                       : launch_pdl(cipher_kernel<false, 64, NSW>, grid, block, p.smem, st, tm_a, tm_pad, tm_B, a);
    return decrypt ? launch_pdl(cipher_kernel<true, 32, NSW>, grid, block, p.smem, st, tm_a, tm_pad, tm_B, a)
                   : launch_pdl(cipher_kernel<false, 32, NSW>, grid, block, p.smem, st, tm_a, tm_pad, tm_B, a);
}

}  // namespace vk
