// kernels.cuh -- launch interface of the sm_100a frame-cipher kernels (kernels.cu).
// Internal to libvcrypt; the public boundary is include/vcrypt.h.
#pragma once
#include <cuda_runtime.h>
#include <stddef.h>
#include <stdint.h>

namespace vk {

struct Geom {
    uint32_t w, h;         // pixels
    uint32_t row_bytes;    // 3w
    uint32_t nD;           // 3(h+w) shift distances per frame
    size_t frame_bytes;    // 3wh
};

inline Geom make_geom(uint32_t w, uint32_t h) {
    Geom g;
    g.w = w; g.h = h; g.row_bytes = 3u * w; g.nD = 3u * (h + w);
    g.frame_bytes = (size_t)3u * w * h;
    return g;
}

// Plan chosen once per context from (w, h) and the device's shared-memory size.
struct Plan {
    bool tiled;            // tiled two-pass path usable (w % 16 == 0, h % 4 == 0, h >= 16, strip and row block fit in shared memory)
    int strip_bytes;       // X: byte columns per strip (64, or 32 for very tall frames)
    int strips_per_frame;  // ceil(3w / X)
    int row_nc;            // row pass: compute threads per CTA (+ 32 for the copy warp)
    int row_ns;            // row pass: stages of the shared-memory ring
    bool row_big;          // row pass: one CTA of up to 1024 threads per SM (wide frames)
    int row_grid_max;      // row pass: persistent CTAs (resident CTAs per SM x SMs)
    int row_nc_dec, row_ns_dec, row_grid_max_dec;  // the same for the inverse row pass (decrypt): three small CTAs per SM where they fit
    size_t smem_row_dec;
    int row_reg;           // register-landing row pass (row_reg_kernel): 0 = not used, 1 = 256-thread CTAs (w <= 1024), 2 = 512-thread
                           // CTAs (w <= 2048), 3 = 512-thread CTAs with two items per thread (w <= 4096)
    bool row_reg_dec;      // ... also for the inverse row pass (every width except 1537 - 2048 pixels: measured, see make_plan)
    int row_reg_grid_max;  // its persistent CTAs
    size_t smem_row_reg;
    uint32_t box_rows;     // column pass: rows per TMA tensor tile (largest divisor of h that is <= 256)
    uint32_t h_magic;      // ceil(2^32 / h): d mod h without a division for d < 2^16
    void *encode_tiled;    // cuTensorMapEncodeTiled, resolved through the runtime (no link-time libcuda dependency)
    int col_ctas_per_sm;   // column pass variant (3: 256-thread CTAs, two or three per SM; 1: one 512-thread CTA per SM)
    size_t smem_row;       // dynamic shared memory of the row pass
    size_t smem_cole;      // dynamic shared memory of the column pass, decrypt direction (the strip)
    size_t smem_cole_enc;  // ... encrypt direction: the strip, or more when that is how two CTAs per SM are asked for
    size_t max_frames_per_launch;  // keeps the intermediate (n * 3wh bytes) L2-resident
};

// row_tma: keep the TMA-staged row pass for every width (test / comparison hook)
cudaError_t make_plan(const Geom &g, int device, bool row_tma, Plan *out);

// Encrypt n frames: row pass (horizontal bit rotation, Eq. 2) then column pass
// (vertical shift, Eq. 3, fused with the XOR of Algorithm 6).  dst may equal src.
// Returns the number of kernels launched through *launches.
cudaError_t encrypt_tiled(const Geom &g, const Plan &p, const uint8_t *src, const uint16_t *D, const uint8_t *B,
                          size_t n, uint8_t *dst, cudaStream_t st, int *launches);
cudaError_t decrypt_tiled(const Geom &g, const Plan &p, const uint8_t *src, const uint16_t *D, const uint8_t *B,
                          size_t n, uint8_t *dst, cudaStream_t st, int *launches);

// ---------------------------------------------------------------------------------------------
// The persistent cipher kernel (cipher.cu): row items and strip items of one call taken by ticket from one launch.
// ---------------------------------------------------------------------------------------------
struct UniTune {               // 0 = chosen from the shape; none of them affects results
    uint32_t row_stages;       // input stages of the row ring
    uint32_t row_item_blocks;  // blocks of 4 rows per row ticket
    uint32_t window;           // frames the leading pass may be ahead of the following one
    uint32_t ring;             // chunks of the strip team's keystream ring (1, 2; 3: none)
};

struct UniPlan {
    bool ok;               // shape takes the tiled path (w % 16 == 0, w >= 64, h % 4 == 0, h >= 16, a strip and a row ring fit in shared memory)
    int X;                 // byte columns per strip (64, or 32 for very tall frames)
    int ns, nob;           // row team: input stages, output buffers
    int bpi;               // row team: blocks per ticket
    int grid_max;          // resident CTAs (one per SM)
    int nring;             // strip team: chunks of the keystream ring
    uint32_t strip_off;    // byte offset of the strip in the dynamic shared memory
    uint32_t bring_off;    // ... of the keystream ring
    size_t smem;           // dynamic shared memory per CTA
    uint32_t nblk;         // blocks of 4 rows per frame
    uint32_t row_items;    // row tickets per frame
    uint32_t strips;       // per frame
    uint32_t window;
    uint32_t box_rows;     // rows per TMA tensor tile of a strip (largest divisor of h that is <= 256)
    uint32_t h_magic;      // ceil(2^32 / h): d mod h without a division for d < 2^16
    void *encode_tiled;    // cuTensorMapEncodeTiled, resolved through the runtime (no link-time libcuda dependency)
};

cudaError_t make_uni_plan(const Geom &g, int device, const UniTune &tune, UniPlan *out);

// Words of launch state cipher_launch needs for n frames (zero before the first use; the kernel leaves it zero).
inline size_t cipher_sched_words(size_t n) { return 4 + 2 * n; }

// Encrypt (row items lead, strip items follow) or decrypt (strip items lead) n frames with ONE launch on `st`.
// dst may equal src.  `sched`: device, cipher_sched_words(n) zeroed words, not shared with a launch that may run concurrently.
cudaError_t cipher_launch(const Geom &g, const UniPlan &p, bool decrypt, const uint8_t *src, const uint16_t *D, const uint8_t *B,
                          size_t n, uint8_t *dst, uint32_t *sched, cudaStream_t st);

// Any-shape path: one thread per output byte, closed-form gather straight from global memory.
// dst must not alias src.
cudaError_t encrypt_generic(const Geom &g, const uint8_t *src, const uint16_t *D, const uint8_t *B, size_t n,
                            uint8_t *dst, cudaStream_t st, int *launches);
cudaError_t decrypt_generic(const Geom &g, const uint8_t *src, const uint16_t *D, const uint8_t *B, size_t n,
                            uint8_t *dst, cudaStream_t st, int *launches);

// Device-side worker systems (derive.cu): D and B of m frames from their LHCS_m records IR (m x 2n x 4 doubles, device),
// written straight into device buffers.  *d_status gets bit 0 set if a chaotic state became non-finite.
cudaError_t derive_device(const Geom &g, const double *d_IR, double gamma, uint32_t n, size_t m, uint16_t *d_D, uint8_t *d_B,
                          uint32_t *d_status, cudaStream_t st);

// Device-side sub-frame hashing (sha256.cu): xor of the SHA-256 digests of row bands band0 .. n-1 of each of m frames
// into d_H (m x 32 bytes, digest byte order).  Needs 16-byte aligned frames and row_bytes % 16 == 0 (cudaErrorInvalidValue otherwise).
cudaError_t hash_device(const Geom &g, const uint8_t *d_frames, uint32_t n, uint32_t band0, size_t m, uint32_t *d_H,
                        cudaStream_t st);

// Statistical evaluation (stats.cu): exact integer sufficient statistics of frames in device memory.
//   stats_device     : d_hist n x 3 x 256 u32 (per channel histogram), d_pairs n x 3 x 3 x 5 u64 (per channel and direction
//                      H, V, D: sum x, sum y, sum xy, sum x^2, sum y^2 over all adjacent pairs)
//   diff_device      : d_out n x 3 x 2 u64 (per channel: differing bytes, sum |a - b|)
//   block_hist_device: d_bh n x k x 3 x 256 u32 (per block and channel histogram; d_xy k x 2 top-left corners, device)
cudaError_t stats_device(const Geom &g, const uint8_t *d_frames, size_t n, uint32_t *d_hist, unsigned long long *d_pairs,
                         cudaStream_t st);
cudaError_t diff_device(const Geom &g, const uint8_t *d_a, const uint8_t *d_b, size_t n, unsigned long long *d_out, cudaStream_t st);
cudaError_t block_hist_device(const Geom &g, const uint8_t *d_frames, size_t n, const uint32_t *d_xy, uint32_t k, uint32_t side,
                              uint32_t *d_bh, cudaStream_t st);
//   diff_device_static: diff_device with its accumulators in a static device array of the library (no allocation anywhere on
//                      the path); results land in h_out (HOST, n x 3 x 2 u64) and the stream has been waited for on return.
//                      At most kDiffStaticMaxFrames frames per call; calls that overlap on one GPU race (see stats.cu).
constexpr size_t kDiffStaticMaxFrames = 512;  // 512 x 6 x 8 bytes = 24 KB of every GPU that loads the library
cudaError_t diff_device_static(const Geom &g, const uint8_t *d_a, const uint8_t *d_b, size_t n, unsigned long long *h_out,
                               cudaStream_t st);

}  // namespace vk
