/*
 * vcrypt.h -- C ABI of libvcrypt: B200-native bit-level confusion + XOR video
 * frame cipher ("Real-Time Bit-Level Encryption of Full High-Definition Video
 * Without Diffusion", arxiv 2505.07158; PAPER.md).
 *
 * The calls follow the paper's problem statement: Algorithm 1's inputs
 * (n, x0, y0, z0, w0, gamma, w, h) go to vcrypt_init, its loop
 * body is vcrypt_encrypt_frames (plaintext frames in, ciphertext frames and
 * the per-frame hash H out; the receiver is sent both), and the
 * inverse transformation is vcrypt_decrypt_frames.
 *
 * Conventions
 *   - Every function returns VCRYPT_OK (0) or a negative VCRYPT_E_* code; no
 *     exception or abort crosses this boundary.  vcrypt_strerror names a code.
 *   - The caller owns every buffer passed in or out.  "host" pointers may be
 *     pageable or pinned (pinned buffers are copied from/to directly, pageable
 *     ones are staged through the context's own pinned ring); "device"
 *     pointers are plain CUDA device addresses on the context's device (for
 *     instance torch.Tensor.data_ptr()), 16-byte aligned.
 *   - Frames are H x W x 3 uint8, tightly packed (byte offset (i*W + j)*3 + c),
 *     `n` frames back to back.  Hashes are n x 32 bytes in standard SHA-256
 *     digest order.  Shift distances D are n x 3(H+W) uint16 with
 *     D[c*(H+W) + i] = d_h(i,c) for i < H and D[c*(H+W) + H + j] = d_v(j,c);
 *     keystream bytes B are n x H x W x 3 with the index of the pixel they mask.
 *   - A context is stateful: the Lorenz hyper-chaotic main system LHCS_m is
 *     chained from frame to frame, so each successful
 *     vcrypt_encrypt_frames / vcrypt_decrypt_frames / vcrypt_derive call
 *     advances the chain by the frames it processed; a failed call leaves the
 *     chain where it was.  Encryption and decryption use separate contexts
 *     created with the same parameters, and the decryptor must see the frames
 *     in the same order from the first one.  One context per caller thread.
 *   - Results never depend on `batch`, `n_streams`, `host_threads` or on which
 *     kernel path (tiled / generic) a shape takes.
 *   - There is no CPU fallback: without a CUDA device vcrypt_init fails with
 *     VCRYPT_E_CUDA unless VCRYPT_FLAG_HOST_ONLY is set, in which case only the
 *     host-side calls (vcrypt_frame_hash, vcrypt_derive, state accessors) work
 *     and every call that needs the GPU returns VCRYPT_E_CUDA.
 */
#ifndef VCRYPT_H
#define VCRYPT_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define VCRYPT_OK 0
#define VCRYPT_E_ARG (-1)    /* null pointer, zero size, misaligned device pointer   */
#define VCRYPT_E_KEY (-2)    /* non-finite key word or gamma outside [-1.52, -0.06]  */
#define VCRYPT_E_SHAPE (-3)  /* width/height/n_workers zero or too large (3*W*H < 2^31) */
#define VCRYPT_E_CUDA (-4)   /* CUDA error, or GPU call on a host-only context       */
#define VCRYPT_E_NOMEM (-5)  /* host or device allocation failed                     */
#define VCRYPT_E_STATE (-6)  /* chaotic state left the finite range                  */
#define VCRYPT_E_LIMIT (-7)  /* n above VCRYPT_NOALLOC_MAX_FRAMES in a *_noalloc call    */

/* vcrypt_params.flags */
#define VCRYPT_FLAG_HOST_ONLY 1u      /* no CUDA: host derivation hooks only (tests on CPU boxes)  */
#define VCRYPT_FLAG_FORCE_GENERIC 2u  /* always take the any-shape gather kernels (test hook)     */
#define VCRYPT_FLAG_HOST_SCALAR 4u    /* host derivation without SHA-NI / AVX lanes (test hook)   */
#define VCRYPT_FLAG_DEVICE_DERIVE 8u  /* worker systems -> D, B on the GPU (same bytes): the host only
                                         hashes and runs the serial LHCS_m chain; D and B never cross PCIe */
#define VCRYPT_FLAG_PERSISTENT 32u    /* one persistent kernel per call (cipher.cu: row team + strip team per SM) instead of the row-pass / column-pass kernel pairs */
#define VCRYPT_FLAG_ROW_TMA 64u       /* row pass through TMA-filled shared-memory stages at every width (test / comparison hook; the default
                                         takes the register-landing row pass where the frame width allows) */
#define VCRYPT_FLAG_DEVICE_HASH 16u   /* sub-frame SHA-256 of vcrypt_encrypt_frames on the GPU, on the frames it
                                         uploads anyway, shared with the host threads band by band (device_hash_bands;
                                         same H); shapes with 3W % 16 != 0 are hashed on the host only */

typedef struct vcrypt_ctx vcrypt_ctx; /* opaque: chain state, host thread pool, streams, device and pinned buffers */

typedef struct vcrypt_params {
    double x0, y0, z0, w0;  /* the 256-bit key: initial values of LHCS_m (PAPER.md:85 Algo 1 inputs; Eq. 12 :449) */
    double gamma;           /* control parameter, -1.52 <= gamma <= -0.06                           */
    uint32_t n_workers;     /* protocol parameter n >= 1: sub-frame count and LHCS pair count;
                               NOT the number of host threads                                                      */
    uint32_t width, height; /* w, h; channels fixed at 3                                                          */
    uint32_t batch;         /* frames per kernel launch in the host-buffer pipeline (0 -> 8)                      */
    uint32_t n_streams;     /* pipeline depth: streams / staging slots (0 -> 3; 12 with VCRYPT_FLAG_DEVICE_HASH)   */
    uint32_t host_threads;  /* host threads for hashing and derivation (0 -> hardware concurrency)                */
    uint32_t flags;         /* VCRYPT_FLAG_*                                                                      */
    int32_t device;         /* CUDA device ordinal (-1 -> current device)                                         */
    uint32_t device_hash_bands; /* with VCRYPT_FLAG_DEVICE_HASH: how many of the n row bands of every frame the GPU
                               hashes (the last ones; the host threads hash the others at the same time);
                               0 or values above n -> all n.  Does not affect results                          */
    uint32_t pipe_frames;   /* vcrypt_{en,de}crypt_device on a resident clip: frames per launch pair when a call brings
                               at least 4 x pipe_frames frames; such a call alternates its launch pairs over
                               `pipe_streams` streams (the caller's + internal ones forked from and joined into it),
                               so that one pair's column pass overlaps the next pair's row pass.  0 -> from the frame
                               size (about 31 MB of frames per pair, in both directions).  Does not affect results                     */
    uint32_t pipe_streams;  /* 0 -> 2; 1 -> off (every launch on the caller's stream); at most 4                    */
    /* tuning of the persistent cipher kernel (0 -> chosen from the frame size); none of them affects results */
    uint32_t tune_row_stages;      /* input stages of the row team's shared-memory ring                            */
    uint32_t tune_row_item_blocks; /* blocks of 4 rows per row ticket                                              */
    uint32_t tune_window;          /* frames the leading pass may run ahead of the following one (0 -> 8)          */
    uint32_t tune_ring;            /* chunks of the strip team's keystream ring in shared memory (1, 2; 3: none)   */
} vcrypt_params;

/* Algorithm 1 set-up (PAPER.md:85 steps 1-2): validates the parameters, whitens the key (reading Q5 of
 * N0 = 20000 RK4 steps), starts the host threads, creates streams and buffers.  The frame chain
 * is at "first frame".  *out is written only on success. */
int vcrypt_init(vcrypt_ctx **out, const vcrypt_params *p);

/* Algorithm 1 steps 3-22 for n frames (hot-path rows a1-a11 of DESIGN.md):
 * H = xor of the sub-frame SHA-256 hashes (:45), reconstruction of the initial values with H (:55), LHCS_m ->
 * IR, worker systems -> D and B (:59), upload, bit-level confusion (Eq. 2, Eq. 3) and XOR (:75) on the GPU,
 * download.  frames, cipher_out: host, n x H x W x 3 (cipher_out may equal frames).  hashes_out: host, n x 32. */
int vcrypt_encrypt_frames(vcrypt_ctx *ctx, const uint8_t *frames, size_t n, uint8_t *cipher_out,
                          uint8_t *hashes_out);

/* The inverse transformation: the receiver holds the key and n and is sent F_e and H.
 * cipher, plain_out: host, n x H x W x 3 (may alias).  hashes: host, n x 32, as returned by the encryptor. */
int vcrypt_decrypt_frames(vcrypt_ctx *ctx, const uint8_t *cipher, const uint8_t *hashes, size_t n,
                          uint8_t *plain_out);

/* Waits for the context's GPU work, stops the host threads, frees everything.  NULL is allowed. */
void vcrypt_destroy(vcrypt_ctx *ctx);

/* Static string for a VCRYPT_* code. */
const char *vcrypt_strerror(int code);

/* Text of the last CUDA error a call on this context hit ("" if none); valid until the next failing call. */
const char *vcrypt_last_cuda_error(const vcrypt_ctx *ctx);

/* One-line description of the compiled-in constants of the method (integrator, dt, N0, K_m, u) and of the
 * host code paths available on this CPU (SHA-NI, AVX-512 / AVX2 lanes).  Static string. */
const char *vcrypt_describe(void);

/* ---- host derivation hooks (work on host-only contexts) ------------------------------------------------ */

/* H of one frame: sub-frame m = rows [floor(m*h/n), floor((m+1)*h/n)), H = xor_m SHA-256(f_m).
 * frame: host, H x W x 3.  H_out: 32 bytes.  Does not touch the chain. */
int vcrypt_frame_hash(vcrypt_ctx *ctx, const uint8_t *frame, uint8_t *H_out);

/* Algorithm 1 steps 7-14 + Algorithm 2 steps 5-10 for one frame whose hash is `hash`:
 * D_out (host, 3(H+W) uint16) and B_out (host, H x W x 3).  Advances the chain by one frame. */
int vcrypt_derive(vcrypt_ctx *ctx, const uint8_t *hash, uint16_t *D_out, uint8_t *B_out);

/* The chain state = last LHCS_m record (x_2n, y_2n, z_2n, w_2n) and the number of frames
 * derived so far: 4 doubles + 1 counter are all a caller needs to checkpoint / resume a stream. */
int vcrypt_get_state(const vcrypt_ctx *ctx, double state_out[4], uint64_t *frames_done);
int vcrypt_set_state(vcrypt_ctx *ctx, const double state[4], uint64_t frames_done); /* VCRYPT_E_STATE unless finite and |v| < 2^53 */

/* Host threads actually started (the `cores` of a CPU-side figure). */
int vcrypt_host_threads(const vcrypt_ctx *ctx);

/* ---- kernel-only path: everything already resident in device memory ------------------------------------ */

/* Algorithms 3-7 fused (rows a6-a10): for each of n frames
 *   F_e(ro,j,c) = B(ro,j,c) xor hrot(F_o)(i0,j,c),  i0 = (ro - d_v(j,c) mod h) mod h,
 * hrot = row i0 of channel c rotated by d_h(i0,c) mod 8w bit positions toward higher columns, LSB first.
 * d_frames, d_B, d_cipher: device, n x H x W x 3; d_D: device, n x 3(H+W) uint16.  d_cipher may equal
 * d_frames (in place); it must not partially overlap.  cuda_stream: a cudaStream_t (NULL = default stream).
 * Asynchronous: returns after enqueueing; launch errors are reported, execution errors surface on sync.
 * Stream order: everything the call enqueues is ordered after the work already in cuda_stream and before whatever
 * the caller enqueues there next -- also when a call on a long resident clip (n >= 4 x pipe_frames) spreads its
 * launch pairs over internal streams (vcrypt_params.pipe_frames / pipe_streams): those fork from cuda_stream at the
 * start of the call and join it at the end (legal under stream capture). */
int vcrypt_encrypt_device(vcrypt_ctx *ctx, const void *d_frames, const void *d_D, const void *d_B, size_t n,
                          void *d_cipher, void *cuda_stream);

/* Inverse of vcrypt_encrypt_device with the same D and B.  d_plain may equal d_cipher. */
int vcrypt_decrypt_device(vcrypt_ctx *ctx, const void *d_cipher, const void *d_D, const void *d_B, size_t n,
                          void *d_plain, void *cuda_stream);

/* Number of kernels the last vcrypt_encrypt_device / vcrypt_decrypt_device call on this context launched,
 * and since vcrypt_init in total (bench bookkeeping). */
int vcrypt_launch_count(const vcrypt_ctx *ctx, uint64_t *last_call, uint64_t *total);

/* Per-stage wall-clock of the last vcrypt_encrypt_frames / vcrypt_decrypt_frames call, milliseconds summed
 * over its batches: [0] hashing, [1] chain + derivation, [2] staging copies on the host, [3] waiting for the GPU.
 * (The paper's Fig. 13 phase split.) */
int vcrypt_last_stage_ms(const vcrypt_ctx *ctx, double out[4]);

/* H of n frames resident in device memory, hashed on the GPU: one thread per (frame, row band), the band
 * digests xor-ed per frame.  d_frames: device, n x H x W x 3, 16-byte aligned; hashes_out: host, n x 32.  Needs
 * 3W % 16 == 0 (VCRYPT_E_SHAPE otherwise).  Synchronises the stream before returning (test hook); does not touch the chain. */
int vcrypt_frame_hash_device(vcrypt_ctx *ctx, const void *d_frames, size_t n, uint8_t *hashes_out, void *cuda_stream);

/* Algorithm 1 steps 7-14 + Algorithm 2 steps 5-10 for one frame with the worker systems on the GPU (PAPER.md:85,
 * :88-110; same bytes as vcrypt_derive): the host reconstructs the initial values with `hash` and runs LHCS_m, the
 * device derives d_D (device, 3(H+W) uint16) and d_B (device, H x W x 3, 8-byte aligned) on `cuda_stream`.
 * Synchronises the stream before returning (test hook); VCRYPT_E_STATE if a chaotic state became non-finite.
 * Advances the chain by one frame on success. */
int vcrypt_derive_device(vcrypt_ctx *ctx, const uint8_t *hash, void *d_D, void *d_B, void *cuda_stream);

/* ---- statistical evaluation of frames resident in device memory (PAPER.md sections III-IV) ---------------- */

/* Per frame and channel c = 0..2 (index of the HWC buffer). */
typedef struct vcrypt_frame_stats {
    double hist_variance[3]; /* Eq. 4: (1/256^2) sum_i sum_j (z_i - z_j)^2 / 2 of the 256-bin histogram   */
    double chi2[3];          /* Eq. 5 (:177): sum_i (z_i - N/256)^2 / (N/256), N = W*H                                    */
    double entropy[3];       /* Eq. 10 (:345): sum_i p_i log2(1/p_i), bits                                                */
    double corr[3][3];       /* Eq. 6-9 (:283-294): correlation coefficient of ALL adjacent pairs, [channel][direction]:
                                0 horizontal (i,j)-(i,j+1), 1 vertical (i,j)-(i+1,j), 2 diagonal (i,j)-(i+1,j+1);
                                NaN when a variance is zero or there is no pair                                          */
} vcrypt_frame_stats;

/* Histogram variance, chi^2, entropy and adjacent-pixel correlation of n frames (one pass over each frame on the GPU;
 * exact integer sums on the device, the final floating-point steps on the host in binary64).
 * d_frames: device, n x H x W x 3.  stats_out: host, n entries.  hist_out: host, n x 3 x 256 uint32, or NULL. */
int vcrypt_frame_stats_device(vcrypt_ctx *ctx, const void *d_frames, size_t n, vcrypt_frame_stats *stats_out,
                              uint32_t *hist_out, void *cuda_stream);

/* NPCR (Eq. 14, 16) and UACI (Eq. 15) in percent between frames d_a[k] and d_b[k], k < n:
 * npcr_out, uaci_out: host, n x 4 doubles = {all three channels together, channel 0, 1, 2}. */
int vcrypt_npcr_uaci_device(vcrypt_ctx *ctx, const void *d_a, const void *d_b, size_t n, double *npcr_out, double *uaci_out,
                            void *cuda_stream);

/* NPCR / UACI (Eq. 14-16) for callers that cannot allocate GPU memory.  Same arguments, same
 * numbers as vcrypt_npcr_uaci_device; the difference is where the per-frame accumulators live.
 *
 * Who this is for.  vcrypt_npcr_uaci_device calls cudaMalloc / cudaFree for its accumulators on every call.  That is
 * not possible, or not acceptable, for some users of a frame cipher:
 *   - a process whose HBM has been handed out in full at start-up (an inference server or a framework memory pool that
 *     reserves the device up front): cudaMalloc simply fails there, however small the request;
 *   - a capture / encode / encrypt loop with a frame deadline: cudaMalloc and cudaFree take a driver lock and
 *     cudaFree waits for the whole device, so one call can stall every other stream for an unbounded time;
 *   - code that runs under a rule of "no allocation after initialisation" (safety-oriented or long-running services
 *     that must not fragment or fail for lack of memory days into a run).
 * Such callers use this entry point: it calls no cudaMalloc, cudaFree, cudaMallocAsync or any other allocating routine,
 * on the device or on the host heap.  The accumulators are a fixed array compiled into libvcrypt.so.
 *
 * The price, and the rules:
 *   - Capacity is fixed: n <= VCRYPT_NOALLOC_MAX_FRAMES (512) per call.  A larger n is refused with VCRYPT_E_LIMIT
 *     before anything is enqueued (vcrypt_last_cuda_error then says how many were asked for); split the clip.
 *   - The array (24 KB) occupies memory on EVERY GPU the process uses this library on, from the time the library's
 *     device code is loaded there until the process exits, also if this function is never called.
 *   - Set-up on first use: the first call on a given device looks up where that device put the array and remembers it.
 *     Make that first call during initialisation, outside any stream capture and before timing-critical work; later
 *     calls on that device only read the remembered address.
 *   - One array per device is shared by all contexts, streams and threads.  A call zeroes the part it uses (in stream
 *     order, ahead of its kernel), so leftovers of earlier calls never leak into a result.  But two calls whose GPU
 *     work may run at the same time on one device -- from two host threads, or on two streams -- race on the array
 *     and return wrong numbers without any error.  Serialise them (the call itself waits for `cuda_stream` before it
 *     returns, so calls made one after another from one thread never overlap).
 * d_a, d_b: device, n x H x W x 3; npcr_out, uaci_out: host, n x 4 doubles, laid out as in vcrypt_npcr_uaci_device. */
#define VCRYPT_NOALLOC_MAX_FRAMES 512u
int vcrypt_npcr_uaci_device_noalloc(vcrypt_ctx *ctx, const void *d_a, const void *d_b, size_t n, double *npcr_out,
                                    double *uaci_out, void *cuda_stream);

/* Local Shannon entropy (Eq. 11): mean over k square blocks (side x side pixels, top-left pixel
 * (x, y) = blocks_xy[2b], blocks_xy[2b+1], chosen by the caller: non-overlapping, inside the frame) of the entropy of
 * each block's histogram, per channel.  The paper's setting is k = 30, side = 44 (T_B = 1936).
 * out: host, n x 3 doubles.  VCRYPT_E_ARG if a block leaves the frame. */
int vcrypt_local_entropy_device(vcrypt_ctx *ctx, const void *d_frames, size_t n, const uint32_t *blocks_xy, uint32_t k,
                                uint32_t side, double *out, void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* VCRYPT_H */
