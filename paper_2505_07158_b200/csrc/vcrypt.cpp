// vcrypt.cpp -- the C ABI of include/vcrypt.h: context, host derivation driver, multi-stream pipeline.
//
// Algorithm 1 re-shaped for one B200: the main-thread loop over frames becomes a loop over
// batches; the worker threads T_w of Algorithm 2 become jobs on a fixed thread pool (the protocol parameter n
// fixes how the work is split, not how many threads run it); upload / GPU steps / download of a batch run on
// one of `n_streams` CUDA streams while the host derives the next batch.
#include <cuda_runtime.h>

#include <atomic>
#include <chrono>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <memory>
#include <new>
#include <thread>
#include <vector>

#pragma GCC visibility push(default)
#include "../../include/vcrypt.h"
#pragma GCC visibility pop
#include "host.hpp"
#include "kernels.cuh"
#include "thread_pool.hpp"

namespace {

using clk = std::chrono::steady_clock;
inline double ms_since(clk::time_point t0) { return std::chrono::duration<double, std::milli>(clk::now() - t0).count(); }

struct Slot {
    cudaStream_t st = nullptr;
    cudaEvent_t done = nullptr;
    // pinned staging (h_F / h_out only when the caller's buffers are pageable)
    uint8_t *h_F = nullptr, *h_B = nullptr, *h_out = nullptr;
    uint16_t *h_D = nullptr;
    // device
    uint8_t *d_F = nullptr, *d_B = nullptr, *d_out = nullptr;  // d_out only on the any-shape kernel path
    uint16_t *d_D = nullptr;
    // device-side derivation (VCRYPT_FLAG_DEVICE_DERIVE): LHCS_m records up, status word down
    double *h_IR = nullptr, *d_IR = nullptr;
    uint32_t *h_status = nullptr, *d_status = nullptr;
    bool status_pending = false;
    // device-side hashing (VCRYPT_FLAG_DEVICE_HASH): H of the batch's frames, and the event that says they are on the host
    uint32_t *d_H = nullptr;
    uint8_t *h_H = nullptr;
    cudaEvent_t hashed = nullptr;
    // work in flight
    bool busy = false;
    uint8_t *user_out = nullptr;  // where h_out goes once `done` fires (nullptr: D2H went straight to the caller)
    size_t out_bytes = 0;
};

}  // namespace

struct vcrypt_ctx {
    vcrypt_params p{};
    vk::Geom g{};
    vk::Plan plan{};
    bool cuda = false;
    int device = -1;
    bool simd = true;
    int isa = 0;
    double S[4] = {0, 0, 0, 0};
    uint64_t frames_done = 0;
    std::unique_ptr<vh::ThreadPool> pool;
    size_t batch = 8;
    std::vector<Slot> slots;
    // per-batch host scratch
    std::vector<double> IR;               // batch x 2n x 4
    std::vector<vh::WorkerSlice> slices;  // batch x n
    std::vector<uint8_t> subhash;         // batch x n x 32
    // resident-clip schedule of the *_device calls (launch pairs alternating over streams): see launch_cipher
    static constexpr int kPipeMax = 4;
    size_t pipe_frames[2] = {0, 0};  // encrypt, decrypt
    int pipe_streams = 2;
    cudaStream_t pipe_st[kPipeMax - 1] = {nullptr, nullptr, nullptr};
    cudaEvent_t pipe_fork = nullptr, pipe_join[kPipeMax - 1] = {nullptr, nullptr, nullptr};
    // persistent cipher kernel (cipher.cu): plan + launch state, one buffer per stream that calls on this context arrive on
    vk::UniPlan uni{};
    static constexpr int kSchedSlots = 32;
    static constexpr size_t kSchedFrames = 4096;  // frames per launch at most (longer calls are cut)
    uint32_t *d_sched = nullptr;                  // kSchedSlots x cipher_sched_words(kSchedFrames), zero between launches
    cudaStream_t sched_owner[kSchedSlots] = {};
    int sched_n = 0;
    // bookkeeping
    uint64_t launches_last = 0, launches_total = 0;
    double stage_ms[4] = {0, 0, 0, 0};
    char cuda_msg[256] = {0};
};

namespace {

int cuda_fail(vcrypt_ctx *c, cudaError_t e, const char *what) {
    if (c) std::snprintf(c->cuda_msg, sizeof c->cuda_msg, "%s: %s", what, cudaGetErrorString(e));
    return VCRYPT_E_CUDA;
}
#define VC_CUDA(ctx, call)                                           \
    do {                                                             \
        cudaError_t e__ = (call);                                    \
        if (e__ != cudaSuccess) return cuda_fail((ctx), e__, #call); \
    } while (0)

// No exception may cross the C ABI (include/vcrypt.h): host allocations inside an entry point become VCRYPT_E_NOMEM.
template <class F>
int guarded(F &&body) noexcept {
    try {
        return body();
    } catch (const std::bad_alloc &) {
        return VCRYPT_E_NOMEM;
    } catch (...) {
        return VCRYPT_E_ARG;
    }
}

// Makes the context's device current for the duration of an entry point and puts the caller's device back afterwards.
struct DeviceScope {
    int prev = -1;
    cudaError_t err = cudaSuccess;
    explicit DeviceScope(int dev) {
        err = cudaGetDevice(&prev);
        if (err == cudaSuccess && prev != dev) err = cudaSetDevice(dev);
        else if (err == cudaSuccess) prev = -1;  // nothing to restore
    }
    ~DeviceScope() {
        if (prev >= 0) cudaSetDevice(prev);
    }
    DeviceScope(const DeviceScope &) = delete;
    DeviceScope &operator=(const DeviceScope &) = delete;
};
#define VC_DEVICE(ctx)                            \
    DeviceScope dev_scope__((ctx)->device);       \
    if (dev_scope__.err != cudaSuccess) return cuda_fail((ctx), dev_scope__.err, "cudaSetDevice")

bool is_pinned(const void *p) {
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    return a.type == cudaMemoryTypeHost;
}

void free_slot(Slot &s) {
    if (s.st) cudaStreamSynchronize(s.st);
    if (s.h_F) cudaFreeHost(s.h_F);
    if (s.h_B) cudaFreeHost(s.h_B);
    if (s.h_out) cudaFreeHost(s.h_out);
    if (s.h_D) cudaFreeHost(s.h_D);
    if (s.d_F) cudaFree(s.d_F);
    if (s.d_B) cudaFree(s.d_B);
    if (s.d_out) cudaFree(s.d_out);
    if (s.d_D) cudaFree(s.d_D);
    if (s.h_IR) cudaFreeHost(s.h_IR);
    if (s.d_IR) cudaFree(s.d_IR);
    if (s.d_H) cudaFree(s.d_H);
    if (s.h_H) cudaFreeHost(s.h_H);
    if (s.hashed) cudaEventDestroy(s.hashed);
    if (s.h_status) cudaFreeHost(s.h_status);
    if (s.d_status) cudaFree(s.d_status);
    if (s.done) cudaEventDestroy(s.done);
    if (s.st) cudaStreamDestroy(s.st);
    s = Slot{};
}

// Device + pinned buffers of one slot, allocated on first use so that contexts used only through the
// *_device calls or the host hooks stay cheap.
int ensure_slot(vcrypt_ctx *c, Slot &s, bool need_hF, bool need_hout) {
    const size_t fb = c->g.frame_bytes * c->batch, db = (size_t)c->g.nD * c->batch * sizeof(uint16_t);
    if (!s.st) VC_CUDA(c, cudaStreamCreateWithFlags(&s.st, cudaStreamNonBlocking));
    if (!s.done) VC_CUDA(c, cudaEventCreateWithFlags(&s.done, cudaEventDisableTiming));
    if (!s.d_F) VC_CUDA(c, cudaMalloc(&s.d_F, fb));
    if (!s.d_B) VC_CUDA(c, cudaMalloc(&s.d_B, fb));
    const bool generic = !c->plan.tiled || (c->p.flags & VCRYPT_FLAG_FORCE_GENERIC);
    if (generic && !s.d_out) VC_CUDA(c, cudaMalloc(&s.d_out, fb));
    if (!s.d_D) VC_CUDA(c, cudaMalloc(&s.d_D, db));
    if (c->p.flags & VCRYPT_FLAG_DEVICE_HASH) {
        if (!s.d_H) VC_CUDA(c, cudaMalloc(&s.d_H, c->batch * 32u));
        if (!s.h_H) VC_CUDA(c, cudaHostAlloc(&s.h_H, c->batch * 32u, cudaHostAllocDefault));
        if (!s.hashed) VC_CUDA(c, cudaEventCreateWithFlags(&s.hashed, cudaEventDisableTiming));
    }
    if (c->p.flags & VCRYPT_FLAG_DEVICE_DERIVE) {
        const size_t irb = c->batch * 2u * (size_t)c->p.n_workers * 4u * sizeof(double);
        if (!s.h_IR) VC_CUDA(c, cudaHostAlloc(&s.h_IR, irb, cudaHostAllocDefault));
        if (!s.d_IR) VC_CUDA(c, cudaMalloc(&s.d_IR, irb));
        if (!s.h_status) VC_CUDA(c, cudaHostAlloc(&s.h_status, sizeof(uint32_t), cudaHostAllocDefault));
        if (!s.d_status) VC_CUDA(c, cudaMalloc(&s.d_status, sizeof(uint32_t)));
    } else {
        if (!s.h_B) VC_CUDA(c, cudaHostAlloc(&s.h_B, fb, cudaHostAllocDefault));
        if (!s.h_D) VC_CUDA(c, cudaHostAlloc(&s.h_D, db, cudaHostAllocDefault));
    }
    if (need_hF && !s.h_F) VC_CUDA(c, cudaHostAlloc(&s.h_F, fb, cudaHostAllocDefault));
    if (need_hout && !s.h_out) VC_CUDA(c, cudaHostAlloc(&s.h_out, fb, cudaHostAllocDefault));
    return VCRYPT_OK;
}

// Waits for a slot's GPU work and hands staged output to the caller.
int retire_slot(vcrypt_ctx *c, Slot &s) {
    if (!s.busy) return VCRYPT_OK;
    const auto t0 = clk::now();
    VC_CUDA(c, cudaEventSynchronize(s.done));
    c->stage_ms[3] += ms_since(t0);
    s.busy = false;
    if (s.status_pending) {
        s.status_pending = false;
        if (*s.h_status) return VCRYPT_E_STATE;  // a worker system left the finite range (Q17)
    }
    if (s.user_out) {
        const auto t1 = clk::now();
        const size_t chunk = (size_t)1 << 20, nch = (s.out_bytes + chunk - 1) / chunk;
        uint8_t *dst = s.user_out;
        const uint8_t *src = s.h_out;
        const size_t total = s.out_bytes;
        c->pool->parallel_for(nch, [&](size_t i) {
            const size_t o = i * chunk, len = total - o < chunk ? total - o : chunk;
            std::memcpy(dst + o, src + o, len);
        });
        c->stage_ms[2] += ms_since(t1);
        s.user_out = nullptr;
    }
    return VCRYPT_OK;
}

// Launch state of the persistent cipher kernel for work enqueued on `st`: launches on one stream follow each other (the
// kernel waits for its predecessor before it touches the state and leaves it zeroed), so one buffer per stream is enough.
int sched_for_stream(vcrypt_ctx *c, cudaStream_t st, uint32_t **out) {
    const size_t words = vk::cipher_sched_words(vcrypt_ctx::kSchedFrames);
    if (!c->d_sched) {
        // One-time zeroing.  cudaMemset of device memory is asynchronous to the host and runs on the legacy default stream, which
        // does not order it before work on a non-blocking stream (the library's own slot streams, torch's, cupy's): the first
        // launch on `st` could read the ticket and the per-frame counters before they are zero.  So the host waits for it here.
        uint32_t *buf = nullptr;
        VC_CUDA(c, cudaMalloc(&buf, vcrypt_ctx::kSchedSlots * words * sizeof(uint32_t)));
        cudaError_t e = cudaMemset(buf, 0, vcrypt_ctx::kSchedSlots * words * sizeof(uint32_t));
        if (e == cudaSuccess) e = cudaStreamSynchronize(cudaStreamLegacy);
        if (e != cudaSuccess) {  // not kept: a buffer that is allocated but not known to be zero must never be handed out
            cudaFree(buf);
            return cuda_fail(c, e, "zeroing the persistent kernel's launch state");
        }
        c->d_sched = buf;
    }
    for (int i = 0; i < c->sched_n; ++i)
        if (c->sched_owner[i] == st) { *out = c->d_sched + (size_t)i * words; return VCRYPT_OK; }
    if (c->sched_n == vcrypt_ctx::kSchedSlots) {  // more streams than buffers: wait for everything, start over
        VC_CUDA(c, cudaDeviceSynchronize());
        c->sched_n = 0;
    }
    c->sched_owner[c->sched_n] = st;
    *out = c->d_sched + (size_t)c->sched_n * words;
    c->sched_n += 1;
    return VCRYPT_OK;
}

int launch_cipher(vcrypt_ctx *c, bool decrypt, const uint8_t *src, const uint16_t *D, const uint8_t *B, size_t n,
                  uint8_t *dst, cudaStream_t st) {
    int launches = 0;
    cudaError_t e;
    const bool aligned = ((((uintptr_t)src) | ((uintptr_t)dst) | ((uintptr_t)B)) & 15u) == 0;
    if (c->uni.ok && aligned && (c->p.flags & VCRYPT_FLAG_PERSISTENT) && !(c->p.flags & VCRYPT_FLAG_FORCE_GENERIC)) {
        // one persistent kernel per call (per kSchedFrames frames): row items and strip items taken by ticket (cipher.cu)
        uint32_t *sched = nullptr;
        const int rs = sched_for_stream(c, st, &sched);
        if (rs != VCRYPT_OK) return rs;
        e = cudaSuccess;
        for (size_t f0 = 0; f0 < n && e == cudaSuccess; f0 += vcrypt_ctx::kSchedFrames) {
            const size_t m = n - f0 < vcrypt_ctx::kSchedFrames ? n - f0 : vcrypt_ctx::kSchedFrames, off = f0 * c->g.frame_bytes;
            e = vk::cipher_launch(c->g, c->uni, decrypt, src + off, D + f0 * c->g.nD, B + off, m, dst + off, sched, st);
            if (e == cudaSuccess) ++launches;
        }
    } else if (c->plan.tiled && aligned && !(c->p.flags & VCRYPT_FLAG_FORCE_GENERIC)) {
        const size_t pf = c->pipe_frames[decrypt ? 1 : 0];
        if (c->pipe_streams >= 2 && n >= 4 * pf) {  // fewer pairs never reach a steady state: the fork / join costs more than it hides
            // Resident clip.  The two passes of a launch pair stress different parts of the memory system (the row pass
            // reads DRAM and fills L2, the column pass's CTAs first pull their strips out of L2 and then stream DRAM), and
            // inside one stream a pass only starts when its predecessor has drained.  Frames are independent, so the
            // pairs go round-robin over `pipe_streams` streams -- the caller's and internal ones that fork from it here
            // and join it below: the column pass of one pair overlaps the row pass of the next.  Pairs are kept small
            // enough for the intermediates of all streams to stay in L2 together (measured).
            const int S = c->pipe_streams;
            e = cudaSuccess;
            for (int i = 0; i + 1 < S && e == cudaSuccess; ++i) {
                if (!c->pipe_st[i]) e = cudaStreamCreateWithFlags(&c->pipe_st[i], cudaStreamNonBlocking);
                if (e == cudaSuccess && !c->pipe_join[i]) e = cudaEventCreateWithFlags(&c->pipe_join[i], cudaEventDisableTiming);
            }
            if (e == cudaSuccess && !c->pipe_fork) e = cudaEventCreateWithFlags(&c->pipe_fork, cudaEventDisableTiming);
            if (e == cudaSuccess) e = cudaEventRecord(c->pipe_fork, st);
            for (int i = 0; i + 1 < S && e == cudaSuccess; ++i) e = cudaStreamWaitEvent(c->pipe_st[i], c->pipe_fork, 0);
            if (e == cudaSuccess) {
                const size_t npairs = (n + pf - 1) / pf, base = n / npairs, extra = n % npairs;  // balanced pairs
                size_t f0 = 0;
                cudaError_t el = cudaSuccess;
                for (size_t k = 0; k < npairs && el == cudaSuccess; ++k) {
                    const size_t m = base + (k < extra ? 1 : 0), off = f0 * c->g.frame_bytes;
                    cudaStream_t sk = (k % S == 0) ? st : c->pipe_st[k % S - 1];
                    el = decrypt ? vk::decrypt_tiled(c->g, c->plan, src + off, D + f0 * c->g.nD, B + off, m, dst + off, sk, &launches)
                                 : vk::encrypt_tiled(c->g, c->plan, src + off, D + f0 * c->g.nD, B + off, m, dst + off, sk, &launches);
                    f0 += m;
                }
                // join even after a failed launch: whatever was enqueued on the internal streams stays ordered before the
                // caller's next operation
                for (int i = 0; i + 1 < S; ++i) {
                    cudaError_t ej = cudaEventRecord(c->pipe_join[i], c->pipe_st[i]);
                    if (ej == cudaSuccess) ej = cudaStreamWaitEvent(st, c->pipe_join[i], 0);
                    if (e == cudaSuccess) e = ej;
                }
                if (el != cudaSuccess) e = el;
            }
        } else {
            e = decrypt ? vk::decrypt_tiled(c->g, c->plan, src, D, B, n, dst, st, &launches)
                        : vk::encrypt_tiled(c->g, c->plan, src, D, B, n, dst, st, &launches);
        }
    } else {
        uint8_t *out = dst;
        const size_t bytes = n * c->g.frame_bytes;
        bool scratch = false;
        if (dst == src) {  // the gather kernels cannot run in place: through a scratch buffer of this call, allocated and freed in
                           // stream order (calls on other streams have their own)
            void *tmp = nullptr;
            VC_CUDA(c, cudaMallocAsync(&tmp, bytes, st));
            out = static_cast<uint8_t *>(tmp);
            scratch = true;
        }
        e = decrypt ? vk::decrypt_generic(c->g, src, D, B, n, out, st, &launches)
                    : vk::encrypt_generic(c->g, src, D, B, n, out, st, &launches);
        if (e == cudaSuccess && out != dst) e = cudaMemcpyAsync(dst, out, bytes, cudaMemcpyDeviceToDevice, st);
        if (scratch) {
            const cudaError_t ef = cudaFreeAsync(out, st);
            if (e == cudaSuccess) e = ef;
        }
    }
    c->launches_last += (uint64_t)launches;
    c->launches_total += (uint64_t)launches;
    if (e != cudaSuccess) return cuda_fail(c, e, decrypt ? "decrypt launch" : "encrypt launch");
    return VCRYPT_OK;
}

}  // namespace

// =====================================================================================================
// context life cycle
// =====================================================================================================
extern "C" int vcrypt_init(vcrypt_ctx **out, const vcrypt_params *p) {
    if (!out || !p) return VCRYPT_E_ARG;
    if (!std::isfinite(p->x0) || !std::isfinite(p->y0) || !std::isfinite(p->z0) || !std::isfinite(p->w0)) return VCRYPT_E_KEY;
    const double lim = 9007199254740992.0;  // 2^53: integer parts stay exact
    if (std::fabs(p->x0) >= lim || std::fabs(p->y0) >= lim || std::fabs(p->z0) >= lim || std::fabs(p->w0) >= lim) return VCRYPT_E_KEY;
    if (!(p->gamma >= -1.52 && p->gamma <= -0.06)) return VCRYPT_E_KEY;
    if (p->n_workers == 0 || p->width == 0 || p->height == 0) return VCRYPT_E_SHAPE;
    if (p->n_workers > (1u << 20) || p->width > (1u << 16) || p->height > (1u << 16)) return VCRYPT_E_SHAPE;
    if ((uint64_t)3 * p->width * p->height >= ((uint64_t)1 << 31)) return VCRYPT_E_SHAPE;  // 32-bit byte offsets inside a frame
    vcrypt_ctx *c = new (std::nothrow) vcrypt_ctx;
    if (!c) return VCRYPT_E_NOMEM;
    int rc = VCRYPT_OK;
    try {
        c->p = *p;
        c->g = vk::make_geom(p->width, p->height);
        c->batch = p->batch ? p->batch : 8;
        c->pipe_streams = p->pipe_streams == 0 ? 2 : (int)(p->pipe_streams > (uint32_t)vcrypt_ctx::kPipeMax ? vcrypt_ctx::kPipeMax : p->pipe_streams);
        {
            // bytes of frames per launch pair, to the nearest frame.  Measured on B200 with two streams (us per frame, 300-frame
            // FHD clip, pairs of 4 / 5 / 6): encrypt 4.77 / 4.70 / 4.79, decrypt 5.65 / 5.68 / 5.56; 640x480 best at 30-40 frames,
            // 4K at 1: two pairs in flight keep their intermediates in L2
            const size_t target[2] = {(size_t)31 << 20, (size_t)31 << 20};  // encrypt, decrypt (decrypt with three small row-pass CTAs per SM: pairs of 4 / 5 / 6 / 7 FHD frames 5.22 / 5.14 / 5.31 / 5.42 us per frame)
            for (int d = 0; d < 2; ++d) {
                const size_t pf = p->pipe_frames ? p->pipe_frames : (target[d] + c->g.frame_bytes / 2) / c->g.frame_bytes;
                c->pipe_frames[d] = pf < 1 ? 1 : pf;
            }
        }
        c->simd = !(p->flags & VCRYPT_FLAG_HOST_SCALAR);
        c->isa = c->simd ? vh::best_isa() : 0;
        unsigned nt = p->host_threads ? p->host_threads : std::thread::hardware_concurrency();
        if (nt < 1) nt = 1;
        if (nt > 256) nt = 256;
        c->pool.reset(new vh::ThreadPool(nt));
        // reading Q5: one-off key whitening
        c->S[0] = p->x0; c->S[1] = p->y0; c->S[2] = p->z0; c->S[3] = p->w0;
        for (int k = 0; k < vh::kWhiten; ++k) vh::rk4_step(c->S, p->gamma);
        if (!vh::finite4(c->S)) rc = VCRYPT_E_STATE;
        c->IR.resize(c->batch * 2u * p->n_workers * 4u);
        c->slices.resize(c->batch * (size_t)p->n_workers);
        c->subhash.resize(c->batch * (size_t)p->n_workers * 32u);
        if (rc == VCRYPT_OK && !(p->flags & VCRYPT_FLAG_HOST_ONLY)) {
            int dev = p->device, prev_dev = -1;
            cudaError_t e = cudaGetDevice(&prev_dev);
            if (e == cudaSuccess && dev < 0) dev = prev_dev;
            if (e == cudaSuccess) e = cudaSetDevice(dev);
            if (e == cudaSuccess) e = vk::make_plan(c->g, dev, (p->flags & VCRYPT_FLAG_ROW_TMA) != 0, &c->plan);
            if (e == cudaSuccess) {
                vk::UniTune tune{p->tune_row_stages, p->tune_row_item_blocks, p->tune_window, p->tune_ring};
                e = vk::make_uni_plan(c->g, dev, tune, &c->uni);
            }
            if (e != cudaSuccess) {
                cudaGetLastError();
                rc = VCRYPT_E_CUDA;
            } else {
                c->cuda = true;
                c->device = dev;
                c->slots.resize(p->n_streams ? p->n_streams : ((p->flags & VCRYPT_FLAG_DEVICE_HASH) ? 12 : 3));  // device hashing wants a deep pipeline (6 ms per band)
            }
            if (prev_dev >= 0 && prev_dev != dev) cudaSetDevice(prev_dev);  // the caller's current device is left as it was
        }
    } catch (const std::bad_alloc &) {
        rc = VCRYPT_E_NOMEM;
    } catch (...) {
        rc = VCRYPT_E_ARG;
    }
    if (rc != VCRYPT_OK) {
        delete c;
        return rc;
    }
    *out = c;
    return VCRYPT_OK;
}

extern "C" void vcrypt_destroy(vcrypt_ctx *c) {
    if (!c) return;
    if (c->cuda) {
        DeviceScope scope(c->device);
        for (Slot &s : c->slots) free_slot(s);
        for (int i = 0; i + 1 < vcrypt_ctx::kPipeMax; ++i) {
            if (c->pipe_st[i]) { cudaStreamSynchronize(c->pipe_st[i]); cudaStreamDestroy(c->pipe_st[i]); }
            if (c->pipe_join[i]) cudaEventDestroy(c->pipe_join[i]);
        }
        if (c->pipe_fork) cudaEventDestroy(c->pipe_fork);
        if (c->d_sched) {
            cudaDeviceSynchronize();
            cudaFree(c->d_sched);
        }
    }
    delete c;
}

extern "C" const char *vcrypt_strerror(int code) {
    switch (code) {
        case VCRYPT_OK: return "ok";
        case VCRYPT_E_ARG: return "invalid argument (null pointer, zero size or misaligned device pointer)";
        case VCRYPT_E_KEY: return "invalid key (non-finite word, or gamma outside [-1.52, -0.06])";
        case VCRYPT_E_SHAPE: return "invalid shape (width, height or n_workers zero or too large)";
        case VCRYPT_E_CUDA: return "CUDA error, or GPU call on a host-only context";
        case VCRYPT_E_NOMEM: return "out of memory";
        case VCRYPT_E_STATE: return "chaotic state left the finite range";
        case VCRYPT_E_LIMIT: return "more frames than the fixed scratch of a no-allocation call holds (VCRYPT_NOALLOC_MAX_FRAMES)";
        default: return "unknown vcrypt error code";
    }
}

extern "C" const char *vcrypt_describe(void) {
    static char buf[512];
    static bool done = false;
    if (!done) {
        std::snprintf(buf, sizeof buf,
                      "vcrypt: LHCS sigma=10 rho=28 beta=8/3, RK4 dt=%.3f, whitening N0=%d steps, IR record stride K_m=%d, "
                      "bound u=%llu, 6 mantissa bytes per variable; host: sha_ni=%d lanes_isa=%d (0 scalar, 1 avx2x4, 2 avx512x8); "
                      "device: sm_100a row pass (register-landing, or TMA-staged warp-specialised) + TMA-tensor T4 column pass (PDL-chained), any-shape gather",
                      vh::kDt, vh::kWhiten, vh::kRecordStride, (unsigned long long)vh::kBound, (int)vh::cpu_has_shani(),
                      vh::best_isa());
        done = true;
    }
    return buf;
}

extern "C" const char *vcrypt_last_cuda_error(const vcrypt_ctx *c) { return c ? c->cuda_msg : ""; }

extern "C" int vcrypt_get_state(const vcrypt_ctx *c, double state_out[4], uint64_t *frames_done) {
    if (!c || !state_out) return VCRYPT_E_ARG;
    std::memcpy(state_out, c->S, sizeof c->S);
    if (frames_done) *frames_done = c->frames_done;
    return VCRYPT_OK;
}

extern "C" int vcrypt_set_state(vcrypt_ctx *c, const double state[4], uint64_t frames_done) {
    if (!c || !state) return VCRYPT_E_ARG;
    if (!vh::finite4(state)) return VCRYPT_E_STATE;
    for (int k = 0; k < 4; ++k)
        if (std::fabs(state[k]) >= 9007199254740992.0) return VCRYPT_E_STATE;  // 2^53, as for the key: integer parts stay exact
    std::memcpy(c->S, state, sizeof c->S);
    c->frames_done = frames_done;
    return VCRYPT_OK;
}

extern "C" int vcrypt_host_threads(const vcrypt_ctx *c) { return c ? (int)c->pool->size() : VCRYPT_E_ARG; }

extern "C" int vcrypt_launch_count(const vcrypt_ctx *c, uint64_t *last_call, uint64_t *total) {
    if (!c) return VCRYPT_E_ARG;
    if (last_call) *last_call = c->launches_last;
    if (total) *total = c->launches_total;
    return VCRYPT_OK;
}

extern "C" int vcrypt_last_stage_ms(const vcrypt_ctx *c, double out[4]) {
    if (!c || !out) return VCRYPT_E_ARG;
    std::memcpy(out, c->stage_ms, sizeof c->stage_ms);
    return VCRYPT_OK;
}

// =====================================================================================================
// host derivation (Algorithm 1 steps 4-14, Algorithm 2)
// =====================================================================================================
namespace {

// H of m frames: every (frame, sub-frame) pair is one job; H = xor of the sub-frame digests.
// Only bands 0 .. nb-1 of every frame are hashed here (nb = n: the whole frame; fewer when the GPU takes the rest).
void hash_frames(vcrypt_ctx *c, const uint8_t *frames, size_t m, uint8_t *hashes, uint32_t nb) {
    const uint32_t n = c->p.n_workers, h = c->g.h;
    const size_t rb = c->g.row_bytes, fb = c->g.frame_bytes;
    uint8_t *sub = c->subhash.data();
    const bool simd = c->simd;
    c->pool->parallel_for(m * nb, [&](size_t job) {
        const size_t f = job / nb;
        const uint32_t k = (uint32_t)(job - f * nb);
        const size_t r0 = vh::band_row(k, n, h), r1 = vh::band_row(k + 1, n, h);
        vh::sha256(frames + f * fb + r0 * rb, (r1 - r0) * rb, sub + (f * n + k) * 32u, simd);
    });
    for (size_t f = 0; f < m; ++f) {
        uint8_t *H = hashes + 32u * f;
        std::memset(H, 0, 32);
        for (uint32_t k = 0; k < nb; ++k)
            for (int b = 0; b < 32; ++b) H[b] ^= sub[(f * n + k) * 32u + b];
    }
}

// D and B of m frames whose hashes are known, written frame after frame into D / B.  S is advanced.
// Returns VCRYPT_E_STATE if a chaotic state became non-finite.
int derive_frames(vcrypt_ctx *c, double S[4], const uint8_t *hashes, size_t m, uint16_t *D, uint8_t *B, bool flush_B = false) {
    const uint32_t n = c->p.n_workers;
    const double gamma = c->p.gamma;
    // the chain is serial in the frame index, and cheap (2n * K_m RK4 steps per frame)
    for (size_t f = 0; f < m; ++f) {
        double *IR = c->IR.data() + f * 2u * n * 4u;
        if (!vh::chain_step(S, gamma, n, hashes + 32u * f, IR)) return VCRYPT_E_STATE;
        vh::make_slices(IR, n, c->g.w, c->g.h, D + f * c->g.nD, B + f * c->g.frame_bytes, c->slices.data() + f * n);
    }
    // a batch whose keystream would stay in the cores' private caches (single-frame calls: latency) is flushed by the jobs
    // that write it; a large batch spills to memory by itself and the flushes would only cost the host-bound pipeline time
    // (only on CPUs that have CLFLUSHOPT: the AVX2 / AVX-512 units are compiled with it, AVX2 alone does not imply it)
    if (flush_B && vh::has_clflushopt() && m * c->g.frame_bytes <= ((size_t)32 << 20))
        for (size_t i = 0; i < m * n; ++i) c->slices[i].flush_B = true;
    const int isa = c->isa;
    const size_t lanes = isa == 2 ? 8 : isa == 1 ? 4 : 1;
    const size_t groups = (n + lanes - 1) / lanes;
    std::atomic<bool> ok{true};
    const vh::WorkerSlice *sl = c->slices.data();
    c->pool->parallel_for(m * groups, [&](size_t job) {
        const size_t f = job / groups, g0 = (job - f * groups) * lanes;
        const size_t cnt = n - g0 < lanes ? n - g0 : lanes;
        if (!vh::derive_workers(sl + f * n + g0, cnt, gamma, isa)) ok.store(false, std::memory_order_relaxed);
    });
    return ok.load() ? VCRYPT_OK : VCRYPT_E_STATE;
}

// The serial part only (Algorithm 1 steps 7-13): IR of m frames, frame after frame, into `IR` (m x 2n x 4 doubles).
int chain_frames(vcrypt_ctx *c, double S[4], const uint8_t *hashes, size_t m, double *IR) {
    const uint32_t n = c->p.n_workers;
    for (size_t f = 0; f < m; ++f)
        if (!vh::chain_step(S, c->p.gamma, n, hashes + 32u * f, IR + f * 2u * n * 4u)) return VCRYPT_E_STATE;
    return VCRYPT_OK;
}

}  // namespace

extern "C" int vcrypt_frame_hash(vcrypt_ctx *c, const uint8_t *frame, uint8_t *H_out) {
    return guarded([&]() -> int {
        if (!c || !frame || !H_out) return VCRYPT_E_ARG;
        hash_frames(c, frame, 1, H_out, c->p.n_workers);
        return VCRYPT_OK;
    });
}

extern "C" int vcrypt_derive(vcrypt_ctx *c, const uint8_t *hash, uint16_t *D_out, uint8_t *B_out) {
    return guarded([&]() -> int {
        if (!c || !hash || !D_out || !B_out) return VCRYPT_E_ARG;
        double S[4];
        std::memcpy(S, c->S, sizeof S);
        const int rc = derive_frames(c, S, hash, 1, D_out, B_out);
        if (rc != VCRYPT_OK) return rc;
        std::memcpy(c->S, S, sizeof S);
        c->frames_done += 1;
        return VCRYPT_OK;
    });
}

extern "C" int vcrypt_frame_hash_device(vcrypt_ctx *c, const void *d_frames, size_t n, uint8_t *hashes_out, void *stream) {
    return guarded([&]() -> int {
        if (!c || !d_frames || !hashes_out || n == 0) return VCRYPT_E_ARG;
        if (!c->cuda) return VCRYPT_E_CUDA;
        if ((((uintptr_t)d_frames) & 15u) || c->g.row_bytes % 16u != 0) return VCRYPT_E_SHAPE;
        VC_DEVICE(c);
        cudaStream_t st = static_cast<cudaStream_t>(stream);
        uint32_t *d_H = nullptr;
        cudaError_t e = cudaMalloc(&d_H, n * 32u);
        if (e == cudaSuccess) e = vk::hash_device(c->g, static_cast<const uint8_t *>(d_frames), c->p.n_workers, 0, n, d_H, st);
        if (e == cudaSuccess) e = cudaMemcpyAsync(hashes_out, d_H, n * 32u, cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (d_H) cudaFree(d_H);
        if (e != cudaSuccess) return cuda_fail(c, e, "device hashing");
        return VCRYPT_OK;
    });
}

extern "C" int vcrypt_derive_device(vcrypt_ctx *c, const uint8_t *hash, void *d_D, void *d_B, void *stream) {
    return guarded([&]() -> int {
        if (!c || !hash || !d_D || !d_B) return VCRYPT_E_ARG;
        if (!c->cuda) return VCRYPT_E_CUDA;
        if ((((uintptr_t)d_B) & 7u) || (((uintptr_t)d_D) & 1u)) return VCRYPT_E_ARG;
        VC_DEVICE(c);
        cudaStream_t st = static_cast<cudaStream_t>(stream);
        const size_t irb = 2u * (size_t)c->p.n_workers * 4u * sizeof(double);
        double S[4];
        std::memcpy(S, c->S, sizeof S);
        std::vector<double> IR(2u * (size_t)c->p.n_workers * 4u);
        int rc = chain_frames(c, S, hash, 1, IR.data());
        if (rc != VCRYPT_OK) return rc;
        double *d_IR = nullptr;
        uint32_t *d_status = nullptr, h_status = 0;
        cudaError_t e = cudaMalloc(&d_IR, irb);
        if (e == cudaSuccess) e = cudaMalloc(&d_status, sizeof(uint32_t));
        if (e == cudaSuccess) e = cudaMemcpyAsync(d_IR, IR.data(), irb, cudaMemcpyHostToDevice, st);
        if (e == cudaSuccess) e = cudaMemsetAsync(d_status, 0, sizeof(uint32_t), st);
        if (e == cudaSuccess)
            e = vk::derive_device(c->g, d_IR, c->p.gamma, c->p.n_workers, 1, static_cast<uint16_t *>(d_D), static_cast<uint8_t *>(d_B),
                                  d_status, st);
        if (e == cudaSuccess) e = cudaMemcpyAsync(&h_status, d_status, sizeof(uint32_t), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (d_IR) cudaFree(d_IR);
        if (d_status) cudaFree(d_status);
        if (e != cudaSuccess) return cuda_fail(c, e, "device derivation");
        if (h_status) return VCRYPT_E_STATE;
        std::memcpy(c->S, S, sizeof S);
        c->frames_done += 1;
        return VCRYPT_OK;
    });
}

// =====================================================================================================
// kernel-only path
// =====================================================================================================
static int device_call(vcrypt_ctx *c, bool decrypt, const void *d_in, const void *d_D, const void *d_B, size_t n,
                       void *d_out, void *stream) {
    if (!c || !d_in || !d_D || !d_B || !d_out) return VCRYPT_E_ARG;
    if (!c->cuda) return VCRYPT_E_CUDA;
    if ((((uintptr_t)d_in) | ((uintptr_t)d_out) | ((uintptr_t)d_B)) & 15u) return VCRYPT_E_ARG;
    if (((uintptr_t)d_D) & 1u) return VCRYPT_E_ARG;
    c->launches_last = 0;
    if (n == 0) return VCRYPT_OK;
    const uint8_t *a = static_cast<const uint8_t *>(d_in);
    uint8_t *o = static_cast<uint8_t *>(d_out);
    const size_t bytes = n * c->g.frame_bytes;
    if (a != o && a < o + bytes && o < a + bytes) return VCRYPT_E_ARG;  // partial overlap
    VC_DEVICE(c);
    return launch_cipher(c, decrypt, a, static_cast<const uint16_t *>(d_D), static_cast<const uint8_t *>(d_B), n, o,
                         static_cast<cudaStream_t>(stream));
}

extern "C" int vcrypt_encrypt_device(vcrypt_ctx *c, const void *d_frames, const void *d_D, const void *d_B, size_t n,
                                     void *d_cipher, void *stream) {
    return guarded([&]() -> int {
        return device_call(c, false, d_frames, d_D, d_B, n, d_cipher, stream);
    });
}

extern "C" int vcrypt_decrypt_device(vcrypt_ctx *c, const void *d_cipher, const void *d_D, const void *d_B, size_t n,
                                     void *d_plain, void *stream) {
    return guarded([&]() -> int {
        return device_call(c, true, d_cipher, d_D, d_B, n, d_plain, stream);
    });
}

// =====================================================================================================
// statistical evaluation (PAPER.md sections III-IV): exact integer sums from the GPU, final steps in binary64
// =====================================================================================================
namespace {

double entropy_bits(const uint32_t *z, double total) {  // Eq. 10
    double H = 0.0;
    for (int i = 0; i < 256; ++i)
        if (z[i]) {
            const double p = (double)z[i] / total;
            H += p * std::log2(1.0 / p);
        }
    return H;
}

}  // namespace

extern "C" int vcrypt_frame_stats_device(vcrypt_ctx *c, const void *d_frames, size_t n, vcrypt_frame_stats *out, uint32_t *hist_out,
                                         void *stream) {
    return guarded([&]() -> int {
        if (!c || !d_frames || !out || n == 0) return VCRYPT_E_ARG;
        if (!c->cuda) return VCRYPT_E_CUDA;
        VC_DEVICE(c);
        cudaStream_t st = static_cast<cudaStream_t>(stream);
        uint32_t *d_hist = nullptr;
        unsigned long long *d_pairs = nullptr;
        std::vector<uint32_t> hist(n * 768u);
        std::vector<unsigned long long> pairs(n * 45u);
        cudaError_t e = cudaMalloc(&d_hist, n * 768u * sizeof(uint32_t));
        if (e == cudaSuccess) e = cudaMalloc(&d_pairs, n * 45u * sizeof(unsigned long long));
        if (e == cudaSuccess) e = vk::stats_device(c->g, static_cast<const uint8_t *>(d_frames), n, d_hist, d_pairs, st);
        if (e == cudaSuccess) e = cudaMemcpyAsync(hist.data(), d_hist, hist.size() * sizeof(uint32_t), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaMemcpyAsync(pairs.data(), d_pairs, pairs.size() * sizeof(unsigned long long), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (d_hist) cudaFree(d_hist);
        if (d_pairs) cudaFree(d_pairs);
        if (e != cudaSuccess) return cuda_fail(c, e, "frame statistics");
        const double N = (double)c->g.w * (double)c->g.h;
        const uint64_t w = c->g.w, h = c->g.h;
        const double npairs[3] = {(double)((w - 1) * h), (double)(w * (h - 1)), (double)((w - 1) * (h - 1))};
        for (size_t f = 0; f < n; ++f) {
            vcrypt_frame_stats &o = out[f];
            for (int ch = 0; ch < 3; ++ch) {
                const uint32_t *z = hist.data() + f * 768u + ch * 256u;
                double s1 = 0.0, s2 = 0.0, chi = 0.0;
                const double ex = N / 256.0;
                for (int i = 0; i < 256; ++i) {
                    s1 += (double)z[i];
                    s2 += (double)z[i] * (double)z[i];
                    chi += ((double)z[i] - ex) * ((double)z[i] - ex) / ex;
                }
                // Eq. 4: (1/256^2) sum_i sum_j (z_i - z_j)^2 / 2 = (256 sum z^2 - (sum z)^2) / 256^2
                o.hist_variance[ch] = (256.0 * s2 - s1 * s1) / 65536.0;
                o.chi2[ch] = chi;
                o.entropy[ch] = entropy_bits(z, N);
                for (int d = 0; d < 3; ++d) {
                    const unsigned long long *p = pairs.data() + f * 45u + (ch * 3 + d) * 5;
                    const double M = npairs[d];
                    if (M <= 0.0) { o.corr[ch][d] = std::nan(""); continue; }
                    // Eq. 6-9 from the exact sums: cov = E[xy] - E[x]E[y], D(x) = E[x^2] - E[x]^2 (integer numerators)
                    const long double sx = (long double)p[0], sy = (long double)p[1], sxy = (long double)p[2], sxx = (long double)p[3],
                                      syy = (long double)p[4], m = (long double)M;
                    const long double cov = m * sxy - sx * sy, dx = m * sxx - sx * sx, dy = m * syy - sy * sy;
                    o.corr[ch][d] = (dx > 0 && dy > 0) ? (double)(cov / std::sqrt(dx * dy)) : std::nan("");
                }
            }
        }
        if (hist_out) std::memcpy(hist_out, hist.data(), hist.size() * sizeof(uint32_t));
        return VCRYPT_OK;
    });
}

extern "C" int vcrypt_npcr_uaci_device(vcrypt_ctx *c, const void *d_a, const void *d_b, size_t n, double *npcr, double *uaci,
                                       void *stream) {
    return guarded([&]() -> int {
        if (!c || !d_a || !d_b || !npcr || !uaci || n == 0) return VCRYPT_E_ARG;
        if (!c->cuda) return VCRYPT_E_CUDA;
        VC_DEVICE(c);
        cudaStream_t st = static_cast<cudaStream_t>(stream);
        unsigned long long *d_out = nullptr;
        std::vector<unsigned long long> r(n * 6u);
        cudaError_t e = cudaMalloc(&d_out, r.size() * sizeof(unsigned long long));
        if (e == cudaSuccess) e = vk::diff_device(c->g, static_cast<const uint8_t *>(d_a), static_cast<const uint8_t *>(d_b), n, d_out, st);
        if (e == cudaSuccess) e = cudaMemcpyAsync(r.data(), d_out, r.size() * sizeof(unsigned long long), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (d_out) cudaFree(d_out);
        if (e != cudaSuccess) return cuda_fail(c, e, "NPCR / UACI");
        const double N = (double)c->g.w * (double)c->g.h;
        for (size_t f = 0; f < n; ++f) {
            unsigned long long ne = 0, ad = 0;
            for (int ch = 0; ch < 3; ++ch) {
                const unsigned long long a = r[f * 6u + 2 * ch], b = r[f * 6u + 2 * ch + 1];
                ne += a;
                ad += b;
                npcr[4 * f + 1 + ch] = 100.0 * (double)a / N;            // Eq. 14, 16
                uaci[4 * f + 1 + ch] = 100.0 * (double)b / (N * 255.0);  // Eq. 15
            }
            npcr[4 * f] = 100.0 * (double)ne / (3.0 * N);
            uaci[4 * f] = 100.0 * (double)ad / (3.0 * N * 255.0);
        }
        return VCRYPT_OK;
    });
}

// The no-allocation twin of vcrypt_npcr_uaci_device (include/vcrypt.h): same sums, same binary64 steps, but the device
// accumulators are the library's static array (stats.cu) and the host landing buffer is on this thread's stack, so nothing
// on the path asks CUDA (or the heap) for memory.
extern "C" int vcrypt_npcr_uaci_device_noalloc(vcrypt_ctx *c, const void *d_a, const void *d_b, size_t n, double *npcr, double *uaci,
                                               void *stream) {
    return guarded([&]() -> int {
        if (!c || !d_a || !d_b || !npcr || !uaci || n == 0) return VCRYPT_E_ARG;
        if (n > VCRYPT_NOALLOC_MAX_FRAMES) {
            std::snprintf(c->cuda_msg, sizeof c->cuda_msg, "vcrypt_npcr_uaci_device_noalloc: n = %zu frames, the static scratch holds %u",
                          n, (unsigned)VCRYPT_NOALLOC_MAX_FRAMES);
            return VCRYPT_E_LIMIT;
        }
        if (!c->cuda) return VCRYPT_E_CUDA;
        VC_DEVICE(c);
        static_assert(VCRYPT_NOALLOC_MAX_FRAMES == vk::kDiffStaticMaxFrames, "header and kernel limits must agree");
        unsigned long long r[vk::kDiffStaticMaxFrames * 6u];  // 24 KB of stack
        const cudaError_t e = vk::diff_device_static(c->g, static_cast<const uint8_t *>(d_a), static_cast<const uint8_t *>(d_b), n, r,
                                                     static_cast<cudaStream_t>(stream));
        if (e != cudaSuccess) return cuda_fail(c, e, "NPCR / UACI (static scratch)");
        const double N = (double)c->g.w * (double)c->g.h;
        for (size_t f = 0; f < n; ++f) {
            unsigned long long ne = 0, ad = 0;
            for (int ch = 0; ch < 3; ++ch) {
                const unsigned long long a = r[f * 6u + 2 * ch], b = r[f * 6u + 2 * ch + 1];
                ne += a;
                ad += b;
                npcr[4 * f + 1 + ch] = 100.0 * (double)a / N;            // Eq. 14, 16
                uaci[4 * f + 1 + ch] = 100.0 * (double)b / (N * 255.0);  // Eq. 15
            }
            npcr[4 * f] = 100.0 * (double)ne / (3.0 * N);
            uaci[4 * f] = 100.0 * (double)ad / (3.0 * N * 255.0);
        }
        return VCRYPT_OK;
    });
}

extern "C" int vcrypt_local_entropy_device(vcrypt_ctx *c, const void *d_frames, size_t n, const uint32_t *xy, uint32_t k, uint32_t side,
                                           double *out, void *stream) {
    return guarded([&]() -> int {
        if (!c || !d_frames || !xy || !out || n == 0 || k == 0 || side == 0) return VCRYPT_E_ARG;
        if (!c->cuda) return VCRYPT_E_CUDA;
        for (uint32_t b = 0; b < k; ++b)
            if ((uint64_t)xy[2 * b] + side > c->g.w || (uint64_t)xy[2 * b + 1] + side > c->g.h) return VCRYPT_E_ARG;
        VC_DEVICE(c);
        cudaStream_t st = static_cast<cudaStream_t>(stream);
        uint32_t *d_xy = nullptr, *d_bh = nullptr;
        std::vector<uint32_t> bh(n * k * 768u);
        cudaError_t e = cudaMalloc(&d_xy, 2u * k * sizeof(uint32_t));
        if (e == cudaSuccess) e = cudaMalloc(&d_bh, bh.size() * sizeof(uint32_t));
        if (e == cudaSuccess) e = cudaMemcpyAsync(d_xy, xy, 2u * k * sizeof(uint32_t), cudaMemcpyHostToDevice, st);
        if (e == cudaSuccess) e = vk::block_hist_device(c->g, static_cast<const uint8_t *>(d_frames), n, d_xy, k, side, d_bh, st);
        if (e == cudaSuccess) e = cudaMemcpyAsync(bh.data(), d_bh, bh.size() * sizeof(uint32_t), cudaMemcpyDeviceToHost, st);
        if (e == cudaSuccess) e = cudaStreamSynchronize(st);
        if (d_xy) cudaFree(d_xy);
        if (d_bh) cudaFree(d_bh);
        if (e != cudaSuccess) return cuda_fail(c, e, "local entropy");
        const double TB = (double)side * (double)side;
        for (size_t f = 0; f < n; ++f)
            for (int ch = 0; ch < 3; ++ch) {
                double acc = 0.0;
                for (uint32_t b = 0; b < k; ++b) acc += entropy_bits(bh.data() + ((f * k + b) * 3u + ch) * 256u, TB);
                out[3 * f + ch] = acc / (double)k;  // Eq. 11
            }
        return VCRYPT_OK;
    });
}

// =====================================================================================================
// host-buffer pipeline: Algorithm 1's loop over frames, batched and overlapped
// =====================================================================================================
static int run_frames(vcrypt_ctx *c, bool decrypt, const uint8_t *in, const uint8_t *hashes_in, size_t n, uint8_t *out,
                      uint8_t *hashes_out) {
    if (!c || !in || !out || (decrypt ? !hashes_in : !hashes_out)) return VCRYPT_E_ARG;
    if (!c->cuda) return VCRYPT_E_CUDA;
    c->launches_last = 0;
    for (double &v : c->stage_ms) v = 0.0;
    if (n == 0) return VCRYPT_OK;
    VC_DEVICE(c);
    const size_t fb = c->g.frame_bytes, nD = c->g.nD;
    const bool in_pinned = is_pinned(in) && is_pinned(in + n * fb - 1);
    const bool out_pinned = is_pinned(out) && is_pinned(out + n * fb - 1);
    const bool generic = !c->plan.tiled || (c->p.flags & VCRYPT_FLAG_FORCE_GENERIC);
    const bool dev_derive = (c->p.flags & VCRYPT_FLAG_DEVICE_DERIVE) != 0;
    // device hashing needs 16-byte rows (128-bit loads); other shapes are hashed on the host: same bytes
    const bool dev_hash = !decrypt && (c->p.flags & VCRYPT_FLAG_DEVICE_HASH) && c->g.row_bytes % 16u == 0;
    // the GPU hashes the last `dev_bands` row bands of every frame, the host threads the others at the same time
    const uint32_t nw = c->p.n_workers;
    const uint32_t dev_bands = !dev_hash ? 0u : c->p.device_hash_bands == 0 || c->p.device_hash_bands > nw ? nw : c->p.device_hash_bands;
    const uint32_t host_bands = nw - dev_bands;
    const size_t S_ = c->slots.size();
    const size_t nbatch = (n + c->batch - 1) / c->batch;
    // Two stages per batch.  Stage A: staging, upload of the frames, hashing (host threads, or the GPU + an event).
    // Stage B: chain + derivation, rest of the upload, cipher kernels, download.  With device hashing stage A runs
    // S / 2 batches ahead, so that the host only waits for hashes that were requested long ago and a slot's stage B has
    // S / 2 iterations to finish before the slot is reused; otherwise A and B of a batch follow each other directly.
    const size_t lag = dev_hash ? S_ / 2 : 0;
    double S[4];
    std::memcpy(S, c->S, sizeof S);
    int rc = VCRYPT_OK;

    auto stage_a = [&](size_t k) -> int {
        const size_t b0 = k * c->batch, m = n - b0 < c->batch ? n - b0 : c->batch;
        Slot &s = c->slots[k % S_];
        int r = retire_slot(c, s);
        if (r != VCRYPT_OK) return r;
        if ((r = ensure_slot(c, s, !in_pinned, !out_pinned)) != VCRYPT_OK) return r;
        const uint8_t *src = in + b0 * fb;
        if (!in_pinned) {
            const auto t0 = clk::now();
            const size_t chunk = (size_t)1 << 20, total = m * fb, nch = (total + chunk - 1) / chunk;
            uint8_t *dst = s.h_F;
            c->pool->parallel_for(nch, [&](size_t i) {
                const size_t o = i * chunk, len = total - o < chunk ? total - o : chunk;
                std::memcpy(dst + o, src + o, len);
            });
            c->stage_ms[2] += ms_since(t0);
        }
        // step 15, first part: the frames do not depend on the derivation, so their upload is enqueued first and runs
        // while the host hashes and derives
        cudaError_t e = cudaMemcpyAsync(s.d_F, in_pinned ? src : s.h_F, m * fb, cudaMemcpyHostToDevice, s.st);
        if (e != cudaSuccess) return cuda_fail(c, e, "upload");
        if (dev_hash) {  // Algorithm 1 steps 4-6, the GPU's share: one thread per (frame, band), xor of the band digests
            e = vk::hash_device(c->g, s.d_F, nw, host_bands, m, s.d_H, s.st);
            if (e == cudaSuccess) e = cudaMemcpyAsync(s.h_H, s.d_H, m * 32u, cudaMemcpyDeviceToHost, s.st);
            if (e == cudaSuccess) e = cudaEventRecord(s.hashed, s.st);
            if (e != cudaSuccess) return cuda_fail(c, e, "device hashing");
            c->launches_last += 2;
            c->launches_total += 2;
        }
        if (!decrypt) {  // Algorithm 1 steps 4-6 on the host threads (all bands, or the host's share)
            const auto t0 = clk::now();
            hash_frames(c, src, m, hashes_out + 32u * b0, host_bands);
            c->stage_ms[0] += ms_since(t0);
        }
        return VCRYPT_OK;
    };

    auto stage_b = [&](size_t k) -> int {
        const size_t b0 = k * c->batch, m = n - b0 < c->batch ? n - b0 : c->batch;
        Slot &s = c->slots[k % S_];
        const uint8_t *hs = decrypt ? hashes_in + 32u * b0 : hashes_out + 32u * b0;
        if (dev_hash) {
            const auto t0 = clk::now();
            const cudaError_t e = cudaEventSynchronize(s.hashed);
            c->stage_ms[0] += ms_since(t0);
            if (e != cudaSuccess) return cuda_fail(c, e, "device hashing");
            for (size_t i = 0; i < m * 32u; ++i) hashes_out[32u * b0 + i] ^= s.h_H[i];  // host share xor device share
        }
        {  // steps 7-14
            const auto t0 = clk::now();
            const int r = dev_derive ? chain_frames(c, S, hs, m, s.h_IR) : derive_frames(c, S, hs, m, s.h_D, s.h_B, true);
            c->stage_ms[1] += ms_since(t0);
            if (r != VCRYPT_OK) return r;
        }
        // steps 15-21: rest of the upload, GPU steps, download -- asynchronous on the slot's stream
        uint8_t *d_res = generic ? s.d_out : s.d_F;
        uint8_t *h_res = out_pinned ? out + b0 * fb : s.h_out;
        cudaError_t e;
        if (dev_derive) {  // the worker systems run on the GPU: only the LHCS_m records go up (2n x 32 bytes per frame)
            e = cudaMemcpyAsync(s.d_IR, s.h_IR, m * 2u * (size_t)c->p.n_workers * 4u * sizeof(double), cudaMemcpyHostToDevice, s.st);
            if (e == cudaSuccess) e = cudaMemsetAsync(s.d_status, 0, sizeof(uint32_t), s.st);
            if (e == cudaSuccess) e = vk::derive_device(c->g, s.d_IR, c->p.gamma, c->p.n_workers, m, s.d_D, s.d_B, s.d_status, s.st);
            if (e == cudaSuccess) e = cudaMemcpyAsync(s.h_status, s.d_status, sizeof(uint32_t), cudaMemcpyDeviceToHost, s.st);
            if (e == cudaSuccess) { s.status_pending = true; c->launches_last += 1; c->launches_total += 1; }
        } else {
            e = cudaMemcpyAsync(s.d_D, s.h_D, m * nD * sizeof(uint16_t), cudaMemcpyHostToDevice, s.st);
            if (e == cudaSuccess) e = cudaMemcpyAsync(s.d_B, s.h_B, m * fb, cudaMemcpyHostToDevice, s.st);
        }
        if (e != cudaSuccess) return cuda_fail(c, e, "upload");
        const int r = launch_cipher(c, decrypt, s.d_F, s.d_D, s.d_B, m, d_res, s.st);
        if (r != VCRYPT_OK) return r;
        e = cudaMemcpyAsync(h_res, d_res, m * fb, cudaMemcpyDeviceToHost, s.st);
        if (e == cudaSuccess) e = cudaEventRecord(s.done, s.st);
        if (e != cudaSuccess) return cuda_fail(c, e, "download");
        s.busy = true;
        s.user_out = out_pinned ? nullptr : out + b0 * fb;
        s.out_bytes = m * fb;
        return VCRYPT_OK;
    };

    for (size_t k = 0; k < nbatch + lag && rc == VCRYPT_OK; ++k) {
        if (k < nbatch) rc = stage_a(k);
        if (rc == VCRYPT_OK && k >= lag) rc = stage_b(k - lag);
    }
    // drain in submission order
    for (size_t i = 0; i < S_; ++i) {
        Slot &s = c->slots[(nbatch + i) % S_];
        const int r2 = retire_slot(c, s);
        if (rc == VCRYPT_OK) rc = r2;
    }
    if (rc != VCRYPT_OK) {  // chain untouched; nothing of this call may still be reading the caller's buffers
        for (Slot &s : c->slots)
            if (s.st) cudaStreamSynchronize(s.st);
        return rc;
    }
    std::memcpy(c->S, S, sizeof S);
    c->frames_done += n;
    return VCRYPT_OK;
}

extern "C" int vcrypt_encrypt_frames(vcrypt_ctx *c, const uint8_t *frames, size_t n, uint8_t *cipher_out,
                                     uint8_t *hashes_out) {
    return guarded([&]() -> int {
        return run_frames(c, false, frames, nullptr, n, cipher_out, hashes_out);
    });
}

extern "C" int vcrypt_decrypt_frames(vcrypt_ctx *c, const uint8_t *cipher, const uint8_t *hashes, size_t n,
                                     uint8_t *plain_out) {
    return guarded([&]() -> int {
        return run_frames(c, true, cipher, hashes, n, plain_out, nullptr);
    });
}
