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
//
// dsmem_probe (vcrypt_dsmem_probe) answers a design question instead: how fast can the CTAs of a
// thread-block cluster exchange an all-to-all through distributed shared memory -- the alternative to passing the
// intermediate between row owners and column owners through L2.
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

// ---------------------------------------------------------------------------------------------
// Distributed-shared-memory exchange: every CTA of a cluster owns `own` bytes of shared memory and, per round, sends
// own / CS bytes to each of the CS CTAs of its cluster (itself included), i.e. the cluster performs one all-to-all of
// CS * own bytes.  mode 0: 16-byte st.shared::cluster stores by the threads; mode 1: one cp.async.bulk shared::cta ->
// shared::cluster per peer with completion on the peer's mbarrier.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t pb_smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ uint32_t pb_mapa(uint32_t addr, uint32_t rank) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
    return r;
}
__device__ __forceinline__ void pb_cluster_sync() {
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}

template <int MODE>
__global__ void __launch_bounds__(512, 1) probe_dsmem(uint32_t own, uint32_t rounds, uint32_t *sink) {
    extern __shared__ __align__(128) uint8_t PS[];
    uint32_t CS, rank;
    asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(CS));
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(rank));
    uint8_t *strip = PS, *src = PS + own;
    uint64_t *bar = reinterpret_cast<uint64_t *>(PS + 2u * own);
    const uint32_t piece = own / CS;
    for (uint32_t i = threadIdx.x; i < own / 4u; i += blockDim.x) reinterpret_cast<uint32_t *>(src)[i] = i * 2654435761u + rank;
    if (threadIdx.x == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(pb_smem_u32(bar)));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    pb_cluster_sync();
    for (uint32_t r = 0; r < rounds; ++r) {
        if (MODE == 0) {
            for (uint32_t i = threadIdx.x; i < own / 16u; i += blockDim.x) {
                const uint32_t byte = i * 16u, p = byte / piece, off = byte - p * piece;
                const uint4 v = *reinterpret_cast<const uint4 *>(src + byte);
                const uint32_t dst = pb_mapa(pb_smem_u32(strip + rank * piece + off), p);
                asm volatile("st.shared::cluster.v4.u32 [%0], {%1,%2,%3,%4};" ::"r"(dst), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w) : "memory");
            }
            pb_cluster_sync();
        } else {
            if (threadIdx.x == 0)
                asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(pb_smem_u32(bar)), "r"(piece * CS) : "memory");
            pb_cluster_sync();  // every barrier of the cluster is armed
            if (threadIdx.x < CS) {
                const uint32_t p = threadIdx.x;
                const uint32_t dst = pb_mapa(pb_smem_u32(strip + rank * piece), p), rbar = pb_mapa(pb_smem_u32(bar), p);
                asm volatile("cp.async.bulk.shared::cluster.shared::cta.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                             "r"(pb_smem_u32(src + p * piece)), "r"(piece), "r"(rbar)
                             : "memory");
            }
            uint32_t ok = 0, spin = 0;
            while (!ok) {
                asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
                             : "=r"(ok)
                             : "r"(pb_smem_u32(bar)), "r"(r & 1u)
                             : "memory");
                if (++spin > (1u << 24)) __trap();  // a copy that never lands must trap, not hang the GPU
            }
            pb_cluster_sync();
        }
    }
    if (threadIdx.x == 0) {
        uint32_t acc = 0;
        for (uint32_t i = 0; i < own / 4u; i += 97u) acc += reinterpret_cast<uint32_t *>(strip)[i];
        sink[blockIdx.x] = acc;
    }
}

cudaError_t dsmem_probe(int cluster_size, size_t own_bytes, int mode, int rounds, double *us_per_round, int *max_active_clusters,
                        int *clusters_launched) {
    if (cluster_size < 1 || cluster_size > 16 || (mode != 0 && mode != 1) || rounds < 1) return cudaErrorInvalidValue;
    if (own_bytes < 16u * (size_t)cluster_size || own_bytes % (16u * (size_t)cluster_size) != 0) return cudaErrorInvalidValue;
    int dev = 0, sms = 0, smem_optin = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (!e) e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (!e) e = cudaDeviceGetAttribute(&smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    if (e) return e;
    const size_t smem = 2 * own_bytes + 64;
    if (smem > (size_t)smem_optin) return cudaErrorInvalidValue;
    void (*k)(uint32_t, uint32_t, uint32_t *) = mode == 0 ? probe_dsmem<0> : probe_dsmem<1>;
    e = cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (!e) e = cudaFuncSetAttribute(k, cudaFuncAttributeNonPortableClusterSizeAllowed, 1);
    if (e) return e;
    cudaLaunchConfig_t cfg{};
    cfg.blockDim = dim3(512);
    cfg.dynamicSmemBytes = smem;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeClusterDimension;
    at[0].val.clusterDim.x = (unsigned)cluster_size;
    at[0].val.clusterDim.y = 1;
    at[0].val.clusterDim.z = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    cfg.gridDim = dim3((unsigned)cluster_size);
    int maxc = 0;
    e = cudaOccupancyMaxActiveClusters(&maxc, k, &cfg);
    if (e) return e;
    if (max_active_clusters) *max_active_clusters = maxc;
    if (maxc < 1) return cudaErrorInvalidValue;
    if (clusters_launched) *clusters_launched = maxc;
    cfg.gridDim = dim3((unsigned)(cluster_size * maxc));  // one resident wave
    uint32_t *sink = nullptr;
    cudaEvent_t e0 = nullptr, e1 = nullptr;
    e = cudaMalloc(&sink, sizeof(uint32_t) * cluster_size * maxc);
    if (!e) e = cudaEventCreate(&e0);
    if (!e) e = cudaEventCreate(&e1);
    if (!e) e = cudaLaunchKernelEx(&cfg, k, (uint32_t)own_bytes, (uint32_t)rounds, sink);  // warm-up
    if (!e) e = cudaEventRecord(e0, 0);
    if (!e) e = cudaLaunchKernelEx(&cfg, k, (uint32_t)own_bytes, (uint32_t)rounds, sink);
    if (!e) e = cudaEventRecord(e1, 0);
    if (!e) e = cudaEventSynchronize(e1);
    float ms = 0.f;
    if (!e) e = cudaEventElapsedTime(&ms, e0, e1);
    if (!e && us_per_round) *us_per_round = 1e3 * (double)ms / rounds;
    cudaDeviceSynchronize();
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(sink);
    return e;
}

}  // namespace vk
