// derive.cu -- device-side worker systems: Algorithm 2 steps 5-10 on the GPU.
//
// Two threads per worker, one per Lorenz hyper-chaotic system (Eq. 1); the two exchange the 48 low
// mantissa bits of x, y, z, w with a shuffle after every RK4 step and the even lane writes the worker's 24 keystream
// bytes: the first ceil(2 nd / 24) steps into its slice of D, the following ceil(nb / 24) into its slice of B
// (readings Q8-Q11 of DESIGN.md) -- straight into the device buffers the cipher kernels read, so neither D nor B
// crosses PCIe and the host is left with hashing and the serial LHCS_m chain.
//
// Bit-exactness: every floating-point operation is an explicit round-to-nearest IEEE binary64 intrinsic (__dadd_rn,
// __dsub_rn, __dmul_rn: never contracted into FMA) in the expression order of DESIGN.md "Bit-exact floating point";
// the file is also compiled with -fmad=false.  The bytes equal the host lanes' and the oracle's.
#include <cuda_runtime.h>
#include <stdint.h>

#include "kernels.cuh"

namespace vk {

namespace {

struct S4 {
    double x, y, z, w;
};

__device__ __forceinline__ S4 rhs(const S4 &s, double gamma) {
    const double B83 = 8.0 / 3.0;
    S4 d;
    d.x = __dadd_rn(__dmul_rn(10.0, __dsub_rn(s.y, s.x)), s.w);                      // 10 (y - x) + w
    d.y = __dsub_rn(__dsub_rn(__dmul_rn(28.0, s.x), s.y), __dmul_rn(s.x, s.z));      // (28 x - y) - x z
    d.z = __dsub_rn(__dmul_rn(s.x, s.y), __dmul_rn(B83, s.z));                       // x y - (8/3) z
    d.w = __dadd_rn(-__dmul_rn(s.y, s.z), __dmul_rn(gamma, s.w));                    // (-(y z)) + gamma w
    return d;
}
__device__ __forceinline__ S4 axpy(const S4 &s, double a, const S4 &k) {
    return S4{__dadd_rn(s.x, __dmul_rn(a, k.x)), __dadd_rn(s.y, __dmul_rn(a, k.y)), __dadd_rn(s.z, __dmul_rn(a, k.z)),
              __dadd_rn(s.w, __dmul_rn(a, k.w))};
}
__device__ __forceinline__ double comb(double s, double dt6, double k1, double k2, double k3, double k4) {
    // s + dt6 * (((k1 + 2 k2) + 2 k3) + k4)
    return __dadd_rn(s, __dmul_rn(dt6, __dadd_rn(__dadd_rn(__dadd_rn(k1, __dmul_rn(2.0, k2)), __dmul_rn(2.0, k3)), k4)));
}
__device__ __forceinline__ void rk4(S4 &s, double gamma) {
    const double dt = 0.005, hdt = 0.5 * 0.005, dt6 = 0.005 / 6.0;  // DESIGN.md Q3; each one rounded constant
    const S4 k1 = rhs(s, gamma);
    const S4 k2 = rhs(axpy(s, hdt, k1), gamma);
    const S4 k3 = rhs(axpy(s, hdt, k2), gamma);
    const S4 k4 = rhs(axpy(s, dt, k3), gamma);
    s.x = comb(s.x, dt6, k1.x, k2.x, k3.x, k4.x);
    s.y = comb(s.y, dt6, k1.y, k2.y, k3.y, k4.y);
    s.z = comb(s.z, dt6, k1.z, k2.z, k3.z, k4.z);
    s.w = comb(s.w, dt6, k1.w, k2.w, k3.w, k4.w);
}

}  // namespace

// One thread per (frame, worker, system).  IR: m x 2n x 4 doubles (the recorded states of LHCS_m of each frame).
__global__ void __launch_bounds__(64) lhcs_kernel(const double *__restrict__ IR, double gamma, uint32_t n, Geom g, uint32_t m,
                                                  uint16_t *D, uint8_t *B, uint32_t *status) {
    const uint32_t L = 2u * n, total = m * L;
    uint32_t t = blockIdx.x * blockDim.x + threadIdx.x;
    const bool live = t < total;
    if (!live) t = total - 1u;  // keeps the warp's shuffles and loop bounds well defined; writes nothing
    const uint32_t f = t / L, gs = t - f * L, wk = gs >> 1, k = gs & 1u;
    const double *ir = IR + (size_t)f * L * 4u;
    // skewed fetch (reading Q4): system g takes x of record g, y of g+1, z of g+2, w of g+3 (mod 2n)
    S4 s;
    s.x = ir[4u * gs + 0u];
    s.y = ir[4u * ((gs + 1u) % L) + 1u];
    s.z = ir[4u * ((gs + 2u) % L) + 2u];
    s.w = ir[4u * ((gs + 3u) % L) + 3u];
    // the worker's slices (reading Q11)
    const uint64_t ND = 3ull * ((uint64_t)g.h + g.w);
    const uint64_t d0 = ((uint64_t)wk * ND) / n, d1 = ((uint64_t)(wk + 1u) * ND) / n;
    const uint64_t r0 = ((uint64_t)wk * g.h) / n, r1 = ((uint64_t)(wk + 1u) * g.h) / n;
    const uint64_t lenD = 2ull * (d1 - d0), lenB = (r1 - r0) * g.row_bytes;
    uint8_t *pD = reinterpret_cast<uint8_t *>(D + (size_t)f * g.nD + d0);
    uint8_t *pB = B + (size_t)f * g.frame_bytes + r0 * g.row_bytes;
    const uint32_t itD = (uint32_t)((lenD + 23u) / 24u), itB = (uint32_t)((lenB + 23u) / 24u);
    const uint32_t iters = __reduce_max_sync(0xffffffffu, itD + itB);  // the warp steps together; surplus steps write nothing
    const uint64_t M48 = 0xFFFFFFFFFFFFull;
    for (uint32_t it = 0; it < iters; ++it) {
        rk4(s, gamma);
        const uint64_t bx = (uint64_t)__double_as_longlong(s.x) & M48, by = (uint64_t)__double_as_longlong(s.y) & M48;
        const uint64_t bz = (uint64_t)__double_as_longlong(s.z) & M48, bw = (uint64_t)__double_as_longlong(s.w) & M48;
        const uint64_t ex = bx ^ __shfl_xor_sync(0xffffffffu, bx, 1), ey = by ^ __shfl_xor_sync(0xffffffffu, by, 1);
        const uint64_t ez = bz ^ __shfl_xor_sync(0xffffffffu, bz, 1), ew = bw ^ __shfl_xor_sync(0xffffffffu, bw, 1);
        if (k != 0u || !live || it >= itD + itB) continue;
        const uint64_t o[3] = {ex | (ey << 48), (ey >> 16) | (ez << 32), (ez >> 32) | (ew << 16)};  // 24 bytes, little-endian
        uint8_t *p;
        uint64_t left;
        if (it < itD) { p = pD + 24ull * it; left = lenD - 24ull * it; }
        else { p = pB + 24ull * (it - itD); left = lenB - 24ull * (it - itD); }
        if (left >= 24u && (reinterpret_cast<uintptr_t>(p) & 7u) == 0u) {
            uint64_t *q = reinterpret_cast<uint64_t *>(p);
            q[0] = o[0]; q[1] = o[1]; q[2] = o[2];
        } else {
            const uint32_t nb = left < 24u ? (uint32_t)left : 24u;
            for (uint32_t b = 0; b < nb; ++b) p[b] = (uint8_t)(o[b >> 3] >> (8u * (b & 7u)));
        }
    }
    const bool fin = isfinite(s.x) && isfinite(s.y) && isfinite(s.z) && isfinite(s.w);
    if (live && !fin) atomicOr(status, 1u);
}

cudaError_t derive_device(const Geom &g, const double *d_IR, double gamma, uint32_t n, size_t m, uint16_t *d_D, uint8_t *d_B,
                          uint32_t *d_status, cudaStream_t st) {
    const uint32_t total = (uint32_t)(m * 2u * n);
    if (!total) return cudaSuccess;
    // 32 threads per CTA: the chains are serial, so spread the few warps over as many SMs as possible
    lhcs_kernel<<<(total + 31u) / 32u, 32, 0, st>>>(d_IR, gamma, n, g, (uint32_t)m, d_D, d_B, d_status);
    return cudaGetLastError();
}

}  // namespace vk
