// host_derive.cpp -- scalar pieces of the host derivation: RK4 step of the Lorenz hyper-chaotic system
// (Eq. 1), initial-condition reconstruction (Fig. 1(a)), the LHCS_m chain step
// (Algorithm 1 steps 7-13) and the split of a frame's D / B into worker slices (Algorithm 2,
// PAPER.md:88-110).  Must be compiled with -ffp-contract=off (no FMA contraction): the expression order below
// is the arithmetic.  Shares nothing with oracle/.
#if defined(__x86_64__)
#include <cpuid.h>
#endif
#include "host.hpp"

#include <cmath>
#include <cstring>

namespace vh {

namespace {
struct V4 {
    double x, y, z, w;
};

// Eq. 1 with sigma = 10, rho = 28, beta = 8/3.
inline V4 rhs(const V4 &s, double gamma) {
    V4 d;
    d.x = 10.0 * (s.y - s.x) + s.w;
    d.y = (28.0 * s.x - s.y) - s.x * s.z;
    d.z = s.x * s.y - (8.0 / 3.0) * s.z;
    d.w = (-(s.y * s.z)) + gamma * s.w;
    return d;
}
inline V4 axpy(const V4 &s, double a, const V4 &k) { return V4{s.x + a * k.x, s.y + a * k.y, s.z + a * k.z, s.w + a * k.w}; }
}  // namespace

void rk4_step(double s[4], double gamma) {
    const double dt = kDt, hdt = 0.5 * kDt, dt6 = kDt / 6.0;
    const V4 s0{s[0], s[1], s[2], s[3]};
    const V4 k1 = rhs(s0, gamma);
    const V4 k2 = rhs(axpy(s0, hdt, k1), gamma);
    const V4 k3 = rhs(axpy(s0, hdt, k2), gamma);
    const V4 k4 = rhs(axpy(s0, dt, k3), gamma);
    s[0] = s0.x + dt6 * (((k1.x + 2.0 * k2.x) + 2.0 * k3.x) + k4.x);
    s[1] = s0.y + dt6 * (((k1.y + 2.0 * k2.y) + 2.0 * k3.y) + k4.y);
    s[2] = s0.z + dt6 * (((k1.z + 2.0 * k2.z) + 2.0 * k3.z) + k4.z);
    s[3] = s0.w + dt6 * (((k1.w + 2.0 * k2.w) + 2.0 * k3.w) + k4.w);
}

bool finite4(const double s[4]) {
    return std::isfinite(s[0]) && std::isfinite(s[1]) && std::isfinite(s[2]) && std::isfinite(s[3]);
}

// integer part's two low bytes XOR two hash bytes, modulo the bound u; the fractional part's six
// low (mantissa) bytes XOR six hash bytes; the two are added.  |v| because states can be negative (reading Q2).
double reconstruct(double v, const uint8_t hb[8]) {
    const double a = std::fabs(v);
    const double fl = std::floor(a);
    const double fr = a - fl;  // exact
    const uint64_t ip = (uint64_t)fl;
    uint64_t hw;
    std::memcpy(&hw, hb, 8);  // little-endian host: hb[0] is the low byte
    const uint64_t I = ((ip ^ hw) & 0xFFFFu) % kBound;
    uint64_t fb;
    std::memcpy(&fb, &fr, 8);
    fb ^= hw >> 16;  // hb[2..7] onto mantissa bits 0..47
    double f2;
    std::memcpy(&f2, &fb, 8);
    return (double)I + f2;
}

bool chain_step(double S[4], double gamma, uint32_t n, const uint8_t H[32], double *IR) {
    double cur[4];
    for (int v = 0; v < 4; ++v) cur[v] = reconstruct(S[v], H + 8 * v);
    const uint32_t L = 2u * n;
    for (uint32_t g = 0; g < L; ++g) {
        for (int k = 0; k < kRecordStride; ++k) rk4_step(cur, gamma);
        std::memcpy(IR + 4u * g, cur, sizeof cur);
    }
    if (!finite4(cur)) return false;
    std::memcpy(S, cur, sizeof cur);
    return true;
}

void make_slices(const double *IR, uint32_t n, uint32_t w, uint32_t h, uint16_t *D, uint8_t *B, WorkerSlice *out) {
    const uint32_t L = 2u * n;
    const uint64_t ND = 3ull * ((uint64_t)h + w);
    const size_t rb = (size_t)w * 3u;
    for (uint32_t m = 0; m < n; ++m) {
        WorkerSlice &s = out[m];
        for (uint32_t k = 0; k < 2; ++k) {
            const uint32_t g = 2u * m + k;  // skewed fetch (reading Q4)
            s.ic[k][0] = IR[4u * g + 0];
            s.ic[k][1] = IR[4u * ((g + 1u) % L) + 1];
            s.ic[k][2] = IR[4u * ((g + 2u) % L) + 2];
            s.ic[k][3] = IR[4u * ((g + 3u) % L) + 3];
        }
        const size_t d0 = (size_t)(((uint64_t)m * ND) / n), d1 = (size_t)(((uint64_t)(m + 1) * ND) / n);
        const size_t b0 = band_row(m, n, h) * rb, b1 = band_row(m + 1, n, h) * rb;
        s.D = D + d0;
        s.nd = d1 - d0;
        s.B = B + b0;
        s.nb = b1 - b0;
        s.flush_B = false;
    }
}

int best_isa() {
#if defined(__x86_64__)
    static const int v = (__builtin_cpu_supports("avx512f") && __builtin_cpu_supports("avx512dq")) ? 2
                         : __builtin_cpu_supports("avx2")                                           ? 1
                                                                                                    : 0;
    return v;
#else
    return 0;
#endif
}

// CLFLUSHOPT is its own CPUID bit (leaf 7, sub-leaf 0, EBX bit 23), not implied by AVX2: Haswell and Broadwell have AVX2
// without it, and the lane code's flush (host_lhcs_lanes.inc) would be an illegal instruction there.
bool has_clflushopt() {
#if defined(__x86_64__)
    static const bool v = [] {
        unsigned a = 0, b = 0, c = 0, d = 0;
        return __get_cpuid_count(7, 0, &a, &b, &c, &d) != 0 && ((b >> 23) & 1u) != 0;
    }();
    return v;
#else
    return false;
#endif
}

bool derive_workers(const WorkerSlice *ws, size_t count, double gamma, int isa) {
#if defined(__x86_64__)
    if (isa >= 2) return derive_workers_avx512(ws, count, gamma);
    if (isa == 1) return derive_workers_avx2(ws, count, gamma);
#endif
    (void)isa;
    return derive_workers_scalar(ws, count, gamma);
}

}  // namespace vh
