// host.hpp -- host subsystem of libvcrypt: sub-frame hashing, initial-condition reconstruction, LHCS_m chain
// and worker-system derivation of D and B (Algorithm 1 steps 4-14, Algorithm 2).
// Internal; the public boundary is include/vcrypt.h.
#pragma once
#include <stddef.h>
#include <stdint.h>

namespace vh {

// ---- constants of the method -------------------------------------------
constexpr double kDt = 0.005;      // Q3: classical RK4 step
constexpr int kWhiten = 20000;     // Q5: one-off RK4 steps applied to the key at init
constexpr int kRecordStride = 16;  // Q4: RK4 steps of LHCS_m per recorded quadruple of IR
constexpr uint64_t kBound = 40;    // Q2: upper bound u of a reconstructed integer part

// ---- SHA-256 (host_sha256.cpp) ------------------------------------------------------------------------------
bool cpu_has_shani();
void sha256(const uint8_t *msg, size_t len, uint8_t out[32], bool allow_simd);

// ---- scalar pieces (host_derive.cpp) ------------------------------------------------------------------------
void rk4_step(double s[4], double gamma);
double reconstruct(double v, const uint8_t hb[8]);
bool finite4(const double s[4]);

// Row band of sub-frame / worker m: rows [band_row(m), band_row(m+1)).
inline size_t band_row(uint32_t m, uint32_t n, uint32_t h) { return (size_t)(((uint64_t)m * h) / n); }

// Algorithm 1 steps 7-13 for one frame: reconstruct the four initial values from the base state S and the
// hash H, iterate LHCS_m, record IR (2n quadruples), move S to the last record.  Returns false if a state
// became non-finite (S is then left untouched).
bool chain_step(double S[4], double gamma, uint32_t n, const uint8_t H[32], double *IR);

// ---- worker systems (host_lhcs_*.cpp) -----------------------------------------------------------------------
// One worker = Algorithm 2 steps 5-10: two LHCS seeded from IR (skewed fetch), advanced in lock-step; every
// step yields 24 bytes (6 low bytes of x, y, z, w of system 0 XOR the same of system 1); the first
// ceil(nd/12) steps fill the worker's slice of D, the following ceil(nb/24) steps its slice of B.
struct WorkerSlice {
    double ic[2][4];  // initial conditions of the two systems
    uint16_t *D;      // slice of the frame's D
    size_t nd;
    uint8_t *B;       // slice of the frame's B
    size_t nb;
    bool flush_B;     // write the slice's cache lines back once it is complete (it goes to the GPU next, see host_lhcs_lanes.inc)
};

// Derives `count` workers (any count; lanes are padded internally).  isa: 0 scalar, 1 AVX2 (4 lanes),
// 2 AVX-512 (8 lanes).  Every isa produces the same bytes.  Returns false on a non-finite state.
bool derive_workers(const WorkerSlice *ws, size_t count, double gamma, int isa);
int best_isa();  // what this CPU supports
bool has_clflushopt();  // CPUID leaf 7 EBX bit 23 (the lane code flushes finished keystream slices only where this holds)

bool derive_workers_scalar(const WorkerSlice *ws, size_t count, double gamma);
bool derive_workers_avx2(const WorkerSlice *ws, size_t count, double gamma);
bool derive_workers_avx512(const WorkerSlice *ws, size_t count, double gamma);

// Fills the WorkerSlice array (n entries) for one frame from IR and the frame's D / B buffers.
void make_slices(const double *IR, uint32_t n, uint32_t w, uint32_t h, uint16_t *D, uint8_t *B, WorkerSlice *out);

}  // namespace vh
