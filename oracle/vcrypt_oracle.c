/*
 * oracle/vcrypt_oracle.c -- plain, slow, single-threaded CPU oracle.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may build, load or call
 * this file.  It shares no code, header, table or helper with the product
 * library (paper_2505_07158_b200/csrc/), and the product never falls back
 * to it.
 *
 * What it is: the protocol of "Real-Time Bit-Level Encryption of Full
 * High-Definition Video Without Diffusion" written out step by
 * step in the paper's own order and notation -- Algorithm 1 (main thread,
 * PAPER.md:85), Algorithm 2 (worker, :88-110), Algorithms 3-7 (GPU threads,
 * :85, :113-156) on EXPLICIT 0/1 bit matrices M_t^c / M_e^c of size 8w x h,
 * and the inverse (:79).  No blocking, fusion or re-ordering.  Where the
 * paper is silent the readings are those of SURVEY.md section 8(c)
 * (Q1..Q17), repeated in DESIGN.md and cited next to each function below.
 *
 * Parity status of each part:
 *   SHA-256 ............. pinned (FIPS 180-4 vectors, hashlib, constants
 *                         re-derived from cube/square roots of primes)
 *   frame hash H ........ pinned (n=1 == SHA-256(frame), XOR-combine)
 *   Algorithms 3-7 ...... pinned (numpy unpackbits/roll reduction, brute
 *                         force on 4x4, bijectivity, invariants)
 *   reconstruction, LHCS iteration, D/B byte layout:
 *                         PARITY UNPINNED against the authors' code (the
 *                         paper prints no vector and fixes no integrator,
 *                         bound u, byte order or burn-in).  Pinned only to
 *                         the mathematics: RK4 order-4 convergence against
 *                         a high-accuracy ODE solve, IEEE field invariants
 *                         of the reconstruction, -O0 == -O2 bit patterns.
 *
 * Arithmetic: IEEE-754 binary64, round-to-nearest-even, no FMA contraction
 * (build with -ffp-contract=off, never -ffast-math), expression order as
 * written.  Bytes of a double are taken arithmetically from its uint64 bit
 * pattern so the result does not depend on host endianness.
 *
 * Build:  gcc -O2 -ffp-contract=off -fno-fast-math -std=c99 -shared -fPIC \
 *             -o oracle/liboracle.so oracle/vcrypt_oracle.c -lm
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* ------------------------------------------------------------------------
 * Constants of the SURVEY.md 8(c) reading.
 * ---------------------------------------------------------------------- */
#define ORC_DT 0.005       /* Q3: classical RK4 step                     */
#define ORC_N0 20000       /* Q5: one-off key whitening steps at init    */
#define ORC_KM 16          /* Q4: RK4 steps of LHCS_m per recorded state */
#define ORC_U 40u          /* Q2: upper bound u_x = u_y = u_z = u_w      */

#define ORC_OK 0
#define ORC_E_ARG (-1)
#define ORC_E_NOMEM (-2)
#define ORC_E_NONFINITE (-3)

/* ========================================================================
 * SHA-256, FIPS 180-4 sections 4.1.2, 4.2.2, 5.1.1, 5.3.3, 6.2.2, written
 * as in the standard (message schedule W_t, working variables a..h).
 * PAPER.md:45 "each T_w^i computing the SHA-256 hash h_i".
 * ====================================================================== */
static const uint32_t SHA_K[64] = {
    0x428a2f98u, 0x71374491u, 0xb5c0fbcfu, 0xe9b5dba5u, 0x3956c25bu, 0x59f111f1u, 0x923f82a4u, 0xab1c5ed5u,
    0xd807aa98u, 0x12835b01u, 0x243185beu, 0x550c7dc3u, 0x72be5d74u, 0x80deb1feu, 0x9bdc06a7u, 0xc19bf174u,
    0xe49b69c1u, 0xefbe4786u, 0x0fc19dc6u, 0x240ca1ccu, 0x2de92c6fu, 0x4a7484aau, 0x5cb0a9dcu, 0x76f988dau,
    0x983e5152u, 0xa831c66du, 0xb00327c8u, 0xbf597fc7u, 0xc6e00bf3u, 0xd5a79147u, 0x06ca6351u, 0x14292967u,
    0x27b70a85u, 0x2e1b2138u, 0x4d2c6dfcu, 0x53380d13u, 0x650a7354u, 0x766a0abbu, 0x81c2c92eu, 0x92722c85u,
    0xa2bfe8a1u, 0xa81a664bu, 0xc24b8b70u, 0xc76c51a3u, 0xd192e819u, 0xd6990624u, 0xf40e3585u, 0x106aa070u,
    0x19a4c116u, 0x1e376c08u, 0x2748774cu, 0x34b0bcb5u, 0x391c0cb3u, 0x4ed8aa4au, 0x5b9cca4fu, 0x682e6ff3u,
    0x748f82eeu, 0x78a5636fu, 0x84c87814u, 0x8cc70208u, 0x90befffau, 0xa4506cebu, 0xbef9a3f7u, 0xc67178f2u};

static const uint32_t SHA_H0[8] = {0x6a09e667u, 0xbb67ae85u, 0x3c6ef372u, 0xa54ff53au,
                                   0x510e527fu, 0x9b05688cu, 0x1f83d9abu, 0x5be0cd19u};

/* exported so the tests can re-derive the constants from first principles */
const uint32_t *orc_sha256_k(void) { return SHA_K; }
const uint32_t *orc_sha256_h0(void) { return SHA_H0; }

static uint32_t rotr32(uint32_t x, unsigned n) { return (x >> n) | (x << (32u - n)); }

static void sha256_block(uint32_t Hs[8], const uint8_t blk[64]) {
    uint32_t W[64];
    uint32_t a, b, c, d, e, f, g, h;
    int t;
    for (t = 0; t < 16; ++t)
        W[t] = ((uint32_t)blk[4 * t] << 24) | ((uint32_t)blk[4 * t + 1] << 16) |
               ((uint32_t)blk[4 * t + 2] << 8) | (uint32_t)blk[4 * t + 3];
    for (t = 16; t < 64; ++t) {
        uint32_t s0 = rotr32(W[t - 15], 7) ^ rotr32(W[t - 15], 18) ^ (W[t - 15] >> 3);
        uint32_t s1 = rotr32(W[t - 2], 17) ^ rotr32(W[t - 2], 19) ^ (W[t - 2] >> 10);
        W[t] = s1 + W[t - 7] + s0 + W[t - 16];
    }
    a = Hs[0]; b = Hs[1]; c = Hs[2]; d = Hs[3];
    e = Hs[4]; f = Hs[5]; g = Hs[6]; h = Hs[7];
    for (t = 0; t < 64; ++t) {
        uint32_t S1 = rotr32(e, 6) ^ rotr32(e, 11) ^ rotr32(e, 25);
        uint32_t ch = (e & f) ^ (~e & g);
        uint32_t T1 = h + S1 + ch + SHA_K[t] + W[t];
        uint32_t S0 = rotr32(a, 2) ^ rotr32(a, 13) ^ rotr32(a, 22);
        uint32_t maj = (a & b) ^ (a & c) ^ (b & c);
        uint32_t T2 = S0 + maj;
        h = g; g = f; f = e; e = d + T1;
        d = c; c = b; b = a; a = T1 + T2;
    }
    Hs[0] += a; Hs[1] += b; Hs[2] += c; Hs[3] += d;
    Hs[4] += e; Hs[5] += f; Hs[6] += g; Hs[7] += h;
}

void orc_sha256(const uint8_t *msg, size_t len, uint8_t out[32]) {
    uint32_t Hs[8];
    uint8_t tail[128];
    size_t full = len / 64, rem = len % 64, i, tl;
    uint64_t bitlen = (uint64_t)len * 8u;
    memcpy(Hs, SHA_H0, sizeof Hs);
    for (i = 0; i < full; ++i) sha256_block(Hs, msg + 64 * i);
    /* padding, FIPS 180-4 section 5.1.1: 0x80, zeros, 64-bit big-endian length */
    memset(tail, 0, sizeof tail);
    if (rem) memcpy(tail, msg + 64 * full, rem);
    tail[rem] = 0x80;
    tl = (rem < 56) ? 64 : 128;
    for (i = 0; i < 8; ++i) tail[tl - 1 - i] = (uint8_t)(bitlen >> (8 * i));
    sha256_block(Hs, tail);
    if (tl == 128) sha256_block(Hs, tail + 64);
    for (i = 0; i < 8; ++i) {
        out[4 * i] = (uint8_t)(Hs[i] >> 24);
        out[4 * i + 1] = (uint8_t)(Hs[i] >> 16);
        out[4 * i + 2] = (uint8_t)(Hs[i] >> 8);
        out[4 * i + 3] = (uint8_t)Hs[i];
    }
}

/* ========================================================================
 * Frame hash.  PAPER.md:45: T_m partitions the frame into sub-frames f_i,
 * each worker hashes its f_i, H = h_1 xor ... xor h_n.
 * Reading Q1: sub-frame m (0-based) = rows [floor(m*h/n), floor((m+1)*h/n))
 * of the tightly packed H x W x 3 buffer (a contiguous byte range, possibly
 * empty -> SHA-256 of the empty message).
 * ====================================================================== */
static size_t band_row(uint32_t m, uint32_t n, uint32_t h) {
    return (size_t)(((uint64_t)m * (uint64_t)h) / (uint64_t)n);
}

int orc_frame_hash(const uint8_t *frame, uint32_t w, uint32_t h, uint32_t n, uint8_t H[32]) {
    uint32_t m;
    int k;
    if (!frame || !H || n == 0 || w == 0 || h == 0) return ORC_E_ARG;
    memset(H, 0, 32);
    for (m = 0; m < n; ++m) {
        uint8_t hm[32];
        size_t r0 = band_row(m, n, h), r1 = band_row(m + 1, n, h);
        orc_sha256(frame + r0 * (size_t)w * 3u, (r1 - r0) * (size_t)w * 3u, hm);
        for (k = 0; k < 32; ++k) H[k] ^= hm[k];
    }
    return ORC_OK;
}

/* ========================================================================
 * LHCS, Eq. (1):  x' = sigma (y - x) + w,  y' = rho x - y - x z,
 * z' = x y - beta z,  w' = -y z + gamma w,  sigma=10, rho=28, beta=8/3.
 * Reading Q3 (paper does not say how the ODE is iterated): classical RK4,
 * dt = 0.005, with the normative expression order of SURVEY.md 8(c) step 10.
 * ====================================================================== */
static void lhcs_f(const double s[4], double gamma, double d[4]) {
    const double x = s[0], y = s[1], z = s[2], w = s[3];
    d[0] = 10.0 * (y - x) + w;
    d[1] = (28.0 * x - y) - x * z;
    d[2] = x * y - (8.0 / 3.0) * z;
    d[3] = (-(y * z)) + gamma * w;
}

void orc_lhcs_rhs(const double s[4], double gamma, double d[4]) { lhcs_f(s, gamma, d); }

void orc_rk4_step(double s[4], double gamma) {
    const double dt = ORC_DT;
    const double hdt = 0.5 * ORC_DT;
    const double dt6 = ORC_DT / 6.0;
    double k1[4], k2[4], k3[4], k4[4], t[4];
    int i;
    lhcs_f(s, gamma, k1);
    for (i = 0; i < 4; ++i) t[i] = s[i] + hdt * k1[i];
    lhcs_f(t, gamma, k2);
    for (i = 0; i < 4; ++i) t[i] = s[i] + hdt * k2[i];
    lhcs_f(t, gamma, k3);
    for (i = 0; i < 4; ++i) t[i] = s[i] + dt * k3[i];
    lhcs_f(t, gamma, k4);
    for (i = 0; i < 4; ++i) s[i] = s[i] + dt6 * (((k1[i] + 2.0 * k2[i]) + 2.0 * k3[i]) + k4[i]);
}

static uint64_t f64_bits(double v) {
    uint64_t b;
    memcpy(&b, &v, 8);
    return b;
}
static double bits_f64(uint64_t b) {
    double v;
    memcpy(&v, &b, 8);
    return v;
}

/* ========================================================================
 * Initial-condition reconstruction, PAPER.md:55 and Fig. 1(a): "an integer
 * via XOR between the two least significant bytes of x0 and two bytes of H,
 * followed by a modulo by the upper bound u_x; a decimal through XOR between
 * the six least significant bytes of the fractional part of x0 and bytes
 * from H; finally, combining".  Eight hash bytes per variable.
 * Reading Q2: |v|; integer part's low 16 bits XOR (hb[0] | hb[1]<<8), mod
 * u=40; IEEE bit pattern of the fractional part XOR the 48-bit little-endian
 * integer hb[2..7] (mantissa bits 0..47 only); one IEEE add.
 * ====================================================================== */
double orc_reconstruct(double v, const uint8_t hb[8]) {
    double a = fabs(v);
    double fl = floor(a);
    uint64_t ip = (uint64_t)fl;
    double fr = a - fl;
    uint64_t I = ((ip & 0xFFFFu) ^ ((uint64_t)hb[0] | ((uint64_t)hb[1] << 8))) % ORC_U;
    uint64_t m48 = (uint64_t)hb[2] | ((uint64_t)hb[3] << 8) | ((uint64_t)hb[4] << 16) |
                   ((uint64_t)hb[5] << 24) | ((uint64_t)hb[6] << 32) | ((uint64_t)hb[7] << 40);
    uint64_t bits = f64_bits(fr) ^ m48;
    return (double)I + bits_f64(bits);
}

/* ========================================================================
 * Context = the state Algorithm 1 carries from frame to frame: the last
 * LHCS_m record (x_2n, y_2n, z_2n, w_2n), gamma, n, w, h.
 * ====================================================================== */
typedef struct orc_ctx {
    double S[4];
    double gamma;
    uint32_t n, w, h;
} orc_ctx;

static int all_finite(const double s[4]) {
    return isfinite(s[0]) && isfinite(s[1]) && isfinite(s[2]) && isfinite(s[3]);
}

/* Algorithm 1 inputs: n, x0, y0, z0, w0, gamma, w, h.
 * Reading Q5: the user key is advanced N0 = 20000 RK4 steps once. */
int orc_init(orc_ctx **out, double x0, double y0, double z0, double w0, double gamma, uint32_t n,
             uint32_t w, uint32_t h) {
    orc_ctx *c;
    int k;
    if (!out || n == 0 || w == 0 || h == 0) return ORC_E_ARG;
    if (!(gamma >= -1.52 && gamma <= -0.06)) return ORC_E_ARG;
    c = (orc_ctx *)malloc(sizeof *c);
    if (!c) return ORC_E_NOMEM;
    c->S[0] = x0; c->S[1] = y0; c->S[2] = z0; c->S[3] = w0;
    c->gamma = gamma; c->n = n; c->w = w; c->h = h;
    if (!all_finite(c->S)) { free(c); return ORC_E_ARG; }
    for (k = 0; k < ORC_N0; ++k) orc_rk4_step(c->S, gamma);
    if (!all_finite(c->S)) { free(c); return ORC_E_NONFINITE; }
    *out = c;
    return ORC_OK;
}

void orc_destroy(orc_ctx *c) { free(c); }
void orc_get_state(const orc_ctx *c, double S[4]) { memcpy(S, c->S, sizeof c->S); }
void orc_set_state(orc_ctx *c, const double S[4]) { memcpy(c->S, S, sizeof c->S); }
size_t orc_num_D(const orc_ctx *c) { return 3u * ((size_t)c->h + c->w); }
size_t orc_num_B(const orc_ctx *c) { return 3u * (size_t)c->h * c->w; }

/* bytes(sys): for x, y, z, w in that order, bytes 0..5 of the little-endian
 * IEEE-754 encoding = mantissa bits 0..47 ("six bytes from the
 * mantissa portion of each iteration result"; reading Q9). */
static void state_bytes(const double s[4], uint8_t e[24]) {
    int v, k;
    for (v = 0; v < 4; ++v) {
        uint64_t b = f64_bits(s[v]);
        for (k = 0; k < 6; ++k) e[6 * v + k] = (uint8_t)((b >> (8 * k)) & 0xFFu);
    }
}

/* Algorithm 1 steps 7-14 + Algorithm 2 steps 5-10 for one frame whose hash
 * is H.  Writes IR (2n x 4 doubles) if IR_out != NULL.  Advances the chain.
 *   D layout (reading Q11 / 8(c) step 7): D[c*(h+w) + i] = d_h(i,c) for i<h,
 *   D[c*(h+w) + h + j] = d_v(j,c).   B[(i*w + j)*3 + c] masks pixel (i,j,c). */
int orc_derive(orc_ctx *c, const uint8_t H[32], uint16_t *D, uint8_t *B, double *IR_out) {
    const uint32_t n = c->n, L = 2u * c->n;
    const size_t ND = orc_num_D(c);
    double s0[4], cur[4];
    double *IR;
    uint32_t g, m;
    int v, k;
    if (!H || !D || !B) return ORC_E_ARG;
    IR = (double *)malloc((size_t)L * 4u * sizeof(double));
    if (!IR) return ORC_E_NOMEM;

    /* Algo 1 steps 7-11: reconstruct (x0,y0,z0,w0) from the base state and H;
     * variable m uses hash bytes H[8m .. 8m+7]. */
    for (v = 0; v < 4; ++v) s0[v] = orc_reconstruct(c->S[v], H + 8 * v);

    /* Algo 1 steps 12-13: iterate LHCS_m, record IR = {x_1..w_1, ..., x_2n..w_2n};
     * reading Q4: one record every K_m = 16 RK4 steps. */
    memcpy(cur, s0, sizeof cur);
    for (g = 0; g < L; ++g) {
        for (k = 0; k < ORC_KM; ++k) orc_rk4_step(cur, c->gamma);
        memcpy(IR + 4u * g, cur, sizeof cur);
    }
    if (!all_finite(cur)) { free(IR); return ORC_E_NONFINITE; }

    /* Algorithm 2 for each worker m (sequentially here). */
    for (m = 0; m < n; ++m) {
        double sys[2][4];
        uint8_t e0[24], e1[24], e[24];
        size_t d0 = (size_t)(((uint64_t)m * ND) / n), d1 = (size_t)(((uint64_t)(m + 1) * ND) / n);
        size_t b0 = band_row(m, n, c->h) * (size_t)c->w * 3u;
        size_t b1 = band_row(m + 1, n, c->h) * (size_t)c->w * 3u;
        size_t nd = d1 - d0, nb = b1 - b0, itD = (nd + 11u) / 12u, itB = (nb + 23u) / 24u, it, q;
        int s;
        /* step 5: "Fetch iteration results from IR"; reading Q4 (skewed fetch):
         * system g = 2m+s takes x from record g, y from g+1, z from g+2, w from g+3 (mod 2n). */
        for (s = 0; s < 2; ++s) {
            g = 2u * m + (uint32_t)s;
            sys[s][0] = IR[4u * g + 0];
            sys[s][1] = IR[4u * ((g + 1u) % L) + 1];
            sys[s][2] = IR[4u * ((g + 2u) % L) + 2];
            sys[s][3] = IR[4u * ((g + 3u) % L) + 3];
        }
        /* steps 6-8: shift distances, d = two bytes little-endian (Q8), XOR of the
         * two systems; first ceil(nd/12) iterations (Q10: disjoint from B's). */
        for (it = 0; it < itD; ++it) {
            orc_rk4_step(sys[0], c->gamma);
            orc_rk4_step(sys[1], c->gamma);
            state_bytes(sys[0], e0);
            state_bytes(sys[1], e1);
            for (k = 0; k < 24; ++k) e[k] = e0[k] ^ e1[k];
            for (q = 0; q < 12; ++q) {
                size_t idx = it * 12u + q;
                if (idx < nd) D[d0 + idx] = (uint16_t)((uint16_t)e[2 * q] | ((uint16_t)e[2 * q + 1] << 8));
            }
        }
        /* steps 9-10: bytes, the following ceil(nb/24) iterations. */
        for (it = 0; it < itB; ++it) {
            orc_rk4_step(sys[0], c->gamma);
            orc_rk4_step(sys[1], c->gamma);
            state_bytes(sys[0], e0);
            state_bytes(sys[1], e1);
            for (q = 0; q < 24; ++q) {
                size_t idx = it * 24u + q;
                if (idx < nb) B[b0 + idx] = (uint8_t)(e0[q] ^ e1[q]);
            }
        }
        if (!all_finite(sys[0]) || !all_finite(sys[1])) { free(IR); return ORC_E_NONFINITE; }
    }
    /* x_2n..w_2n of this frame are the base state for the next. */
    memcpy(c->S, IR + 4u * (L - 1u), sizeof c->S);
    if (IR_out) memcpy(IR_out, IR, (size_t)L * 4u * sizeof(double));
    free(IR);
    return ORC_OK;
}

/* ========================================================================
 * Algorithms 3-7 on explicit bit matrices.  One matrix per channel,
 * M[c][i][p], i = 0..h-1 (row), p = 0..8w-1 (bit column), one byte per bit.
 * Each function is "all GPU threads T_g^c(i,j) execute Algorithm k".
 * ====================================================================== */
#define MIDX(c, i, p) (((size_t)(c) * h + (size_t)(i)) * (8u * (size_t)w) + (size_t)(p))

/* Algorithm 3: M_t^c(i, 8j+k) <- (F^c(i,j) >> k) AND 1. */
void orc_bit_extract(const uint8_t *F, uint32_t w, uint32_t h, uint8_t *Mt) {
    uint32_t i, j, c, k;
    for (c = 0; c < 3; ++c)
        for (i = 0; i < h; ++i)
            for (j = 0; j < w; ++j) {
                uint8_t temp = F[((size_t)i * w + j) * 3u + c];
                for (k = 0; k < 8; ++k) {
                    Mt[MIDX(c, i, 8u * j + k)] = temp & 0x01u;
                    temp = (uint8_t)(temp >> 1);
                }
            }
}

/* Algorithm 4 (Eq. 2 :67):
 *   M_e^c(i, (8j+k + (d_h MOD 8w)) MOD 8w) <- M_t^c(i, 8j+k),  d_h = D[c(h+w)+i].
 * inverse != 0 applies the inverse map (M_e^c(i, 8j+k) <- M_t^c(i, dest)). */
void orc_hshift(const uint8_t *Mt, uint8_t *Me, uint32_t w, uint32_t h, const uint16_t *D, int inverse) {
    uint32_t i, j, c, k;
    const uint64_t W8 = 8u * (uint64_t)w;
    for (c = 0; c < 3; ++c)
        for (i = 0; i < h; ++i) {
            uint64_t dh = D[(size_t)c * (h + w) + i];
            for (j = 0; j < w; ++j)
                for (k = 0; k < 8; ++k) {
                    uint64_t src = 8u * (uint64_t)j + k;
                    uint64_t dst = (src + (dh % W8)) % W8;
                    if (!inverse) Me[MIDX(c, i, dst)] = Mt[MIDX(c, i, src)];
                    else Me[MIDX(c, i, src)] = Mt[MIDX(c, i, dst)];
                }
        }
}

/* Algorithm 5 (Eq. 3 :72 with reading Q7):
 *   M_e^c((i + (d_v MOD h)) MOD h, 8j+k) <- M_t^c(i, 8j+k),  d_v = D[c(h+w)+h+j]
 * (reading Q6: one d_v per pixel column and channel, all 8 bit columns move together). */
void orc_vshift(const uint8_t *Mt, uint8_t *Me, uint32_t w, uint32_t h, const uint16_t *D, int inverse) {
    uint32_t i, j, c, k;
    for (c = 0; c < 3; ++c)
        for (i = 0; i < h; ++i)
            for (j = 0; j < w; ++j) {
                uint64_t dv = D[(size_t)c * (h + w) + h + j];
                uint64_t di = ((uint64_t)i + (dv % h)) % h;
                for (k = 0; k < 8; ++k) {
                    if (!inverse) Me[MIDX(c, di, 8u * j + k)] = Mt[MIDX(c, i, 8u * j + k)];
                    else Me[MIDX(c, i, 8u * j + k)] = Mt[MIDX(c, di, 8u * j + k)];
                }
            }
}

/* Algorithm 6: b = B(i,j,c);
 *   M_e^c(i, 8j+k) <- M_t^c(i, 8j+k) XOR (b AND 1); b <- b >> 1. */
void orc_xor_bits(const uint8_t *Mt, uint8_t *Me, uint32_t w, uint32_t h, const uint8_t *B) {
    uint32_t i, j, c, k;
    for (c = 0; c < 3; ++c)
        for (i = 0; i < h; ++i)
            for (j = 0; j < w; ++j) {
                uint8_t b = B[((size_t)i * w + j) * 3u + c];
                for (k = 0; k < 8; ++k) {
                    uint8_t temp = b & 0x01u;
                    Me[MIDX(c, i, 8u * j + k)] = Mt[MIDX(c, i, 8u * j + k)] ^ temp;
                    b = (uint8_t)(b >> 1);
                }
            }
}

/* Algorithm 7: for k = 7 down to 0:
 *   F_e <- F_e OR M_e^c(i, 8j+k); if k != 0: F_e <- F_e << 1. */
void orc_pack(const uint8_t *Me, uint32_t w, uint32_t h, uint8_t *Fe) {
    uint32_t i, j, c;
    int k;
    for (c = 0; c < 3; ++c)
        for (i = 0; i < h; ++i)
            for (j = 0; j < w; ++j) {
                uint8_t v = 0;
                for (k = 7; k >= 0; --k) {
                    v = (uint8_t)(v | Me[MIDX(c, i, 8u * j + (uint32_t)k)]);
                    if (k != 0) v = (uint8_t)(v << 1);
                }
                Fe[((size_t)i * w + j) * 3u + c] = v;
            }
}

/* Algorithm 1 steps 16-20: "for k = 3..7: execute Algo k on all threads;
 * M_t^c <- M_e^c". */
int orc_confuse_xor(const uint8_t *Fo, uint32_t w, uint32_t h, const uint16_t *D, const uint8_t *B,
                    uint8_t *Fe) {
    size_t nbits = 3u * (size_t)h * 8u * (size_t)w;
    uint8_t *Mt = (uint8_t *)malloc(nbits), *Me = (uint8_t *)malloc(nbits);
    if (!Mt || !Me) { free(Mt); free(Me); return ORC_E_NOMEM; }
    orc_bit_extract(Fo, w, h, Mt);      /* Algo 3 */
    orc_hshift(Mt, Me, w, h, D, 0);     /* Algo 4 */
    memcpy(Mt, Me, nbits);
    orc_vshift(Mt, Me, w, h, D, 0);     /* Algo 5 */
    memcpy(Mt, Me, nbits);
    orc_xor_bits(Mt, Me, w, h, B);      /* Algo 6 */
    memcpy(Mt, Me, nbits);
    orc_pack(Me, w, h, Fe);             /* Algo 7 */
    free(Mt); free(Me);
    return ORC_OK;
}

/* Decryption = the inverse transformation: XOR, inverse vertical,
 * inverse horizontal, with the same D and B. */
int orc_unconfuse_xor(const uint8_t *Fe, uint32_t w, uint32_t h, const uint16_t *D, const uint8_t *B,
                      uint8_t *Fo) {
    size_t nbits = 3u * (size_t)h * 8u * (size_t)w;
    uint8_t *Mt = (uint8_t *)malloc(nbits), *Me = (uint8_t *)malloc(nbits);
    if (!Mt || !Me) { free(Mt); free(Me); return ORC_E_NOMEM; }
    orc_bit_extract(Fe, w, h, Mt);
    orc_xor_bits(Mt, Me, w, h, B);
    memcpy(Mt, Me, nbits);
    orc_vshift(Mt, Me, w, h, D, 1);
    memcpy(Mt, Me, nbits);
    orc_hshift(Mt, Me, w, h, D, 1);
    orc_pack(Me, w, h, Fo);
    free(Mt); free(Me);
    return ORC_OK;
}

/* ========================================================================
 * Algorithm 1 as a whole, and its receiver-side inverse (the
 * receiver holds the key and n, and is sent F_e and H for every frame).
 * frames: nframes tightly packed H x W x 3 buffers; hashes: nframes x 32.
 * ====================================================================== */
int orc_encrypt_frames(orc_ctx *c, const uint8_t *frames, size_t nframes, uint8_t *cipher, uint8_t *hashes) {
    const size_t fb = orc_num_B(c);
    uint16_t *D = (uint16_t *)malloc(orc_num_D(c) * sizeof(uint16_t));
    uint8_t *B = (uint8_t *)malloc(fb);
    size_t f;
    int rc = ORC_OK;
    if (!D || !B) { free(D); free(B); return ORC_E_NOMEM; }
    for (f = 0; f < nframes && rc == ORC_OK; ++f) {
        uint8_t *H = hashes + 32u * f;
        rc = orc_frame_hash(frames + f * fb, c->w, c->h, c->n, H);
        if (rc == ORC_OK) rc = orc_derive(c, H, D, B, NULL);
        if (rc == ORC_OK) rc = orc_confuse_xor(frames + f * fb, c->w, c->h, D, B, cipher + f * fb);
    }
    free(D); free(B);
    return rc;
}

int orc_decrypt_frames(orc_ctx *c, const uint8_t *cipher, const uint8_t *hashes, size_t nframes, uint8_t *plain) {
    const size_t fb = orc_num_B(c);
    uint16_t *D = (uint16_t *)malloc(orc_num_D(c) * sizeof(uint16_t));
    uint8_t *B = (uint8_t *)malloc(fb);
    size_t f;
    int rc = ORC_OK;
    if (!D || !B) { free(D); free(B); return ORC_E_NOMEM; }
    for (f = 0; f < nframes && rc == ORC_OK; ++f) {
        rc = orc_derive(c, hashes + 32u * f, D, B, NULL);
        if (rc == ORC_OK) rc = orc_unconfuse_xor(cipher + f * fb, c->w, c->h, D, B, plain + f * fb);
    }
    free(D); free(B);
    return rc;
}
