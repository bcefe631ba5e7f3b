// vx_blake3.cuh -- BLAKE3 keyed hash of one short nonce, whole state in registers (sm_100a).
//
// What it computes: PAPER.md L41-43 (I-A) / L91 (III-B): "each thread independently converts its
// global ID to a little-endian nonce, computes a Blake3 keyed hash".  One compression of one
// 64-byte block (BLAKE3 spec, paper ref [4]): 7 rounds x 8 G over a 16-word state; only output
// words 0 and 1 are needed (HASH_SIZE = 8, reading A4), so the tail of round 7 that does not feed
// v0, v1, v8, v9 is never emitted.
//
// B200 specifics (differs from the paper's one-thread-per-nonce V100 kernel only in the details):
//   * the message block is all zero except word 0 (and the low byte of word 1 when NONCE_SIZE = 5),
//     so the schedule below is resolved at compile time and every "+ 0" disappears;
//   * columns 1..3 of round 1 do not depend on the nonce: the host folds them once per plot into
//     VxHashConst (12 state words) -- 3 of the 56 G functions leave the device entirely;
//   * the key and those words arrive as kernel parameters, i.e. in the constant bank, and are
//     read with uniform-register / constant-operand instructions (the paper's __constant__ key);
//   * rotations are single funnel shifts (SHF.R.W) or byte permutes (PRMT) on the ALU pipe, adds
//     are left to ptxas to place on the FMA pipe (IMAD.IADD) -- see DESIGN.md "hash kernel".
#pragma once
#include <stdint.h>

struct VxHashConst {
    uint32_t k[8];     // key words (little-endian), the chaining value
    uint32_t s04;      // k0 + k4, first add of column 0
    uint32_t col[12];  // v1,v5,v9,v13, v2,v6,v10,v14, v3,v7,v11,v15 after round-1 columns 1..3
    uint32_t block_len; // NONCE_SIZE
};

#define VX_IV0 0x6A09E667u
#define VX_IV1 0xBB67AE85u
#define VX_IV2 0x3C6EF372u
#define VX_IV3 0xA54FF53Au
#define VX_FLAGS 27u /* CHUNK_START | CHUNK_END | ROOT | KEYED_HASH */

#if defined(__CUDACC__)

__device__ __forceinline__ uint32_t vx_rotr(uint32_t x, int r) { return __funnelshift_r(x, x, r); }

// One G with both message words possibly absent (compile-time zero).
#define VX_G(a, b, c, d, x, y)            \
    do {                                  \
        a = a + b + (x);                  \
        d = vx_rotr(d ^ a, 16);           \
        c = c + d;                        \
        b = vx_rotr(b ^ c, 12);           \
        a = a + b + (y);                  \
        d = vx_rotr(d ^ a, 8);            \
        c = c + d;                        \
        b = vx_rotr(b ^ c, 7);            \
    } while (0)

// Message schedule: after r applications of the BLAKE3 permutation P, slot i of round r holds
// original word idx[r][i].  Generated from P at compile time (no hand-derived table), so that
// vx_msg<R, SLOT> folds to m0, m1 or the literal 0.
struct VxSchedule {
    int idx[7][16];
    __host__ __device__ constexpr VxSchedule() : idx{} {
        const int P[16] = {2, 6, 3, 10, 7, 0, 4, 13, 1, 11, 12, 5, 9, 14, 15, 8};
        for (int i = 0; i < 16; i++) idx[0][i] = i;
        for (int r = 1; r < 7; r++)
            for (int i = 0; i < 16; i++) idx[r][i] = idx[r - 1][P[i]];
    }
};

// (m2 is the compile-time constant 0 everywhere except in the 10-byte pair hash of the re-keying)
template <int R, int SLOT>
__device__ __forceinline__ uint32_t vx_msg(uint32_t m0, uint32_t m1, uint32_t m2)
{
    constexpr VxSchedule S{};
    constexpr int w = S.idx[R][SLOT];
    return w == 0 ? m0 : (w == 1 ? m1 : (w == 2 ? m2 : 0u));
}

template <int R>
__device__ __forceinline__ void vx_round(uint32_t (&v)[16], uint32_t m0, uint32_t m1, uint32_t m2 = 0u)
{
    VX_G(v[0], v[4], v[8], v[12], (vx_msg<R, 0>(m0, m1, m2)), (vx_msg<R, 1>(m0, m1, m2)));
    VX_G(v[1], v[5], v[9], v[13], (vx_msg<R, 2>(m0, m1, m2)), (vx_msg<R, 3>(m0, m1, m2)));
    VX_G(v[2], v[6], v[10], v[14], (vx_msg<R, 4>(m0, m1, m2)), (vx_msg<R, 5>(m0, m1, m2)));
    VX_G(v[3], v[7], v[11], v[15], (vx_msg<R, 6>(m0, m1, m2)), (vx_msg<R, 7>(m0, m1, m2)));
    VX_G(v[0], v[5], v[10], v[15], (vx_msg<R, 8>(m0, m1, m2)), (vx_msg<R, 9>(m0, m1, m2)));
    VX_G(v[1], v[6], v[11], v[12], (vx_msg<R, 10>(m0, m1, m2)), (vx_msg<R, 11>(m0, m1, m2)));
    VX_G(v[2], v[7], v[8], v[13], (vx_msg<R, 12>(m0, m1, m2)), (vx_msg<R, 13>(m0, m1, m2)));
    VX_G(v[3], v[4], v[9], v[14], (vx_msg<R, 14>(m0, m1, m2)), (vx_msg<R, 15>(m0, m1, m2)));
}

// H(n) as the big-endian u64 of the first 8 digest bytes (readings A4, A5).
// NONCE5 = false: m1 is the compile-time constant 0 (NONCE_SIZE = 4, K <= 32).
template <bool NONCE5>
__device__ __forceinline__ uint64_t vx_blake3_h(const VxHashConst &hc, uint32_t m0, uint32_t m1_in)
{
    const uint32_t m1 = NONCE5 ? m1_in : 0u;
    uint32_t v[16];
    // round 1, column 0: the only nonce-dependent column
    v[0] = hc.s04 + m0;                 // k0 + k4 + m0
    v[12] = vx_rotr(v[0], 16);          // v12 = counter low = 0
    v[8] = VX_IV0 + v[12];
    v[4] = vx_rotr(hc.k[4] ^ v[8], 12);
    v[0] = v[0] + v[4] + m1;
    v[12] = vx_rotr(v[12] ^ v[0], 8);
    v[8] = v[8] + v[12];
    v[4] = vx_rotr(v[4] ^ v[8], 7);
    // round 1, columns 1..3: folded on the host
    v[1] = hc.col[0]; v[5] = hc.col[1]; v[9] = hc.col[2];  v[13] = hc.col[3];
    v[2] = hc.col[4]; v[6] = hc.col[5]; v[10] = hc.col[6]; v[14] = hc.col[7];
    v[3] = hc.col[8]; v[7] = hc.col[9]; v[11] = hc.col[10]; v[15] = hc.col[11];
    // round 1, diagonals (message words 8..15 are zero)
    VX_G(v[0], v[5], v[10], v[15], 0u, 0u);
    VX_G(v[1], v[6], v[11], v[12], 0u, 0u);
    VX_G(v[2], v[7], v[8], v[13], 0u, 0u);
    VX_G(v[3], v[4], v[9], v[14], 0u, 0u);
    vx_round<1>(v, m0, m1);
    vx_round<2>(v, m0, m1);
    vx_round<3>(v, m0, m1);
    vx_round<4>(v, m0, m1);
    vx_round<5>(v, m0, m1);
    vx_round<6>(v, m0, m1);
    const uint32_t w0 = v[0] ^ v[8], w1 = v[1] ^ v[9];
    // digest bytes 0..7 = w0, w1 little-endian; H reads them big-endian
    return ((uint64_t)__byte_perm(w0, 0, 0x0123) << 32) | (uint64_t)__byte_perm(w1, 0, 0x0123);
}

// H2 of a pair of 5-byte nonces (re-keying, reading A19): the 10 message bytes nonce1 LE || nonce2 LE are
// the words m0, m1, m2; column 1 of round 1 then depends on the message (m2) and is computed here from
// the key instead of being taken from the host fold; columns 2 and 3 are the folded ones (hc.block_len = 10).
__device__ __forceinline__ uint64_t vx_blake3_h3(const VxHashConst &hc, uint32_t m0, uint32_t m1, uint32_t m2)
{
    uint32_t v[16];
    v[0] = hc.s04 + m0;
    v[12] = vx_rotr(v[0], 16);
    v[8] = VX_IV0 + v[12];
    v[4] = vx_rotr(hc.k[4] ^ v[8], 12);
    v[0] = v[0] + v[4] + m1;
    v[12] = vx_rotr(v[12] ^ v[0], 8);
    v[8] = v[8] + v[12];
    v[4] = vx_rotr(v[4] ^ v[8], 7);
    // column 1: G(v1, v5, v9, v13, m2, 0) with v1 = k1, v5 = k5, v9 = IV1, v13 = counter high = 0
    v[1] = hc.k[1]; v[5] = hc.k[5]; v[9] = VX_IV1; v[13] = 0u;
    VX_G(v[1], v[5], v[9], v[13], m2, 0u);
    v[2] = hc.col[4]; v[6] = hc.col[5]; v[10] = hc.col[6]; v[14] = hc.col[7];
    v[3] = hc.col[8]; v[7] = hc.col[9]; v[11] = hc.col[10]; v[15] = hc.col[11];
    VX_G(v[0], v[5], v[10], v[15], 0u, 0u);
    VX_G(v[1], v[6], v[11], v[12], 0u, 0u);
    VX_G(v[2], v[7], v[8], v[13], 0u, 0u);
    VX_G(v[3], v[4], v[9], v[14], 0u, 0u);
    vx_round<1>(v, m0, m1, m2);
    vx_round<2>(v, m0, m1, m2);
    vx_round<3>(v, m0, m1, m2);
    vx_round<4>(v, m0, m1, m2);
    vx_round<5>(v, m0, m1, m2);
    vx_round<6>(v, m0, m1, m2);
    const uint32_t w0 = v[0] ^ v[8], w1 = v[1] ^ v[9];
    return ((uint64_t)__byte_perm(w0, 0, 0x0123) << 32) | (uint64_t)__byte_perm(w1, 0, 0x0123);
}

#endif // __CUDACC__
