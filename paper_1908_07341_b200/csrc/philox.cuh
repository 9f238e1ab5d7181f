// philox.cuh -- Philox4x32-10 in registers for the shaken-dynamics kernels (device side of libshaken).
//
// The generator is the public counter-based algorithm of Salmon, Moraes, Dror, Shaw (SC'11): ten rounds of
//     (c0, c1, c2, c3) <- (hi(M1*c2) ^ c1 ^ k0,  lo(M1*c2),  hi(M0*c0) ^ c3 ^ k1,  lo(M0*c0))
// with the key bumped by the two Weyl constants between rounds.  The paper itself used cuRAND's default
// generator and stored the uniforms in a 4-byte global matrix; here the 32 random
// bits of a site never leave registers (include/shaken.h gives the site -> counter mapping).
//
// This file is part of the product path and shares nothing with oracle/ (which carries its own Philox).
#pragma once
#include <stdint.h>

namespace shaken {

constexpr uint32_t PHILOX_M0 = 0xD2511F53u;
constexpr uint32_t PHILOX_M1 = 0xCD9E8D57u;
constexpr uint32_t PHILOX_W0 = 0x9E3779B9u;
constexpr uint32_t PHILOX_W1 = 0xBB67AE85u;

__host__ __device__ __forceinline__ void mul_wide(uint32_t a, uint32_t b, uint32_t &hi, uint32_t &lo)
{
    uint64_t p = (uint64_t)a * (uint64_t)b;   // one IMAD.WIDE.U32 on the FMA pipe
    hi = (uint32_t)(p >> 32);
    lo = (uint32_t)p;
}

// Generic form (init stream, test hook, conversions): any counter, any key.
__host__ __device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                                       uint32_t k0, uint32_t k1, uint32_t out[4])
{
#pragma unroll
    for (int i = 0; i < 10; ++i) {
        uint32_t h0, l0, h1, l1;
        mul_wide(PHILOX_M0, c0, h0, l0);
        mul_wide(PHILOX_M1, c2, h1, l1);
        c0 = h1 ^ c1 ^ k0;
        c1 = l1;
        c2 = h0 ^ c3 ^ k1;
        c3 = l0;
        k0 += PHILOX_W0;
        k1 += PHILOX_W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// ---------------------------------------------------------------------------------------------------
// Hoisted form for the half-step kernels.  In counter = (n, chain, g_lo, g_hi) only n = site >> 2 varies
// inside a launch, so round 0 needs one multiply (M0*n; M1*g_lo is uniform) and round 1 needs one
// (M1*a2; M0*a0 is uniform per chain): 18 instead of 20 IMAD.WIDE per call, 19 XORs instead of 20.
//
// StepKeys is filled on the host once per half-step launch and lives in the kernel parameter block
// (constant bank 0), so round keys are constant-bank operands of LOP3 and cost no registers.
// ---------------------------------------------------------------------------------------------------
struct StepKeys {
    uint32_t k0[10];   // k0 + i*W0
    uint32_t k1[10];   // k1 + i*W1
    uint32_t hi1;      // hi(M1 * g_lo)
    uint32_t xa2;      // g_hi ^ k1[0]                  : a2 = hi(M0*n) ^ xa2
    uint32_t xb0;      // lo(M1 * g_lo) ^ k0[1]          : b0 = hi(M1*a2) ^ xb0
    uint32_t pad;
};

// Per-chain uniform part (three integer ops per task).
struct ChainKeys {
    uint32_t xb2;      // hi(M0*a0) ^ k1[1]              : b2 = lo(M0*n) ^ xb2
    uint32_t xd2;      // lo(M0*a0) ^ k1[2]              : d2 = hi(M0*b0) ^ xd2
};

inline void make_step_keys(uint64_t seed, uint64_t g, StepKeys &K)
{
    uint32_t k0 = (uint32_t)seed, k1 = (uint32_t)(seed >> 32);
    for (int i = 0; i < 10; ++i) {
        K.k0[i] = k0 + (uint32_t)i * PHILOX_W0;
        K.k1[i] = k1 + (uint32_t)i * PHILOX_W1;
    }
    uint32_t g_lo = (uint32_t)g, g_hi = (uint32_t)(g >> 32), hi, lo;
    mul_wide(PHILOX_M1, g_lo, hi, lo);
    K.hi1 = hi;
    K.xa2 = g_hi ^ K.k1[0];
    K.xb0 = lo ^ K.k0[1];
    K.pad = 0;
}

__device__ __forceinline__ ChainKeys make_chain_keys(const StepKeys &K, uint32_t chain)
{
    uint32_t a0 = K.hi1 ^ chain ^ K.k0[0];
    uint32_t h, l;
    mul_wide(PHILOX_M0, a0, h, l);
    ChainKeys c;
    c.xb2 = h ^ K.k1[1];
    c.xd2 = l ^ K.k1[2];
    return c;
}

// The four random words of sites 4n .. 4n+3, with the round-0 product (h0:l0) = M0 * n supplied by the caller.  Inside a strip n moves by constants (to the next vector
// word, to the next row), so the 64-bit product can be carried along by 64-bit ADDITIONS (two IADD3 on the ALU port)
// instead of one IMAD.WIDE per call on the multiplier pipe, which is the pipe that bounds the kernels: 17 multiplies per
// call instead of 18.  Exact as long as n itself does not wrap, which it never does (n < L^2 / 4 <= 2^30).
__device__ __forceinline__ void philox_site_words_prod(uint32_t h0, uint32_t l0, const StepKeys &K, const uint32_t xa2, const uint32_t xb0,
                                                       const ChainKeys &C, uint32_t r[4])
{
    uint32_t h1, l1;
    uint32_t a2 = h0 ^ xa2, a3 = l0;
    // round 1: c = (a0 [uniform], a1 [uniform], a2, a3)
    mul_wide(PHILOX_M1, a2, h1, l1);
    uint32_t c0 = h1 ^ xb0, c1 = l1, c2 = a3 ^ C.xb2;            // c3 = lo(M0*a0), folded into xd2
    // round 2
    mul_wide(PHILOX_M0, c0, h0, l0);
    mul_wide(PHILOX_M1, c2, h1, l1);
    c0 = h1 ^ c1 ^ K.k0[2];
    c1 = l1;
    c2 = h0 ^ C.xd2;
    uint32_t c3 = l0;
#pragma unroll
    for (int i = 3; i < 10; ++i) {
        mul_wide(PHILOX_M0, c0, h0, l0);
        mul_wide(PHILOX_M1, c2, h1, l1);
        c0 = h1 ^ c1 ^ K.k0[i];
        c1 = l1;
        c2 = h0 ^ c3 ^ K.k1[i];
        c3 = l0;
    }
    r[0] = c0; r[1] = c1; r[2] = c2; r[3] = c3;
}


// The four random words of sites 4n .. 4n+3.  xa2, xb0: the per-half-step uniform words (StepKeys::xa2, ::xb0,
// or the same values computed on the device by a kernel that loops over steps itself).
__device__ __forceinline__ void philox_site_words(uint32_t n, const StepKeys &K, const uint32_t xa2, const uint32_t xb0,
                                                  const ChainKeys &C, uint32_t r[4])
{
    uint32_t h0, l0;
    mul_wide(PHILOX_M0, n, h0, l0);      // round 0: c = (n, chain, g_lo, g_hi)
    philox_site_words_prod(h0, l0, K, xa2, xb0, C, r);
}

// N independent calls advanced round by round (the source order a scheduler would want: N multiply chains in flight)
// PROD: n[t] is not used, (ph[t]:pl[t]) = M0 * n[t] is supplied (see philox_site_words_prod)
template <int N, bool PROD = false>
__device__ __forceinline__ void philox_site_words_xn(const uint32_t (&n)[N], const StepKeys &K, const uint32_t xa2, const uint32_t xb0,
                                                     const ChainKeys &C, uint32_t (&r)[N][4], const uint32_t *ph = nullptr,
                                                     const uint32_t *pl = nullptr)
{
    uint32_t c0[N], c1[N], c2[N], c3[N];
#pragma unroll
    for (int t = 0; t < N; ++t) {
        uint32_t h0, l0, h1, l1;
        if constexpr (PROD) { h0 = ph[t]; l0 = pl[t]; }
        else mul_wide(PHILOX_M0, n[t], h0, l0);
        const uint32_t a2 = h0 ^ xa2, a3 = l0;
        mul_wide(PHILOX_M1, a2, h1, l1);
        c0[t] = h1 ^ xb0; c1[t] = l1; c2[t] = a3 ^ C.xb2;
    }
#pragma unroll
    for (int t = 0; t < N; ++t) {
        uint32_t h0, l0, h1, l1;
        mul_wide(PHILOX_M0, c0[t], h0, l0);
        mul_wide(PHILOX_M1, c2[t], h1, l1);
        c0[t] = h1 ^ c1[t] ^ K.k0[2];
        c1[t] = l1;
        c2[t] = h0 ^ C.xd2;
        c3[t] = l0;
    }
#pragma unroll
    for (int i = 3; i < 10; ++i) {
#pragma unroll
        for (int t = 0; t < N; ++t) {
            uint32_t h0, l0, h1, l1;
            mul_wide(PHILOX_M0, c0[t], h0, l0);
            mul_wide(PHILOX_M1, c2[t], h1, l1);
            c0[t] = h1 ^ c1[t] ^ K.k0[i];
            c1[t] = l1;
            c2[t] = h0 ^ c3[t] ^ K.k1[i];
            c3[t] = l0;
        }
    }
#pragma unroll
    for (int t = 0; t < N; ++t) { r[t][0] = c0[t]; r[t][1] = c1[t]; r[t][2] = c2[t]; r[t][3] = c3[t]; }
}

// 64-bit (hi:lo) += (ahi:alo), as two 32-bit additions with carry (kept off the multiplier pipe on purpose)
__device__ __forceinline__ void add64(uint32_t &hi, uint32_t &lo, uint32_t ahi, uint32_t alo)
{
    asm("add.cc.u32 %0, %0, %2;\n\taddc.u32 %1, %1, %3;" : "+r"(lo), "+r"(hi) : "r"(alo), "r"(ahi));
}

__device__ __forceinline__ void philox_site_words(uint32_t n, const StepKeys &K, const ChainKeys &C, uint32_t r[4])
{
    philox_site_words(n, K, K.xa2, K.xb0, C, r);
}

// Device-side form of the per-half-step part of make_step_keys + make_chain_keys, for kernels that advance
// several steps in one launch: K supplies only the round keys k0[], k1[] (functions of the seed).
__device__ __forceinline__ void device_half_step_keys(const StepKeys &K, uint64_t g, uint32_t chain, uint32_t &xa2, uint32_t &xb0, ChainKeys &C)
{
    uint32_t hi, lo;
    mul_wide(PHILOX_M1, (uint32_t)g, hi, lo);
    xa2 = (uint32_t)(g >> 32) ^ K.k1[0];
    xb0 = lo ^ K.k0[1];
    const uint32_t a0 = hi ^ chain ^ K.k0[0];
    uint32_t h, l;
    mul_wide(PHILOX_M0, a0, h, l);
    C.xb2 = h ^ K.k1[1];
    C.xd2 = l ^ K.k1[2];
}

} // namespace shaken
