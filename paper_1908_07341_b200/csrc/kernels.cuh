// kernels.cuh -- initialisation, layout conversion, validation, test hook.
// (The half-step kernels are in kernel_i8.cuh and kernel_pk.cuh; shared declarations in kernels_common.cuh.)
#pragma once
#include "kernels_common.cuh"
#include "kernel_i8.cuh"
#include "kernel_pk.cuh"
#include "kernel_small.cuh"
#include "kernel_cluster.cuh"
#include "kernel_flow.cuh"
#include "kernel_band.cuh"
#include "kernel_alt.cuh"
#include "kernel_slab.cuh"

namespace shaken {

// ===================================================================================================
// Initialisation, layout conversion, validation, test hook
// ===================================================================================================

// iid start: spin = +1 iff init-stream word < 2^31; counter = (site>>2, chain, which, 0xFFFFFFFF).
// One thread per Philox call (4 sites) per sublattice.  packed: 8 calls per word handled by one thread.
// n_offset: Philox counter word 0 of the first call (a slab of one lattice starts at row0 * L / 4, a whole torus at 0)
__global__ void init_iid_i8(uint8_t *sigma, uint8_t *tau, int n_chains, uint32_t chain0, long long calls_per_chain, uint32_t k0, uint32_t k1, uint32_t n_offset)
{
    const long long total = (long long)n_chains * calls_per_chain;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
        const uint32_t chain = chain0 + (uint32_t)(i / calls_per_chain);
        const uint32_t n = (uint32_t)(i % calls_per_chain);
#pragma unroll
        for (int which = 0; which < 2; ++which) {
            uint32_t w[4];
            philox4x32_10(n + n_offset, chain, (uint32_t)which, 0xFFFFFFFFu, k0, k1, w);
            uint32_t out = 0;
#pragma unroll
            for (int b = 0; b < 4; ++b) out |= (w[b] < 0x80000000u ? 0x01u : 0xFFu) << (8 * b);
            reinterpret_cast<uint32_t *>(which ? tau : sigma)[i] = out;
        }
    }
}

__global__ void init_iid_pk(uint32_t *sigma, uint32_t *tau, int n_chains, uint32_t chain0, long long words_per_chain, uint32_t k0, uint32_t k1)
{
    const long long total = (long long)n_chains * words_per_chain;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
        const uint32_t chain = chain0 + (uint32_t)(i / words_per_chain);
        const uint32_t wd = (uint32_t)(i % words_per_chain);
#pragma unroll
        for (int which = 0; which < 2; ++which) {
            uint32_t out = 0;
            for (int q = 0; q < 8; ++q) {
                uint32_t w[4];
                philox4x32_10(wd * 8u + (uint32_t)q, chain, (uint32_t)which, 0xFFFFFFFFu, k0, k1, w);
#pragma unroll
                for (int b = 0; b < 4; ++b) out |= (w[b] < 0x80000000u ? 1u : 0u) << (4 * q + b);
            }
            (which ? tau : sigma)[i] = out;
        }
    }
}

// packed words -> +-1 bytes (one thread per word, 32 bytes out)
__global__ void unpack_words(const uint32_t *pk, uint8_t *bytes, long long n_words)
{
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n_words; i += (long long)gridDim.x * blockDim.x) {
        const uint32_t w = pk[i];
        uint4 o[2];
        uint32_t *ow = reinterpret_cast<uint32_t *>(o);
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            uint32_t x = 0;
#pragma unroll
            for (int b = 0; b < 4; ++b) x |= (((w >> (4 * j + b)) & 1u) ? 0x01u : 0xFFu) << (8 * b);
            ow[j] = x;
        }
        reinterpret_cast<uint4 *>(bytes)[2 * i] = o[0];
        reinterpret_cast<uint4 *>(bytes)[2 * i + 1] = o[1];
    }
}

// +-1 bytes -> packed words; counts bytes that are neither 0x01 nor 0xFF
__global__ void pack_words(const uint8_t *bytes, uint32_t *pk, long long n_words, unsigned long long *bad)
{
    unsigned int nbad = 0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n_words; i += (long long)gridDim.x * blockDim.x) {
        const uint4 a = reinterpret_cast<const uint4 *>(bytes)[2 * i];
        const uint4 b4 = reinterpret_cast<const uint4 *>(bytes)[2 * i + 1];
        const uint32_t in[8] = {a.x, a.y, a.z, a.w, b4.x, b4.y, b4.z, b4.w};
        uint32_t w = 0;
#pragma unroll
        for (int j = 0; j < 8; ++j)
#pragma unroll
            for (int b = 0; b < 4; ++b) {
                const uint32_t x = (in[j] >> (8 * b)) & 0xFFu;
                if (x == 0x01u) w |= 1u << (4 * j + b);
                else if (x != 0xFFu) ++nbad;
            }
        pk[i] = w;
    }
    if (nbad) atomicAdd(bad, (unsigned long long)nbad);
}

// counts bytes that are neither 0x01 nor 0xFF (16 bytes per thread-iteration)
__global__ void validate_bytes(const uint8_t *bytes, long long n_vec, unsigned long long *bad)
{
    unsigned int nbad = 0;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n_vec; i += (long long)gridDim.x * blockDim.x) {
        const uint4 a = reinterpret_cast<const uint4 *>(bytes)[i];
        const uint32_t in[4] = {a.x, a.y, a.z, a.w};
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            // valid bytes: 0x01 or 0xFF  <=>  bit 0 set and bits 1..7 all equal
            const uint32_t x = in[j];
            const uint32_t m = (x >> 1) & 0x01010101u;          // bit 1 of each byte
            const uint32_t expect = (m * 0xFEu) | 0x01010101u;  // 0xFF where minus, 0x01 where plus
            const uint32_t d = x ^ expect;
            if (d) {
#pragma unroll
                for (int b = 0; b < 4; ++b) nbad += ((d >> (8 * b)) & 0xFFu) != 0;
            }
        }
    }
    if (nbad) atomicAdd(bad, (unsigned long long)nbad);
}

// "sandwich" start: the first chain of every coupling group all +1, the others all -1, both layers.
// vec_per_chain 16-byte vectors per chain; plus / minus are the byte patterns of the layout (int8: 0x01 / 0xFF, packed: 0xFF / 0x00).
__global__ void init_sandwich(uint4 *sigma, uint4 *tau, long long n_vec, long long vec_per_chain, int group, uint32_t plus, uint32_t minus)
{
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n_vec; i += (long long)gridDim.x * blockDim.x) {
        const long long chain = i / vec_per_chain;
        const uint32_t w = (chain % group == 0) ? plus : minus;
        sigma[i] = make_uint4(w, w, w, w);
        tau[i] = make_uint4(w, w, w, w);
    }
}

// Coalescence (T = min{n : X_n = Y_n}).  compare: every member of a not yet coalesced group against the
// group's first chain, 16 bytes at a time; any difference stamps diff[group] with the step index (all writers store the
// same value).  finalize: a group whose stamp is not this step's has coalesced now.
__global__ void coalesce_compare(const uint4 *sigma, long long vec_per_chain, int group, long long n_groups, const long long *coal,
                                 unsigned long long *diff, unsigned long long stamp)
{
    const long long per_group = (long long)(group - 1) * vec_per_chain, total = n_groups * per_group;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
        const long long gi = i / per_group, rest = i - gi * per_group;
        if (coal[gi] >= 0) continue;
        if (__ldcg(diff + gi) == stamp) continue;          // a difference of this step is already on record: nothing left to find
        const long long m = 1 + rest / vec_per_chain, v = rest % vec_per_chain;
        const uint4 a = sigma[(gi * group) * vec_per_chain + v], b = sigma[(gi * group + m) * vec_per_chain + v];
        if (a.x != b.x || a.y != b.y || a.z != b.z || a.w != b.w) diff[gi] = stamp;
    }
}

__global__ void coalesce_finalize(long long *coal, const unsigned long long *diff, long long n_groups, unsigned long long stamp)
{
    for (long long gi = (long long)blockIdx.x * blockDim.x + threadIdx.x; gi < n_groups; gi += (long long)gridDim.x * blockDim.x)
        if (coal[gi] < 0 && diff[gi] != stamp) coal[gi] = (long long)stamp;
}

// Diagonal correlation sums of the sigma layer (Table 1), translation-summed over the torus:
//   out[chain][e][0] = sum sigma[r][c] sigma[r+l][c+l]  (SW-NE),  out[chain][e][1] = sum sigma[r+l][c] sigma[r][c+l]  (NW-SE).
// One thread per 32-bit word of row r; the partner word, l columns to the right, is a funnel shift of two aligned
// words (int8: by 8 (l mod 4) bits, products by IDP.4A; packed: by l mod 32 bits, products by popcount of the XOR).
// grid = (blocks per chain, min(n_chains, 65535)), chains beyond gridDim.y are looped over; one int64 atomic per warp and sum.
template <bool PACKED>
__global__ void diag_corr(const uint32_t *sigma, int L, int n_chains, int ell, long long *out, int n_ell, int e)
{
    const int SPW = PACKED ? 32 : 4;                    // sites per word
    const int W = L / SPW;                              // L * W <= 2^30: the int indices below cannot overflow
    const int wsh = ell / SPW, sh = (ell % SPW) * (PACKED ? 1 : 8);
    for (int chain = blockIdx.y; chain < n_chains; chain += gridDim.y) {
    const uint32_t *sg = sigma + (size_t)chain * L * W;
    long long swne = 0, nwse = 0;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < L * W; i += gridDim.x * blockDim.x) {
        const int r = i / W, cw = i - r * W;
        const int r2 = r + ell >= L ? r + ell - L : r + ell;
        const int w0 = (cw + wsh) % W, w1 = w0 + 1 == W ? 0 : w0 + 1;
        const uint32_t a = sg[r * W + cw], a2 = sg[r2 * W + cw];
        const uint32_t b2 = __funnelshift_r(sg[r2 * W + w0], sg[r2 * W + w1], sh);   // sites (r+l, c+l ..)
        const uint32_t b = __funnelshift_r(sg[r * W + w0], sg[r * W + w1], sh);      // sites (r, c+l ..)
        if (PACKED) {
            swne += 32 - 2 * __popc(a ^ b2);
            nwse += 32 - 2 * __popc(a2 ^ b);
        } else {
            swne += __dp4a((int)a, (int)b2, 0);
            nwse += __dp4a((int)a2, (int)b, 0);
        }
    }
    for (int o = 16; o > 0; o >>= 1) {
        swne += __shfl_down_sync(0xFFFFFFFFu, swne, o);
        nwse += __shfl_down_sync(0xFFFFFFFFu, nwse, o);
    }
    if ((threadIdx.x & 31) == 0) {
        long long *dst = out + ((size_t)chain * n_ell + e) * 2;
        atomicAdd(reinterpret_cast<unsigned long long *>(dst), (unsigned long long)swne);
        atomicAdd(reinterpret_cast<unsigned long long *>(dst + 1), (unsigned long long)nwse);
    }
    }
}

// Measurement hook (shaken_selftest_philox_rate): the half-step kernels' own hoisted Philox4x32-10 (philox.cuh: 18
// IMAD.WIDE + 19 LOP3 per call of 4 sites) with one compare-and-count per random word and NOTHING else -- no loads, no
// stores, no neighbours, no table.  Its rate is the practical ceiling of any kernel that draws 32 Philox bits per site
// on this chip (SURVEY 8(d) "first experiment of the build"); bench.py reports it beside the HBM fraction.
__global__ void __launch_bounds__(256) philox_rate(uint32_t *out, const __grid_constant__ StepKeys K, int iters)
{
    const ChainKeys ck = make_chain_keys(K, 0u);
    uint32_t n = (blockIdx.x * 256u + threadIdx.x) * 4u * (uint32_t)iters, acc = 0;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            uint32_t r[4];
            philox_site_words(n + j, K, ck, r);
            acc += (r[0] < 0x80000000u) + (r[1] < 0x70000000u) + (r[2] < 0x60000000u) + (r[3] < 0x50000000u);
        }
        n += 4;
    }
    if (acc == 0x12345678u) out[0] = acc;          // keeps the arithmetic alive; practically never taken
}

__global__ void philox_hook(const uint32_t *ctr, const uint32_t *key, uint32_t *out, long long n)
{
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        uint32_t w[4];
        philox4x32_10(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3], key[2 * i], key[2 * i + 1], w);
        out[4 * i] = w[0]; out[4 * i + 1] = w[1]; out[4 * i + 2] = w[2]; out[4 * i + 3] = w[3];
    }
}

} // namespace shaken
