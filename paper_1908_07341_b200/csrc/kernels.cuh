// kernels.cuh -- bit-packed half-step kernel, initialisation, layout conversion, validation, test hook.
// (The int8 half-step kernel is in kernel_i8.cuh; shared declarations in kernels_common.cuh.)
#pragma once
#include "kernels_common.cuh"
#include "kernel_i8.cuh"

namespace shaken {

// ===================================================================================================
// Bit-packed layout: 32 spins per word, bit 1 <-> +1.  A word is spread into eight byte-SIMD registers
// Y4[k] = 4 * (bits k, 8+k, 16+k, 24+k), so that the left (right) neighbour of site 8m+k is byte m of
// Y4[k-1] (Y4[k+1]) with no shift; only k = 0 (k = 7) needs a byte funnel shift and the neighbouring word.
// Table order: natural, index = c + 2 (v + h) = 2k + c.
// ===================================================================================================
__device__ __forceinline__ void spread4(uint32_t W, uint32_t Y4[8])
{
#pragma unroll
    for (int k = 0; k < 8; ++k) Y4[k] = (k <= 2 ? (W << (2 - k)) : (W >> (k - 2))) & 0x04040404u;
}

template <int HALF, int FLAGS>
__global__ void __launch_bounds__(BLOCK_THREADS, 2) half_step_pk(const __grid_constant__ StepParams p)
{
    constexpr bool OBS = (FLAGS & F_OBS) != 0;
    constexpr bool BONDS = (FLAGS & F_BONDS) != 0;
    constexpr bool UPDATE = (FLAGS & F_NOUPDATE) == 0;
    static_assert(!(BONDS && HALF == 1), "bond sums ride on half-step 0");

    __shared__ uint32_t s_tab[WARPS_PER_BLOCK][8];
    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    uint32_t *tabw = s_tab[warp];

    const int L = p.L;
    const int L4 = L >> 2;
    const int W = p.nvec;                 // words per row
    const int R = p.rows_per_task;
    const size_t plane = (size_t)L * (size_t)W;

    int cur_chain = -1;
    ChainKeys ck = {0u, 0u};
    int cnt0 = 0, cnt1 = 0, cnt2 = 0;

    auto flush = [&](int chain) {
        if (HALF == 1) {
            if (OBS) {
                warp_add_to(p.rec_cur + (size_t)chain * 6 + 0, cnt0);
                warp_add_to(p.rec_cur + (size_t)chain * 6 + 2, cnt1);
                warp_add_to(p.rec_cur + (size_t)chain * 6 + 3, cnt2);
            }
        } else {
            if (OBS) warp_add_to(p.rec_cur + (size_t)chain * 6 + 1, cnt0);
            if (BONDS) {
                warp_add_to(p.rec_prev + (size_t)chain * 6 + 4, cnt1);
                warp_add_to(p.rec_prev + (size_t)chain * 6 + 5, cnt2);
            }
        }
        cnt0 = cnt1 = cnt2 = 0;
    };

    const long long nw = (long long)gridDim.x * WARPS_PER_BLOCK;
    for (long long task = (long long)blockIdx.x * WARPS_PER_BLOCK + warp; task < p.ntasks; task += nw) {
        const int seg = (int)(task % p.nseg);
        const long long t2 = task / p.nseg;
        const int rb = (int)(t2 % p.nrb);
        const int chain = (int)(t2 / p.nrb);
        if (chain != cur_chain) {
            if ((OBS || BONDS) && cur_chain >= 0) flush(cur_chain);
            cur_chain = chain;
            if (UPDATE) {
                ck = make_chain_keys(p.keys, p.chain0 + (uint32_t)chain);
                __syncwarp();
                if (lane < 8) tabw[lane] = p.gtab ? p.gtab[(size_t)chain * 8 + lane] : p.utab[lane];
                __syncwarp();
            }
        }
        const int cv = seg * 32 + lane;
        if (cv >= W) continue;

        const int r_first = rb * R;
        const int r_last = min(L, r_first + R) - 1;
        const int rows = r_last - r_first + 1;
        const uint32_t *sbase = reinterpret_cast<const uint32_t *>(p.src) + (size_t)chain * plane;
        uint32_t *dbase = reinterpret_cast<uint32_t *>(p.dst) + (size_t)chain * plane;

        const int dir = HALF ? -1 : +1;
        int r = HALF ? r_last : r_first;
        const int rh = HALF ? (r_last + 1 == L ? 0 : r_last + 1) : (r_first == 0 ? L - 1 : r_first - 1);
        const int ce = HALF ? (cv + 1 == W ? 0 : cv + 1) : (cv == 0 ? W - 1 : cv - 1);

        uint32_t V = __ldg(sbase + (size_t)rh * W + cv);
        uint32_t S = __ldg(sbase + (size_t)r * W + cv);
        uint32_t e = __ldg(sbase + (size_t)r * W + ce);
        uint32_t n = (uint32_t)r * (uint32_t)L4 + (uint32_t)cv * 8u;

        uint32_t Yv[8];
        if (UPDATE) spread4(V, Yv);
        int a0 = 0, a1 = 0, a2 = 0;     // popcount partials of this task

        for (int i = 0; i < rows; ++i) {
            uint32_t Sn = S, en = e;
            if (i + 1 < rows) {
                const int rn = r + dir;
                Sn = __ldg(sbase + (size_t)rn * W + cv);
                en = __ldg(sbase + (size_t)rn * W + ce);
            }
            // horizontal neighbour plane: left (half 0) or right (half 1)
            const uint32_t Hp = HALF == 0 ? ((S << 1) | (e >> 31)) : ((S >> 1) | (e << 31));
            uint32_t out = 0;
            if (UPDATE) {
                uint32_t Y[8];
                spread4(S, Y);
                uint32_t off[8];
#pragma unroll
                for (int k = 0; k < 8; ++k) {
                    uint32_t H;
                    if (HALF == 0) H = k >= 1 ? Y[k - 1] : ((Y[7] << 8) | ((e >> 31) << 2));
                    else           H = k <= 6 ? Y[k + 1] : ((Y[0] >> 8) | ((e & 1u) << 26));
                    off[k] = Y[k] + 2u * (Yv[k] + H);
                }
#pragma unroll
                for (int q = 0; q < 8; ++q) {
                    uint32_t rw[4];
                    philox_site_words(n + (uint32_t)q, p.keys, ck, rw);
#pragma unroll
                    for (int b = 0; b < 4; ++b) {
                        const int site = 4 * q + b, m = site >> 3, k = site & 7;
                        const uint32_t o = (off[k] >> (8 * m)) & 0xFFu;
                        const uint32_t T = *reinterpret_cast<const uint32_t *>(reinterpret_cast<const char *>(tabw) + o);
                        out |= (rw[b] < T ? 1u : 0u) << site;
                    }
                }
                dbase[(size_t)r * W + cv] = out;
#pragma unroll
                for (int k = 0; k < 8; ++k) Yv[k] = Y[k];
            }
            if (HALF == 1) {
                if (OBS) {
                    a0 += __popc(out);
                    a1 += __popc(out ^ V) + __popc(out ^ Hp);
                    a2 += __popc(out ^ S);
                }
            } else {
                if (OBS) a0 += __popc(out);
                if (BONDS) {
                    a1 += __popc(S ^ Hp);
                    a2 += __popc(S ^ V);
                }
            }
            V = S; S = Sn; e = en;
            r += dir;
            n += (uint32_t)(dir * L4);
        }
        if (OBS || BONDS) {
            const int ns = rows * 32;
            if (HALF == 1) {
                if (OBS) {
                    cnt0 += 2 * a0 - ns;
                    cnt1 += 2 * ns - 2 * a1;
                    cnt2 += ns - 2 * a2;
                }
            } else {
                if (OBS) cnt0 += 2 * a0 - ns;
                if (BONDS) {
                    cnt1 += ns - 2 * a1;
                    cnt2 += ns - 2 * a2;
                }
            }
        }
    }
    if ((OBS || BONDS) && cur_chain >= 0) flush(cur_chain);
}

// ===================================================================================================
// Initialisation, layout conversion, validation, test hook
// ===================================================================================================

// iid start: spin = +1 iff init-stream word < 2^31; counter = (site>>2, chain, which, 0xFFFFFFFF).
// One thread per Philox call (4 sites) per sublattice.  packed: 8 calls per word handled by one thread.
__global__ void init_iid_i8(uint8_t *sigma, uint8_t *tau, int n_chains, uint32_t chain0, long long calls_per_chain, uint32_t k0, uint32_t k1)
{
    const long long total = (long long)n_chains * calls_per_chain;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < total; i += (long long)gridDim.x * blockDim.x) {
        const uint32_t chain = chain0 + (uint32_t)(i / calls_per_chain);
        const uint32_t n = (uint32_t)(i % calls_per_chain);
#pragma unroll
        for (int which = 0; which < 2; ++which) {
            uint32_t w[4];
            philox4x32_10(n, chain, (uint32_t)which, 0xFFFFFFFFu, k0, k1, w);
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

__global__ void philox_hook(const uint32_t *ctr, const uint32_t *key, uint32_t *out, long long n)
{
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        uint32_t w[4];
        philox4x32_10(ctr[4 * i], ctr[4 * i + 1], ctr[4 * i + 2], ctr[4 * i + 3], key[2 * i], key[2 * i + 1], w);
        out[4 * i] = w[0]; out[4 * i + 1] = w[1]; out[4 * i + 2] = w[2]; out[4 * i + 3] = w[3];
    }
}

} // namespace shaken
