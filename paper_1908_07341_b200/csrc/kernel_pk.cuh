// kernel_pk.cuh -- the bit-packed ("multispin") half-step kernel: 32 spins per uint32,
// bit b of word w of row r = site c = 32 w + b, bit 1 <-> +1.
//
// The acceptance needs a 32-bit compare per SITE, so packing saves memory traffic (0.25 B per update), not
// integer work.  The per-site table index is formed 4 sites at a time in byte-SIMD registers:
//   Y[k]  = 4 * (bits k, 8+k, 16+k, 24+k of the word)                       (k = 0..7: one shift + one AND)
//   C[k]  = Y[k] + 2 * (Yv[k] + Yh[k])  = 4 * (c + 2 (v + h)) = 4 * (2 k_plus + c)  per byte,
// where Yv is the previous row's Y (kept in registers) and Yh[k] = Y[k-1] (left, half 0) or Y[k+1] (right,
// half 1): in this strided grouping the horizontal neighbour of site 8m+k sits in the SAME byte m of the
// adjacent group, so only k = 0 (k = 7) needs a byte funnel shift and one bit of the neighbouring word.
// Byte m of C[k] is the byte offset of T[2k+c] for site 8m+k; the eight C words go through a per-thread
// shared-memory slot and come back one byte at a time (LDS.U8), exactly as in the int8 kernel.
// Observables are population counts of XORed words.
#pragma once
#include "kernels_common.cuh"

namespace shaken {

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

    __shared__ uint32_t s_tab[8];                       // T[2k + c], natural order
    __shared__ uint32_t s_idx[8][BLOCK_THREADS];        // per-thread staging of the eight C words

    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const int L = p.L;
    const int L4 = L >> 2;
    const int W = p.nvec;                               // words per row
    const int R = p.rows_per_task;
    const size_t plane = (size_t)L * (size_t)W;
    const int tpc = p.nrb * p.nseg;
    const int bpc = (tpc + WARPS_PER_BLOCK - 1) / WARPS_PER_BLOCK;

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

    for (long long bt = blockIdx.x; bt < p.ntasks; bt += gridDim.x) {
        const int chain = (int)(bt / bpc);
        const int lt = (int)(bt % bpc) * WARPS_PER_BLOCK + warp;
        if (chain != cur_chain) {                                    // block-uniform
            if ((OBS || BONDS) && cur_chain >= 0) flush(cur_chain);
            cur_chain = chain;
            if (UPDATE) {
                ck = make_chain_keys(p.keys, p.chain0 + (uint32_t)chain);
                __syncthreads();
                if (threadIdx.x < 8) s_tab[threadIdx.x] = p.gtab ? p.gtab[(size_t)chain * 8 + threadIdx.x] : p.utab[threadIdx.x];
                __syncthreads();
            }
        }
        const int seg = lt % p.nseg;
        const int rb = lt / p.nseg;
        const int cv = seg * 32 + lane;
        if (lt < tpc && cv < W) {
            const int r_first = rb * R;
            const int r_last = min(L, r_first + R) - 1;
            const int rows = r_last - r_first + 1;
            const uint32_t *sbase = reinterpret_cast<const uint32_t *>(p.src) + (size_t)chain * plane;
            uint32_t *dbase = reinterpret_cast<uint32_t *>(p.dst) + (size_t)chain * plane;

            const int dir = HALF ? -1 : +1;
            const int r0 = HALF ? r_last : r_first;
            const int rh = HALF ? (r_last + 1 == L ? 0 : r_last + 1) : (r_first == 0 ? L - 1 : r_first - 1);
            const int ce = HALF ? (cv + 1 == W ? 0 : cv + 1) : (cv == 0 ? W - 1 : cv - 1);

            const ptrdiff_t stride = (ptrdiff_t)dir * W;
            const uint32_t *pc = sbase + (size_t)r0 * W + cv;
            const uint32_t *pe = sbase + (size_t)r0 * W + ce;
            uint32_t *pd = dbase + (size_t)r0 * W + cv;
            uint32_t n = (uint32_t)r0 * (uint32_t)L4 + (uint32_t)cv * 8u;
            const uint32_t nstep = (uint32_t)(dir * L4);
            uint32_t *const my_idx = &s_idx[0][threadIdx.x];

            uint32_t V = __ldg(sbase + (size_t)rh * W + cv);
            uint32_t S = __ldg(pc);
            uint32_t e = __ldg(pe);
            uint32_t Yv[8];
            if (UPDATE) spread4(V, Yv);
            int a0 = 0, a1 = 0, a2 = 0;     // popcount partials of this task

            for (int i = 0; i < rows; ++i) {
                uint32_t Sn = S, en = e;
                if (i + 1 < rows) {
                    Sn = __ldg(pc + stride);
                    en = __ldg(pe + stride);
                }
                // horizontal neighbour plane: left (half 0) or right (half 1)
                const uint32_t Hp = HALF == 0 ? ((S << 1) | (e >> 31)) : ((S >> 1) | (e << 31));
                uint32_t out = 0;
                if (UPDATE) {
                    uint32_t Y[8];
                    spread4(S, Y);
#pragma unroll
                    for (int k = 0; k < 8; ++k) {
                        uint32_t H;
                        if (HALF == 0) H = k >= 1 ? Y[k - 1] : ((Y[7] << 8) | ((e >> 31) << 2));
                        else           H = k <= 6 ? Y[k + 1] : ((Y[0] >> 8) | ((e & 1u) << 26));
                        const uint32_t C = Y[k] + 2u * (Yv[k] + H);
                        *reinterpret_cast<volatile uint32_t *>(my_idx + k * BLOCK_THREADS) = C;
                    }
#pragma unroll
                    for (int q = 0; q < 8; ++q) {
                        uint32_t rw[4];
                        philox_site_words(n + (uint32_t)q, p.keys, ck, rw);
#pragma unroll
                        for (int b = 0; b < 4; ++b) {
                            const int site = 4 * q + b, m = site >> 3, k = site & 7;
                            const uint32_t code = reinterpret_cast<volatile const uint8_t *>(my_idx + k * BLOCK_THREADS)[m];
                            const uint32_t T = *reinterpret_cast<const uint32_t *>(reinterpret_cast<const char *>(s_tab) + code);
                            out = xor_if_less(out, rw[b], T, 1u << site);
                        }
                    }
                    *pd = out;
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
                pc += stride; pe += stride; pd += stride;
                n += nstep;
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
    }
    if ((OBS || BONDS) && cur_chain >= 0) flush(cur_chain);
}

} // namespace shaken
