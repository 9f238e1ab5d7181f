// kernel_pk.cuh -- the bit-packed ("multispin") half-step kernel: 32 spins per uint32,
// bit b of word w of row r = site c = 32 w + b, bit 1 <-> +1.
//
// The acceptance needs a 32-bit compare per SITE, so packing saves memory traffic (0.25 B per update), not
// integer work.  The per-site table index is formed 4 sites at a time in byte-SIMD registers:
//   Y[k]  = 2 * (bits k, 8+k, 16+k, 24+k of the word)                       (k = 0..7: one shift + one AND)
//   C[k]  = Y[k] + 2 * (Yv[k] + Yh[k])  = 2 * (c + 2 (v + h)) = 2 * (2 k_plus + c) = 2 idx   per byte,
// where Yv is the previous row's Y (kept in registers) and Yh[k] = Y[k-1] (left, half 0) or Y[k+1] (right,
// half 1): in this strided grouping the horizontal neighbour of site 8m+k sits in the SAME byte m of the
// adjacent group, so only k = 0 (k = 7) needs a byte funnel shift and one bit of the neighbouring word.
// Two sites share one lookup: P[j] = C[2j] + 8 C[2j+1] holds in byte m the pair code 2 (idx_a + 8 idx_b) of the
// consecutive sites a = 8m+2j, b = a+1 (both of the same Philox call), one IDP.4A turns that byte into the byte
// offset 256 (idx_a + 8 idx_b) + 8 lane, and one LDS.64 fetches {T[idx_a], T[idx_b]} from a lane-replicated table
// (46 entries x 256 B; lane l always reads banks 2l, 2l+1: conflict-free for any mix of indices).
// Accepted sites are added into the output word with a predicated IADD (half the ALU-port cost of a LOP3).
// Observables are population counts of XORed words.
#pragma once
#include "kernels_common.cuh"

namespace shaken {

constexpr int PK_THREADS = 512;     // one 512-thread block per SM, up to 128 registers per thread
constexpr int PK_PAIR_ENTRIES = 46; // idx_a + 8 idx_b, idx in 0..5

__device__ __forceinline__ void spread2(uint32_t W, uint32_t Y2[8])
{
#pragma unroll
    for (int k = 0; k < 8; ++k) Y2[k] = (k == 0 ? (W << 1) : (W >> (k - 1))) & 0x02020202u;
}

template <int HALF, int FLAGS>
__global__ void __launch_bounds__(PK_THREADS, 1) half_step_pk(const __grid_constant__ StepParams p)
{
    constexpr bool OBS = (FLAGS & F_OBS) != 0;
    constexpr bool BONDS = (FLAGS & F_BONDS) != 0;
    constexpr bool UPDATE = (FLAGS & F_NOUPDATE) == 0;
    constexpr bool COAL = (FLAGS & F_COAL) != 0;            // compare the sigma read here with the group's first chain
    constexpr int WPB = PK_THREADS / 32;
    static_assert(!(BONDS && HALF == 1), "bond sums ride on half-step 0");

    __shared__ uint2 s_pair[PK_PAIR_ENTRIES][32];

    const int lane = threadIdx.x & 31;
    const int warp = threadIdx.x >> 5;
    const uint32_t lane8 = (uint32_t)lane * 8u;
    const int L = p.L;
    const int L4 = L >> 2;
    const int W = p.nvec;                               // words per row
    const int R = p.rows_per_task;
    const size_t plane = (size_t)L * (size_t)W;
    const int tpc = p.nrb * p.nseg;
    const int bpc = (tpc + WPB - 1) / WPB;

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

    let_next_kernel_launch();
    wait_for_previous_kernel();
    if (HALF == 1) finalize_coalescence(p);
    for (long long bt = blockIdx.x; bt < p.ntasks; bt += gridDim.x) {
        const int chain = (int)(bt / bpc);
        const int lt = (int)(bt % bpc) * WPB + warp;
        if (chain != cur_chain) {                                    // block-uniform
            if ((OBS || BONDS) && cur_chain >= 0) flush(cur_chain);
            cur_chain = chain;
            if (UPDATE) {
                ck = make_chain_keys(p.keys, rng_chain(p, chain));
                __syncthreads();
                for (int t = threadIdx.x; t < PK_PAIR_ENTRIES * 32; t += PK_THREADS) {
                    const int e = t >> 5, ia = e & 7, ib = e >> 3;
                    if (ia < 6 && ib < 6) {
                        const uint32_t Ta = p.gtab ? p.gtab[(size_t)chain * 8 + ia] : p.utab[ia];
                        const uint32_t Tb = p.gtab ? p.gtab[(size_t)chain * 8 + ib] : p.utab[ib];
                        s_pair[e][t & 31] = make_uint2(Ta, Tb);
                    }
                }
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
            // M0 * (Philox counter word 0 of the word's first call), carried by 64-bit additions (philox.cuh)
            uint32_t ph, pl;
            mul_wide(PHILOX_M0, (uint32_t)r0 * (uint32_t)L4 + (uint32_t)cv * 8u, ph, pl);
            const long long pstep = (long long)PHILOX_M0 * (long long)(dir * L4);
            const uint32_t pstep_hi = (uint32_t)((unsigned long long)pstep >> 32), pstep_lo = (uint32_t)pstep;

            // the row in use, and the next two already on their way (prefetch distance 2)
            uint32_t V = __ldg(sbase + (size_t)rh * W + cv);
            uint32_t S0 = __ldg(pc), E0 = __ldg(pe), S1 = S0, E1 = E0, S2 = S0, E2 = E0;
            if (rows > 1) { S1 = __ldg(pc + stride); E1 = __ldg(pe + stride); }
            uint32_t Yv[8];
            if (UPDATE) spread2(V, Yv);
            int a0 = 0, a1 = 0, a2 = 0;     // popcount partials of this task
            // coalescence test: members other than the first of a group that has not coalesced yet
            const int member = COAL ? chain % p.group : 0;
            // (not yet coalesced, and no difference of this step on record yet: one is enough)
            const bool cmp = COAL && member != 0 && p.coal[chain / p.group] < 0 && __ldcg(p.diff + chain / p.group) != p.cstamp;
            const ptrdiff_t to_first = -(ptrdiff_t)member * (ptrdiff_t)plane;
            uint32_t differs = 0;

            for (int i = 0; i < rows; ++i) {
                if (i + 2 < rows) {
                    S2 = __ldg(pc + 2 * stride);
                    E2 = __ldg(pe + 2 * stride);
                }
                const uint32_t S = S0, e = E0;
                if (COAL && cmp) differs |= S ^ __ldg(pc + to_first);   // the same word of the group's first chain
                // horizontal neighbour plane: left (half 0) or right (half 1)
                const uint32_t Hp = HALF == 0 ? ((S << 1) | (e >> 31)) : ((S >> 1) | (e << 31));
                uint32_t out = 0;
                if (UPDATE) {
                    uint32_t Y[8], C[8], P[4];
                    spread2(S, Y);
#pragma unroll
                    for (int k = 0; k < 8; ++k) {
                        uint32_t H;
                        if (HALF == 0) H = k >= 1 ? Y[k - 1] : ((Y[7] << 8) | ((e >> 31) << 1));
                        else           H = k <= 6 ? Y[k + 1] : ((Y[0] >> 8) | ((e & 1u) << 25));
                        C[k] = Y[k] + 2u * (Yv[k] + H);
                    }
#pragma unroll
                    for (int j = 0; j < 4; ++j) P[j] = C[2 * j] + 8u * C[2 * j + 1];
                    uint32_t RW[4][4];
#pragma unroll
                    for (int q = 0; q < 8; ++q) {
                        if ((q & 3) == 0) {                            // four calls at a time, round by round
                            uint32_t qh[4] = {ph, ph, ph, ph}, ql[4] = {pl, pl, pl, pl};   // M0 * (n + q + t)
#pragma unroll
                            for (int t = 0; t < 4; ++t)
                                if (q + t) add64(qh[t], ql[t], (uint32_t)(((unsigned long long)PHILOX_M0 * (q + t)) >> 32), (uint32_t)((unsigned long long)PHILOX_M0 * (q + t)));
                            const uint32_t nn[4] = {0u, 0u, 0u, 0u};
                            philox_site_words_xn<4, true>(nn, p.keys, p.keys.xa2, p.keys.xb0, ck, RW, qh, ql);
                        }
                        const uint32_t (&rw)[4] = RW[q & 3];
                        const int m = q >> 1, j0 = (q & 1) * 2;
                        const uint32_t o01 = __dp4a(P[j0], 0x80u << (8 * m), lane8), o23 = __dp4a(P[j0 + 1], 0x80u << (8 * m), lane8);
                        const uint2 t01 = *reinterpret_cast<const uint2 *>(reinterpret_cast<const char *>(s_pair) + o01);
                        const uint2 t23 = *reinterpret_cast<const uint2 *>(reinterpret_cast<const char *>(s_pair) + o23);
                        out = add_if_less(out, rw[0], t01.x, 1u << (4 * q));
                        out = add_if_less(out, rw[1], t01.y, 2u << (4 * q));
                        out = add_if_less(out, rw[2], t23.x, 4u << (4 * q));
                        out = add_if_less(out, rw[3], t23.y, 8u << (4 * q));
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
                V = S; S0 = S1; E0 = E1; S1 = S2; E1 = E2;
                pc += stride; pe += stride; pd += stride;
                add64(ph, pl, pstep_hi, pstep_lo);
            }
            if (COAL && differs != 0) p.diff[chain / p.group] = p.cstamp;   // every writer stores the same value
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
