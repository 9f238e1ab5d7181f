// kernel_alt.cuh -- the alternate parallel heat bath on the SQUARE lattice ("a parallel version of the
// heat bath dynamics that updates, alternatively, the spins on the odd and the even sites of the lattice"; its
// equilibrium measure is the Gibbs measure of the square-lattice Ising model).  SURVEY 8(f) rank 3.
//
// One spin field (the context's sigma array, updated IN PLACE; tau is not touched).  Site (r, c) has colour (r + c) & 1;
// half-step HALF of full step t redraws every site of colour HALF: +1 iff rnd < A[k], k = number of +1 among the four
// neighbours (field h = J (2k - 4)).  The m-th site of a colour in row-major order, m = (r L + c) >> 1, draws word
// m & 3 of Philox counter (m >> 2, chain, g lo, g hi), g = 2t + HALF -- so one call serves eight consecutive sites of a
// row and no random word is thrown away.
//
// In place is safe: every neighbour of a redrawn site has the other colour and is not written with a different value
// during the launch (a thread stores whole vectors, but the bytes or bits of the passive colour go back unchanged).
// For the same reason the loads are plain coherent loads, not the read-only path.
//
// Work: a warp takes `rows_per_task` rows of one chain; its lanes stride over the (row, vector) pairs.  A vector is
// 16 int8 spins (two Philox calls) or one packed word of 32 spins (four calls).  The sums of a recorded step are fused
// into half-step 1: every bond joins a site redrawn there to a passive one, so  C_x = sum_{x odd} s_x (left + right),
// C_y = sum_{x odd} s_x (up + down)  and M is the sum of the stored vectors.
#pragma once
#include "kernels_common.cuh"

namespace shaken {

constexpr int ALT_THREADS = 256;

struct AltParams {
    void *sigma;
    int L;
    int nvec;               // vectors per row: L/16 (int8) or L/32 (packed)
    int n_chains;
    uint32_t chain0;
    int group;              // coupling group size (random numbers of the group's first chain)
    int rows_per_task;
    int nrb;                // row blocks per chain = ceil(L / rows_per_task)
    long long ntasks;       // n_chains * nrb
    const uint32_t *gtab;   // per-chain thresholds [n_chains][8] (A[0..4] used) or nullptr: utab
    uint32_t utab[8];
    long long *rec;         // [n_chains][6] record of this step (half-step 1 only) or nullptr
    StepKeys keys;
};

template <int HALF, bool OBS, bool PACKED>
__global__ void __launch_bounds__(ALT_THREADS) alt_half(const __grid_constant__ AltParams p)
{
    __shared__ uint32_t s_tab[ALT_THREADS / 32][8];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int L = p.L, nvec = p.nvec;
    const int wpr = PACKED ? nvec : 4 * nvec;                      // 32-bit words per row
    uint32_t *tab = s_tab[warp];

    for (long long task = (long long)blockIdx.x * (ALT_THREADS / 32) + warp; task < p.ntasks;
         task += (long long)gridDim.x * (ALT_THREADS / 32)) {
        const int chain = (int)(task / p.nrb), rb = (int)(task - (long long)chain * p.nrb);
        const int r_begin = rb * p.rows_per_task, r_end = min(L, r_begin + p.rows_per_task);
        __syncwarp();
        if (lane < 8) tab[lane] = p.gtab ? p.gtab[(size_t)chain * 8 + lane] : p.utab[lane];
        __syncwarp();
        const ChainKeys ck = make_chain_keys(p.keys, p.chain0 + (uint32_t)((chain / p.group) * p.group));
        uint32_t *base = reinterpret_cast<uint32_t *>(p.sigma) + (size_t)chain * L * wpr;
        int accM = 0, accX = 0, accY = 0;
        const int items = (r_end - r_begin) * nvec;
        for (int it = lane; it < items; it += 32) {
            const int r = r_begin + it / nvec, v = it - (it / nvec) * nvec;
            uint32_t *row = base + (size_t)r * wpr;
            const uint32_t *up = base + (size_t)(r + 1 == L ? 0 : r + 1) * wpr;
            const uint32_t *dn = base + (size_t)(r == 0 ? L - 1 : r - 1) * wpr;
            const int pc = (r + HALF) & 1;                         // parity of the redrawn columns of this row
            if constexpr (!PACKED) {
                const uint4 c4 = *reinterpret_cast<const uint4 *>(row + 4 * v);
                const uint4 u4 = *reinterpret_cast<const uint4 *>(up + 4 * v);
                const uint4 d4 = *reinterpret_cast<const uint4 *>(dn + 4 * v);
                const uint32_t prev = row[v == 0 ? wpr - 1 : 4 * v - 1];        // holds the spin left of the vector
                const uint32_t next = row[v + 1 == nvec ? 0 : 4 * v + 4];       // holds the spin right of it
                const uint32_t c[6] = {prev, c4.x, c4.y, c4.z, c4.w, next};
                const uint32_t u[4] = {u4.x, u4.y, u4.z, u4.w}, d[4] = {d4.x, d4.y, d4.z, d4.w};
                uint32_t rnd[8];
                const uint32_t n0 = (uint32_t)r * (uint32_t)(L >> 3) + 2u * (uint32_t)v;
                philox_site_words(n0, p.keys, ck, rnd);
                philox_site_words(n0 + 1u, p.keys, ck, rnd + 4);
                const uint32_t active = 0x00FF00FFu << (8 * pc);
                uint32_t out[4];
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const uint32_t lw = __funnelshift_l(c[j], c[j + 1], 8);     // byte b = spin left of column b
                    const uint32_t rw = __funnelshift_r(c[j + 1], c[j + 2], 8); // byte b = spin right of column b
                    const uint32_t hsum = __vadd4(lw, rw), vsum = __vadd4(u[j], d[j]);
                    // k = (sum of the four +-1 neighbours + 4) / 2, per byte
                    const uint32_t kq = (__vadd4(__vadd4(hsum, vsum), 0x04040404u) >> 1) & 0x07070707u;
                    uint32_t o = c[j + 1] & ~active;
#pragma unroll
                    for (int i = 0; i < 2; ++i) {
                        const int sh = 8 * (pc + 2 * i);
                        const uint32_t T = tab[(kq >> sh) & 7u];
                        o |= (rnd[2 * j + i] < T ? 0x01u : 0xFFu) << sh;
                    }
                    out[j] = o;
                    if constexpr (OBS) {
                        accM = __dp4a((int)o, 0x01010101, accM);
                        accX = __dp4a((int)(o & active), (int)hsum, accX);
                        accY = __dp4a((int)(o & active), (int)vsum, accY);
                    }
                }
                *reinterpret_cast<uint4 *>(row + 4 * v) = make_uint4(out[0], out[1], out[2], out[3]);
            } else {
                const uint32_t c = row[v], a = up[v], b = dn[v];
                const uint32_t prev = row[v == 0 ? nvec - 1 : v - 1], next = row[v + 1 == nvec ? 0 : v + 1];
                const uint32_t lw = __funnelshift_l(prev, c, 1);                // bit i = spin left of column i
                const uint32_t rw = __funnelshift_r(c, next, 1);                // bit i = spin right of column i
                // bit-sliced count of +1 among (a, b, lw, rw): k = s0 + 2 s1 + 4 s2
                const uint32_t ab = a & b, axb = a ^ b, lr = lw & rw, lxr = lw ^ rw;
                const uint32_t s0 = axb ^ lxr, s1 = (ab ^ lr) ^ (axb & lxr), s2 = ab & lr;
                const uint32_t n0 = (uint32_t)r * (uint32_t)(L >> 3) + 4u * (uint32_t)v;
                uint32_t nb = 0;
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    uint32_t rnd[4];
                    philox_site_words(n0 + (uint32_t)q, p.keys, ck, rnd);
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        const int bit = 2 * (4 * q + i) + pc;
                        const uint32_t k = ((s0 >> bit) & 1u) | (((s1 >> bit) & 1u) << 1) | (((s2 >> bit) & 1u) << 2);
                        nb |= (rnd[i] < tab[k] ? 1u : 0u) << bit;
                    }
                }
                const uint32_t active = 0x55555555u << pc;
                const uint32_t o = (c & ~active) | nb;
                row[v] = o;
                if constexpr (OBS) {
                    accM += 2 * __popc(o) - 32;
                    accX += 2 * (__popc(~(o ^ lw) & active) + __popc(~(o ^ rw) & active)) - 32;
                    accY += 2 * (__popc(~(o ^ a) & active) + __popc(~(o ^ b) & active)) - 32;
                }
            }
        }
        if constexpr (OBS) {
            long long *rec = p.rec + (size_t)chain * 6;
            warp_add_to(rec + 0, accM);
            warp_add_to(rec + 4, accX);
            warp_add_to(rec + 5, accY);
        }
    }
}

} // namespace shaken
