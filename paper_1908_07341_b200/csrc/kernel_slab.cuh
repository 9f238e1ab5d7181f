// kernel_slab.cuh -- row-slab sharding of ONE large lattice over several GPUs (second bullet).
//
// Rank k holds rows [row0, row0 + n_rows) of sigma and tau.  The fields of eq. (14) reach one row
// across a slab edge in each half-step (the down row in half 0, the up row in half 1).  As in the band kernel
// (kernel_band.cuh) a slab redraws the tau row ABOVE itself redundantly -- a site's random word is a function of (seed,
// step, half, GLOBAL site index), so the bits are identical on both sides -- and the ranks exchange only sigma rows, once
// per full step: after half-step 1 a rank stores its bottom sigma row into the "from above" inbox of the rank below and its
// top row into the "from below" inbox of the rank above (peer stores over NVLink, `slab_publish`), and before half-step 0
// it polls its own inbox (`slab_edge`).  A row travels as {word, stamp} pairs, each ONE 64-bit relaxed system-scope access:
// a reader that sees the stamp of the exchange has the word written with it (no flag, no fence); two parities of inbox
// rows keep a fast rank from overwriting a row its neighbour has not read yet.  The two big launches of a step are the
// ordinary strip kernels (kernel_i8.cuh with slab_rows / row0); the arrays hold the halo rows in place (sigma rows -1 and
// n_rows, tau row n_rows), so the hot loops know nothing about slabs.  int64 sums are per slab; the host adds them.
#pragma once
#include "kernels_common.cuh"

namespace shaken {

constexpr int SLAB_THREADS = 256;

struct SlabParams {
    uint8_t *sigma;          // the slab's row 0 of sigma; rows -1 and n_rows exist in the array
    uint8_t *tau;            // the slab's row 0 of tau; row n_rows exists
    int L;
    int n_rows;
    uint32_t row0;           // global index of the slab's row 0
    uint32_t chain;          // Philox counter word 1
    uint2 *inbox;            // own inbox: [2 sides][2 parities][L/4] pairs; side 0 = sigma row row0-1, side 1 = row row0+n_rows
    uint2 *to_below;         // inbox of the rank that owns row row0-1 (its side 1 receives this slab's bottom row)
    uint2 *to_above;         // inbox of the rank that owns row row0+n_rows (its side 0 receives this slab's top row)
    uint32_t stamp;          // stamp of this exchange (its parity selects the inbox rows)
    uint32_t utab[8];        // thresholds T[2k + c]
    StepKeys keys;           // of half-step 0 of the step that follows the exchange
    int redraw;              // slab_edge: also redraw tau row n_rows (0 for the collect that only closes a record)
};

__device__ __forceinline__ uint2 ld_pair_sys(const uint2 *p)
{
    unsigned long long v;
    asm volatile("ld.relaxed.sys.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return make_uint2((uint32_t)v, (uint32_t)(v >> 32));
}
__device__ __forceinline__ void st_pair_sys(uint2 *p, uint32_t word, uint32_t stamp)
{
    asm volatile("st.relaxed.sys.global.u64 [%0], %1;" :: "l"(p), "l"(((unsigned long long)stamp << 32) | word) : "memory");
}

// after half-step 1: bottom row -> rank below (its side 1), top row -> rank above (its side 0)
__global__ void __launch_bounds__(SLAB_THREADS) slab_publish(const __grid_constant__ SlabParams p)
{
    const int W = p.L >> 2;
    const uint32_t *bottom = reinterpret_cast<const uint32_t *>(p.sigma);
    const uint32_t *top = reinterpret_cast<const uint32_t *>(p.sigma + (size_t)(p.n_rows - 1) * p.L);
    uint2 *dst_b = p.to_below + ((size_t)(2 + (p.stamp & 1u))) * W;     // side 1 of the rank below
    uint2 *dst_a = p.to_above + ((size_t)(0 + (p.stamp & 1u))) * W;     // side 0 of the rank above
    for (int i = blockIdx.x * SLAB_THREADS + threadIdx.x; i < W; i += gridDim.x * SLAB_THREADS) {
        st_pair_sys(dst_b + i, bottom[i], p.stamp);
        st_pair_sys(dst_a + i, top[i], p.stamp);
    }
}

// before half-step 0: wait for the neighbours' rows of this exchange, put them into the arrays (sigma rows -1 and n_rows)
// and redraw tau row n_rows from them (eq. (15), the same rule and the same random words as the rank above uses).
// One thread per 16-byte vector; each polls exactly the pairs it needs (its four words of either row, and the word left
// of its vector in the upper row for the horizontal edge spin).
__global__ void __launch_bounds__(SLAB_THREADS) slab_edge(const __grid_constant__ SlabParams p)
{
    const int L = p.L, W = L >> 2, nvec = W >> 2;
    const uint2 *below = p.inbox + ((size_t)(0 + (p.stamp & 1u))) * W;
    const uint2 *above = p.inbox + ((size_t)(2 + (p.stamp & 1u))) * W;
    uint32_t *row_m1 = reinterpret_cast<uint32_t *>(p.sigma) - W;
    uint32_t *row_n = reinterpret_cast<uint32_t *>(p.sigma + (size_t)p.n_rows * L);
    const uint32_t *row_top = reinterpret_cast<const uint32_t *>(p.sigma + (size_t)(p.n_rows - 1) * L);
    uint32_t *tau_n = reinterpret_cast<uint32_t *>(p.tau + (size_t)p.n_rows * L);
    uint32_t gr = p.row0 + (uint32_t)p.n_rows;                        // global row of tau row n_rows
    if (gr >= (uint32_t)L) gr -= (uint32_t)L;
    ChainKeys ck = make_chain_keys(p.keys, p.chain);
    for (int cv = blockIdx.x * SLAB_THREADS + threadIdx.x; cv < nvec; cv += gridDim.x * SLAB_THREADS) {
        uint32_t lo[4], up[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            uint2 a, b;
            do { a = ld_pair_sys(below + 4 * cv + j); b = ld_pair_sys(above + 4 * cv + j); } while (a.y != p.stamp || b.y != p.stamp);
            lo[j] = a.x;
            up[j] = b.x;
        }
        *reinterpret_cast<uint4 *>(row_m1 + 4 * cv) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
        *reinterpret_cast<uint4 *>(row_n + 4 * cv) = make_uint4(up[0], up[1], up[2], up[3]);
        if (!p.redraw) continue;
        uint2 e;
        const uint2 *pe = above + (cv == 0 ? W - 1 : 4 * cv - 1);
        do { e = ld_pair_sys(pe); } while (e.y != p.stamp);
        const uint4 v4 = *reinterpret_cast<const uint4 *>(row_top + 4 * cv);          // sigma row n_rows-1: the down neighbours
        const uint32_t vw[4] = {v4.x, v4.y, v4.z, v4.w};
        uint32_t o[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const uint32_t sw = up[j];
            const uint32_t hw = __funnelshift_l(j == 0 ? e.x : up[j - 1], sw, 8);      // left neighbours
            uint32_t rw[4];
            philox_site_words(gr * (uint32_t)W + 4u * (uint32_t)cv + (uint32_t)j, p.keys, ck, rw);
            uint32_t out = 0;
#pragma unroll
            for (int b = 0; b < 4; ++b) {
                const int ms = (sw >> (8 * b + 1)) & 1, mh = (hw >> (8 * b + 1)) & 1, mv = (vw[j] >> (8 * b + 1)) & 1;   // minus flags
                const uint32_t T = p.utab[2 * (2 - mh - mv) + (1 - ms)];               // T[2k + c]
                out |= (rw[b] < T ? 0x01u : 0xFFu) << (8 * b);
            }
            o[j] = out;
        }
        *reinterpret_cast<uint4 *>(tau_n + 4 * cv) = make_uint4(o[0], o[1], o[2], o[3]);
    }
}

} // namespace shaken
