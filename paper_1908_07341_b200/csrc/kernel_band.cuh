// kernel_band.cuh -- mid-size lattices (128 < L <= 2048, few chains): a half-step is a microsecond of work, so one
// launch per half-step is mostly launch latency (cfg 2: 4.9 us per launch for 0.8 us of arithmetic).  Here the whole
// run is ONE cooperative launch.  Every CTA owns a band of rows of one chain and keeps both sublattices of the band in
// shared memory.  The fields of eq. (14) reach one row across a band edge in each half-step: the
// down row in half 0, the up row in half 1.  Because a site's random word is a function of (seed, chain, step, half,
// site) alone, a band can redraw the tau row ABOVE itself redundantly (from the sigma row above, which it receives, and
// its own top sigma row), so bands exchange only sigma rows, ONCE per full step: after half-step 1 a band publishes its
// bottom and top sigma rows, and in the next half-step 0 it needs the top row of the band below and the bottom row of
// the band above.  One hand-over latency per step instead of two, at the price of one extra row of half-step 0.
//
// The hand-over goes through a small global buffer in "data + stamp" form: every 64-bit store carries a spin word and
// the step's stamp, so a reader that sees the stamp has the data (no fence, no separate flag; see ld_pair / st_pairs2).
// The thread that computes a vector of a boundary row polls for exactly the words it needs and the thread that computed
// a published vector stores it itself: no staging warp, no barrier on the exchange path.  Work is ordered so that the
// rows that wait for a neighbour come LAST in half-step 0 and the rows a neighbour waits for come FIRST in half-step 1:
// the hand-over latency hides behind the interior rows.  There is no grid-wide barrier: only neighbouring bands wait
// for each other, which is why all CTAs must be co-resident -- the cooperative launch guarantees it.
// Site -> random word mapping, thresholds and rule are those of kernel_i8.cuh; only the schedule differs.
#pragma once
#include <type_traits>

#include "kernels_common.cuh"

namespace shaken {

constexpr int BAND_THREADS = 512;
constexpr int BAND_L_MAX = 2048;   // W = L/4 <= 512 words per row

struct BandParams {
    uint8_t *sigma;          // [n_chains][L][L] int8
    uint8_t *tau;
    int L;
    int n_chains;
    uint32_t chain0;
    unsigned long long t0;   // global full-step index of the first step of this launch
    long long n_steps;
    long long obs_every;     // 0 = never
    long long *rec;          // first free record slot, [record][n_chains][6] (zeroed)
    const uint32_t *gtab;    // per-chain tables [n_chains][8] (natural order) or nullptr: utab
    uint32_t utab[8];
    StepKeys keys;           // only k0[], k1[] are used
    int bpc;                 // bands per chain
    int rows_per_band;
    uint2 *xtop;             // [2][n_bands][L/4] {word, stamp}: TOP sigma row of each band after a full step (by parity of the step)
    uint2 *xbot;             // [2][n_bands][L/4] {word, stamp}: BOTTOM sigma row of each band after a full step
    uint32_t magicV;         // floor(2^32 / (L/16)) + 1: c / (L/16) == __umulhi(c, magicV) for the small c used here
    uint32_t magicW;         // floor(2^32 / (L/4)) + 1: the same for word indices c / W
    unsigned long long slot_group;   // band_flow_i8: nibble s = the group (row) that warp slot s works for, 15 = none (flow_slot_groups)
    uint32_t stamp0;         // stamps of this launch are stamp0 + 1 .. stamp0 + n_steps (never seen before in xtop, xbot)
};

// dynamic shared memory: sigma rows r0-1 .. r1 (halo below, band, halo above) and tau rows r0 .. r1 (band, redundant row)
__host__ __device__ inline size_t band_smem_bytes(int L, int rows_per_band) { return (size_t)(2 * rows_per_band + 3) * (size_t)(L / 4) * sizeof(uint32_t); }

// A {word, stamp} pair crosses between CTAs as ONE naturally aligned 64-bit scalar, relaxed at gpu scope on both sides:
// the PTX memory model makes such an access single-copy atomic (the elements of a vector access count as separate scalar
// accesses, which is all that is needed: every pair validates itself), so a reader that sees the stamp of a step has
// the spin word written with it.  No fence, no flag.
__device__ __forceinline__ void ld_pairs2(const uint2 *p, uint2 &a, uint2 &b)
{
    unsigned long long x, y;
    asm volatile("ld.relaxed.gpu.global.v2.u64 {%0, %1}, [%2];" : "=l"(x), "=l"(y) : "l"(p) : "memory");
    a = make_uint2((uint32_t)x, (uint32_t)(x >> 32));
    b = make_uint2((uint32_t)y, (uint32_t)(y >> 32));
}
__device__ __forceinline__ uint2 ld_pair(const uint2 *p)
{
    unsigned long long v;
    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return make_uint2((uint32_t)v, (uint32_t)(v >> 32));
}
__device__ __forceinline__ void st_pair(uint2 *p, uint32_t word, uint32_t stamp)
{
    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" :: "l"(p), "l"(((unsigned long long)stamp << 32) | word) : "memory");
}
__device__ __forceinline__ void st_pairs2(uint2 *p, uint32_t w0, uint32_t w1, uint32_t stamp)
{
    const unsigned long long s = (unsigned long long)stamp << 32;
    asm volatile("st.relaxed.gpu.global.v2.u64 [%0], {%1, %2};" :: "l"(p), "l"(s | w0), "l"(s | w1) : "memory");
}

__global__ void __launch_bounds__(BAND_THREADS, 1) band_run_i8(const __grid_constant__ BandParams p)
{
    extern __shared__ __align__(16) uint32_t smem[];
    __shared__ uint2 s_pair[64][32];              // paired thresholds, lane-replicated (see kernel_i8.cuh)
    __shared__ long long s_red[BAND_THREADS / 32][6];
    __shared__ int s_acc[6];                      // the band's partial sums of the record in progress

    const int L = p.L, W = L >> 2;
    const int band = blockIdx.x, chain = band / p.bpc, k = band - chain * p.bpc;
    const int r0 = k * p.rows_per_band;
    const int nr = min(L, r0 + p.rows_per_band) - r0;                 // rows of this band (>= 1)
    const int below = chain * p.bpc + (k == 0 ? p.bpc - 1 : k - 1);   // band that owns row r0 - 1
    const int above = chain * p.bpc + (k == p.bpc - 1 ? 0 : k + 1);   // band that owns row r0 + nr
    const int nb = gridDim.x;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t lane8 = (uint32_t)lane * 8u;

    uint32_t *sg = smem;                          // sigma rows: index 0 = row r0-1 (halo), 1 .. nr = the band, nr+1 = row r0+nr (halo)
    uint32_t *ta = smem + (p.rows_per_band + 2) * W;   // tau rows: index 0 .. nr-1 = the band, nr = row r0+nr (redrawn redundantly)

    const size_t plane = (size_t)L * L;
    uint32_t *gs = reinterpret_cast<uint32_t *>(p.sigma + (size_t)chain * plane);
    uint32_t *gt = reinterpret_cast<uint32_t *>(p.tau + (size_t)chain * plane);
    const int row_below = r0 == 0 ? L - 1 : r0 - 1, row_above = r0 + nr == L ? 0 : r0 + nr;
    for (int i = tid; i < nr * W; i += BAND_THREADS) { sg[W + i] = gs[(size_t)r0 * W + i]; ta[i] = gt[(size_t)r0 * W + i]; }
    for (int i = tid; i < W; i += BAND_THREADS) { sg[i] = gs[(size_t)row_below * W + i]; sg[(nr + 1) * W + i] = gs[(size_t)row_above * W + i]; }
    for (int t = tid; t < 64 * 32; t += BAND_THREADS) {
        const int e = t >> 5;
        uint32_t T2[2];
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const int c = h ? (e >> 3) : (e & 7);
            const int ms = c & 1, mh = (c >> 1) & 1, mv = c >> 2;
            const int idx = 2 * (2 - mh - mv) + (1 - ms);          // T[2k + c]
            T2[h] = p.gtab ? p.gtab[(size_t)chain * 8 + idx] : p.utab[idx];
        }
        s_pair[e][t & 31] = make_uint2(T2[0], T2[1]);
    }
    if (tid < 6) s_acc[tid] = 0;
    __syncthreads();

    uint32_t xa2 = 0, xb0 = 0;
    ChainKeys ck = {0u, 0u};

    // one 16-byte vector (16 sites = 4 Philox calls, interleaved by the compiler) of the new sublattice:
    // s4 = own words, v4 = vertical neighbours, e = the word holding the horizontal edge spin, n = Philox counter of word 0.
    auto update_vector = [&](const int half, const uint4 s4, const uint4 v4, const uint32_t e, const uint32_t n) -> uint4 {
        const uint32_t w[4] = {s4.x, s4.y, s4.z, s4.w}, vw[4] = {v4.x, v4.y, v4.z, v4.w};
        uint32_t o[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const uint32_t hl = __funnelshift_l(j == 0 ? e : w[j - 1], w[j], 8);      // left neighbours (half 0)
            const uint32_t hr = __funnelshift_r(w[j], j == 3 ? e : w[j + 1], 8);      // right neighbours (half 1)
            const uint32_t hw = half ? hr : hl;
            const uint32_t y = (hw & 0x40044004u) | (vw[j] & ~0x40044004u);
            const uint32_t z = ((w[j] & 0x20022002u) | (y & ~0x20022002u)) & 0xE00EE00Eu;
            const uint32_t o01 = __dp4a(z, 0x00004080u, lane8), o23 = __dp4a(z, 0x40800000u, lane8);
            const uint2 t01 = *reinterpret_cast<const uint2 *>(reinterpret_cast<const char *>(s_pair) + o01);
            const uint2 t23 = *reinterpret_cast<const uint2 *>(reinterpret_cast<const char *>(s_pair) + o23);
            uint32_t rw[4];
            philox_site_words(n + (uint32_t)j, p.keys, xa2, xb0, ck, rw);
            uint32_t out = 0x01010101u;
            out = add_if_not_less(out, rw[0], t01.x, 0xFEu);
            out = add_if_not_less(out, rw[1], t01.y, 0xFEu << 8);
            out = add_if_not_less(out, rw[2], t23.x, 0xFEu << 16);
            out = add_if_not_less(out, rw[3], t23.y, 0xFEu << 24);
            o[j] = out;
        }
        return make_uint4(o[0], o[1], o[2], o[3]);
    };

    // The same vector in two stages, for the rows that wait for a neighbour: a site's random word does not depend on any
    // spin, so the Philox calls (85 % of the instructions) are made BEFORE the wait and only the table lookups and the
    // compares are left for after it.
    auto draw = [&](const uint32_t n, uint32_t (&R)[4][4]) {
#pragma unroll
        for (int j = 0; j < 4; ++j) philox_site_words(n + (uint32_t)j, p.keys, xa2, xb0, ck, R[j]);
    };
    auto apply0 = [&](const uint4 s4, const uint4 v4, const uint32_t e, const uint32_t (&R)[4][4]) -> uint4 {
        const uint32_t w[4] = {s4.x, s4.y, s4.z, s4.w}, vw[4] = {v4.x, v4.y, v4.z, v4.w};
        uint32_t o[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const uint32_t hw = __funnelshift_l(j == 0 ? e : w[j - 1], w[j], 8);      // left neighbours
            const uint32_t y = (hw & 0x40044004u) | (vw[j] & ~0x40044004u);
            const uint32_t z = ((w[j] & 0x20022002u) | (y & ~0x20022002u)) & 0xE00EE00Eu;
            const uint32_t o01 = __dp4a(z, 0x00004080u, lane8), o23 = __dp4a(z, 0x40800000u, lane8);
            const uint2 t01 = *reinterpret_cast<const uint2 *>(reinterpret_cast<const char *>(s_pair) + o01);
            const uint2 t23 = *reinterpret_cast<const uint2 *>(reinterpret_cast<const char *>(s_pair) + o23);
            uint32_t out = 0x01010101u;
            out = add_if_not_less(out, R[j][0], t01.x, 0xFEu);
            out = add_if_not_less(out, R[j][1], t01.y, 0xFEu << 8);
            out = add_if_not_less(out, R[j][2], t23.x, 0xFEu << 16);
            out = add_if_not_less(out, R[j][3], t23.y, 0xFEu << 24);
            o[j] = out;
        }
        return make_uint4(o[0], o[1], o[2], o[3]);
    };

    // block-wide sums of up to six int partials into one record (int64 atomics: bands of a chain share the record)
    auto reduce_to = [&](long long *dst, const int (&v)[6], const int first, const int count) {
#pragma unroll
        for (int j = 0; j < 6; ++j) {
            const int w = __reduce_add_sync(0xFFFFFFFFu, v[j]);
            if (lane == 0) s_red[warp][j] = w;
        }
        __syncthreads();
        if (tid < count) {
            long long tot = 0;
            for (int w = 0; w < BAND_THREADS / 32; ++w) tot += s_red[w][first + tid];
            atomicAdd(reinterpret_cast<unsigned long long *>(dst + first + tid), (unsigned long long)tot);
        }
        __syncthreads();
    };

    // C_x, C_y of the record taken after the previous step: sigma is final, sg row 0 holds the new sigma row below the band
    auto bond_sums = [&](long long *dst) {
        int v[6] = {0, 0, 0, 0, 0, 0};
        for (int c = tid; c < nr * W; c += BAND_THREADS) {
            const int r = (int)__umulhi((uint32_t)c, p.magicW), cw = c - r * W;
            const uint32_t *row = sg + (r + 1) * W;
            const uint32_t s0 = row[cw];
            v[4] = __dp4a((int)s0, (int)__funnelshift_l(row[cw == 0 ? W - 1 : cw - 1], s0, 8), v[4]);   // sigma_x sigma_{x left}
            v[5] = __dp4a((int)s0, (int)row[cw - W], v[5]);                                              // sigma_x sigma_{x down}
        }
        reduce_to(dst, v, 4, 2);
    };

    const int nvec = W >> 2;                      // vectors per row
    const int n0 = (nr + 1) * nvec, n1 = nr * nvec;   // vectors of half-step 0 (band + redundant row) and of half-step 1
    long long *pending = nullptr;
    long long nrec = 0;
    // full steps until the next recorded one: a countdown instead of a 64-bit modulo per step
    long long until_rec = p.obs_every > 0 ? p.obs_every - (long long)(p.t0 % (unsigned long long)p.obs_every) : 0;
    // The sums of a recorded step are taken where their operands are in registers anyway: M_sigma, M_tau, E_J, E_q in the
    // half-step 1 that produces the recorded sigma, C_x and C_y in the NEXT half-step 0, which reads that sigma together
    // with its left and down neighbours (incl. the neighbour band's new row).  Per-thread int partials -> warp sum ->
    // shared-memory atomics; after the block barrier that ends the half-step anyway, six threads add the band's totals to
    // the record (int64 atomics: the bands of a chain share it).  No extra pass, no extra barrier.
    auto add_partials = [&](const int (&v)[6], const int first, const int count) {
        for (int j = first; j < first + count; ++j) {
            const int w = __reduce_add_sync(0xFFFFFFFFu, v[j]);
            if (lane == 0 && w != 0) atomicAdd(&s_acc[j], w);
        }
    };
    auto flush_partials = [&](long long *dst, const int first, const int count) {     // right after a block barrier
        if (tid >= first && tid < first + count) {
            atomicAdd(reinterpret_cast<unsigned long long *>(dst + tid), (unsigned long long)(long long)s_acc[tid]);
            s_acc[tid] = 0;                       // next written after at least one more block barrier
        }
    };
#pragma unroll 1
    for (long long s = 0; s < p.n_steps; ++s) {
        const unsigned long long t = p.t0 + (unsigned long long)s;
        const bool rec = p.obs_every > 0 && --until_rec == 0;                        // block-uniform
        if (rec) until_rec = p.obs_every;
        // hand-over buffers: the rows published after step s-1 (parity (s-1) & 1) are read now
        const uint32_t stamp_in = p.stamp0 + (uint32_t)s;
        const uint2 *in_below = p.xtop + ((size_t)((s + 1) & 1) * nb + below) * W;   // top row of the band below = row r0-1
        const uint2 *in_above = p.xbot + ((size_t)((s + 1) & 1) * nb + above) * W;   // bottom row of the band above = row r0+nr

        // ---- half-step 0: tau <- sigma, field from the down and left neighbours (eq. (15)); rows 0 .. nr of the tau array.
        // Order: the interior rows first, then row 0 (needs the sigma row below the band), then row nr (needs the sigma
        // row above the band): those two wait for the neighbours' rows of the previous step (none on the first step of a
        // launch: the halo rows came from global memory).
        device_half_step_keys(p.keys, 2ull * t, p.chain0 + (uint32_t)chain, xa2, xb0, ck);
        int v[6] = {0, 0, 0, 0, 0, 0};
#pragma unroll 1
        for (int c = tid; c < n0; c += BAND_THREADS) {
            const int kk = (int)__umulhi((uint32_t)c, p.magicV), cv = c - kk * nvec;
            const int i = kk < nr - 1 ? kk + 1 : (kk == nr - 1 ? 0 : nr);      // tau row
            const uint32_t *self = sg + (i + 1) * W, *downr = sg + i * W;
            int gr = r0 + i;
            if (gr >= L) gr -= L;
            const uint32_t n = (uint32_t)gr * (uint32_t)W + 4u * (uint32_t)cv;
            uint4 o, s4, v4;
            uint32_t e;
            if (s > 0 && i == 0) {
                // vertical neighbours from the band below, straight from the hand-over buffer; random words first
                uint32_t R[4][4];
                draw(n, R);
                uint2 a, b, c2, d;
                do { ld_pairs2(in_below + 4 * cv, a, b); ld_pairs2(in_below + 4 * cv + 2, c2, d); }
                while (a.y != stamp_in || b.y != stamp_in || c2.y != stamp_in || d.y != stamp_in);
                v4 = make_uint4(a.x, b.x, c2.x, d.x);
                *reinterpret_cast<uint4 *>(sg + 4 * cv) = v4;                  // (row index 0 of sg mirrors the row below the band)
                s4 = *reinterpret_cast<const uint4 *>(self + 4 * cv);
                e = self[cv == 0 ? W - 1 : 4 * cv - 1];
                o = apply0(s4, v4, e, R);
            } else if (s > 0 && i == nr) {
                // the row above the band: own words and the left edge spin from the band above; random words first
                uint32_t R[4][4];
                draw(n, R);
                uint2 a, b, c2, d, ee;
                const uint2 *pe = in_above + (cv == 0 ? W - 1 : 4 * cv - 1);
                do { ld_pairs2(in_above + 4 * cv, a, b); ld_pairs2(in_above + 4 * cv + 2, c2, d); ee = ld_pair(pe); }
                while (a.y != stamp_in || b.y != stamp_in || c2.y != stamp_in || d.y != stamp_in || ee.y != stamp_in);
                s4 = make_uint4(a.x, b.x, c2.x, d.x);
                v4 = *reinterpret_cast<const uint4 *>(downr + 4 * cv);
                e = ee.x;
                o = apply0(s4, v4, e, R);
            } else {
                s4 = *reinterpret_cast<const uint4 *>(self + 4 * cv);
                v4 = *reinterpret_cast<const uint4 *>(downr + 4 * cv);
                e = self[cv == 0 ? W - 1 : 4 * cv - 1];
                o = update_vector(0, s4, v4, e, n);
            }
            *reinterpret_cast<uint4 *>(ta + i * W + 4 * cv) = o;
            if (__builtin_expect(pending != nullptr, 0) && i < nr) {
                // C_x, C_y of the record taken after the previous step: sigma_x sigma_{x left}, sigma_x sigma_{x down}
                const uint32_t w[4] = {s4.x, s4.y, s4.z, s4.w}, dw[4] = {v4.x, v4.y, v4.z, v4.w};
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    v[4] = __dp4a((int)w[j], (int)__funnelshift_l(j == 0 ? e : w[j - 1], w[j], 8), v[4]);
                    v[5] = __dp4a((int)w[j], (int)dw[j], v[5]);
                }
            }
        }
        if (pending) add_partials(v, 4, 2);
        __syncthreads();
        if (pending) { flush_partials(pending, 4, 2); pending = nullptr; }

        // ---- half-step 1: sigma <- tau, up and right neighbours (eq. (16)); rows 0 .. nr-1.  Order: the top row and the
        // bottom row first -- the neighbours wait for them -- each vector published by the thread that computed it.
        device_half_step_keys(p.keys, 2ull * t + 1ull, p.chain0 + (uint32_t)chain, xa2, xb0, ck);
        const uint32_t stamp_out = p.stamp0 + (uint32_t)s + 1u;
        uint2 *out_top = p.xtop + ((size_t)(s & 1) * nb + band) * W;
        uint2 *out_bot = p.xbot + ((size_t)(s & 1) * nb + band) * W;
#pragma unroll 1
        for (int c = tid; c < n1; c += BAND_THREADS) {
            const int kk = (int)__umulhi((uint32_t)c, p.magicV), cv = c - kk * nvec;
            const int i = kk == 0 ? nr - 1 : (kk == 1 ? 0 : kk - 1);          // sigma row
            const uint32_t *self = ta + i * W;
            const uint4 s4 = *reinterpret_cast<const uint4 *>(self + 4 * cv);
            const uint4 v4 = *reinterpret_cast<const uint4 *>(self + W + 4 * cv);
            const uint32_t e = self[cv == nvec - 1 ? 0 : 4 * cv + 4];
            const uint4 o = update_vector(1, s4, v4, e, (uint32_t)(r0 + i) * (uint32_t)W + 4u * (uint32_t)cv);
            *reinterpret_cast<uint4 *>(sg + (i + 1) * W + 4 * cv) = o;
            if (i == nr - 1) { st_pairs2(out_top + 4 * cv, o.x, o.y, stamp_out); st_pairs2(out_top + 4 * cv + 2, o.z, o.w, stamp_out); }
            if (i == 0) { st_pairs2(out_bot + 4 * cv, o.x, o.y, stamp_out); st_pairs2(out_bot + 4 * cv + 2, o.z, o.w, stamp_out); }
            if (__builtin_expect(rec, 0)) {
                // M_sigma, M_tau, E_J = sigma'_x (tau_{x up} + tau_{x right}), E_q = sigma'_x tau_x  (row nr of ta is the redrawn row above the band)
                const uint32_t ow[4] = {o.x, o.y, o.z, o.w}, tw[4] = {s4.x, s4.y, s4.z, s4.w}, uw[4] = {v4.x, v4.y, v4.z, v4.w};
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    v[0] = __dp4a((int)ow[j], 0x01010101, v[0]);
                    v[1] = __dp4a((int)tw[j], 0x01010101, v[1]);
                    v[2] = __dp4a((int)ow[j], (int)uw[j], v[2]);
                    v[2] = __dp4a((int)ow[j], (int)__funnelshift_r(tw[j], j == 3 ? e : tw[j + 1], 8), v[2]);
                    v[3] = __dp4a((int)ow[j], (int)tw[j], v[3]);
                }
            }
        }
        if (rec) add_partials(v, 0, 4);
        __syncthreads();
        if (rec) {
            long long *dst = p.rec + ((size_t)nrec * p.n_chains + chain) * 6;
            flush_partials(dst, 0, 4);
            pending = dst;
            ++nrec;
        }
    }
    if (pending) {
        // the last step was recorded: fetch the final sigma row below the band (the neighbour published it after its last step)
        const uint32_t stamp_in = p.stamp0 + (uint32_t)p.n_steps;
        const uint2 *in_below = p.xtop + ((size_t)((p.n_steps + 1) & 1) * nb + below) * W;
        for (int i = tid; i < W; i += BAND_THREADS) {
            uint2 a;
            do { a = ld_pair(in_below + i); } while (a.y != stamp_in);
            sg[i] = a.x;
        }
        __syncthreads();
        bond_sums(pending);
    }
    for (int i = tid; i < nr * W; i += BAND_THREADS) { gs[(size_t)r0 * W + i] = sg[W + i]; gt[(size_t)r0 * W + i] = ta[i]; }
}

} // namespace shaken
