// kernel_band.cuh -- mid-size lattices (128 < L <= 2048, few chains): a half-step is a microsecond of work, so one
// launch per half-step is mostly launch latency (cfg 2: 4.9 us per launch for 0.8 us of arithmetic).  Here the whole
// run is ONE cooperative launch.  Every CTA owns a band of rows of one chain and keeps both sublattices of the band in
// shared memory; per half-step it needs exactly one row from a neighbouring band (eq. (14): the field
// uses the down row in half 0, the up row in half 1), which the neighbour publishes through a small global buffer in
// "data + stamp" form: every 64-bit store carries the spin word and the half-step stamp, so a reader that sees the
// stamp has the data (no fence, no separate flag; see st_pair).  A CTA computes the row its neighbour waits for first, one word per
// thread, and every word is published by the thread that computed it; one warp does no arithmetic and polls for the
// row the CTA itself needs next.  There is no grid-wide barrier: only neighbouring
// bands wait for each other, which is why all CTAs must be co-resident -- the cooperative launch guarantees it.
// Site -> random word mapping, thresholds and rule are those of kernel_i8.cuh; only the schedule differs.
#pragma once
#include "kernels_common.cuh"

namespace shaken {

constexpr int BAND_THREADS = 512;
constexpr int BAND_L_MAX = 2048;   // W = L/4 <= 512: a published row is at most 8 words per lane of the collecting warp

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
    uint2 *xs;               // [2][n_bands][L/4] {word, stamp}: last sigma row of each band after half-step 1
    uint2 *xt;               // [2][n_bands][L/4] {word, stamp}: first tau row of each band after half-step 0
    uint32_t magicV;         // floor(2^32 / (L/16)) + 1: the same for vector indices c / (L/16)
    uint32_t magicW;         // floor(2^32 / (L/4)) + 1: c / W == __umulhi(c, magicW) for the small c used here
    uint32_t stamp0;         // stamps of this launch are stamp0 + 1 .. stamp0 + 2 n_steps (never seen before in xs, xt)
};

// A {word, stamp} pair crosses between CTAs as ONE naturally aligned 64-bit scalar access, relaxed at gpu scope on both
// sides: the PTX memory model makes such an access single-copy atomic (a vector access would count as two scalar ones),
// so a reader that sees the stamp of a half-step has the spin word written with it.  No fence, no flag.
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

__global__ void __launch_bounds__(BAND_THREADS, 1) band_run_i8(const __grid_constant__ BandParams p)
{
    extern __shared__ __align__(16) uint32_t smem[];
    __shared__ uint2 s_pair[64][32];              // paired thresholds, lane-replicated (see kernel_i8.cuh)
    __shared__ long long s_red[BAND_THREADS / 32][6];

    const int L = p.L, W = L >> 2;
    const int band = blockIdx.x, chain = band / p.bpc, k = band - chain * p.bpc;
    const int r0 = k * p.rows_per_band;
    const int nr = min(L, r0 + p.rows_per_band) - r0;
    const int down = chain * p.bpc + (k == 0 ? p.bpc - 1 : k - 1);
    const int up = chain * p.bpc + (k == p.bpc - 1 ? 0 : k + 1);
    const int nb = gridDim.x;
    const int ncalls = nr * W;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t lane8 = (uint32_t)lane * 8u;
    const bool duty_warp = warp == BAND_THREADS / 32 - 1;
    constexpr int WORKERS = BAND_THREADS - 32;   // polls for the neighbour's row while the other warps compute

    uint32_t *sg = smem;                          // sigma band [nr][W]
    uint32_t *ta = smem + p.rows_per_band * W;    // tau band
    uint32_t *hs = ta + p.rows_per_band * W;      // sigma row below the band
    uint32_t *ht = hs + W;                        // tau row above the band

    const size_t plane = (size_t)L * L;
    uint32_t *gs = reinterpret_cast<uint32_t *>(p.sigma + (size_t)chain * plane);
    uint32_t *gt = reinterpret_cast<uint32_t *>(p.tau + (size_t)chain * plane);
    for (int i = tid; i < ncalls; i += BAND_THREADS) { sg[i] = gs[(size_t)r0 * W + i]; ta[i] = gt[(size_t)r0 * W + i]; }
    for (int i = tid; i < W; i += BAND_THREADS) hs[i] = gs[(size_t)(r0 == 0 ? L - 1 : r0 - 1) * W + i];
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
    __syncthreads();

    uint32_t xa2 = 0, xb0 = 0;
    ChainKeys ck = {0u, 0u};

    // one word (4 sites) of the new sublattice
    auto update_word = [&](const uint32_t sw, const uint32_t hw, const uint32_t vw, const uint32_t n) -> uint32_t {
        const uint32_t y = (hw & 0x40044004u) | (vw & ~0x40044004u);
        const uint32_t z = ((sw & 0x20022002u) | (y & ~0x20022002u)) & 0xE00EE00Eu;
        const uint32_t o01 = __dp4a(z, 0x00004080u, lane8), o23 = __dp4a(z, 0x40800000u, lane8);
        const uint2 t01 = *reinterpret_cast<const uint2 *>(reinterpret_cast<const char *>(s_pair) + o01);
        const uint2 t23 = *reinterpret_cast<const uint2 *>(reinterpret_cast<const char *>(s_pair) + o23);
        uint32_t rw[4];
        philox_site_words(n, p.keys, xa2, xb0, ck, rw);
        uint32_t out = 0x01010101u;
        out = add_if_not_less(out, rw[0], t01.x, 0xFEu);
        out = add_if_not_less(out, rw[1], t01.y, 0xFEu << 8);
        out = add_if_not_less(out, rw[2], t23.x, 0xFEu << 16);
        out = add_if_not_less(out, rw[3], t23.y, 0xFEu << 24);
        return out;
    };

    // One 16-byte vector (4 words = 16 sites = 4 Philox calls) per thread per trip, as in kernel_i8.cuh: the four
    // independent chains interleave, the horizontal neighbours of three of the four words are in registers already.
    // half 0: tau from sigma, rows ascending.  half 1: sigma from tau, rows walked from the last one down.
    // `half` is a run-time value on purpose: one copy of this code serves both half-steps and every trip.
    const int nvec = W >> 2, nvecs = nr * nvec;   // vectors per row, per band
    auto update_vector = [&](const int half, const int c, uint2 *xmine, const uint32_t stamp) {
        const uint32_t *src = half ? ta : sg;
        uint32_t *dst = half ? sg : ta;
        const uint32_t *halo = half ? ht : hs;
        const int rr = (int)__umulhi((uint32_t)c, p.magicV), cv = c - rr * nvec;
        const int r = half ? nr - 1 - rr : rr;
        const int at = r * W + 4 * cv;
        const uint4 s4 = *reinterpret_cast<const uint4 *>(src + at);
        const bool edge = half ? r == nr - 1 : r == 0;
        const uint4 v4 = *reinterpret_cast<const uint4 *>(edge ? halo + 4 * cv : src + (half ? at + W : at - W));
        const int ce = half ? (cv == nvec - 1 ? 0 : 4 * cv + 4) : (cv == 0 ? W - 1 : 4 * cv - 1);
        const uint32_t e = src[r * W + ce];
        const uint32_t w[4] = {s4.x, s4.y, s4.z, s4.w}, vw[4] = {v4.x, v4.y, v4.z, v4.w};
        const uint32_t n = (uint32_t)(r0 + r) * (uint32_t)W + 4u * (uint32_t)cv;
        uint32_t o[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const uint32_t hl = __funnelshift_l(j == 0 ? e : w[j - 1], w[j], 8);      // left neighbours (half 0)
            const uint32_t hr = __funnelshift_r(w[j], j == 3 ? e : w[j + 1], 8);      // right neighbours (half 1)
            o[j] = update_word(w[j], half ? hr : hl, vw[j], n + (uint32_t)j);
        }
        *reinterpret_cast<uint4 *>(dst + at) = make_uint4(o[0], o[1], o[2], o[3]);
        if (rr == 0) {                            // (tall bands only, see below) a vector of the row the neighbour waits for
#pragma unroll
            for (int j = 0; j < 4; ++j) st_pair(xmine + 4 * cv + j, o[j], stamp);
        }
    };

    // The first row in walking order (first tau row in half 0, last sigma row in half 1) is the one the neighbouring band
    // waits for and the only one that reads the incoming row: it is done one WORD per thread (a single Philox call, the
    // shortest latency there is), ahead of the vectors, and each word leaves at once for the neighbour as a
    // {word, stamp} pair -- no barrier on the critical path of the ring.
    auto boundary_word = [&](const int half, const int cw, uint2 *xmine, const uint32_t stamp) {
        const uint32_t *src = half ? ta : sg;
        uint32_t *dst = half ? sg : ta;
        const uint32_t *halo = half ? ht : hs;
        const int r = half ? nr - 1 : 0, at = r * W + cw;
        const uint32_t sw = src[at];
        const uint32_t e = src[r * W + (half ? (cw == W - 1 ? 0 : cw + 1) : (cw == 0 ? W - 1 : cw - 1))];
        const uint32_t hw = half ? __funnelshift_r(sw, e, 8) : __funnelshift_l(e, sw, 8);
        const uint32_t out = update_word(sw, hw, halo[cw], (uint32_t)(r0 + r) * (uint32_t)W + (uint32_t)cw);
        dst[at] = out;
        st_pair(xmine + cw, out, stamp);
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

    // C_x, C_y of the record taken after the previous step: sigma is final, hs holds the sigma row below the band
    auto bond_sums = [&](long long *dst) {
        int v[6] = {0, 0, 0, 0, 0, 0};
        for (int c = tid; c < ncalls; c += BAND_THREADS) {
            const int r = (int)__umulhi((uint32_t)c, p.magicW), cw = c - r * W;
            const uint32_t s0 = sg[c];
            const uint32_t e = sg[r * W + (cw == 0 ? W - 1 : cw - 1)];
            v[4] = __dp4a((int)s0, (int)__funnelshift_l(e, s0, 8), v[4]);             // sigma_x sigma_{x left}
            v[5] = __dp4a((int)s0, (int)(r == 0 ? hs[cw] : sg[c - W]), v[5]);         // sigma_x sigma_{x down}
        }
        reduce_to(dst, v, 4, 2);
    };

    // Receiving side of the exchange (polling warp only): copy the neighbour's published row into shared memory as soon
    // as every word carries this half-step's stamp.
    auto collect = [&](const uint2 *src, const uint32_t stamp, uint32_t *dst) {
        // W <= 512: at most two rounds of 8 words per lane.  The loads are unconditional (indices past the row are
        // clamped to its last word) and all eight are in flight together; a round is repeated until every word carries
        // the stamp.  (A version with predicated loads compiled into a loop that was 3.7x slower.)
        for (int i0 = 0; i0 < W; i0 += 256) {
            uint2 v[8];
            bool ok;
            do {
                ok = true;
#pragma unroll
                for (int j = 0; j < 8; ++j) v[j] = ld_pair(src + min(i0 + j * 32 + lane, W - 1));
#pragma unroll
                for (int j = 0; j < 8; ++j)
                    if (v[j].y != stamp) ok = false;
            } while (!ok);
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const int i = i0 + j * 32 + lane;
                if (i < W) dst[i] = v[j].x;
            }
        }
    };

    long long *pending = nullptr;
    long long nrec = 0;
    // full steps until the next recorded one: a countdown instead of a 64-bit modulo per step
    long long until_rec = p.obs_every > 0 ? p.obs_every - (long long)(p.t0 % (unsigned long long)p.obs_every) : 0;
#pragma unroll 1
    for (long long h = 0; h < 2 * p.n_steps; ++h) {
        const long long s = h >> 1;
        const int half = (int)(h & 1);
        const unsigned long long t = p.t0 + (unsigned long long)s;
        const int par = (int)(s & 1);
        // half 0: tau <- sigma, field from the down and left neighbours (eq. (15)); hs is in place (loaded at the start,
        // collected during the previous half-step 1 afterwards).  half 1: sigma <- tau, up and right neighbours (eq. (16)).
        if (half == 0 && pending) { bond_sums(pending); pending = nullptr; }
        device_half_step_keys(p.keys, 2ull * t + (unsigned long long)half, p.chain0 + (uint32_t)chain, xa2, xb0, ck);

        // half 0 hands the first tau row to the band below, half 1 the last sigma row to the band above; the row this
        // band needs next (tau above for half 1, sigma below for the next half 0 and for the bond sums) comes back the
        // same way.  hs is not read during half-step 1, ht not during half-step 0.
        const uint32_t stamp = p.stamp0 + (uint32_t)(h + 1);
        uint2 *xmine = (half ? p.xs : p.xt) + ((size_t)par * nb + band) * W;
        const uint2 *xnbr = (half ? p.xs : p.xt) + ((size_t)par * nb + (half ? down : up)) * W;
        // The last warp does no arithmetic: it polls for the neighbour's row from the start of the half-step, so the
        // handshake (one L2 round trip after the neighbour's first vectors are done) hides behind the other 15 warps.
        if (duty_warp) collect(xnbr, stamp, half ? hs : ht);
        else if (nvecs <= 3 * WORKERS) {
            // short bands: the hand-over is the critical path, so the neighbour's row goes first, word by word
#pragma unroll 1
            for (int cw = tid; cw < W; cw += WORKERS) boundary_word(half, cw, xmine, stamp);
#pragma unroll 1
            for (int c = nvec + tid; c < nvecs; c += WORKERS) update_vector(half, c, xmine, stamp);   // rows 1 .. nr-1
        } else {
            // tall bands: several trips of vectors hide the hand-over anyway; the row is part of the first trip
#pragma unroll 1
            for (int c = tid; c < nvecs; c += WORKERS) update_vector(half, c, xmine, stamp);
        }
        __syncthreads();

        // record (M_sigma, M_tau, E_J, E_q now; C_x, C_y at the start of the next half-step 0)
        if (half == 1 && p.obs_every > 0 && --until_rec == 0) {
            until_rec = p.obs_every;
            long long *dst = p.rec + ((size_t)nrec * p.n_chains + chain) * 6;
            int v[6] = {0, 0, 0, 0, 0, 0};
            for (int c = tid; c < ncalls; c += BAND_THREADS) {
                const int r = (int)__umulhi((uint32_t)c, p.magicW), cw = c - r * W;
                const uint32_t s0 = sg[c], t0w = ta[c];
                const uint32_t tu = r == nr - 1 ? ht[cw] : ta[c + W];
                const uint32_t tr = __funnelshift_r(t0w, ta[r * W + (cw == W - 1 ? 0 : cw + 1)], 8);
                v[0] = __dp4a((int)s0, 0x01010101, v[0]);
                v[1] = __dp4a((int)t0w, 0x01010101, v[1]);
                v[2] = __dp4a((int)s0, (int)tu, v[2]);
                v[2] = __dp4a((int)s0, (int)tr, v[2]);
                v[3] = __dp4a((int)s0, (int)t0w, v[3]);
            }
            reduce_to(dst, v, 0, 4);
            pending = dst;
            ++nrec;
        }
    }
    if (pending) bond_sums(pending);              // hs already holds the final sigma row below the band
    for (int i = tid; i < ncalls; i += BAND_THREADS) { gs[(size_t)r0 * W + i] = sg[i]; gt[(size_t)r0 * W + i] = ta[i]; }
}

} // namespace shaken
