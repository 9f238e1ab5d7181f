// kernel_flow.cuh -- the band path (kernel_band.cuh) as a DATA-FLOW schedule, for bands of at most 7 rows (cfg 2).
//
// band_run_i8 marches a CTA through a full step in two phases separated by block barriers; a row that needs a neighbour
// band's row makes the whole CTA wait for the hand-over (store -> L2 -> poll, ~0.35 us) once per step, and every barrier
// lines all warps up at the same pipeline stage.  Here a ROW of the band belongs to a fixed group of warps for the whole
// run (row i of sigma and row i of tau to group i; group nr redraws the redundant tau row above the band), and a group
// starts a half-step as soon as ITS inputs exist:
//   half-step 0 of row i (eq. (15)) needs sigma rows i (own) and i-1 (group i-1, or the band below),
//   half-step 1 of row i (eq. (16), :169-172)         needs tau   rows i (own) and i+1 (group i+1).
// Groups meet through named barriers in producer / consumer form: the consumer group `bar.sync`s on its barrier, which
// also collects its own warps (a vector's horizontal edge spin was written by the neighbouring thread), the producer
// group only `bar.arrive`s.  One barrier per group and half (X0_i, X1_i): 2 nr + 1 <= 15 hardware barriers, hence the
// limit of 7 rows.  There is no block-wide barrier inside the step loop, so the hand-over latency delays only the two
// groups that touch a neighbour band, and those have slack: the step time is bounded by the arithmetic, not by the sum
// of the phases.  Write-after-read hazards are covered by the same edges: group i overwrites tau row i in half-step 0 of
// step s+1 only after group i-1 arrived at X0_i, i.e. after its half-step 1 of step s, the last reader of that row;
// group i overwrites sigma row i in half-step 1 only after group i+1 arrived at X1_i, i.e. after its half-step 0.
// Records: per-warp partial sums go to a ring of shared-memory slots by atomics that count their contributors, and the LAST
// warp to deliver its part of a sum adds the band's total to the record in global memory (no barrier, no fence: `deliver`).
// Exchange protocol ({word, stamp} pairs), site -> random word mapping, thresholds and rule: exactly band_run_i8's.
#pragma once
#include "kernel_band.cuh"

namespace shaken {

constexpr int FLOW_MAX_ROWS = 7;           // rows per band: 2 * 7 + 1 named barriers (+ barrier 0)
constexpr int FLOW_BIAS = 2048;            // makes a warp's part of a sum non-negative (|part| <= 1024)
constexpr int FLOW_RING = 8;               // records in flight inside a band: groups drift at most nr + 1 half-steps apart

__device__ __forceinline__ void bar_sync_n(int id, int n) { __syncwarp(); asm volatile("bar.sync %0, %1;" :: "r"(id), "r"(n) : "memory"); }
__device__ __forceinline__ void bar_arrive_n(int id, int n) { __syncwarp(); asm volatile("bar.arrive %0, %1;" :: "r"(id), "r"(n) : "memory"); }

// host side: does the data-flow kernel apply to bands of rows_per_band rows of an L x L lattice?
__host__ __device__ inline bool flow_applies(int L, int rows_per_band)
{
    const int wpr = (L / 16 + 31) / 32;                              // warps per row
    return rows_per_band <= FLOW_MAX_ROWS && wpr * (rows_per_band + 1) <= BAND_THREADS / 32;
}

// Which warps work for which group.  A slot = wpr consecutive warps; slot s sits on SM sub-partition(s) s % ncol (ncol = 4
// sub-partitions for one warp per row, 2 pairs of them for two).  Group 0 is on the critical cycle between neighbouring bands
// twice per step (it waits for the band below AND publishes the row that band waits for), the redundant last group has half
// the work of the others: group 0 goes where the load is lightest (alone, or with the last group), the others are spread
// evenly.  Measured at 1024^2: 1.98 us per step against 2.21 with groups simply in warp order (which puts group 0 on the
// fully loaded sub-partitions), 768^2 1.84 against 2.09, 512^2 1.37 against 1.50; all 35 / 70 placements were timed.
inline unsigned long long flow_slot_groups(int L, int rows_per_band)
{
    const int wpr = (L / 16 + 31) / 32, ncol = wpr == 1 ? 4 : 2, depth = (BAND_THREADS / 32) / wpr / ncol;
    const int ng = rows_per_band + 1;
    double load[4] = {0.0, 0.0, 0.0, 0.0};
    int used[4] = {0, 0, 0, 0};
    unsigned long long map = ~0ull;                                   // every nibble 15 = no group
    for (int g = 0; g < ng; ++g) {
        const double w = g == 0 ? 1.5 : (g == ng - 1 ? 0.5 : 1.0);    // group 0 counts as one and a half: it ends up lightest
        int best = -1;
        for (int c = 0; c < ncol; ++c)
            if (used[c] < depth && (best < 0 || load[c] < load[best])) best = c;
        const int slot = best + ncol * used[best];
        map = (map & ~(15ull << (4 * slot))) | ((unsigned long long)g << (4 * slot));
        load[best] += w;
        used[best]++;
    }
    return map;
}

__global__ void __launch_bounds__(BAND_THREADS, 1) band_flow_i8(const __grid_constant__ BandParams p)
{
    extern __shared__ __align__(16) uint32_t smem[];
    __shared__ uint2 s_pair[64][32];              // paired thresholds, lane-replicated (see kernel_i8.cuh)
    __shared__ int s_acc[FLOW_RING][6];           // the band's partial sums of the records in flight, with their contributor counts (see deliver)
    __shared__ long long s_red[BAND_THREADS / 32][2];

    const int L = p.L, W = L >> 2, nvec = W >> 2;
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
    for (int t = tid; t < FLOW_RING * 6; t += BAND_THREADS) (&s_acc[0][0])[t] = 0;
    __syncthreads();

    const int wpr = (nvec + 31) >> 5;             // warps per row
    const int slot = warp / wpr;                  // wpr consecutive warps form a slot; the host decides which group a slot serves
    const int gi = (int)((p.slot_group >> (4 * slot)) & 15ull);   // this warp's group = its row of the band (nr: the redundant row above)
    const int cv = (warp - slot * wpr) * 32 + lane; // its vector of the row
    const bool member = gi <= nr;                 // (warps beyond the last group only help with loading and storing)
    const bool mine = member && cv < nvec;
    const int gt_threads = wpr * 32;              // threads of one group
    const int n_contrib = nr * wpr;               // warps that deliver sums (groups 0 .. nr-1)
    const int X0 = 1 + gi, X1 = 1 + (p.rows_per_band + 1) + gi;      // this group's barriers of half-step 0 and 1

    uint32_t xa2 = 0, xb0 = 0;
    ChainKeys ck = {0u, 0u};
    auto draw = [&](const uint32_t n, uint32_t (&R)[4][4]) {
#pragma unroll
        for (int j = 0; j < 4; ++j) philox_site_words(n + (uint32_t)j, p.keys, xa2, xb0, ck, R[j]);
    };
    // s4 = own words, v4 = vertical neighbours, e = the word holding the horizontal edge spin, R = the vector's random words
    auto apply = [&](const int half, const uint4 s4, const uint4 v4, const uint32_t e, const uint32_t (&R)[4][4]) -> uint4 {
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
            uint32_t out = 0x01010101u;
            out = add_if_not_less(out, R[j][0], t01.x, 0xFEu);
            out = add_if_not_less(out, R[j][1], t01.y, 0xFEu << 8);
            out = add_if_not_less(out, R[j][2], t23.x, 0xFEu << 16);
            out = add_if_not_less(out, R[j][3], t23.y, 0xFEu << 24);
            o[j] = out;
        }
        return make_uint4(o[0], o[1], o[2], o[3]);
    };
    // A warp's part of a record.  The lanes' partial sums travel two to an int through the warp reduction (a * 65536 + b; a warp
    // holds 512 sites of a row, so |a|, |b| <= 1024).  Lane k then adds sum k to its word of the record's slot in shared
    // memory with ONE atomic that also counts the contributors: word = count * 2^26 + sum of (v + FLOW_BIAS).  The warp whose
    // atomic returns count == n_contrib - 1 is the last one for that word: old value + own part is the band's total, which it
    // adds to the record in global memory (int64 atomics: the bands of a chain share it), and it clears the word.  Data and count
    // in one atomic: no fence, no ordering between separate words to rely on.  Fields [first, first + 2 count) of the record.
    auto deliver = [&](const int x0, const int x1, const int count, const int first, const int slot, long long *dst) {
        const int w0 = __reduce_add_sync(0xFFFFFFFFu, x0);
        const int w1 = count > 1 ? __reduce_add_sync(0xFFFFFFFFu, x1) : 0;
        if (lane < 2 * count) {                                       // lane k carries field first + k
            const int wk = lane < 2 ? w0 : w1;
            const int lo = (int)(short)(wk & 0xFFFF);
            const int fk = (lane & 1) ? lo : (wk - lo) >> 16;
            unsigned int *acc = reinterpret_cast<unsigned int *>(&s_acc[slot][first + lane]);
            const unsigned int old = atomicAdd(acc, (1u << 26) + (unsigned int)(fk + FLOW_BIAS));
            if ((old >> 26) == (unsigned int)(n_contrib - 1)) {
                const int tot = (int)(old & 0x3FFFFFFu) + fk + FLOW_BIAS - n_contrib * FLOW_BIAS;
                *reinterpret_cast<volatile unsigned int *>(acc) = 0u;               // (the slot is next used FLOW_RING records later)
                atomicAdd(reinterpret_cast<unsigned long long *>(dst + first + lane), (unsigned long long)(long long)tot);
            }
        }
    };

    long long *pending = nullptr;                 // record that still lacks C_x, C_y (taken in the next half-step 0)
    int pending_slot = 0;
    long long nrec = 0;
    long long until_rec = p.obs_every > 0 ? p.obs_every - (long long)(p.t0 % (unsigned long long)p.obs_every) : 0;
    if (member) {
        int gr = r0 + gi;                         // the group's row of the lattice, for both sublattices
        if (gr >= L) gr -= L;
        const uint32_t n = (uint32_t)gr * (uint32_t)W + 4u * (uint32_t)(mine ? cv : 0);
        const int cvs = mine ? cv : 0;            // (lanes beyond the row compute nothing but pass every barrier)
        uint32_t *self_s = sg + (gi + 1) * W, *down_s = sg + gi * W;     // sigma rows gi and gi-1
        uint32_t *self_t = ta + gi * W;                                  // tau row gi; row gi+1 is self_t + W
        // one full step of this group; two copies of the body: steps that touch a record (rec: this step is recorded; pending: the
        // previous one was) carry the sums, the others do not pay for them (registers, schedule)
        auto step = [&](auto with_sums, const long long s, const bool rec) {
            constexpr bool SUMS = decltype(with_sums)::value;
            const unsigned long long t = p.t0 + (unsigned long long)s;
            const uint32_t stamp_in = p.stamp0 + (uint32_t)s;
            const uint2 *in_below = p.xtop + ((size_t)((s + 1) & 1) * nb + below) * W;   // top row of the band below = row r0-1
            const uint2 *in_above = p.xbot + ((size_t)((s + 1) & 1) * nb + above) * W;   // bottom row of the band above = row r0+nr
            int v[6] = {0, 0, 0, 0, 0, 0};
            uint32_t R[4][4];

            // ---- half-step 0: tau row gi <- sigma rows gi, gi-1.  Random words first: they depend on no spin.
            device_half_step_keys(p.keys, 2ull * t, p.chain0 + (uint32_t)chain, xa2, xb0, ck);
            if (mine) draw(n, R);
            if (s > 0) bar_sync_n(X0, gi >= 1 ? 2 * gt_threads : gt_threads);   // own sigma row complete; row gi-1 too
            if (mine) {
                uint4 s4, v4;
                uint32_t e;
                if (s > 0 && gi == 0) {
                    uint2 a, b, c2, d;                                  // the row below the band: from the band below
                    do { ld_pairs2(in_below + 4 * cvs, a, b); ld_pairs2(in_below + 4 * cvs + 2, c2, d); }
                    while (a.y != stamp_in || b.y != stamp_in || c2.y != stamp_in || d.y != stamp_in);
                    v4 = make_uint4(a.x, b.x, c2.x, d.x);
                    *reinterpret_cast<uint4 *>(sg + 4 * cvs) = v4;      // (row index 0 of sg mirrors the row below the band)
                    s4 = *reinterpret_cast<const uint4 *>(self_s + 4 * cvs);
                    e = self_s[cvs == 0 ? W - 1 : 4 * cvs - 1];
                } else if (s > 0 && gi == nr) {
                    uint2 a, b, c2, d, ee;                              // the row above the band: own words and edge from the band above
                    const uint2 *pe = in_above + (cvs == 0 ? W - 1 : 4 * cvs - 1);
                    do { ld_pairs2(in_above + 4 * cvs, a, b); ld_pairs2(in_above + 4 * cvs + 2, c2, d); ee = ld_pair(pe); }
                    while (a.y != stamp_in || b.y != stamp_in || c2.y != stamp_in || d.y != stamp_in || ee.y != stamp_in);
                    s4 = make_uint4(a.x, b.x, c2.x, d.x);
                    v4 = *reinterpret_cast<const uint4 *>(down_s + 4 * cvs);
                    e = ee.x;
                } else {
                    s4 = *reinterpret_cast<const uint4 *>(self_s + 4 * cvs);
                    v4 = *reinterpret_cast<const uint4 *>(down_s + 4 * cvs);
                    e = self_s[cvs == 0 ? W - 1 : 4 * cvs - 1];
                }
                const uint4 o = apply(0, s4, v4, e, R);
                *reinterpret_cast<uint4 *>(self_t + 4 * cvs) = o;
                if constexpr (SUMS) if (pending != nullptr && gi < nr) {
                    // C_x, C_y of the record taken after the previous step: sigma_x sigma_{x left}, sigma_x sigma_{x down}
                    const uint32_t w[4] = {s4.x, s4.y, s4.z, s4.w}, dw[4] = {v4.x, v4.y, v4.z, v4.w};
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        v[4] = __dp4a((int)w[j], (int)__funnelshift_l(j == 0 ? e : w[j - 1], w[j], 8), v[4]);
                        v[5] = __dp4a((int)w[j], (int)dw[j], v[5]);
                    }
                }
            }
            if (gi >= 1) bar_arrive_n(X1 - 1, 2 * gt_threads);          // tau row gi exists: group gi-1 may start its half-step 1
            if constexpr (SUMS) if (pending) {
                if (gi < nr) deliver(v[4] * 65536 + v[5], 0, 1, 4, pending_slot, pending);
                pending = nullptr;
            }

            // ---- half-step 1: sigma row gi <- tau rows gi, gi+1 (the redundant row's group has none)
            if (gi < nr) {
                device_half_step_keys(p.keys, 2ull * t + 1ull, p.chain0 + (uint32_t)chain, xa2, xb0, ck);
                if (mine) draw(n, R);
                bar_sync_n(X1, 2 * gt_threads);                         // own tau row complete; row gi+1 too
                if (mine) {
                    const uint32_t stamp_out = p.stamp0 + (uint32_t)s + 1u;
                    const uint4 s4 = *reinterpret_cast<const uint4 *>(self_t + 4 * cvs);
                    const uint4 v4 = *reinterpret_cast<const uint4 *>(self_t + W + 4 * cvs);
                    const uint32_t e = self_t[cvs == nvec - 1 ? 0 : 4 * cvs + 4];
                    const uint4 o = apply(1, s4, v4, e, R);
                    *reinterpret_cast<uint4 *>(self_s + 4 * cvs) = o;
                    if (gi == nr - 1) {
                        uint2 *out_top = p.xtop + ((size_t)(s & 1) * nb + band) * W;
                        st_pairs2(out_top + 4 * cvs, o.x, o.y, stamp_out); st_pairs2(out_top + 4 * cvs + 2, o.z, o.w, stamp_out);
                    }
                    if (gi == 0) {
                        uint2 *out_bot = p.xbot + ((size_t)(s & 1) * nb + band) * W;
                        st_pairs2(out_bot + 4 * cvs, o.x, o.y, stamp_out); st_pairs2(out_bot + 4 * cvs + 2, o.z, o.w, stamp_out);
                    }
                    if constexpr (SUMS) if (rec) {
                        // M_sigma, M_tau, E_J = sigma'_x (tau_{x up} + tau_{x right}), E_q = sigma'_x tau_x
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
                if (s + 1 < p.n_steps) bar_arrive_n(X0 + 1, 2 * gt_threads);   // sigma row gi exists: group gi+1 may start the next step
            }
            if constexpr (SUMS) if (rec) {
                long long *dst = p.rec + ((size_t)nrec * p.n_chains + chain) * 6;
                const int slot = (int)(nrec & (FLOW_RING - 1));
                if (gi < nr) deliver(v[0] * 65536 + v[1], v[2] * 65536 + v[3], 2, 0, slot, dst);
                pending = dst;
                pending_slot = slot;
                ++nrec;
            }
        };
#pragma unroll 1
        for (long long s = 0; s < p.n_steps; ++s) {
            const bool rec = p.obs_every > 0 && --until_rec == 0;        // the same in every warp
            if (rec) until_rec = p.obs_every;
            if (rec || pending) step(std::true_type{}, s, rec);
            else step(std::false_type{}, s, false);
        }
    } else {
        // a warp without a row: only the bookkeeping that decides whether the last step was recorded
        for (long long s = 0; s < p.n_steps; ++s) {
            const bool rec = p.obs_every > 0 && --until_rec == 0;
            if (rec) { until_rec = p.obs_every; pending = p.rec + ((size_t)nrec * p.n_chains + chain) * 6; ++nrec; }
            else pending = nullptr;
        }
    }
    __syncthreads();                              // every group is through its last half-step
    if (pending) {
        // the last step was recorded: C_x, C_y of the final sigma; the row below the band comes from the neighbour's last publish
        const uint32_t stamp_in = p.stamp0 + (uint32_t)p.n_steps;
        const uint2 *in_below = p.xtop + ((size_t)((p.n_steps + 1) & 1) * nb + below) * W;
        for (int i = tid; i < W; i += BAND_THREADS) {
            uint2 a;
            do { a = ld_pair(in_below + i); } while (a.y != stamp_in);
            sg[i] = a.x;
        }
        __syncthreads();
        int a0 = 0, a1 = 0;
        for (int c = tid; c < nr * W; c += BAND_THREADS) {
            const int r = (int)__umulhi((uint32_t)c, p.magicW), cw = c - r * W;
            const uint32_t *row = sg + (r + 1) * W;
            const uint32_t s0 = row[cw];
            a0 = __dp4a((int)s0, (int)__funnelshift_l(row[cw == 0 ? W - 1 : cw - 1], s0, 8), a0);   // sigma_x sigma_{x left}
            a1 = __dp4a((int)s0, (int)row[cw - W], a1);                                              // sigma_x sigma_{x down}
        }
        a0 = __reduce_add_sync(0xFFFFFFFFu, a0);
        a1 = __reduce_add_sync(0xFFFFFFFFu, a1);
        if (lane == 0) { s_red[warp][0] = a0; s_red[warp][1] = a1; }
        __syncthreads();
        if (tid < 2) {
            long long tot = 0;
            for (int w = 0; w < BAND_THREADS / 32; ++w) tot += s_red[w][tid];
            atomicAdd(reinterpret_cast<unsigned long long *>(pending + 4 + tid), (unsigned long long)tot);
        }
    }
    for (int i = tid; i < nr * W; i += BAND_THREADS) { gs[(size_t)r0 * W + i] = sg[W + i]; gt[(size_t)r0 * W + i] = ta[i]; }
}

} // namespace shaken
