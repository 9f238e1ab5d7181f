// kernel_cluster.cuh -- ONE small chain (L <= 128) spread over a thread-block cluster of 8 SMs.
//
// kernel_small.cuh runs a small chain on one SM: a half-step of a 64 x 64 lattice is 256 vectors = 8 warps, and 2 warps per
// SM sub-partition need 0.47 us for it whatever they do (the ALU port), 2.1 us per recorded step in
// all.  When only a few chains run (cfg 1: one), the other 147 SMs idle.  Here the 8 CTAs of a cluster share the chain: each
// keeps L / 8 rows of both sublattices in its shared memory, one 32-bit word (4 sites, ONE Philox call: the shortest
// dependent chain there is) per thread.  The fields of eq. (14) reach one row across a CTA edge per
// half-step (the down row in half-step 0, the up row in half-step 1).  As in the band kernel, a CTA redraws the tau row ABOVE
// its rows redundantly (a site's random word depends on (seed, chain, step, half, site) alone; the threads that do it would
// idle otherwise), so half-step 1 needs nothing from a neighbour and ONE cluster barrier per full step is enough: half-step 0
// reads the neighbours' sigma rows straight out of their shared memory (distributed shared memory), a block barrier separates
// the half-steps, a cluster barrier the steps.  sigma is double-buffered (a step writes the buffer the previous step did not
// read), so a CTA that is already in half-step 1 never overwrites a row a slower neighbour still reads in its half-step 0.
// A thread draws the random words of BOTH half-steps of the next step between its arrival at the cluster barrier and its
// wait: the two Philox calls (most of a step's latency) hide the barrier's round trip.  The sums of a recorded step are
// fused into the half-steps (operands in registers), reduced per warp and collected per CTA in a shared-memory ring of
// CLUSTER_STAGE records, which is added to the records in global memory (int64 atomics: the 8 CTAs share a record) once it is
// full and at the end: a global atomic inside the step loop would make the next `barrier.cluster.arrive.release` wait for it.
// Site -> random word mapping, thresholds and rule are those of kernel_i8.cuh; only the schedule differs.
#pragma once
#include <cooperative_groups.h>

#include "kernels_common.cuh"
#include "kernel_small.cuh"

namespace shaken {

constexpr int CLUSTER_CTAS = 8;            // portable cluster size; L % 16 == 0 makes L / 8 an integer
constexpr int CLUSTER_STAGE = 64;          // records a CTA collects in shared memory between two flushes to global memory


// dynamic shared memory of cluster_run_i8: two buffers of the CTA's sigma rows, its tau rows and the redundant tau row above them
__host__ __device__ inline size_t cluster_smem_bytes(int L) { return (size_t)(3 * (L / CLUSTER_CTAS) + 1) * (L / 4) * sizeof(uint32_t); }
// threads per CTA: one per word of half-step 0 (the CTA's rows + the redundant row): at most 17 rows x 32 words at L = 128
constexpr int CLUSTER_MAX_THREADS = 544;
__host__ __device__ inline int cluster_threads(int L) { return (((L / CLUSTER_CTAS + 1) * (L / 4) + 31) / 32) * 32; }

__global__ void __launch_bounds__(CLUSTER_MAX_THREADS, 1) cluster_run_i8(const __grid_constant__ SmallParams p)
{
    namespace cg = cooperative_groups;
    cg::cluster_group cluster = cg::this_cluster();
    extern __shared__ __align__(16) uint32_t smem[];
    __shared__ uint2 s_pair[64][32];              // paired thresholds, lane-replicated (see kernel_i8.cuh)
    __shared__ int s_stage[CLUSTER_STAGE][6];     // this CTA's partial sums of the records not yet flushed (ring, by record index)

    const int L = p.L, W = L >> 2, rpb = L / CLUSTER_CTAS;
    const int rank = (int)cluster.block_rank();
    const int chain = blockIdx.x / CLUSTER_CTAS;
    const int r0 = rank * rpb;                    // first row of this CTA
    const int nwords = rpb * W;                   // words of the CTA's rows = words of half-step 1
    const int n0 = nwords + W;                    // words of half-step 0: the rows and the redundant row above them
    const int tid = threadIdx.x, lane = tid & 31;
    const uint32_t lane8 = (uint32_t)lane * 8u;
    // sigma is double-buffered: step s reads the buffer at smem + (s & 1) * nwords and writes the other one
    uint32_t *ta = smem + 2 * nwords;             // tau rows 0 .. rpb (row rpb = the row above the CTA's rows, redrawn redundantly)
    // the sigma buffers of the CTAs that own the rows below (rank - 1) and above (rank + 1) on the torus
    const uint32_t *sm_below = cluster.map_shared_rank(smem, (rank + CLUSTER_CTAS - 1) % CLUSTER_CTAS);
    const uint32_t *sm_above = cluster.map_shared_rank(smem, (rank + 1) % CLUSTER_CTAS);

    const size_t plane = (size_t)L * L;
    uint32_t *gs = reinterpret_cast<uint32_t *>(p.sigma + (size_t)chain * plane) + (size_t)r0 * W;
    uint32_t *gt = reinterpret_cast<uint32_t *>(p.tau + (size_t)chain * plane) + (size_t)r0 * W;
    for (int i = tid; i < nwords; i += blockDim.x) { smem[i] = gs[i]; ta[i] = gt[i]; }
    for (int t = tid; t < 64 * 32; t += blockDim.x) {
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
    for (int i = tid; i < CLUSTER_STAGE * 6; i += blockDim.x) (&s_stage[0][0])[i] = 0;
    cluster.sync();

    long long nrec = 0, flushed = 0, done = 0;    // records begun / added to global memory / complete as of the previous step
    bool pending = false;                         // the last record still lacks C_x, C_y (taken in the next half-step 0)
    // records [flushed, upto) of the ring -> global memory; every thread of the CTA calls it at the same point
    auto flush = [&](const long long upto) {
        const int count = (int)(upto - flushed);
        for (int i = tid; i < count * 6; i += blockDim.x) {
            const long long r = flushed + i / 6;
            const int f = i - (i / 6) * 6;
            int *src = &s_stage[(int)(r % CLUSTER_STAGE)][f];
            const int v = *reinterpret_cast<volatile int *>(src);
            *reinterpret_cast<volatile int *>(src) = 0;
            if (v != 0) atomicAdd(reinterpret_cast<unsigned long long *>(p.rec + ((size_t)r * p.n_chains + chain) * 6 + f), (unsigned long long)(long long)v);
        }
        flushed = upto;
        __syncthreads();                          // the cleared slots are used again right away
    };
    // threshold lookup, compare and pack of one word: sw = own spins, hw = horizontal, vw = vertical neighbours, rw = random words
    auto redraw = [&](const uint32_t sw, const uint32_t hw, const uint32_t vw, const uint32_t (&rw)[4]) -> uint32_t {
        const uint32_t y = (hw & 0x40044004u) | (vw & ~0x40044004u);
        const uint32_t z = ((sw & 0x20022002u) | (y & ~0x20022002u)) & 0xE00EE00Eu;
        const uint32_t o01 = __dp4a(z, 0x00004080u, lane8), o23 = __dp4a(z, 0x40800000u, lane8);
        const uint2 t01 = *reinterpret_cast<const uint2 *>(reinterpret_cast<const char *>(s_pair) + o01);
        const uint2 t23 = *reinterpret_cast<const uint2 *>(reinterpret_cast<const char *>(s_pair) + o23);
        uint32_t out = 0x01010101u;
        out = add_if_not_less(out, rw[0], t01.x, 0xFEu);
        out = add_if_not_less(out, rw[1], t01.y, 0xFEu << 8);
        out = add_if_not_less(out, rw[2], t23.x, 0xFEu << 16);
        out = add_if_not_less(out, rw[3], t23.y, 0xFEu << 24);
        return out;
    };

    // Thread tid owns word tid of half-step 0 (rows 0 .. rpb, the last one redundant) and word tid of half-step 1 (rows
    // 0 .. rpb-1): one Philox call per thread and half-step.
    const bool act0 = tid < n0, act1 = tid < nwords;
    const int wr = (act0 ? tid : 0) / W, wc = (act0 ? tid : 0) - wr * W;    // row and word-in-row
    int gr = r0 + wr;
    if (gr >= L) gr -= L;                         // (the redundant row of the top CTA is row 0)
    const uint32_t wn = (uint32_t)gr * (uint32_t)W + (uint32_t)wc;          // Philox counter = global word index
    uint32_t rw0[4] = {0u, 0u, 0u, 0u}, rw1[4] = {0u, 0u, 0u, 0u};
    // the random words of both half-steps of full step t: they depend on no spin
    auto draw_step = [&](const unsigned long long t) {
        uint32_t xa2, xb0;
        ChainKeys ck;
        device_half_step_keys(p.keys, 2ull * t, p.chain0 + (uint32_t)chain, xa2, xb0, ck);
        if (act0) philox_site_words(wn, p.keys, xa2, xb0, ck, rw0);
        device_half_step_keys(p.keys, 2ull * t + 1ull, p.chain0 + (uint32_t)chain, xa2, xb0, ck);
        if (act1) philox_site_words(wn, p.keys, xa2, xb0, ck, rw1);
    };
    draw_step(p.t0);
    long long until_rec = p.obs_every > 0 ? p.obs_every - (long long)(p.t0 % (unsigned long long)p.obs_every) : 0;
#pragma unroll 1
    for (long long s = 0; s < p.n_steps; ++s) {
        const bool rec = p.obs_every > 0 && --until_rec == 0;       // uniform over the cluster
        if (rec) until_rec = p.obs_every;
        const int off = (int)(s & 1) * nwords;    // the buffer this step reads
        const uint32_t *cur = smem + off, *below = sm_below + off, *above = sm_above + off;
        uint32_t *nxt = smem + (nwords - off);

        // ---- half-step 0: tau rows 0 .. rpb <- sigma, down and left neighbours (eq. (15))
        const bool sums0 = pending;
        int a0 = 0, a1 = 0, a2 = 0, a3 = 0, c0 = 0, c1 = 0;
        if (act0) {
                const int r = wr, cw = wc;
                const uint32_t *row = r < rpb ? cur + r * W : above;                              // (row rpb: the first row of the CTA above)
                const uint32_t sw = row[cw];
                const uint32_t hw = __funnelshift_l(row[cw == 0 ? W - 1 : cw - 1], sw, 8);        // left neighbours
                const uint32_t vw = r == 0 ? below[(rpb - 1) * W + cw] : cur[(r - 1) * W + cw];   // down: row 0 reads the last row of the CTA below
                ta[tid] = redraw(sw, hw, vw, rw0);
                if (sums0 && r < rpb) {
                    c0 = __dp4a((int)sw, (int)hw, 0);               // C_x: sigma_x sigma_{x left}
                    c1 = __dp4a((int)sw, (int)vw, 0);               // C_y: sigma_x sigma_{x down}
                }
            }
        __syncthreads();                          // tau rows 0 .. rpb of this CTA are complete: half-step 1 needs nothing else

        // ---- half-step 1: sigma rows 0 .. rpb-1 <- tau, up and right neighbours (eq. (16)), into the other sigma buffer
        if (act1) {
            const int r = wr, cw = wc;
            const uint32_t sw = ta[tid];
            const uint32_t hw = __funnelshift_r(sw, ta[r * W + (cw == W - 1 ? 0 : cw + 1)], 8);   // right neighbours
            const uint32_t vw = ta[tid + W];                                                      // up (row rpb: the redundant row)
            const uint32_t out = redraw(sw, hw, vw, rw1);
            nxt[tid] = out;
            if (rec) {
                a0 = __dp4a((int)out, 0x01010101, 0);               // M_sigma
                a1 = __dp4a((int)sw, 0x01010101, 0);                // M_tau
                a2 = __dp4a((int)out, (int)vw, 0);                  // sigma'_x tau_{x up}
                a2 = __dp4a((int)out, (int)hw, a2);                 // sigma'_x tau_{x right}
                a3 = __dp4a((int)out, (int)sw, 0);                  // E_q
            }
        }
        asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");   // my rows of the new sigma are written
        // in the shadow of the barrier: the next step's random words, and this step's sums into the ring
        if (s + 1 < p.n_steps) draw_step(p.t0 + (unsigned long long)(s + 1));
        if (sums0) {
            c0 = __reduce_add_sync(0xFFFFFFFFu, c0);
            c1 = __reduce_add_sync(0xFFFFFFFFu, c1);
            if (lane == 0) { int *d = s_stage[(int)((nrec - 1) % CLUSTER_STAGE)]; atomicAdd(d + 4, c0); atomicAdd(d + 5, c1); }
        }
        if (rec) {
            a0 = __reduce_add_sync(0xFFFFFFFFu, a0);
            a1 = __reduce_add_sync(0xFFFFFFFFu, a1);
            a2 = __reduce_add_sync(0xFFFFFFFFu, a2);
            a3 = __reduce_add_sync(0xFFFFFFFFu, a3);
            if (lane == 0) { int *d = s_stage[(int)(nrec % CLUSTER_STAGE)]; atomicAdd(d + 0, a0); atomicAdd(d + 1, a1); atomicAdd(d + 2, a2); atomicAdd(d + 3, a3); }
        }
        asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");     // ... and so are everybody else's
        // The sums above were added AFTER this thread's arrival, so they are ordered for the other threads only by the NEXT
        // barrier: what may be flushed now are the records that were complete one step ago (`done`, from the previous trip).
        if (done - flushed >= CLUSTER_STAGE / 2) flush(done);
        pending = rec;
        if (rec) ++nrec;
        done = pending ? nrec - 1 : nrec;         // complete once this trip's sums have landed; at most three more are in flight
    }
    const int fin_off = (int)(p.n_steps & 1) * nwords;
    const uint32_t *fin = smem + fin_off, *fin_below = sm_below + fin_off;
    if (pending) {
        // the last step was recorded: C_x, C_y of the final sigma (the row below this CTA's rows is in the neighbour's memory)
        int a0 = 0, a1 = 0;
        for (int c = tid; c < nwords; c += blockDim.x) {
            const int r = c / W, cw = c - r * W;
            const uint32_t sw = fin[c];
            a0 = __dp4a((int)sw, (int)__funnelshift_l(fin[r * W + (cw == 0 ? W - 1 : cw - 1)], sw, 8), a0);
            a1 = __dp4a((int)sw, (int)(r == 0 ? fin_below[(rpb - 1) * W + cw] : fin[c - W]), a1);
        }
        a0 = __reduce_add_sync(0xFFFFFFFFu, a0);
        a1 = __reduce_add_sync(0xFFFFFFFFu, a1);
        if (lane == 0) { int *d = s_stage[(int)((nrec - 1) % CLUSTER_STAGE)]; atomicAdd(d + 4, a0); atomicAdd(d + 5, a1); }
    }
    __syncthreads();                              // every warp's last sums have landed
    flush(nrec);
    for (int i = tid; i < nwords; i += blockDim.x) { gs[i] = fin[i]; gt[i] = ta[i]; }
    cluster.sync();                               // nobody leaves while a neighbour may still read its shared memory
}

} // namespace shaken
