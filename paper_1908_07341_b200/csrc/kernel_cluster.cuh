// kernel_cluster.cuh -- ONE small chain (L <= 128) spread over a thread-block cluster of 8 SMs.
//
// kernel_small.cuh runs a small chain on one SM: a half-step of a 64 x 64 lattice is 256 vectors = 8 warps, and 2 warps per
// SM sub-partition need 0.47 us for it whatever they do (the ALU port), 2.1 us per recorded step in
// all.  When only a few chains run (cfg 1: one), the other 147 SMs idle.  Here the 8 CTAs of a cluster share the chain: each
// keeps L / 8 rows of both sublattices in its shared memory, one 32-bit word (4 sites, ONE Philox call: the shortest
// dependent chain there is) per thread, and the one row a half-step needs from the neighbouring CTA (eq. (14),
// the down row in half-step 0, the up row in half-step 1) is read straight out of that CTA's shared memory
// (distributed shared memory); a cluster barrier separates the half-steps, and a thread draws the random words of the
// next half-step between its arrival at that barrier and its wait.  The sums of a recorded step are fused into the
// half-steps (operands in registers), reduced per warp and collected per CTA in a shared-memory ring of CLUSTER_STAGE
// records, which is added to the records in global memory (int64 atomics: the 8 CTAs share a record) once it is full and
// at the end: a global atomic inside the step loop would make the next `barrier.cluster.arrive.release` wait for it
// (measured: 1.49 us per recorded step with a flush per step, 1.21 without).
// Site -> random word mapping, thresholds and rule are those of kernel_i8.cuh; only the schedule differs.
#pragma once
#include <cooperative_groups.h>

#include "kernels_common.cuh"
#include "kernel_small.cuh"

namespace shaken {

constexpr int CLUSTER_CTAS = 8;            // portable cluster size; L % 16 == 0 makes L / 8 an integer
constexpr int CLUSTER_STAGE = 64;          // records a CTA collects in shared memory between two flushes to global memory

// dynamic shared memory of cluster_run_i8: the CTA's rows of sigma and of tau
__host__ __device__ inline size_t cluster_smem_bytes(int L) { return (size_t)2 * (L / CLUSTER_CTAS) * (L / 4) * sizeof(uint32_t); }

__global__ void __launch_bounds__(512, 1) cluster_run_i8(const __grid_constant__ SmallParams p)
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
    const int nwords = rpb * W;
    const int tid = threadIdx.x, lane = tid & 31;
    const uint32_t lane8 = (uint32_t)lane * 8u;
    uint32_t *sg = smem, *ta = smem + nwords;
    // the same arrays in the CTA that owns the rows below (rank - 1) and above (rank + 1) on the torus
    const uint32_t *sg_below = cluster.map_shared_rank(sg, (rank + CLUSTER_CTAS - 1) % CLUSTER_CTAS);
    const uint32_t *ta_above = cluster.map_shared_rank(ta, (rank + 1) % CLUSTER_CTAS);

    const size_t plane = (size_t)L * L;
    uint32_t *gs = reinterpret_cast<uint32_t *>(p.sigma + (size_t)chain * plane) + (size_t)r0 * W;
    uint32_t *gt = reinterpret_cast<uint32_t *>(p.tau + (size_t)chain * plane) + (size_t)r0 * W;
    for (int i = tid; i < nwords; i += blockDim.x) { sg[i] = gs[i]; ta[i] = gt[i]; }
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

    long long nrec = 0, flushed = 0;              // records begun / added to global memory so far
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
    long long until_rec = p.obs_every > 0 ? p.obs_every - (long long)(p.t0 % (unsigned long long)p.obs_every) : 0;
    // A CTA has at most L^2 / 32 <= 512 words: one word per thread, no loop.  The random words of a half-step depend on no
    // spin, so a thread draws them BETWEEN its arrival at the cluster barrier and its wait: the Philox call (most of a
    // half-step's latency) hides the barrier's round trip.
    const bool active = tid < nwords;
    const int r = tid / W, cw = tid - r * W;
    const uint32_t n = (uint32_t)(r0 + r) * (uint32_t)W + (uint32_t)cw;
    uint32_t rw[4] = {0u, 0u, 0u, 0u};
    {
        uint32_t xa2, xb0;
        ChainKeys ck;
        device_half_step_keys(p.keys, 2ull * p.t0, p.chain0 + (uint32_t)chain, xa2, xb0, ck);
        if (active) philox_site_words(n, p.keys, xa2, xb0, ck, rw);
    }
    bool rec = false;
#pragma unroll 1
    for (long long h = 0; h < 2 * p.n_steps; ++h) {
        const int half = (int)(h & 1);
        if (half == 0) {
            rec = p.obs_every > 0 && --until_rec == 0;               // uniform over the cluster
            if (rec) until_rec = p.obs_every;
        }
        const uint32_t *src = half ? ta : sg;
        uint32_t *dst = half ? sg : ta;
        const bool sums1 = half == 1 && rec, sums0 = half == 0 && pending;
        int a0 = 0, a1 = 0, a2 = 0, a3 = 0;
        if (active) {
            const uint32_t sw = src[tid];
            uint32_t hw, vw;
            if (half == 0) {
                hw = __funnelshift_l(src[r * W + (cw == 0 ? W - 1 : cw - 1)], sw, 8);                 // left neighbours
                vw = r == 0 ? sg_below[(rpb - 1) * W + cw] : src[tid - W];                           // down: last row of the CTA below
            } else {
                hw = __funnelshift_r(sw, src[r * W + (cw == W - 1 ? 0 : cw + 1)], 8);                 // right neighbours
                vw = r == rpb - 1 ? ta_above[cw] : src[tid + W];                                     // up: first row of the CTA above
            }
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
            dst[tid] = out;
            if (sums1) {
                a0 = __dp4a((int)out, 0x01010101, 0);               // M_sigma
                a1 = __dp4a((int)sw, 0x01010101, 0);                // M_tau
                a2 = __dp4a((int)out, (int)vw, 0);                  // sigma'_x tau_{x up}
                a2 = __dp4a((int)out, (int)hw, a2);                 // sigma'_x tau_{x right}
                a3 = __dp4a((int)out, (int)sw, 0);                  // E_q
            }
            if (sums0) {
                a0 = __dp4a((int)sw, (int)hw, 0);                   // C_x: sigma_x sigma_{x left}
                a1 = __dp4a((int)sw, (int)vw, 0);                   // C_y: sigma_x sigma_{x down}
            }
        }
        if (sums1 || sums0) {
            a0 = __reduce_add_sync(0xFFFFFFFFu, a0);
            a1 = __reduce_add_sync(0xFFFFFFFFu, a1);
            a2 = __reduce_add_sync(0xFFFFFFFFu, a2);
            a3 = __reduce_add_sync(0xFFFFFFFFu, a3);
            if (lane == 0) {
                if (sums1) { int *d = s_stage[(int)(nrec % CLUSTER_STAGE)]; atomicAdd(d + 0, a0); atomicAdd(d + 1, a1); atomicAdd(d + 2, a2); atomicAdd(d + 3, a3); }
                else { int *d = s_stage[(int)((nrec - 1) % CLUSTER_STAGE)]; atomicAdd(d + 4, a0); atomicAdd(d + 5, a1); }
            }
        }
        asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");   // my part of the new sublattice is written
        if (h + 1 < 2 * p.n_steps) {
            uint32_t xa2, xb0;
            ChainKeys ck;
            device_half_step_keys(p.keys, 2ull * p.t0 + (unsigned long long)(h + 1), p.chain0 + (uint32_t)chain, xa2, xb0, ck);
            if (active) philox_site_words(n, p.keys, xa2, xb0, ck, rw);
        }
        asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");     // ... and so is everybody else's
        if (sums0) {
            pending = false;
            if (nrec - flushed == CLUSTER_STAGE) flush(nrec);        // the ring is full of complete records
        }
        if (sums1) {
            pending = true;
            ++nrec;
        }
    }
    if (pending) {
        // the last step was recorded: C_x, C_y of the final sigma (the row below this CTA's rows is still in the neighbour's memory)
        int a0 = 0, a1 = 0;
        for (int c = tid; c < nwords; c += blockDim.x) {
            const int r = c / W, cw = c - r * W;
            const uint32_t sw = sg[c];
            a0 = __dp4a((int)sw, (int)__funnelshift_l(sg[r * W + (cw == 0 ? W - 1 : cw - 1)], sw, 8), a0);
            a1 = __dp4a((int)sw, (int)(r == 0 ? sg_below[(rpb - 1) * W + cw] : sg[c - W]), a1);
        }
        a0 = __reduce_add_sync(0xFFFFFFFFu, a0);
        a1 = __reduce_add_sync(0xFFFFFFFFu, a1);
        if (lane == 0) { int *d = s_stage[(int)((nrec - 1) % CLUSTER_STAGE)]; atomicAdd(d + 4, a0); atomicAdd(d + 5, a1); }
        __syncthreads();
    }
    flush(nrec);
    for (int i = tid; i < nwords; i += blockDim.x) { gs[i] = sg[i]; gt[i] = ta[i]; }
    cluster.sync();                               // nobody leaves while a neighbour may still read its shared memory
}

} // namespace shaken
