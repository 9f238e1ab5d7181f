// kernel_small.cuh -- small-lattice path: one CTA owns one whole chain.
//
// For L <= 128 a half-step is a few thousand sites: one launch per half-step would be pure launch latency
// (about 4 us against well under 1 us of work).  Here both sublattices of a chain live in shared memory and ONE
// launch advances n_steps full steps, with a block barrier between half-steps (eq. (15) then eq. (16),
// PAPER.md:162-172) and the six sums of a recorded step reduced inside the block -- no atomics, one CTA per
// chain, grid = n_chains (the shape of the paper's 32x32 coalescence runs, and of (q,J) scans).
// Coupled chains (shaken_set_coupling) share a CTA: every Philox call is made once per GROUP and serves all its members
// ("the same sequence of random numbers"), and the coalescence test is one block-wide vote per step.
// Site -> random word mapping, thresholds and index encoding are those of kernel_i8.cuh; only the schedule differs.
#pragma once
#include "kernels_common.cuh"

namespace shaken {

constexpr int SMALL_L_MAX = 128;        // always the one-CTA-per-chain path
constexpr int SMALL_L_BATCH_MAX = 288;  // ... and up to here for batches that fill the machine (2 L^2 + 16 KiB <= 200 KiB)
constexpr int SMALL_GROUP_MAX = 8;   // coupled chains of one group share a CTA (and every Philox call)

struct SmallParams {
    uint8_t *sigma;          // [n_chains][L][L] int8
    uint8_t *tau;
    int L;
    int n_chains;
    int group;               // coupling group size: one CTA per group, grid = n_chains / group
    uint32_t chain0;
    unsigned long long t0;   // global full-step index of the first step of this launch
    long long n_steps;
    long long obs_every;     // 0 = never
    long long *rec;          // first free record slot, [record][n_chains][6]
    long long *coal;         // [n_chains / group] coalescence times (-1 = not yet) or nullptr (group == 1)
    const uint32_t *gtab;    // per-chain tables [n_chains][8] (natural order) or nullptr: utab
    uint32_t utab[8];
    StepKeys keys;           // only k0[], k1[] are used (functions of the seed)
};

// dynamic shared memory of small_run_i8: G members x (sigma words, tau words), then G paired threshold tables
__host__ __device__ inline size_t small_smem_bytes(int L, int G) { return (size_t)G * ((size_t)2 * L * L + 64 * 32 * sizeof(uint2)); }

// MAXT: the largest block this instance is launched with (256 for L <= 64, 512 above: up to 128 registers for the four
// interleaved Philox calls)
template <int MAXT>
__global__ void __launch_bounds__(MAXT, 1) small_run_i8(const __grid_constant__ SmallParams p)
{
    extern __shared__ __align__(16) uint32_t smem[];
    const int L = p.L;
    const int W = L >> 2;                         // 32-bit words (= Philox calls) per row
    const int ncalls = L * W;                     // per sublattice
    const int nvec = L >> 4, nvecs = L * nvec;    // 16-byte vectors per row / per sublattice
    const int G = p.group;
    uint2 *s_pair = reinterpret_cast<uint2 *>(smem + 2 * G * ncalls);   // [G][64][32], see kernel_i8.cuh EXTRACT_PAIR
    __shared__ int s_red[32][6];

    const int gi = blockIdx.x, chain_first = gi * G;
    const int tid = threadIdx.x;
    const int lane = tid & 31, warp = tid >> 5;
    const int nwarps = blockDim.x >> 5;
    const uint32_t lane8 = (uint32_t)lane * 8u;
    const size_t plane = (size_t)L * L;
    // member m: sigma words at smem + 2 m ncalls, tau words right behind
    for (int m = 0; m < G; ++m) {
        const uint32_t *gs = reinterpret_cast<const uint32_t *>(p.sigma + (size_t)(chain_first + m) * plane);
        const uint32_t *gt = reinterpret_cast<const uint32_t *>(p.tau + (size_t)(chain_first + m) * plane);
        uint32_t *sg = smem + 2 * m * ncalls, *ta = sg + ncalls;
        for (int i = tid; i < ncalls; i += blockDim.x) { sg[i] = gs[i]; ta[i] = gt[i]; }
        for (int t = tid; t < 64 * 32; t += blockDim.x) {
            const int e = t >> 5;
            uint32_t T2[2];
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int c = h ? (e >> 3) : (e & 7);
                const int ms = c & 1, mh = (c >> 1) & 1, mv = c >> 2;
                const int idx = 2 * (2 - mh - mv) + (1 - ms);          // T[2k + c]
                T2[h] = p.gtab ? p.gtab[(size_t)(chain_first + m) * 8 + idx] : p.utab[idx];
            }
            s_pair[(size_t)m * 64 * 32 + t] = make_uint2(T2[0], T2[1]);
        }
    }
    __syncthreads();

    bool coalesced = p.coal ? p.coal[gi] >= 0 : true;   // block-uniform
    long long nrec = 0;
    for (long long s = 0; s < p.n_steps; ++s) {
        const unsigned long long t = p.t0 + (unsigned long long)s;
#pragma unroll 1
        for (int half = 0; half < 2; ++half) {
            uint32_t xa2, xb0;
            ChainKeys ck;
            // one sequence of random numbers for the whole group: the words of its first chain
            device_half_step_keys(p.keys, 2ull * t + (unsigned)half, p.chain0 + (uint32_t)chain_first, xa2, xb0, ck);
            // one 16-byte vector (4 words, 4 interleaved Philox calls) per thread per trip, as in kernel_i8.cuh
#pragma unroll 1
            for (int c = tid; c < nvecs; c += blockDim.x) {
                const int r = c / nvec, cv = c - r * nvec;
                const int at = r * W + 4 * cv;
                uint32_t rw[4][4];
#pragma unroll
                for (int j = 0; j < 4; ++j) philox_site_words((uint32_t)(at + j), p.keys, xa2, xb0, ck, rw[j]);
                const int av = half == 0 ? (r == 0 ? L - 1 : r - 1) * W + 4 * cv : (r == L - 1 ? 0 : r + 1) * W + 4 * cv;
                const int ae = half == 0 ? r * W + (cv == 0 ? W - 1 : 4 * cv - 1) : r * W + (cv == nvec - 1 ? 0 : 4 * cv + 4);
#pragma unroll 1
                for (int m = 0; m < G; ++m) {
                    const uint32_t *src = smem + 2 * m * ncalls + (half ? ncalls : 0);
                    uint32_t *dst = smem + 2 * m * ncalls + (half ? 0 : ncalls);
                    const char *tab = reinterpret_cast<const char *>(s_pair + (size_t)m * 64 * 32);
                    const uint4 s4 = *reinterpret_cast<const uint4 *>(src + at);
                    const uint4 v4 = *reinterpret_cast<const uint4 *>(src + av);
                    const uint32_t e = src[ae];
                    const uint32_t w[4] = {s4.x, s4.y, s4.z, s4.w}, vw[4] = {v4.x, v4.y, v4.z, v4.w};
                    uint32_t o[4];
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        const uint32_t hw = half == 0 ? __funnelshift_l(j == 0 ? e : w[j - 1], w[j], 8)
                                                      : __funnelshift_r(w[j], j == 3 ? e : w[j + 1], 8);
                        const uint32_t y = (hw & 0x40044004u) | (vw[j] & ~0x40044004u);
                        const uint32_t z = ((w[j] & 0x20022002u) | (y & ~0x20022002u)) & 0xE00EE00Eu;
                        const uint32_t o01 = __dp4a(z, 0x00004080u, lane8), o23 = __dp4a(z, 0x40800000u, lane8);
                        const uint2 t01 = *reinterpret_cast<const uint2 *>(tab + o01);
                        const uint2 t23 = *reinterpret_cast<const uint2 *>(tab + o23);
                        uint32_t out = 0x01010101u;
                        out = add_if_not_less(out, rw[j][0], t01.x, 0xFEu);
                        out = add_if_not_less(out, rw[j][1], t01.y, 0xFEu << 8);
                        out = add_if_not_less(out, rw[j][2], t23.x, 0xFEu << 16);
                        out = add_if_not_less(out, rw[j][3], t23.y, 0xFEu << 24);
                        o[j] = out;
                    }
                    *reinterpret_cast<uint4 *>(dst + at) = make_uint4(o[0], o[1], o[2], o[3]);
                }
            }
            __syncthreads();
        }
        if (!coalesced) {
            // coalescence time T = min{n : X_n = Y_n}: sigma of every member against the first one
            int differ = 0;
            for (int c = tid; c < ncalls; c += blockDim.x)
                for (int m = 1; m < G; ++m) differ |= smem[c] != smem[2 * m * ncalls + c];
            if (!__syncthreads_or(differ)) {
                coalesced = true;
                if (tid == 0) p.coal[gi] = (long long)(t + 1);
            }
        }
        if (p.obs_every > 0 && (t + 1) % (unsigned long long)p.obs_every == 0) {
            // six sums on (sigma', tau') of every member -- signed-byte dot products over the words in shared memory
            for (int m = 0; m < G; ++m) {
                const uint32_t *sg = smem + 2 * m * ncalls, *ta = sg + ncalls;
                int v[6] = {0, 0, 0, 0, 0, 0};
                for (int c = tid; c < nvecs; c += blockDim.x) {       // one 16-byte vector of each layer per trip
                    const int r = c / nvec, cv = c - r * nvec;
                    const int at = r * W + 4 * cv;
                    const int up = (r == L - 1 ? 0 : r + 1) * W + 4 * cv;
                    const int rt = r * W + (cv == nvec - 1 ? 0 : 4 * cv + 4);
                    const uint4 s4 = *reinterpret_cast<const uint4 *>(sg + at), t4 = *reinterpret_cast<const uint4 *>(ta + at);
                    const uint4 su4 = *reinterpret_cast<const uint4 *>(sg + up), tu4 = *reinterpret_cast<const uint4 *>(ta + up);
                    const uint32_t sw[5] = {s4.x, s4.y, s4.z, s4.w, sg[rt]}, tw[5] = {t4.x, t4.y, t4.z, t4.w, ta[rt]};
                    const uint32_t su[4] = {su4.x, su4.y, su4.z, su4.w}, tu[4] = {tu4.x, tu4.y, tu4.z, tu4.w};
#pragma unroll
                    for (int j = 0; j < 4; ++j) {
                        const int s0 = (int)sw[j], t0w = (int)tw[j];
                        const int sr = (int)__funnelshift_r(sw[j], sw[j + 1], 8), tr = (int)__funnelshift_r(tw[j], tw[j + 1], 8);
                        v[0] = __dp4a(s0, 0x01010101, v[0]);
                        v[1] = __dp4a(t0w, 0x01010101, v[1]);
                        v[2] = __dp4a(s0, (int)tu[j], v[2]);
                        v[2] = __dp4a(s0, tr, v[2]);
                        v[3] = __dp4a(s0, t0w, v[3]);
                        v[4] = __dp4a(s0, sr, v[4]);
                        v[5] = __dp4a(s0, (int)su[j], v[5]);
                    }
                }
#pragma unroll
                for (int k = 0; k < 6; ++k) {
                    const int w = __reduce_add_sync(0xFFFFFFFFu, v[k]);
                    if (lane == 0) s_red[warp][k] = w;
                }
                __syncthreads();
                if (warp == 0) {                       // second level: one warp sums the per-warp partials (|sum| <= 2 L^2)
#pragma unroll
                    for (int k = 0; k < 6; ++k) {
                        const int tot = __reduce_add_sync(0xFFFFFFFFu, lane < nwarps ? s_red[lane][k] : 0);
                        if (lane == 0) p.rec[((size_t)nrec * p.n_chains + chain_first + m) * 6 + k] = (long long)tot;
                    }
                }
                __syncthreads();
            }
            ++nrec;
        }
    }
    for (int m = 0; m < G; ++m) {
        uint32_t *os = reinterpret_cast<uint32_t *>(p.sigma + (size_t)(chain_first + m) * plane);
        uint32_t *ot = reinterpret_cast<uint32_t *>(p.tau + (size_t)(chain_first + m) * plane);
        const uint32_t *sg = smem + 2 * m * ncalls, *ta = sg + ncalls;
        for (int i = tid; i < ncalls; i += blockDim.x) { os[i] = sg[i]; ot[i] = ta[i]; }
    }
}

} // namespace shaken
