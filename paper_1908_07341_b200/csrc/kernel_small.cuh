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

constexpr int SMALL_L_MAX = 128;
constexpr int SMALL_THREADS = 1024;
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

__global__ void __launch_bounds__(SMALL_THREADS, 1) small_run_i8(const __grid_constant__ SmallParams p)
{
    extern __shared__ __align__(16) uint32_t smem[];
    const int L = p.L;
    const int W = L >> 2;                         // 32-bit words (= Philox calls) per row
    const int ncalls = L * W;                     // per sublattice
    const int G = p.group;
    __shared__ uint32_t s_tab[SMALL_GROUP_MAX][64];
    __shared__ int s_red[32][6];

    const int gi = blockIdx.x, chain_first = gi * G;
    const int tid = threadIdx.x;
    const int lane = tid & 31, warp = tid >> 5;
    const int nwarps = blockDim.x >> 5;
    const size_t plane = (size_t)L * L;
    // member m: sigma words at smem + 2 m ncalls, tau words right behind
    for (int m = 0; m < G; ++m) {
        const uint32_t *gs = reinterpret_cast<const uint32_t *>(p.sigma + (size_t)(chain_first + m) * plane);
        const uint32_t *gt = reinterpret_cast<const uint32_t *>(p.tau + (size_t)(chain_first + m) * plane);
        uint32_t *sg = smem + 2 * m * ncalls, *ta = sg + ncalls;
        for (int i = tid; i < ncalls; i += blockDim.x) { sg[i] = gs[i]; ta[i] = gt[i]; }
    }
    if (tid < 8 * G) {
        const int m = tid >> 3, t = tid & 7;
        const int ms = t & 1, mh = (t >> 1) & 1, mv = t >> 2;
        const int idx = 2 * (2 - mh - mv) + (1 - ms);
        s_tab[m][(((uint32_t)ms << 3) | ((uint32_t)mh << 4) | (mv ? 0xE4u : 0u)) >> 2] =
            p.gtab ? p.gtab[(size_t)(chain_first + m) * 8 + idx] : p.utab[idx];
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
            for (int c = tid; c < ncalls; c += blockDim.x) {
                const int r = c / W, cw = c - r * W;
                uint32_t rw[4];
                philox_site_words((uint32_t)c, p.keys, xa2, xb0, ck, rw);
                const int cv = half == 0 ? (r == 0 ? L - 1 : r - 1) * W + cw : (r == L - 1 ? 0 : r + 1) * W + cw;
                const int ce = half == 0 ? r * W + (cw == 0 ? W - 1 : cw - 1) : r * W + (cw == W - 1 ? 0 : cw + 1);
#pragma unroll 1
                for (int m = 0; m < G; ++m) {
                    const uint32_t *src = smem + 2 * m * ncalls + (half ? ncalls : 0);
                    uint32_t *dst = smem + 2 * m * ncalls + (half ? 0 : ncalls);
                    const uint32_t sw = src[c], vw = src[cv], e = src[ce];
                    const uint32_t hw = half == 0 ? __funnelshift_l(e, sw, 8) : __funnelshift_r(sw, e, 8);
                    const uint32_t y = (hw & 0x10101010u) | (vw & ~0x10101010u);
                    const uint32_t z = ((sw & 0x08080808u) | (y & ~0x08080808u)) & 0xFCFCFCFCu;
                    uint32_t out = 0xFFFFFFFFu;
#pragma unroll
                    for (int b = 0; b < 4; ++b) {
                        const uint32_t code = b == 3 ? (z >> 24) : __byte_perm(z, 0u, 0x4440u + b);
                        const uint32_t T = *reinterpret_cast<const uint32_t *>(reinterpret_cast<const char *>(s_tab[m]) + code);
                        out = xor_if_less(out, rw[b], T, 0xFEu << (8 * b));
                    }
                    dst[c] = out;
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
                for (int c = tid; c < ncalls; c += blockDim.x) {
                    const int r = c / W, cw = c - r * W;
                    const int up = (r == L - 1 ? 0 : r + 1) * W + cw;
                    const int rt = r * W + (cw == W - 1 ? 0 : cw + 1);
                    const uint32_t s0 = sg[c], t0w = ta[c];
                    const int sr = (int)__funnelshift_r(s0, sg[rt], 8), tr = (int)__funnelshift_r(t0w, ta[rt], 8);
                    v[0] = __dp4a((int)s0, 0x01010101, v[0]);
                    v[1] = __dp4a((int)t0w, 0x01010101, v[1]);
                    v[2] = __dp4a((int)s0, (int)ta[up], v[2]);
                    v[2] = __dp4a((int)s0, tr, v[2]);
                    v[3] = __dp4a((int)s0, (int)t0w, v[3]);
                    v[4] = __dp4a((int)s0, sr, v[4]);
                    v[5] = __dp4a((int)s0, (int)sg[up], v[5]);
                }
#pragma unroll
                for (int k = 0; k < 6; ++k) {
                    const int w = __reduce_add_sync(0xFFFFFFFFu, v[k]);
                    if (lane == 0) s_red[warp][k] = w;
                }
                __syncthreads();
                if (tid < 6) {
                    long long tot = 0;
                    for (int w = 0; w < nwarps; ++w) tot += s_red[w][tid];
                    p.rec[((size_t)nrec * p.n_chains + chain_first + m) * 6 + tid] = tot;
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
