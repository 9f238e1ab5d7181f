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
#include <type_traits>

#include "kernels_common.cuh"
#include "kernel_small.cuh"
#include "kernel_band.cuh"

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

// One int8 vector (16 sites, the 8 of parity PC redrawn).  c = {word left of the vector, its four words, word right of
// it}; fu, fd = minus-flags of the rows above and below.  A minus-flag word has 4 in every byte whose spin is -1
// (0xFF & 0x04) and 0 where it is +1, so the four flag words of a site's neighbours add up, without carries, to
// 4 * (number of -1 neighbours): the byte offset of its threshold in `tab` (which is stored in that order).
// Sums: a1 += sum of redrawn spins, ah += sum of redrawn spin * 4 * (minus among left, right), av likewise for up, down.
__device__ __forceinline__ uint32_t minus4(uint32_t x) { return x & 0x04040404u; }

// The 5-entry table of a warp sits at a 256-byte aligned shared-memory address, so the address of an entry is the table
// address with its low byte replaced by the offset byte: one PRMT picks the byte out of the flag sum AND forms the address.
constexpr int ALT_TAB_WORDS = 64;
__device__ __forceinline__ uint32_t shared_addr(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ uint32_t lds_u32(uint32_t saddr)
{
    uint32_t v;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(saddr));
    return v;
}

template <int PC, bool OBS>
__device__ __forceinline__ uint4 alt_vector_i8(const uint32_t (&c)[6], const uint32_t (&fu)[4], const uint32_t (&fd)[4],
                                               const uint32_t (&rnd)[8], const uint32_t tab, int &accM, int &a1, int &ah, int &av)
{
    constexpr uint32_t active = 0x00FF00FFu << (8 * PC);
    uint32_t fc[6], out[4];
#pragma unroll
    for (int j = 0; j < 6; ++j) fc[j] = minus4(c[j]);
#pragma unroll
    for (int j = 0; j < 4; ++j) {
        const uint32_t fl = __funnelshift_l(fc[j], fc[j + 1], 8);         // byte b: flag of the spin left of column b
        const uint32_t fr = __funnelshift_r(fc[j + 1], fc[j + 2], 8);     // byte b: flag of the spin right of column b
        const uint32_t hs = fl + fr, vs = fu[j] + fd[j], nm = hs + vs;
        uint32_t o = c[j + 1] | active;                                   // redrawn bytes start as -1 (0xFF)
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            constexpr uint32_t FE = 0xFEu;
            const int b = PC + 2 * i;
            const uint32_t T = lds_u32(__byte_perm(nm, tab, 0x7650u | (uint32_t)b));
            o = xor_if_less(o, rnd[2 * j + i], T, FE << (8 * b));         // 0xFF ^ 0xFE = +1
        }
        out[j] = o;
        if constexpr (OBS) {
            const uint32_t oa = o & active;
            accM = __dp4a((int)o, 0x01010101, accM);
            a1 = __dp4a((int)oa, 0x01010101, a1);
            ah = __dp4a((int)oa, (int)hs, ah);
            av = __dp4a((int)oa, (int)vs, av);
        }
    }
    return make_uint4(out[0], out[1], out[2], out[3]);
}

// Packed word: the 16 redrawn bits (parity PC) from the bit-sliced neighbour count k = s0 + 2 s1 + 4 s2.  Site j of the
// word's redrawn sites sits at bit 2j + PC and draws rnd[j].  For q = j & 3 the four sites j = 4m + q lie in byte m at
// bit 2q + PC, so one word W_q collects, per byte, 4 s0 + 8 s1 + 16 s2 = the byte offset of A[k] in `tab`: six
// shift-and-mask operations serve four sites, then one PRMT, one LDS and one predicated add per site.
template <int FROM, int TO>
__device__ __forceinline__ uint32_t shift_bit(uint32_t x)
{
    if constexpr (FROM >= TO) return x >> (FROM - TO);
    else return x << (TO - FROM);
}

template <int PC>
__device__ __forceinline__ uint32_t alt_offsets_pk(uint32_t s0, uint32_t s1, uint32_t s2, int q)
{
    // bit (2q + PC) of every byte of s0, s1, s2 moved to bits 2, 3, 4 of that byte
    switch (q) {
        case 0: return (shift_bit<0 + PC, 2>(s0) & 0x04040404u) | (shift_bit<0 + PC, 3>(s1) & 0x08080808u) | (shift_bit<0 + PC, 4>(s2) & 0x10101010u);
        case 1: return (shift_bit<2 + PC, 2>(s0) & 0x04040404u) | (shift_bit<2 + PC, 3>(s1) & 0x08080808u) | (shift_bit<2 + PC, 4>(s2) & 0x10101010u);
        case 2: return (shift_bit<4 + PC, 2>(s0) & 0x04040404u) | (shift_bit<4 + PC, 3>(s1) & 0x08080808u) | (shift_bit<4 + PC, 4>(s2) & 0x10101010u);
        default: return (shift_bit<6 + PC, 2>(s0) & 0x04040404u) | (shift_bit<6 + PC, 3>(s1) & 0x08080808u) | (shift_bit<6 + PC, 4>(s2) & 0x10101010u);
    }
}

template <int PC>
__device__ __forceinline__ uint32_t alt_bits_pk(uint32_t s0, uint32_t s1, uint32_t s2, const uint32_t (&rnd)[16], const uint32_t tab)
{
    uint32_t nb = 0;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const uint32_t W = alt_offsets_pk<PC>(s0, s1, s2, q);
#pragma unroll
        for (int m = 0; m < 4; ++m) {
            const uint32_t T = lds_u32(__byte_perm(W, tab, 0x7650u | (uint32_t)m));
            nb = add_if_less(nb, rnd[4 * m + q], T, 1u << (8 * m + 2 * q + PC));
        }
    }
    return nb;
}

// generic form: lanes stride over the (row, vector) pairs of a block of rows -- any L, also rows much narrower than a warp
template <int HALF, bool OBS, bool PACKED>
__global__ void __launch_bounds__(ALT_THREADS) alt_half(const __grid_constant__ AltParams p)
{
    __shared__ __align__(256) uint32_t s_tab[ALT_THREADS / 32][ALT_TAB_WORDS];
    let_next_kernel_launch();                                      // programmatic dependent launch (kernels_common.cuh)
    wait_for_previous_kernel();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int L = p.L, nvec = p.nvec;
    const int wpr = PACKED ? nvec : 4 * nvec;                      // 32-bit words per row
    const uint32_t magic = (uint32_t)(4294967296ull / (uint32_t)nvec) + 1u;   // it / nvec = umulhi(it, magic) for it * nvec < 2^32
    uint32_t *tab = s_tab[warp];

    for (long long task = (long long)blockIdx.x * (ALT_THREADS / 32) + warp; task < p.ntasks;
         task += (long long)gridDim.x * (ALT_THREADS / 32)) {
        const int chain = (int)(task / p.nrb), rb = (int)(task - (long long)chain * p.nrb);
        const int r_begin = rb * p.rows_per_task, r_end = min(L, r_begin + p.rows_per_task);
        __syncwarp();
        // int8: entry i = A[4 - i], addressed by 4 * (number of -1 neighbours); packed: entry k = A[k]
        if (lane < 5) tab[lane] = p.gtab ? p.gtab[(size_t)chain * 8 + (PACKED ? lane : 4 - lane)] : p.utab[PACKED ? lane : 4 - lane];
        __syncwarp();
        const ChainKeys ck = make_chain_keys(p.keys, p.chain0 + (uint32_t)((chain / p.group) * p.group));
        uint32_t *base = reinterpret_cast<uint32_t *>(p.sigma) + (size_t)chain * L * wpr;
        int accM = 0, accX = 0, accY = 0, a1 = 0;
        const int items = (r_end - r_begin) * nvec;
        for (int it = lane; it < items; it += 32) {
            const int dr = nvec == 1 ? it : (int)__umulhi((uint32_t)it, magic);
            const int r = r_begin + dr, v = it - dr * nvec;
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
                const uint32_t fu[4] = {minus4(u4.x), minus4(u4.y), minus4(u4.z), minus4(u4.w)};
                const uint32_t fd[4] = {minus4(d4.x), minus4(d4.y), minus4(d4.z), minus4(d4.w)};
                uint32_t rnd[8];
                const uint32_t n0 = (uint32_t)r * (uint32_t)(L >> 3) + 2u * (uint32_t)v;
                philox_site_words(n0, p.keys, ck, rnd);
                philox_site_words(n0 + 1u, p.keys, ck, rnd + 4);
                uint4 o;
                if (pc) o = alt_vector_i8<1, OBS>(c, fu, fd, rnd, shared_addr(tab), accM, a1, accX, accY);
                else o = alt_vector_i8<0, OBS>(c, fu, fd, rnd, shared_addr(tab), accM, a1, accX, accY);
                *reinterpret_cast<uint4 *>(row + 4 * v) = o;
            } else {
                const uint32_t c = row[v], a = up[v], b = dn[v];
                const uint32_t prev = row[v == 0 ? nvec - 1 : v - 1], next = row[v + 1 == nvec ? 0 : v + 1];
                const uint32_t lw = __funnelshift_l(prev, c, 1);                // bit i = spin left of column i
                const uint32_t rw = __funnelshift_r(c, next, 1);                // bit i = spin right of column i
                // bit-sliced count of +1 among (a, b, lw, rw): k = s0 + 2 s1 + 4 s2
                const uint32_t ab = a & b, axb = a ^ b, lr = lw & rw, lxr = lw ^ rw;
                const uint32_t s0 = axb ^ lxr, s1 = (ab ^ lr) ^ (axb & lxr), s2 = ab & lr;
                const uint32_t n0 = (uint32_t)r * (uint32_t)(L >> 3) + 4u * (uint32_t)v;
                uint32_t rr[4][4];
                {
                    const uint32_t nn[4] = {n0, n0 + 1u, n0 + 2u, n0 + 3u};
                    philox_site_words_xn<4>(nn, p.keys, p.keys.xa2, p.keys.xb0, ck, rr);
                }
                const uint32_t rnd[16] = {rr[0][0], rr[0][1], rr[0][2], rr[0][3], rr[1][0], rr[1][1], rr[1][2], rr[1][3],
                                          rr[2][0], rr[2][1], rr[2][2], rr[2][3], rr[3][0], rr[3][1], rr[3][2], rr[3][3]};
                const uint32_t nb = pc ? alt_bits_pk<1>(s0, s1, s2, rnd, shared_addr(tab)) : alt_bits_pk<0>(s0, s1, s2, rnd, shared_addr(tab));
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
            if constexpr (!PACKED) {
                // s * (l + r) = s * (2 - 2 * minus) per site: ah, av hold 4 * minus, so they are multiples of 4
                accX = 2 * a1 - accX / 2;
                accY = 2 * a1 - accY / 2;
            }
            long long *rec = p.rec + (size_t)chain * 6;
            warp_add_to(rec + 0, accM);
            warp_add_to(rec + 4, accX);
            warp_add_to(rec + 5, accY);
        }
    }
}

// Strip form for wide int8 rows (nvec >= 32): a warp owns a strip 32 vectors wide and rows_per_task (even) rows high and
// walks it row by row; every row is loaded once, the minus-flags of the rows above and below stay in registers (the flags
// of a row's PASSIVE bytes do not change when the row is redrawn, and only those are read by its neighbours), and the
// column parity of the redrawn sites is a compile-time constant of each of the two unrolled row bodies.
// p.ntasks = n_chains * nrb * nseg with nseg = ceil(nvec / 32); rows_per_task and the first row of every task are even.
struct AltRow {
    uint4 c;
    uint32_t prev, next;
};

// row = pointer to the lane's own vector of that row; off_prev / off_next = word offsets (relative to it) of the words
// that hold the spins left and right of the vector (torus wrap included)
__device__ __forceinline__ AltRow alt_load_row(const uint32_t *row, int off_prev, int off_next)
{
    AltRow x;
    x.c = *reinterpret_cast<const uint4 *>(row);
    x.prev = row[off_prev];
    x.next = row[off_next];
    return x;
}

__device__ __forceinline__ void minus4(const uint4 &x, uint32_t (&f)[4])
{
    f[0] = minus4(x.x); f[1] = minus4(x.y); f[2] = minus4(x.z); f[3] = minus4(x.w);
}

template <int HALF, bool OBS>
__global__ void __launch_bounds__(ALT_THREADS, 2) alt_strip_i8(const __grid_constant__ AltParams p)
{
    __shared__ __align__(256) uint32_t s_tab[ALT_THREADS / 32][ALT_TAB_WORDS];
    let_next_kernel_launch();                                      // programmatic dependent launch (kernels_common.cuh)
    wait_for_previous_kernel();
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const int L = p.L, nvec = p.nvec, wpr = 4 * nvec;
    const int nseg = (nvec + 31) >> 5;
    uint32_t *tab_ptr = s_tab[warp];
    const uint32_t tab = shared_addr(tab_ptr);

    for (long long task = (long long)blockIdx.x * (ALT_THREADS / 32) + warp; task < p.ntasks;
         task += (long long)gridDim.x * (ALT_THREADS / 32)) {
        const int per_chain = p.nrb * nseg;
        const int chain = (int)(task / per_chain), rest = (int)(task - (long long)chain * per_chain);
        const int rb = rest / nseg, seg = rest - rb * nseg;
        const int r_begin = rb * p.rows_per_task, r_end = min(L, r_begin + p.rows_per_task);
        __syncwarp();
        if (lane < 5) tab_ptr[lane] = p.gtab ? p.gtab[(size_t)chain * 8 + 4 - lane] : p.utab[4 - lane];
        __syncwarp();
        const ChainKeys ck = make_chain_keys(p.keys, p.chain0 + (uint32_t)((chain / p.group) * p.group));
        const bool live = seg * 32 + lane < nvec;
        const int v = live ? seg * 32 + lane : nvec - 1;          // idle lanes of a ragged last strip repeat the last vector
        uint32_t *col = reinterpret_cast<uint32_t *>(p.sigma) + (size_t)chain * L * wpr + 4 * v;   // the lane's vector of row 0
        const int off_prev = v == 0 ? wpr - 1 : -1, off_next = v + 1 == nvec ? 4 - wpr : 4;
        int accM = 0, a1 = 0, ah = 0, av = 0;

        // Two schedules of the same walk, chosen by measurement (profiles/r1c_ncu_alt_cfg4.md): the launch with the sums
        // is 12 % faster when the vectors are fetched two trips ahead (its memory stalls go from 2.7 to 0.3 per issued
        // instruction); the plain launch is limited by issue slots, and the same change costs it 6 % in extra instructions.
        if constexpr (OBS) {
            // rows held: r0 = row r, r1 = row r + 1, r2 = row r + 2 (the "up" of row r + 1, and the next trip's row r);
            // n3, n4 = the vectors of rows r + 3, r + 4, fetched a trip ago; fd = minus-flags of row r - 1.
            // Every trip fetches the vectors of rows r + 5, r + 6 (two trips ahead: DRAM latency) and the edge words of rows
            // r + 3, r + 4 (one trip ahead: their lines are in L1 or L2 by now).  Nothing is fetched past the halo row r_end.
            // Only the halo row can be row L (= row 0): rows at odd distance from r are odd and L is even.
            uint32_t fd[4];
            minus4(*reinterpret_cast<const uint4 *>(col + (size_t)(r_begin == 0 ? L - 1 : r_begin - 1) * wpr), fd);
            uint32_t *row = col + (size_t)r_begin * wpr;             // row r
            AltRow r0 = alt_load_row(row, off_prev, off_next);
            AltRow r1 = alt_load_row(row + wpr, off_prev, off_next); // L even and r_begin even: rows r + 1 exists
            AltRow r2 = alt_load_row(r_begin + 2 == L ? col : row + 2 * wpr, off_prev, off_next);
            uint4 n3 = make_uint4(0, 0, 0, 0), n4 = n3;
            if (r_begin + 2 < r_end) {
                n3 = *reinterpret_cast<const uint4 *>(row + 3 * wpr);
                n4 = *reinterpret_cast<const uint4 *>(r_begin + 4 == L ? col : row + 4 * wpr);
            }
            uint32_t n0 = (uint32_t)r_begin * (uint32_t)(L >> 3) + 2u * (uint32_t)v;
            const uint32_t dn = (uint32_t)(L >> 3);

            for (int r = r_begin; r < r_end; r += 2) {
                const bool more = r + 2 < r_end, more2 = r + 4 < r_end;
                uint4 m5 = make_uint4(0, 0, 0, 0), m6 = m5;
                uint32_t e3p = 0, e3n = 0, e4p = 0, e4n = 0;
                if (more2) {
                    m5 = *reinterpret_cast<const uint4 *>(row + 5 * wpr);
                    m6 = *reinterpret_cast<const uint4 *>(r + 6 == L ? col : row + 6 * wpr);
                }
                if (more) {
                    const uint32_t *p3 = row + 3 * wpr, *p4 = r + 4 == L ? col : row + 4 * wpr;
                    e3p = p3[off_prev]; e3n = p3[off_next];
                    e4p = p4[off_prev]; e4n = p4[off_next];
                }
                uint32_t rr[4][4];
                {
                    const uint32_t nn[4] = {n0, n0 + 1u, n0 + dn, n0 + dn + 1u};
                    philox_site_words_xn<4>(nn, p.keys, p.keys.xa2, p.keys.xb0, ck, rr);
                }
                const uint32_t rnd0[8] = {rr[0][0], rr[0][1], rr[0][2], rr[0][3], rr[1][0], rr[1][1], rr[1][2], rr[1][3]};
                const uint32_t rnd1[8] = {rr[2][0], rr[2][1], rr[2][2], rr[2][3], rr[3][0], rr[3][1], rr[3][2], rr[3][3]};
                n0 += 2u * dn;
                int m = 0, b1 = 0, bh = 0, bv = 0;
                uint32_t f1[4], f2[4], f0[4];
                minus4(r1.c, f1);
                minus4(r2.c, f2);
                minus4(r0.c, f0);
                const uint32_t c0[6] = {r0.prev, r0.c.x, r0.c.y, r0.c.z, r0.c.w, r0.next};
                const uint32_t c1[6] = {r1.prev, r1.c.x, r1.c.y, r1.c.z, r1.c.w, r1.next};
                // even row r: redrawn columns have parity HALF; odd row r + 1: parity 1 - HALF
                const uint4 o0 = alt_vector_i8<HALF, OBS>(c0, f1, fd, rnd0, tab, m, b1, bh, bv);
                const uint4 o1 = alt_vector_i8<1 - HALF, OBS>(c1, f2, f0, rnd1, tab, m, b1, bh, bv);
                if (live) {
                    *reinterpret_cast<uint4 *>(row) = o0;
                    *reinterpret_cast<uint4 *>(row + wpr) = o1;
                    if constexpr (OBS) { accM += m; a1 += b1; ah += bh; av += bv; }
                }
                row += 2 * wpr;
    #pragma unroll
                for (int j = 0; j < 4; ++j) fd[j] = f1[j];           // flags of the OLD row r + 1: its passive bytes are what row r + 2 reads
                if (more) {
                    r0 = r2;
                    r1.c = n3; r1.prev = e3p; r1.next = e3n;
                    r2.c = n4; r2.prev = e4p; r2.next = e4n;
                    n3 = m5;
                    n4 = m6;
                }
            }
        } else {
            // rows held: r0 = row r, r1 = row r + 1, r2 = row r + 2 (the "up" of row r + 1, and the next iteration's row r);
            // fd = minus-flags of row r - 1
            uint32_t fd[4];
            minus4(*reinterpret_cast<const uint4 *>(col + (size_t)(r_begin == 0 ? L - 1 : r_begin - 1) * wpr), fd);
            uint32_t *row = col + (size_t)r_begin * wpr;             // row r
            AltRow r0 = alt_load_row(row, off_prev, off_next);
            AltRow r1 = alt_load_row(row + wpr, off_prev, off_next); // L even and r_begin even: rows r + 1 exists
            const uint32_t *pa = r_begin + 2 >= L ? col : row + 2 * wpr;   // row r + 2 (mod L)
            AltRow r2 = alt_load_row(pa, off_prev, off_next);
            uint32_t n0 = (uint32_t)r_begin * (uint32_t)(L >> 3) + 2u * (uint32_t)v;
            const uint32_t dn = (uint32_t)(L >> 3);

            for (int r = r_begin; r < r_end; r += 2) {
                // fetch rows r + 3 and r + 4 before computing rows r and r + 1 (not past the strip's upper halo row r_end)
                AltRow a3, a4;
                const bool more = r + 2 < r_end;
                if (more) {
                    a3 = alt_load_row(pa + wpr, off_prev, off_next);               // r + 3 <= r_end - 1 < L: no wrap
                    const uint32_t *p4 = r + 4 >= L ? col : pa + 2 * wpr;
                    a4 = alt_load_row(p4, off_prev, off_next);
                    pa = p4;
                }
                uint32_t rr[4][4];
                {
                    const uint32_t nn[4] = {n0, n0 + 1u, n0 + dn, n0 + dn + 1u};
                    philox_site_words_xn<4>(nn, p.keys, p.keys.xa2, p.keys.xb0, ck, rr);
                }
                const uint32_t rnd0[8] = {rr[0][0], rr[0][1], rr[0][2], rr[0][3], rr[1][0], rr[1][1], rr[1][2], rr[1][3]};
                const uint32_t rnd1[8] = {rr[2][0], rr[2][1], rr[2][2], rr[2][3], rr[3][0], rr[3][1], rr[3][2], rr[3][3]};
                n0 += 2u * dn;
                int m = 0, b1 = 0, bh = 0, bv = 0;
                uint32_t f1[4], f2[4], f0[4];
                minus4(r1.c, f1);
                minus4(r2.c, f2);
                minus4(r0.c, f0);
                const uint32_t c0[6] = {r0.prev, r0.c.x, r0.c.y, r0.c.z, r0.c.w, r0.next};
                const uint32_t c1[6] = {r1.prev, r1.c.x, r1.c.y, r1.c.z, r1.c.w, r1.next};
                // even row r: redrawn columns have parity HALF; odd row r + 1: parity 1 - HALF
                const uint4 o0 = alt_vector_i8<HALF, OBS>(c0, f1, fd, rnd0, tab, m, b1, bh, bv);
                const uint4 o1 = alt_vector_i8<1 - HALF, OBS>(c1, f2, f0, rnd1, tab, m, b1, bh, bv);
                if (live) {
                    *reinterpret_cast<uint4 *>(row) = o0;
                    *reinterpret_cast<uint4 *>(row + wpr) = o1;
                    if constexpr (OBS) { accM += m; a1 += b1; ah += bh; av += bv; }
                }
                row += 2 * wpr;
    #pragma unroll
                for (int j = 0; j < 4; ++j) fd[j] = f1[j];           // flags of the OLD row r + 1: its passive bytes are what row r + 2 reads
                if (more) {
                    r0 = r2;
                    r1 = a3;
                    r2 = a4;
                }
            }
        }
        if constexpr (OBS) {
            long long *rec = p.rec + (size_t)chain * 6;
            warp_add_to(rec + 0, accM);
            warp_add_to(rec + 4, 2 * a1 - ah / 2);
            warp_add_to(rec + 5, 2 * a1 - av / 2);
        }
    }
}

// Small lattices (L <= 128): one CTA per coupling group keeps the sigma arrays of its members in shared memory and ONE
// launch advances n_steps full steps (block barrier between half-steps), as kernel_small.cuh does for the shaken
// dynamics -- a launch per half-step would be pure launch latency here.  Every Philox call is made once per group and
// serves all its members; the coalescence test is one block-wide vote per step; the sums of a recorded
// step go through shared-memory atomics.  p.tau is not used.
__host__ __device__ inline size_t alt_small_smem_bytes(int L, int G) { return (size_t)G * L * L; }

__global__ void __launch_bounds__(256) alt_small_i8(const __grid_constant__ SmallParams p)
{
    extern __shared__ __align__(16) uint32_t smem[];
    __shared__ __align__(256) uint32_t s_tab[SMALL_GROUP_MAX][ALT_TAB_WORDS];
    __shared__ int s_acc[SMALL_GROUP_MAX][4];
    const int L = p.L, W = L >> 2, nvec = L >> 4, nvecs = L * nvec, G = p.group;
    const int words = L * W;
    const int gi = blockIdx.x, chain_first = gi * G, tid = threadIdx.x;
    for (int m = 0; m < G; ++m) {
        const uint32_t *gs = reinterpret_cast<const uint32_t *>(p.sigma + (size_t)(chain_first + m) * L * L);
        for (int i = tid; i < words; i += blockDim.x) smem[m * words + i] = gs[i];
    }
    if (tid < G * 8) {
        const int m = tid >> 3, i = tid & 7;
        // entry i = A[4 - i]: addressed by 4 * (number of -1 neighbours), see alt_vector_i8
        s_tab[m][i] = i < 5 ? (p.gtab ? p.gtab[(size_t)(chain_first + m) * 8 + 4 - i] : p.utab[4 - i]) : 0u;
        if (i < 4) s_acc[m][i] = 0;
    }
    __syncthreads();

    bool coalesced = p.coal ? p.coal[gi] >= 0 : true;   // block-uniform
    long long nrec = 0;
    // full steps until the next recorded one: a countdown instead of a 64-bit modulo per step
    long long until_rec = p.obs_every > 0 ? p.obs_every - (long long)(p.t0 % (unsigned long long)p.obs_every) : 0;
    for (long long s = 0; s < p.n_steps; ++s) {
        const unsigned long long t = p.t0 + (unsigned long long)s;
        const bool rec = p.obs_every > 0 && --until_rec == 0;
        if (rec) until_rec = p.obs_every;
#pragma unroll 1
        for (int half = 0; half < 2; ++half) {
            uint32_t xa2, xb0;
            ChainKeys ck;
            device_half_step_keys(p.keys, 2ull * t + (unsigned)half, p.chain0 + (uint32_t)chain_first, xa2, xb0, ck);
            const bool sums = rec && half == 1;
#pragma unroll 1
            for (int c = tid; c < nvecs; c += blockDim.x) {
                const int r = c / nvec, v = c - r * nvec;
                uint32_t rnd[8];
                const uint32_t n0 = (uint32_t)(r * (L >> 3) + 2 * v);
                philox_site_words(n0, p.keys, xa2, xb0, ck, rnd);
                philox_site_words(n0 + 1u, p.keys, xa2, xb0, ck, rnd + 4);
                const int at = r * W + 4 * v;
                const int au = (r + 1 == L ? 0 : r + 1) * W + 4 * v, ad = (r == 0 ? L - 1 : r - 1) * W + 4 * v;
                const int ap = r * W + (v == 0 ? W - 1 : 4 * v - 1), an = r * W + (v + 1 == nvec ? 0 : 4 * v + 4);
                const int pc = (r + half) & 1;
#pragma unroll 1
                for (int m = 0; m < G; ++m) {
                    uint32_t *sg = smem + m * words;
                    const uint4 c4 = *reinterpret_cast<const uint4 *>(sg + at);
                    const uint32_t cw[6] = {sg[ap], c4.x, c4.y, c4.z, c4.w, sg[an]};
                    uint32_t fu[4], fd[4];
                    minus4(*reinterpret_cast<const uint4 *>(sg + au), fu);
                    minus4(*reinterpret_cast<const uint4 *>(sg + ad), fd);
                    int mM = 0, b1 = 0, bh = 0, bv = 0;
                    uint4 o;
                    const uint32_t tb = shared_addr(s_tab[m]);
                    if (sums) o = pc ? alt_vector_i8<1, true>(cw, fu, fd, rnd, tb, mM, b1, bh, bv) : alt_vector_i8<0, true>(cw, fu, fd, rnd, tb, mM, b1, bh, bv);
                    else o = pc ? alt_vector_i8<1, false>(cw, fu, fd, rnd, tb, mM, b1, bh, bv) : alt_vector_i8<0, false>(cw, fu, fd, rnd, tb, mM, b1, bh, bv);
                    *reinterpret_cast<uint4 *>(sg + at) = o;
                    if (sums) {
                        atomicAdd(&s_acc[m][0], mM);
                        atomicAdd(&s_acc[m][1], 2 * b1 - bh / 2);
                        atomicAdd(&s_acc[m][2], 2 * b1 - bv / 2);
                    }
                }
            }
            __syncthreads();
        }
        if (!coalesced) {                                 // T = min{n : X_n = Y_n}, in full steps
            uint32_t diff = 0;
            for (int i = tid; i < (G - 1) * words; i += blockDim.x) {
                const int m = 1 + i / words, w = i - (m - 1) * words;
                diff |= smem[w] ^ smem[m * words + w];
            }
            if (!__syncthreads_or(diff != 0)) {
                coalesced = true;
                if (tid == 0) p.coal[gi] = (long long)(t + 1);
            }
        }
        if (rec) {
            if (tid < G) {
                long long *out = p.rec + ((size_t)nrec * p.n_chains + chain_first + tid) * 6;
                out[0] = s_acc[tid][0];
                out[4] = s_acc[tid][1];
                out[5] = s_acc[tid][2];
                s_acc[tid][0] = s_acc[tid][1] = s_acc[tid][2] = 0;   // next used after the barrier of a later half-step
            }
            ++nrec;
        }
    }
    for (int m = 0; m < G; ++m) {
        uint32_t *gs = reinterpret_cast<uint32_t *>(p.sigma + (size_t)(chain_first + m) * L * L);
        for (int i = tid; i < words; i += blockDim.x) gs[i] = smem[m * words + i];
    }
}

// Mid-size lattices (128 < L <= 2048, few chains): the whole run in ONE cooperative launch, row bands in shared memory,
// as kernel_band.cuh does for the shaken dynamics (two launches per step are 6-9 us of launch latency for well under a
// microsecond of work at 1024^2).  Here a redrawn site reads the rows above AND below, so a band keeps TWO halo rows on
// either side and redraws, in half-step 0, also the nearest halo row on each side (redundantly: the random word of a site
// is a function of the site), which makes the halo of half-step 1 valid without a hand-over in between.  Bands exchange
// once per full step: after half-step 1 a band publishes its two bottom and its two top rows ({word, stamp} pairs, see
// kernel_band.cuh) and collects the neighbours' rows at the start of the next step.  rows_per_band is even, so every
// band has at least two rows.  BandParams: xtop / xbot hold [2][n_bands][2][L/4] pairs, utab / gtab the table A[0..4].
__host__ __device__ inline size_t alt_band_smem_bytes(int L, int rows_per_band) { return (size_t)(rows_per_band + 4) * (size_t)(L / 4) * sizeof(uint32_t); }

__global__ void __launch_bounds__(BAND_THREADS, 1) alt_band_i8(const __grid_constant__ BandParams p)
{
    extern __shared__ __align__(16) uint32_t smem[];
    __shared__ __align__(256) uint32_t s_tab[ALT_TAB_WORDS];
    __shared__ int s_acc[3];                      // the band's partial sums (M, C_x, C_y) of the record in progress

    const int L = p.L, W = L >> 2, nvec = W >> 2;
    const int band = blockIdx.x, chain = band / p.bpc, k = band - chain * p.bpc;
    const int r0 = k * p.rows_per_band;
    const int nr = min(L, r0 + p.rows_per_band) - r0;                 // rows of this band (even, >= 2)
    const int below = chain * p.bpc + (k == 0 ? p.bpc - 1 : k - 1);
    const int above = chain * p.bpc + (k == p.bpc - 1 ? 0 : k + 1);
    const int nb = gridDim.x;
    const int tid = threadIdx.x, lane = tid & 31;
    uint32_t *sg = smem;                          // row index j holds global row r0 - 2 + j (mod L), j = 0 .. nr + 3
    uint32_t *gs = reinterpret_cast<uint32_t *>(p.sigma + (size_t)chain * L * L);
    for (int i = tid; i < (nr + 4) * W; i += BAND_THREADS) {
        const int j = (int)__umulhi((uint32_t)i, p.magicW), cw = i - j * W;
        int gr = r0 - 2 + j;
        gr = gr < 0 ? gr + L : (gr >= L ? gr - L : gr);
        sg[i] = gs[(size_t)gr * W + cw];
    }
    if (tid < 8) s_tab[tid] = tid < 5 ? (p.gtab ? p.gtab[(size_t)chain * 8 + 4 - tid] : p.utab[4 - tid]) : 0u;   // entry i = A[4 - i]
    if (tid < 3) s_acc[tid] = 0;
    __syncthreads();
    const uint32_t tb = shared_addr(s_tab);

    uint32_t xa2 = 0, xb0 = 0;
    ChainKeys ck = {0u, 0u};
    // one vector (16 sites, the 8 of the row's active parity redrawn) of row index j, in place
    int accM = 0, a1 = 0, ah = 0, av = 0;         // partial sums of a recorded step (see alt_vector_i8)
    auto redraw = [&](const int half, const int j, const int v, const bool sums) -> uint4 {
        int gr = r0 - 2 + j;
        gr = gr < 0 ? gr + L : (gr >= L ? gr - L : gr);
        uint32_t *row = sg + j * W;
        const uint4 c4 = *reinterpret_cast<const uint4 *>(row + 4 * v);
        const uint32_t cw[6] = {row[v == 0 ? W - 1 : 4 * v - 1], c4.x, c4.y, c4.z, c4.w, row[v + 1 == nvec ? 0 : 4 * v + 4]};
        uint32_t fu[4], fd[4];
        minus4(*reinterpret_cast<const uint4 *>(row + W + 4 * v), fu);
        minus4(*reinterpret_cast<const uint4 *>(row - W + 4 * v), fd);
        uint32_t rnd[8];
        const uint32_t n0 = (uint32_t)gr * (uint32_t)(L >> 3) + 2u * (uint32_t)v;
        philox_site_words(n0, p.keys, xa2, xb0, ck, rnd);
        philox_site_words(n0 + 1u, p.keys, xa2, xb0, ck, rnd + 4);
        uint4 o;
        if (sums) o = ((gr + half) & 1) ? alt_vector_i8<1, true>(cw, fu, fd, rnd, tb, accM, a1, ah, av) : alt_vector_i8<0, true>(cw, fu, fd, rnd, tb, accM, a1, ah, av);
        else o = ((gr + half) & 1) ? alt_vector_i8<1, false>(cw, fu, fd, rnd, tb, accM, a1, ah, av) : alt_vector_i8<0, false>(cw, fu, fd, rnd, tb, accM, a1, ah, av);
        *reinterpret_cast<uint4 *>(row + 4 * v) = o;
        return o;
    };
    // neighbours' rows of the step just finished: row indices 0, 1 from the band below, nr + 2, nr + 3 from the band above
    auto collect = [&](const long long s_done) {
        const uint32_t stamp_in = p.stamp0 + (uint32_t)s_done;
        const uint2 *in_below = p.xtop + ((size_t)((s_done + 1) & 1) * nb + below) * 2 * W;
        const uint2 *in_above = p.xbot + ((size_t)((s_done + 1) & 1) * nb + above) * 2 * W;
        for (int i = tid; i < 4 * W; i += BAND_THREADS) {
            const uint2 *src = i < 2 * W ? in_below + i : in_above + (i - 2 * W);
            uint2 a;
            do { a = ld_pair(src); } while (a.y != stamp_in);
            sg[i < 2 * W ? i : (nr + 2) * W + (i - 2 * W)] = a.x;
        }
    };

    long long nrec = 0;
    long long until_rec = p.obs_every > 0 ? p.obs_every - (long long)(p.t0 % (unsigned long long)p.obs_every) : 0;
#pragma unroll 1
    for (long long s = 0; s < p.n_steps; ++s) {
        const unsigned long long t = p.t0 + (unsigned long long)s;
        const bool rec = p.obs_every > 0 && --until_rec == 0;            // block-uniform
        if (rec) until_rec = p.obs_every;
        // half-step 0: colour 0 of row indices 1 .. nr + 2 (the band and one halo row on either side).  First the rows
        // that read only the band's own rows (indices 3 .. nr), then the neighbours' rows of the previous step are
        // collected -- they were published early in the neighbours' half-step 1 and have had all that time to arrive --
        // and the four rows next to them follow (indices 1, 2, nr + 1, nr + 2).
        device_half_step_keys(p.keys, 2ull * t, p.chain0 + (uint32_t)chain, xa2, xb0, ck);
#pragma unroll 1
        for (int c = tid; c < (nr - 2) * nvec; c += BAND_THREADS) {
            const int kk = (int)__umulhi((uint32_t)c, p.magicV);
            redraw(0, 3 + kk, c - kk * nvec, false);
        }
        if (s > 0) collect(s);
        __syncthreads();
#pragma unroll 1
        for (int c = tid; c < 4 * nvec; c += BAND_THREADS) {
            const int kk = (int)__umulhi((uint32_t)c, p.magicV);
            redraw(0, kk < 2 ? 1 + kk : nr - 1 + kk, c - kk * nvec, false);
        }
        __syncthreads();
        // half-step 1: colour 1 of the band's rows (indices 2 .. nr + 1); the two top rows and the two bottom rows first,
        // each vector published by the thread that computed it.  On a recorded step the sums are fused in: every bond of
        // the lattice joins a site redrawn here to a passive one (final since half-step 0, also in the halo rows), so
        // M = sum of the stored vectors, C_x = sum_{x redrawn} s_x (left + right), C_y = sum_{x redrawn} s_x (up + down),
        // each bond counted once, by the band that owns its redrawn end -- no neighbour row is waited for.
        device_half_step_keys(p.keys, 2ull * t + 1ull, p.chain0 + (uint32_t)chain, xa2, xb0, ck);
        const uint32_t stamp_out = p.stamp0 + (uint32_t)s + 1u;
        uint2 *out_top = p.xtop + ((size_t)(s & 1) * nb + band) * 2 * W;   // rows r1-2, r1-1
        uint2 *out_bot = p.xbot + ((size_t)(s & 1) * nb + band) * 2 * W;   // rows r0, r0+1
#pragma unroll 1
        for (int c = tid; c < nr * nvec; c += BAND_THREADS) {
            const int kk = (int)__umulhi((uint32_t)c, p.magicV), v = c - kk * nvec;
            const int j = kk == 0 ? nr + 1 : (kk == 1 ? nr : kk);              // row index: nr+1, nr, 2, 3, 4 .. nr-1
            const uint4 o = redraw(1, j, v, rec);
            if (j >= nr) {
                uint2 *x = out_top + (j - nr) * W + 4 * v;
                st_pair(x, o.x, stamp_out); st_pair(x + 1, o.y, stamp_out); st_pair(x + 2, o.z, stamp_out); st_pair(x + 3, o.w, stamp_out);
            }
            if (j <= 3) {
                uint2 *x = out_bot + (j - 2) * W + 4 * v;
                st_pair(x, o.x, stamp_out); st_pair(x + 1, o.y, stamp_out); st_pair(x + 2, o.z, stamp_out); st_pair(x + 3, o.w, stamp_out);
            }
        }
        if (rec) {
            // s * (l + r) = s * (2 - 2 * minus) per site: ah, av hold 4 * minus, so they are multiples of 4 (see alt_half)
            const int w0 = __reduce_add_sync(0xFFFFFFFFu, accM), w1 = __reduce_add_sync(0xFFFFFFFFu, 2 * a1 - ah / 2),
                      w2 = __reduce_add_sync(0xFFFFFFFFu, 2 * a1 - av / 2);
            if (lane == 0) { atomicAdd(&s_acc[0], w0); atomicAdd(&s_acc[1], w1); atomicAdd(&s_acc[2], w2); }
            accM = a1 = ah = av = 0;
        }
        __syncthreads();
        if (rec) {
            if (tid < 3) {
                long long *dst = p.rec + ((size_t)nrec * p.n_chains + chain) * 6;
                atomicAdd(reinterpret_cast<unsigned long long *>(dst + (tid ? 3 + tid : 0)), (unsigned long long)(long long)s_acc[tid]);   // M, C_x, C_y at 0, 4, 5
                s_acc[tid] = 0;                   // next written after at least one more block barrier
            }
            ++nrec;
        }
    }
    for (int i = tid; i < nr * W; i += BAND_THREADS) gs[(size_t)r0 * W + i] = sg[2 * W + i];
}

} // namespace shaken
