// kernels_common.cuh -- sm_100a kernels of libshaken: the shaken-dynamics half-step (eq. (15)-(16))
// on int8 and bit-packed spins, with fused observable sums (eq. (17) :196, eq. (5) :81-84).
//
// Work decomposition (both layouts).  A *task* is a column strip of one warp: 32 lanes x one vector
// (int8: 16 spins = one 16-byte load; packed: one 32-spin word) wide, `rows_per_task` rows high, of one chain.
// A lane walks its strip row by row IN THE DIRECTION OF THE FIELD (half 0 reads down/left, so rows ascend
// and the previous row in registers is the "down" neighbour; half 1 reads up/right, rows descend), which
// leaves one halo row per task and, per row, the one spin left (right) of the lane's vector, taken from
// an extra 4-byte load that hits the line the neighbouring lane just fetched.  The next row is loaded
// before the current one is computed.  Warps loop over tasks with a grid sized to the machine.
//
// Acceptance ("rand() < p"): new spin = +1 iff rnd < T[idx], T looked up in shared memory
// by a byte offset that is computed for 4 sites at a time with byte-SIMD integer arithmetic.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "philox.cuh"

namespace shaken {

constexpr int I8_THREADS = 512;         // int8 half-step: one 512-thread block per SM, up to 128 registers per thread
constexpr int MAX_ROWS_PER_TASK = 4096;   // int32 observable partials: 2 * 512 * rows per warp stay far below 2^31

enum : int { F_OBS = 1, F_BONDS = 2, F_NOUPDATE = 4, F_COAL = 8 };

struct StepParams {
    const void *src;        // sublattice that is read   (half 0: sigma, half 1: tau)
    void *dst;              // sublattice that is redrawn (half 0: tau,   half 1: sigma)
    int L;                  // lattice side
    int nvec;               // vectors per row: L/16 (int8) or L/32 (packed)
    int n_chains;
    uint32_t chain0;        // global index of chain 0 of this context (Philox counter word 1 = chain0 + rng chain)
    int group;              // coupling group size (>= 1): chains c with equal c / group draw the words of chain
                            // (c / group) * group, i.e. evolve with the same random numbers
    int rows_per_task;
    int nseg;               // warp-wide strips per row = ceil(nvec / 32)
    int nrb;                // row blocks = ceil(L / rows_per_task)
    long long ntasks;       // block tasks: n_chains * ceil(nrb * nseg / warps per block); per-warp lists: number of ranges
    long long rows_total;   // per-warp lists: n_chains * nseg * rows = strip-rows in the launch
    int range_len;          // per-warp lists: strip-rows per range (<= MAX_ROWS_PER_TASK)
    int slab_rows;          // 0: a whole L x L torus.  > 0: a SLAB of one lattice (row-slab sharding, kernel_slab.cuh): this
                            // many rows are redrawn; src / dst point at the slab's row 0 and the arrays hold the rows just
                            // below (index -1) and above (index slab_rows) as well, so vertical neighbours never wrap
    uint32_t row0;          // global index of the slab's row 0 (enters the Philox counter); 0 for a whole torus
    const uint32_t *gtab;   // per-chain tables [n_chains][8] in global memory, or nullptr: use utab
    uint32_t utab[8];       // one table for all chains (kernel parameters live in constant memory)
    long long *rec_cur;     // [n_chains][6] record of the step being computed (F_OBS) or nullptr
    long long *rec_prev;    // [n_chains][6] record whose C_x, C_y are still owed (F_BONDS) or nullptr
    // coupled chains (group > 1), PAPER.md:234 T = min{n : X_n = Y_n}: half-step 0 launches with F_COAL compare the sigma
    // they read (the state after `cstamp` full steps) of every member with the group's first chain and stamp diff[group]
    // with cstamp where they differ; the half-step 1 launch that follows (do_fin, fin_stamp) turns "no difference stamped"
    // into the coalescence time (do_fin).  coal: [n_groups] times, -1 = not yet; diff: [n_groups] stamps.
    long long *coal;
    unsigned long long *diff;
    unsigned long long cstamp;
    unsigned long long fin_stamp;
    int do_fin;
    StepKeys keys;
};

// coalescence bookkeeping at the start of a half-step 1 launch (block 0 only; the half-step 0 launch that stamped the
// differences has completed: wait_for_previous_kernel)
__device__ __forceinline__ void finalize_coalescence(const StepParams &p)
{
    if (p.do_fin && blockIdx.x == 0) {
        const long long ng = p.n_chains / p.group;
        for (long long gi = threadIdx.x; gi < ng; gi += blockDim.x)
            if (p.coal[gi] < 0 && p.diff[gi] != p.fin_stamp) p.coal[gi] = (long long)p.fin_stamp;
    }
}

// counter word 1 of a chain: its own global index, or that of the first chain of its coupling group
__device__ __forceinline__ uint32_t rng_chain(const StepParams &p, int chain) { return p.chain0 + (uint32_t)((chain / p.group) * p.group); }

__device__ __forceinline__ uint4 ldg128(const void *p) { return __ldg(reinterpret_cast<const uint4 *>(p)); }
__device__ __forceinline__ uint32_t ldg32(const void *p) { return __ldg(reinterpret_cast<const uint32_t *>(p)); }

__device__ __forceinline__ int bytes_sum(uint32_t acc) { return (int)__dp4a(acc, 0x01010101u, 0u); }

__device__ __forceinline__ void warp_add_to(long long *addr, int v)
{
    int s = __reduce_add_sync(0xFFFFFFFFu, v);
    if ((threadIdx.x & 31) == 0 && s != 0) atomicAdd(reinterpret_cast<unsigned long long *>(addr), (unsigned long long)(long long)s);
}

// Programmatic dependent launch: the half-step kernels of a run are launched back to back with
// cudaLaunchAttributeProgrammaticStreamSerialization, so the launch of kernel n+1 is processed while kernel n still runs;
// kernel n+1 must not touch memory before kernel n has completed and flushed, which is what this waits for (a no-op
// for a kernel launched the ordinary way).
__device__ __forceinline__ void wait_for_previous_kernel() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void let_next_kernel_launch() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// out ^= c if a < b (unsigned): one ISETP and one predicated LOP3
__device__ __forceinline__ uint32_t xor_if_less(uint32_t out, uint32_t a, uint32_t b, uint32_t c)
{
    asm("{\n\t.reg .pred p;\n\tsetp.lo.u32 p, %1, %2;\n\t@p xor.b32 %0, %0, %3;\n\t}" : "+r"(out) : "r"(a), "r"(b), "r"(c));
    return out;
}

// out += c if a < b (unsigned): one ISETP and one predicated add
__device__ __forceinline__ uint32_t add_if_less(uint32_t out, uint32_t a, uint32_t b, uint32_t c)
{
    asm("{\n\t.reg .pred p;\n\tsetp.lo.u32 p, %1, %2;\n\t@p add.u32 %0, %0, %3;\n\t}" : "+r"(out) : "r"(a), "r"(b), "r"(c));
    return out;
}

// out += c if !(a < b) (unsigned): one ISETP and one predicated add (IADD3 costs about half a LOP3 on the ALU port)
__device__ __forceinline__ uint32_t add_if_not_less(uint32_t out, uint32_t a, uint32_t b, uint32_t c)
{
    asm("{\n\t.reg .pred p;\n\tsetp.hs.u32 p, %1, %2;\n\t@p add.u32 %0, %0, %3;\n\t}" : "+r"(out) : "r"(a), "r"(b), "r"(c));
    return out;
}

} // namespace shaken
