// pipe_rates.cu -- measurement tool: issue intervals of the sm_100a integer instructions that bound the half-step
// kernels, alone and in pairs (do two instruction kinds overlap or add?), and the rate of the product's own hoisted
// Philox4x32-10 (philox.cuh) with no memory traffic.  DESIGN.md "Rooflines" takes its ALU ceiling from the numbers
// this prints (profiles/r1_pipe_rates.md).
//
//   build:  python -m paper_1908_07341_b200.build --pipe-rates      run:  paper_1908_07341_b200/pipe_rates
#include <cstdint>
#include <cstdio>
#include <cuda_runtime.h>

#include "philox.cuh"

#define ITERS 2048
#define CH 8
enum { WIDE, IMADLO, LOP3, IADD3, ISETPX, SHF, PRMT, LDS, IDP, FFMA, NONE };
const char *names[] = {"WIDE", "IMADLO", "LOP3", "IADD3", "ISETP+@pLOP3", "SHF", "PRMT", "LDS", "IDP", "FFMA", "-"};
template <int OP> __device__ __forceinline__ void op(uint32_t &x, uint32_t &y, uint32_t ka, uint32_t kb, const uint32_t *sm)
{
    if (OP == WIDE) { uint64_t p; asm volatile("mul.wide.u32 %0, %1, 0xD2511F53;" : "=l"(p) : "r"(x)); x = (uint32_t)(p >> 32); y = (uint32_t)p; }
    else if (OP == IMADLO) { asm volatile("mad.lo.u32 %0, %1, 0xD2511F53, %2;" : "=r"(x) : "r"(x), "r"(y)); }
    else if (OP == LOP3) { asm volatile("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(x) : "r"(x), "r"(y), "r"(ka)); }
    else if (OP == IADD3) { asm volatile("add.u32 %0, %1, %2;" : "=r"(x) : "r"(x), "r"(y)); }
    else if (OP == ISETPX) { asm volatile("{\n\t.reg .pred p;\n\tsetp.lo.u32 p, %1, %2;\n\t@p xor.b32 %0, %0, %3;\n\t}" : "+r"(x) : "r"(y), "r"(ka), "r"(kb)); }
    else if (OP == SHF) { asm volatile("shf.l.wrap.b32 %0, %1, %2, 8;" : "=r"(x) : "r"(x), "r"(y)); }
    else if (OP == PRMT) { asm volatile("prmt.b32 %0, %1, %2, 0x4321;" : "=r"(x) : "r"(x), "r"(y)); }
    else if (OP == LDS) { asm volatile("ld.shared.u32 %0, [%1];" : "=r"(x) : "r"((uint32_t)(x & 0x7Cu) + (uint32_t)__cvta_generic_to_shared(sm))); }
    else if (OP == IDP) { x = (uint32_t)__dp4a((int)y, (int)x, (int)x); }
    else if (OP == FFMA) { float a = __uint_as_float(x), b = __uint_as_float(y); asm volatile("fma.rn.f32 %0, %1, %2, %3;" : "=f"(a) : "f"(a), "f"(b), "f"(b)); x = __float_as_uint(a); }
}
template <int A, int NA, int B, int NB> __global__ void __launch_bounds__(256) k(uint32_t *out, uint32_t seed, uint32_t ka, uint32_t kb)
{
    __shared__ uint32_t sm[64];
    if (threadIdx.x < 64) sm[threadIdx.x] = (threadIdx.x * 4) & 0x7C;
    __syncthreads();
    uint32_t x[CH], y[CH], u[CH], v[CH];
#pragma unroll
    for (int i = 0; i < CH; ++i) { x[i] = seed + threadIdx.x * 977u + i * 131u + blockIdx.x; y[i] = x[i] ^ 0x5bd1e995u; u[i] = y[i] * 3u; v[i] = u[i] + 17u; }
    for (int it = 0; it < ITERS; ++it) {
#pragma unroll
        for (int r = 0; r < (NA > NB ? NA : NB); ++r)
#pragma unroll
            for (int i = 0; i < CH; ++i) {
                if (r < NA) op<A>(x[i], y[i], ka, kb, sm);
                if (r < NB) op<B>(u[i], v[i], ka, kb, sm);
            }
    }
    uint32_t acc = 0;
#pragma unroll
    for (int i = 0; i < CH; ++i) acc ^= x[i] ^ y[i] ^ u[i] ^ v[i];
    if (acc == 0x12345678u) out[threadIdx.x] = acc;
}
template <int A, int NA, int B, int NB> void run()
{
    const int bps = 4;
    uint32_t *d; cudaMalloc(&d, 4096);
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    k<A, NA, B, NB><<<148 * bps, 256>>>(d, 1, 0x9E3779B9u, 0xBB67AE85u); cudaDeviceSynchronize();
    cudaEventRecord(e0); k<A, NA, B, NB><<<148 * bps, 256>>>(d, 1, 0x9E3779B9u, 0xBB67AE85u); cudaEventRecord(e1); cudaEventSynchronize(e1);
    float ms; cudaEventElapsedTime(&ms, e0, e1);
    double n = (double)bps * 2 * ITERS * CH;
    printf("%d x %-13s + %d x %-13s : %6.2f cyc/warp-iter/SMSP\n", NA, names[A], NB, names[B], ms * 1e6 / n * 1.965);
    cudaFree(d);
}
// the product's hoisted Philox (18 IMAD.WIDE + 19 LOP3 per 4 sites) with a compare per word and nothing else
__global__ void __launch_bounds__(256) philox_only(uint32_t *out, const __grid_constant__ shaken::StepKeys K, int iters)
{
    const shaken::ChainKeys ck = shaken::make_chain_keys(K, 0u);
    uint32_t n = (blockIdx.x * 256u + threadIdx.x) * 4u * (uint32_t)iters, acc = 0;
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            uint32_t r[4];
            shaken::philox_site_words(n + j, K, ck, r);
            acc += (r[0] < 0x80000000u) + (r[1] < 0x70000000u) + (r[2] < 0x60000000u) + (r[3] < 0x50000000u);
        }
        n += 4;
    }
    if (acc == 0x12345678u) out[0] = acc;
}

int main()
{
    int sms = 0, khz = 0;
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, 0);
    cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, 0);
    printf("SMs=%d  max SM clock=%d MHz; cycles below assume 1965 MHz (bench.py samples the clock under load)\n", sms, khz / 1000);
    printf("-- one instruction kind alone (8 independent chains per thread, 8 warps per SMSP)\n");
    run<WIDE,1,NONE,0>(); run<IMADLO,1,NONE,0>(); run<LOP3,1,NONE,0>(); run<IADD3,1,NONE,0>(); run<ISETPX,1,NONE,0>(); run<SHF,1,NONE,0>(); run<PRMT,1,NONE,0>(); run<LDS,1,NONE,0>(); run<IDP,1,NONE,0>(); run<FFMA,1,NONE,0>();
    printf("-- IMAD.WIDE beside another kind\n");
    run<WIDE,1,IMADLO,1>(); run<WIDE,1,LOP3,1>(); run<WIDE,1,LOP3,2>(); run<WIDE,1,LOP3,3>(); run<WIDE,1,IADD3,1>(); run<WIDE,1,ISETPX,1>(); run<WIDE,1,SHF,1>(); run<WIDE,1,PRMT,1>(); run<WIDE,1,LDS,1>(); run<WIDE,1,LDS,2>(); run<WIDE,1,IDP,1>(); run<WIDE,1,FFMA,1>();
    printf("-- LOP3 beside another kind\n");
    run<LOP3,1,IMADLO,1>(); run<LOP3,1,IADD3,1>(); run<LOP3,1,SHF,1>(); run<LOP3,1,PRMT,1>(); run<LOP3,1,LDS,1>(); run<LOP3,1,IDP,1>(); run<LOP3,1,FFMA,1>(); run<LOP3,1,ISETPX,1>(); run<IMADLO,1,IDP,1>();
    printf("-- one Philox round's mix: 2 IMAD.WIDE + 2 LOP3\n");
    run<WIDE,2,LOP3,2>();

    shaken::StepKeys K;
    shaken::make_step_keys(3, 12345, K);
    uint32_t *d;
    cudaMalloc(&d, 64);
    for (int b = 2; b <= 8; b *= 2) {
        const int iters = 2048;
        cudaEvent_t e0, e1;
        cudaEventCreate(&e0); cudaEventCreate(&e1);
        philox_only<<<sms * b, 256>>>(d, K, iters);
        cudaDeviceSynchronize();
        cudaEventRecord(e0);
        philox_only<<<sms * b, 256>>>(d, K, iters);
        cudaEventRecord(e1);
        cudaEventSynchronize(e1);
        float ms;
        cudaEventElapsedTime(&ms, e0, e1);
        printf("hoisted Philox4x32-10 only, blocks/SM=%d: %8.3f ms  %7.1f sites/ns (32 random bits per site)\n", b, ms, (double)sms * b * 256 * iters * 16 / (ms * 1e6));
    }
    return 0;
}
