// micro-benchmarks of integer pipes on B200: thread-instructions per clock per SM
#include <cstdio>
#include <cstdint>
#include <cuda_runtime.h>
#define ITER 4096
#define NCH 8
template <int MODE>
__global__ void __launch_bounds__(256) k(uint32_t *out, uint32_t seed, unsigned long long *clk)
{
    uint32_t x[NCH], y[NCH];
    for (int i = 0; i < NCH; ++i) { x[i] = seed + threadIdx.x * 7 + i; y[i] = seed ^ (i * 0x9E3779B9u); }
    unsigned long long t0 = clock64();
    for (int it = 0; it < ITER; ++it) {
#pragma unroll
        for (int i = 0; i < NCH; ++i) {
            if (MODE == 0) {          // LOP3 chain
                asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(x[i]) : "r"(y[i]), "r"(seed));
            } else if (MODE == 1) {   // IMAD.WIDE.U32
                unsigned long long p = (unsigned long long)x[i] * 0xD2511F53ull;
                x[i] = (uint32_t)(p >> 32) ^ 0; y[i] += (uint32_t)p;   // uses both halves (adds IADD)
            } else if (MODE == 2) {   // mul.wide only, hi feeds next
                uint32_t lo, hi;
                asm volatile("{.reg .u64 p; mul.wide.u32 p, %2, 0xD2511F53; mov.b64 {%0,%1}, p;}" : "=r"(lo), "=r"(hi) : "r"(x[i]));
                x[i] = hi; y[i] = lo;
            } else if (MODE == 3) {   // 1 mul.wide + 1 lop3 (philox-like)
                uint32_t lo, hi;
                asm volatile("{.reg .u64 p; mul.wide.u32 p, %2, 0xD2511F53; mov.b64 {%0,%1}, p;}" : "=r"(lo), "=r"(hi) : "r"(x[i]));
                asm volatile("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(x[i]) : "r"(hi), "r"(y[i]), "r"(seed));
                y[i] = lo;
            } else if (MODE == 4) {   // 1 mul.wide + 2 lop3
                uint32_t lo, hi;
                asm volatile("{.reg .u64 p; mul.wide.u32 p, %2, 0xD2511F53; mov.b64 {%0,%1}, p;}" : "=r"(lo), "=r"(hi) : "r"(x[i]));
                asm volatile("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(x[i]) : "r"(hi), "r"(y[i]), "r"(seed));
                asm volatile("lop3.b32 %0, %1, %2, %3, 0xe8;" : "=r"(y[i]) : "r"(lo), "r"(y[i]), "r"(x[i]));
            } else if (MODE == 5) {   // mul.hi
                x[i] = __umulhi(x[i], 0xD2511F53u);
            } else if (MODE == 6) {   // mul.lo
                x[i] = x[i] * 0xD2511F53u;
            } else if (MODE == 7) {   // popc + add
                x[i] += __popc(x[i]);
            } else if (MODE == 8) {   // shf
                x[i] = __funnelshift_r(x[i], y[i], 5);
            } else if (MODE == 9) {   // iadd3
                asm volatile("add.u32 %0, %0, %1;" : "+r"(x[i]) : "r"(y[i]));
            } else if (MODE == 10) {  // 1 mul.wide + 3 lop3
                uint32_t lo, hi;
                asm volatile("{.reg .u64 p; mul.wide.u32 p, %2, 0xD2511F53; mov.b64 {%0,%1}, p;}" : "=r"(lo), "=r"(hi) : "r"(x[i]));
                asm volatile("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(x[i]) : "r"(hi), "r"(y[i]), "r"(seed));
                asm volatile("lop3.b32 %0, %1, %2, %3, 0xe8;" : "=r"(y[i]) : "r"(lo), "r"(y[i]), "r"(x[i]));
                asm volatile("lop3.b32 %0, %1, %2, %3, 0x1e;" : "=r"(x[i]) : "r"(lo), "r"(y[i]), "r"(x[i]));
            } else if (MODE == 11) {  // mul.lo + mul.hi pair (same result as wide)
                uint32_t lo = x[i] * 0xD2511F53u, hi = __umulhi(x[i], 0xD2511F53u);
                x[i] = hi; y[i] ^= lo;
            } else if (MODE >= 20 && MODE < 30) {  // mul.hi + mul.lo + (MODE-20) lop3
                uint32_t lo = x[i] * 0xD2511F53u, hi = __umulhi(x[i], 0xD2511F53u);
                asm volatile("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(x[i]) : "r"(hi), "r"(y[i]), "r"(seed));
                if (MODE >= 22) asm volatile("lop3.b32 %0, %1, %2, %3, 0xe8;" : "=r"(y[i]) : "r"(lo), "r"(y[i]), "r"(x[i]));
                else y[i] = lo;
                if (MODE >= 23) asm volatile("lop3.b32 %0, %1, %2, %3, 0x1e;" : "=r"(x[i]) : "r"(lo), "r"(y[i]), "r"(x[i]));
                if (MODE >= 24) asm volatile("lop3.b32 %0, %1, %2, %3, 0x2e;" : "=r"(y[i]) : "r"(lo), "r"(y[i]), "r"(x[i]));
            } else if (MODE >= 30 && MODE < 40) {  // mul.wide + (MODE-30) lop3
                uint32_t lo, hi;
                asm volatile("{.reg .u64 p; mul.wide.u32 p, %2, 0xD2511F53; mov.b64 {%0,%1}, p;}" : "=r"(lo), "=r"(hi) : "r"(x[i]));
                asm volatile("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(x[i]) : "r"(hi), "r"(y[i]), "r"(seed));
                if (MODE >= 32) asm volatile("lop3.b32 %0, %1, %2, %3, 0xe8;" : "=r"(y[i]) : "r"(lo), "r"(y[i]), "r"(x[i]));
                else y[i] = lo;
                if (MODE >= 33) asm volatile("lop3.b32 %0, %1, %2, %3, 0x1e;" : "=r"(x[i]) : "r"(lo), "r"(y[i]), "r"(x[i]));
                if (MODE >= 34) asm volatile("lop3.b32 %0, %1, %2, %3, 0x2e;" : "=r"(y[i]) : "r"(lo), "r"(y[i]), "r"(x[i]));
            } else if (MODE == 40) {  // mul.hi + 1 lop3 + 1 iadd
                uint32_t hi = __umulhi(x[i], 0xD2511F53u);
                asm volatile("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(x[i]) : "r"(hi), "r"(y[i]), "r"(seed));
            } else if (MODE == 41) {  // mul.hi + 2 lop3
                uint32_t hi = __umulhi(x[i], 0xD2511F53u);
                asm volatile("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(x[i]) : "r"(hi), "r"(y[i]), "r"(seed));
                asm volatile("lop3.b32 %0, %1, %2, %3, 0xe8;" : "=r"(y[i]) : "r"(hi), "r"(y[i]), "r"(x[i]));
            } else if (MODE == 42) {  // mul.hi + 3 lop3
                uint32_t hi = __umulhi(x[i], 0xD2511F53u);
                asm volatile("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(x[i]) : "r"(hi), "r"(y[i]), "r"(seed));
                asm volatile("lop3.b32 %0, %1, %2, %3, 0xe8;" : "=r"(y[i]) : "r"(hi), "r"(y[i]), "r"(x[i]));
                asm volatile("lop3.b32 %0, %1, %2, %3, 0x1e;" : "=r"(x[i]) : "r"(hi), "r"(y[i]), "r"(x[i]));
            } else if (MODE == 43) {  // mul.lo + 2 lop3
                uint32_t lo = x[i] * 0xD2511F53u;
                asm volatile("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(x[i]) : "r"(lo), "r"(y[i]), "r"(seed));
                asm volatile("lop3.b32 %0, %1, %2, %3, 0xe8;" : "=r"(y[i]) : "r"(lo), "r"(y[i]), "r"(x[i]));
            } else if (MODE == 44) {  // mul.lo + 1 lop3
                uint32_t lo = x[i] * 0xD2511F53u;
                asm volatile("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(x[i]) : "r"(lo), "r"(y[i]), "r"(seed));
            } else if (MODE == 12) {  // lop3 + iadd
                asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(x[i]) : "r"(y[i]), "r"(seed));
                asm volatile("add.u32 %0, %0, %1;" : "+r"(y[i]) : "r"(x[i]));
            }
        }
    }
    unsigned long long t1 = clock64();
    uint32_t s = 0;
    for (int i = 0; i < NCH; ++i) s ^= x[i] ^ y[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
    if (threadIdx.x == 0) clk[blockIdx.x] = t1 - t0;
}
template <int MODE>
void run(const char *name, double instr_per_iter_per_chain)
{
    const int blocks = 148 * 4;   // 4 blocks of 256 per SM = 32 warps/SM
    uint32_t *out; unsigned long long *clk;
    cudaMalloc(&out, blocks * 256 * 4); cudaMalloc(&clk, blocks * 8);
    k<MODE><<<blocks, 256>>>(out, 12345u, clk);
    cudaDeviceSynchronize();
    cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
    cudaEventRecord(e0);
    k<MODE><<<blocks, 256>>>(out, 12345u, clk);
    cudaEventRecord(e1); cudaEventSynchronize(e1);
    float ms; cudaEventElapsedTime(&ms, e0, e1);
    unsigned long long h[148 * 4]; cudaMemcpy(h, clk, sizeof h, cudaMemcpyDeviceToHost);
    double avg = 0; for (int i = 0; i < blocks; ++i) avg += h[i]; avg /= blocks;
    double instr_per_sm = 4.0 * 256 * ITER * NCH * instr_per_iter_per_chain;
    printf("%-28s %.3f ms  %6.2f cycles/group/SMSP  (%.1f thread-instr/clk/SM)\n", name, ms, ms*1e-3*1.965e9/(8.0*ITER*NCH), 4.0*256*ITER*NCH*instr_per_iter_per_chain/(ms*1e-3*1.965e9));
    cudaFree(out); cudaFree(clk);
}
int main()
{
    run<0>("lop3", 1);
    run<1>("imad.wide+use both", 1);
    run<2>("mul.wide only", 1);
    run<3>("1 mul.wide + 1 lop3 (count 2)", 2);
    run<4>("1 mul.wide + 2 lop3 (count 3)", 3);
    run<10>("1 mul.wide + 3 lop3 (count 4)", 4);
    run<5>("mul.hi", 1);
    run<6>("mul.lo", 1);
    run<11>("mul.lo + mul.hi + xor (3)", 3);
    run<7>("popc + add (count 2)", 2);
    run<8>("shf", 1);
    run<9>("iadd", 1);
    run<12>("lop3 + iadd (count 2)", 2);
    run<21>("mul.lo+mul.hi + 1 lop3", 3);
    run<22>("mul.lo+mul.hi + 2 lop3", 4);
    run<23>("mul.lo+mul.hi + 3 lop3", 5);
    run<24>("mul.lo+mul.hi + 4 lop3", 6);
    run<31>("mul.wide + 1 lop3", 2);
    run<32>("mul.wide + 2 lop3", 3);
    run<33>("mul.wide + 3 lop3", 4);
    run<34>("mul.wide + 4 lop3", 5);
    run<40>("mul.hi + 1 lop3", 2);
    run<41>("mul.hi + 2 lop3", 3);
    run<42>("mul.hi + 3 lop3", 4);
    run<44>("mul.lo + 1 lop3", 2);
    run<43>("mul.lo + 2 lop3", 3);
    return 0;
}
