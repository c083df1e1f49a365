// ubench.cuh -- the integer-dispatch micro-benchmark behind bench.py's "alu" roofline peak.
//
// The half-sweep kernels are bound by one 16-lane dispatch per SM sub-partition that LOP3-class
// instructions (ALU pipe) and the 32x32->64 multiplies of Philox (IMAD.WIDE / IMAD.HI) share
// (DESIGN.md section 6).  Instead of quoting a nominal 64 lanes/clk/SM, bench.py runs this kernel
// in the same process and uses the MEASURED thread-instructions per clock per SM as the peak.
// Cycles come from clock64() inside the kernel, so the figure does not depend on the SM clock:
// per SM, the span from the earliest start to the latest end over ALL warps that ran on it (the
// warp schedulers favour old warps, so one warp's own span understates the time), and the
// instructions of the blocks that actually landed on that SM.
//   mode 0: independent LOP3 chains                       (the ALU pipe alone)
//   mode 1: 1 mul.wide.u32 + 1 LOP3 per step              (the Philox round mix, 1 : 1)
//   mode 2: 1 mul.wide.u32 + 3 LOP3 per step              (the half-sweep's overall mix, ~1 : 3)
//   mode 3: POPC (+ an uncounted IADD) per step           (the measurement kernels' popcount pipe)
#pragma once
#include <stdint.h>

namespace lat {

constexpr int UB_ITER = 4096, UB_CHAINS = 8, UB_BLOCKS_PER_SM = 4, UB_MAX_SM = 512;

template <int MODE>
__global__ void __launch_bounds__(256) ubench_kernel(uint32_t *out, uint32_t seed, unsigned long long *clk)
{
    // clk[3 * smid + {0, 1, 2}] = earliest start, latest end, number of blocks on that SM
    uint32_t smid;
    asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
    uint32_t x[UB_CHAINS], y[UB_CHAINS];
#pragma unroll
    for (int i = 0; i < UB_CHAINS; ++i) { x[i] = seed + threadIdx.x * 7u + i; y[i] = seed ^ (i * 0x9E3779B9u); }
    const unsigned long long t0 = clock64();
    for (int it = 0; it < UB_ITER; ++it) {
#pragma unroll
        for (int i = 0; i < UB_CHAINS; ++i) {
            if (MODE == 0) {
                asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(x[i]) : "r"(y[i]), "r"(seed));
            } else if (MODE == 1 || MODE == 2) {
                uint32_t lo, hi;
                asm volatile("{.reg .u64 p; mul.wide.u32 p, %2, 0xD2511F53; mov.b64 {%0,%1}, p;}"
                             : "=r"(lo), "=r"(hi) : "r"(x[i]));
                asm volatile("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(x[i]) : "r"(hi), "r"(y[i]), "r"(seed));
                if (MODE == 2) {
                    asm volatile("lop3.b32 %0, %1, %2, %3, 0xe8;" : "=r"(y[i]) : "r"(lo), "r"(y[i]), "r"(x[i]));
                    asm volatile("lop3.b32 %0, %1, %2, %3, 0x1e;" : "=r"(x[i]) : "r"(lo), "r"(y[i]), "r"(x[i]));
                } else {
                    y[i] = lo;
                }
            } else {
                x[i] += __popc(x[i]);
            }
        }
    }
    const unsigned long long t1 = clock64();
    uint32_t s = 0;
#pragma unroll
    for (int i = 0; i < UB_CHAINS; ++i) s ^= x[i] ^ y[i];
    out[blockIdx.x * blockDim.x + threadIdx.x] = s;
    if ((threadIdx.x & 31u) == 0 && smid < UB_MAX_SM) {
        atomicMin(clk + 3 * smid, t0);
        atomicMax(clk + 3 * smid + 1, t1);
        if (threadIdx.x == 0) atomicAdd(clk + 3 * smid + 2, 1ull);
    }
}

// thread-instructions of the counted classes per step of one chain
__host__ inline double ubench_instr_per_step(int mode)
{
    return mode == 0 ? 1.0 : mode == 1 ? 2.0 : mode == 2 ? 4.0 : 1.0;     // mode 3 counts the POPC only
}

}  // namespace lat
