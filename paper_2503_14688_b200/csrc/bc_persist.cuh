// bc_persist.cuh -- many sweeps of a cache-resident Blume-Capel lattice in ONE cooperative kernel.
//
// SURVEY.md section 8(f) NEXT-4 ("persistent multi-sweep kernels for cache-resident sizes"), the
// Blume-Capel counterpart of ising_persist.cuh: BASELINE config 3 (L = 16384, Delta = 0, 64 MiB at
// 2 bits/spin, inside the 126 MB L2) is one launch per lattice_sweep(n) call instead of 2n.  The grid
// is launched once (cudaLaunchCooperativeKernel, every block resident), loops over sweeps and colours
// and separates the half-sweeps with a grid-wide barrier.  What is computed is exactly what 2n
// launches of bc_march_kernel compute: the same bc_march_thread() runs, with the per-half-sweep
// arguments (sweep index, colour, folded Philox constants, threshold truth tables) rebuilt in shared
// memory by one thread per block from a per-sweep table the host uploads.  Threshold tables of the
// Delta = 0 structure only (bc_march.cuh); any other table keeps the per-launch path.
#pragma once
#include <cooperative_groups.h>

#include "bc_march.cuh"

namespace lat {

struct BCSweepParams {        // what changes from sweep to sweep (built on the host from beta)
    uint32_t lut[8];
    uint32_t lut_always;
    uint32_t pad;
    unsigned long long thr[8];
};

#ifdef __CUDACC__
// What a thread of the persistent kernel marches with: the launch-constant fields (lattice shape,
// Philox round keys) stay kernel parameters, i.e. constant-bank operands exactly as in
// bc_march_kernel; only what changes per half-sweep is read from shared memory into registers, and
// the per-plane truth tables are read from shared memory when they are needed.
struct BCPersistArgs : BCMarchArgs {
    const uint32_t *lut_s;
    __device__ __forceinline__ uint32_t lut_k(int k) const { return lut_s[k]; }
};

__global__ void __launch_bounds__(256, 2) bc_persist_kernel(const BCMarchArgs a0, uint32_t *buf, const BCSweepParams *sp,
                                                            uint32_t n_sweeps)
{
    namespace cg = cooperative_groups;
    cg::grid_group grid = cg::this_grid();
    __shared__ uint4 s_q[8][2 * TIE_Q_SLOTS];
    __shared__ BCMarchArgs a;                    // the current half-sweep's arguments
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const uint32_t stride = gridDim.x * 256u;
    const unsigned long long pw = (unsigned long long)a0.L * a0.wpr;      // words per plane

    if (threadIdx.x == 0) a = a0;
    for (uint32_t s = 0; s < n_sweeps; ++s) {
        for (uint32_t colour = 0; colour < 2; ++colour) {
            if (threadIdx.x == 0) {
                if (colour == 0) {
                    const BCSweepParams p = sp[s];
                    for (int k = 0; k < 8; ++k) { a.lut[k] = p.lut[k]; a.thr[k] = p.thr[k]; }
                    a.lut_always = p.lut_always;
                    a.t = a0.t + s;
                }
                a.colour = colour;
                a.tnz = buf + (size_t)(2u * colour) * pw;
                a.tsg = buf + (size_t)(2u * colour + 1u) * pw;
                a.onz = buf + (size_t)(2u * (1u - colour)) * pw;
                a.osg = buf + (size_t)(2u * (1u - colour) + 1u) * pw;
                build_plane_fold(a0.K, a.t, colour, TAG_ACC_PLANE, a.F);
                a.fbp = (colour | (TAG_PROP_PLANE << 8)) ^ a0.K.k1[0];
            }
            __syncthreads();
            BCTieQueue<false> queue{a, s_q[warp], lane, 0u};       // ties (rare) read the shared copy
            BCPersistArgs al;
            static_cast<BCMarchArgs &>(al) = a0;
            al.tnz = a.tnz; al.tsg = a.tsg; al.onz = a.onz; al.osg = a.osg;
            al.t = a.t; al.colour = colour;
            al.F.fa = a.F.fa; al.F.fh = a.F.fh; al.F.fl = a.F.fl; al.F.fb[0] = a.F.fb[0];
            al.fbp = a.fbp;
            al.lut_always = a.lut_always;
            al.lut_s = a.lut;
            for (uint32_t g = blockIdx.x * 256u + threadIdx.x; g - lane < a0.threads; g += stride) {
                if (colour == 0) bc_march_thread<0, false, false>(al, g, queue);
                else bc_march_thread<1, false, false>(al, g, queue);
            }
            queue.drain();
            __threadfence();
            if (gridDim.x == 1) __syncthreads();   // one block: the block barrier is the grid barrier
            else grid.sync();                    // every move of this colour is visible to the next
        }
    }
}
#endif

}  // namespace lat
