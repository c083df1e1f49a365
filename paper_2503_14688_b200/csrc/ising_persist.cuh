// ising_persist.cuh -- many sweeps of a cache-resident Ising lattice in ONE cooperative kernel.
//
// SURVEY.md section 8(f) NEXT-4 ("persistent multi-sweep kernels for cache-resident sizes").  For
// L <= 8192 a half-sweep is a few microseconds: the grid does not fill the GPU and the time is
// the latency of one thread's rows plus the launch gap.  Measured gain over back-to-back launches
// (512 sweeps per call): 1358 -> 1528 updates/ns at L = 4096, 340 -> 391 at 2048, 85 -> 99 at 1024,
// 2724 -> 2764 at 8192: the row latency (~1.5 us per row, 2 rows per thread), not the launch,
// dominates.  Here the grid is launched once (cudaLaunchCooperativeKernel, every block resident), loops over the
// sweeps and colours itself and separates the half-sweeps with a grid-wide barrier; the lattice
// stays in L2.  What is computed is exactly what n launches of ising_march_kernel compute: the
// same march_thread() (or, for the smallest lattices, row_thread()) runs, with the per-half-sweep arguments (sweep index, colour, folded
// Philox constants, thresholds) rebuilt in shared memory by one thread per block from a
// per-sweep table the host uploads.
#pragma once
#include <cooperative_groups.h>

#include "ising_march.cuh"

namespace lat {

struct SweepParams {          // what changes from sweep to sweep (built on the host, fp64 -> u32)
    unsigned long long thr4, thr8;
    uint32_t mask4, mask8;
    uint32_t pcase[8];
};

#ifdef __CUDACC__
template <bool EDGE, bool ONE_ROW>
__global__ void __launch_bounds__(256) ising_persist_kernel(const IsingMarchArgs a0, uint32_t *buf0,
                                                            uint32_t *buf1, const SweepParams *sp,
                                                            uint32_t n_sweeps)
{
    namespace cg = cooperative_groups;
    cg::grid_group grid = cg::this_grid();
    __shared__ uint4 s_q[8][TIE_Q_SLOTS];
    __shared__ IsingMarchArgs a;                 // the current half-sweep's arguments
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const uint32_t stride = gridDim.x * 256u;

    if (threadIdx.x == 0) a = a0;
    SweepParams p = sp[0];                       // thread 0 uses it; the next one is prefetched
    for (uint32_t s = 0; s < n_sweeps; ++s) {
        for (uint32_t colour = 0; colour < 2; ++colour) {
            if (threadIdx.x == 0) {
                if (colour == 0) {
                    a.thr4 = p.thr4; a.thr8 = p.thr8; a.mask4 = p.mask4; a.mask8 = p.mask8;
                    for (int k = 0; k < 8; ++k) a.pcase[k] = p.pcase[k];
                    a.t = a0.t + s;
                    if (s + 1 < n_sweeps) p = sp[s + 1];          // in flight during this sweep
                }
                a.colour = colour;
                a.tgt = colour ? buf1 : buf0;
                a.opp = colour ? buf0 : buf1;
                build_plane_fold(a0.K, a.t, colour, TAG_ACC_PLANE, a.F);
            }
            __syncthreads();
            WarpTieQueue<false> queue{a, s_q[warp], lane, 0u};
            for (uint32_t g = blockIdx.x * 256u + threadIdx.x; g - lane < a0.threads; g += stride) {
                if (ONE_ROW) {
                    if (colour == 0) row_thread<0, EDGE>(a, g, queue);
                    else row_thread<1, EDGE>(a, g, queue);
                } else {
                    if (colour == 0) march_thread<0, EDGE, false>(a, g, queue);
                    else march_thread<1, EDGE, false>(a, g, queue);
                }
            }
            queue.drain();
            __threadfence();
            if (gridDim.x == 1) __syncthreads();   // one block: the block barrier is the grid barrier
            else grid.sync();                    // every flip of this colour is visible to the next
        }
    }
}
#endif

}  // namespace lat
