// ising_persist.cuh -- many sweeps of a cache-resident Ising lattice in ONE cooperative kernel.
//
// SURVEY.md section 8(f) NEXT-4 ("persistent multi-sweep kernels for cache-resident sizes").  The grid
// is launched once (cudaLaunchCooperativeKernel, every block resident), loops over the sweeps and
// colours itself and separates the half-sweeps with a grid-wide barrier; the lattice stays in L2.
// What is computed is exactly what n launches of ising_march_kernel compute: the same march_thread()
// (or, for the smallest lattices, row_thread()) runs, with the per-half-sweep arguments (sweep index,
// colour, folded Philox constants, thresholds) rebuilt in shared memory by one thread per block from
// a per-sweep table the host uploads.
//
// Measured (B200, updates/ns, persistent vs two launches per sweep, >= 2 s timed, round 2, grids sized
// so that every block strides over the same number of 256-thread groups):
//   L = 4096: 1677 vs 1366;  8192: 2997 vs 2732;  16384: 4112 vs 4094.
// It wins where a half-sweep is a few microseconds and the launch gap shows; at L = 16384 back-to-back
// launches overlap as well, and the persistent variant pays for its arguments living in registers
// instead of the constant bank (108-127 registers against 63: half the resident warps) and for the
// grid barrier.  lattice_sweep therefore takes this path by itself for L <= 8192; L = 16384 takes it on
// request (lattice_set_persist_blocks), which is what the parity tests of that variant do.  (With a
// grid of simply "all resident blocks" L = 8192 ran at 2090: 444 blocks over 512 groups leave most of
// them idle in the second round.)
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
// PC >= 0: every sweep of the call has the packed plane cases PC (a constant-beta run at one of the
// specialised temperatures, ising_march.cuh): the plane compare is compiled in as in the per-launch kernels.
template <bool EDGE, bool ONE_ROW, int PC = -1>
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
            WarpTieQueue<false> queue{a, s_q[warp], lane, 0u};     // ties (rare) read the shared copy
            // the marching code reads the launch-constant fields (shape, Philox round keys) from the
            // kernel parameters, i.e. as constant-bank operands exactly like ising_march_kernel; only
            // what changes per half-sweep comes from shared memory into registers
            IsingMarchArgs al = a0;
            al.tgt = a.tgt; al.opp = a.opp; al.t = a.t; al.colour = colour;
            al.F.fa = a.F.fa; al.F.fh = a.F.fh; al.F.fl = a.F.fl; al.F.fb[0] = a.F.fb[0];
            if (EDGE) { al.mask4 = a.mask4; al.mask8 = a.mask8; }
            if (PC < 0) {
#pragma unroll
                for (int k = 0; k < 8; ++k) al.pcase[k] = a.pcase[k];
            }
            for (uint32_t g = blockIdx.x * 256u + threadIdx.x; g - lane < a0.threads; g += stride) {
                if (ONE_ROW) {
                    if (colour == 0) row_thread<0, EDGE>(al, g, queue);
                    else row_thread<1, EDGE>(al, g, queue);
                } else {
                    if (colour == 0) march_thread<0, EDGE, false, PC>(al, g, queue);
                    else march_thread<1, EDGE, false, PC>(al, g, queue);
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
