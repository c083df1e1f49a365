// slab_flags.cuh -- device-side ordering of the colours between row slabs.
//
// A slab's half-sweep h = 2 t + colour + 1 may start when both neighbours have finished half-sweep
// h - 1: their mirrors of the other colour have landed in this slab's halo rows, and they no longer
// read the halo rows this half-sweep is about to overwrite in THEIR buffers.  Each slab publishes the
// number of half-sweeps it has completed in a 64-bit word of its own buffer; the neighbours read that
// word through their peer / IPC mapping.  With lattice_slab_set_flags every half-sweep launch is
//     slab_wait_kernel (1 thread: spin until both neighbours' words are >= h - 1)
//     the marching kernel (stores its boundary rows into the neighbours' halos)
//     slab_publish_kernel (1 thread: system-scope fence, release store of h)
// in stream order, so a driver can enqueue any number of sweeps without a host barrier per colour.
// The hot kernels are unchanged.  The wait is bounded: a protocol error traps instead of hanging.
// NOT exercised with a wait that actually spins: on one GPU ranks whose kernels wait on one another
// must not be run (B200_PROFILING.md); with all slabs in one stream the words are already there.
#pragma once
#include <stdint.h>

namespace lat {

#ifdef __CUDACC__
__global__ void slab_wait_kernel(const unsigned long long *up, const unsigned long long *dn, unsigned long long target)
{
    const long long t0 = clock64();
    for (;;) {
        unsigned long long a, b;
        asm volatile("ld.acquire.sys.global.u64 %0, [%1];" : "=l"(a) : "l"(up) : "memory");
        asm volatile("ld.acquire.sys.global.u64 %0, [%1];" : "=l"(b) : "l"(dn) : "memory");
        if (a >= target && b >= target) return;
        if (clock64() - t0 > (1ll << 35)) __trap();          // ~17 s
        __nanosleep(200);
    }
}

__global__ void slab_publish_kernel(unsigned long long *mine, unsigned long long value)
{
    __threadfence_system();                                   // after every store of the kernels before this one
    asm volatile("st.release.sys.global.u64 [%0], %1;" ::"l"(mine), "l"(value) : "memory");
}
#endif

}  // namespace lat
