// measure.cuh -- exact integer reductions: M, Q and the axis correlation sums S_x(r), S_y(r).
//
// Paper: C(r;t), Eq. 2, measured along the lattice axes; E from r = 1, Eq. 3
// (PAPER.md:47-50).  BASELINE.json north_star (c): XOR/popcount of shifted rows, warp-shuffle
// reductions, exact 64-bit integer counts.
//
// With the sublattice packing the partner of site (i, p) of colour c at distance r is
//   y axis: row i+r, same p, colour c ^ (r & 1)
//   x axis: row i,  r = 2d   -> colour c,     p + d
//                   r = 2d+1 -> colour c ^ 1, p + d + ((i + c) & 1)
// (all periodic), i.e. a whole word of partners is one funnel shift of two partner words.
// Ising: s s' = 1 - 2 (bit ^ bit'), so S(r) = N - 2 popc(xor).  Blume-Capel:
// s s' = +1 / -1 / 0 -> S(r) = popc(nz & nz') - 2 popc(nz & nz' & (sg ^ sg')).
//
// Counters (device, unsigned 64-bit, zeroed by the host before launch):
//   cnt[0], cnt[1]                         Ising: #(+1), unused      BC: #(+1), #(-1)
//   cnt[2 + 2*(axis*r_max + r-1) + {0,1}]  Ising: popc(xor), unused  BC: #both nonzero, #opposite
#pragma once
#include <stdint.h>

namespace lat {

struct MeasArgs {
    const uint32_t *buf;
    uint32_t L, wpr, model;          // model: 0 Ising, 1 Blume-Capel
    uint32_t i0, n_rows;             // base rows i0 .. i0+n_rows-1
    uint32_t r_max;
    uint32_t r0;                     // this launch covers r = r0+1 .. r0+gridDim.y
    unsigned long long *cnt;
};

__device__ __forceinline__ unsigned long long warp_sum(unsigned long long v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// block-wide sum of two counters, then one atomic each from thread 0
__device__ __forceinline__ void block_add2(unsigned long long a, unsigned long long b,
                                           unsigned long long *dst)
{
    __shared__ unsigned long long sh[2][8];
    a = warp_sum(a);
    b = warp_sum(b);
    const uint32_t wid = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) { sh[0][wid] = a; sh[1][wid] = b; }
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long sa = 0, sb = 0;
        for (uint32_t w = 0; w < (blockDim.x >> 5); ++w) { sa += sh[0][w]; sb += sh[1][w]; }
        if (sa) atomicAdd(dst, sa);
        if (sb) atomicAdd(dst + 1, sb);
    }
}

// word k of (colour, plane) in row i
__device__ __forceinline__ const uint32_t *plane_ptr(const MeasArgs &a, uint32_t colour, uint32_t plane)
{
    const size_t pw = (size_t)a.L * a.wpr;
    return a.model == 0 ? a.buf + (size_t)colour * pw : a.buf + (size_t)(2 * colour + plane) * pw;
}

__global__ void __launch_bounds__(256) measure_mq_kernel(const MeasArgs a)
{
    const unsigned long long total = 2ull * a.n_rows * a.wpr;
    unsigned long long c0 = 0, c1 = 0;
    for (unsigned long long g = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; g < total;
         g += (unsigned long long)gridDim.x * blockDim.x) {
        const uint32_t colour = (uint32_t)(g / ((unsigned long long)a.n_rows * a.wpr));
        const unsigned long long rem = g % ((unsigned long long)a.n_rows * a.wpr);
        const size_t off = ((size_t)a.i0 * a.wpr) + rem;
        if (a.model == 0) {
            c0 += __popc(plane_ptr(a, colour, 0)[off]);
        } else {
            const uint32_t nz = plane_ptr(a, colour, 0)[off], sg = plane_ptr(a, colour, 1)[off];
            c0 += __popc(nz & ~sg);
            c1 += __popc(nz & sg);
        }
    }
    block_add2(c0, c1, a.cnt);
}

// grid = (blocks_x, n_r, 2): r = r0 + blockIdx.y + 1, blockIdx.z = axis (0 = x, 1 = y)
__global__ void __launch_bounds__(256) measure_corr_kernel(const MeasArgs a)
{
    const uint32_t r = a.r0 + blockIdx.y + 1, axis = blockIdx.z;
    const uint32_t L = a.L, wpr = a.wpr;
    const unsigned long long per_colour = (unsigned long long)a.n_rows * wpr;
    const unsigned long long total = 2ull * per_colour;
    unsigned long long c0 = 0, c1 = 0;
    for (unsigned long long g = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; g < total;
         g += (unsigned long long)gridDim.x * blockDim.x) {
        const uint32_t colour = (uint32_t)(g / per_colour);
        const unsigned long long rem = g % per_colour;
        const uint32_t i = a.i0 + (uint32_t)(rem / wpr), k = (uint32_t)(rem % wpr);
        uint32_t c2, i2, k1, k2, bo;
        if (axis == 1) {
            c2 = colour ^ (r & 1u);
            i2 = (uint32_t)(((unsigned long long)i + r) % L);
            k1 = k; k2 = k; bo = 0;
        } else {
            c2 = colour ^ (r & 1u);
            i2 = i;
            const uint32_t s = (r >> 1) + ((r & 1u) ? ((i + colour) & 1u) : 0u);
            k1 = (k + (s >> 5)) % wpr;
            k2 = (k1 + 1 == wpr) ? 0 : k1 + 1;
            bo = s & 31u;
        }
        const size_t o0 = (size_t)i * wpr + k, o1 = (size_t)i2 * wpr + k1, o2 = (size_t)i2 * wpr + k2;
        if (a.model == 0) {
            const uint32_t *w0 = plane_ptr(a, colour, 0), *w1 = plane_ptr(a, c2, 0);
            const uint32_t partner = __funnelshift_r(w1[o1], w1[o2], bo);
            c0 += __popc(w0[o0] ^ partner);
        } else {
            const uint32_t *n0 = plane_ptr(a, colour, 0), *s0 = plane_ptr(a, colour, 1);
            const uint32_t *n1 = plane_ptr(a, c2, 0), *s1 = plane_ptr(a, c2, 1);
            const uint32_t pn = __funnelshift_r(n1[o1], n1[o2], bo);
            const uint32_t ps = __funnelshift_r(s1[o1], s1[o2], bo);
            const uint32_t both = n0[o0] & pn;
            c0 += __popc(both);
            c1 += __popc(both & (s0[o0] ^ ps));
        }
    }
    block_add2(c0, c1, a.cnt + 2 + 2 * ((size_t)axis * a.r_max + (r - 1)));
}

// ---- unpacked windows (tests, windowed replay, checkpoints) --------------------------------
struct WindowArgs {
    uint32_t *buf;
    uint32_t L, wpr, model;
    uint32_t i0, j0, h, w;
    int8_t *spins;                   // device, row-major h x w
};

__device__ __forceinline__ void site_addr(const WindowArgs &a, uint32_t i, uint32_t j,
                                          size_t &word, uint32_t &bit, uint32_t &colour)
{
    colour = (i + j) & 1u;
    const uint32_t p = j >> 1;
    word = (size_t)i * a.wpr + (p >> 5);
    bit = p & 31u;
}

__global__ void __launch_bounds__(256) get_spins_kernel(const WindowArgs a)
{
    const unsigned long long g = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= (unsigned long long)a.h * a.w) return;
    const uint32_t i = (uint32_t)((a.i0 + g / a.w) % a.L), j = (uint32_t)((a.j0 + g % a.w) % a.L);
    size_t word; uint32_t bit, colour;
    site_addr(a, i, j, word, bit, colour);
    const size_t pw = (size_t)a.L * a.wpr;
    if (a.model == 0) {
        a.spins[g] = ((a.buf[(size_t)colour * pw + word] >> bit) & 1u) ? 1 : -1;
    } else {
        const uint32_t nz = (a.buf[(size_t)(2 * colour) * pw + word] >> bit) & 1u;
        const uint32_t sg = (a.buf[(size_t)(2 * colour + 1) * pw + word] >> bit) & 1u;
        a.spins[g] = nz ? (sg ? -1 : 1) : 0;
    }
}

__global__ void __launch_bounds__(256) set_spins_kernel(const WindowArgs a)
{
    const unsigned long long g = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= (unsigned long long)a.h * a.w) return;
    const uint32_t i = (uint32_t)((a.i0 + g / a.w) % a.L), j = (uint32_t)((a.j0 + g % a.w) % a.L);
    size_t word; uint32_t bit, colour;
    site_addr(a, i, j, word, bit, colour);
    const size_t pw = (size_t)a.L * a.wpr;
    const int s = a.spins[g];
    const uint32_t m = 1u << bit;
    if (a.model == 0) {
        uint32_t *p = a.buf + (size_t)colour * pw + word;
        if (s > 0) atomicOr(p, m); else atomicAnd(p, ~m);
    } else {
        uint32_t *pn = a.buf + (size_t)(2 * colour) * pw + word;
        uint32_t *ps = a.buf + (size_t)(2 * colour + 1) * pw + word;
        if (s != 0) atomicOr(pn, m); else atomicAnd(pn, ~m);
        if (s < 0) atomicOr(ps, m); else atomicAnd(ps, ~m);
    }
}

}  // namespace lat
