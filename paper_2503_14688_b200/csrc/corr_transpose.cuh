// corr_transpose.cuh -- transposed copy of a band of lattice rows, for the x-axis correlations.
//
// S_x(r) = sum_i sum_j s(i,j) s(i,j+r) (Eq. 2) contracts over the ROWS i for every
// pair of columns.  Read from the lattice as it is stored, that is 8 bytes per row and colour for a
// 128-column tile: at L = 2^20 (rows 64 KiB apart) every such read is its own DRAM burst and the
// tiles of neighbouring CTAs do not meet in L2 (profiles/r2_launches_default.md: 15-18 TB for 1.4 TB
// of distinct data; the x axis is what that traffic makes it).  So the x axis runs on a TRANSPOSED copy
// instead, band by band: a band of B rows (B <= 65536) of the L columns is written as a lattice T of L
// rows and B columns in the same sublattice packing, T(j, i) = s(i0 + i, j), and the y-axis kernel --
// contraction along a stored row, 16 contiguous bytes per lane and two steps -- is run on T: its row
// Gram band IS the band's contribution to S_x.  The bands' contributions add up.
//
// Packing: word W of row i of colour c holds p = 32 W + beta, column
// j = 2 p + ((i + c) & 1).  A site keeps its colour under transposition (both are (i + j) & 1 for an
// even first row i0), so with i = 64 w + 2 b + pi (band-local, pi = row parity) and sigma = (pi + c) & 1
//     T[c][j = 64 W + 2 beta + sigma][w] bit b  =  O[c][i0 + 64 w + 2 b + pi][W] bit beta :
// a 32 x 32 bit-block transpose per (c, pi, w, W).  A block of 8 warps takes 8 consecutive w and 32
// consecutive W: lane l of warp k loads word W0 + l of its 32 rows (coalesced), transposes the 32 words
// it then holds IN REGISTERS (five butterfly stages), and the block writes 32 contiguous bytes (8 words
// w) of 1024 rows of T through shared memory.
#pragma once
#include <stdint.h>

namespace lat {

struct TransposeArgs {
    const uint32_t *src;             // the lattice buffer: [plane][rows][wpr]
    uint32_t *dst;                   // T: [plane][L][B / 64]
    uint32_t rows, wpr;              // rows per plane and words per row of the lattice
    uint32_t i0;                     // first row of the band (even)
    uint32_t B;                      // rows in the band: a multiple of 512
    uint32_t L;                      // columns of the lattice = rows of T; wpr % 32 == 0
    uint32_t bc;                     // 1: planes are [colour][nz, sg] (Blume-Capel), 0: [colour]
};

#ifdef __CUDACC__
// out[beta] bit b = in[b] bit beta, in place
__device__ __forceinline__ void bit_transpose32(uint32_t (&a)[32])
{
    uint32_t m = 0x0000ffffu;
#pragma unroll
    for (int j = 16; j != 0; j >>= 1, m ^= m << j) {
#pragma unroll
        for (int k = 0; k < 32; k = (k + j + 1) & ~j) {
            const uint32_t t = ((a[k] >> j) ^ a[k + j]) & m;
            a[k] ^= t << j;
            a[k + j] ^= t;
        }
    }
}

// grid: (wpr / 32, B / 512, planes * 2), 256 threads
__global__ void __launch_bounds__(256) band_transpose_kernel(const TransposeArgs a)
{
    __shared__ uint32_t S[1024 * 9];                 // [beta][l][k], rows padded to 9 words
    const uint32_t lane = threadIdx.x & 31u, k = threadIdx.x >> 5;
    const uint32_t q = blockIdx.z >> 1, pi = blockIdx.z & 1u;            // plane, row parity
    const uint32_t c = a.bc ? q >> 1 : q;                                // colour of the plane
    const uint32_t w = blockIdx.y * 8u + k, W = blockIdx.x * 32u + lane;
    const uint32_t wprT = a.B >> 6;
    const uint32_t *sp = a.src + (size_t)q * a.rows * a.wpr + (size_t)(a.i0 + 64u * w + pi) * a.wpr + W;
    uint32_t r[32];
#pragma unroll
    for (int b = 0; b < 32; ++b) r[b] = sp[(size_t)(2 * b) * a.wpr];
    bit_transpose32(r);
#pragma unroll
    for (int beta = 0; beta < 32; ++beta) S[((uint32_t)beta * 32u + lane) * 9u + k] = r[beta];
    __syncthreads();
    const uint32_t sigma = (pi + c) & 1u;
    uint32_t *dp = a.dst + (size_t)q * a.L * wprT + blockIdx.y * 8u;
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        const uint32_t row = threadIdx.x + 256u * (uint32_t)e;           // beta * 32 + l
        const uint32_t beta = row >> 5, l = row & 31u;
        const uint32_t j = 64u * (blockIdx.x * 32u + l) + 2u * beta + sigma;
        const uint32_t *s = S + row * 9u;
        uint4 *d = reinterpret_cast<uint4 *>(dp + (size_t)j * wprT);
        d[0] = make_uint4(s[0], s[1], s[2], s[3]);
        d[1] = make_uint4(s[4], s[5], s[6], s[7]);
    }
}
#endif

}  // namespace lat
