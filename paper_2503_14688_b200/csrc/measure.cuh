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
    uint32_t axis0;                  // axis of blockIdx.z == 0 (0 = x, 1 = y)
    unsigned long long *cnt;
    // batch of replicas: blockIdx.x = replica * bpr + block; replica k reads buf + k * rep_words
    // and adds to cnt + k * cnt_stride (bpr = gridDim.x, strides 0 for a single lattice)
    uint32_t bpr;
    unsigned long long rep_words, cnt_stride;
    // sparse list of r (lattice_measure_list): when non-null, blockIdx.y indexes rlist (device) and
    // the counters, r_max being the length of the list
    const uint32_t *rlist;
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

// word k of (colour, plane) in row i of the lattice that starts at buf
__device__ __forceinline__ const uint32_t *plane_ptr(const MeasArgs &a, const uint32_t *buf, uint32_t colour,
                                                     uint32_t plane)
{
    const size_t pw = (size_t)a.L * a.wpr;
    return a.model == 0 ? buf + (size_t)colour * pw : buf + (size_t)(2 * colour + plane) * pw;
}

__global__ void __launch_bounds__(256) measure_mq_kernel(const MeasArgs a)
{
    const uint32_t rep = blockIdx.x / a.bpr, bx = blockIdx.x - rep * a.bpr;
    const uint32_t *buf = a.buf + rep * a.rep_words;
    // the base rows of one colour (and plane) are one contiguous range of n_rows * wpr words
    const unsigned long long n = (unsigned long long)a.n_rows * a.wpr, stride = (unsigned long long)a.bpr * blockDim.x;
    const size_t off = (size_t)a.i0 * a.wpr;
    unsigned long long c0 = 0, c1 = 0;
    for (uint32_t colour = 0; colour < 2; ++colour) {
        const uint32_t *p0 = plane_ptr(a, buf, colour, 0) + off, *p1 = plane_ptr(a, buf, colour, 1) + off;
        if ((a.wpr & 3u) == 0) {                 // 16-byte loads (rows are whole 128-bit runs)
            const uint4 *q0 = reinterpret_cast<const uint4 *>(p0), *q1 = reinterpret_cast<const uint4 *>(p1);
            for (unsigned long long g = (unsigned long long)bx * blockDim.x + threadIdx.x; g < n / 4; g += stride) {
                const uint4 nz = q0[g];
                if (a.model == 0) {
                    c0 += __popc(nz.x) + __popc(nz.y) + __popc(nz.z) + __popc(nz.w);
                } else {
                    const uint4 sg = q1[g];
                    c0 += __popc(nz.x & ~sg.x) + __popc(nz.y & ~sg.y) + __popc(nz.z & ~sg.z) + __popc(nz.w & ~sg.w);
                    c1 += __popc(nz.x & sg.x) + __popc(nz.y & sg.y) + __popc(nz.z & sg.z) + __popc(nz.w & sg.w);
                }
            }
        } else {
            for (unsigned long long g = (unsigned long long)bx * blockDim.x + threadIdx.x; g < n; g += stride) {
                if (a.model == 0) {
                    c0 += __popc(p0[g]);
                } else {
                    const uint32_t nz = p0[g], sg = p1[g];
                    c0 += __popc(nz & ~sg);
                    c1 += __popc(nz & sg);
                }
            }
        }
    }
    block_add2(c0, c1, a.cnt + rep * a.cnt_stride);
}

// grid = (replicas * bpr, n_r, n_axes): r = r0 + blockIdx.y + 1, axis = axis0 + blockIdx.z (0 = x, 1 = y)
__global__ void __launch_bounds__(256) measure_corr_kernel(const MeasArgs a)
{
    const uint32_t rep = blockIdx.x / a.bpr, bx = blockIdx.x - rep * a.bpr;
    const uint32_t *buf = a.buf + rep * a.rep_words;
    const uint32_t ridx = a.r0 + blockIdx.y, axis = a.axis0 + blockIdx.z;
    const uint32_t r = a.rlist ? a.rlist[ridx] : ridx + 1;
    const uint32_t L = a.L, wpr = a.wpr;
    const unsigned long long per_colour = (unsigned long long)a.n_rows * wpr;
    const unsigned long long total = 2ull * per_colour;
    unsigned long long c0 = 0, c1 = 0;
    for (unsigned long long g = (unsigned long long)bx * blockDim.x + threadIdx.x; g < total;
         g += (unsigned long long)a.bpr * blockDim.x) {
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
            const uint32_t *w0 = plane_ptr(a, buf, colour, 0), *w1 = plane_ptr(a, buf, c2, 0);
            const uint32_t partner = __funnelshift_r(w1[o1], w1[o2], bo);
            c0 += __popc(w0[o0] ^ partner);
        } else {
            const uint32_t *n0 = plane_ptr(a, buf, colour, 0), *s0 = plane_ptr(a, buf, colour, 1);
            const uint32_t *n1 = plane_ptr(a, buf, c2, 0), *s1 = plane_ptr(a, buf, c2, 1);
            const uint32_t pn = __funnelshift_r(n1[o1], n1[o2], bo);
            const uint32_t ps = __funnelshift_r(s1[o1], s1[o2], bo);
            const uint32_t both = n0[o0] & pn;
            c0 += __popc(both);
            c1 += __popc(both & (s0[o0] ^ ps));
        }
    }
    block_add2(c0, c1, a.cnt + rep * a.cnt_stride + 2 + 2 * ((size_t)axis * a.r_max + ridx));
}

// ---- row-blocked kernels (the production measurement path) ----------------------------------
//
// The generic kernel above re-reads the lattice once per (r, axis) and pays one POPC per word.
// The two kernels below keep 16 base words per thread in registers, slide the partner words
// past them (one new row, or one more bit of funnel shift, per step of r) and reduce the 16
// XOR words of one r with a carry-save adder tree (30 LOP3) before 5 POPCs, so the cost per
// (word, r) is ~3 (y axis) to ~4 (x axis) ALU instructions and the lattice is read from DRAM
// about once per chunk of MEAS_RC values of r.  Per-r counts are summed over the warp with
// REDUX and accumulated in shared memory; one 64-bit atomic per (block, r) reaches global
// memory.  blockIdx.y selects the chunk r = r0+1 .. r0+MEAS_RC, r0 = MEAS_RC * blockIdx.y.
constexpr int MEAS_NB = 16;      // base words per thread (rows for the y axis, words for the x axis)
constexpr int MEAS_RC = 64;      // values of r per chunk (even)

// population count of 16 words as 5 bit-sliced words of weight 1, 2, 4, 8, 16
// (explicit LOP3 truth tables: left to itself the compiler regroups the XOR + majority tree and
// ends up with ~30 % more LOP3 than the 2 per adder written here)
__device__ __forceinline__ void csa(uint32_t a, uint32_t b, uint32_t c, uint32_t &s, uint32_t &cy)
{
    asm("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(s) : "r"(a), "r"(b), "r"(c));      // a ^ b ^ c
    asm("lop3.b32 %0, %1, %2, %3, 0xE8;" : "=r"(cy) : "r"(a), "r"(b), "r"(c));     // majority
}
__device__ __forceinline__ uint32_t weighted_popc16(const uint32_t (&x)[16])
{
    uint32_t s[4], t[8], u[4], v[2];
    // weight 1: 16 -> 1 (+ 8 of weight 2)
    uint32_t a0, a1, a2, a3, a4, a5, a6;
    csa(x[0], x[1], x[2], a0, t[0]);
    csa(x[3], x[4], x[5], a1, t[1]);
    csa(x[6], x[7], x[8], a2, t[2]);
    csa(x[9], x[10], x[11], a3, t[3]);
    csa(x[12], x[13], x[14], a4, t[4]);
    csa(a0, a1, a2, a5, t[5]);
    csa(a3, a4, x[15], a6, t[6]);
    const uint32_t w1 = a5 ^ a6;
    t[7] = a5 & a6;
    // weight 2: 8 -> 1 (+ 4 of weight 4)
    csa(t[0], t[1], t[2], s[0], u[0]);
    csa(t[3], t[4], t[5], s[1], u[1]);
    csa(s[0], s[1], t[6], s[2], u[2]);
    const uint32_t w2 = s[2] ^ t[7];
    u[3] = s[2] & t[7];
    // weight 4: 4 -> 1 (+ 2 of weight 8)
    csa(u[0], u[1], u[2], s[3], v[0]);
    const uint32_t w4 = s[3] ^ u[3];
    v[1] = s[3] & u[3];
    // weight 8: 2 -> 1 (+ 1 of weight 16)
    const uint32_t w8 = v[0] ^ v[1];
    const uint32_t w16 = v[0] & v[1];
    return __popc(w1) + 2u * __popc(w2) + 4u * __popc(w4) + 8u * __popc(w8) + 16u * __popc(w16);
}

struct MeasBlkArgs {
    const uint32_t *buf;
    uint32_t L, wpr;
    uint32_t i0;                     // first base row
    uint32_t n;                      // y kernel: number of 16-row blocks; x kernel: number of rows
    uint32_t r_max;
    unsigned long long *cnt;         // same layout as MeasArgs::cnt
};

template <int MODEL, class Args>
__device__ __forceinline__ const uint32_t *blk_plane(const Args &a, uint32_t colour, uint32_t plane)
{
    const size_t pw = (size_t)a.L * a.wpr;
    return MODEL == 0 ? a.buf + (size_t)colour * pw : a.buf + (size_t)(2 * colour + plane) * pw;
}

// shared-memory accumulation of one r: counts summed over the live lanes of the warp
__device__ __forceinline__ void add_r(unsigned int (*s_cnt)[2], uint32_t slot, uint32_t mask, uint32_t leader,
                                      uint32_t lane, uint32_t c0, uint32_t c1, bool two)
{
    const uint32_t v0 = __reduce_add_sync(mask, c0);
    const uint32_t v1 = two ? __reduce_add_sync(mask, c1) : 0u;
    if (lane == leader) {
        atomicAdd(&s_cnt[slot][0], v0);
        if (two) atomicAdd(&s_cnt[slot][1], v1);
    }
}

// y axis (and M, Q in chunk 0): thread = (colour c, 16-row block, word column k)
template <int MODEL>
__global__ void __launch_bounds__(128) measure_y_kernel(const MeasBlkArgs a)
{
    __shared__ unsigned int s_cnt[MEAS_RC][2];
    __shared__ unsigned long long s_mq[2];
    for (uint32_t t = threadIdx.x; t < MEAS_RC * 2; t += blockDim.x) (&s_cnt[0][0])[t] = 0;
    if (threadIdx.x < 2) s_mq[threadIdx.x] = 0;
    __syncthreads();
    const uint32_t r0 = blockIdx.y * MEAS_RC;
    const uint32_t g = blockIdx.x * blockDim.x + threadIdx.x;
    const uint32_t per_colour = a.n * a.wpr;
    const bool live = g < 2u * per_colour;
    const uint32_t mask = __ballot_sync(0xffffffffu, live);
    const uint32_t lane = threadIdx.x & 31u;
    if (live) {
        const uint32_t leader = __ffs(mask) - 1;
        const uint32_t c = g >= per_colour ? 1u : 0u;
        const uint32_t rem = g - c * per_colour;
        const uint32_t rb = rem / a.wpr, k = rem - rb * a.wpr;
        const uint32_t ib0 = a.i0 + MEAS_NB * rb;
        const unsigned long long plane_words = (unsigned long long)a.L * a.wpr;
        const uint32_t *bp0 = blk_plane<MODEL>(a, c, 0), *bp1 = blk_plane<MODEL>(a, c, 1);
        const uint32_t *op0 = blk_plane<MODEL>(a, c ^ 1u, 0), *op1 = blk_plane<MODEL>(a, c ^ 1u, 1);

        uint32_t B0[MEAS_NB], B1[MEAS_NB];          // base words (Ising: spins; BC: nz, sg)
        {
            unsigned long long o = (unsigned long long)ib0 * a.wpr + k;
#pragma unroll
            for (int j = 0; j < MEAS_NB; ++j) {
                B0[j] = bp0[o];
                B1[j] = MODEL ? bp1[o] : 0u;
                o += a.wpr;
            }
        }
        if (blockIdx.y == 0) {                       // M and Q of the base rows
            uint32_t m0 = 0, m1 = 0;
#pragma unroll
            for (int j = 0; j < MEAS_NB; ++j) {
                if (MODEL == 0) m0 += __popc(B0[j]);
                else { m0 += __popc(B0[j] & ~B1[j]); m1 += __popc(B0[j] & B1[j]); }
            }
            const uint32_t v0 = __reduce_add_sync(mask, m0);
            const uint32_t v1 = MODEL ? __reduce_add_sync(mask, m1) : 0u;
            if (lane == leader) {
                atomicAdd(&s_mq[0], (unsigned long long)v0);
                if (MODEL) atomicAdd(&s_mq[1], (unsigned long long)v1);
            }
        }
        // partner windows: odd r -> opposite colour rows ib0 + r + j, even r -> same colour.
        // WO[x & 15] holds opposite-colour row ib0 + r0 + 1 + x, WS[x & 15] same-colour row
        // ib0 + r0 + 2 + x; step m uses x = 2m .. 2m+15 of both.
        uint32_t WO0[MEAS_NB], WO1[MEAS_NB], WS0[MEAS_NB], WS1[MEAS_NB];
        unsigned long long oo = ((unsigned long long)((ib0 + r0 + 1u) % a.L)) * a.wpr + k;
        unsigned long long os = ((unsigned long long)((ib0 + r0 + 2u) % a.L)) * a.wpr + k;
#pragma unroll
        for (int x = 0; x < MEAS_NB; ++x) {
            WO0[x] = op0[oo]; WO1[x] = MODEL ? op1[oo] : 0u;
            WS0[x] = bp0[os]; WS1[x] = MODEL ? bp1[os] : 0u;
            oo += a.wpr; if (oo >= plane_words) oo -= plane_words;
            os += a.wpr; if (os >= plane_words) os -= plane_words;
        }
        for (uint32_t mm = 0; mm < MEAS_RC / 2; mm += 8) {
            if (r0 + 2 * mm + 1 > a.r_max) break;
#pragma unroll
            for (int u = 0; u < 8; ++u) {
                const uint32_t r_odd = r0 + 2 * (mm + u) + 1;
#pragma unroll
                for (int par = 0; par < 2; ++par) {
                    const uint32_t r = r_odd + par;
                    if (r <= a.r_max) {
                        uint32_t X[MEAS_NB], Y[MEAS_NB];
#pragma unroll
                        for (int j = 0; j < MEAS_NB; ++j) {
                            const int sl = (j + 2 * u) & 15;
                            const uint32_t p0 = par ? WS0[sl] : WO0[sl];
                            const uint32_t p1 = par ? WS1[sl] : WO1[sl];
                            if (MODEL == 0) X[j] = B0[j] ^ p0;
                            else { X[j] = B0[j] & p0; Y[j] = X[j] & (B1[j] ^ p1); }
                        }
                        const uint32_t c0 = weighted_popc16(X);
                        const uint32_t c1 = MODEL ? weighted_popc16(Y) : 0u;
                        add_r(s_cnt, r - r0 - 1, mask, leader, lane, c0, c1, MODEL != 0);
                    }
                }
                // slide both windows by two rows: slots (2u)&15 and (2u+1)&15 are free now
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                    const int sl = (2 * u + e) & 15;
                    WO0[sl] = op0[oo]; WO1[sl] = MODEL ? op1[oo] : 0u;
                    WS0[sl] = bp0[os]; WS1[sl] = MODEL ? bp1[os] : 0u;
                    oo += a.wpr; if (oo >= plane_words) oo -= plane_words;
                    os += a.wpr; if (os >= plane_words) os -= plane_words;
                }
            }
        }
    }
    __syncthreads();
    for (uint32_t t = threadIdx.x; t < MEAS_RC * 2; t += blockDim.x) {
        const uint32_t r = r0 + (t >> 1) + 1;
        const unsigned int v = (&s_cnt[0][0])[t];
        if (r <= a.r_max && v) atomicAdd(a.cnt + 2 + 2 * ((size_t)a.r_max + (r - 1)) + (t & 1u), (unsigned long long)v);
    }
    if (threadIdx.x < 2 && s_mq[threadIdx.x]) atomicAdd(a.cnt + threadIdx.x, s_mq[threadIdx.x]);
}

// x axis: thread = (colour c, row i, segment of 16 words); requires wpr % 16 == 0.
// r = 2d   -> same colour, bit shift d;   r = 2d+1 -> opposite colour, bit shift d + ((i+c)&1).
// With r0/2 a multiple of 32 the chunk needs source words k0 + r0/64 + [0, 16] of each colour
// and funnel shifts by 0..32 bits (clamped form).
template <int MODEL>
__global__ void __launch_bounds__(128) measure_x_kernel(const MeasBlkArgs a)
{
    __shared__ unsigned int s_cnt[MEAS_RC][2];
    for (uint32_t t = threadIdx.x; t < MEAS_RC * 2; t += blockDim.x) (&s_cnt[0][0])[t] = 0;
    __syncthreads();
    const uint32_t r0 = blockIdx.y * MEAS_RC;
    const uint32_t g = blockIdx.x * blockDim.x + threadIdx.x;
    const uint32_t nseg = a.wpr / MEAS_NB;
    const uint32_t per_colour = a.n * nseg;
    const bool live = g < 2u * per_colour;
    const uint32_t mask = __ballot_sync(0xffffffffu, live);
    const uint32_t lane = threadIdx.x & 31u;
    if (live) {
        const uint32_t leader = __ffs(mask) - 1;
        const uint32_t c = g >= per_colour ? 1u : 0u;
        const uint32_t rem = g - c * per_colour;
        const uint32_t ir = rem / nseg, sg = rem - ir * nseg;
        const uint32_t i = a.i0 + ir, k0 = sg * MEAS_NB;
        const uint32_t par = (i + c) & 1u;
        const unsigned long long ro = (unsigned long long)i * a.wpr;
        const uint32_t *bp0 = blk_plane<MODEL>(a, c, 0) + ro, *bp1 = blk_plane<MODEL>(a, c, 1) + ro;
        const uint32_t *op0 = blk_plane<MODEL>(a, c ^ 1u, 0) + ro, *op1 = blk_plane<MODEL>(a, c ^ 1u, 1) + ro;

        uint32_t B0[MEAS_NB], B1[MEAS_NB];
#pragma unroll
        for (int j = 0; j < MEAS_NB; j += 4) {
            const uint4 v = *reinterpret_cast<const uint4 *>(bp0 + k0 + j);
            B0[j] = v.x; B0[j + 1] = v.y; B0[j + 2] = v.z; B0[j + 3] = v.w;
            if (MODEL) {
                const uint4 w = *reinterpret_cast<const uint4 *>(bp1 + k0 + j);
                B1[j] = w.x; B1[j + 1] = w.y; B1[j + 2] = w.z; B1[j + 3] = w.w;
            } else { B1[j] = B1[j + 1] = B1[j + 2] = B1[j + 3] = 0u; }
        }
        uint32_t SS0[MEAS_NB + 1], SS1[MEAS_NB + 1], SO0[MEAS_NB + 1], SO1[MEAS_NB + 1];
        {
            uint32_t kk = k0 + (r0 >> 6);
            if (kk >= a.wpr) kk -= a.wpr;
#pragma unroll
            for (int x = 0; x <= MEAS_NB; ++x) {
                SS0[x] = bp0[kk]; SS1[x] = MODEL ? bp1[kk] : 0u;
                SO0[x] = op0[kk]; SO1[x] = MODEL ? op1[kk] : 0u;
                if (++kk == a.wpr) kk = 0;
            }
        }
#pragma unroll 1
        for (uint32_t b = 0; b < MEAS_RC / 2; ++b) {
            const uint32_t r_odd = r0 + 2 * b + 1;
            if (r_odd > a.r_max) break;
            {   // r = 2d+1, d = r0/2 + b: opposite colour, shift b + par (0..32)
                const uint32_t sh = b + par;
                uint32_t X[MEAS_NB], Y[MEAS_NB];
#pragma unroll
                for (int j = 0; j < MEAS_NB; ++j) {
                    const uint32_t p0 = __funnelshift_rc(SO0[j], SO0[j + 1], sh);
                    if (MODEL == 0) X[j] = B0[j] ^ p0;
                    else {
                        const uint32_t p1 = __funnelshift_rc(SO1[j], SO1[j + 1], sh);
                        X[j] = B0[j] & p0; Y[j] = X[j] & (B1[j] ^ p1);
                    }
                }
                const uint32_t c0 = weighted_popc16(X);
                const uint32_t c1 = MODEL ? weighted_popc16(Y) : 0u;
                add_r(s_cnt, r_odd - r0 - 1, mask, leader, lane, c0, c1, MODEL != 0);
            }
            if (r_odd + 1 <= a.r_max) {   // r = 2d, d = r0/2 + b + 1: same colour, shift b + 1 (1..32)
                const uint32_t sh = b + 1;
                uint32_t X[MEAS_NB], Y[MEAS_NB];
#pragma unroll
                for (int j = 0; j < MEAS_NB; ++j) {
                    const uint32_t p0 = __funnelshift_rc(SS0[j], SS0[j + 1], sh);
                    if (MODEL == 0) X[j] = B0[j] ^ p0;
                    else {
                        const uint32_t p1 = __funnelshift_rc(SS1[j], SS1[j + 1], sh);
                        X[j] = B0[j] & p0; Y[j] = X[j] & (B1[j] ^ p1);
                    }
                }
                const uint32_t c0 = weighted_popc16(X);
                const uint32_t c1 = MODEL ? weighted_popc16(Y) : 0u;
                add_r(s_cnt, r_odd - r0, mask, leader, lane, c0, c1, MODEL != 0);
            }
        }
    }
    __syncthreads();
    for (uint32_t t = threadIdx.x; t < MEAS_RC * 2; t += blockDim.x) {
        const uint32_t r = r0 + (t >> 1) + 1;
        const unsigned int v = (&s_cnt[0][0])[t];
        if (r <= a.r_max && v) atomicAdd(a.cnt + 2 + 2 * (size_t)(r - 1) + (t & 1u), (unsigned long long)v);
    }
}

// ---- sparse lists of r (lattice_measure_list) --------------------------------------------------
//
// The paper samples C(r;t) sparsely in r.  Same thread layout and carry-save
// reduction as the dense kernels, but the partner words of each listed r are loaded afresh: one
// partner read per (word, r, axis) instead of a sliding window.  blockIdx.y selects a chunk of
// MEAS_LIST_CHUNK list entries; counters as in the dense kernels with r - 1 replaced by the index
// in the list and r_max by its length n_r.
constexpr int MEAS_LIST_CHUNK = 32;

struct MeasListArgs {
    const uint32_t *buf;
    uint32_t L, wpr;                 // rows per plane, words per row
    uint32_t i0, n;                  // first base row, number of 16-row blocks
    const uint32_t *rlist;           // device, n_r entries, each in [1, L/2]
    uint32_t n_r;
    uint32_t mq;                     // also count M, Q (chunk 0)
    uint32_t axes;                   // measure_list_kernel: bit 0 = x axis, bit 1 = y axis
    unsigned long long *cnt;
};

// Both axes in one kernel: thread = (colour c, 16-row block, word column k) keeps its 16 base words
// (one per row) in registers; for every listed r it loads, coalesced along k,
//   y axis: the 16 words of rows i + r at the same k (colour c if r is even, else 1 - c),
//   x axis: per row the two words k + (s >> 5), + 1 of the partner colour, funnel-shifted by
//           s & 31, with s = r/2 (+ the row's parity (i + c) & 1 for odd r).
template <int MODEL>
__global__ void __launch_bounds__(128) measure_list_kernel(const MeasListArgs a)
{
    __shared__ unsigned int s_cnt[2][MEAS_LIST_CHUNK][2];          // [axis][entry][count]
    __shared__ unsigned long long s_mq[2];
    for (uint32_t t = threadIdx.x; t < 2 * MEAS_LIST_CHUNK * 2; t += blockDim.x) (&s_cnt[0][0][0])[t] = 0;
    if (threadIdx.x < 2) s_mq[threadIdx.x] = 0;
    __syncthreads();
    const uint32_t q0 = blockIdx.y * MEAS_LIST_CHUNK;
    const uint32_t g = blockIdx.x * blockDim.x + threadIdx.x;
    const uint32_t per_colour = a.n * a.wpr;
    const bool live = g < 2u * per_colour;
    const uint32_t mask = __ballot_sync(0xffffffffu, live);
    const uint32_t lane = threadIdx.x & 31u;
    if (live) {
        const uint32_t leader = __ffs(mask) - 1;
        const uint32_t c = g >= per_colour ? 1u : 0u;
        const uint32_t rem = g - c * per_colour;
        const uint32_t rb = rem / a.wpr, k = rem - rb * a.wpr;
        const uint32_t ib0 = a.i0 + MEAS_NB * rb;
        const uint32_t par0 = (ib0 + c) & 1u;                         // (i + c) & 1 of the block's first row
        const uint32_t *bp0 = blk_plane<MODEL>(a, c, 0), *bp1 = blk_plane<MODEL>(a, c, 1);
        const uint32_t *op0 = blk_plane<MODEL>(a, c ^ 1u, 0), *op1 = blk_plane<MODEL>(a, c ^ 1u, 1);
        const unsigned long long plane_words = (unsigned long long)a.L * a.wpr;
        const unsigned long long ob = (unsigned long long)ib0 * a.wpr;
        uint32_t B0[MEAS_NB], B1[MEAS_NB];
#pragma unroll
        for (int j = 0; j < MEAS_NB; ++j) {
            B0[j] = bp0[ob + (unsigned long long)j * a.wpr + k];
            B1[j] = MODEL ? bp1[ob + (unsigned long long)j * a.wpr + k] : 0u;
        }
        if (blockIdx.y == 0 && a.mq) {
            uint32_t m0 = 0, m1 = 0;
#pragma unroll
            for (int j = 0; j < MEAS_NB; ++j) {
                if (MODEL == 0) m0 += __popc(B0[j]);
                else { m0 += __popc(B0[j] & ~B1[j]); m1 += __popc(B0[j] & B1[j]); }
            }
            const uint32_t v0 = __reduce_add_sync(mask, m0);
            const uint32_t v1 = MODEL ? __reduce_add_sync(mask, m1) : 0u;
            if (lane == leader) {
                atomicAdd(&s_mq[0], (unsigned long long)v0);
                if (MODEL) atomicAdd(&s_mq[1], (unsigned long long)v1);
            }
        }
        const uint32_t q1 = min(q0 + (uint32_t)MEAS_LIST_CHUNK, a.n_r);
        for (uint32_t q = q0; q < q1; ++q) {
            const uint32_t r = a.rlist[q];
            const uint32_t *p0 = (r & 1u) ? op0 : bp0, *p1 = (r & 1u) ? op1 : bp1;
            uint32_t X[MEAS_NB], Y[MEAS_NB];
            if (a.axes & 2u) {   // y axis
                uint32_t row = ib0 + r;                                // < 2 L
                if (row >= a.L) row -= a.L;
                unsigned long long o = (unsigned long long)row * a.wpr + k;
                if (row + MEAS_NB <= a.L) {
                    // the 16 partner rows do not wrap: one running pointer, no per-row checks (the
                    // address arithmetic of the general form below cost more than the counting)
                    const uint32_t *q0 = p0 + o, *q1 = p1 + o;
#pragma unroll
                    for (int j = 0; j < MEAS_NB; ++j) {
                        const uint32_t w0 = *q0;
                        if (MODEL == 0) X[j] = B0[j] ^ w0;
                        else { X[j] = B0[j] & w0; Y[j] = X[j] & (B1[j] ^ *q1); }
                        q0 += a.wpr; q1 += a.wpr;
                    }
                } else {
#pragma unroll
                for (int j = 0; j < MEAS_NB; ++j) {
                    const uint32_t w0 = p0[o];
                    if (MODEL == 0) X[j] = B0[j] ^ w0;
                    else { X[j] = B0[j] & w0; Y[j] = X[j] & (B1[j] ^ p1[o]); }
                    o += a.wpr; if (o >= plane_words) o -= plane_words;
                }
                }
                const uint32_t c0 = weighted_popc16(X);
                const uint32_t c1 = MODEL ? weighted_popc16(Y) : 0u;
                add_r(s_cnt[1], q - q0, mask, leader, lane, c0, c1, MODEL != 0);
            }
            if (a.axes & 1u) {   // x axis: rows j and j+1 have parities par0 and par0 ^ 1
                const uint32_t sA = (r >> 1) + ((r & 1u) ? par0 : 0u), sB = (r >> 1) + ((r & 1u) ? (par0 ^ 1u) : 0u);
                uint32_t kA = k + (sA >> 5), kB = k + (sB >> 5);     // s >> 5 <= wpr / 2
                if (kA >= a.wpr) kA -= a.wpr;
                if (kB >= a.wpr) kB -= a.wpr;
                const uint32_t kA1 = (kA + 1 == a.wpr) ? 0 : kA + 1, kB1 = (kB + 1 == a.wpr) ? 0 : kB + 1;
                const uint32_t bA = sA & 31u, bB = sB & 31u;
                // four running pointers (rows of either parity: first and second word), advanced by
                // two rows per use: the 64-bit index arithmetic of `p0[o + ka]` per load cost more than
                // the counting
                const uint32_t *pa = p0 + ob + kA, *pa1 = p0 + ob + kA1;
                const uint32_t *pb = p0 + ob + a.wpr + kB, *pb1 = p0 + ob + a.wpr + kB1;
                const size_t two = 2 * (size_t)a.wpr, dpl = (size_t)(p1 - p0);
#pragma unroll
                for (int j = 0; j < MEAS_NB; j += 2) {
                    const uint32_t wA = __funnelshift_r(*pa, *pa1, bA), wB = __funnelshift_r(*pb, *pb1, bB);
                    if (MODEL == 0) { X[j] = B0[j] ^ wA; X[j + 1] = B0[j + 1] ^ wB; }
                    else {
                        const uint32_t vA = __funnelshift_r(pa[dpl], pa1[dpl], bA), vB = __funnelshift_r(pb[dpl], pb1[dpl], bB);
                        X[j] = B0[j] & wA; Y[j] = X[j] & (B1[j] ^ vA);
                        X[j + 1] = B0[j + 1] & wB; Y[j + 1] = X[j + 1] & (B1[j + 1] ^ vB);
                    }
                    pa += two; pa1 += two; pb += two; pb1 += two;
                }
                const uint32_t c0 = weighted_popc16(X);
                const uint32_t c1 = MODEL ? weighted_popc16(Y) : 0u;
                add_r(s_cnt[0], q - q0, mask, leader, lane, c0, c1, MODEL != 0);
            }
        }
    }
    __syncthreads();
    for (uint32_t t = threadIdx.x; t < 2 * MEAS_LIST_CHUNK * 2; t += blockDim.x) {
        const uint32_t axis = t / (MEAS_LIST_CHUNK * 2), e = t % (MEAS_LIST_CHUNK * 2);
        const uint32_t q = q0 + (e >> 1);
        const unsigned int v = (&s_cnt[0][0][0])[t];
        if (q < a.n_r && v)
            atomicAdd(a.cnt + 2 + 2 * ((size_t)axis * a.n_r + q) + (e & 1u), (unsigned long long)v);
    }
    if (threadIdx.x < 2 && s_mq[threadIdx.x]) atomicAdd(a.cnt + threadIdx.x, s_mq[threadIdx.x]);
}

// ---- r_max == 1: M, Q and the nearest-neighbour sums (the energy) in one pass ---------------
//
// The per-step record of a run (e, m, q) needs only r = 1.  One thread owns one 128-bit run of
// both colours and marches down MEAS_E1_ROWS rows with the previous row in registers, so the
// lattice is read from HBM exactly once (plus one row in MEAS_E1_ROWS and one side word per run):
//   y axis: colour c of row i pairs with colour c^1 of row i+1 at the same packed position;
//   x axis: r = 1 pairs colour c of row i with colour c^1 at p + ((i+c)&1): one of the two
//           colours pairs in place, the other with the opposite colour shifted by one bit.
// Requires wpr % 4 == 0.  Counts are reduced two rows at a time with the carry-save tree.
constexpr int MEAS_E1_ROWS = 32;

struct MeasE1Args {
    const uint32_t *buf;
    uint32_t rows, wpr;              // rows allocated per plane (L, or n_rows + 2 for a row slab)
    uint32_t i0, n_rows;             // local index of the first base row, number of base rows
    uint32_t par_off;                // parity of the global row of local row 0 (0 for a whole lattice)
    unsigned long long *cnt;         // [6]: MeasArgs::cnt layout with r_max = 1
};

template <int MODEL>
struct E1Row {                       // one 128-bit run of both colours (+ planes) of one row
    uint32_t a0[4], a1[4];           // colour 0: spins (Ising) or nz, sg (BC)
    uint32_t b0[4], b1[4];           // colour 1
    uint32_t e0, e1;                 // the word after the run of the colour whose bits pair shifted
};

// Row `row` (local index; == a.rows wraps to 0) of run kw; ODD = parity of the GLOBAL row: the colour
// c with (i + c) odd pairs along x with colour 1-c shifted down by one bit, i.e. it needs the word
// after the run (kn) of colour ODD.
template <int MODEL, int ODD>
__device__ __forceinline__ void e1_load(const MeasE1Args &a, uint32_t row, uint32_t kw, uint32_t kn, E1Row<MODEL> &r)
{
    const size_t pw = (size_t)a.rows * a.wpr;
    const unsigned long long ro = (row == a.rows) ? 0ull : (unsigned long long)row * a.wpr;
    const uint32_t *p = a.buf + ro + kw;
    const uint4 x = *reinterpret_cast<const uint4 *>(p);
    r.a0[0] = x.x; r.a0[1] = x.y; r.a0[2] = x.z; r.a0[3] = x.w;
    if (MODEL == 0) {
        const uint4 y = *reinterpret_cast<const uint4 *>(p + pw);
        r.b0[0] = y.x; r.b0[1] = y.y; r.b0[2] = y.z; r.b0[3] = y.w;
#pragma unroll
        for (int w = 0; w < 4; ++w) { r.a1[w] = 0; r.b1[w] = 0; }
        r.e0 = a.buf[(size_t)ODD * pw + ro + kn];
        r.e1 = 0;
    } else {
        const uint4 xs = *reinterpret_cast<const uint4 *>(p + pw);
        const uint4 y = *reinterpret_cast<const uint4 *>(p + 2 * pw);
        const uint4 ys = *reinterpret_cast<const uint4 *>(p + 3 * pw);
        r.a1[0] = xs.x; r.a1[1] = xs.y; r.a1[2] = xs.z; r.a1[3] = xs.w;
        r.b0[0] = y.x; r.b0[1] = y.y; r.b0[2] = y.z; r.b0[3] = y.w;
        r.b1[0] = ys.x; r.b1[1] = ys.y; r.b1[2] = ys.z; r.b1[3] = ys.w;
        r.e0 = a.buf[(size_t)(2 * ODD) * pw + ro + kn];
        r.e1 = a.buf[(size_t)(2 * ODD + 1) * pw + ro + kn];
    }
}

// The 8 words per tree that base row `cur` (global parity ODD) contributes, at tree slots o..o+7:
// XM / XN: +1 / -1 sites; XX (XXo): x-axis pairs (and those of opposite sign); XY (XYo): y axis.
template <int MODEL, int ODD>
__device__ __forceinline__ void e1_row(const E1Row<MODEL> &cur, const E1Row<MODEL> &nxt, int o, uint32_t (&XM)[16],
                                       uint32_t (&XN)[16], uint32_t (&XX)[16], uint32_t (&XXo)[16], uint32_t (&XY)[16],
                                       uint32_t (&XYo)[16])
{
#pragma unroll
    for (int w = 0; w < 4; ++w) {
        // partner-colour words shifted by one bit: colour ODD is the shifted partner of colour 1-ODD
        const uint32_t p0lo = ODD ? cur.b0[w] : cur.a0[w];
        const uint32_t p0hi = w < 3 ? (ODD ? cur.b0[w < 3 ? w + 1 : 0] : cur.a0[w < 3 ? w + 1 : 0]) : cur.e0;
        const uint32_t sh0 = __funnelshift_r(p0lo, p0hi, 1);
        const uint32_t t0 = ODD ? cur.a0[w] : cur.b0[w];              // the shifted pairing's base colour
        if (MODEL == 0) {
            XM[o + w] = cur.a0[w]; XM[o + w + 4] = cur.b0[w];
            XX[o + w] = cur.a0[w] ^ cur.b0[w];                        // in-place pairing
            XX[o + w + 4] = t0 ^ sh0;
            XY[o + w] = cur.a0[w] ^ nxt.b0[w];
            XY[o + w + 4] = cur.b0[w] ^ nxt.a0[w];
        } else {
            const uint32_t p1lo = ODD ? cur.b1[w] : cur.a1[w];
            const uint32_t p1hi = w < 3 ? (ODD ? cur.b1[w < 3 ? w + 1 : 0] : cur.a1[w < 3 ? w + 1 : 0]) : cur.e1;
            const uint32_t sh1 = __funnelshift_r(p1lo, p1hi, 1);
            const uint32_t t1 = ODD ? cur.a1[w] : cur.b1[w];
            XM[o + w] = cur.a0[w] & ~cur.a1[w]; XM[o + w + 4] = cur.b0[w] & ~cur.b1[w];
            XN[o + w] = cur.a0[w] & cur.a1[w]; XN[o + w + 4] = cur.b0[w] & cur.b1[w];
            XX[o + w] = cur.a0[w] & cur.b0[w];
            XXo[o + w] = XX[o + w] & (cur.a1[w] ^ cur.b1[w]);
            XX[o + w + 4] = t0 & sh0;
            XXo[o + w + 4] = XX[o + w + 4] & (t1 ^ sh1);
            XY[o + w] = cur.a0[w] & nxt.b0[w];
            XYo[o + w] = XY[o + w] & (cur.a1[w] ^ nxt.b1[w]);
            XY[o + w + 4] = cur.b0[w] & nxt.a0[w];
            XYo[o + w + 4] = XY[o + w + 4] & (cur.b1[w] ^ nxt.a1[w]);
        }
    }
}

// The march of one thread over base rows ia .. ia+nr-1 (local indices), two rows per step, with the
// two rows of the NEXT step already in flight while the current pair is reduced (the kernel is
// bound by HBM latency x bytes in flight, not by arithmetic).  P0 = global parity of row ia.
template <int MODEL, int P0>
__device__ __forceinline__ void e1_march(const MeasE1Args &a, uint32_t kw, uint32_t kn, uint32_t ia, uint32_t nr,
                                         uint32_t (&acc)[6])
{
    E1Row<MODEL> r0, r1, r2, r3, r4;                 // rows ia+rr .. ia+rr+4 of the current step
    e1_load<MODEL, P0>(a, ia, kw, kn, r0);
    e1_load<MODEL, P0 ^ 1>(a, ia + 1, kw, kn, r1);   // nr >= 1: row ia+1 is at least a partner row
    if (nr >= 2) e1_load<MODEL, P0>(a, ia + 2, kw, kn, r2);
    for (uint32_t rr = 0; rr < nr; rr += 2) {
        if (rr + 3 <= nr) e1_load<MODEL, P0 ^ 1>(a, ia + rr + 3, kw, kn, r3);
        if (rr + 4 <= nr) e1_load<MODEL, P0>(a, ia + rr + 4, kw, kn, r4);
        uint32_t XM[16], XN[16], XX[16], XXo[16], XY[16], XYo[16];
        e1_row<MODEL, P0>(r0, r1, 0, XM, XN, XX, XXo, XY, XYo);
        if (rr + 1 < nr) {
            e1_row<MODEL, P0 ^ 1>(r1, r2, 8, XM, XN, XX, XXo, XY, XYo);
        } else {
#pragma unroll
            for (int o = 8; o < 16; ++o) { XM[o] = XN[o] = XX[o] = XXo[o] = XY[o] = XYo[o] = 0; }
        }
        acc[0] += weighted_popc16(XM);
        acc[2] += weighted_popc16(XX);
        acc[4] += weighted_popc16(XY);
        if (MODEL) {
            acc[1] += weighted_popc16(XN);
            acc[3] += weighted_popc16(XXo);
            acc[5] += weighted_popc16(XYo);
        }
        r0 = r2; r1 = r3; r2 = r4;
    }
}

template <int MODEL>
__global__ void __launch_bounds__(128) measure_e1_kernel(const MeasE1Args a)
{
    const uint32_t nq = a.wpr >> 2;
    const uint32_t nslab = (a.n_rows + MEAS_E1_ROWS - 1) / MEAS_E1_ROWS;
    const uint32_t g = blockIdx.x * blockDim.x + threadIdx.x;
    uint32_t acc[6] = {0, 0, 0, 0, 0, 0};       // m0, m1, x0, x1, y0, y1 (MeasArgs::cnt order)
    if (g < nq * nslab) {
        const uint32_t q = g % nq, sl = g / nq;
        const uint32_t kw = q << 2;
        const uint32_t kn = (kw + 4 == a.wpr) ? 0 : kw + 4;       // word after the run (periodic)
        const uint32_t ia = a.i0 + sl * MEAS_E1_ROWS;
        const uint32_t nr = min((uint32_t)MEAS_E1_ROWS, a.i0 + a.n_rows - ia);
        if ((ia + a.par_off) & 1u) e1_march<MODEL, 1>(a, kw, kn, ia, nr, acc);
        else e1_march<MODEL, 0>(a, kw, kn, ia, nr, acc);
    }
    __shared__ unsigned long long sh[6];
    if (threadIdx.x < 6) sh[threadIdx.x] = 0;
    __syncthreads();
#pragma unroll
    for (int e = 0; e < 6; ++e) {
        if (MODEL == 0 && (e & 1)) continue;
        const uint32_t v = __reduce_add_sync(0xffffffffu, acc[e]);
        if ((threadIdx.x & 31u) == 0 && v) atomicAdd(&sh[e], (unsigned long long)v);
    }
    __syncthreads();
    if (threadIdx.x < 6 && sh[threadIdx.x]) atomicAdd(a.cnt + threadIdx.x, sh[threadIdx.x]);
}

// ---- unpacked windows (tests, windowed replay, checkpoints) --------------------------------
struct WindowArgs {
    uint32_t *buf;
    uint32_t L, wpr, model;
    uint32_t rows, row_base;         // rows allocated per plane and the global row of local row 0
                                     // (L and 0 for a whole lattice; n_rows + 2 and row0 - 1 for a slab)
    uint32_t i0, j0, h, w;
    int8_t *spins;                   // device, row-major h x w
};

__device__ __forceinline__ void site_addr(const WindowArgs &a, uint32_t i, uint32_t j,
                                          size_t &word, uint32_t &bit, uint32_t &colour)
{
    colour = (i + j) & 1u;
    const uint32_t p = j >> 1;
    const uint32_t li = i >= a.row_base ? i - a.row_base : i + a.L - a.row_base;   // local row
    word = (size_t)li * a.wpr + (p >> 5);
    bit = p & 31u;
}

__global__ void __launch_bounds__(256) get_spins_kernel(const WindowArgs a)
{
    const unsigned long long g = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= (unsigned long long)a.h * a.w) return;
    const uint32_t i = (uint32_t)((a.i0 + g / a.w) % a.L), j = (uint32_t)((a.j0 + g % a.w) % a.L);
    size_t word; uint32_t bit, colour;
    site_addr(a, i, j, word, bit, colour);
    const size_t pw = (size_t)a.rows * a.wpr;
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
    const size_t pw = (size_t)a.rows * a.wpr;
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
