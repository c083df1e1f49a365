// ising.cuh -- packed checkerboard Metropolis half-sweep for the spin-1/2 Ising model.
//
// Paper: Metropolis + checkerboard + multispin coding, Eq. 1 in the Ising
// limit.  1 bit per spin (bit = 1 <-> s = +1), packed by sublattice:
// word k of colour c in row i holds p = 32k..32k+31, column j = 2p + ((i+c)&1).
//
// For a target word T[i][k] of colour c the four neighbour words are opposite-colour words
//   U = O[i-1][k], D = O[i+1][k], C = O[i][k] and the side word
//   S = (C << 1) | (O[i][k-1] >> 31)   if (i+c) is even   (neighbour at p-1)
//   S = (C >> 1) | (O[i][k+1] << 31)   if (i+c) is odd    (neighbour at p+1)
// (indices periodic).  The number of "+1" neighbours is added bit-sliced (two carry-save
// steps), turned into the two classes that need a random decision
//   c4: exactly 3 neighbours aligned with s (dE = 4),  c8: all 4 aligned (dE = 8)
// and every other lane flips unconditionally (dE <= 0).
//
// Acceptance u32(site) < thr[dE] is evaluated without ever materialising u32 per site
// (scheme 1): the top byte of u32 comes from 8 Philox bit-planes shared by the thread's 128
// sites and is compared bit-serially against the top byte of the lane's threshold; only a
// lane whose top byte ties (probability 2^-8) needs its own tail block for the low 24 bits.
// Scheme 0 draws one 32-bit word per site (4 sites per Philox block) and compares directly.
#pragma once
#include "philox.cuh"

namespace lat {

struct IsingArgs {
    uint32_t *tgt;            // colour being updated   [L][wpr]
    const uint32_t *opp;      // opposite colour        [L][wpr]
    uint32_t L;
    uint32_t wpr;             // 32-bit words per row per colour = L/64
    uint32_t t;               // sweep index
    uint32_t colour;          // 0 = black ((i+j) even), 1 = white
    uint32_t thr4, thr8;      // thresholds for dE = 4, 8 (valid when not "always")
    uint32_t always4, always8;// threshold == 2^32: class accepts unconditionally
    uint32_t tq_log2;         // tile width in quads (WPT=4 kernel): 1 << tq_log2
    RoundKeys K;
};

__device__ __forceinline__ uint32_t maj3(uint32_t a, uint32_t b, uint32_t c)
{
    return (a & b) | (a & c) | (b & c);
}

// One thread updates WPT consecutive words kw..kw+WPT-1 of row i.  WPT = 4 requires
// wpr % 4 == 0 and kw % 4 == 0, so that the run is exactly one 128-site RNG unit.
template <int WPT, int SCHEME>
__device__ __forceinline__ void ising_update_run(const IsingArgs &a, uint32_t i, uint32_t kw)
{
    const uint32_t L = a.L, wpr = a.wpr;
    const uint32_t iu = (i == 0) ? L - 1 : i - 1;
    const uint32_t id = (i + 1 == L) ? 0 : i + 1;
    const size_t row = (size_t)i * wpr, rowu = (size_t)iu * wpr, rowd = (size_t)id * wpr;
    const uint32_t par = (i + a.colour) & 1u;

    uint32_t T[WPT], U[WPT], D[WPT], C[WPT], S[WPT];
    if constexpr (WPT == 4) {
        const uint4 t4 = *reinterpret_cast<const uint4 *>(a.tgt + row + kw);
        const uint4 u4 = *reinterpret_cast<const uint4 *>(a.opp + rowu + kw);
        const uint4 d4 = *reinterpret_cast<const uint4 *>(a.opp + rowd + kw);
        const uint4 c4 = *reinterpret_cast<const uint4 *>(a.opp + row + kw);
        T[0] = t4.x; T[1] = t4.y; T[2] = t4.z; T[3] = t4.w;
        U[0] = u4.x; U[1] = u4.y; U[2] = u4.z; U[3] = u4.w;
        D[0] = d4.x; D[1] = d4.y; D[2] = d4.z; D[3] = d4.w;
        C[0] = c4.x; C[1] = c4.y; C[2] = c4.z; C[3] = c4.w;
    } else {
#pragma unroll
        for (int w = 0; w < WPT; ++w) {
            T[w] = a.tgt[row + kw + w];
            U[w] = a.opp[rowu + kw + w];
            D[w] = a.opp[rowd + kw + w];
            C[w] = a.opp[row + kw + w];
        }
    }
    // side neighbour: one extra word, direction by row parity (periodic in the row)
    if (par == 0) {
        const uint32_t ke = (kw == 0) ? wpr - 1 : kw - 1;
        const uint32_t E = a.opp[row + ke];
#pragma unroll
        for (int w = 0; w < WPT; ++w) S[w] = __funnelshift_l(w == 0 ? E : C[w > 0 ? w - 1 : 0], C[w], 1);
    } else {
        const uint32_t ke = (kw + WPT == wpr) ? 0 : kw + WPT;
        const uint32_t E = a.opp[row + ke];
#pragma unroll
        for (int w = 0; w < WPT; ++w)
            S[w] = __funnelshift_r(C[w], w == WPT - 1 ? E : C[w < WPT - 1 ? w + 1 : 0], 1);
    }

    // bit-sliced count of "+1" neighbours: n = s0 + 2*(c1 + c2)
    uint32_t c4[WPT], c8[WPT];
#pragma unroll
    for (int w = 0; w < WPT; ++w) {
        const uint32_t s1 = U[w] ^ D[w] ^ C[w];
        const uint32_t c1 = maj3(U[w], D[w], C[w]);
        const uint32_t s0 = s1 ^ S[w];
        const uint32_t c2 = s1 & S[w];
        const uint32_t t = T[w];
        // aligned count k = t ? n : 4 - n.  k == 4: (t & n==4) | (~t & n==0)
        const uint32_t g = (t & c1 & c2) | (~t & ~(c1 | c2));
        c8[w] = g & (t | ~s0);
        // k == 3: s0 & (t ? exactly one of c1,c2 : none of them)
        const uint32_t h = (t & (c1 ^ c2)) | (~t & ~(c1 | c2));
        c4[w] = s0 & h;
    }
    if (a.always4) {
#pragma unroll
        for (int w = 0; w < WPT; ++w) c4[w] = 0;
    }
    if (a.always8) {
#pragma unroll
        for (int w = 0; w < WPT; ++w) c8[w] = 0;
    }

    const unsigned long long P0 = (unsigned long long)i * (L >> 1) + ((unsigned long long)kw << 5);
    uint32_t acc[WPT];   // lanes of c4|c8 whose move is accepted
#pragma unroll
    for (int w = 0; w < WPT; ++w) acc[w] = 0;

    if (SCHEME == 1) {
        const unsigned long long G = P0 >> 7;
        const uint32_t sub = (uint32_t)(P0 >> 5) & 3u;   // used when WPT == 1
        uint32_t eq[WPT];
#pragma unroll
        for (int w = 0; w < WPT; ++w) eq[w] = c4[w] | c8[w];
        // top byte, least significant plane first: m <- MAJ(tau, ~b, m) is "u < thr" on the
        // bits seen so far; eq tracks lanes whose top byte still equals the threshold's.
#pragma unroll
        for (int k = 7; k >= 0; --k) {
            const uint4 blk = philox_unit(G, a.t, a.colour, TAG_ACC_PLANE, (uint32_t)k, a.K);
            const uint32_t t4k = ((a.thr4 >> (31 - k)) & 1u) ? 0xffffffffu : 0u;
            const uint32_t t8k = ((a.thr8 >> (31 - k)) & 1u) ? 0xffffffffu : 0u;
#pragma unroll
            for (int w = 0; w < WPT; ++w) {
                const uint32_t b = (WPT == 4) ? pick(blk, w) : pick(blk, sub + w);
                const uint32_t tau = (c4[w] & t4k) | (c8[w] & t8k);
                acc[w] = maj3(tau, ~b, acc[w]);
                eq[w] &= ~(b ^ tau);
            }
        }
        // rare ties: low 24 bits from the site's own tail block
#pragma unroll
        for (int w = 0; w < WPT; ++w) {
            uint32_t e = eq[w];
            while (e) {
                const uint32_t bit = __ffs(e) - 1;
                e &= e - 1;
                const unsigned long long P = P0 + 32u * w + bit;
                const uint4 blk = philox_unit(P, a.t, a.colour, TAG_ACC_TAIL, 0, a.K);
                const uint32_t thr = ((c8[w] >> bit) & 1u) ? a.thr8 : a.thr4;
                if ((blk.x >> 8) < (thr & 0x00ffffffu)) acc[w] |= 1u << bit;
            }
        }
    } else {
        // scheme 0: one 32-bit word per site, 4 sites per block
#pragma unroll
        for (int w = 0; w < WPT; ++w) {
            const uint32_t need = c4[w] | c8[w];
#pragma unroll 1
            for (int q = 0; q < 8; ++q) {
                if (((need >> (4 * q)) & 0xfu) == 0) continue;
                const unsigned long long unit = (P0 + 32u * w + 4u * q) >> 2;
                const uint4 blk = philox_unit(unit, a.t, a.colour, TAG_ACC_QUAD, 0, a.K);
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const uint32_t bit = 4 * q + j;
                    const uint32_t thr = ((c8[w] >> bit) & 1u) ? a.thr8 : a.thr4;
                    if (pick(blk, j) < thr) acc[w] |= 1u << bit;
                }
            }
            acc[w] &= need;
        }
    }

#pragma unroll
    for (int w = 0; w < WPT; ++w) T[w] ^= (~(c4[w] | c8[w])) | acc[w];

    if constexpr (WPT == 4) {
        *reinterpret_cast<uint4 *>(a.tgt + row + kw) = make_uint4(T[0], T[1], T[2], T[3]);
    } else {
#pragma unroll
        for (int w = 0; w < WPT; ++w) a.tgt[row + kw + w] = T[w];
    }
}

// 128-bit runs: block = 256 threads = (1 << tq_log2) quads wide x (256 >> tq_log2) rows; rows of
// a tile are enumerated even-first so that every warp works on rows of one parity (the side
// neighbour direction is then warp-uniform).
template <int SCHEME>
__global__ void __launch_bounds__(256) ising_half_sweep_v4(const IsingArgs a)
{
    const uint32_t tq = 1u << a.tq_log2;
    const uint32_t tr = 256u >> a.tq_log2;
    const uint32_t nq = a.wpr >> 2;
    const uint32_t tiles_x = nq >> a.tq_log2;
    const uint32_t bx = blockIdx.x % tiles_x, by = blockIdx.x / tiles_x;
    const uint32_t q = bx * tq + (threadIdx.x & (tq - 1));
    const uint32_t r = threadIdx.x >> a.tq_log2;
    const uint32_t half = tr >> 1;
    const uint32_t rr = (r < half) ? 2 * r : 2 * (r - half) + 1;
    const uint32_t i = by * tr + rr;
    if (i >= a.L) return;
    ising_update_run<4, SCHEME>(a, i, q * 4);
}

// generic path (any L % 64 == 0, in particular L = 64 and 128): one word per thread
template <int SCHEME>
__global__ void __launch_bounds__(256) ising_half_sweep_v1(const IsingArgs a)
{
    const unsigned long long g = (unsigned long long)blockIdx.x * 256u + threadIdx.x;
    if (g >= (unsigned long long)a.L * a.wpr) return;
    const uint32_t i = (uint32_t)(g / a.wpr), k = (uint32_t)(g % a.wpr);
    ising_update_run<1, SCHEME>(a, i, k);
}

// Disordered start: s = +1 iff the site's INIT-plane bit is 1.  One thread per
// 128-site unit of one colour (or per word when a row is not a whole number of units).
struct IsingInitArgs {
    uint32_t *buf;            // [2][L][wpr]
    uint32_t L, wpr;
    RoundKeys K;
};

__global__ void __launch_bounds__(256) ising_init_kernel(const IsingInitArgs a)
{
    const unsigned long long words = (unsigned long long)a.L * a.wpr;   // per colour
    const unsigned long long g = (unsigned long long)blockIdx.x * 256u + threadIdx.x;
    if (g >= 2 * words) return;
    const uint32_t colour = g >= words;
    const unsigned long long wi = g - (colour ? words : 0);
    // same-colour linear index of the word's first site: rows are L/2 = 32*wpr sites long
    const unsigned long long P0 = wi << 5;
    const uint4 blk = philox_unit(P0 >> 7, 0, colour, TAG_INIT_PLANE, 0, a.K);
    a.buf[g] = pick(blk, (uint32_t)(P0 >> 5) & 3u);
}

// Row-slab variant of the disordered start: the slab holds local rows 0 .. rows-1 per colour,
// local row l being global row (row_base + l) mod L (local rows 0 and rows-1 are halo rows).
// Keying uses global coordinates, so the halos are born consistent with their owners.
struct IsingSlabInitArgs {
    uint32_t *buf;            // [2][rows][wpr]
    uint32_t L, wpr, rows, row_base;
    RoundKeys K;
};

__global__ void __launch_bounds__(256) ising_init_slab_kernel(const IsingSlabInitArgs a)
{
    const unsigned long long words = (unsigned long long)a.rows * a.wpr;   // per colour
    const unsigned long long g = (unsigned long long)blockIdx.x * 256u + threadIdx.x;
    if (g >= 2 * words) return;
    const uint32_t colour = g >= words;
    const unsigned long long wi = g - (colour ? words : 0);
    const uint32_t li = (uint32_t)(wi / a.wpr), k = (uint32_t)(wi % a.wpr);
    const uint32_t gi = (a.row_base + li) % a.L;
    const unsigned long long P0 = ((unsigned long long)gi * a.wpr + k) << 5;
    const uint4 blk = philox_unit(P0 >> 7, 0, colour, TAG_INIT_PLANE, 0, a.K);
    a.buf[g] = pick(blk, (uint32_t)(P0 >> 5) & 3u);
}

}  // namespace lat
