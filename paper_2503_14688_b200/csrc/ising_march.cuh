// ising_march.cuh -- the production Ising half-sweep (RNG scheme 1, L a multiple of 256).
//
// Paper: Metropolis + checkerboard + multispin coding, Eq. 1 in the Ising
// limit, 32-bit acceptance compare.  Same packing, neighbour
// geometry and acceptance rule as ising.cuh (which stays as the generic path: scheme 0 and
// lattices whose rows are not a whole number of 128-bit runs); what changes is how the work
// is laid on the machine, because the kernel is bound by the integer pipes (DESIGN.md
// "Rooflines"), not by HBM:
//
//   * one thread owns one 128-bit run (4 words = 128 same-colour sites = one RNG unit G) and
//     MARCHES down R consecutive rows, keeping the opposite-colour rows i-1, i, i+1 in
//     registers: per row it loads 2 x 128 bits + 1 side word instead of 4 x 128 bits + 1;
//   * the 8 acceptance bit-planes of unit G come from the folded Philox streams of philox.cuh
//     (16 instead of 20 multiplies per plane, the first rounds shared by the planes);
//   * the rare lanes whose top random byte ties with the threshold's (2^-8 per deciding lane)
//     are not resolved in place -- that would make all 32 threads of a warp walk through a
//     Philox block whenever one of them has a tie -- but pushed into a per-warp queue in shared
//     memory; whenever 32 entries are pending the warp resolves them, one entry per thread,
//     and applies the accepted flips with a global atomic XOR on the already-stored word.
//
// Everything that decides a spin is computed in march_row()/tail_accept(), which are plain
// functions of their arguments; the queue is a policy so that the same code can be driven
// sequentially in a host harness.
#pragma once
#include "ising.cuh"

namespace lat {

struct IsingMarchArgs {
    uint32_t *tgt;            // colour being updated   [L][wpr]
    const uint32_t *opp;      // opposite colour        [L][wpr]
    uint32_t L, wpr;
    uint32_t t, colour;
    uint32_t thr4, thr8;      // thresholds for dE = 4, 8 (low 24 bits used by the tails)
    uint32_t always4, always8;// threshold == 2^32: the class flips unconditionally
    uint32_t top4, top8;      // top bytes of thr4, thr8
    uint32_t R;               // rows per thread (even, divides L)
    uint32_t threads;         // (wpr/4) * (L/R), a multiple of 32
    PlaneFold F;              // folded ACC_PLANE stream of (t, colour)
    RoundKeys K;
};

__host__ __device__ __forceinline__ uint32_t fsl1(uint32_t lo, uint32_t hi)   // (hi:lo << 1) high word
{
#ifdef __CUDA_ARCH__
    return __funnelshift_l(lo, hi, 1);
#else
    return (hi << 1) | (lo >> 31);
#endif
}
__host__ __device__ __forceinline__ uint32_t fsr1(uint32_t lo, uint32_t hi)   // (hi:lo >> 1) low word
{
#ifdef __CUDA_ARCH__
    return __funnelshift_r(lo, hi, 1);
#else
    return (lo >> 1) | (hi << 31);
#endif
}
__host__ __device__ __forceinline__ uint32_t maj3m(uint32_t a, uint32_t b, uint32_t c)
{
    return (a & b) | (a & c) | (b & c);
}
__host__ __device__ __forceinline__ uint32_t w4(const uint4 &v, int i)
{
    return i == 0 ? v.x : i == 1 ? v.y : i == 2 ? v.z : v.w;
}

// One row of one 128-bit run.  T: target words; U, C, D: opposite-colour words of rows i-1, i,
// i+1 at the same packed position; E: the side word (PAR == 0: the word before the run,
// PAR == 1: the word after it).  Returns the updated words with every tie treated as a
// rejection; eq = lanes whose top byte ties (to be resolved by tail_accept), c8q = eq & class 8.
template <int PAR>
__host__ __device__ __forceinline__ uint4 march_row(const IsingMarchArgs &a, uint32_t G, const uint4 &T4,
                                                    const uint4 &U4, const uint4 &C4, const uint4 &D4,
                                                    uint32_t E, uint4 &eq4, uint4 &c8q4)
{
    uint32_t T[4] = {T4.x, T4.y, T4.z, T4.w};
    const uint32_t U[4] = {U4.x, U4.y, U4.z, U4.w};
    const uint32_t C[4] = {C4.x, C4.y, C4.z, C4.w};
    const uint32_t D[4] = {D4.x, D4.y, D4.z, D4.w};
    uint32_t S[4];
    if (PAR == 0) {           // neighbour at p-1
        S[0] = fsl1(E, C[0]); S[1] = fsl1(C[0], C[1]); S[2] = fsl1(C[1], C[2]); S[3] = fsl1(C[2], C[3]);
    } else {                  // neighbour at p+1
        S[0] = fsr1(C[0], C[1]); S[1] = fsr1(C[1], C[2]); S[2] = fsr1(C[2], C[3]); S[3] = fsr1(C[3], E);
    }
    uint32_t c4[4], c8[4], acc[4], eq[4];
#pragma unroll
    for (int w = 0; w < 4; ++w) {
        // bit-sliced count of "+1" neighbours n = s0 + 2 (c1 + c2); aligned count k = t ? n : 4-n
        const uint32_t s1 = U[w] ^ D[w] ^ C[w];
        const uint32_t c1 = maj3m(U[w], D[w], C[w]);
        const uint32_t s0 = s1 ^ S[w];
        const uint32_t c2 = s1 & S[w];
        const uint32_t t = T[w];
        const uint32_t g = (t & c1 & c2) | (~t & ~(c1 | c2));
        c8[w] = g & (t | ~s0);                                   // k == 4: dE = 8
        const uint32_t h = (t & (c1 ^ c2)) | (~t & ~(c1 | c2));
        c4[w] = s0 & h;                                          // k == 3: dE = 4
    }
    if (a.always4) {
#pragma unroll
        for (int w = 0; w < 4; ++w) c4[w] = 0;
    }
    if (a.always8) {
#pragma unroll
        for (int w = 0; w < 4; ++w) c8[w] = 0;
    }
#pragma unroll
    for (int w = 0; w < 4; ++w) { acc[w] = 0; eq[w] = c4[w] | c8[w]; }

    // top byte of u32(site) against the top byte of the lane's threshold, least significant
    // plane first: acc <- MAJ(tau, ~b, acc) is "u < thr" on the bits seen so far
    const PlaneShared ps = plane_shared(G, a.F);
#pragma unroll
    for (int k = 7; k >= 0; --k) {
        const uint4 b4 = plane_block(ps, a.F.fb[k], a.F, a.K);
        const uint32_t b[4] = {b4.x, b4.y, b4.z, b4.w};
        const uint32_t m4 = (a.top4 >> (7 - k)) & 1u, m8 = (a.top8 >> (7 - k)) & 1u;   // warp-uniform
        if (m4 == m8) {
            if (m4) {
#pragma unroll
                for (int w = 0; w < 4; ++w) {
                    const uint32_t tau = c4[w] | c8[w];
                    acc[w] = maj3m(tau, ~b[w], acc[w]);
                    eq[w] &= ~(b[w] ^ tau);
                }
            } else {
#pragma unroll
                for (int w = 0; w < 4; ++w) { acc[w] &= ~b[w]; eq[w] &= ~b[w]; }
            }
        } else if (m4) {
#pragma unroll
            for (int w = 0; w < 4; ++w) {
                acc[w] = maj3m(c4[w], ~b[w], acc[w]);
                eq[w] &= ~(b[w] ^ c4[w]);
            }
        } else {
#pragma unroll
            for (int w = 0; w < 4; ++w) {
                acc[w] = maj3m(c8[w], ~b[w], acc[w]);
                eq[w] &= ~(b[w] ^ c8[w]);
            }
        }
    }
    // lanes outside c4|c8 flip unconditionally (dE <= 0); ties stay put until resolved
#pragma unroll
    for (int w = 0; w < 4; ++w) T[w] ^= ~(c4[w] | c8[w]) | acc[w];   // a tied lane has acc = 0
    eq4 = make_uint4(eq[0], eq[1], eq[2], eq[3]);
    c8q4 = make_uint4(eq[0] & c8[0], eq[1] & c8[1], eq[2] & c8[2], eq[3] & c8[3]);
    return make_uint4(T[0], T[1], T[2], T[3]);
}

// Resolve the ties of one queued run: low 24 bits of u32(site) from the site's own tail block
// against the low 24 bits of its threshold.  wo = word offset i*wpr + kw of the run (so that
// the site index is P = 32 (wo + w) + bit).  Returns, per word, the lanes that flip after all.
__host__ __device__ __forceinline__ uint4 tail_accept(const IsingMarchArgs &a, unsigned long long wo, uint4 eq4,
                                                      const uint4 &c8q4)
{
    uint32_t e[4] = {eq4.x, eq4.y, eq4.z, eq4.w};
    const uint32_t c8[4] = {c8q4.x, c8q4.y, c8q4.z, c8q4.w};
    uint32_t flip[4] = {0, 0, 0, 0};
    // one tie per iteration, whichever word it is in: a warp iterates max-over-lanes(#ties)
    // times (ties are sparse: usually one per queued run)
    for (;;) {
        const int w = e[0] ? 0 : e[1] ? 1 : e[2] ? 2 : 3;
        const uint32_t ew = e[0] ? e[0] : e[1] ? e[1] : e[2] ? e[2] : e[3];
        if (!ew) break;
#ifdef __CUDA_ARCH__
        const uint32_t bit = __ffs(ew) - 1;
#else
        const uint32_t bit = __builtin_ctz(ew);
#endif
        const uint32_t m = 1u << bit;
        const unsigned long long P = ((wo + (unsigned)w) << 5) + bit;
        const uint4 blk = philox4x32_10((uint32_t)P, (uint32_t)(P >> 32), a.t,
                                        a.colour | (TAG_ACC_TAIL << 8), a.K);
        const uint32_t c8w = w == 0 ? c8[0] : w == 1 ? c8[1] : w == 2 ? c8[2] : c8[3];
        const uint32_t thr = (c8w & m) ? a.thr8 : a.thr4;
        const uint32_t hit = ((blk.x >> 8) < (thr & 0x00ffffffu)) ? m : 0u;
        if (w == 0) { e[0] &= ~m; flip[0] |= hit; }
        else if (w == 1) { e[1] &= ~m; flip[1] |= hit; }
        else if (w == 2) { e[2] &= ~m; flip[2] |= hit; }
        else { e[3] &= ~m; flip[3] |= hit; }
    }
    return make_uint4(flip[0], flip[1], flip[2], flip[3]);
}

// The march of one thread: rows i0 .. i0+R-1 of run q.  Q is the tie-queue policy:
//   q.push(has, eq, c8q, wo)  collective over the warp; wo = word offset of the run
//   q.drain()                 collective; resolves everything still pending
template <int COLOUR, class Q>
__host__ __device__ __forceinline__ void march_thread(const IsingMarchArgs &a, uint32_t g, Q &queue)
{
    const uint32_t L = a.L, wpr = a.wpr, nq = wpr >> 2;
    const uint32_t q = g % nq, s = g / nq;
    const uint32_t kw = q << 2;
    const uint32_t i0 = s * a.R;
    const uint32_t iu = (i0 == 0) ? L - 1 : i0 - 1;
    // side words: PAR == 0 reads the word before the run, PAR == 1 the word after it (periodic)
    const uint32_t ke0 = (kw == 0) ? wpr - 1 : kw - 1;
    const uint32_t ke1 = (kw + 4 == wpr) ? 0 : kw + 4;

    unsigned long long ro = (unsigned long long)i0 * wpr;            // word offset of row i
    uint4 U = *reinterpret_cast<const uint4 *>(a.opp + (unsigned long long)iu * wpr + kw);
    uint4 C = *reinterpret_cast<const uint4 *>(a.opp + ro + kw);
    uint32_t G = i0 * nq + q;                                        // (i*(L/2) + 32 kw) >> 7

    for (uint32_t r = 0; r < a.R; r += 2) {
        {   // row i0 + r: (i + colour) & 1 == COLOUR because i0 and r are even
            const uint32_t i = i0 + r;
            const unsigned long long rd = (i + 1 == L) ? 0ull : ro + wpr;
            const uint4 T = *reinterpret_cast<const uint4 *>(a.tgt + ro + kw);
            const uint4 D = *reinterpret_cast<const uint4 *>(a.opp + rd + kw);
            const uint32_t E = a.opp[ro + (COLOUR == 0 ? ke0 : ke1)];
            uint4 eq, c8q;
            const uint4 Tn = march_row<COLOUR>(a, G, T, U, C, D, E, eq, c8q);
            *reinterpret_cast<uint4 *>(a.tgt + ro + kw) = Tn;
            queue.push((eq.x | eq.y | eq.z | eq.w) != 0, eq, c8q, ro + kw);
            U = C; C = D; ro = rd; G += nq;
        }
        {   // row i0 + r + 1: the other parity
            const uint32_t i = i0 + r + 1;
            const unsigned long long rd = (i + 1 == L) ? 0ull : ro + wpr;
            const uint4 T = *reinterpret_cast<const uint4 *>(a.tgt + ro + kw);
            const uint4 D = *reinterpret_cast<const uint4 *>(a.opp + rd + kw);
            const uint32_t E = a.opp[ro + (COLOUR == 0 ? ke1 : ke0)];
            uint4 eq, c8q;
            const uint4 Tn = march_row<COLOUR ^ 1>(a, G, T, U, C, D, E, eq, c8q);
            *reinterpret_cast<uint4 *>(a.tgt + ro + kw) = Tn;
            queue.push((eq.x | eq.y | eq.z | eq.w) != 0, eq, c8q, ro + kw);
            U = C; C = D; ro = rd; G += nq;
        }
    }
    queue.drain();
}

#ifdef __CUDACC__
// Per-warp tie queue in shared memory.  At most 31 entries are pending before a push and a
// push adds at most 32, so 64 slots are enough.  Entries are resolved 32 at a time, one per
// thread, which keeps the Philox tail blocks dense in the warp.
struct WarpTieQueue {
    const IsingMarchArgs &a;
    uint4 *eq, *c8;            // [64] each, this warp's slice
    unsigned long long *wo;    // [64]
    uint32_t lane, pending;

    __device__ __forceinline__ void resolve(uint32_t idx)
    {
        const uint4 e = eq[idx], c = c8[idx];
        const unsigned long long o = wo[idx];
        const uint4 f = tail_accept(a, o, e, c);
        if (f.x) atomicXor(a.tgt + o, f.x);
        if (f.y) atomicXor(a.tgt + o + 1, f.y);
        if (f.z) atomicXor(a.tgt + o + 2, f.z);
        if (f.w) atomicXor(a.tgt + o + 3, f.w);
    }
    __device__ __forceinline__ void push(bool has, const uint4 &e, const uint4 &c, unsigned long long o)
    {
        const uint32_t m = __ballot_sync(0xffffffffu, has);
        if (m == 0) return;
        if (has) {
            const uint32_t slot = pending + __popc(m & ((1u << lane) - 1u));
            eq[slot] = e; c8[slot] = c; wo[slot] = o;
        }
        pending += __popc(m);
        __syncwarp();
        if (pending >= 32) {
            pending -= 32;
            resolve(pending + lane);
            __syncwarp();
        }
    }
    __device__ __forceinline__ void drain()
    {
        __syncwarp();
        if (lane < pending) resolve(lane);
        pending = 0;
    }
};

template <int COLOUR>
__global__ void __launch_bounds__(256) ising_march_kernel(const IsingMarchArgs a)
{
    __shared__ uint4 s_eq[8][64];
    __shared__ uint4 s_c8[8][64];
    __shared__ unsigned long long s_wo[8][64];
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const uint32_t g = blockIdx.x * 256u + threadIdx.x;
    if (g - lane >= a.threads) return;          // a.threads is a multiple of 32: whole warps only
    WarpTieQueue queue{a, s_eq[warp], s_c8[warp], s_wo[warp], lane, 0u};
    march_thread<COLOUR>(a, g, queue);
}
#endif

}  // namespace lat
