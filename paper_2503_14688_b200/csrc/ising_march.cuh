// ising_march.cuh -- the production Ising half-sweep (RNG scheme 1, L a multiple of 256).
//
// Paper: Metropolis + checkerboard + multispin coding, Eq. 1 in the Ising
// limit, 32-bit acceptance compare.  Same packing, neighbour
// geometry and acceptance rule as ising.cuh (which stays as the generic path: scheme 0 and
// lattices whose rows are not a whole number of 128-bit runs); what changes is how the work
// is laid on the machine, because the kernel is bound by the 16-lane integer dispatch
// (DESIGN.md section 6), not by HBM -- every LOP3-class instruction and every wide multiply
// costs two dispatch cycles, so the design minimises exactly those:
//
//   * one thread owns one 128-bit run (4 words = 128 same-colour sites = one RNG unit G) and
//     MARCHES down R consecutive rows, keeping the opposite-colour rows i-1, i, i+1 in
//     registers: per row it loads 2 x 128 bits + 1 side word instead of 4 x 128 bits + 1;
//   * 5 LOP3 per word turn the four neighbour words into the two class masks
//       need = "dE > 0" (3 or 4 neighbours aligned),  c8 = "dE = 8" (all 4 aligned);
//   * the 8 acceptance bit-planes of unit G come from the folded Philox streams of philox.cuh
//     (16 instead of 20 multiplies per plane, the first rounds shared by the planes);
//   * the bit-serial compare "top byte of u32 < top byte of the lane's threshold" costs 2 LOP3
//     per word per plane: with tau = c8 ? bit_k(thr8) : bit_k(thr4),
//       acc <- MAJ(tau, ~b, acc)      eq <- eq & ~(b ^ tau)
//     are 3-input functions of (c8, b, acc) and (eq, b, c8) whose truth tables depend only on the
//     warp-uniform pair (bit_k(thr4), bit_k(thr8)): a 4-way brx.idx per plane picks the LOP3
//     immediates (inline PTX);
//   * the rare lanes whose top random byte ties with the threshold's (2^-8 per deciding lane)
//     are not resolved in place; the words that contain them are pushed (loop-free, one ballot
//     per word) into a per-warp queue in shared memory; whenever 32 entries are pending the
//     warp resolves them, one entry per thread (tail Philox block per tied lane), and applies the
//     accepted flips with a global atomic XOR on the already-stored word.
#pragma once
#include "ising.cuh"

namespace lat {

struct IsingMarchArgs {
    uint32_t *tgt;            // colour being updated   [L][wpr]
    const uint32_t *opp;      // opposite colour        [L][wpr]
    uint32_t L, wpr;          // L = rows allocated per colour (lattice side, or n_rows + 2 for a slab)
    // row-slab mode (all zero / null for a whole lattice):
    uint32_t row_off;         // local index of the first own row (1: local row 0 is a halo row)
    uint32_t g_off;           // added to the RNG unit index: (global row of local row 0) * (wpr/4)
    long long p_off;          // global minus local word offset, for the tail keying
    uint32_t *mir_up;         // where the first / last own row of tgt is mirrored: the neighbour
    uint32_t *mir_dn;         // slabs' halo rows (possibly peer-GPU memory), same [wpr] layout
    uint32_t t, colour;
    unsigned long long thr4, thr8;   // thresholds for dE = 4, 8 on the 2^64 scale (scheme 1: thr32 << 32):
                              // top byte -> pcase, low 56 bits -> compared with the 56 tail bits
    uint32_t mask4, mask8;    // 0 if the class flips unconditionally (threshold == 2^32), else ~0
    uint32_t pcase[8];        // plane k: bit_k(thr4) | bit_k(thr8) << 1, bit_k = bit (31-k)
    uint32_t R;               // rows per thread (even, divides L)
    uint32_t threads;         // (wpr/4) * (L/R), a multiple of 32
    PlaneFold F;              // folded ACC_PLANE stream of (t, colour)
    RoundKeys K;
    unsigned long long *rec;  // REC kernels: [REC_SLOTS][4] counters (anti-aligned x bonds, y bonds, up whites, up blacks)
};

constexpr int REC_SLOTS = 64;  // blocks spread their record atomics over this many counter sets

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

#ifdef __CUDACC__
// f(a, b, c) with the truth table LUT (bit (a<<2 | b<<1 | c)): one LOP3 where the compiler's own
// decomposition of a 3-input expression would take two or three
template <int LUT>
__device__ __forceinline__ uint32_t lop3(uint32_t a, uint32_t b, uint32_t c)
{
    uint32_t r;
    asm("lop3.b32 %0, %1, %2, %3, %4;" : "=r"(r) : "r"(a), "r"(b), "r"(c), "n"(LUT));
    return r;
}

// One plane of the bit-serial compare for the 4 words of a run (see the header comment).
// pcase = t4 | t8 << 1 (warp-uniform).  LOP3 truth tables, inputs (a, b, c) <-> (0xF0, 0xCC, 0xAA):
//   acc' = f(c8, b, acc):  tau = 0: ~b & acc = 0x22;  tau = ~c8: 0x2B;  tau = c8: 0xB2;  tau = 1: ~b | acc = 0xBB
//   eq'  = g(eq, b, c8):   tau = 0: eq & ~b = 0x30;   tau = ~c8: 0x60;  tau = c8: 0x90;  tau = 1: eq & b = 0xC0
#define LAT_PL(ta, te)                                                                            \
    "lop3.b32 %0, %8, %13, %0, " #ta "; lop3.b32 %1, %9, %14, %1, " #ta                           \
    "; lop3.b32 %2, %10, %15, %2, " #ta "; lop3.b32 %3, %11, %16, %3, " #ta                       \
    "; lop3.b32 %4, %4, %13, %8, " #te "; lop3.b32 %5, %5, %14, %9, " #te                         \
    "; lop3.b32 %6, %6, %15, %10, " #te "; lop3.b32 %7, %7, %16, %11, " #te "; bra PE;\n\t"

__device__ __forceinline__ void plane_compare(uint32_t pcase, const uint32_t (&c8)[4], const uint4 &b,
                                              uint32_t (&acc)[4], uint32_t (&eq)[4])
{
    asm("{\n\t"
        "pt: .branchtargets P0, P1, P2, P3;\n\t"
        "brx.idx %12, pt;\n\t"
        "P0: " LAT_PL(0x22, 0x30)
        "P1: " LAT_PL(0x2B, 0x60)
        "P2: " LAT_PL(0xB2, 0x90)
        "P3: " LAT_PL(0xBB, 0xC0)
        "PE:\n\t"
        "}"
        : "+r"(acc[0]), "+r"(acc[1]), "+r"(acc[2]), "+r"(acc[3]), "+r"(eq[0]), "+r"(eq[1]), "+r"(eq[2]), "+r"(eq[3])
        : "r"(c8[0]), "r"(c8[1]), "r"(c8[2]), "r"(c8[3]), "r"(pcase), "r"(b.x), "r"(b.y), "r"(b.z), "r"(b.w));
}
#undef LAT_PL

// Launch-time specialisation: the plane cases depend only on the top bytes of the two thresholds,
// i.e. on beta.  For the inverse temperatures the workloads actually run at (constant-beta runs are
// all of Table I; the two-step protocol has two values) the host picks a kernel
// instantiated with the packed cases PC = sum_k pcase[k] << 2k, where every LOP3 immediate is a
// compile-time constant and the eight brx.idx dispatches are gone.  PC < 0: the generic path above.
template <int PCASE>
__device__ __forceinline__ void plane_compare_fixed(const uint32_t (&c8)[4], const uint4 &b, uint32_t (&acc)[4],
                                                    uint32_t (&eq)[4])
{
    constexpr int TA = PCASE == 0 ? 0x22 : PCASE == 1 ? 0x2B : PCASE == 2 ? 0xB2 : 0xBB;
    constexpr int TE = PCASE == 0 ? 0x30 : PCASE == 1 ? 0x60 : PCASE == 2 ? 0x90 : 0xC0;
    const uint32_t bw[4] = {b.x, b.y, b.z, b.w};
#pragma unroll
    for (int w = 0; w < 4; ++w) {
        acc[w] = lop3<TA>(c8[w], bw[w], acc[w]);
        eq[w] = lop3<TE>(eq[w], bw[w], c8[w]);
    }
}

// planes K, K-1, ..., 0 (least significant plane first) of unit ps
template <int PC, int K>
struct PlaneLoop {
    template <class Args>
    static __device__ __forceinline__ void run(const Args &a, const PlaneShared &ps, const uint32_t (&c8)[4],
                                               uint32_t (&acc)[4], uint32_t (&eq)[4])
    {
        // fb[k] = fb[0] ^ (k << 16): the plane index enters as an immediate of the first XOR
        const uint4 b4 = plane_block(ps, a.F.fb[0] ^ ((uint32_t)K << 16), a.F, a.K);
        if constexpr (PC >= 0) plane_compare_fixed<(PC >> (2 * K)) & 3>(c8, b4, acc, eq);
        else plane_compare(a.pcase[K], c8, b4, acc, eq);
        if constexpr (K > 0) PlaneLoop<PC, K - 1>::run(a, ps, c8, acc, eq);
    }
};

// Per-warp queue of words that contain tied lanes.  One 128-bit entry per word:
//   x = the tied lanes of the word, y = which of them are class dE = 8, (z, w) = word offset.
// Pushing is loop-free (one ballot per word of the run); the bits of a word are only
// enumerated when the entry is resolved, 32 entries at a time, one entry per thread.  At most
// 31 entries are pending before a row and a row adds at most 4 x 32.
constexpr int TIE_Q_SLOTS = 160;

// REC (the fused r = 1 record of the white half-sweep, see march_row): a late flip changes the four
// bonds of its site, which the row has already counted with the unflipped value; the resolving thread
// re-reads the neighbour words (rare path) and keeps the differences in rx, ry, rm.
template <bool SLAB, bool REC = false>
struct WarpTieQueue {
    const IsingMarchArgs &a;
    uint4 *q;                  // [TIE_Q_SLOTS] this warp's slice
    uint32_t lane, pending;
    int rx, ry, rm;            // REC: corrections to the anti-aligned x / y bond counts and the up-white count

    // entry.w = word offset bits 32..35 | column word << 4 | mirror flag << 30 (1 = up, 2 = down)
    __device__ __forceinline__ void resolve(uint32_t idx)
    {
        const uint4 e = q[idx];
        const unsigned long long wo = ((unsigned long long)(e.w & 0xFu) << 32) | e.z;
        uint32_t ties = e.x, flip = 0;
        while (ties) {
            const uint32_t bit = __ffs(ties) - 1;
            ties &= ties - 1;
            const unsigned long long P = ((SLAB ? wo + a.p_off : wo) << 5) + bit;
            const uint4 blk = philox4x32_10((uint32_t)P, (uint32_t)(P >> 32), a.t,
                                            a.colour | (TAG_ACC_TAIL << 8), a.K);
            // low 56 bits: (tail word 0 >> 8) : tail word 1 against the threshold's (for scheme 1
            // the threshold's low word is 0, so word 1 never decides: u32 < thr32 exactly)
            const unsigned long long thr = ((e.y >> bit) & 1u) ? a.thr8 : a.thr4;
            const unsigned long long u56 = ((unsigned long long)(blk.x >> 8) << 32) | blk.y;
            if (u56 < (thr & 0x00ffffffffffffffull)) flip |= 1u << bit;
        }
        if (flip) {
            const uint32_t was = atomicXor(a.tgt + wo, flip);
            if constexpr (REC) {
                const uint32_t now = was ^ flip;
                const uint32_t row = (uint32_t)(wo / a.wpr), k = (uint32_t)(wo - (unsigned long long)row * a.wpr);
                const uint32_t *rp = a.opp + (unsigned long long)row * a.wpr;
                const uint32_t C = rp[k];
                const uint32_t U = a.opp[(unsigned long long)(row == 0 ? a.L - 1 : row - 1) * a.wpr + k];
                const uint32_t D = a.opp[(unsigned long long)(row + 1 == a.L ? 0 : row + 1) * a.wpr + k];
                const uint32_t S = ((row + a.colour) & 1u) == 0 ? fsl1(rp[k == 0 ? a.wpr - 1 : k - 1], C)
                                                                : fsr1(C, rp[k + 1 == a.wpr ? 0 : k + 1]);
                rx += __popc((now ^ C) & flip) + __popc((now ^ S) & flip) - __popc((was ^ C) & flip) - __popc((was ^ S) & flip);
                ry += __popc((now ^ U) & flip) + __popc((now ^ D) & flip) - __popc((was ^ U) & flip) - __popc((was ^ D) & flip);
                rm += __popc(now & flip) - __popc(was & flip);
            }
            const uint32_t mf = SLAB ? e.w >> 30 : 0u;
            if (mf) {
                // the mirror row may be peer-GPU memory: order this late flip after the plain
                // mirror store of the row (made by another lane of this warp) at system scope
                __threadfence_system();
                atomicXor_system((mf == 1 ? a.mir_up : a.mir_dn) + ((e.w >> 4) & 0x3ffffu), flip);
            }
        }
    }
    // collective over the warp: queue the words of this run that hold ties
    __device__ __forceinline__ void push(const uint32_t (&eq)[4], const uint32_t (&c8)[4], unsigned long long wo,
                                         uint32_t mir_tag)
    {
        const uint32_t below = (1u << lane) - 1u;
#pragma unroll
        for (int w = 0; w < 4; ++w) {
            const bool has = eq[w] != 0;
            const uint32_t m = __ballot_sync(0xffffffffu, has);
            if (has) {
                const unsigned long long o = wo + (unsigned)w;
                q[pending + __popc(m & below)] =
                    make_uint4(eq[w], c8[w], (uint32_t)o,
                               SLAB ? (uint32_t)(o >> 32) | (mir_tag + ((unsigned)w << 4)) : (uint32_t)(o >> 32));
            }
            pending += __popc(m);
        }
        __syncwarp();
        while (pending >= 32) {
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

// One row of one 128-bit run at word offset wo.  U, C, D: opposite-colour words of rows i-1, i,
// i+1 at the same packed position; E: the side word (PAR == 0: the word before the run,
// PAR == 1: the word after it).  Stores the updated words with every tie treated as a rejection
// and queues the ties.  EDGE: some class has threshold 2^32 (beta = 0): mask it out of `need`.
// mir / mir_tag: slab mode only -- where this row is mirrored (null: nowhere) and the queue tag
// (column word << 4 | flag << 30) that lets a late flip reach the mirror too.
// REC: what the fused r = 1 record of a thread adds up (march_row<.., REC = true>, white half-sweep)
struct RecAcc {
    uint32_t ax, ay, mw, mb;  // anti-aligned x bonds, y bonds, up spins of this colour, of the other colour
};

// REC = true (white half-sweep only): the row also counts the r = 1 record.  Every bond of the lattice
// joins one white and one black site, so summing over the white sites their two horizontal bonds
// (black words C and S) and two vertical bonds (U and D) counts every bond once: with the black rows
// final and the white word as stored, anti-aligned pairs of an axis = popc(n1 ^ n2) + 2 popc((T ^ n1) &
// (T ^ n2)); S_axis(1) = L^2 - 2 anti, M = 2 (up whites + up blacks) - L^2.  Per word 4 LOP3 + 1 SHF +
// 6 POPC: ~5 % of the half-sweep instead of a separate 24 ms pass over the lattice (Eq. 2-3,
// PAPER.md:42-50).  Late tie flips are corrected in WarpTieQueue::resolve.
template <int PAR, bool EDGE, bool SLAB, int PC = -1, bool REC = false, class Queue>
__device__ __forceinline__ void march_row(const IsingMarchArgs &a, uint32_t G, unsigned long long wo, uint32_t *tp,
                                          const uint4 &U4, const uint4 &C4, const uint4 &D4, uint32_t E,
                                          Queue &queue, uint32_t *mir = nullptr, uint32_t mir_tag = 0,
                                          RecAcc *rec = nullptr)
{
    const uint4 T4 = *reinterpret_cast<const uint4 *>(tp);       // tp == a.tgt + wo
    uint32_t T[4] = {T4.x, T4.y, T4.z, T4.w};
    const uint32_t U[4] = {U4.x, U4.y, U4.z, U4.w};
    const uint32_t C[4] = {C4.x, C4.y, C4.z, C4.w};
    const uint32_t D[4] = {D4.x, D4.y, D4.z, D4.w};
    uint32_t need[4], c8[4], acc[4], eq[4];
#pragma unroll
    for (int w = 0; w < 4; ++w) {
        uint32_t S;
        if (PAR == 0) S = fsl1(w == 0 ? E : C[w > 0 ? w - 1 : 0], C[w]);      // neighbour at p-1
        else S = fsr1(C[w], w == 3 ? E : C[w < 3 ? w + 1 : 0]);               // neighbour at p+1
        // "+1" neighbours: n = s1 + S + 2 c1;  aligned k = t ? n : 4 - n
        const uint32_t s1 = U[w] ^ D[w] ^ C[w];
        const uint32_t c1 = maj3m(U[w], D[w], C[w]);
        const uint32_t t = T[w];
        // k >= 3:  t = 1: c1 & (s1 | S);   t = 0: ~c1 & ~(s1 & S)
        const uint32_t m = lop3<0xE7>(t, s1, S);         // (t & (s1 | S)) | (~t & ~(s1 & S))
        uint32_t nd = lop3<0x82>(c1, t, m);              // ~(c1 ^ t) & m
        uint32_t k4 = lop3<0x90>(nd, s1, S);             // nd & ~(s1 ^ S): k == 4
        if (EDGE) {
            // classes whose threshold is 2^32 flip unconditionally: drop them from need
            const uint32_t k3 = nd & ~k4;
            nd = (k3 & a.mask4) | (k4 & a.mask8);
            k4 &= a.mask8;
        }
        need[w] = nd; c8[w] = k4; eq[w] = nd; acc[w] = 0;
    }
    // top byte of u32(site) against the top byte of the lane's threshold, least significant
    // plane first
    const PlaneShared ps = plane_shared(G, a.F);
    PlaneLoop<PC, 7>::run(a, ps, c8, acc, eq);
    // lanes outside need flip unconditionally (dE <= 0); a tied lane has acc = 0 and stays put
#pragma unroll
    for (int w = 0; w < 4; ++w) T[w] = lop3<0x4B>(T[w], need[w], acc[w]);    // T ^ (~need | acc)
    *reinterpret_cast<uint4 *>(tp) = make_uint4(T[0], T[1], T[2], T[3]);
    if constexpr (REC) {
#pragma unroll
        for (int w = 0; w < 4; ++w) {
            uint32_t S;
            if (PAR == 0) S = fsl1(w == 0 ? E : C[w > 0 ? w - 1 : 0], C[w]);
            else S = fsr1(C[w], w == 3 ? E : C[w < 3 ? w + 1 : 0]);
            rec->ax += __popc(C[w] ^ S) + 2u * __popc(lop3<0x18>(T[w], C[w], S));      // (T ^ C) & (T ^ S)
            rec->ay += __popc(U[w] ^ D[w]) + 2u * __popc(lop3<0x18>(T[w], U[w], D[w]));
            rec->mw += __popc(T[w]);
            rec->mb += __popc(C[w]);
        }
    }
    if (SLAB && mir) {
        *reinterpret_cast<uint4 *>(mir) = make_uint4(T[0], T[1], T[2], T[3]);
        __threadfence_system();      // before any late flip of this row (resolve) reaches the mirror
    }
    queue.push(eq, c8, wo, mir_tag);
}

// The march of one thread: rows i0 .. i0+R-1 of run q, g = s * (wpr/4) + q (ties are queued, not
// drained).
template <int COLOUR, bool EDGE, bool SLAB, int PC = -1, bool REC = false, class Queue>
__device__ __forceinline__ void march_thread(const IsingMarchArgs &a, uint32_t g, Queue &queue, RecAcc *rec = nullptr)
{
    const uint32_t L = a.L, wpr = a.wpr, nq = wpr >> 2;
    const uint32_t q = g % nq, s = g / nq;
    const uint32_t kw = q << 2;
    const uint32_t i0 = s * a.R + (SLAB ? a.row_off : 0u);
    const uint32_t iu = (i0 == 0) ? L - 1 : i0 - 1;
    // side words: PAR == 0 reads the word before the run, PAR == 1 the word after it (periodic)
    const uint32_t ke0 = (kw == 0) ? wpr - 1 : kw - 1;
    const uint32_t ke1 = (kw + 4 == wpr) ? 0 : kw + 4;

    const unsigned long long ro = (unsigned long long)i0 * wpr;      // word offset of row i0
    uint4 U = *reinterpret_cast<const uint4 *>(a.opp + (unsigned long long)iu * wpr + kw);
    uint4 C = *reinterpret_cast<const uint4 *>(a.opp + ro + kw);
    uint32_t G = i0 * nq + q + (SLAB ? a.g_off : 0u);                // (global i*(L/2) + 32 kw) >> 7
    // slab mode: the first own row is mirrored into the upper neighbour's halo, the last into the
    // lower neighbour's (this slab's own halos when it is the only one)
    const bool top = SLAB && s == 0, bot = SLAB && (s + 1) * nq == a.threads;
    // running pointers: the slab's own rows never wrap; only row i+1 of the last lattice row does
    const uint32_t *op = a.opp + ro;                                 // row i of the opposite colour
    uint32_t *tp = a.tgt + ro + kw;                                  // this run in row i
    unsigned long long wo = ro + kw;
    uint32_t left = L - i0;                                          // rows from i to the lattice end

    for (uint32_t r = 0; r < a.R; r += 2) {
        {   // row i0 + r: (i + colour) & 1 == COLOUR because i0 and r are even
            const uint32_t *dn = op + wpr;                           // row i + 1 (left >= 2 here)
            const uint4 D = *reinterpret_cast<const uint4 *>(dn + kw);
            const uint32_t E = op[COLOUR == 0 ? ke0 : ke1];
            if (SLAB && top && r == 0)
                march_row<COLOUR, EDGE, SLAB, PC>(a, G, wo, tp, U, C, D, E, queue, a.mir_up + kw, (kw << 4) | (1u << 30));
            else
                march_row<COLOUR, EDGE, SLAB, PC, REC>(a, G, wo, tp, U, C, D, E, queue, nullptr, 0, rec);
            U = C; C = D; op = dn; tp += wpr; wo += wpr; G += nq;
        }
        {   // row i0 + r + 1: the other parity; its row i + 1 wraps to row 0 at the lattice end
            left -= 2;
            const uint32_t *dn = left ? op + wpr : a.opp;
            const uint4 D = *reinterpret_cast<const uint4 *>(dn + kw);
            const uint32_t E = op[COLOUR == 0 ? ke1 : ke0];
            if (SLAB && bot && r + 2 == a.R)
                march_row<COLOUR ^ 1, EDGE, SLAB, PC>(a, G, wo, tp, U, C, D, E, queue, a.mir_dn + kw, (kw << 4) | (2u << 30));
            else
                march_row<COLOUR ^ 1, EDGE, SLAB, PC, REC>(a, G, wo, tp, U, C, D, E, queue, nullptr, 0, rec);
            U = C; C = D; op = dn; tp += wpr; wo += wpr; G += nq;
        }
    }
}

// One row per thread, for lattices too small to fill the GPU with marching threads (there the
// time of a half-sweep is the latency of ONE thread's rows, so fewer rows per thread is faster
// even though every thread now loads all three neighbour rows itself).  g enumerates
// (row slot s, run q) with the even rows first and the odd rows after them, so that every warp
// works on rows of one parity (wpr/4 * L/2 is a multiple of 32) and the branch is warp-uniform.
template <int COLOUR, bool EDGE, class Queue>
__device__ __forceinline__ void row_thread(const IsingMarchArgs &a, uint32_t g, Queue &queue)
{
    const uint32_t L = a.L, wpr = a.wpr, nq = wpr >> 2, half = L >> 1;
    const uint32_t q = g % nq, s = g / nq;
    const uint32_t i = s < half ? 2u * s : 2u * (s - half) + 1u;
    const uint32_t kw = q << 2;
    const uint32_t iu = (i == 0) ? L - 1 : i - 1, id = (i + 1 == L) ? 0 : i + 1;
    const unsigned long long ro = (unsigned long long)i * wpr;
    const uint4 U = *reinterpret_cast<const uint4 *>(a.opp + (unsigned long long)iu * wpr + kw);
    const uint4 C = *reinterpret_cast<const uint4 *>(a.opp + ro + kw);
    const uint4 D = *reinterpret_cast<const uint4 *>(a.opp + (unsigned long long)id * wpr + kw);
    const uint32_t G = i * nq + q;
    if (((i + COLOUR) & 1u) == 0) {
        const uint32_t E = a.opp[ro + ((kw == 0) ? wpr - 1 : kw - 1)];
        march_row<0, EDGE, false>(a, G, ro + kw, a.tgt + ro + kw, U, C, D, E, queue);
    } else {
        const uint32_t E = a.opp[ro + ((kw + 4 == wpr) ? 0 : kw + 4)];
        march_row<1, EDGE, false>(a, G, ro + kw, a.tgt + ro + kw, U, C, D, E, queue);
    }
}

template <int COLOUR, bool EDGE>
__global__ void __launch_bounds__(256) ising_row_kernel(const IsingMarchArgs a)
{
    __shared__ uint4 s_q[8][TIE_Q_SLOTS];
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const uint32_t g = blockIdx.x * 256u + threadIdx.x;
    if (g - lane >= a.threads) return;          // a.threads = wpr/4 * L, a multiple of 32
    WarpTieQueue<false> queue{a, s_q[warp], lane, 0u};
    row_thread<COLOUR, EDGE>(a, g, queue);
    queue.drain();
}

// The plane-case values with a specialised instantiation (host side: ising_pc_index):
//   0xF910  beta_c = ln(1 + sqrt 2)/2: thr4 = 0x2B......, thr8 = 0x07......  (BASELINE configs 1, 2, 4)
//   0x7440  T_1 = 1.66 of the paper's two-step protocol (Table II)
//   0xAD10  T_2 = 2.27414861561203 of the same protocol, and beta_c/1.01 (plateau of config 5a)
#define LAT_ISING_PC_LIST(X) X(0xF910) X(0x7440) X(0xAD10)

template <int COLOUR, bool EDGE, bool SLAB, int PC = -1, bool REC = false>
__global__ void __launch_bounds__(256) ising_march_kernel(const IsingMarchArgs a)
{
    __shared__ uint4 s_q[8][TIE_Q_SLOTS];
    __shared__ unsigned int s_rec[4];
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const uint32_t g = blockIdx.x * 256u + threadIdx.x;
    if constexpr (REC) {
        if (threadIdx.x < 4) s_rec[threadIdx.x] = 0;
        __syncthreads();
    }
    if (g - lane >= a.threads) return;          // a.threads is a multiple of 32: whole warps only
    WarpTieQueue<SLAB, REC> queue{a, s_q[warp], lane, 0u};
    RecAcc rec{0u, 0u, 0u, 0u};
    march_thread<COLOUR, EDGE, SLAB, PC, REC>(a, g, queue, &rec);
    queue.drain();
    if constexpr (REC) {
        // thread -> warp (REDUX) -> block (shared atomics) -> one of REC_SLOTS counter sets; a thread's
        // sums may be "negative" (it only corrected late flips of other threads' rows): the sums are
        // modulo 2^32 and a warp's total is the exact count of its own rows
        const uint32_t v[4] = {__reduce_add_sync(0xffffffffu, rec.ax + (uint32_t)queue.rx),
                               __reduce_add_sync(0xffffffffu, rec.ay + (uint32_t)queue.ry),
                               __reduce_add_sync(0xffffffffu, rec.mw + (uint32_t)queue.rm),
                               __reduce_add_sync(0xffffffffu, rec.mb)};
        if (lane == 0) {
#pragma unroll
            for (int k = 0; k < 4; ++k) atomicAdd(&s_rec[k], v[k]);
        }
        __syncthreads();                        // warps that returned above have exited: they do not count
        if (threadIdx.x < 4)
            atomicAdd(a.rec + (blockIdx.x % REC_SLOTS) * 4u + threadIdx.x, (unsigned long long)s_rec[threadIdx.x]);
    }
}
#endif

}  // namespace lat
