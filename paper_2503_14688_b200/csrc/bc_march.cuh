// bc_march.cuh -- the production Blume-Capel half-sweep (RNG scheme 1, L a multiple of 256,
// threshold tables with the "integer dE" structure that Delta = 0 gives).
//
// Paper: Eq. 1 with crystal field Delta; every run of the paper uses
// Delta = 0.  Metropolis + checkerboard + multispin coding,
// 32-bit acceptance compare.  Same packing, neighbour geometry, proposal rule and
// acceptance rule as bc.cuh, which stays as the generic path (any Delta, scheme 0, narrow rows).
//
// With r the per-lane reference sign of bc.cuh and x = (#neighbours of sign r) - (#of sign -r),
// the move types cost dE = 2x (flip), x - Delta (vacate), x + Delta (occupy).  When the host
// finds that every entry with x <= 0 is "always" and vacate/occupy share their thresholds for
// x = 1..4 (true for Delta = 0 at any beta), a lane that needs a random decision is in one of
// 8 classes (F, x) with F = flip and x = 1..4, i.e. 3 bits per lane:
//     F = flip,   Y1 = (x >= 3),   H0 = (x odd)
// and bit k of the lane's threshold is a 3-input boolean function of those bits -- exactly one
// LOP3 whose truth table (8 bits per plane) the host derives from the threshold table.  LOP3's
// truth table is an immediate, so the kernel dispatches once per plane (warp-uniform, 256-way
// jump table) to the LOP3 with the right immediate.  This replaces ~90 LOP3 per word of class
// selection in bc.cuh by 1 per word per plane.
//
// Work layout as in ising_march.cuh: one thread owns a 128-bit run and marches down R rows with
// the opposite-colour rows i-1, i, i+1 in registers; folded Philox bit-planes; ties (top byte of
// u32 equal to the top byte of the lane's threshold) are queued per warp, one entry per word that
// holds ties, and resolved 32 entries at a time, accepted late moves applied with global atomic XORs.
#pragma once
#include "bc.cuh"
#include "ising_march.cuh"

namespace lat {

struct BCMarchArgs {
    uint32_t *tnz, *tsg;            // colour being updated
    const uint32_t *onz, *osg;      // opposite colour
    uint32_t L, wpr, t, colour;     // L = rows allocated per plane (lattice side, or n_rows + 2 for a slab)
    // row-slab mode (same meaning as in IsingMarchArgs; zero / null for a whole lattice)
    uint32_t row_off, g_off;
    long long p_off;
    uint32_t *mir_up_nz, *mir_up_sg, *mir_dn_nz, *mir_dn_sg;
    uint32_t R;                     // rows per thread (even, divides L)
    uint32_t threads;               // (wpr/4) * (L/R), a multiple of 32
    uint32_t lut[8];                // truth table of threshold bit (31-k) over (F, Y1, H0)
    uint32_t lut_always;            // truth table of "threshold == 2^32" over (F, Y1, H0)
    unsigned long long thr[8];      // threshold of class (F<<2 | Y1<<1 | H0) on the 2^64 scale (scheme 1:
                                    // thr32 << 32); the low 56 bits are compared with the 56 tail bits
    // general crystal field (GEN kernels; Delta != 0): per move type an 8-entry table indexed by
    // idx = (hA << 2 | h1 << 1 | h0) of the lane's x + 4 (hA = h3 for flips, h2 otherwise; see
    // bc_march_row_gen): truth tables of threshold bit (63-k) and of "always", thresholds for ties
    // Table A serves the flips (idx 1..4) and the one of vacate / occupy whose x <= 0 entries are all
    // "always" (idx 5, 6, 7, 0 for x = 1..4): vacate for Delta >= 0 (share_v = 1), occupy otherwise;
    // table B serves the other type (all eight idx).
    uint32_t lutA[8], lutB[8];
    uint32_t lutA_always, lutB_always;
    uint32_t share_v;
    unsigned long long thrG[24];    // [type 0 flip, 1 vacate, 2 occupy][idx]
    uint32_t fbp;                   // folded counter word of the PROP plane
    PlaneFold F;                    // folded ACC_PLANE stream of (t, colour)
    RoundKeys K;
#ifdef __CUDACC__
    // truth table of plane k (a runtime index: a kernel parameter is read from the constant bank;
    // bc_persist.cuh overrides this with a shared-memory read)
    __device__ __forceinline__ uint32_t lut_k(int k) const { return lut[k]; }
#endif
};

// out[w] = f(a[w], b[w], c[w]), w = 0..3, with f given by the runtime truth table `lut` (LOP3
// convention: bit (a<<2 | b<<1 | c) of lut).  One PTX block: a 256-entry jump table (brx.idx)
// into 256 groups of four LOP3 with the truth table as immediate.  Labels are scoped by the
// braces, so the block can be inlined more than once.  lut should be warp-uniform.
#define LAT_LC(h, l)                                                                              \
    "L" #h #l ": lop3.b32 %0, %4, %8, %13, 0x" #h #l "; lop3.b32 %1, %5, %9, %14, 0x" #h #l       \
    "; lop3.b32 %2, %6, %10, %15, 0x" #h #l "; lop3.b32 %3, %7, %11, %16, 0x" #h #l "; bra LE;\n\t"
#define LAT_LR(h)                                                                                 \
    LAT_LC(h, 0) LAT_LC(h, 1) LAT_LC(h, 2) LAT_LC(h, 3) LAT_LC(h, 4) LAT_LC(h, 5) LAT_LC(h, 6)    \
    LAT_LC(h, 7) LAT_LC(h, 8) LAT_LC(h, 9) LAT_LC(h, a) LAT_LC(h, b) LAT_LC(h, c) LAT_LC(h, d)    \
    LAT_LC(h, e) LAT_LC(h, f)
#define LAT_TR(h)                                                                                 \
    "L" #h "0, L" #h "1, L" #h "2, L" #h "3, L" #h "4, L" #h "5, L" #h "6, L" #h "7, L" #h        \
    "8, L" #h "9, L" #h "a, L" #h "b, L" #h "c, L" #h "d, L" #h "e, L" #h "f"

__device__ __forceinline__ void lut3_dispatch(uint32_t lut, const uint32_t (&a)[4], const uint32_t (&b)[4],
                                              const uint32_t (&c)[4], uint32_t (&out)[4])
{
    asm("{\n\t"
        "ts: .branchtargets " LAT_TR(0) ", " LAT_TR(1) ", " LAT_TR(2) ", " LAT_TR(3) ", " LAT_TR(4) ", "
        LAT_TR(5) ", " LAT_TR(6) ", " LAT_TR(7) ", " LAT_TR(8) ", " LAT_TR(9) ", " LAT_TR(a) ", "
        LAT_TR(b) ", " LAT_TR(c) ", " LAT_TR(d) ", " LAT_TR(e) ", " LAT_TR(f) ";\n\t"
        "brx.idx %12, ts;\n\t"
        LAT_LR(0) LAT_LR(1) LAT_LR(2) LAT_LR(3) LAT_LR(4) LAT_LR(5) LAT_LR(6) LAT_LR(7)
        LAT_LR(8) LAT_LR(9) LAT_LR(a) LAT_LR(b) LAT_LR(c) LAT_LR(d) LAT_LR(e) LAT_LR(f)
        "LE:\n\t"
        "}"
        : "=r"(out[0]), "=r"(out[1]), "=r"(out[2]), "=r"(out[3])
        : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b[0]), "r"(b[1]), "r"(b[2]), "r"(b[3]),
          "r"(lut & 0xffu), "r"(c[0]), "r"(c[1]), "r"(c[2]), "r"(c[3]));
}

#undef LAT_LC
#undef LAT_LR
#undef LAT_TR

// Launch-time specialisation (as for the Ising kernel, ising_march.cuh): the eight per-plane truth
// tables depend only on the top bytes of the eight class thresholds, i.e. on beta.  For the
// temperatures the workloads run at, LS >= 0 selects a set of tables compiled in: every dispatched
// LOP3 becomes a LOP3 with an immediate, the eight 256-way brx.idx jumps are gone and the plane loop is
// unrolled.  All sets have lut_always == 0 (no class threshold is 2^32).  LS < 0: the generic path.
//   0: T = 1.6934 (BASELINE config 3), T_c = 1.69355839821214427 (Table I) and
//      T_2 = 1.69661396797728 of the two-step protocol (Table II)
//   1: beta = (1/1.6934)/1.01, the plateau of BASELINE config 5b's ramp
//   2: T_1 = 1.24 of the two-step protocol
constexpr int BC_LUT_SETS = 3;
__host__ __device__ constexpr uint32_t bc_lut_set(int ls, int k)
{
    constexpr uint32_t T[BC_LUT_SETS][8] = {{0x02, 0x21, 0x08, 0x14, 0x3f, 0xa3, 0xe9, 0x8a},
                                            {0x02, 0x21, 0x08, 0x14, 0x3f, 0xab, 0xe3, 0xa1},
                                            {0x00, 0x02, 0x23, 0x2b, 0x14, 0x08, 0xbf, 0x21}};
    return T[ls][k];
}

#ifdef __CUDACC__
// planes K, K-1, ..., 0 with the truth tables of set LS as LOP3 immediates
template <int LS, int K>
struct BCPlaneLoop {
    template <class Args>
    static __device__ __forceinline__ void run(const Args &a, const PlaneShared &ps, const uint32_t (&Fm)[4],
                                               const uint32_t (&Y1)[4], const uint32_t (&H0)[4],
                                               uint32_t (&acc)[4], uint32_t (&eq)[4])
    {
        const uint4 b4 = plane_block(ps, a.F.fb[0] ^ ((uint32_t)K << 16), a.F, a.K);
        const uint32_t b[4] = {b4.x, b4.y, b4.z, b4.w};
        constexpr int LUT = (int)bc_lut_set(LS, K);
#pragma unroll
        for (int w = 0; w < 4; ++w) {
            const uint32_t tau = LUT == 0 ? 0u : lop3<LUT>(Fm[w], Y1[w], H0[w]);
            acc[w] = maj3m(tau, ~b[w], acc[w]);
            eq[w] &= ~(b[w] ^ tau);
        }
        if constexpr (K > 0) BCPlaneLoop<LS, K - 1>::run(a, ps, Fm, Y1, H0, acc, eq);
    }
};
#endif

// Per-warp queue of words that contain tied lanes (same scheme as WarpTieQueue in
// ising_march.cuh).  Two 128-bit halves per entry:
//   [0] = (tied lanes, F, Y1, H0 of the word)    [1] = (nz-toggle mask, sg-toggle mask, word offset)
// Pushing is loop-free (one ballot per word); the tied lanes of a word are enumerated when the
// entry is resolved, 32 entries at a time, one entry per thread.
template <bool SLAB>
struct BCTieQueue {
    const BCMarchArgs &a;
    uint4 *q;                   // [2 * TIE_Q_SLOTS] this warp's slice
    uint32_t lane, pending;

    // e1.w = word offset bits 32..35 | column word << 4 | mirror flag << 30 (1 = up, 2 = down)
    __device__ __forceinline__ void resolve(uint32_t idx)
    {
        const uint4 e0 = q[2 * idx], e1 = q[2 * idx + 1];
        const unsigned long long wo = ((unsigned long long)(e1.w & 0xFu) << 32) | e1.z;
        uint32_t ties = e0.x, hit = 0;
        while (ties) {
            const uint32_t bit = __ffs(ties) - 1;
            ties &= ties - 1;
            const uint32_t cls = (((e0.y >> bit) & 1u) << 2) | (((e0.z >> bit) & 1u) << 1) | ((e0.w >> bit) & 1u);
            const unsigned long long P = ((SLAB ? wo + a.p_off : wo) << 5) + bit;
            const uint4 blk = philox4x32_10((uint32_t)P, (uint32_t)(P >> 32), a.t,
                                            a.colour | (TAG_ACC_TAIL << 8), a.K);
            const unsigned long long u56 = ((unsigned long long)(blk.x >> 8) << 32) | blk.y;
            if (u56 < (a.thr[cls] & 0x00ffffffffffffffull)) hit |= 1u << bit;
        }
        const uint32_t dnz = hit & e1.x, dsg = hit & e1.y;
        if (dnz) atomicXor(a.tnz + wo, dnz);
        if (dsg) atomicXor(a.tsg + wo, dsg);
        const uint32_t mf = SLAB ? e1.w >> 30 : 0u;
        if (mf && (dnz | dsg)) {
            // possibly peer-GPU memory: system-scope atomics, ordered after the row's mirror store
            const uint32_t col = (e1.w >> 4) & 0x3ffffu;
            __threadfence_system();
            if (dnz) atomicXor_system((mf == 1 ? a.mir_up_nz : a.mir_dn_nz) + col, dnz);
            if (dsg) atomicXor_system((mf == 1 ? a.mir_up_sg : a.mir_dn_sg) + col, dsg);
        }
    }
    __device__ __forceinline__ void push(const uint32_t (&eq)[4], const uint32_t (&Fm)[4], const uint32_t (&Y1)[4],
                                         const uint32_t (&H0)[4], const uint32_t (&nf)[4],
                                         const uint32_t (&gg)[4], unsigned long long wo, uint32_t mir_tag)
    {
        const uint32_t below = (1u << lane) - 1u;
#pragma unroll
        for (int w = 0; w < 4; ++w) {
            const bool has = eq[w] != 0;
            const uint32_t m = __ballot_sync(0xffffffffu, has);
            if (has) {
                const unsigned long long o = wo + (unsigned)w;
                const uint32_t slot = pending + __popc(m & below);
                q[2 * slot] = make_uint4(eq[w], Fm[w], Y1[w], H0[w]);
                q[2 * slot + 1] = make_uint4(nf[w], gg[w], (uint32_t)o,
                                             SLAB ? (uint32_t)(o >> 32) | (mir_tag + ((unsigned)w << 4))
                                                  : (uint32_t)(o >> 32));
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

struct BCRow {
    uint32_t nz[4], sg[4];
};

__device__ __forceinline__ void bcm_load(const uint32_t *nzp, const uint32_t *sgp, unsigned long long off, BCRow &v)
{
    const uint4 x = *reinterpret_cast<const uint4 *>(nzp + off);
    const uint4 y = *reinterpret_cast<const uint4 *>(sgp + off);
    v.nz[0] = x.x; v.nz[1] = x.y; v.nz[2] = x.z; v.nz[3] = x.w;
    v.sg[0] = y.x; v.sg[1] = y.y; v.sg[2] = y.z; v.sg[3] = y.w;
}

// One row of one 128-bit run.  PAR == 0: side neighbour at p-1 (En, Es = word before the run),
// PAR == 1: at p+1 (word after it).  Stores the updated words (ties treated as rejections) and
// queues the ties.
template <int PAR, bool SLAB, int LS, class Args>
__device__ __forceinline__ void bc_march_row(const Args &a, uint32_t G, unsigned long long wo,
                                             uint32_t *tn, uint32_t *ts,
                                             const BCRow &U, const BCRow &C, const BCRow &D,
                                             uint32_t En, uint32_t Es, BCTieQueue<SLAB> &queue,
                                             uint32_t *mir_nz = nullptr, uint32_t *mir_sg = nullptr,
                                             uint32_t mir_tag = 0)
{
    BCRow T;
    bcm_load(tn, ts, 0, T);                                       // tn == a.tnz + wo, ts == a.tsg + wo
    const PlaneShared ps = plane_shared(G, a.F);
    uint32_t Fm[4], Y1[4], H0[4], pos[4], nf[4], gg[4];
    {
        const uint4 pb = plane_block(ps, a.fbp, a.F, a.K);        // proposal bits
        const uint32_t b[4] = {pb.x, pb.y, pb.z, pb.w};
#pragma unroll
        for (int w = 0; w < 4; ++w) {
            uint32_t Sn, Ss;
            if (PAR == 0) {
                Sn = fsl1(w == 0 ? En : C.nz[w > 0 ? w - 1 : 0], C.nz[w]);
                Ss = fsl1(w == 0 ? Es : C.sg[w > 0 ? w - 1 : 0], C.sg[w]);
            } else {
                Sn = fsr1(C.nz[w], w == 3 ? En : C.nz[w < 3 ? w + 1 : 0]);
                Ss = fsr1(C.sg[w], w == 3 ? Es : C.sg[w < 3 ? w + 1 : 0]);
            }
            const uint32_t nz = T.nz[w], sg = T.sg[w], bw = b[w];
            Fm[w] = lop3<0x90>(nz, sg, bw);                       // flip: nz & ~(sg ^ b)
            nf[w] = ~Fm[w];                                       // nz toggles unless the move is a flip
            // sg toggles on flip, vacate of -1, occupy to -1: Fm | (nz & sg & ~b) | (~nz & b)
            gg[w] = lop3<0xDA>(nz, sg, bw);
            const uint32_t r = lop3<0xC5>(nz, sg, bw);            // (nz & sg) | (~nz & ~b)
            // x + 4 = sum over the 4 neighbours of [sign r] + [not sign -r], bit-sliced
            // explicit truth tables (inputs nz, sg, r): [sign r] = nz & ~(sg ^ r) = 0x90,
            // [not sign -r] = ~(nz & (sg ^ r)) = 0x9F; adders: xor3 = 0x96, majority = 0xE8
            const uint32_t a1 = lop3<0x90>(U.nz[w], U.sg[w], r), n1 = lop3<0x9F>(U.nz[w], U.sg[w], r);
            const uint32_t a2 = lop3<0x90>(D.nz[w], D.sg[w], r), n2 = lop3<0x9F>(D.nz[w], D.sg[w], r);
            const uint32_t a3 = lop3<0x90>(C.nz[w], C.sg[w], r), n3 = lop3<0x9F>(C.nz[w], C.sg[w], r);
            const uint32_t a4 = lop3<0x90>(Sn, Ss, r), n4 = lop3<0x9F>(Sn, Ss, r);
            const uint32_t s1 = lop3<0x96>(a1, a2, a3), c1 = lop3<0xE8>(a1, a2, a3);
            const uint32_t s2 = lop3<0x96>(n1, n2, n3), c2 = lop3<0xE8>(n1, n2, n3);
            const uint32_t s3 = lop3<0x96>(s1, s2, a4), c3 = lop3<0xE8>(s1, s2, a4);
            const uint32_t h0 = s3 ^ n4, c4 = s3 & n4;            // weight 1 done
            const uint32_t t1 = lop3<0x96>(c1, c2, c3), d1 = lop3<0xE8>(c1, c2, c3);
            const uint32_t h1 = t1 ^ c4, d2 = t1 & c4;            // weight 2 done
            const uint32_t h2 = d1 ^ d2, h3 = d1 & d2;            // weights 4, 8
            H0[w] = h0;
            Y1[w] = lop3<0xF8>(h3, h1, h0);                       // h3 | (h1 & h0): x >= 3  (x+4 in {7, 8})
            pos[w] = h3 | lop3<0xE0>(h2, h1, h0);                 // h3 | (h2 & (h1 | h0)): x >= 1
        }
    }
    uint32_t alw[4], acc[4], eq[4];
    if constexpr (LS >= 0) { alw[0] = alw[1] = alw[2] = alw[3] = 0u; }      // the sets have lut_always == 0
    else lut3_dispatch(a.lut_always, Fm, Y1, H0, alw);
#pragma unroll
    for (int w = 0; w < 4; ++w) {
        const uint32_t need = pos[w] & ~alw[w];
        alw[w] = ~need;                                           // x <= 0, or threshold 2^32
        pos[w] = need;
        eq[w] = need;
        acc[w] = 0;
    }
    if constexpr (LS >= 0) {
        BCPlaneLoop<LS, 7>::run(a, ps, Fm, Y1, H0, acc, eq);
    } else {
#pragma unroll 1                     // unrolling replicates the 256-entry tables: slower (I-cache)
        for (int k = 7; k >= 0; --k) {
            const uint4 b4 = plane_block(ps, a.F.fb[0] ^ ((uint32_t)k << 16), a.F, a.K);
            const uint32_t b[4] = {b4.x, b4.y, b4.z, b4.w};
            uint32_t tau[4];
            lut3_dispatch(a.lut_k(k), Fm, Y1, H0, tau);
#pragma unroll
            for (int w = 0; w < 4; ++w) {
                acc[w] = maj3m(tau[w], ~b[w], acc[w]);
                eq[w] &= ~(b[w] ^ tau[w]);
            }
        }
    }
#pragma unroll
    for (int w = 0; w < 4; ++w) {
        const uint32_t ok = alw[w] | (acc[w] & pos[w]);           // a tied lane has acc = 0
        T.nz[w] ^= ok & nf[w];
        T.sg[w] ^= ok & gg[w];
    }
    *reinterpret_cast<uint4 *>(tn) = make_uint4(T.nz[0], T.nz[1], T.nz[2], T.nz[3]);
    *reinterpret_cast<uint4 *>(ts) = make_uint4(T.sg[0], T.sg[1], T.sg[2], T.sg[3]);
    if (SLAB && mir_nz) {       // slab mode: this row is also a neighbour's halo row
        *reinterpret_cast<uint4 *>(mir_nz) = make_uint4(T.nz[0], T.nz[1], T.nz[2], T.nz[3]);
        *reinterpret_cast<uint4 *>(mir_sg) = make_uint4(T.sg[0], T.sg[1], T.sg[2], T.sg[3]);
        __threadfence_system();
    }
    queue.push(eq, Fm, Y1, H0, nf, gg, wo, mir_tag);
}

// ---- any crystal field Delta (|Delta| <= 4) -------------------------------------------------------
//
// For Delta != 0 vacate (dE = x - Delta) and occupy (dE = x + Delta) no longer share thresholds and
// x <= 0 is no longer "always" for them (Eq. 1), so a deciding lane is in one of up
// to 4 + 8 + 8 classes.  Per move type the threshold bit of plane k is still a function of three
// bits of the bit-sliced x + 4 = (h3 h2 h1 h0):
//   flip   : only x = 1..4 can need a decision; (h3, h1, h0) tells 5, 6, 7, 8 apart;
//   vacate / occupy : x = -3..4 <-> (x + 4) & 7 = (h2, h1, h0), with x = 4 on index 0 -- legal when
//            x = -4 is "always" for both (true for |Delta| <= 4; the host checks the table and
//            falls back to the generic kernel otherwise).
// With hA = flip ? h3 : h2 every table takes the same inputs (hA, h1, h0).  Two tables suffice: for
// Delta >= 0 a vacate with x <= 0 is always accepted (dE = x - Delta <= 0), so its deciding entries
// x = 1..4 sit on idx 5, 6, 7, 0 and share table A with the flips (idx 1..4), while occupy owns table
// B; for Delta < 0 vacate and occupy swap roles.  Per word per plane: two dispatched LOP3, one select
// by table, then the same two-LOP3 compare as before.
template <bool SLAB>
struct BCTieQueueGen {
    const BCMarchArgs &a;
    uint4 *q;                   // [3 * TIE_Q_SLOTS] this warp's slice
    uint32_t lane, pending;

    // [0] = (tied lanes, F, V, hA)   [1] = (h1, h0, nz-toggle mask, sg-toggle mask)
    // [2] = (word offset lo, bits 32..35 | column word << 4 | mirror flag << 30, -, -)
    __device__ __forceinline__ void resolve(uint32_t idx)
    {
        const uint4 e0 = q[3 * idx], e1 = q[3 * idx + 1], e2 = q[3 * idx + 2];
        const unsigned long long wo = ((unsigned long long)(e2.y & 0xFu) << 32) | e2.x;
        uint32_t ties = e0.x, hit = 0;
        while (ties) {
            const uint32_t bit = __ffs(ties) - 1;
            ties &= ties - 1;
            const uint32_t type = ((e0.y >> bit) & 1u) ? 0u : ((e0.z >> bit) & 1u) ? 1u : 2u;
            const uint32_t i3 = (((e0.w >> bit) & 1u) << 2) | (((e1.x >> bit) & 1u) << 1) | ((e1.y >> bit) & 1u);
            const unsigned long long P = ((SLAB ? wo + a.p_off : wo) << 5) + bit;
            const uint4 blk = philox4x32_10((uint32_t)P, (uint32_t)(P >> 32), a.t,
                                            a.colour | (TAG_ACC_TAIL << 8), a.K);
            const unsigned long long u56 = ((unsigned long long)(blk.x >> 8) << 32) | blk.y;
            if (u56 < (a.thrG[type * 8u + i3] & 0x00ffffffffffffffull)) hit |= 1u << bit;
        }
        const uint32_t dnz = hit & e1.z, dsg = hit & e1.w;
        if (dnz) atomicXor(a.tnz + wo, dnz);
        if (dsg) atomicXor(a.tsg + wo, dsg);
        const uint32_t mf = SLAB ? e2.y >> 30 : 0u;
        if (mf && (dnz | dsg)) {
            const uint32_t col = (e2.y >> 4) & 0x3ffffu;
            __threadfence_system();
            if (dnz) atomicXor_system((mf == 1 ? a.mir_up_nz : a.mir_dn_nz) + col, dnz);
            if (dsg) atomicXor_system((mf == 1 ? a.mir_up_sg : a.mir_dn_sg) + col, dsg);
        }
    }
    __device__ __forceinline__ void push(const uint32_t (&eq)[4], const uint32_t (&Fm)[4], const uint32_t (&Vm)[4],
                                         const uint32_t (&hA)[4], const uint32_t (&H1)[4], const uint32_t (&H0)[4],
                                         const uint32_t (&nf)[4], const uint32_t (&gg)[4], unsigned long long wo,
                                         uint32_t mir_tag)
    {
        const uint32_t below = (1u << lane) - 1u;
#pragma unroll
        for (int w = 0; w < 4; ++w) {
            const bool has = eq[w] != 0;
            const uint32_t m = __ballot_sync(0xffffffffu, has);
            if (has) {
                const unsigned long long o = wo + (unsigned)w;
                const uint32_t slot = pending + __popc(m & below);
                q[3 * slot] = make_uint4(eq[w], Fm[w], Vm[w], hA[w]);
                q[3 * slot + 1] = make_uint4(H1[w], H0[w], nf[w], gg[w]);
                q[3 * slot + 2] = make_uint4((uint32_t)o, SLAB ? (uint32_t)(o >> 32) | (mir_tag + ((unsigned)w << 4))
                                                               : (uint32_t)(o >> 32), 0u, 0u);
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

template <int PAR, bool SLAB>
__device__ __forceinline__ void bc_march_row_gen(const BCMarchArgs &a, uint32_t G, unsigned long long wo,
                                                 uint32_t *tn, uint32_t *ts,
                                                 const BCRow &U, const BCRow &C, const BCRow &D,
                                                 uint32_t En, uint32_t Es, BCTieQueueGen<SLAB> &queue,
                                                 uint32_t *mir_nz = nullptr, uint32_t *mir_sg = nullptr,
                                                 uint32_t mir_tag = 0)
{
    BCRow T;
    bcm_load(tn, ts, 0, T);
    const PlaneShared ps = plane_shared(G, a.F);
    uint32_t Fm[4], Vm[4], hA[4], H1[4], H0[4], pos[4], z4[4], nf[4], gg[4];
    {
        const uint4 pb = plane_block(ps, a.fbp, a.F, a.K);        // proposal bits
        const uint32_t b[4] = {pb.x, pb.y, pb.z, pb.w};
#pragma unroll
        for (int w = 0; w < 4; ++w) {
            uint32_t Sn, Ss;
            if (PAR == 0) {
                Sn = fsl1(w == 0 ? En : C.nz[w > 0 ? w - 1 : 0], C.nz[w]);
                Ss = fsl1(w == 0 ? Es : C.sg[w > 0 ? w - 1 : 0], C.sg[w]);
            } else {
                Sn = fsr1(C.nz[w], w == 3 ? En : C.nz[w < 3 ? w + 1 : 0]);
                Ss = fsr1(C.sg[w], w == 3 ? Es : C.sg[w < 3 ? w + 1 : 0]);
            }
            const uint32_t nz = T.nz[w], sg = T.sg[w], bw = b[w];
            Fm[w] = lop3<0x90>(nz, sg, bw);                       // flip: nz & ~(sg ^ b)
            Vm[w] = nz & ~Fm[w];                                  // vacate; occupy = ~nz
            nf[w] = ~Fm[w];
            gg[w] = lop3<0xDA>(nz, sg, bw);
            const uint32_t r = lop3<0xC5>(nz, sg, bw);            // reference sign (bc_march_row)
            const uint32_t a1 = lop3<0x90>(U.nz[w], U.sg[w], r), n1 = lop3<0x9F>(U.nz[w], U.sg[w], r);
            const uint32_t a2 = lop3<0x90>(D.nz[w], D.sg[w], r), n2 = lop3<0x9F>(D.nz[w], D.sg[w], r);
            const uint32_t a3 = lop3<0x90>(C.nz[w], C.sg[w], r), n3 = lop3<0x9F>(C.nz[w], C.sg[w], r);
            const uint32_t a4 = lop3<0x90>(Sn, Ss, r), n4 = lop3<0x9F>(Sn, Ss, r);
            const uint32_t s1 = lop3<0x96>(a1, a2, a3), c1 = lop3<0xE8>(a1, a2, a3);
            const uint32_t s2 = lop3<0x96>(n1, n2, n3), c2 = lop3<0xE8>(n1, n2, n3);
            const uint32_t s3 = lop3<0x96>(s1, s2, a4), c3 = lop3<0xE8>(s1, s2, a4);
            const uint32_t h0 = s3 ^ n4, c4 = s3 & n4;
            const uint32_t t1 = lop3<0x96>(c1, c2, c3), d1 = lop3<0xE8>(c1, c2, c3);
            const uint32_t h1 = t1 ^ c4, d2 = t1 & c4;
            const uint32_t h2 = d1 ^ d2, h3 = d1 & d2;
            H0[w] = h0; H1[w] = h1;
            hA[w] = lop3<0xCA>(Fm[w], h3, h2);                    // flip ? h3 : h2
            pos[w] = h3 | lop3<0xE0>(h2, h1, h0);                 // x >= 1
            z4[w] = ~(h3 | h2 | h1 | h0);                         // x == -4
        }
    }
    uint32_t aA[4], aB[4], selA[4], need[4], acc[4], eq[4];
    lut3_dispatch(a.lutA_always, hA, H1, H0, aA);
    lut3_dispatch(a.lutB_always, hA, H1, H0, aB);
#pragma unroll
    for (int w = 0; w < 4; ++w) {
        // lanes of table A: flips and the sharing type (nz lanes if vacate shares, else flip | ~nz)
        selA[w] = a.share_v ? (Fm[w] | Vm[w]) : ~Vm[w];
        // table A lanes decide only for x >= 1; table B lanes unless "always" (x = -4 always is)
        need[w] = lop3<0xCA>(selA[w], pos[w] & ~aA[w], ~(aB[w] | z4[w]));
        eq[w] = need[w];
        acc[w] = 0;
    }
#pragma unroll 1                     // two 256-entry dispatch tables per iteration: keep one copy
    for (int k = 7; k >= 0; --k) {
        const uint4 b4 = plane_block(ps, a.F.fb[0] ^ ((uint32_t)k << 16), a.F, a.K);
        const uint32_t b[4] = {b4.x, b4.y, b4.z, b4.w};
        uint32_t gA[4], gB[4];
        lut3_dispatch(a.lutA[k], hA, H1, H0, gA);
        lut3_dispatch(a.lutB[k], hA, H1, H0, gB);
#pragma unroll
        for (int w = 0; w < 4; ++w) {
            const uint32_t tau = lop3<0xCA>(selA[w], gA[w], gB[w]);
            acc[w] = maj3m(tau, ~b[w], acc[w]);
            eq[w] &= ~(b[w] ^ tau);
        }
    }
#pragma unroll
    for (int w = 0; w < 4; ++w) {
        const uint32_t ok = ~need[w] | acc[w];                    // a tied lane has acc = 0
        T.nz[w] ^= ok & nf[w];
        T.sg[w] ^= ok & gg[w];
    }
    *reinterpret_cast<uint4 *>(tn) = make_uint4(T.nz[0], T.nz[1], T.nz[2], T.nz[3]);
    *reinterpret_cast<uint4 *>(ts) = make_uint4(T.sg[0], T.sg[1], T.sg[2], T.sg[3]);
    if (SLAB && mir_nz) {
        *reinterpret_cast<uint4 *>(mir_nz) = make_uint4(T.nz[0], T.nz[1], T.nz[2], T.nz[3]);
        *reinterpret_cast<uint4 *>(mir_sg) = make_uint4(T.sg[0], T.sg[1], T.sg[2], T.sg[3]);
        __threadfence_system();
    }
    queue.push(eq, Fm, Vm, hA, H1, H0, nf, gg, wo, mir_tag);
}

// GEN = false: the integer-dE (Delta = 0 type) rows above; GEN = true: bc_march_row_gen
template <bool GEN, int PAR, bool SLAB, int LS, class Args, class Queue>
__device__ __forceinline__ void bc_row(const Args &a, uint32_t G, unsigned long long wo, uint32_t *tn,
                                       uint32_t *ts, const BCRow &U, const BCRow &C, const BCRow &D, uint32_t En,
                                       uint32_t Es, Queue &queue, uint32_t *mir_nz = nullptr,
                                       uint32_t *mir_sg = nullptr, uint32_t mir_tag = 0)
{
    if constexpr (GEN) bc_march_row_gen<PAR, SLAB>(a, G, wo, tn, ts, U, C, D, En, Es, queue, mir_nz, mir_sg, mir_tag);
    else bc_march_row<PAR, SLAB, LS>(a, G, wo, tn, ts, U, C, D, En, Es, queue, mir_nz, mir_sg, mir_tag);
}

template <bool GEN, bool SLAB>
struct BCQueueOf { using type = BCTieQueue<SLAB>; };
template <bool SLAB>
struct BCQueueOf<true, SLAB> { using type = BCTieQueueGen<SLAB>; };

// The march of one thread: rows i0 .. i0+R-1 of run q, g = s * (wpr/4) + q (ties are queued, not
// drained) -- shared by bc_march_kernel and bc_persist_kernel (bc_persist.cuh).
template <int COLOUR, bool SLAB, bool GEN, int LS = -1, class Args, class Queue>
__device__ __forceinline__ void bc_march_thread(const Args &a, uint32_t g, Queue &queue)
{
    const uint32_t L = a.L, wpr = a.wpr, nq = wpr >> 2;
    const uint32_t q = g % nq, s = g / nq;
    const uint32_t kw = q << 2;
    const uint32_t i0 = s * a.R + (SLAB ? a.row_off : 0u);
    const uint32_t iu = (i0 == 0) ? L - 1 : i0 - 1;
    const uint32_t ke0 = (kw == 0) ? wpr - 1 : kw - 1;       // word before the run (periodic)
    const uint32_t ke1 = (kw + 4 == wpr) ? 0 : kw + 4;       // word after it
    const unsigned long long ro = (unsigned long long)i0 * wpr;
    BCRow U, C, D;
    bcm_load(a.onz, a.osg, (unsigned long long)iu * wpr + kw, U);
    bcm_load(a.onz, a.osg, ro + kw, C);
    uint32_t G = i0 * nq + q + (SLAB ? a.g_off : 0u);
    const bool top = SLAB && s == 0, bot = SLAB && (s + 1) * nq == a.threads;
    // running pointers: the slab's own rows never wrap; only row i+1 of the last lattice row does
    // (the sg plane sits one plane stride pw = L * wpr words after the nz plane)
    const unsigned long long pw = (unsigned long long)L * wpr;
    const uint32_t *on = a.onz + ro;                                // row i of the opposite colour (nz)
    uint32_t *tn = a.tnz + ro + kw;                                 // this run in row i (nz)
    unsigned long long wo = ro + kw;
    uint32_t left = L - i0;
    for (uint32_t r = 0; r < a.R; r += 2) {
        {   // row i0 + r: (i + colour) & 1 == COLOUR
            const uint32_t *dn = on + wpr;
            bcm_load(dn, dn + pw, kw, D);
            const uint32_t ke = COLOUR == 0 ? ke0 : ke1;
            if (SLAB && top && r == 0)
                bc_row<GEN, COLOUR, SLAB, LS>(a, G, wo, tn, tn + pw, U, C, D, on[ke], on[pw + ke], queue,
                                     a.mir_up_nz + kw, a.mir_up_sg + kw, (kw << 4) | (1u << 30));
            else
                bc_row<GEN, COLOUR, SLAB, LS>(a, G, wo, tn, tn + pw, U, C, D, on[ke], on[pw + ke], queue);
            U = C; C = D; on = dn; tn += wpr; wo += wpr; G += nq;
        }
        {   // row i0 + r + 1: the other parity; its row i + 1 wraps to row 0 at the lattice end
            left -= 2;
            const uint32_t *dn = left ? on + wpr : a.onz;
            bcm_load(dn, dn + pw, kw, D);
            const uint32_t ke = COLOUR == 0 ? ke1 : ke0;
            if (SLAB && bot && r + 2 == a.R)
                bc_row<GEN, COLOUR ^ 1, SLAB, LS>(a, G, wo, tn, tn + pw, U, C, D, on[ke], on[pw + ke], queue,
                                         a.mir_dn_nz + kw, a.mir_dn_sg + kw, (kw << 4) | (2u << 30));
            else
                bc_row<GEN, COLOUR ^ 1, SLAB, LS>(a, G, wo, tn, tn + pw, U, C, D, on[ke], on[pw + ke], queue);
            U = C; C = D; on = dn; tn += wpr; wo += wpr; G += nq;
        }
    }
}

template <int COLOUR, bool SLAB, bool GEN = false, int LS = -1>
__global__ void __launch_bounds__(256, GEN ? 2 : 3) bc_march_kernel(const BCMarchArgs a)
{
    // the general queue (3 x 16 bytes per entry, 60 KiB per block) exceeds the static limit: dynamic
    extern __shared__ uint4 s_dyn[];
    __shared__ uint4 s_fix[GEN ? 1 : 8][GEN ? 1 : 2 * TIE_Q_SLOTS];
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const uint32_t g = blockIdx.x * 256u + threadIdx.x;
    if (g - lane >= a.threads) return;          // a.threads is a multiple of 32: whole warps only
    typename BCQueueOf<GEN, SLAB>::type queue{a, GEN ? s_dyn + warp * (3 * TIE_Q_SLOTS) : s_fix[GEN ? 0 : warp], lane, 0u};
    bc_march_thread<COLOUR, SLAB, GEN, LS>(a, g, queue);
    queue.drain();
}

}  // namespace lat
