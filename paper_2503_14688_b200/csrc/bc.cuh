// bc.cuh -- packed checkerboard Metropolis half-sweep for the spin-1 Blume-Capel model.
//
// Paper: Eq. 1 with crystal field Delta, Metropolis + checkerboard + multispin
// coding.  Proposal (BASELINE.json; the paper is silent): one of the two other
// spin values with probability 1/2 each, code' = (code + 1 + b) mod 3 with code = s + 1 and b
// the site's PROPOSAL-plane bit.  2 bits per spin as two bit-planes per colour:
//   nz = (s != 0), sg = (s < 0)   (sg = 0 wherever nz = 0)
// with the same [row][word] layout and neighbour geometry as the Ising kernel (ising.cuh).
//
// Every proposed move is one of three types, and with a per-lane reference sign r its energy
// change depends on one small integer x = (#neighbours of sign r) - (#neighbours of sign -r):
//   flip    (+-1 -> -+1): nz & (sg == b),  r = sg,  dE = 2x
//   vacate  (+-1 -> 0)  : nz & (sg != b),  r = sg,  dE = x - Delta
//   occupy  (0 -> s')   : ~nz, s' = b ? -1 : +1,  r = ~b (sign of -s'),  dE = x + Delta
// (dE = (s - s')h + Delta (s'^2 - s^2) of Eq. 1 written per type.)  The 27 (type, x) entries
// of the threshold table are classified on the host into always / never / decide; the lanes of
// a "decide" entry get their per-lane threshold bits OR-ed into 8 bit-planes tau_k, after which
// the bit-serial compare is the same as for Ising.
#pragma once
#include "ising.cuh"

namespace lat {

enum { BC_FLIP = 0, BC_VACATE = 1, BC_OCCUPY = 2 };

struct BCArgs {
    uint32_t *tnz, *tsg;            // colour being updated
    const uint32_t *onz, *osg;      // opposite colour
    uint32_t L, wpr, t, colour;
    uint32_t tq_log2;
    uint32_t always_mask;           // bit e = type*9 + (x+4): threshold == 2^32
    uint32_t decide_mask;           // bit e: 0 < threshold < 2^32
    uint32_t thr[27];               // thresholds of the "decide" entries
    RoundKeys K;
};

template <int WPT>
struct BCWords {
    uint32_t nz[WPT], sg[WPT];
};

template <int WPT>
__device__ __forceinline__ void bc_load(const uint32_t *nzp, const uint32_t *sgp, size_t off,
                                        BCWords<WPT> &v)
{
    if constexpr (WPT == 4) {
        const uint4 a = *reinterpret_cast<const uint4 *>(nzp + off);
        const uint4 b = *reinterpret_cast<const uint4 *>(sgp + off);
        v.nz[0] = a.x; v.nz[1] = a.y; v.nz[2] = a.z; v.nz[3] = a.w;
        v.sg[0] = b.x; v.sg[1] = b.y; v.sg[2] = b.z; v.sg[3] = b.w;
    } else {
#pragma unroll
        for (int w = 0; w < WPT; ++w) { v.nz[w] = nzp[off + w]; v.sg[w] = sgp[off + w]; }
    }
}

// per-lane entry index e = type*9 + (x+4) of lane `bit` (tails and scheme 0 only)
__device__ __forceinline__ uint32_t bc_lane_entry(uint32_t bit, uint32_t flipm, uint32_t vacm,
                                                  uint32_t A0, uint32_t A1, uint32_t A2,
                                                  uint32_t O0, uint32_t O1, uint32_t O2)
{
    const uint32_t type = ((flipm >> bit) & 1u) ? BC_FLIP : ((vacm >> bit) & 1u) ? BC_VACATE : BC_OCCUPY;
    const int A = (int)(((A0 >> bit) & 1u) | (((A1 >> bit) & 1u) << 1) | (((A2 >> bit) & 1u) << 2));
    const int O = (int)(((O0 >> bit) & 1u) | (((O1 >> bit) & 1u) << 1) | (((O2 >> bit) & 1u) << 2));
    return type * 9u + (uint32_t)(A - O + 4);
}

template <int WPT, int SCHEME>
__device__ __forceinline__ void bc_update_run(const BCArgs &a, uint32_t i, uint32_t kw)
{
    const uint32_t L = a.L, wpr = a.wpr;
    const uint32_t iu = (i == 0) ? L - 1 : i - 1;
    const uint32_t id = (i + 1 == L) ? 0 : i + 1;
    const size_t row = (size_t)i * wpr, rowu = (size_t)iu * wpr, rowd = (size_t)id * wpr;
    const uint32_t par = (i + a.colour) & 1u;

    BCWords<WPT> T, U, D, C, S;
    bc_load<WPT>(a.tnz, a.tsg, row + kw, T);
    bc_load<WPT>(a.onz, a.osg, rowu + kw, U);
    bc_load<WPT>(a.onz, a.osg, rowd + kw, D);
    bc_load<WPT>(a.onz, a.osg, row + kw, C);
    if (par == 0) {
        const uint32_t ke = (kw == 0) ? wpr - 1 : kw - 1;
        const uint32_t En = a.onz[row + ke], Es = a.osg[row + ke];
#pragma unroll
        for (int w = 0; w < WPT; ++w) {
            S.nz[w] = __funnelshift_l(w == 0 ? En : C.nz[w > 0 ? w - 1 : 0], C.nz[w], 1);
            S.sg[w] = __funnelshift_l(w == 0 ? Es : C.sg[w > 0 ? w - 1 : 0], C.sg[w], 1);
        }
    } else {
        const uint32_t ke = (kw + WPT == wpr) ? 0 : kw + WPT;
        const uint32_t En = a.onz[row + ke], Es = a.osg[row + ke];
#pragma unroll
        for (int w = 0; w < WPT; ++w) {
            S.nz[w] = __funnelshift_r(C.nz[w], w == WPT - 1 ? En : C.nz[w < WPT - 1 ? w + 1 : 0], 1);
            S.sg[w] = __funnelshift_r(C.sg[w], w == WPT - 1 ? Es : C.sg[w < WPT - 1 ? w + 1 : 0], 1);
        }
    }

    const unsigned long long P0 = (unsigned long long)i * (L >> 1) + ((unsigned long long)kw << 5);
    const unsigned long long G = P0 >> 7;
    const uint32_t sub = (uint32_t)(P0 >> 5) & 3u;

    // proposal bits
    uint32_t b[WPT];
    {
        const uint4 blk = philox_unit(G, a.t, a.colour, TAG_PROP_PLANE, 0, a.K);
#pragma unroll
        for (int w = 0; w < WPT; ++w) b[w] = (WPT == 4) ? pick(blk, w) : pick(blk, sub + w);
    }

    uint32_t flipm[WPT], vacm[WPT], occm[WPT];
    uint32_t A0[WPT], A1[WPT], A2[WPT], O0[WPT], O1[WPT], O2[WPT];
    uint32_t alw[WPT], need[WPT], tau[8][WPT];
#pragma unroll
    for (int w = 0; w < WPT; ++w) {
        const uint32_t nz = T.nz[w], sg = T.sg[w];
        flipm[w] = nz & ~(sg ^ b[w]);
        vacm[w] = nz & (sg ^ b[w]);
        occm[w] = ~nz;
        const uint32_t r = (nz & sg) | (~nz & ~b[w]);
        // neighbours of sign r ("a") and of sign -r ("o"), counted bit-sliced
        const uint32_t a1 = U.nz[w] & ~(U.sg[w] ^ r), o1 = U.nz[w] & (U.sg[w] ^ r);
        const uint32_t a2 = D.nz[w] & ~(D.sg[w] ^ r), o2 = D.nz[w] & (D.sg[w] ^ r);
        const uint32_t a3 = C.nz[w] & ~(C.sg[w] ^ r), o3 = C.nz[w] & (C.sg[w] ^ r);
        const uint32_t a4 = S.nz[w] & ~(S.sg[w] ^ r), o4 = S.nz[w] & (S.sg[w] ^ r);
        {
            const uint32_t s1 = a1 ^ a2 ^ a3, c1 = maj3(a1, a2, a3), c2 = s1 & a4;
            A0[w] = s1 ^ a4; A1[w] = c1 ^ c2; A2[w] = c1 & c2;
        }
        {
            const uint32_t s1 = o1 ^ o2 ^ o3, c1 = maj3(o1, o2, o3), c2 = s1 & o4;
            O0[w] = s1 ^ o4; O1[w] = c1 ^ c2; O2[w] = c1 & c2;
        }
        // one-hots of A and O (both <= 4, A + O <= 4)
        uint32_t Ah[5], Oh[5];
        Ah[0] = ~(A0[w] | A1[w] | A2[w]); Ah[1] = A0[w] & ~A1[w]; Ah[2] = ~A0[w] & A1[w];
        Ah[3] = A0[w] & A1[w]; Ah[4] = A2[w];
        Oh[0] = ~(O0[w] | O1[w] | O2[w]); Oh[1] = O0[w] & ~O1[w]; Oh[2] = ~O0[w] & O1[w];
        Oh[3] = O0[w] & O1[w]; Oh[4] = O2[w];
        uint32_t X[9];   // X[x+4] = lanes with A - O == x
        X[8] = Ah[4];
        X[7] = Ah[3] & Oh[0];
        X[6] = (Ah[2] & Oh[0]) | (Ah[3] & Oh[1]);
        X[5] = (Ah[1] & Oh[0]) | (Ah[2] & Oh[1]);
        X[4] = (Ah[0] & Oh[0]) | (Ah[1] & Oh[1]) | (Ah[2] & Oh[2]);
        X[3] = (Ah[0] & Oh[1]) | (Ah[1] & Oh[2]);
        X[2] = (Ah[0] & Oh[2]) | (Ah[1] & Oh[3]);
        X[1] = Ah[0] & Oh[3];
        X[0] = Oh[4];
        uint32_t al = 0, nd = 0, tk[8] = {0, 0, 0, 0, 0, 0, 0, 0};
#pragma unroll
        for (int type = 0; type < 3; ++type) {
            const uint32_t tm = type == BC_FLIP ? flipm[w] : type == BC_VACATE ? vacm[w] : occm[w];
#pragma unroll
            for (int xi = 0; xi < 9; ++xi) {
                const int e = type * 9 + xi;
                if ((a.always_mask >> e) & 1u) al |= tm & X[xi];
                if ((a.decide_mask >> e) & 1u) {
                    const uint32_t cls = tm & X[xi];
                    nd |= cls;
                    const uint32_t thr = a.thr[e];
#pragma unroll
                    for (int k = 0; k < 8; ++k)
                        if ((thr >> (31 - k)) & 1u) tk[k] |= cls;
                }
            }
        }
        alw[w] = al;
        need[w] = nd;
#pragma unroll
        for (int k = 0; k < 8; ++k) tau[k][w] = tk[k];
    }

    uint32_t acc[WPT];
#pragma unroll
    for (int w = 0; w < WPT; ++w) acc[w] = 0;

    if (SCHEME == 1) {
        uint32_t eq[WPT];
#pragma unroll
        for (int w = 0; w < WPT; ++w) eq[w] = need[w];
#pragma unroll
        for (int k = 7; k >= 0; --k) {
            const uint4 blk = philox_unit(G, a.t, a.colour, TAG_ACC_PLANE, (uint32_t)k, a.K);
#pragma unroll
            for (int w = 0; w < WPT; ++w) {
                const uint32_t pb = (WPT == 4) ? pick(blk, w) : pick(blk, sub + w);
                acc[w] = maj3(tau[k][w], ~pb, acc[w]);
                eq[w] &= ~(pb ^ tau[k][w]);
            }
        }
#pragma unroll
        for (int w = 0; w < WPT; ++w) {
            uint32_t e = eq[w];
            while (e) {
                const uint32_t bit = __ffs(e) - 1;
                e &= e - 1;
                const unsigned long long P = P0 + 32u * w + bit;
                const uint4 blk = philox_unit(P, a.t, a.colour, TAG_ACC_TAIL, 0, a.K);
                const uint32_t thr = a.thr[bc_lane_entry(bit, flipm[w], vacm[w], A0[w], A1[w], A2[w],
                                                         O0[w], O1[w], O2[w])];
                if ((blk.x >> 8) < (thr & 0x00ffffffu)) acc[w] |= 1u << bit;
            }
        }
    } else {
#pragma unroll
        for (int w = 0; w < WPT; ++w) {
#pragma unroll 1
            for (int q = 0; q < 8; ++q) {
                if (((need[w] >> (4 * q)) & 0xfu) == 0) continue;
                const unsigned long long unit = (P0 + 32u * w + 4u * q) >> 2;
                const uint4 blk = philox_unit(unit, a.t, a.colour, TAG_ACC_QUAD, 0, a.K);
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    const uint32_t bit = 4 * q + j;
                    if (!((need[w] >> bit) & 1u)) continue;
                    const uint32_t thr = a.thr[bc_lane_entry(bit, flipm[w], vacm[w], A0[w], A1[w],
                                                             A2[w], O0[w], O1[w], O2[w])];
                    if (pick(blk, j) < thr) acc[w] |= 1u << bit;
                }
            }
        }
    }

    // apply accepted moves
#pragma unroll
    for (int w = 0; w < WPT; ++w) {
        const uint32_t ok = alw[w] | (acc[w] & need[w]);
        const uint32_t nz = T.nz[w], sg = T.sg[w];
        T.nz[w] = nz ^ (ok & ~flipm[w]);
        T.sg[w] = ((sg ^ (ok & flipm[w])) & ~(ok & vacm[w])) | (ok & occm[w] & b[w]);
    }
    if constexpr (WPT == 4) {
        *reinterpret_cast<uint4 *>(a.tnz + row + kw) = make_uint4(T.nz[0], T.nz[1], T.nz[2], T.nz[3]);
        *reinterpret_cast<uint4 *>(a.tsg + row + kw) = make_uint4(T.sg[0], T.sg[1], T.sg[2], T.sg[3]);
    } else {
#pragma unroll
        for (int w = 0; w < WPT; ++w) { a.tnz[row + kw + w] = T.nz[w]; a.tsg[row + kw + w] = T.sg[w]; }
    }
}

template <int SCHEME>
__global__ void __launch_bounds__(256, 2) bc_half_sweep_v4(const BCArgs a)
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
    bc_update_run<4, SCHEME>(a, i, q * 4);
}

template <int SCHEME>
__global__ void __launch_bounds__(256) bc_half_sweep_v1(const BCArgs a)
{
    const unsigned long long g = (unsigned long long)blockIdx.x * 256u + threadIdx.x;
    if (g >= (unsigned long long)a.L * a.wpr) return;
    bc_update_run<1, SCHEME>(a, (uint32_t)(g / a.wpr), (uint32_t)(g % a.wpr));
}

// Disordered start: uniform on {-1,0,+1}: code = floor(3 u / 2^32) with u the site's INIT_QUAD
// word, s = code - 1 (reading 11).  One thread per word (8 Philox blocks).
struct BCInitArgs {
    uint32_t *buf;            // [2 colours][2 planes][L][wpr]
    uint32_t L, wpr;
    RoundKeys K;
};

__global__ void __launch_bounds__(256) bc_init_kernel(const BCInitArgs a)
{
    const unsigned long long words = (unsigned long long)a.L * a.wpr;   // per colour per plane
    const unsigned long long g = (unsigned long long)blockIdx.x * 256u + threadIdx.x;
    if (g >= 2 * words) return;
    const uint32_t colour = g >= words;
    const unsigned long long wi = g - (colour ? words : 0);
    const unsigned long long P0 = wi << 5;
    uint32_t nz = 0, sg = 0;
#pragma unroll 1
    for (int q = 0; q < 8; ++q) {
        const uint4 blk = philox_unit((P0 >> 2) + q, 0, colour, TAG_INIT_QUAD, 0, a.K);
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const uint32_t code = __umulhi(pick(blk, j), 3u);
            nz |= (uint32_t)(code != 1u) << (4 * q + j);
            sg |= (uint32_t)(code == 0u) << (4 * q + j);
        }
    }
    a.buf[(size_t)(2 * colour) * words + wi] = nz;
    a.buf[(size_t)(2 * colour + 1) * words + wi] = sg;
}

// Row-slab variant of the disordered start (see ising_init_slab_kernel): local rows 0 .. rows-1,
// local row l = global row (row_base + l) mod L, keyed by global coordinates.
struct BCSlabInitArgs {
    uint32_t *buf;            // [2 colours][2 planes][rows][wpr]
    uint32_t L, wpr, rows, row_base;
    RoundKeys K;
};

__global__ void __launch_bounds__(256) bc_init_slab_kernel(const BCSlabInitArgs a)
{
    const unsigned long long words = (unsigned long long)a.rows * a.wpr;   // per colour per plane
    const unsigned long long g = (unsigned long long)blockIdx.x * 256u + threadIdx.x;
    if (g >= 2 * words) return;
    const uint32_t colour = g >= words;
    const unsigned long long wi = g - (colour ? words : 0);
    const uint32_t li = (uint32_t)(wi / a.wpr), k = (uint32_t)(wi % a.wpr);
    const uint32_t gi = (a.row_base + li) % a.L;
    const unsigned long long P0 = ((unsigned long long)gi * a.wpr + k) << 5;
    uint32_t nz = 0, sg = 0;
#pragma unroll 1
    for (int q = 0; q < 8; ++q) {
        const uint4 blk = philox_unit((P0 >> 2) + q, 0, colour, TAG_INIT_QUAD, 0, a.K);
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const uint32_t code = __umulhi(pick(blk, j), 3u);
            nz |= (uint32_t)(code != 1u) << (4 * q + j);
            sg |= (uint32_t)(code == 0u) << (4 * q + j);
        }
    }
    a.buf[(size_t)(2 * colour) * words + wi] = nz;
    a.buf[(size_t)(2 * colour + 1) * words + wi] = sg;
}

}  // namespace lat
