// philox.cuh -- Philox4x32-10 in registers, and the (seed, sweep, colour, site) keying.
//
// Counter-based generator of Salmon, Moraes, Dror & Shaw (SC'11): ten rounds of
//   (c0,c1,c2,c3) <- (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0))
// with the key bumped by the Weyl constants after every round.  The ten round keys depend
// only on the seed, so the host expands them once (RoundKeys) and they reach the kernels as
// launch parameters (constant bank operands of the XORs).  Nothing is ever stored to memory:
// the paper's "32-bit random numbers" live in registers only.
//
// Keying contract (BASELINE.json: keyed by (seed, sweep, colour, site)):
//   key     = (seed lo, seed hi)
//   counter = (unit lo, unit hi, t, colour | tag << 8 | plane << 16)
// with P = i*(L/2) + (j>>1) the same-colour linear site index and
//   tag 0 INIT_PLANE  unit = P>>7   one bit per site: lane l = P&127 is bit (l&31) of word l>>5
//   tag 1 INIT_QUAD   unit = P>>2   word P&3 is the site's 32-bit number
//   tag 2 ACC_QUAD    unit = P>>2   scheme 0: u32(site) = word P&3
//   tag 3 ACC_PLANE   unit = P>>7   scheme 1: plane k = 0..7 gives bit (31-k) of u32(site)
//   tag 4 ACC_TAIL    unit = P      scheme 1: low 24 bits of u32(site) = word 0 >> 8
//   tag 5 PROP_PLANE  unit = P>>7   Blume-Capel proposal bit
#pragma once
#include <stdint.h>

namespace lat {

struct RoundKeys {
    uint32_t k0[10];
    uint32_t k1[10];
};

enum : uint32_t {
    TAG_INIT_PLANE = 0, TAG_INIT_QUAD = 1, TAG_ACC_QUAD = 2, TAG_ACC_PLANE = 3,
    TAG_ACC_TAIL = 4, TAG_PROP_PLANE = 5
};

static inline void expand_round_keys(uint64_t seed, RoundKeys &K)
{
    uint32_t a = (uint32_t)(seed & 0xffffffffull), b = (uint32_t)(seed >> 32);
    for (int r = 0; r < 10; ++r) {
        K.k0[r] = a;
        K.k1[r] = b;
        a += 0x9E3779B9u;
        b += 0xBB67AE85u;
    }
}

// ---- folded bit-plane streams (tags 0, 3, 5: unit = P>>7 < 2^32, so the counter's second word is 0) ----
// For a fixed launch (seed, t, colour, tag) the counter of plane k of unit G is (G, 0, t, ctr3_k):
// only the first word varies per thread and only the fourth per plane.  Writing the rounds out,
//   round 0:  c0 <- N0 = hi(M1 t) ^ k0[0]          (launch constant)
//             c1 <- A1 = lo(M1 t)                  (launch constant)
//             c2 <- hi(M0 G) ^ ctr3_k ^ k1[0]      = xh ^ fb[k]
//             c3 <- lo(M0 G)                       = xl          (shared by the planes of G)
//   round 1:  c0 <- hi(M1 c2) ^ A1 ^ k0[1]         = hi(M1 c2) ^ fa
//             c1 <- lo(M1 c2)
//             c2 <- hi(M0 N0) ^ xl ^ k1[1]         = fh ^ xl     (shared by the planes of G)
//             c3 <- lo(M0 N0) = L0                 (launch constant)
//   round 2:  c0 <- hi(M1 (fh^xl)) ^ c1 ^ k0[2]    = yh ^ c1 ^ k0[2]   (y shared by the planes)
//             c1 <- lo(M1 (fh^xl))                 = yl
//             c2 <- hi(M0 c0) ^ L0 ^ k1[2]         = hi(M0 c0) ^ fl
//             c3 <- lo(M0 c0)
// and rounds 3..9 are generic.  Per plane this is 16 multiplies instead of 20 (plus 2 shared by
// all planes of G); the result is bit-identical to philox4x32_10 on the full counter.
struct PlaneFold {
    uint32_t fa;              // lo(M1 t) ^ k0[1]
    uint32_t fh;              // hi(M0 N0) ^ k1[1]
    uint32_t fl;              // lo(M0 N0) ^ k1[2]
    uint32_t fb[8];           // ctr3(colour, tag, k) ^ k1[0], k = 0..7
};

#ifdef __CUDACC__
__host__ __device__
#endif
static inline void build_plane_fold(const RoundKeys &K, uint32_t t, uint32_t colour, uint32_t tag,
                                    PlaneFold &f)
{
    const unsigned long long p1 = 0xCD9E8D57ull * (unsigned long long)t;
    const uint32_t N0 = (uint32_t)(p1 >> 32) ^ K.k0[0];
    const unsigned long long p0 = 0xD2511F53ull * (unsigned long long)N0;
    f.fa = (uint32_t)p1 ^ K.k0[1];
    f.fh = (uint32_t)(p0 >> 32) ^ K.k1[1];
    f.fl = (uint32_t)p0 ^ K.k1[2];
    for (uint32_t k = 0; k < 8; ++k) f.fb[k] = (colour | (tag << 8) | (k << 16)) ^ K.k1[0];
}

#ifdef __CUDACC__
// the part of a folded plane block that all planes of unit G share
struct PlaneShared {
    uint32_t xh, xl, yh, yl;
};

__host__ __device__ __forceinline__ PlaneShared plane_shared(uint32_t G, const PlaneFold &f)
{
    PlaneShared s;
    const unsigned long long x = (unsigned long long)G * 0xD2511F53ull;
    s.xh = (uint32_t)(x >> 32);
    s.xl = (uint32_t)x;
    const unsigned long long y = (unsigned long long)(f.fh ^ s.xl) * 0xCD9E8D57ull;
    s.yh = (uint32_t)(y >> 32);
    s.yl = (uint32_t)y;
    return s;
}

// 128-bit block of plane k (fbk = f.fb[k]) of the unit whose shared part is s
__host__ __device__ __forceinline__ uint4 plane_block(const PlaneShared &s, uint32_t fbk, const PlaneFold &f,
                                             const RoundKeys &K)
{
    // round 1
    const unsigned long long q1 = (unsigned long long)(s.xh ^ fbk) * 0xCD9E8D57ull;
    uint32_t c0 = (uint32_t)(q1 >> 32) ^ f.fa;
    uint32_t c1 = (uint32_t)q1;
    // round 2
    const unsigned long long q0 = (unsigned long long)c0 * 0xD2511F53ull;
    c0 = s.yh ^ c1 ^ K.k0[2];
    c1 = s.yl;
    uint32_t c2 = (uint32_t)(q0 >> 32) ^ f.fl;
    uint32_t c3 = (uint32_t)q0;
#pragma unroll
    for (int r = 3; r < 10; ++r) {
        const unsigned long long p0 = (unsigned long long)c0 * 0xD2511F53ull;
        const unsigned long long p1 = (unsigned long long)c2 * 0xCD9E8D57ull;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ K.k0[r];
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ K.k1[r];
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
    }
    return make_uint4(c0, c1, c2, c3);
}

__host__ __device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                               const RoundKeys &K)
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const unsigned long long p0 = (unsigned long long)c0 * 0xD2511F53ull;
        const unsigned long long p1 = (unsigned long long)c2 * 0xCD9E8D57ull;
        const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ K.k0[r];
        const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ K.k1[r];
        c1 = (uint32_t)p1;
        c3 = (uint32_t)p0;
        c0 = n0;
        c2 = n2;
    }
    return make_uint4(c0, c1, c2, c3);
}

__device__ __forceinline__ uint32_t ctr3(uint32_t colour, uint32_t tag, uint32_t plane)
{
    return colour | (tag << 8) | (plane << 16);
}

// 128-bit block of a 128-site unit (tags 0, 3, 5)
__device__ __forceinline__ uint4 philox_unit(unsigned long long unit, uint32_t t, uint32_t colour,
                                             uint32_t tag, uint32_t plane, const RoundKeys &K)
{
    return philox4x32_10((uint32_t)unit, (uint32_t)(unit >> 32), t, ctr3(colour, tag, plane), K);
}

__device__ __forceinline__ uint32_t pick(const uint4 v, uint32_t idx)
{
    return idx == 0 ? v.x : idx == 1 ? v.y : idx == 2 ? v.z : v.w;
}
#endif

}  // namespace lat
