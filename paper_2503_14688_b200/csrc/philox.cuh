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

#ifdef __CUDACC__
__device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
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
