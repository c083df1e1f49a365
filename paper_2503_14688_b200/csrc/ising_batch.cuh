// ising_batch.cuh -- many independent Ising replicas per launch (lattice_create_batch).
//
// The paper's statistics are 40-4000 independent runs per point (Tables I-II, PAPER.md:126-153;
// errors by the jackknife over realisations).  One small lattice cannot fill
// the GPU: at L = 4096 a half-sweep is 2^23 updates (1.7 us of work), at L = 64 it is 2048.  A
// batch handle holds n replicas [replica][colour][row][word] that differ only in their Philox
// key (seed), every replica evolving bit for bit like a stand-alone lattice with that seed:
//
//   * ising_march_batch_kernel -- the production marching kernel over all replicas at once
//     (L a multiple of 256): blockIdx.y is the replica; its ten round keys come from a table in
//     the kernel parameters, indexed by blockIdx.y, i.e. uniform-register operands of the Philox
//     XORs exactly like the single-lattice kernel's launch constants (no extra registers);
//   * ising_block_kernel -- 256 <= L <= 512: one thread block per replica runs ALL n sweeps of the
//     call, a block barrier between the colours instead of a launch;
//   * ising_tiny_kernel -- L = 64 and 128 (one or two words per row): a half-warp (L = 64) or a
//     warp (L = 128) owns a whole replica IN REGISTERS, each lane four consecutive rows = whole
//     128-site RNG units, neighbour rows come by warp shuffle, and ALL n sweeps of the call run
//     inside the one launch with no barrier at all (lanes of a warp run in lock step).  BASELINE
//     config 1 (L = 64, 2000 sweeps) is then one launch instead of 4000.
//
// Same arithmetic as ising_march.cuh (class masks, folded Philox planes, plane compare by brx.idx or
// with the plane cases compiled in); in ising_tiny_kernel the lanes of a replica resolve its ties
// together before the next half-sweep (state lives in registers, so there is nothing to patch later).
#pragma once
#include "ising_march.cuh"
#include "ising_persist.cuh"

namespace lat {

#ifndef LAT_TINY_MINB
#define LAT_TINY_MINB 4        // resident blocks per SM of ising_tiny_kernel<1> (measured: 4 > 6; see below)
#endif

constexpr int BATCH_CHUNK = 128;             // replicas per launch of the marching batch kernel

struct BatchKeys {                           // 10 KiB of kernel parameters
    RoundKeys K[BATCH_CHUNK];
};

#ifdef __CUDACC__
template <int COLOUR, bool EDGE, bool ONE_ROW, int PC = -1>
__global__ void __launch_bounds__(256) ising_march_batch_kernel(const IsingMarchArgs a0,
                                                                const __grid_constant__ BatchKeys bk,
                                                                unsigned long long rep_stride)
{
    __shared__ uint4 s_q[8][TIE_Q_SLOTS];
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    const uint32_t g = blockIdx.x * 256u + threadIdx.x;
    if (g - lane >= a0.threads) return;          // a0.threads (per replica) is a multiple of 32
    const uint32_t rep = blockIdx.y;
    IsingMarchArgs a = a0;
    a.tgt = a0.tgt + rep * rep_stride;
    a.opp = a0.opp + rep * rep_stride;
    a.K = bk.K[rep];
    build_plane_fold(a.K, a.t, a.colour, TAG_ACC_PLANE, a.F);
    WarpTieQueue<false> queue{a, s_q[warp], lane, 0u};
    if (ONE_ROW) row_thread<COLOUR, EDGE>(a, g, queue);
    else march_thread<COLOUR, EDGE, false, PC>(a, g, queue);
    queue.drain();
}

// ---- 256 <= L <= 512: one thread block per replica, all sweeps of the call in one launch ---------
//
// A half-sweep of such a replica is a few thousand thread-rows: launched on its own it costs more
// in launch latency than in work.  Here block b owns replica b for the whole call: its threads take
// one row of one 128-bit run each (row_thread, strided over the replica), the two colours are
// separated by a block barrier instead of a kernel boundary, and the per-half-sweep arguments are
// rebuilt in shared memory exactly as in ising_persist_kernel.  The replica (<= 128 KiB) stays in
// L1/L2; replicas are independent, so no block ever waits for another.
constexpr int BLOCK_KERNEL_THREADS = 512;

template <bool EDGE>
__global__ void __launch_bounds__(BLOCK_KERNEL_THREADS, 2) ising_block_kernel(const IsingMarchArgs a0, uint32_t *buf,
                                                                           const RoundKeys *keys,
                                                                           const SweepParams *sp, uint32_t n_sweeps,
                                                                           unsigned long long rep_words)
{
    __shared__ uint4 s_q[BLOCK_KERNEL_THREADS / 32][TIE_Q_SLOTS];
    __shared__ IsingMarchArgs a;
    const uint32_t lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    uint32_t *base = buf + blockIdx.x * rep_words;
    const unsigned long long pw = (unsigned long long)a0.L * a0.wpr;
    if (threadIdx.x == 0) { a = a0; a.K = keys[blockIdx.x]; }
    SweepParams p = sp[0];                       // thread 0 uses it; the next one is prefetched
    for (uint32_t s = 0; s < n_sweeps; ++s) {
        for (uint32_t colour = 0; colour < 2; ++colour) {
            if (threadIdx.x == 0) {
                if (colour == 0) {
                    a.thr4 = p.thr4; a.thr8 = p.thr8; a.mask4 = p.mask4; a.mask8 = p.mask8;
                    for (int k = 0; k < 8; ++k) a.pcase[k] = p.pcase[k];
                    a.t = a0.t + s;
                    if (s + 1 < n_sweeps) p = sp[s + 1];
                }
                a.colour = colour;
                a.tgt = base + colour * pw;
                a.opp = base + (1u - colour) * pw;
                build_plane_fold(a.K, a.t, colour, TAG_ACC_PLANE, a.F);
            }
            __syncthreads();
            WarpTieQueue<false> queue{a, s_q[warp], lane, 0u};
            for (uint32_t g = threadIdx.x; g - lane < a0.threads; g += blockDim.x) {
                if (colour == 0) row_thread<0, EDGE>(a, g, queue);
                else row_thread<1, EDGE>(a, g, queue);
            }
            queue.drain();
            __threadfence();                     // late tie flips (atomics) before the other colour reads them
            __syncthreads();
        }
    }
}

// ---- L = 64, 128: a replica in the registers of 16 / 32 lanes ----------------------------------
//
// WPR = words per row per colour (1 or 2), L = 64 WPR, LANES = 16 WPR lanes per replica, lane l
// owns rows 4l .. 4l+3 of both colours (4 WPR words per colour).  With P = i (L/2) + p the RNG
// unit is G = P >> 7: L = 64: G = i >> 2 = l (rows 4l..4l+3 are the block's words x, y, z, w);
// L = 128: G = i >> 1 = 2l + u, u = 0, 1 (rows 4l+2u, 4l+2u+1: words (row even: 0, 1; odd: 2, 3)).
// what PlaneLoop (ising_march.cuh) reads from its argument
struct TinyPlaneView {
    const PlaneFold &F;
    const RoundKeys &K;
    const uint32_t (&pcase)[8];
};

// Ties (top byte of u32 equal to the threshold's; 2^-8 per deciding lane) are resolved by the
// replica's lanes TOGETHER: the words that hold ties are queued in shared memory (one ballot per
// word, as in WarpTieQueue), then every lane takes one entry, evaluates the tail blocks of its tied
// bits and leaves the accepted flips in a per-word buffer that the owner reads back.  A lane that
// looped over its own ties alone would make the warp pay max-over-lanes(ties) tail blocks per
// half-sweep (~2.5) instead of ~1.
//   q    [LANES * NW] entries (tied lanes of the word, their dE = 8 mask, word offset, -)
//   fbuf [LANES * NW] accepted flips per word of the replica's colour
template <int COLOUR, int WPR, int PC>
__device__ __forceinline__ void tiny_half_sweep(uint32_t (&T)[4 * WPR], const uint32_t (&O)[4 * WPR],
                                                const RoundKeys &K, uint32_t t, const SweepParams &p,
                                                uint32_t ln, uint4 *q, uint32_t *fbuf)
{
    constexpr uint32_t LANES = 16 * WPR;
    PlaneFold F;
    build_plane_fold(K, t, (uint32_t)COLOUR, TAG_ACC_PLANE, F);
    const TinyPlaneView view{F, K, p.pcase};
    // opposite-colour rows 4l-1 (last row of the lane above) and 4l+4 (first row of the lane below)
    uint32_t up[WPR], dn[WPR];
#pragma unroll
    for (int w = 0; w < WPR; ++w) {
        up[w] = __shfl_sync(0xffffffffu, O[3 * WPR + w], (ln + LANES - 1u) % LANES, LANES);
        dn[w] = __shfl_sync(0xffffffffu, O[w], (ln + 1u) % LANES, LANES);
    }
    constexpr int NW = 4 * WPR;
    uint32_t need[NW], c8[NW], acc[NW], eq[NW];              // word x = r * WPR + w of the lane
#pragma unroll
    for (int u = 0; u < WPR; ++u) {
        uint32_t uc8[4], uacc[4], ueq[4];
#pragma unroll
        for (int qq = 0; qq < 4; ++qq) {
            const int r = WPR == 1 ? qq : 2 * u + (qq >> 1), w = WPR == 1 ? 0 : (qq & 1), x = r * WPR + w;
            const uint32_t U = r == 0 ? up[w] : O[(r > 0 ? r - 1 : 0) * WPR + w];
            const uint32_t D = r == 3 ? dn[w] : O[(r < 3 ? r + 1 : 3) * WPR + w];
            const uint32_t C = O[x];
            uint32_t S;                                               // (i + colour) & 1 = (r + COLOUR) & 1
            if (((r + COLOUR) & 1) == 0) S = fsl1(O[r * WPR + (w + WPR - 1) % WPR], C);   // neighbour at p-1
            else S = fsr1(C, O[r * WPR + (w + 1) % WPR]);                                // neighbour at p+1
            const uint32_t s1 = U ^ D ^ C, c1 = maj3m(U, D, C), tt = T[x];
            const uint32_t m = lop3<0xE7>(tt, s1, S);
            const uint32_t nd = lop3<0x82>(c1, tt, m);               // k >= 3
            const uint32_t k4 = lop3<0x90>(nd, s1, S);               // k == 4
            // classes whose threshold is 2^32 flip unconditionally (masks are ~0 otherwise)
            need[x] = ((nd & ~k4) & p.mask4) | (k4 & p.mask8);
            uc8[qq] = k4 & p.mask8;
            ueq[qq] = need[x];
            uacc[qq] = 0;
        }
        const uint32_t G = WPR == 1 ? ln : 2u * ln + (uint32_t)u;
        const PlaneShared ps = plane_shared(G, F);
        PlaneLoop<PC, 7>::run(view, ps, uc8, uacc, ueq);
#pragma unroll
        for (int qq = 0; qq < 4; ++qq) {
            const int r = WPR == 1 ? qq : 2 * u + (qq >> 1), w = WPR == 1 ? 0 : (qq & 1), x = r * WPR + w;
            c8[x] = uc8[qq]; acc[x] = uacc[qq]; eq[x] = ueq[qq];
        }
    }
    // ---- ties: queue the words (group = the LANES lanes of this replica), resolve together ----
    const uint32_t lane = threadIdx.x & 31u;
    const uint32_t gmask = WPR == 1 ? 0xffffu << (lane & 16u) : 0xffffffffu;
    const uint32_t below = gmask & ((1u << lane) - 1u);
    uint32_t pending = 0;
#pragma unroll
    for (int x = 0; x < NW; ++x) {
        const bool has = eq[x] != 0;
        const uint32_t m = __ballot_sync(0xffffffffu, has) & gmask;
        if (has) q[pending + __popc(m & below)] = make_uint4(eq[x], c8[x], ln * (uint32_t)NW + (uint32_t)x, 0u);
        pending += __popc(m);
    }
    __syncwarp();
    if (__any_sync(0xffffffffu, pending != 0u)) {
        for (uint32_t base = 0; __any_sync(0xffffffffu, base < pending); base += LANES) {
            const uint32_t idx = base + ln;
            if (idx < pending) {
                const uint4 e = q[idx];
                uint32_t ties = e.x, flip = 0;
                while (ties) {
                    const uint32_t bit = __ffs(ties) - 1;
                    ties &= ties - 1;
                    const uint32_t P = (e.z << 5) + bit;             // word offset i * wpr + w = 4 ln WPR + x
                    const uint4 blk = philox4x32_10(P, 0u, t, (uint32_t)COLOUR | (TAG_ACC_TAIL << 8), K);
                    const unsigned long long thr = ((e.y >> bit) & 1u) ? p.thr8 : p.thr4;
                    const unsigned long long u56 = ((unsigned long long)(blk.x >> 8) << 32) | blk.y;
                    if (u56 < (thr & 0x00ffffffffffffffull)) flip |= 1u << bit;
                }
                fbuf[e.z] = flip;
            }
        }
        __syncwarp();
#pragma unroll
        for (int x = 0; x < NW; ++x)
            if (eq[x]) acc[x] |= fbuf[ln * (uint32_t)NW + (uint32_t)x];
        __syncwarp();                                            // before the next half-sweep reuses q / fbuf
    }
#pragma unroll
    for (int x = 0; x < NW; ++x) T[x] = lop3<0x4B>(T[x], need[x], acc[x]);       // T ^ (~need | acc)
}

// resident blocks of 128 threads per SM: 4 (<= 128 registers) measured fastest for L = 64; L = 128
// keeps twice the state per lane and would spill under that cap.  PC >= 0: every sweep of the call
// has the packed plane cases PC (ising_march.cuh) compiled in.
template <int WPR, int PC = -1>
__global__ void __launch_bounds__(128, WPR == 1 ? LAT_TINY_MINB : 3) ising_tiny_kernel(uint32_t *buf, const RoundKeys *keys,
                                                         const SweepParams *sp, uint32_t n_rep,
                                                         uint32_t t0, uint32_t n_sweeps)
{
    constexpr uint32_t L = 64 * WPR, LANES = 16 * WPR, NW = 4 * WPR;
    __shared__ uint4 s_q[128 * NW];                           // [group][LANES * NW]
    __shared__ uint32_t s_f[128 * NW];
    const uint32_t gt = blockIdx.x * blockDim.x + threadIdx.x;
    const uint32_t rep = gt / LANES, ln = gt % LANES;
    if ((gt & ~31u) / LANES >= n_rep) return;                 // the whole warp is past the last replica
    const bool live = rep < n_rep;                            // L = 64: a warp may hold one live half
    const uint32_t r_eff = live ? rep : n_rep - 1u;           // dead lanes shadow the last replica
    uint32_t *base = buf + (size_t)r_eff * (2u * L * WPR) + (size_t)(4u * ln) * WPR;
    uint4 *q = s_q + (threadIdx.x / LANES) * (LANES * NW);
    uint32_t *fbuf = s_f + (threadIdx.x / LANES) * (LANES * NW);
    const RoundKeys K = keys[r_eff];
    uint32_t s0[NW], s1[NW];                                  // colour 0 / 1, rows 4 ln .. 4 ln + 3
#pragma unroll
    for (int j = 0; j < (int)NW; j += 4) {
        const uint4 a = *reinterpret_cast<const uint4 *>(base + j);
        const uint4 b = *reinterpret_cast<const uint4 *>(base + (size_t)L * WPR + j);
        s0[j] = a.x; s0[j + 1] = a.y; s0[j + 2] = a.z; s0[j + 3] = a.w;
        s1[j] = b.x; s1[j + 1] = b.y; s1[j + 2] = b.z; s1[j + 3] = b.w;
    }
#pragma unroll 1
    for (uint32_t sw = 0; sw < n_sweeps; ++sw) {
        const SweepParams p = sp[sw];
        tiny_half_sweep<0, WPR, PC>(s0, s1, K, t0 + sw, p, ln, q, fbuf);   // black sees the old white
        tiny_half_sweep<1, WPR, PC>(s1, s0, K, t0 + sw, p, ln, q, fbuf);   // white sees the new black
    }
    if (live) {
#pragma unroll
        for (int j = 0; j < (int)NW; j += 4) {
            *reinterpret_cast<uint4 *>(base + j) = make_uint4(s0[j], s0[j + 1], s0[j + 2], s0[j + 3]);
            *reinterpret_cast<uint4 *>(base + (size_t)L * WPR + j) = make_uint4(s1[j], s1[j + 1], s1[j + 2], s1[j + 3]);
        }
    }
}
#endif

}  // namespace lat
