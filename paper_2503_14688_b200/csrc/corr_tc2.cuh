// corr_tc2.cuh -- dense axis correlations on the tensor cores with CTA PAIRS (tcgen05 cta_group::2).
//
// Same mathematics, operand encoding and exactness argument as corr_tc.cuh (Eq. 2: the
// band of the row / column Gram matrix; spins as fp8 +-1.0 / 0.0, fp32 accumulators holding exact
// integers).  What changes is how the work is laid on the machine.  corr_tc_kernel is bound by the
// L1/shared-memory data pipe (profiles/r2_corr_tc.md): per 128-step stage one CTA stores 80 KiB of
// expanded operands, the tensor core reads 96 KiB of them (the base tile once per N tile) and every
// expanded byte is first a per-lane global load.  Here a cluster of two CTAs (the two SMs of a TPC)
// shares one work item of 256 base x 512 partner positions: one `tcgen05.mma.cta_group::2` of shape
// 256 x 256 x 32 takes the 128 base rows of EACH CTA from that CTA's own shared memory and HALF of the
// 256 partner rows from each, and leaves each CTA's half of the accumulator in its own tensor memory.
// Per CTA and stage that is 48 KiB stored and 64 KiB read (112 instead of 176 KiB through the pipe) and
// 0.6 x the global loads, and four stages fit in shared memory instead of two.
//
//   * CTA rank 0 (the leader) issues all MMAs; the `full` barriers live in its shared memory and collect
//     one arrival per producer warp of BOTH CTAs (the peer arrives through the cluster address);
//   * `tcgen05.commit ... multicast::cluster` releases a stage / publishes the accumulators in both CTAs;
//   * each CTA's warps 0-3 read their own accumulator half back and bin it; the leader waits for both
//     epilogues (`tfree`) before the first MMA of the next item overwrites the accumulators.
#pragma once
#include "corr_tc.cuh"

namespace lat {

constexpr int T2_M = 128;             // base positions per CTA (256 per pair)
constexpr int T2_N = 256;             // partner positions per MMA (128 staged by each CTA)
constexpr int T2_NT = 2;              // N tiles per item: 2 * 256 fp32 columns = the 512 TMEM columns
constexpr int T2_KC = 128;            // contraction positions per stage
constexpr int T2_STAGES = 4;
constexpr int T2_BLK_BYTES = 128 * T2_KC;                     // one 128-row block: 16 KiB
constexpr int T2_STAGE_BYTES = (1 + T2_NT) * T2_BLK_BYTES;    // A + two B halves: 48 KiB
constexpr int T2_PRODUCERS = 768;     // one 64-byte chunk per thread and stage (24 warps); warp 24 issues the MMAs
constexpr int T2_THREADS = T2_PRODUCERS + 32;
constexpr int T2_HIST = T2_NT * T2_N + 2 * T2_M;              // r - 512 pass + 255 in [0, 767)
constexpr int T2_SMEM_BYTES = T2_STAGES * T2_STAGE_BYTES + 1024 /* alignment */ + T2_HIST * 4 + 64;

#ifdef __CUDACC__
namespace tc {

__device__ __forceinline__ uint32_t cluster_rank()
{
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_sync()
{
    asm volatile("barrier.cluster.arrive.release.aligned;\n\tbarrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// address of the same shared-memory location in CTA `rank` of the cluster
__device__ __forceinline__ uint32_t map_to_rank(uint32_t saddr, uint32_t rank)
{
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(saddr), "r"(rank));
    return r;
}
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t cluster_addr)
{
    // default semantics (release at CTA scope), as CUTLASS' ClusterBarrier::arrive does: what the barrier
    // orders is read by the tensor cores (made visible by fence.proxy.async / tcgen05 fences), not by
    // generic loads of the waiting thread; `.release.cluster` here compiled to a full MEMBAR per arrive
    // and `.acquire.cluster` on the waits to a cache invalidate per poll (1.4 x slower than one CTA)
    asm volatile("mbarrier.arrive.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
// bounded spin on a barrier that is (also) arrived at from the peer CTA or by a multicast commit
__device__ __forceinline__ void mbar_wait_cluster(uint32_t bar, uint32_t parity)
{
    for (uint32_t spin = 0;; ++spin) {
        uint32_t ok;
        asm volatile("{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
                     "selp.u32 %0, 1, 0, p;\n\t}"
                     : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
        if (ok) return;
        if (spin > (1u << 28)) __trap();
    }
}
// D[tmem of both CTAs] (+)= A[smem of both] * B[smem halves of both], kind::f8f6f4, issued by one thread of the leader
__device__ __forceinline__ void umma2_f8(uint32_t tmem_d, uint64_t desc_a, uint64_t desc_b, uint32_t idesc,
                                         uint32_t accumulate)
{
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::2.kind::f8f6f4 [%0], %1, %2, %3, p;\n\t}"
                 ::"r"(tmem_d), "l"(desc_a), "l"(desc_b), "r"(idesc), "r"(accumulate) : "memory");
}
// arrive (once all MMAs issued so far are done) on the barrier at this offset in BOTH CTAs
__device__ __forceinline__ void umma2_commit_both(uint32_t bar)
{
    asm volatile("{\n\t.reg .b16 m;\n\tmov.b16 m, 3;\n\t"
                 "tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], m;\n\t}"
                 ::"r"(bar) : "memory");
}

}  // namespace tc

// AXIS 1 (y): positions are rows, the contraction runs over the columns of a row.
// AXIS 0 (x): positions are columns, the contraction runs over rows i0 .. i0 + n_rows - 1.
// a.n_tiles counts PAIR tiles of 256 base positions; a.n_pass = ceil((r_max + 256) / 512).
template <int MODEL, int AXIS>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(T2_THREADS, 1) corr_tc2_kernel(const CorrTCArgs a)
{
    using namespace tc;
    extern __shared__ uint8_t tc2_smem_raw[];
    uint8_t *smem = (uint8_t *)(((uintptr_t)tc2_smem_raw + 1023) & ~(uintptr_t)1023);     // swizzle atoms: 1 KiB
    int *hist = (int *)(smem + T2_STAGES * T2_STAGE_BYTES);
    __shared__ __align__(8) unsigned long long bars[2 * T2_STAGES + 2];
    __shared__ uint32_t tmem_base_s;

    // two producer groups, each owning pairs of stages (below): measured -4 % for Ising (7.6 -> 7.4 s at
    // L = 2^20), +6 % for Blume-Capel (its second plane costs registers: spills under the 80-register cap)
    constexpr bool T2_GROUPS = AXIS == 1 && MODEL == 0;
    const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31u;
    const uint32_t rank = cluster_rank();                     // 0 = leader (issues the MMAs)
    const uint32_t full0 = smem_u32(&bars[0]), empty0 = smem_u32(&bars[T2_STAGES]),
                   accf = smem_u32(&bars[2 * T2_STAGES]), tfree = smem_u32(&bars[2 * T2_STAGES + 1]);
    const uint32_t full0_leader = map_to_rank(full0, 0u), tfree_leader = map_to_rank(tfree, 0u);

    if (threadIdx.x == 0) {
        for (int s = 0; s < T2_STAGES; ++s) {
            // one arrive per producer warp that fills the stage, in both CTAs: all 24 warps (x axis), or the
            // 12 warps of the group that owns the stage (Ising y axis, below)
            mbar_init(full0 + 8 * s, T2_GROUPS ? T2_PRODUCERS / 32 : 2 * (T2_PRODUCERS / 32));
            mbar_init(empty0 + 8 * s, 1);                         // tcgen05.commit (multicast)
        }
        mbar_init(accf, 1);
        mbar_init(tfree, 8);                                      // the four epilogue warps of both CTAs
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == T2_PRODUCERS / 32) {                              // the same warp in both CTAs
        asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)), "n"(512));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::);
    }
    fence_before_sync();
    __syncthreads();
    cluster_sync();                                               // the peer's barriers exist before anyone arrives
    fence_after_sync();
    const uint32_t tmem = tmem_base_s;

    const size_t pw = (size_t)a.rows * a.wpr;                     // words per plane
    const uint32_t n_kc = AXIS == 1 ? a.L / T2_KC : (a.n_rows + T2_KC - 1) / T2_KC;
    // instruction descriptor: fp32 accumulate, e4m3 x e4m3, N >> 3 in [17,23), M >> 4 in [24,29) with the
    // PAIR's M = 256, bits 15 / 16 = MN-major A / B (x axis)
    const uint32_t idesc = (1u << 4) | ((uint32_t)(T2_N >> 3) << 17) | ((uint32_t)((2 * T2_M) >> 4) << 24) |
                           (AXIS == 0 ? (1u << 15) | (1u << 16) : 0u);
    const uint32_t n_pairs = gridDim.x >> 1, pair = blockIdx.x >> 1;

    uint32_t sbase = 0, acc_phase = 0;                            // stages done before this item
    for (uint32_t item = pair; item < a.n_items; item += n_pairs, sbase += n_kc) {
        const uint32_t pass = item / a.n_tiles, tile = item - pass * a.n_tiles;
        // first base position of the pair's tile; this CTA's own base block starts 128 * rank further
        const uint32_t p0 = (AXIS == 1 ? a.i0 : 0u) + tile * (2u * T2_M);
        const uint32_t w0 = p0 + pass * (T2_NT * T2_N);           // first partner position of the pass
        // ===== epilogue (warps 0-3: TMEM lane quarter = warp): this CTA's 128 base positions =====
        auto epilogue = [&]() {
            if (warp < 4) {
            for (uint32_t t = threadIdx.x; t < (uint32_t)T2_HIST; t += 128u) hist[t] = 0;
            asm volatile("bar.sync 1, 128;" ::: "memory");
            mbar_wait_cluster(accf, acc_phase);
            fence_after_sync();
            const uint32_t m = warp * 32u + lane;             // base position index in this CTA's block
            // position of byte index x inside a 128-block: natural for y; [64 even | 64 odd] and the
            // byte order of expand_word inside each 32-byte group for x (corr_tc.cuh)
            const int pm = (int)(T2_M * rank) +
                           (AXIS == 1 ? (int)m : (int)(2u * ((m & 32u) + tc_spin_of_byte(m & 31u)) + (m >> 6)));
#pragma unroll 1
            for (uint32_t cb = 0; cb < (uint32_t)(T2_NT * T2_N); cb += 16u) {
                uint32_t v[16];
                asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 "
                             "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
                             : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]),
                               "=r"(v[7]), "=r"(v[8]), "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]),
                               "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
                             : "r"(tmem + ((warp * 32u) << 16) + cb));
                asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
                for (int e = 0; e < 16; ++e) {
                    // column n of the accumulators <-> partner position: N tile n >> 8, inside it the
                    // leader's 128 partner rows first, then the peer's: the natural order of the window
                    const uint32_t n = cb + (uint32_t)e;
                    int pn;
                    if (AXIS == 1) pn = (int)n;
                    else {
                        const uint32_t nb = n & 127u;
                        pn = (int)((n & ~127u) + 2u * ((nb & 32u) + tc_spin_of_byte(nb & 31u)) + (nb >> 6));
                    }
                    const int d = pn - pm;                     // r - 512 pass, in (-256, 512)
                    const long long r = (long long)d + (long long)pass * (T2_NT * T2_N);
                    const int val = __float2int_rn(__uint_as_float(v[e]));
                    if (r >= 1 && r <= (long long)a.r_max && val) atomicAdd(&hist[d + (2 * T2_M - 1)], val);
                }
            }
            // this CTA's accumulators are read: tell the leader (it waits for both CTAs)
            fence_before_sync();
            __syncwarp();
            if (lane == 0) mbar_arrive_cluster(tfree_leader);
            asm volatile("bar.sync 1, 128;" ::: "memory");
            for (uint32_t t = threadIdx.x; t < (uint32_t)T2_HIST; t += 128u) {
                const long long r = (long long)t - (2 * T2_M - 1) + (long long)pass * (T2_NT * T2_N);
                if (hist[t] && r >= 1 && r <= (long long)a.r_max)
                    atomicAdd((unsigned long long *)(a.S + (r - 1) * a.s_stride), (unsigned long long)(long long)hist[t]);
            }
            asm volatile("bar.sync 1, 128;" ::: "memory");
        }
        };
        if (T2_GROUPS && warp < T2_PRODUCERS / 32) {
            // ===== producers, Ising y axis: two groups of 12 warps; group g fills the stage PAIRS 4 j + 2 g, 4 j + 2 g + 1
            // of the item (one 16-byte load = both stages of a pair), two 64-byte chunks per thread and
            // stage.  The per-stage overhead of a warp (barrier wait, proxy fence, arrive) is paid once per
            // two chunks, and one group expands while the other waits for its stores to drain.
            constexpr uint32_t GRP = T2_PRODUCERS / 2;            // 384 threads
            const uint32_t grp = threadIdx.x / GRP, tg = threadIdx.x - grp * GRP;
            const uint32_t *src[2];
            uint32_t dst[2], r7[2], c0[2];
            bool zero[2];
#pragma unroll
            for (int q = 0; q < 2; ++q) {
                const uint32_t it = tg + (uint32_t)q * GRP, tr = it >> 1, h = it & 1u;   // 0..127 base rows, 128..383 partner rows
                const uint32_t mb = tr / T2_M, srow = tr % T2_M;
                uint32_t i;
                zero[q] = false;
                if (mb == 0) { i = p0 + T2_M * rank + srow; zero[q] = i >= a.i0 + a.n_rows; }
                else i = w0 + (mb - 1u) * T2_N + T2_M * rank + srow;
                const uint32_t row_l = i % a.rows, c = (row_l & 1u) ^ h;
                src[q] = a.buf + (MODEL == 0 ? (size_t)c * pw : (size_t)(2u * c) * pw) + (size_t)row_l * a.wpr;
                dst[q] = mb * T2_BLK_BYTES + (srow >> 3) * 1024u + (srow & 7u) * 128u;
                r7[q] = srow & 7u; c0[q] = h << 2;
            }
            uint4 cur[2], curs[2], nxt[2], nxts[2];
#pragma unroll
            for (int q = 0; q < 2; ++q) {
                cur[q] = curs[q] = nxt[q] = nxts[q] = make_uint4(0u, 0u, 0u, 0u);
                const uint32_t k0 = 2u * grp, k1 = k0 + 4u;                              // first stages of the first two pairs
                if (!zero[q] && k0 < n_kc) {
                    cur[q] = *reinterpret_cast<const uint4 *>(src[q] + 2 * (size_t)k0);
                    if (MODEL) curs[q] = *reinterpret_cast<const uint4 *>(src[q] + 2 * (size_t)k0 + pw);
                }
                if (!zero[q] && k1 < n_kc) {
                    nxt[q] = *reinterpret_cast<const uint4 *>(src[q] + 2 * (size_t)k1);
                    if (MODEL) nxts[q] = *reinterpret_cast<const uint4 *>(src[q] + 2 * (size_t)k1 + pw);
                }
            }
            for (uint32_t kp = 2u * grp; kp < n_kc; kp += 4u) {
#pragma unroll
                for (int v = 0; v < 2; ++v) {
                    const uint32_t sg = sbase + kp + (uint32_t)v, slot = sg % T2_STAGES;
                    mbar_wait_cluster(empty0 + 8 * slot, ((sg / T2_STAGES) & 1u) ^ 1u);
                    const uint32_t st = smem_u32(smem) + slot * T2_STAGE_BYTES;
#pragma unroll
                    for (int q = 0; q < 2; ++q) {
                        uint4 o[4];
                        if (zero[q]) o[0] = o[1] = o[2] = o[3] = make_uint4(0u, 0u, 0u, 0u);
                        else {
                            expand_word<MODEL>(v ? cur[q].z : cur[q].x, v ? curs[q].z : curs[q].x, o[0], o[1]);
                            expand_word<MODEL>(v ? cur[q].w : cur[q].y, v ? curs[q].w : curs[q].y, o[2], o[3]);
                        }
#pragma unroll
                        for (int e = 0; e < 4; ++e)
                            asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(st + dst[q] + (((c0[q] + (uint32_t)e) ^ r7[q]) << 4)),
                                         "r"(o[e].x), "r"(o[e].y), "r"(o[e].z), "r"(o[e].w) : "memory");
                    }
                    fence_proxy_async();                          // generic-proxy writes -> visible to the tensor core
                    __syncwarp();
                    if (lane == 0) mbar_arrive_cluster(full0_leader + 8 * slot);
                }
                const uint32_t nk = kp + 8u;                      // the pair after the next one
#pragma unroll
                for (int q = 0; q < 2; ++q) {
                    cur[q] = nxt[q]; curs[q] = nxts[q];
                    nxt[q] = nxts[q] = make_uint4(0u, 0u, 0u, 0u);
                    if (!zero[q] && nk < n_kc) {
                        nxt[q] = *reinterpret_cast<const uint4 *>(src[q] + 2 * (size_t)nk);
                        if (MODEL) nxts[q] = *reinterpret_cast<const uint4 *>(src[q] + 2 * (size_t)nk + pw);
                    }
                }
            }
            epilogue();
            acc_phase ^= 1u;
        } else if (warp < T2_PRODUCERS / 32) {
            // ===== producers: one 64-byte chunk of the stage per thread =====
            // blocks of 128 smem rows: 0 = this CTA's base block, 1 + nt = this CTA's half of N tile nt
            const uint32_t it = threadIdx.x;
            uint32_t h, srow, mb, row_l, word, kc_zero = 0xffffffffu;
            if (AXIS == 1) {
                const uint32_t tr = it >> 1;                      // 0..127 base rows, 128..383 partner rows
                h = it & 1u;
                mb = tr / T2_M;
                srow = tr % T2_M;
                uint32_t i;
                if (mb == 0) { i = p0 + T2_M * rank + srow; if (i >= a.i0 + a.n_rows) kc_zero = 0u; }
                else i = w0 + (mb - 1u) * T2_N + T2_M * rank + srow;
                row_l = i % a.rows;
                word = 0u;                                        // + 2 words (64 packed positions) per step
            } else {
                // chunks 0..511: the two partner blocks, the block index varying faster than the upper bits
                // of the row, so that the 32 lanes of a load read 16 rows x 2 blocks (16 lines, the blocks of a
                // row are 32 bytes apart) while a quarter-warp still stores to 8 consecutive rows;
                // chunks 512..767: the base block (srow = contraction index = lattice row of the stage)
                if (it < 4u * T2_KC) {
                    srow = ((it >> 4) & 15u) * 8u + (it & 7u);
                    mb = 1u + ((it >> 3) & 1u);
                    h = it >> 8;
                } else {
                    srow = it % T2_KC;
                    mb = 0u;
                    h = (it - 4u * T2_KC) / T2_KC;
                }
                row_l = a.i0 + srow;                              // + T2_KC rows per step; never wraps
                kc_zero = srow < a.n_rows ? (a.n_rows - srow + T2_KC - 1) / T2_KC : 0u;
                const uint32_t col0 = (mb == 0 ? p0 + T2_M * rank : w0 + (mb - 1u) * T2_N + T2_M * rank) % a.L;
                word = col0 / 64u;                                // 128 columns = 64 packed positions = 2 words
            }
            const uint32_t c = (row_l & 1u) ^ h;                  // even columns of row i live in colour i & 1
            const uint32_t *src = a.buf + (MODEL == 0 ? (size_t)c * pw : (size_t)(2u * c) * pw) + (size_t)row_l * a.wpr + word;
            // canonical 128-byte swizzle: 8-row atoms of 1 KiB, 16-byte chunk index ^ (row & 7)
            const uint32_t dst = mb * T2_BLK_BYTES + (srow >> 3) * 1024u + (srow & 7u) * 128u;
            const uint32_t r7 = srow & 7u, c0 = h << 2;
            auto put = [&](uint32_t st, uint32_t wa, uint32_t sa_, uint32_t wb_, uint32_t sb_, bool zero) {
                uint4 o[4];
                if (zero) o[0] = o[1] = o[2] = o[3] = make_uint4(0u, 0u, 0u, 0u);
                else { expand_word<MODEL>(wa, sa_, o[0], o[1]); expand_word<MODEL>(wb_, sb_, o[2], o[3]); }
#pragma unroll
                for (int e = 0; e < 4; ++e)
                    asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(st + dst + (((c0 + (uint32_t)e) ^ r7) << 4)),
                                 "r"(o[e].x), "r"(o[e].y), "r"(o[e].z), "r"(o[e].w) : "memory");
            };
            auto publish = [&](uint32_t slot) {
                fence_proxy_async();                              // generic-proxy writes -> visible to the tensor core
                __syncwarp();
                if (lane == 0) mbar_arrive_cluster(full0_leader + 8 * slot);
            };
            const size_t step = AXIS == 1 ? 2u : (size_t)T2_KC * a.wpr;      // words per contraction step
            if constexpr (AXIS == 1) {
                // 16-byte loads = two steps each (rows are 16-byte aligned: L % 256 == 0; n_kc is even);
                // ring of TC2_PF such loads, reloaded for step kc + 2 TC2_PF after the second of its steps
                constexpr int TC2_PF = 2;
                uint4 wb[TC2_PF], sb[TC2_PF];
#pragma unroll
                for (int u = 0; u < TC2_PF; ++u) {
                    wb[u] = sb[u] = make_uint4(0u, 0u, 0u, 0u);
                    if (2u * (uint32_t)u < n_kc && kc_zero != 0u) {
                        wb[u] = *reinterpret_cast<const uint4 *>(src + 4 * u);
                        if (MODEL) sb[u] = *reinterpret_cast<const uint4 *>(src + 4 * u + pw);
                    }
                }
                for (uint32_t kc0 = 0; kc0 < n_kc; kc0 += 2u * TC2_PF) {
#pragma unroll
                    for (int uv = 0; uv < 2 * TC2_PF; ++uv) {
                        const int u = uv >> 1, v = uv & 1;
                        const uint32_t kc = kc0 + (uint32_t)uv;
                        if (kc >= n_kc) break;
                        const uint32_t s = sbase + kc, slot = s % T2_STAGES;
                        mbar_wait_cluster(empty0 + 8 * slot, ((s / T2_STAGES) & 1u) ^ 1u);
                        put(smem_u32(smem) + slot * T2_STAGE_BYTES, v ? wb[u].z : wb[u].x, v ? sb[u].z : sb[u].x,
                            v ? wb[u].w : wb[u].y, v ? sb[u].w : sb[u].y, kc_zero == 0u);
                        publish(slot);
                        if (v == 1) {
                            const uint32_t nk = kc0 + 2u * (uint32_t)u + 2u * TC2_PF;
                            wb[u] = sb[u] = make_uint4(0u, 0u, 0u, 0u);
                            if (nk < n_kc && kc_zero != 0u) {
                                wb[u] = *reinterpret_cast<const uint4 *>(src + 2 * (size_t)nk);
                                if (MODEL) sb[u] = *reinterpret_cast<const uint4 *>(src + 2 * (size_t)nk + pw);
                            }
                        }
                    }
                }
            } else {
                constexpr int TC2_PF = 4;                         // one step per 8-byte load, 4 steps ahead
                uint2 wb[TC2_PF], sb[TC2_PF];
#pragma unroll
                for (int u = 0; u < TC2_PF; ++u) {
                    wb[u] = sb[u] = make_uint2(0u, 0u);
                    if ((uint32_t)u < n_kc && (uint32_t)u < kc_zero) {
                        wb[u] = *reinterpret_cast<const uint2 *>(src + (size_t)u * step);
                        if (MODEL) sb[u] = *reinterpret_cast<const uint2 *>(src + (size_t)u * step + pw);
                    }
                }
                for (uint32_t kc0 = 0; kc0 < n_kc; kc0 += TC2_PF) {
#pragma unroll
                    for (int u = 0; u < TC2_PF; ++u) {
                        const uint32_t kc = kc0 + (uint32_t)u;
                        if (kc >= n_kc) break;
                        const uint32_t s = sbase + kc, slot = s % T2_STAGES;
                        mbar_wait_cluster(empty0 + 8 * slot, ((s / T2_STAGES) & 1u) ^ 1u);
                        put(smem_u32(smem) + slot * T2_STAGE_BYTES, wb[u].x, sb[u].x, wb[u].y, sb[u].y, kc >= kc_zero);
                        publish(slot);
                        const uint32_t nk = kc + (uint32_t)TC2_PF;
                        wb[u] = sb[u] = make_uint2(0u, 0u);
                        if (nk < n_kc && nk < kc_zero) {
                            wb[u] = *reinterpret_cast<const uint2 *>(src + (size_t)nk * step);
                            if (MODEL) sb[u] = *reinterpret_cast<const uint2 *>(src + (size_t)nk * step + pw);
                        }
                    }
                }
            }
            epilogue();
            acc_phase ^= 1u;
        } else if (rank == 0) {
            // ===== MMA issuer: one elected thread of the leader CTA =====
            if (sbase) {                                          // accumulators of the previous item read back?
                mbar_wait_cluster(tfree, acc_phase ^ 1u);
                fence_after_sync();
            }
            for (uint32_t kc = 0; kc < n_kc; ++kc) {
                const uint32_t s = sbase + kc, slot = s % T2_STAGES;
                mbar_wait_cluster(full0 + 8 * slot, (s / T2_STAGES) & 1u);
                fence_after_sync();
                if (lane == 0) {
                    const uint32_t sa = smem_u32(smem) + slot * T2_STAGE_BYTES;
#pragma unroll
                    for (uint32_t k = 0; k < T2_KC / 32; ++k) {
#pragma unroll
                        for (uint32_t nt = 0; nt < (uint32_t)T2_NT; ++nt) {
                            const uint32_t sb = sa + (1u + nt) * T2_BLK_BYTES;
                            uint64_t da, db;
                            if (AXIS == 1) {
                                // K-major: rows of 128 bytes along K, 8-row atoms 1 KiB apart; a K step of
                                // 32 bytes moves the start address inside the swizzled row
                                da = umma_desc(sa + k * 32u, 16u, 1024u);
                                db = umma_desc(sb + k * 32u, 16u, 1024u);
                            } else {
                                // MN-major: one 128-column block per CTA and operand, one smem row per
                                // contraction index, 8-row atoms along K 1 KiB apart; a K step of 32 = 4 atoms
                                da = umma_desc(sa + k * 4096u, T2_BLK_BYTES, 1024u);
                                db = umma_desc(sb + k * 4096u, T2_BLK_BYTES, 1024u);
                            }
                            umma2_f8(tmem + nt * T2_N, da, db, idesc, (kc | k) ? 1u : 0u);
                        }
                    }
                    umma2_commit_both(empty0 + 8 * slot);         // slot reusable in both CTAs once these MMAs are done
                    if (kc + 1 == n_kc) umma2_commit_both(accf);  // accumulators complete in both CTAs
                }
                __syncwarp();
            }
            acc_phase ^= 1u;
        } else {
            acc_phase ^= 1u;                                      // the peer's MMA warp only owns the TMEM allocation
        }
    }
    fence_before_sync();
    __syncthreads();
    cluster_sync();                                               // nobody touches the peer's memory any more
    if (warp == T2_PRODUCERS / 32) {
        fence_after_sync();
        asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(512));
    }
}
#endif

}  // namespace lat
