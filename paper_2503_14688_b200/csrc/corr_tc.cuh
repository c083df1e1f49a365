// corr_tc.cuh -- dense axis correlations S_x(r), S_y(r), r <= r_max, on the 5th-generation tensor
// cores (tcgen05 + TMEM): the one-CTA-per-item kernel.  Since round 2's last third the CTA-pair
// kernel of corr_tc2.cuh (which reuses the helpers and the operand encoding defined here) takes the y
// axis and, on transposed bands (corr_transpose.cuh), the x axis; this kernel keeps the x axis of rows
// that are not whole 512-row bands, of odd first rows and of lattices with L not a multiple of 2048 (its
// MN-major operands need no copy), and both axes on request (lattice_set_measure_path 4).
//
// Paper: C(r;t), Eq. 2, along the lattice axes.  Dense in r this IS a dense
// contraction: S_y(r) = sum_i G[i, i+r] with the band of the row Gram matrix
//     G[i, i'] = sum_j s(i, j) s(i', j),
// and S_x(r) the same with rows and columns exchanged.  The XOR/popcount kernels of measure.cuh
// pay ~3 integer instructions per (32 spins, r); on the tensor cores one tcgen05.mma of shape
// 128 x 256 x 32 (fp8 e4m3, fp32 accumulate) does 2^20 spin products.  Spins are exactly
// representable (+1 = 0x38, -1 = 0xB8, 0 = 0x00) and |G| <= L <= 2^20 < 2^24, so the fp32
// accumulators hold exact integers: the result is the same exact integer count as the popcount path.
//
// One CTA per SM, persistent over work items (tile of 128 base positions, pass of 512 partner
// positions starting at the tile's first position + 512 * pass).  Per item the whole lattice extent
// along the contraction axis streams through a 2-stage shared-memory ring:
//   * 20 producer warps read the packed words (1 or 2 bits per spin), expand them to fp8 bytes and
//     write them into the canonical 128-byte-swizzled UMMA layout (K-major for the y axis, where the
//     contraction runs along a row; MN-major for the x axis, where it runs across rows);
//   * one thread of a 21st warp issues 8 tcgen05.mma per stage (4 K-steps x 2 N-tiles of 256) into
//     two 128 x 256 fp32 accumulators that fill the 512 TMEM columns, and commits to the stage's
//     "empty" mbarrier;
//   * after the last stage warps 0-3 read the accumulators back (tcgen05.ld, lane = base position)
//     and add every element with 1 <= r <= r_max to a per-item histogram in shared memory, which is
//     flushed to 64-bit global counters.
// Within a 128-position block the byte order is [64 even columns | 64 odd columns] of the row for
// the x axis (and the same split of the contraction index for the y axis), and within each 32-spin
// word the order expand_word produces: that is the order the sublattice packing and the cheapest
// bit -> byte expansion deliver, the same for both operands, and the epilogue undoes it.
#pragma once
#include <stdint.h>

namespace lat {

constexpr int TC_M = 128;            // base positions per item
constexpr int TC_N = 256;            // partner positions per MMA
constexpr int TC_NT = 2;             // N tiles per item (TC_NT * TC_N = 512 TMEM columns)
constexpr int TC_KC = 128;           // contraction positions per stage (one 128-byte swizzle row)
constexpr int TC_STAGES = 2;
constexpr int TC_PRODUCERS = 640;    // producer threads (warps 0-19: 2 chunks of 64 bytes each per stage); warp 20 issues the MMAs
constexpr int TC_THREADS = TC_PRODUCERS + 32;
constexpr int TC_STAGE_BYTES = (TC_M + TC_NT * TC_N) * TC_KC;            // 80 KiB
constexpr int TC_HIST = TC_NT * TC_N + TC_M;                             // r - 512 pass + 127 in [0, 639)
constexpr int TC_SMEM_BYTES = TC_STAGES * TC_STAGE_BYTES + 1024 /* alignment */ + TC_HIST * 4 + 64;

struct CorrTCArgs {
    const uint32_t *buf;
    uint32_t L;                      // lattice side: extent of a row, period along x
    uint32_t rows;                   // rows per plane in the buffer (L, or a view's row count): period along y
    uint32_t wpr;
    uint32_t i0, n_rows;             // base rows i0 .. i0 + n_rows - 1
    uint32_t r_max;
    uint32_t n_tiles, n_pass, n_items;
    long long *S;                    // signed sums of this axis: S[(r - 1) * s_stride] (device, zeroed by the host)
    uint32_t s_stride;
};

#ifdef __CUDACC__
namespace tc {

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
// bounded spin: a protocol error traps instead of hanging the GPU
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
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
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void fence_before_sync() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void fence_after_sync() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// UMMA shared-memory descriptor, 128-byte swizzle, version 1 (Blackwell): start address >> 4 in
// bits [0,14), leading byte offset >> 4 in [16,30), stride byte offset >> 4 in [32,46), version in
// [46,48), layout type (2 = SWIZZLE_128B) in [61,64)
__device__ __forceinline__ uint64_t umma_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes)
{
    return (uint64_t)((saddr & 0x3FFFFu) >> 4) | ((uint64_t)(lbo_bytes >> 4) << 16) |
           ((uint64_t)(sbo_bytes >> 4) << 32) | (1ull << 46) | (2ull << 61);
}

// D[tmem] (+)= A[smem] * B[smem], kind::f8f6f4, issued by one thread
__device__ __forceinline__ void umma_f8(uint32_t tmem_d, uint64_t desc_a, uint64_t desc_b, uint32_t idesc,
                                        uint32_t accumulate)
{
    asm volatile("{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
                 "tcgen05.mma.cta_group::1.kind::f8f6f4 [%0], %1, %2, %3, p;\n\t}"
                 ::"r"(tmem_d), "l"(desc_a), "l"(desc_b), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void umma_commit(uint32_t bar)
{
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}

// 32 spins of word w (and sign plane s for Blume-Capel) -> 32 fp8 bytes, in the order
//     byte 4 k + b  <->  bit 8 b + 7 - k of the word        (k = 0..7, b = 0..3)
// (tc_spin_of_byte below): shifting the word left by k puts bits 7-k, 15-k, 23-k, 31-k at the top of
// its four bytes, and one PRMT with the sign-replicating selector 0xBA98 spreads each of them over a
// byte (0x00 / 0xFF).  Ising: +1.0 = 0x38 for a set bit, -1.0 = 0xB8 otherwise, i.e. 0xB8 ^ (m & 0x80):
// per 4 bytes one shift (an IMAD on the FMA pipe), one PRMT and one LOP3.  Blume-Capel: nz ? (sg ? -1.0
// : +1.0) : 0.0 = m_nz & (0x38 | (m_sg & 0x80)).  The order of the bytes within a word is the same for
// both operands of the MMA, so a contraction along it is unaffected (y axis) and the epilogue undoes it
// where the bytes are matrix rows / columns (x axis).
__device__ __forceinline__ uint32_t sign_bytes(uint32_t x)
{
    uint32_t m;
    asm("prmt.b32 %0, %1, %1, 0xBA98;" : "=r"(m) : "r"(x));
    return m;
}
__host__ __device__ __forceinline__ uint32_t tc_spin_of_byte(uint32_t y)      // y = 0..31 -> bit of the word
{
    return 8u * (y & 3u) + 7u - (y >> 2);
}

template <int MODEL>
__device__ __forceinline__ void expand_word(uint32_t w, uint32_t s, uint4 &lo, uint4 &hi)
{
    uint32_t o[8];
#pragma unroll
    for (int k = 0; k < 8; ++k) {
        const uint32_t m = sign_bytes(w << k);
        if (MODEL == 0) o[k] = 0xB8B8B8B8u ^ (m & 0x80808080u);
        else o[k] = m & (0x38383838u | (sign_bytes(s << k) & 0x80808080u));
    }
    lo = make_uint4(o[0], o[1], o[2], o[3]);
    hi = make_uint4(o[4], o[5], o[6], o[7]);
}

}  // namespace tc

// AXIS 1 (y): positions are rows, the contraction runs over the columns of a row.
// AXIS 0 (x): positions are columns, the contraction runs over rows i0 .. i0 + n_rows - 1.
template <int MODEL, int AXIS>
__global__ void __launch_bounds__(TC_THREADS, 1) corr_tc_kernel(const CorrTCArgs a)
{
    using namespace tc;
    extern __shared__ uint8_t tc_smem_raw[];
    uint8_t *smem = (uint8_t *)(((uintptr_t)tc_smem_raw + 1023) & ~(uintptr_t)1023);      // swizzle atoms: 1 KiB
    int *hist = (int *)(smem + TC_STAGES * TC_STAGE_BYTES);
    __shared__ __align__(8) unsigned long long bars[2 * TC_STAGES + 1];
    __shared__ uint32_t tmem_base_s;

    const uint32_t warp = threadIdx.x >> 5, lane = threadIdx.x & 31u;
    const uint32_t full0 = smem_u32(&bars[0]), empty0 = smem_u32(&bars[TC_STAGES]), accf = smem_u32(&bars[2 * TC_STAGES]);

    if (threadIdx.x == 0) {
        for (int s = 0; s < TC_STAGES; ++s) {
            mbar_init(full0 + 8 * s, TC_PRODUCERS / 32);      // one arrive per producer warp
            mbar_init(empty0 + 8 * s, 1);                     // tcgen05.commit
        }
        mbar_init(accf, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == TC_PRODUCERS / 32) {                          // the MMA warp owns the tensor memory
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&tmem_base_s)), "n"(512));
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::);
    }
    fence_before_sync();
    __syncthreads();
    fence_after_sync();
    const uint32_t tmem = tmem_base_s;

    const size_t pw = (size_t)a.rows * a.wpr;                 // words per plane
    // contraction extent: y: the L columns of a row; x: the base rows
    const uint32_t n_kc = AXIS == 1 ? a.L / TC_KC : (a.n_rows + TC_KC - 1) / TC_KC;
    // instruction descriptor: fp32 accumulate, e4m3 x e4m3, N >> 3 in [17,23), M >> 4 in [24,29),
    // bits 15 / 16 = MN-major A / B (x axis)
    const uint32_t idesc = (1u << 4) | ((uint32_t)(TC_N >> 3) << 17) | ((uint32_t)(TC_M >> 4) << 24) |
                           (AXIS == 0 ? (1u << 15) | (1u << 16) : 0u);

    uint32_t stage = 0, phase = 0, acc_phase = 0;
    for (uint32_t item = blockIdx.x; item < a.n_items; item += gridDim.x) {
        const uint32_t pass = item / a.n_tiles, tile = item - pass * a.n_tiles;
        // first base position of the tile and first partner position of the pass
        const uint32_t p0 = (AXIS == 1 ? a.i0 : 0u) + tile * TC_M;
        if (warp < TC_PRODUCERS / 32) {
            // ===== producers =====
            // A stage is (128 + 512) x 2 chunks of 64 bytes; thread t owns chunks t, t + 256, ...
            // (TC_PER_THREAD of them) for the whole item: source pointer, shared-memory offset and
            // the contraction step at which its lattice row leaves the base rows are fixed per item.
            constexpr int TC_PER_THREAD = (TC_M + TC_NT * TC_N) * 2 / TC_PRODUCERS;      // 5
            const uint32_t *src[TC_PER_THREAD];
            uint32_t dst[TC_PER_THREAD], xr[TC_PER_THREAD], kc_zero[TC_PER_THREAD];
#pragma unroll
            for (int q = 0; q < TC_PER_THREAD; ++q) {
                const uint32_t it = threadIdx.x + (uint32_t)q * TC_PRODUCERS;
                uint32_t h, srow, blk, row_l, word;          // half, smem row, block, lattice row, word in row
                kc_zero[q] = 0xffffffffu;                    // first contraction step that is all zeros
                if (AXIS == 1) {
                    const uint32_t tr = it >> 1;              // 0..127 base rows, 128..639 partner rows
                    h = it & 1u;
                    blk = tr < TC_M ? 0u : 1u + (tr - TC_M) / TC_N;
                    srow = tr < TC_M ? tr : (tr - TC_M) % TC_N;
                    uint32_t i;
                    if (tr < TC_M) { i = p0 + tr; if (i >= a.i0 + a.n_rows) kc_zero[q] = 0u; }
                    else i = p0 + pass * (TC_NT * TC_N) + (tr - TC_M);
                    row_l = i % a.rows;
                    word = 0u;                                // + 2 words (64 packed positions) per step
                } else {
                    // smem row = contraction index (lattice row), 128-column blocks along MN:
                    // block 0 = base columns, blocks 1..4 = the pass's partner columns; the second
                    // 128-column block of an N tile sits TC_KC rows (16 KiB) further (MN-major LBO)
                    // chunks 0..255: the base block (mb = 0), one 8-byte word pair per (row, half);
                    // chunks 256..1279: the four partner blocks, with the block index varying faster
                    // than the upper bits of the row: the 32 lanes of a load instruction then read the
                    // 4 x 8 contiguous bytes of 8 rows (8 lines) instead of 8 bytes of 32 rows, while the
                    // 8 lanes of a quarter-warp still store to 8 consecutive rows (conflict-free)
                    uint32_t kk, mb;
                    if (it < 2u * TC_KC) { kk = it % TC_KC; h = it / TC_KC; mb = 0u; }
                    else {
                        const uint32_t b = it - 2u * TC_KC;
                        kk = ((b >> 5) & 15u) * 8u + (b & 7u);
                        mb = 1u + ((b >> 3) & 3u);
                        h = b >> 9;
                    }
                    blk = mb == 0 ? 0u : 1u + (mb - 1u) / 2u;
                    srow = kk + ((mb == 0 ? 0u : (mb - 1u) & 1u) * TC_KC);
                    row_l = a.i0 + kk;                        // + TC_KC rows per step; never wraps
                    kc_zero[q] = kk < a.n_rows ? (a.n_rows - kk + TC_KC - 1) / TC_KC : 0u;
                    const uint32_t col0 = mb == 0 ? p0 : (p0 + pass * (TC_NT * TC_N) + (mb - 1u) * TC_M) % a.L;
                    word = col0 / 64u;                        // 128 columns = 64 packed positions = 2 words
                }
                const uint32_t c = (row_l & 1u) ^ h;          // even columns of row i live in colour i & 1
                src[q] = a.buf + (MODEL == 0 ? (size_t)c * pw : (size_t)(2u * c) * pw) + (size_t)row_l * a.wpr + word;
                // canonical 128-byte swizzle: 8-row atoms of 1 KiB, 16-byte chunk index ^ (row & 7)
                dst[q] = (blk == 0 ? 0u : TC_M * TC_KC + (blk - 1u) * (TC_N * TC_KC)) + (srow >> 3) * 1024u + (srow & 7u) * 128u;
                xr[q] = (srow & 7u) | (h << 2 << 8);          // low byte: row & 7, bits 8..: first chunk h * 4
            }
            const size_t step = AXIS == 1 ? 2u : (size_t)TC_KC * a.wpr;      // words per contraction step
            if constexpr (AXIS == 1) {
                // y axis: a thread's consecutive steps read consecutive 8-byte pieces of one lattice row,
                // so it loads 16 bytes = two steps at a time (rows are 16-byte aligned: L % 256 == 0, and
                // n_kc = L / 128 is even).  Every lane of a load reads another row -- 32 lines, 32
                // wavefronts of the L1 data pipe whatever the width -- and that pipe (stores of the
                // expanded bytes + operand reads of the tensor core + these loads) is what binds the
                // kernel (profiles/r2_corr_tc.md): half as many loads is what counts.  Ring of TC_PF2
                // such loads per chunk, reloaded for step kc + 2 TC_PF2 after the second of its steps.
                constexpr int TC_PF2 = 2;
                uint4 wb[TC_PF2][TC_PER_THREAD], sb[TC_PF2][TC_PER_THREAD];
#pragma unroll
                for (int u = 0; u < TC_PF2; ++u)
#pragma unroll
                    for (int q = 0; q < TC_PER_THREAD; ++q) {
                        wb[u][q] = sb[u][q] = make_uint4(0u, 0u, 0u, 0u);
                        if (2u * (uint32_t)u < n_kc && kc_zero[q] != 0u) {
                            wb[u][q] = *reinterpret_cast<const uint4 *>(src[q] + 4 * u);
                            if (MODEL) sb[u][q] = *reinterpret_cast<const uint4 *>(src[q] + 4 * u + pw);
                        }
                    }
                for (uint32_t kc0 = 0; kc0 < n_kc; kc0 += 2u * TC_PF2) {
#pragma unroll
                    for (int uv = 0; uv < 2 * TC_PF2; ++uv) {
                        const int u = uv >> 1, v = uv & 1;
                        const uint32_t kc = kc0 + (uint32_t)uv;
                        if (kc >= n_kc) break;
                        mbar_wait(empty0 + 8 * stage, phase ^ 1u);
                        const uint32_t st = smem_u32(smem) + stage * TC_STAGE_BYTES;
#pragma unroll
                        for (int q = 0; q < TC_PER_THREAD; ++q) {
                            uint4 o[4];
                            if (kc_zero[q] == 0u) {
                                o[0] = o[1] = o[2] = o[3] = make_uint4(0u, 0u, 0u, 0u);
                            } else {
                                expand_word<MODEL>(v ? wb[u][q].z : wb[u][q].x, v ? sb[u][q].z : sb[u][q].x, o[0], o[1]);
                                expand_word<MODEL>(v ? wb[u][q].w : wb[u][q].y, v ? sb[u][q].w : sb[u][q].y, o[2], o[3]);
                            }
                            const uint32_t r7 = xr[q] & 7u, c0 = xr[q] >> 8;
#pragma unroll
                            for (int e = 0; e < 4; ++e)
                                asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(st + dst[q] + (((c0 + (uint32_t)e) ^ r7) << 4)),
                                             "r"(o[e].x), "r"(o[e].y), "r"(o[e].z), "r"(o[e].w) : "memory");
                        }
                        fence_proxy_async();                  // generic-proxy writes -> visible to the tensor core
                        __syncwarp();
                        if (lane == 0) mbar_arrive(full0 + 8 * stage);
                        if (++stage == TC_STAGES) { stage = 0; phase ^= 1u; }
                        if (v == 1) {
                            const uint32_t nk = kc0 + 2u * (uint32_t)u + 2u * TC_PF2;
#pragma unroll
                            for (int q = 0; q < TC_PER_THREAD; ++q) {
                                wb[u][q] = sb[u][q] = make_uint4(0u, 0u, 0u, 0u);
                                if (nk < n_kc && kc_zero[q] != 0u) {
                                    wb[u][q] = *reinterpret_cast<const uint4 *>(src[q] + 2 * (size_t)nk);
                                    if (MODEL) sb[u][q] = *reinterpret_cast<const uint4 *>(src[q] + 2 * (size_t)nk + pw);
                                }
                            }
                        }
                    }
                }
            } else {
            // The packed words of the next TC_PF contraction steps live in registers (a ring indexed by
            // kc % TC_PF, the loop unrolled by TC_PF so that the index is static): the loads of step
            // kc + TC_PF are issued at the end of step kc, after the proxy fence (which would otherwise
            // wait for them).  A producer iteration is a few hundred cycles of work, far less than a
            // global-load latency under load: with a distance of one step (round 2's first version)
            // 40 % of all stall samples sat on the first use of the loaded word.
            constexpr int TC_PF = MODEL == 0 ? 4 : 3;
            uint2 wb[TC_PF][TC_PER_THREAD], sb[TC_PF][TC_PER_THREAD];
#pragma unroll
            for (int u = 0; u < TC_PF; ++u)
#pragma unroll
                for (int q = 0; q < TC_PER_THREAD; ++q) {
                    wb[u][q] = sb[u][q] = make_uint2(0u, 0u);
                    if ((uint32_t)u < n_kc && (uint32_t)u < kc_zero[q]) {
                        wb[u][q] = *reinterpret_cast<const uint2 *>(src[q] + (size_t)u * step);
                        if (MODEL) sb[u][q] = *reinterpret_cast<const uint2 *>(src[q] + (size_t)u * step + pw);
                    }
                }
            for (uint32_t kc0 = 0; kc0 < n_kc; kc0 += TC_PF) {
#pragma unroll
                for (int u = 0; u < TC_PF; ++u) {
                    const uint32_t kc = kc0 + (uint32_t)u;
                    if (kc >= n_kc) break;
                    mbar_wait(empty0 + 8 * stage, phase ^ 1u);
                    const uint32_t st = smem_u32(smem) + stage * TC_STAGE_BYTES;
#pragma unroll
                    for (int q = 0; q < TC_PER_THREAD; ++q) {
                        uint4 o[4];
                        if (kc >= kc_zero[q]) {
                            o[0] = o[1] = o[2] = o[3] = make_uint4(0u, 0u, 0u, 0u);
                        } else {
                            expand_word<MODEL>(wb[u][q].x, sb[u][q].x, o[0], o[1]);
                            expand_word<MODEL>(wb[u][q].y, sb[u][q].y, o[2], o[3]);
                        }
                        const uint32_t r7 = xr[q] & 7u, c0 = xr[q] >> 8;
#pragma unroll
                        for (int e = 0; e < 4; ++e)
                            asm volatile("st.shared.v4.b32 [%0], {%1, %2, %3, %4};" ::"r"(st + dst[q] + (((c0 + (uint32_t)e) ^ r7) << 4)),
                                         "r"(o[e].x), "r"(o[e].y), "r"(o[e].z), "r"(o[e].w) : "memory");
                    }
                    fence_proxy_async();                      // generic-proxy writes -> visible to the tensor core
                    __syncwarp();
                    if (lane == 0) mbar_arrive(full0 + 8 * stage);
                    if (++stage == TC_STAGES) { stage = 0; phase ^= 1u; }
                    const uint32_t nk = kc + (uint32_t)TC_PF;
#pragma unroll
                    for (int q = 0; q < TC_PER_THREAD; ++q) {
                        wb[u][q] = sb[u][q] = make_uint2(0u, 0u);
                        if (nk < n_kc && nk < kc_zero[q]) {
                            wb[u][q] = *reinterpret_cast<const uint2 *>(src[q] + (size_t)nk * step);
                            if (MODEL) sb[u][q] = *reinterpret_cast<const uint2 *>(src[q] + (size_t)nk * step + pw);
                        }
                    }
                }
            }
            }
            // ===== epilogue (warps 0-3: TMEM lane quarter = warp) =====
            if (warp < 4) {
                for (uint32_t t = threadIdx.x; t < (uint32_t)TC_HIST; t += 128u) hist[t] = 0;
                asm volatile("bar.sync 1, 128;" ::: "memory");
                mbar_wait(accf, acc_phase);
                fence_after_sync();
                const uint32_t m = warp * 32u + lane;         // base position index in the tile
                // position of byte index x inside a 128-block: [64 even | 64 odd] for the x axis
                // (and inside each 32-byte group the byte order of expand_word)
                const int pm = AXIS == 1 ? (int)m : (int)(2u * ((m & 32u) + tc_spin_of_byte(m & 31u)) + (m >> 6));
#pragma unroll 1
                for (uint32_t cb = 0; cb < (uint32_t)(TC_NT * TC_N); cb += 16u) {
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
                        const uint32_t n = cb + (uint32_t)e;
                        int pn;
                        if (AXIS == 1) pn = (int)n;
                        else {
                            const uint32_t nb = n & 127u;
                            pn = (int)((n & ~127u) + 2u * ((nb & 32u) + tc_spin_of_byte(nb & 31u)) + (nb >> 6));
                        }
                        const int d = pn - pm;                 // r - 512 pass, in (-128, 512)
                        const long long r = (long long)d + (long long)pass * (TC_NT * TC_N);
                        const int val = __float2int_rn(__uint_as_float(v[e]));
                        if (r >= 1 && r <= (long long)a.r_max && val) atomicAdd(&hist[d + (TC_M - 1)], val);
                    }
                }
                fence_before_sync();
                asm volatile("bar.sync 1, 128;" ::: "memory");
                for (uint32_t t = threadIdx.x; t < (uint32_t)TC_HIST; t += 128u) {
                    const long long r = (long long)t - (TC_M - 1) + (long long)pass * (TC_NT * TC_N);
                    if (hist[t] && r >= 1 && r <= (long long)a.r_max)
                        atomicAdd((unsigned long long *)(a.S + (r - 1) * a.s_stride), (unsigned long long)(long long)hist[t]);
                }
                asm volatile("bar.sync 1, 128;" ::: "memory");
            }
            acc_phase ^= 1u;
        } else {
            // ===== MMA issuer (one elected thread of warp 8) =====
            for (uint32_t kc = 0; kc < n_kc; ++kc) {
                mbar_wait(full0 + 8 * stage, phase);
                fence_after_sync();
                if (lane == 0) {
                    const uint32_t sa = smem_u32(smem + (size_t)stage * TC_STAGE_BYTES);
                    const uint32_t sb = sa + TC_M * TC_KC;
#pragma unroll
                    for (uint32_t k = 0; k < TC_KC / 32; ++k) {
#pragma unroll
                        for (uint32_t nt = 0; nt < (uint32_t)TC_NT; ++nt) {
                            uint64_t da, db;
                            if (AXIS == 1) {
                                // K-major: rows of 128 bytes along K, 8-row atoms 1 KiB apart; a K step of
                                // 32 bytes moves the start address inside the swizzled row
                                da = umma_desc(sa + k * 32u, 16u, 1024u);
                                db = umma_desc(sb + nt * (TC_N * TC_KC) + k * 32u, 16u, 1024u);
                            } else {
                                // MN-major: rows of 128 bytes along M / N, one row per contraction index;
                                // 8-row atoms along K 1 KiB apart (SBO), the second 128-column block of an
                                // N tile TC_KC * 128 bytes further (LBO); a K step of 32 = 4 atoms
                                da = umma_desc(sa + k * 4096u, TC_KC * 128u, 1024u);
                                db = umma_desc(sb + nt * (TC_N * TC_KC) + k * 4096u, TC_KC * 128u, 1024u);
                            }
                            umma_f8(tmem + nt * TC_N, da, db, idesc, (kc | k) ? 1u : 0u);
                        }
                    }
                    umma_commit(empty0 + 8 * stage);          // stage reusable once these MMAs are done
                    if (kc + 1 == n_kc) umma_commit(accf);    // accumulators complete
                }
                __syncwarp();
                if (++stage == TC_STAGES) { stage = 0; phase ^= 1u; }
            }
        }
    }
    fence_before_sync();
    __syncthreads();
    if (warp == TC_PRODUCERS / 32) {
        fence_after_sync();
        asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "n"(512));
    }
}
#endif

}  // namespace lat
