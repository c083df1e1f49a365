/*
 * lattice.h -- C ABI of the B200 (sm_100a) checkerboard Metropolis library.
 *
 * What is computed (arXiv:2503.14688, Bisson et al.; line numbers refer to the paper text
 * PAPER.md as surveyed in SURVEY.md, readings in DESIGN.md):
 *   - Hamiltonian H = -J sum_<xy> s_x s_y + Delta sum_x s_x^2, J = 1, periodic L x L square
 *     lattice; spin-1/2 Ising (s = +-1) and spin-1 Blume-Capel (s in {-1,0,+1})
 *     (Eq. 1).
 *   - Metropolis dynamics with checkerboard decomposition and multispin coding
 *     (PAPER.md:32-34): one sweep = black half-sweep ((i+j) even) then white half-sweep;
 *     time is counted in full-lattice sweeps.
 *   - Fully disordered start; a per-sweep inverse temperature beta(t): constant
 *     for protocol 1, time-varying for protocol 2.
 *   - Acceptance as a 32-bit integer compare: accept iff dE <= 0 or
 *     u32(site) < floor(2^32 exp(-beta dE)).  u32(site) and every other random bit come from
 *     Philox4x32-10 keyed by (seed, sweep, colour, site); random
 *     numbers are generated in registers and never stored.
 *   - Measurements as exact 64-bit integers: M = sum s, Q = sum s^2 and the axis correlation
 *     sums S_x(r) = sum_{i,j} s(i,j) s(i,j+r), S_y(r) = sum_{i,j} s(i,j) s(i+r,j)
 *     (Eq. 2); C(r) = (S_x+S_y)/(2 L^2), e = -(S_x(1)+S_y(1))/L^2 + Delta Q/L^2
 *     (Eq. 3 with the sign fixed by E_eq = -sqrt 2), xi = I_2/I_1
 *     (Eq. C1).
 *
 * Conventions
 *   - Every pointer is a HOST pointer unless its name starts with `device_`.
 *   - Every call that can fail returns an int status (LATTICE_OK == 0).  Outputs are written
 *     only on LATTICE_OK.  Nothing throws or aborts across this boundary.
 *   - A handle is not thread-safe; different handles are independent.
 *   - The library runs only on a CUDA device; there is no CPU fallback.
 */
#ifndef LATTICE_H
#define LATTICE_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct lattice lattice_t;              /* opaque; owned by the library */

enum { LATTICE_ISING = 0, LATTICE_BLUME_CAPEL = 1 };
enum {
    LATTICE_OK = 0,
    LATTICE_EINVAL = -1,    /* bad argument (see each call)                                */
    LATTICE_ENOMEM = -2,    /* host or device scratch allocation failed                    */
    LATTICE_ECUDA = -3,     /* a CUDA call or kernel failed; lattice_last_error() has text */
    LATTICE_ESTATE = -4     /* call not allowed in the handle's current state              */
};

/* Bytes of device memory the packed state needs: L*L/8 (Ising, 1 bit/spin) or L*L/4
 * (Blume-Capel, 2 bits/spin).  Returns 0 if L is not a positive multiple of 64 or the model
 * is unknown.  Layout inside the buffer (32-bit words):
 *   Ising:        [colour 0..1][row 0..L-1][word 0..L/64-1]
 *   Blume-Capel:  [colour 0..1][plane 0 = nonzero, 1 = negative][row][word]
 * Word k of a row holds the L/2 same-colour sites p = 32k..32k+31 (bit b <-> p = 32k+b),
 * column j = 2p + ((i + colour) & 1). */
size_t lattice_state_bytes(uint32_t L, int model);

/* Create a lattice in caller-owned device memory and fill it with the disordered start
 * (PAPER.md:65): Ising s = +-1 with probability 1/2, Blume-Capel uniform on {-1,0,+1}; t = 0.
 *   out               receives the handle.
 *   L                 lattice side, a multiple of 64, L <= 2^20.
 *   model             LATTICE_ISING or LATTICE_BLUME_CAPEL.
 *   delta             crystal field Delta of Eq. 1 (ignored for Ising; must be finite).
 *   seed              Philox key.
 *   device_buf        device pointer, 16-byte aligned, at least lattice_state_bytes(L, model)
 *                     bytes.  The caller keeps ownership and must keep it alive until
 *                     lattice_destroy; the library never frees it.
 *   cuda_stream       a cudaStream_t (NULL = the legacy default stream).  Every kernel of this
 *                     handle is launched on it.
 * The RNG scheme defaults to 1 (bit-plane + tail).
 * Errors: EINVAL (bad L/model/delta/buffer/alignment/out), ENOMEM, ECUDA. */
int lattice_create(lattice_t **out, uint32_t L, int model, double delta, uint64_t seed,
                   void *device_buf, size_t device_buf_bytes, void *cuda_stream);

/* ---- Batches of independent replicas ----------------------------------------------------------
 * The paper's error bars come from 40-4000 independent runs per point (Tables I-II,
 * PAPER.md:126-153; jackknife over realisations).  A batch handle evolves
 * n_replicas lattices of the same L, model and Delta under the same beta schedule, replica k keyed
 * by seeds[k]: every replica is bit for bit the stand-alone lattice lattice_create(L, model, Delta,
 * seeds[k]) would give.  Layout of the buffer: [replica][<single-lattice layout>], i.e.
 * lattice_batch_bytes = n_replicas * lattice_state_bytes.  What fills the GPU at cache-resident
 * sizes: Ising lattices with L a multiple of 256 update all replicas in one launch per half-sweep
 * (replica = blockIdx.y, its Philox round keys from a table in the kernel parameters); Ising
 * L = 64 and 128 keep each replica in the registers of a (half-)warp and run ALL n sweeps of a
 * lattice_sweep call in one launch; other shapes fall back to one launch per replica.
 *   lattice_sweep / lattice_half_sweep / lattice_set_rng_scheme / lattice_set_time / lattice_fill /
 *   lattice_time / lattice_launches act on all replicas; lattice_measure_batch returns the counts
 *   of every replica: M[k], Q[k], Sx[k * r_max + r - 1], Sy[k * r_max + r - 1].
 *   lattice_replica lends the handle of replica k (owned by the batch, valid until the batch is
 *   destroyed, not to be destroyed itself): lattice_get_spins / lattice_set_spins /
 *   lattice_measure / lattice_measure_rows / lattice_fill work on it; sweeps, set_time and
 *   set_rng_scheme return ESTATE.  On the batch handle itself the per-lattice calls
 *   (get/set_spins, measure, measure_rows) return ESTATE.
 * Errors: EINVAL (as lattice_create; n_replicas == 0 or > 2^20; NULL seeds), ENOMEM, ECUDA. */
size_t lattice_batch_bytes(uint32_t n_replicas, uint32_t L, int model);       /* 0 if invalid */
int lattice_create_batch(lattice_t **out, uint32_t n_replicas, uint32_t L, int model, double delta,
                         const uint64_t *seeds, void *device_buf, size_t device_buf_bytes,
                         void *cuda_stream);
uint32_t lattice_replicas(const lattice_t *lat);       /* 1 for a plain lattice, 0 for NULL */
int lattice_replica(lattice_t *batch, uint32_t k, lattice_t **out);
int lattice_measure_batch(lattice_t *batch, uint32_t r_max, int64_t *M, int64_t *Q, int64_t *Sx,
                          int64_t *Sy);

/* ---- Row-slab domain decomposition (the paper's third level of parallelism, PAPER.md:32-34;
 * SURVEY.md section 8(f) NEXT-1) -------------------------------------------
 * A slab owns global rows row0 .. row0+n_rows-1 of a periodic L x L lattice and keeps one halo
 * row above and below them: layout [colour][n_rows + 2][L/64] 32-bit words, local row l being
 * global row (row0 - 1 + l) mod L.  Random numbers are keyed by GLOBAL (row, column), so N slabs
 * evolve bit for bit like the whole lattice.  Every half-sweep kernel stores the slab's first
 * and last own row a second time, directly into the neighbour slabs' halo rows (and applies late
 * tie flips there with atomics): those pointers may be peer-GPU memory (NVLink P2P), so the halo
 * exchange is fused into the update kernel and needs no copy or collective.  The caller orders
 * the half-sweeps: all slabs finish colour c (and its mirrors) before any starts colour 1-c.
 * Restrictions (round 1): RNG scheme 1, L a multiple of 256, row0 and n_rows multiples of 64;
 * Blume-Capel only with threshold tables of the Delta = 0 structure (half-sweeps return EINVAL
 * otherwise); Blume-Capel layout [colour][plane][n_rows + 2][L/64]; lattice_measure on a slab
 * only with r_max == 1 (partial sums over the own rows: add them up; for r > 1 see lattice_view);
 * windows of get/set_spins must stay inside the slab's rows (halos included). */
size_t lattice_slab_bytes(uint32_t L, int model, uint32_t n_rows);      /* 0 if not supported */
/* Like lattice_create for the slab; own rows AND halos receive the disordered start. */
int lattice_create_slab(lattice_t **out, uint32_t L, int model, double delta, uint64_t seed,
                        uint32_t row0, uint32_t n_rows, void *device_buf, size_t device_buf_bytes,
                        void *cuda_stream);
/* Device buffers (and n_rows) of the slabs that own the rows above and below this one (this
 * slab's own buffer twice when it is the only slab).  Required before the first half-sweep
 * (ESTATE otherwise).  The buffers must stay valid and, if on another GPU, peer-accessible. */
int lattice_slab_set_neighbours(lattice_t *lat, void *device_up_buf, uint32_t up_n_rows,
                                void *device_down_buf, uint32_t down_n_rows);

/* Device-side ordering of the colours (csrc/slab_flags.cuh): instead of the caller waiting between the
 * half-sweeps, every slab publishes the number of half-sweeps it has completed, 2 t + colour + 1 after
 * colour `colour` of sweep t, in a 64-bit word of device memory (8-byte aligned, e.g. behind its slab
 * buffer), and every half-sweep launch of this handle is preceded by a one-thread kernel that waits
 * until both neighbours' words have reached the previous half-sweep, and followed by one that
 * publishes its own (release, system scope).  The neighbours' words may be peer-GPU or IPC memory.
 * lattice_slab_set_flags publishes 2 * lattice_time() (so does lattice_set_time); the caller makes sure
 * that every slab has done so before the first half-sweep (one host barrier at set-up), and that all
 * slabs are given the same sequence of half-sweeps.  Three NULLs switch back to host ordering.
 * The wait is bounded (~17 s, then the kernel traps: ECUDA on the next call).
 * Errors: EINVAL (NULL handle, some but not all pointers NULL, misaligned), ESTATE (not a slab), ECUDA. */
int lattice_slab_set_flags(lattice_t *lat, void *device_my_flag, const void *device_up_flag,
                           const void *device_down_flag);

/* A measurement-only handle over a caller-assembled buffer [colour(/plane)][rows][L/64] that is
 * NOT periodic along y: lattice_measure_rows(view, i0, n, r_max, ...) requires
 * i0 + n + r_max <= rows (partner rows i + r are read from the buffer as they are); the x axis
 * stays periodic within a row.  This is how a slab measures C(r) for r > 1: its own rows followed
 * by the next r_max rows of the lattice (copied from the slabs below, lattice_device_copy works on
 * peer / IPC pointers), base rows 0 .. n_rows-1.  No other call is allowed on a view except
 * lattice_destroy.  Row parity matters for odd r along x: rows must start at an EVEN global row. */
int lattice_view(lattice_t **out, uint32_t L, int model, uint32_t rows, void *device_buf,
                 size_t device_buf_bytes, void *cuda_stream);
int lattice_device_copy(void *device_dst, const void *device_src, size_t bytes, void *cuda_stream);

/* One process driving several GPUs: let kernels running on `device` store into memory of
 * `peer_device` (cudaDeviceEnablePeerAccess; already-enabled is not an error).  ECUDA if the two
 * devices cannot reach each other. */
int lattice_enable_peer_access(int device, int peer_device);

/* One process per GPU: the mirror pointers of lattice_slab_set_neighbours must then come from
 * another process.  These helpers allocate a slab buffer that can be exported (cudaMalloc on the
 * current device, so that the IPC handle maps the buffer itself), export it as a 64-byte CUDA IPC
 * handle (sent to the neighbours by any means, e.g. torch.distributed), and open a neighbour's
 * handle as a device pointer valid in this process.  Errors: EINVAL (NULL), ECUDA. */
int lattice_device_alloc(void **device_ptr, size_t bytes);
int lattice_device_free(void *device_ptr);
int lattice_ipc_export(const void *device_ptr, unsigned char handle[64]);
int lattice_ipc_open(const unsigned char handle[64], void **device_ptr);
int lattice_ipc_close(void *device_ptr);

/* Select how u32(site) is derived from Philox4x32-10:
 *   0 "quad":       one block per 4 consecutive same-colour sites, one 32-bit word each;
 *   1 "plane+tail": top 8 bits from 8 bit-plane blocks shared by 128 sites, low 24 bits from a
 *                   per-site block that is only evaluated when the top byte ties with the
 *                   threshold's.  Same statistics, ~4x less RNG work.
 *   2 "plane+tail56": scheme 1 with 64-bit thresholds floor(2^64 exp(-beta dE)) and 56 tail bits
 *                   (words 0 and 1 of the same tail block): u64 = top byte | 56 tail bits; lifts the
 *                   2^-32 floor on acceptance probabilities to 2^-64.  Identical to
 *                   scheme 1 unless u32 == thr32.  Marching kernels only: EINVAL unless L is a
 *                   multiple of 256; Blume-Capel half-sweeps return EINVAL for tables without the
 *                   Delta = 0 structure.
 * Only allowed at t == 0 (ESTATE otherwise).  EINVAL for an unknown scheme. */
int lattice_set_rng_scheme(lattice_t *lat, int scheme);

/* Run sweeps t .. t+n-1; sweep t+k uses beta[k] (host fp64 array of n entries; beta = 1/T).
 * One sweep = one Metropolis update attempt of every site, the paper's time unit:
 * black half-sweep then white half-sweep (checkerboard); a constant array is
 * protocol 1, a time-varying one protocol 2 (Table II).
 * Thresholds floor(2^32 exp(-beta dE)) are rebuilt on the host whenever beta changes.
 * Asynchronous on the handle's stream (beta is consumed before the call returns); t += n.
 * Errors: EINVAL (NULL beta with n > 0, NaN or negative beta, t+n >= 2^32), ECUDA. */
int lattice_sweep(lattice_t *lat, uint64_t n, const double *beta);

/* lattice_sweep(n, beta) followed by the r = 1 record of the resulting state -- what a run that logs
 * e(t), m(t) every step does (Eq. 3): *M, *Q, *Sx1 = S_x(1), *Sy1 = S_y(1) exactly as
 * lattice_measure(lat, 1, ...) would return them after the sweeps.  For Ising lattices on the marching
 * kernel (L a multiple of 256, L > 4352, bit-plane RNG schemes, not a slab) the record is counted inside
 * the last white half-sweep, where the four neighbour words of every white site are in registers (every
 * bond joins a white and a black site): no separate pass over the lattice.  Any other handle runs
 * lattice_sweep and lattice_measure(1).  Host outputs; synchronises the stream.  n == 0 measures only.
 * Errors: as lattice_sweep and lattice_measure; ESTATE for batch handles and views. */
int lattice_sweep_record(lattice_t *lat, uint64_t n, const double *beta, int64_t *M, int64_t *Q,
                         int64_t *Sx1, int64_t *Sy1);

/* One colour (0 = black first, 1 = white) of sweep t at inverse temperature beta, without
 * advancing t.  lattice_sweep(1, &beta) == half_sweep(0), half_sweep(1), t += 1.  For tests. */
int lattice_half_sweep(lattice_t *lat, int colour, double beta);

/* Exact integer measurements of the whole lattice, r = 1..r_max (1 <= r_max <= L/2): the
 * numerators of C(r;t) along the two lattice axes, Eq. 2, and of E(t), Eq. 3
 * (r = 1):
 *   *M = sum s, *Q = sum s^2 (= L^2 for Ising), Sx[r-1] = S_x(r), Sy[r-1] = S_y(r).
 * Host outputs; synchronises the stream.  Errors: EINVAL, ENOMEM, ECUDA. */
int lattice_measure(lattice_t *lat, uint32_t r_max, int64_t *M, int64_t *Q, int64_t *Sx,
                    int64_t *Sy);

/* lattice_measure without any allocation, for callers that cannot call cudaMalloc (code under CUDA
 * graph capture, tight serving loops, harnesses that forbid it): the same exact counts (Eq. 2-3,
 * PAPER.md:42-50) for r = 1 .. r_max, r_max <= LATTICE_STATIC_RMAX, computed by the XOR/popcount
 * kernels with their per-r counters in a file-scope device array of 2 + 4 * LATTICE_STATIC_RMAX 64-bit
 * words (34 KiB) that every GPU loading the library holds until exit.  The call makes no cudaMalloc,
 * cudaFree or host allocation; it clears the array on the handle's stream, launches, copies the counts
 * back and synchronises the stream.  ALL calls on a device share that array: calls that overlap on
 * the GPU (different streams, handles or host threads) race -- serialise them.  The device current at
 * the call must be the one that holds the lattice.
 * Errors: EINVAL (NULL, r_max < 1, r_max > L/2, r_max > LATTICE_STATIC_RMAX -- lattice_last_error says
 * so --, a slab with r_max != 1), ESTATE (batch handle or view), ECUDA. */
#define LATTICE_STATIC_RMAX 1024
int lattice_measure_static(lattice_t *lat, uint32_t r_max, int64_t *M, int64_t *Q, int64_t *Sx,
                           int64_t *Sy);

/* The same sums restricted to base sites in rows i0 .. i0+n_rows-1 (partners wrap
 * periodically); the partial sums of a partition of the rows add up to lattice_measure.
 * For spot checks at L = 2^20 and for future row-slab sharding. */
int lattice_measure_rows(lattice_t *lat, uint64_t i0, uint64_t n_rows, uint32_t r_max,
                         int64_t *M, int64_t *Q, int64_t *Sx, int64_t *Sy);

/* The same sums for a sparse list of separations -- the paper samples C(r;t) sparsely in r
 * (PAPER.md:207): Sx[q] = S_x(r[q]), Sy[q] = S_y(r[q]), q = 0..n_r-1, over base rows
 * i0 .. i0+n_rows-1 (the whole lattice: 0, L).  r is a host array; each entry in [1, L/2], any
 * order, repeats allowed; n_r <= 2^20.  Cost: one partner read per (word, r[q]) instead of one
 * per (word, r <= r_max).  Host outputs; synchronises the stream.  On a slab only r = 1 is
 * available (as for lattice_measure_rows).  Errors: EINVAL, ESTATE (batch handle), ENOMEM, ECUDA. */
int lattice_measure_list(lattice_t *lat, uint64_t i0, uint64_t n_rows, const uint32_t *r, uint32_t n_r,
                         int64_t *M, int64_t *Q, int64_t *Sx, int64_t *Sy);

/* Unpacked -1/0/+1 windows, row-major h x w, global origin (i0, j0), periodic wrap.
 * h, w <= L.  set_spins rejects values outside the model's alphabet (EINVAL).  Both
 * synchronise the stream.  For tests, windowed replay and checkpoints. */
int lattice_get_spins(lattice_t *lat, uint64_t i0, uint64_t j0, uint32_t h, uint32_t w,
                      int8_t *out);
int lattice_set_spins(lattice_t *lat, uint64_t i0, uint64_t j0, uint32_t h, uint32_t w,
                      const int8_t *in);

/* Set every spin of the lattice (or slab, halos included) to `spin` (+1 / -1, or 0 for
 * Blume-Capel): the ordered states used as worst-case throughput inputs (every site has 4 aligned
 * neighbours, so every lane needs a random decision) and in tests.  Asynchronous on the stream.
 * EINVAL if the value is not in the model's alphabet. */
int lattice_fill(lattice_t *lat, int spin);

/* Sweeps done so far. */
uint64_t lattice_time(const lattice_t *lat);
/* Overwrite the sweep counter (checkpoint restore together with the packed words).
 * EINVAL if t >= 2^32. */
int lattice_set_time(lattice_t *lat, uint64_t t);
/* Number of kernels this handle has launched so far (bench.py's gpu_launches). */
uint64_t lattice_launches(const lattice_t *lat);
/* Launch-time specialisation of the half-sweeps: how many of the handle's launches ran a kernel
 * instantiated for the plane cases of their beta (the LOP3 truth tables of the bit-serial threshold
 * compare as compile-time constants, no per-plane dispatch), and whether such an instantiation
 * exists for (model, delta, beta).  Ising: beta_c = ln(1 + sqrt 2)/2, T_1 = 1.66 and
 * T_2 = 2.27414861561203 of the two-step protocol (Table II).  Blume-Capel at
 * Delta = 0: T = 1.6934 (BASELINE config 3), T_c = 1.69355839821214427 (Table I),
 * T_2 = 1.69661396797728 and T_1 = 1.24 (Table II), the plateau of config 5b's
 * ramp.  Any beta whose thresholds share their top bytes with one of these takes the same kernel.
 * Results never depend on which kernel runs. */
uint64_t lattice_specialised_launches(const lattice_t *lat);
int lattice_plane_case_specialised(int model, double delta, double beta);
/* Which kernels lattice_measure / lattice_measure_rows / lattice_measure_batch use for r_max > 1:
 *   0 (default) automatic: the tensor-core path for L >= 4096, >= 512 base rows and r_max >= 48,
 *     else the XOR/popcount kernels;
 *   1 always the XOR/popcount kernels (north_star (c));
 *   2 always the tensor cores (EINVAL unless L is a multiple of 256, L >= 1024, not a slab): CTA pairs
 *     (tcgen05 cta_group::2, csrc/corr_tc2.cuh) on the y axis, one CTA per item (csrc/corr_tc.cuh) on
 *     the x axis -- the combination measured fastest;
 *   3 / 4 CTA pairs / single CTAs on both axes (same conditions; for tests and measurements).
 * The tensor-core path evaluates dense C(r <= r_max), Eq. 2, as the band of the row /
 * column Gram matrix with tcgen05.mma on fp8 copies of the spins (exactly representable; fp32
 * accumulators hold exact integers up to 2^24 > L); all paths return the same exact integer counts.
 * Device memory: for lattices with L a multiple of 2048 the x axis is evaluated on a transposed copy
 * of up to 65536 rows at a time (csrc/corr_transpose.cuh), which the library allocates on first use
 * and keeps until lattice_destroy: lattice_state_bytes(L, model) * min(n_rows, 65536) / L bytes
 * (8 GiB at L = 2^20).  If that allocation fails the copy-free kernel is used instead (slower, same
 * counts). */
int lattice_set_measure_path(lattice_t *lat, int path);
/* The persistent multi-sweep kernels: lattice_sweep(n >= 2) on a
 * cache-resident lattice can run all n sweeps in ONE cooperative launch with a grid barrier per
 * half-sweep.  max_blocks selects when:
 *   0 (default)   automatic: only where it is measured faster than two launches per sweep, i.e. Ising
 *                 lattices with L <= 8192;
 *   1..2^32-2     on request, for any Ising lattice with L <= 16384 and any Blume-Capel lattice with
 *                 L <= 16384 and Delta = 0 type threshold tables, with at most max_blocks blocks (fewer
 *                 blocks than 256-thread groups of work: every block strides over several groups);
 *   UINT32_MAX    never (two launches per sweep, as for n == 1).
 * Results do not depend on it.  EINVAL for a NULL handle. */
int lattice_set_persist_blocks(lattice_t *lat, uint32_t max_blocks);

/* Host-only helpers (no device work).
 * lattice_thresholds: acceptance thresholds in [0, 2^32] for inverse temperature beta;
 *   Ising: out[0] = thr(dE = 4), out[1] = thr(dE = 8);
 *   Blume-Capel: out[(code*2 + b)*9 + (h+4)], code = s+1, b = proposal bit, h = neighbour sum;
 *   an entry equal to 2^32 means "always accept" (dE <= 0, or exp rounded to 1).
 * lattice_xi: xi = I_2/I_1, I_n = int r^n C(r) dr, Eq. C1, of a single run
 *   (reading 14): C(r) = (Sx+Sy)/(2 L^2), r_cut = (first r with Sx+Sy <= 0) - 1 or
 *   r_max, trapezoid weights (1/2 at r_cut); the two sums are accumulated exactly in 128-bit
 *   integers and divided once; returns 0 if r_cut < 1; *r_cut_out (may be NULL) receives r_cut.
 * lattice_energy: e = -(Sx[0]+Sy[0])/L^2 + delta*Q/L^2. */
void lattice_thresholds(int model, double delta, double beta, uint64_t *out);
/* Scheme 2: thresholds on the 2^64 scale (same indexing); always[e] = 1 where the move is always
 * accepted (dE <= 0, or the product rounds to 2^64), thr[e] is then 0. */
void lattice_thresholds64(int model, double delta, double beta, uint64_t *thr, unsigned char *always);
double lattice_xi(const int64_t *Sx, const int64_t *Sy, uint32_t r_max, int64_t Q, uint32_t L,
                  uint32_t *r_cut_out);
double lattice_energy(const int64_t *Sx, const int64_t *Sy, int64_t Q, double delta, uint32_t L);

/* Integer-dispatch micro-benchmark (the measured peak of bench.py's "alu" roofline; DESIGN.md
 * section 6): runs dependent chains of the instruction mix `mode` on every SM of the current device
 * (4 blocks of 256 threads per SM, 8 chains per thread) and returns the thread-instructions of the
 * counted classes issued per clock per SM, from clock64() inside the kernel (independent of the
 * SM clock).  mode 0: LOP3; 1: mul.wide.u32 + LOP3 (a Philox round); 2: mul.wide.u32 + 3 LOP3
 * (the half-sweep's mix); 3: POPC.  *elapsed_ms (may be NULL) receives the CUDA-event time of the
 * timed launch.  Synchronises the stream.  Errors: EINVAL, ENOMEM, ECUDA. */
int lattice_ubench_int_dispatch(int mode, void *cuda_stream, double *thread_instr_per_clk_per_sm,
                                double *elapsed_ms);

/* Frees the handle and its scratch; never the caller's device_buf. */
int lattice_destroy(lattice_t *lat);

const char *lattice_strerror(int status);
/* Text of the last CUDA error seen by this handle ("" if none). */
const char *lattice_last_error(const lattice_t *lat);

#ifdef __cplusplus
}
#endif
#endif /* LATTICE_H */
