/*
 * rosen.h -- C ABI of librosen.so: Rosenbluth self-avoiding-walk chain generation on one B200.
 *
 * The data-parallel hot path of arXiv 1704.04381 (Guo & Baulin, "GPU Implementation of the
 * Rosenbluth Generation Method for Static Monte Carlo Simulations", CPC 2017), re-designed for
 * sm_100a. Citations are /root/reference/PAPER.md line numbers; the numeric specification both
 * this library and the CPU oracle restate independently is DESIGN.md section 3.
 *
 * Conventions
 *   - Every entry point returns ROSEN_OK (0) or a negative ROSEN_E* code; nothing throws.
 *   - All pointers inside rosen_outputs point to CALLER-OWNED memory; `memory` says whether they
 *     are device pointers (ROSEN_MEM_DEVICE, the usual case: PyTorch tensors) or host pointers
 *     (ROSEN_MEM_HOST: the library stages through its own device buffers and copies back inside
 *     the call). NULL members are not written. The library allocates nothing the caller must free.
 *   - `summary` is always a HOST pointer (may be NULL). When it is non-NULL the call returns after
 *     the work has completed on `cuda_stream` (the stream is synchronised); when it is NULL and
 *     all outputs are device memory the call only enqueues work on `cuda_stream`.
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).
 *   - Chain ids: chain i of a call has id chain_offset + i. Every per-chain result is a pure
 *     function of (seed, id, parameters): any sub-range reproduces bit-identically, which is how
 *     multi-GPU sharding, resume and sampled parity checks work.
 *   - Calls on one device share that device's scratch (block partials; the long-chain workspace). The library keeps them
 *     apart itself: host threads are serialised per device for the duration of a call, and a call enqueued on another
 *     stream than the previous call of that device first waits (cudaStreamWaitEvent) for that call's work; this holds for
 *     the _async calls too, which are thereby ordered across streams on the device. Calls on different devices are
 *     independent.
 *   - There is no CPU fallback: without a CUDA device every generate call fails with ROSEN_ECUDA.
 */
#ifndef ROSEN_H
#define ROSEN_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define ROSEN_API __attribute__((visibility("default")))
#else
#define ROSEN_API
#endif

#define ROSEN_OK        0
#define ROSEN_EINVAL   (-1)  /* N < 2, n_chains == 0, k_trials outside 1..255, bond_len <= 0, sigma < 0, NaN/inf */
#define ROSEN_ERANGE   (-2)  /* N beyond the supported chain length (lattice 16383, real space 16383)            */
#define ROSEN_ECUDA    (-3)  /* a CUDA runtime call failed (no device, launch error, ...); see rosen_last_error */
#define ROSEN_ENOMEM   (-4)  /* staging / workspace allocation failed                                           */

#define ROSEN_MEM_DEVICE 0
#define ROSEN_MEM_HOST   1

#define ROSEN_LATTICE_SCAN_MAX_N 512  /* longest chain of the shared-memory scan kernel (lattice.cu)                   */
#define ROSEN_LATTICE_HASH_MIN_N 193  /* from here on the hash-map kernel is faster and is used (measured crossover)   */
#define ROSEN_LATTICE_MAX_N  16383   /* beyond: per-chain hash set in HBM (lattice_hash.cu), the range of the paper's
                                        "global-memory version", Table 1 PAPER.md:282-288 (N = 100 ... 10000)        */
#define ROSEN_REALSPACE_SCAN_MAX_N 2048  /* longest chain of the shared-memory scan kernel (realspace.cu) = the paper's
                                           longest shared-memory chain, Table 2                          */
#define ROSEN_REALSPACE_CELL_MIN_N 400   /* from here on the cell-list kernel is faster and is used (measured crossover) */
#define ROSEN_REALSPACE_MAX_N 16383     /* beyond: chain + cell list in HBM, one warp per chain (realspace_long.cu),
                                           the range of Table 2's "global-memory version" rows, PAPER.md:315-320      */

/*
 * Ensemble summary, Eq. 2 and Eq. 6 (:362). w_c = exp(lnW_c - ln_shift) for a chain
 * that reached N monomers and 0 for a dead chain; dead chains stay in every denominator
 * (reading A6 in DESIGN.md 4). All sums are deterministic: fixed chain->thread->block mapping,
 * warp shuffle tree, block tree, then a second kernel over the block partials; no float atomics.
 */
typedef struct rosen_summary {
    uint64_t n_chains;            /* chains attempted                                                  */
    uint64_t n_dead;              /* chains that hit m_s = 0                                           */
    uint64_t n_steps_attempted;   /* sum over chains of growth steps attempted (= monomer-steps)       */
    double   ln_shift;            /* L: lattice ln6 + (N-2) ln5, real space (N-1) ln k; long chains    */
                                  /*    (lattice N > 512, real space N > 2048): the largest lnW of the */
                                  /*    call, 0 if no chain is alive (reading A18)        */
    double   sum_w, sum_w_ree2, sum_w_rg2, sum_w2;
    double   mean_ree2;           /* sum_w_ree2 / sum_w   : W-weighted <R_ee^2>                        */
    double   mean_rg2;            /* sum_w_rg2 / sum_w    : W-weighted <R_g^2>                         */
    double   attrition;           /* n_dead / n_chains                                                 */
    double   ln_mean_W;           /* L + ln(sum_w / n_chains) = ln Z_N estimate (Eq. 6)                */
    uint64_t digest_xor;          /* XOR / wrapping sum of the per-chain digests; 0 unless             */
    uint64_t digest_sum;          /*   outputs->digest was requested                                   */
} rosen_summary;

/*
 * Optional per-chain outputs ("coordinates of each conformation and corresponding Rosenbluth
 * weight are flushed to the global memory"). Layouts are chain-major, C order.
 */
typedef struct rosen_outputs {
    double*   lnW;     /* [n_chains]            ln W = sum_s ln m_s (Eq. 3, :58); -inf for dead chains        */
    uint8_t*  alive;   /* [n_chains]            1 = reached N monomers                                         */
    uint8_t*  m_seq;   /* [n_chains][N-1]       m_s = number of free trials at step s; 0 from death on         */
    uint64_t* digest;  /* [n_chains]            FNV-1a fold of (m_s | choice_s << 8) per attempted step        */
    void*     conf;    /* [n_chains][N][3]      int32 (lattice) / float (real space); 0 after the death step   */
    double*   ree2;    /* [n_chains]            |r_{N-1} - r_0|^2; 0 for dead chains                           */
    double*   rg2;     /* [n_chains]            (1/N) sum_i |r_i - r_cm|^2; 0 for dead chains                  */
    int32_t   memory;  /* ROSEN_MEM_DEVICE or ROSEN_MEM_HOST for ALL pointers above                            */
    int32_t   reserved;
} rosen_outputs;

/*
 * Cubic-lattice Rosenbluth generation (sec. 3.3.2 + Algorithm 1; weight Eq. 3).
 * Each chain starts at the origin and grows to N monomers; at step s (1..N-1) the 6 neighbours of
 * r_{s-1}, in the order +x,-x,+y,-y,+z,-z, are tested against all earlier monomers, m_s = number
 * of free ones, lnW += ln m_s, and the ((u_s * m_s) >> 32)-th free neighbour is taken, u_s being
 * word s&3 of Philox4x32-10(key = seed, counter = (id_lo, id_hi, s>>2, 0)). m_s = 0 kills the
 * chain (W = 0, kept). 2 <= N <= ROSEN_LATTICE_MAX_N. For N >= ROSEN_LATTICE_HASH_MIN_N the library keeps device
 * workspace (at most 12 GiB of per-chain hash tables + 40 bytes per chain of the largest call) until
 * rosen_workspace_release(); decisions (trajectory, m sequence, digest) do not depend on which kernel ran, lnW and the sums agree to 1e-12
 * (different rounding order). The tables are cleared only when they are allocated or their layout changes. That workspace is one per
 * device; the library keeps the calls that share it apart itself (see Conventions above).
 */
ROSEN_API int rosen_lattice_generate(int32_t N, uint64_t n_chains, uint64_t seed, uint64_t chain_offset,
                           const rosen_outputs* outputs, rosen_summary* summary, void* cuda_stream);

/*
 * Real-space (off-lattice) Rosenbluth generation (PAPER.md:185-187 sec. 3.3.3, :202-262 Alg. 2).
 * At step s, k_trials unit directions u_t come from Philox blocks (id_lo, id_hi, s, 1 + (t>>1))
 * (words 0,1 for even t, 2,3 for odd t) through the fp32 map of DESIGN.md 3.3; trial_t =
 * fma(bond_len, u_t, r_{s-1}); it overlaps if fma(dz,dz,fma(dy,dy,dx*dx)) < sigma*sigma (fp32)
 * for some j <= s-2; m_s = number of non-overlapping trials; the ((u_s*m_s)>>32)-th of them in
 * trial order is taken, u_s as in the lattice call. 2 <= N <= ROSEN_REALSPACE_MAX_N,
 * 1 <= k_trials <= 255, bond_len > 0, sigma >= 0, both finite. N >= ROSEN_REALSPACE_CELL_MIN_N uses the library's
 * long-chain workspace like the lattice call.
 */
ROSEN_API int rosen_realspace_generate(int32_t N, uint64_t n_chains, int32_t k_trials, float bond_len, float sigma,
                             uint64_t seed, uint64_t chain_offset,
                             const rosen_outputs* outputs, rosen_summary* summary, void* cuda_stream);

/*
 * Other trial sets and Boltzmann-weighted trials (readings A19-A21).
 *
 * Lattice: z = 6 (the order above) or z = 26, "all z = 26 possible lattice space" (sec. 3.3.2): the 26 sites
 * (dx,dy,dz) in {-1,0,1}^3 \ {0} around r_{s-1}, trial d = rank of (dx+1) + 3(dy+1) + 9(dz+1), site exclusion only.
 * Energy U = -eps per non-bonded contact (Eq. 1-2): a free trial t whose site has c_t earlier monomers
 * j <= s-2 on its z neighbour sites carries Q[c_t], Q[c] = round(q^c 2^16), q = exp(beta_eps) (fixed point: exact sums);
 * W_s = sum_t Q[c_t]; the trial taken is the first, in trial order, whose cumulative sum exceeds floor(u_s W_s / 2^32);
 * lnW += log(W_s 2^-16). m_seq = number of free trials; the chain is dead when that is 0. beta_eps = 0 reproduces
 * rosen_lattice_generate decision for decision. 2 <= N <= ROSEN_LATTICE_MODEL_MAX_N, 0 <= beta_eps <= ROSEN_MODEL_MAX_BETA_EPS.
 * summary->ln_shift is the largest lnW of the call. Uses 40 bytes per chain of library workspace (rosen_workspace_release).
 *
 * Real space: square well of range lambda sigma (lambda >= 1) and depth eps around every monomer: c_t = number of earlier
 * monomers j <= s-2 with d2 < fl32(fl32(lambda sigma)^2), d2 the fp32 expression of the overlap test, capped at 31; the
 * rest as on the lattice. 2 <= N <= ROSEN_REALSPACE_MODEL_MAX_N.
 */
#define ROSEN_LATTICE_MODEL_MAX_N    256
#define ROSEN_REALSPACE_MODEL_MAX_N  399
#define ROSEN_MODEL_MAX_BETA_EPS     0.85
ROSEN_API int rosen_lattice_generate_model(int32_t N, uint64_t n_chains, uint64_t seed, uint64_t chain_offset,
                                 int32_t z, double beta_eps,
                                 const rosen_outputs* outputs, rosen_summary* summary, void* cuda_stream);
ROSEN_API int rosen_realspace_generate_model(int32_t N, uint64_t n_chains, int32_t k_trials, float bond_len, float sigma,
                                   float lambda, double beta_eps, uint64_t seed, uint64_t chain_offset,
                                   const rosen_outputs* outputs, rosen_summary* summary, void* cuda_stream);

/*
 * PERM, the pruned-enriched Rosenbluth method, on the cubic lattice. The paper names
 * it only as the topic of its supplement (not available); the algorithm is P. Grassberger's (Phys. Rev. E
 * 56, 3682 (1997)), depth-first, one TOUR per id: the chain grows as in rosen_lattice_generate; after a step that brings it
 * to n monomers (2 <= n <= N-1) with weight W, lnW > ln_hi[n] replaces it by two copies of weight W/2 (enrichment),
 * lnW < ln_lo[n] kills it with probability 1/2 and doubles its weight otherwise (pruning); every chain of the tour that
 * reaches N monomers is a leaf. ln_lo, ln_hi: HOST arrays of N+1 doubles (entries 2..N-1 are read; -inf / +inf switch
 * the control off, and a tour is then exactly the chain of the same id). The estimate of Z_N is unbiased for any
 * thresholds. ln_ref: leaf weights are summed inside a tour as exp(lnW - ln_ref) (choose ~ ln Z_N). A tour stops after
 * max_nodes growth steps. Random words: DESIGN.md 3.7.
 * Per-tour outputs (tour i has id tour_offset + i): lnW = ln(sum of its leaf weights), -inf without a leaf; ree2 / rg2 =
 * its weight-averaged leaf observables; alive = 1 (some leaf), 0 (none), 2 (stopped at max_nodes); digest of its decisions;
 * m_seq and conf must be NULL. Summary: n_chains = tours, n_dead = tours without a leaf, n_steps_attempted = growth steps
 * of all tours, sums over tours of exp(lnW - ln_shift) with ln_shift = the largest lnW, mean_ree2 / mean_rg2 = weighted means
 * over all leaves, ln_mean_W = estimate of ln Z_N (Eq. 6). 2 <= N <= ROSEN_PERM_MAX_N.
 */
#define ROSEN_PERM_MAX_N 512
ROSEN_API int rosen_lattice_perm(int32_t N, uint64_t n_tours, uint64_t seed, uint64_t tour_offset,
                       const double* ln_lo, const double* ln_hi, double ln_ref, uint32_t max_nodes,
                       const rosen_outputs* outputs, rosen_summary* summary, void* cuda_stream);

/*
 * Enqueue-only variants: same computation, but nothing is synchronised. All outputs must be device
 * memory (outputs->memory == ROSEN_MEM_DEVICE, else ROSEN_EINVAL); `summary_device` is a DEVICE
 * pointer (may be NULL) that the second reduction pass fills on `cuda_stream`, derived fields
 * included. Used to time the path with inputs/outputs resident in HBM and to overlap calls. The one exception to
 * "enqueue only": a long-chain call (N >= ROSEN_LATTICE_HASH_MIN_N / ROSEN_REALSPACE_CELL_MIN_N) that finds the library's
 * workspace missing or too small allocates it, which synchronises the device once; repeated calls of a size do not.
 */
ROSEN_API int rosen_lattice_generate_async(int32_t N, uint64_t n_chains, uint64_t seed, uint64_t chain_offset,
                                 const rosen_outputs* outputs, rosen_summary* summary_device, void* cuda_stream);
ROSEN_API int rosen_realspace_generate_async(int32_t N, uint64_t n_chains, int32_t k_trials, float bond_len, float sigma,
                                   uint64_t seed, uint64_t chain_offset,
                                   const rosen_outputs* outputs, rosen_summary* summary_device, void* cuda_stream);

/*
 * rosen_lattice_generate_noalloc -- the lattice call for callers that must not allocate device memory.
 *
 * Who needs it: a host program that gave the whole GPU to its own allocator at start-up (a simulation code with one big
 * arena, a framework whose caching allocator already holds every free byte) finds that a cudaMalloc inside a library
 * either fails or takes memory the program had budgeted for itself; a service with a fixed, audited memory footprint
 * may not let a library grow it behind its back; and a loop that must not stall cannot afford cudaMalloc / cudaFree,
 * which synchronise the whole device. Every other generate call of this header allocates on its first use (block
 * partials, a pinned summary mirror, events; workspaces for long chains). This one allocates nothing, ever: it makes no
 * cudaMalloc*, cudaFree*, cudaHostAlloc, stream / event creation or other allocating call, on the first call or later.
 *
 * What it computes: exactly rosen_lattice_generate_async (same kernel -- the shared-memory scan kernel of lattice.cu --
 * same chain ids, same virtual-block partition, same reduction order), so per-chain outputs and every field of the
 * summary are bit-identical to that call for N < ROSEN_LATTICE_HASH_MIN_N; for longer chains the regular call switches
 * kernels, and the two agree decision for decision with lnW and the sums within 1e-12, as documented above.
 *
 * Where the scratch lives: the kernel's scratch (one 64-byte block partial per virtual block + the virtual-block
 * ticket) sits in a static __device__ array inside librosen.so, ROSEN_NOALLOC_SCRATCH_BYTES = 512 KiB + 256 B. The
 * CUDA runtime places it on every GPU on which the process uses this library, and it stays there until the process
 * exits; that is the whole price.
 *
 * Limits: 2 <= N <= ROSEN_NOALLOC_MAX_N (the scan kernel's range; longer chains need gigabytes of hash tables, which
 * no static array can hold) and 1 <= n_chains <= ROSEN_NOALLOC_MAX_CHAINS per call (one partial per 2048 chains fills
 * the array). Anything beyond returns ROSEN_ERANGE with a message naming the limit and launches nothing; cover a
 * larger population with several calls over consecutive chain_offset ranges and merge the summaries with
 * rosen_summary_merge (bit-identical per chain; that is what the ids are for).
 *
 * Arguments: outputs (may be NULL) must hold DEVICE pointers only (memory == ROSEN_MEM_DEVICE, else ROSEN_EINVAL: a
 * host destination would need a staging allocation). summary_device (may be NULL) is a DEVICE pointer to
 * sizeof(rosen_summary) caller-owned bytes, 8-byte aligned, filled on cuda_stream, derived fields included; copy it
 * out yourself. The call only enqueues work (one cudaMemsetAsync of the 4-byte ticket, the generation kernel, and the
 * second reduction pass when summary_device is set) and returns; nothing is synchronised.
 *
 * First call on each device: it looks up the device address of the static array (cudaGetSymbolAddress, with that device
 * current) and remembers it; this is also when the CUDA runtime loads the library's kernels onto that device. Make that
 * first call during start-up, outside any stream capture; later calls on the device do no set-up at all.
 *
 * Sharing: all no-allocation calls on a device use the SAME array. The ticket is re-zeroed on the stream by every call
 * and every partial the second pass reads is rewritten by the kernel first, so a call never sees what the previous one
 * left behind -- provided the calls do not overlap on the GPU. Two such calls in flight at once on one device (different
 * streams without an event between them) race on the array and give wrong sums: keep them on one stream or order them
 * yourself; the library takes no lock and records no event here, since creating one would allocate. The array is
 * private to this entry point, so these calls do not disturb, and are not disturbed by, the other calls of this header.
 */
#define ROSEN_NOALLOC_MAX_N         ROSEN_LATTICE_SCAN_MAX_N
#define ROSEN_NOALLOC_MAX_CHAINS    (1ull << 24)
#define ROSEN_NOALLOC_SCRATCH_BYTES (8192 * 64 + 256)
ROSEN_API int rosen_lattice_generate_noalloc(int32_t N, uint64_t n_chains, uint64_t seed, uint64_t chain_offset,
                                   const rosen_outputs* outputs, rosen_summary* summary_device, void* cuda_stream);

/*
 * The direction map "rngonsphere" of Alg. 2 line 10 (reading A10) alone, as the real-space
 * kernels evaluate it: dir_xyz[3 i .. 3 i + 2] = unit vector of the Philox word pair (wz[i], wphi[i]). A component of
 * step R1 exposed so that parity tests can sweep it exhaustively (all 2^23 polar values; every azimuth octant) against
 * the oracle and against IEEE arithmetic on the host. wz, wphi, dir_xyz: n, n and 3 n elements, all device pointers
 * (memory == ROSEN_MEM_DEVICE, enqueue only) or all host pointers (ROSEN_MEM_HOST: staged, synchronous).
 */
ROSEN_API int rosen_direction_eval(const uint32_t* wz, const uint32_t* wphi, uint64_t n, float* dir_xyz, int32_t memory,
                                   void* cuda_stream);

/*
 * Conformation dump alone (the store path of PAPER.md:80 / :189, BASELINE config 5): identical to
 * the generate calls with outputs = {conf, lnW} only, provided as named entry points.
 * conf/lnW are DEVICE pointers when memory == ROSEN_MEM_DEVICE, host pointers otherwise.
 */
ROSEN_API int rosen_lattice_dump(int32_t N, uint64_t n_chains, uint64_t seed, uint64_t chain_offset,
                       int32_t* conf, double* lnW, int32_t memory, rosen_summary* summary, void* cuda_stream);
ROSEN_API int rosen_realspace_dump(int32_t N, uint64_t n_chains, int32_t k_trials, float bond_len, float sigma,
                         uint64_t seed, uint64_t chain_offset,
                         float* conf, double* lnW, int32_t memory, rosen_summary* summary, void* cuda_stream);

/*
 * The store phase of rosen_realspace_dump ALONE ("HBM GB/s is only meaningful for the store phase
 * measured alone ... a dump-only kernel"): every lane group keeps one synthetic chain (r_i = (i, i/2, -i)) resident in
 * shared memory and stores it to conf[c][N][3] (and (double)c to lnW[c], if non-NULL) for every chain c < n_chains, with
 * the store routine, block size and grid of the config-5 kernel realspace_kernel<G=32>. Enqueue only; conf, lnW are
 * DEVICE pointers of 3 N n_chains floats / n_chains doubles. A measurement entry: bytes stored = n_chains (12 N + 8).
 */
ROSEN_API int rosen_realspace_dump_probe(int32_t N, uint64_t n_chains, float* conf, double* lnW, void* cuda_stream);

/*
 * Merge the summaries of disjoint chain ranges generated with the same (N, k_trials) -- the only
 * "exchange" a multi-GPU run needs. Sums are added in array order (deterministic),
 * derived fields recomputed. Parts with different ln_shift (long chains) are rescaled to the largest shift of a
 * part with sum_w > 0. Returns ROSEN_EINVAL if count == 0 or a shift is not finite.
 * Pure host function.
 */
ROSEN_API int rosen_summary_merge(const rosen_summary* parts, int32_t count, rosen_summary* merged);

/*
 * Scaling analysis of a length sweep (sec. 4.1: Eq. 4 <R_N^2> = a N^(2 nu); Eq. 5-7
 * ln Z_N ~ N ln mu + (gamma - 1) ln N with Z_N = <W_N>, Eq. 6). Ordinary least squares over `count` lengths:
 *   ln mean_ree2[i] = ln a + 2 nu ln x_i                       (count >= 2)
 *   ln_mean_W[i]    = c + x_i ln mu + (gamma - 1) ln x_i       (count >= 3; skipped, fields NaN, if count == 2)
 * with x_i = N[i] - 1 (number of steps; reading A14 of DESIGN.md 4) if use_steps != 0, else x_i = N[i].
 * Pure host function over the summaries of rosen_lattice_generate / rosen_realspace_generate calls
 * (ln_mean_W of real space must have (N-1) ln k subtracted by the caller if mu per trial is wanted).
 * Returns ROSEN_EINVAL on count < 2, N[i] < 2, non-positive mean_ree2, non-finite input or a singular system.
 */
typedef struct rosen_fit {
    double nu, ln_a;              /* Eq. 4 */
    double mu, gamma, c;          /* Eq. 5-7 */
    double rms_ree2, rms_lnZ;     /* root-mean-square residuals of the two fits (log scale) */
} rosen_fit;

ROSEN_API int rosen_fit_exponents(const int32_t* N, const double* mean_ree2, const double* ln_mean_W,
                                  int32_t count, int32_t use_steps, rosen_fit* fit);

/* Bytes of device memory the library currently keeps on the current device (informational): block partials and the summary
 * slot (always), plus whatever the calls made so far left behind -- the long-chain tables (at most 12 GiB) with their
 * generation counters (4 MiB), 40 bytes per chain of the largest long-chain / model / PERM call, the PERM thresholds (8 KiB).
 * Not counted: staging buffers of ROSEN_MEM_HOST calls. Those are stream-ordered allocations from the device's DEFAULT memory
 * pool, whose release threshold the library raises on first use so that freed staging memory (3.2 GB at BASELINE config 5)
 * stays in the pool for the next call instead of going back to the driver at every synchronisation; other users of
 * cudaMalloc on the device do not see that memory as free until rosen_workspace_release() trims the pool. */
ROSEN_API size_t rosen_workspace_bytes(void);

/* Free what the calls on the current device left behind: the long-chain / model / PERM workspace, the mapped flags, copy
 * stream and ordering event of earlier calls, and the unused part of the default memory pool (cudaMemPoolTrimTo 0). Waits for
 * calls of other host threads on this device to return, then synchronises the device. Always ROSEN_OK; later calls allocate
 * again what they need. */
ROSEN_API int rosen_workspace_release(void);

/*
 * Test and tuning knobs (process-wide; value 0 restores the default). The library never reads the environment: these are
 * the only way to change which kernel serves a chain length, so a stray variable cannot alter results at the 1e-12 level.
 *   "lattice_hash_min_n"   2 .. 513   chain length from which rosen_lattice_generate uses the hash-map kernel
 *   "realspace_cell_min_n" 2 .. 2049  same for rosen_realspace_generate and the cell-list kernel
 *   "realspace_cand_cap"   33 .. 160  candidates a warp of the cell-list kernel buffers before a flush (33: every round)
 *   "hash_blocks_per_sm"   1 .. 32    cap on resident blocks of the hash-map kernel (tuning)
 *   "generations_left"     >= 0       not a knob but an action on the current device's long-chain workspace (there must be
 *                                     one): every thread / warp of the next long-chain calls of the same layout wraps its
 *                                     generation counter -- clears its table and restarts -- after `value` more chains.
 *                                     Clears the tables (no old entry may carry a generation that is about to be used
 *                                     again) and synchronises the device.
 * Decisions (trajectory, m sequence, digest) never depend on a knob. Returns ROSEN_EINVAL for an unknown name or a value
 * out of range.
 */
ROSEN_API int rosen_debug_set(const char* knob, int64_t value);

/*
 * Number of kernel launches the last generate/dump call on this thread enqueued, and the name of
 * the main kernel variant it chose (static string). For bench.py's gpu_launches and profiles.
 */
ROSEN_API int32_t     rosen_last_launch_count(void);
ROSEN_API const char* rosen_last_kernel_name(void);

/* Static description of an error code; rosen_last_error() adds the CUDA error text of the last
 * failing call on this thread (empty string if none). */
ROSEN_API const char* rosen_strerror(int code);
ROSEN_API const char* rosen_last_error(void);

/* Library version string, e.g. "rosen-b200 0.1 (sm_100a)". */
ROSEN_API const char* rosen_version(void);

#ifdef __cplusplus
}
#endif
#endif /* ROSEN_H */
