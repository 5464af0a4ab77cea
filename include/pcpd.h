/*
 * pcpd.h - C ABI of libpcpd.so: the B200-native (sm_100a) hot path of
 * arXiv 1301.6082 (Schram, "Reaction-diffusion model Monte Carlo simulations on
 * the GPU"): multispin Monte Carlo update of the 1+1-D pair contact process
 * with diffusion (PCPD, eq. (1); Alg. 1; bitwise
 * form Alg. 2) and its TCPD variant, with 64
 * independent replicas bit-packed per uint64 word (classic multispin coding,
 * PAPER.md:94-96).
 *
 * Conventions
 *   L sites, periodic.  R = n_replicas, W = R/64 words per site.  Word (i, w)
 *   holds replicas 64w .. 64w+63 at site i; bit j <-> replica 64w+j.
 *   CANONICAL order of a host lattice buffer: words[i*W + w].  (The device
 *   layout is private: column-major [W][L].)
 *   One sweep = one time unit = L attempted updates per replica.
 *   The update schedule, random streams and mask definition are the contract
 *   C1..C9 of DESIGN.md section 3 (SD2(T_s, D, A) shifted domains, Philox-4x32-10
 *   keyed by seed / sweep / slot / word, K = 32-plane Bernoulli masks).
 *
 * All pointers are HOST pointers unless the name ends in _dev.  Buffers are
 * caller-owned; the library owns all device memory of a handle.  Every call
 * returns 0 (PCPD_OK) or a negative pcpd_status; pcpd_create* return NULL on
 * error.  The message of the last error on the calling thread is available from
 * pcpd_last_error().  No C++ exception crosses this boundary.  A handle is used
 * by one host thread at a time; distinct handles are independent.  There is NO
 * CPU fallback: without a CUDA device of compute capability 10.x every compute
 * call fails with PCPD_ERR_DEVICE.
 */
#ifndef PCPD_H
#define PCPD_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define PCPD_API __attribute__((visibility("default")))
#else
#define PCPD_API
#endif

typedef struct pcpd_s pcpd_t;

enum pcpd_status {
    PCPD_OK = 0,
    PCPD_ERR_ARG = -1,     /* invalid argument (see pcpd_last_error) */
    PCPD_ERR_DEVICE = -2,  /* no usable sm_100 device / CUDA runtime error */
    PCPD_ERR_ALLOC = -3,   /* device allocation failed */
    PCPD_ERR_RANGE = -4    /* sweep counter would exceed 2^32 - 1 */
};

/* 0 PCPD (eq. (1)); 1 TCPD (config 5: triples, 5-site footprint); 2 QCPD (quadruplets
 * AAAA0/0AAAA -> AAAAA at (1-p)(1-d)/2 each, AAAA -> 0000 at p(1-d), A0 <-> 0A at d; 6-site footprint
 * {x-1 .. x+4}; needs D >= 11). */
/* 3 CPD: the contact process with diffusion, the one-particle member of that family (directed-percolation
 * class; this build's reading of the "DP" model of PAPER.md:15, 21): A0/0A -> AA at (1-p)(1-d)/2 each, A -> 0 at
 * p(1-d), A0 <-> 0A at d; 3-site footprint {x-1, x, x+1}; needs D >= 5. */
enum pcpd_variant { PCPD_VARIANT_PCPD = 0, PCPD_VARIANT_TCPD = 1, PCPD_VARIANT_QCPD = 2, PCPD_VARIANT_CPD = 3 };
/* Flag to OR into `variant`: use the PAPER's OWN annihilation mask instead of independent
 * per-lane Bernoulli(p) bits (Alg. 2 lines 12-13; section 4.3):
 * lane j of Pm = a0_j & a1_j & [u < 4p], a0/a1 = the two 64-lane planes of ANNI block 0 (an
 * independent 1/4-bit per lane), u = x3 of the MISC block, ONE draw per attempt-word shared by
 * its 64 lanes, compared as a 32-bit integer with floor(4p * 2^32).  Each lane is 1 w.p. p but
 * lanes of a word are partially correlated.  Requires p < 1/4 (else PCPD_ERR_ARG).
 * Costs 3 Philox blocks per attempt-word when d is a short dyadic (d = 1/2, 1/4, 3/4: the
 * paper's AND/OR recipe for d, is what C3 reduces to for such d). */
#define PCPD_VARIANT_PMASK_PAPER 0x100
/* With PCPD_VARIANT_PMASK_PAPER: the other members of the paper's mask family (section 4.3): per-lane
 * independent "decorrelation" bits that are 1 w.p. b, ANDed with the ONE word-wide draw, now 1 w.p. p/b (compared as
 * floor((p/b) * 2^32) with p/b formed as 4p, 2p, p, 4p/3).  Default b = 1/4 (Alg. 2: two raw words ANDed);
 * _BOUND_HALF: b = 1/2 (one raw word, plane lo of ANNI block 0); _BOUND_ONE: b = 1, no decorrelation - "all N_r bits
 * are set to 1 with probability p and all 0 otherwise", fully correlated lanes; _BOUND_3_4: b = 3/4 (two
 * raw words ORed; "correlated bits that are one with probability 4p/3").  Requires p < b; the bound bits
 * without PCPD_VARIANT_PMASK_PAPER are an error.  This is the paper's "number of decorrelation bits" knob. */
#define PCPD_VARIANT_PMASK_BOUND_HALF 0x400
#define PCPD_VARIANT_PMASK_BOUND_ONE 0x800
#define PCPD_VARIANT_PMASK_BOUND_3_4 0xC00
/* Flag to OR into `variant`: the PAPER's CONNECTED multispin lattice instead of
 * 64 independent replicas per word: the 64 bit-lanes of a word column are 64 consecutive segments of
 * ONE periodic lattice of 64*L sites (strand position lane*L + site); the successor of (site L-1,
 * lane j) is (site 0, lane (j+1) mod 64).  n_replicas/64 such lattices are simulated; pcpd_density
 * still returns per-lane counts (sum 64 consecutive entries for a lattice's particle number).
 * Schedule, streams and masks are unchanged: an attempt-word updates 64 positions L sites apart. */
#define PCPD_VARIANT_CONNECTED 0x200
enum pcpd_init_mode { PCPD_INIT_FULL = 0, PCPD_INIT_BERNOULLI = 1, PCPD_INIT_EMPTY = 2 };

/* Default schedule constants of SD2 (C5). */
#define PCPD_DEFAULT_TS 2048u
#define PCPD_DEFAULT_D 64u
#define PCPD_DEFAULT_A 4u

/* ---- plumbing: device memory and stream come from the host framework ------
 * Optional.  alloc(bytes, stream) returns a DEVICE pointer (NULL on failure),
 * release(ptr) frees it.  The Python binding installs PyTorch's CUDA caching
 * allocator here; without it the library uses cudaMalloc/cudaFree.  Process
 * wide; every handle remembers the pair it was created with and frees its buffers
 * through it.  PCPD_ERR_ARG while any handle is alive, or if only one of the two is given.
 * Thread-safe, like pcpd_create* (first-use configuration of a device is serialised). */
typedef void *(*pcpd_alloc_fn)(size_t bytes, void *cuda_stream);
typedef void (*pcpd_free_fn)(void *dev_ptr);
PCPD_API int pcpd_set_allocator(pcpd_alloc_fn alloc, pcpd_free_fn release);

/* cudaStream_t (as void*) every later call of this handle enqueues on.
 * Default: the legacy default stream. */
PCPD_API int pcpd_set_stream(pcpd_t *h, void *cuda_stream);

/* ---- the path -------------------------------------------------------------
 * pcpd_create: variant 0 = PCPD, 1 = TCPD.  Schedule SD2(2048, 64, 4).
 * Errors (NULL): n_replicas == 0 or not a multiple of 64; L not a multiple of
 * the domain length D, or L < D; T_s is clamped to L when L < T_s, otherwise
 * L % T_s != 0 is an error; d, p outside [0,1] or NaN; L > 2^31 or
 * W >= 2^32; unknown variant; allocation failure; no sm_100 device. */
PCPD_API pcpd_t *pcpd_create(uint64_t L, uint64_t n_replicas, double d, double p, uint64_t seed, int variant);

/* Test hook: with the environment variable PCPD_FORCE_BLOCK_KERNEL=1 set at create time the handle
 * runs the generic block-per-tile sweep kernel instead of the warp-per-tile one (same results, bit
 * for bit; used by the parity tests to cross-check the two kernels at full size). */

/* Same with explicit schedule constants (D | T_s | L, A | D, D >= 2*Rr+3 with
 * Rr = 2 PCPD / 3 TCPD / 4 QCPD / 1 CPD; T_s*8 bytes (one tile column) must fit the 227 KB shared memory) and
 * a global word offset: the handle simulates word columns
 * word_offset .. word_offset + W - 1 of a larger run (multi-GPU sharding by
 * replica words); columns never interact, so the union of
 * shards is bit-identical to one big run. */
PCPD_API pcpd_t *pcpd_create_ex(uint64_t L, uint64_t n_replicas, double d, double p, uint64_t seed, int variant,
                       uint32_t T_s, uint32_t D, uint32_t A, uint64_t word_offset);

/* Per-word-column probabilities (one run scans p across p_c; contract C11 of DESIGN.md): word column w of the
 * handle (global column word_offset + w) uses d_w[w], p_w[w] - HOST arrays of n_replicas/64 doubles, copied at
 * create time - instead of one (d, p); everything else is as in pcpd_create_ex, and column w evolves bit for bit
 * as it would in a uniform run with (d_w[w], p_w[w]).  Errors as pcpd_create_ex, plus: NULL arrays, any entry
 * outside [0,1] or NaN, the PCPD_VARIANT_PMASK_PAPER flag (not available in this mode), a schedule the
 * warp-per-tile-column kernel cannot run (more than 32 domains per tile, T_s / D > 32, or a tile column above
 * 200 KiB, T_s > 25598).  pcpd_thresholds reports column 0's thresholds. */
PCPD_API pcpd_t *pcpd_create_scan(uint64_t L, uint64_t n_replicas, const double *d_w, const double *p_w, uint64_t seed,
                         int variant, uint32_t T_s, uint32_t D, uint32_t A, uint64_t word_offset);

/* mode 0: all sites occupied; 1: i.i.d. Bernoulli(1/2) from the INIT stream
 * (C8: word(i,w) = low 64 bits of block (i, 0, w, 4<<24)); 2: empty.
 * Resets the sweep counter to 0.  Asynchronous. */
PCPD_API int pcpd_init(pcpd_t *h, int mode);

/* Advance sweeps t0 .. t0+n-1, t0 = the handle's counter, so that
 * run(a); run(b) == run(a+b) bit for bit.  Asynchronous on the handle's stream.
 * PCPD_ERR_RANGE if the counter would pass 2^32 - 1. */
PCPD_API int pcpd_run(pcpd_t *h, uint64_t n_sweeps);

/* out_counts[r] = number of particles of replica r (C9; density = count / L is
 * the caller's division), r < n_replicas.  Synchronises the stream. */
PCPD_API int pcpd_density(pcpd_t *h, uint32_t *out_counts);

/* out_pairs[r] = number of adjacent occupied pairs sum_i q(i) q(next(i)) whose left site lies in
 * replica lane r (pair density of PAPER.md:203-208, Figs 5-6).  Independent replicas: next(L-1) =
 * site 0 of the same lane.  PCPD_VARIANT_CONNECTED: next(site L-1, lane j) = (site 0, lane j+1 mod 64)
 * of the same word column, so 64 consecutive entries sum to the pair count of that ring.  Synchronises. */
PCPD_API int pcpd_pair_density(pcpd_t *h, uint32_t *out_pairs);

/* A whole time series in one call (the paper's observable is rho(t) at many times, Fig. 1; pair
 * density PAPER.md:203-208): for k = 0 .. n_times-1 advance to sweep times[k] (absolute sweep indices, ascending,
 * times[0] >= the current counter; equal entries allowed) and record the per-replica particle counts into
 * out_counts[k*n_replicas + r] and / or the pair counts into out_pairs[k*n_replicas + r] (either may be NULL, not
 * both).  Same numbers as pcpd_run + pcpd_density / pcpd_pair_density called in a loop, but the records stay on the
 * device until the end: one read-back and one synchronisation for the series instead of one per record.
 * PCPD_ERR_ARG for non-ascending times, PCPD_ERR_RANGE past 2^32 - 1; on error the counter stays where it got to. */
PCPD_API int pcpd_run_series(pcpd_t *h, const uint64_t *times, uint64_t n_times, uint32_t *out_counts, uint32_t *out_pairs);

/* pcpd_run_series WITHOUT any allocation, for callers that cannot call cudaMalloc (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid it).  pcpd_run_series takes its device-side record buffer from the
 * allocator on every call; this variant keeps the records in ONE buffer of fixed size that is part of the library
 * image - a file-scope `static __device__` array of PCPD_STATIC_SERIES_MAX_COUNTS uint32 (2 MiB; every GPU that loads
 * the library holds it until the process exits) - and calls no cudaMalloc, cudaFree or allocating library routine.
 * Arguments, results and errors are those of pcpd_run_series, bit for bit, plus:
 *   PCPD_ERR_ARG if n_times * n_replicas * (number of non-NULL outputs) > PCPD_STATIC_SERIES_MAX_COUNTS;
 *   PCPD_ERR_ARG if the handle's first sweep would still compile its run-time specialised kernel (NVRTC and the
 *     module load allocate): run one sweep with pcpd_run first;
 *   PCPD_ERR_DEVICE if the current device is not the one the handle was created on.
 * The buffer is shared by ALL handles and calls on a device and keeps the last call's contents; each call clears the
 * part it uses on its own stream before use.  Calls that overlap on the GPU (two handles on different streams, or two
 * host threads) race on it: serialise them.  Synchronises the handle's stream before it returns. */
#define PCPD_STATIC_SERIES_MAX_COUNTS 524288u
PCPD_API int pcpd_run_series_static(pcpd_t *h, const uint64_t *times, uint64_t n_times, uint32_t *out_counts,
                                    uint32_t *out_pairs);

/* Effective exponent of a density series (host-side analysis; eq. (2) and Figs 5-6:
 * "a straight line is obtained by plotting delta_eff as a function of rho"):
 *     rho[k]   = mean over the n_replicas replicas of series[k*n_replicas + r] / L
 *     delta[k] = - ln(rho[k+m] / rho[k-m]) / ln(times[k+m] / times[k-m]),   m = half_window >= 1
 * i.e. delta_eff = -d ln rho / d ln t as a central difference in log-log coordinates.  `series` is what
 * pcpd_run_series wrote (particle counts or pair counts), `times` the sweep indices it was given.  out_rho,
 * out_delta: n_times doubles each; delta[k] is NaN where the window does not fit, where a time in it is 0 or
 * repeated, or where a density in it is 0.  Plain host arithmetic in double; no device is touched.
 * PCPD_ERR_ARG for NULL pointers, n_times == 0, n_replicas == 0, L == 0, half_window == 0 or descending times. */
PCPD_API int pcpd_delta_eff(const uint64_t *times, uint64_t n_times, const uint32_t *series, uint64_t n_replicas,
                            uint64_t L, uint32_t half_window, double *out_rho, double *out_delta);

/* Lattice in canonical order words[i*W + w], L*W uint64.  Synchronise. */
PCPD_API int pcpd_get_lattice(pcpd_t *h, uint64_t *out_words);
PCPD_API int pcpd_set_lattice(pcpd_t *h, const uint64_t *in_words);

/* One step from a HOST lattice, pipelined: the same result as
 *     pcpd_set_lattice(h, in_words); pcpd_run(h, n_sweeps); pcpd_density(h, out_counts);
 * (out_counts may be NULL: no density), but the upload is cut into chunks of 8 word columns - columns never
 * interact, so a chunk can run all its n_sweeps sweeps as soon as it has arrived - and the host-to-device copy of
 * chunk c+1 (a strided 2-D copy out of the canonical [i][w] layout, on a copy stream) overlaps the sweeps of chunk c.
 * in_words: canonical words[i*W + w], L*W uint64, pinned host memory for the copies to be asynchronous.  Handles
 * with fewer than 16 word columns, or whose 8-column chunks would not fill the GPU, run the plain sequence.
 * Synchronises.  Errors as the three calls. */
PCPD_API int pcpd_step_from_host(pcpd_t *h, const uint64_t *in_words, uint64_t n_sweeps, uint32_t *out_counts);

/* The same step from a host lattice in COLUMN-MAJOR order, in_columns[w*L + i] (word column w contiguous - the order
 * the device keeps; e.g. a checkpoint written from the device layout): a chunk of columns is then one contiguous copy
 * straight into the lattice, with no staging buffer and no transpose, at the full host-to-device rate (the strided
 * copy of pcpd_step_from_host out of 8 W-byte rows runs at about half of it), and the call allocates nothing on the
 * device.  Chunks are whole multiples of the most columns that fit two waves of warps, a short first one (the only
 * exposed copy) and growing ones after it (PCPD_STEP_CHUNK = columns per chunk overrides: uniform chunks).  Same result as pcpd_step_from_host on the transposed buffer, bit
 * for bit.  in_columns: L*W uint64, pinned host memory for the copies to be asynchronous.  Synchronises. */
PCPD_API int pcpd_step_from_host_columns(pcpd_t *h, const uint64_t *in_columns, uint64_t n_sweeps, uint32_t *out_counts);

/* Schedule / precision constants in force for this handle (T_s after
 * clamping; K = 32 planes), so an independent implementation can be run with
 * the same ones.  Any out pointer may be NULL. */
PCPD_API int pcpd_schedule_info(const pcpd_t *h, uint32_t *T_s, uint32_t *D, uint32_t *A, uint32_t *K);

/* 32-bit-resolution thresholds T_d, T_p = floor(q * 2^32) in force (C3). */
PCPD_API int pcpd_thresholds(const pcpd_t *h, uint64_t *T_d, uint64_t *T_p);

PCPD_API uint64_t pcpd_sweep(const pcpd_t *h);           /* current sweep counter      */
PCPD_API int pcpd_set_sweep(pcpd_t *h, uint64_t sweep);  /* checkpoint/resume          */
PCPD_API int pcpd_synchronize(pcpd_t *h);                /* cudaStreamSynchronize      */
PCPD_API void pcpd_destroy(pcpd_t *h);                   /* NULL-safe                  */
PCPD_API const char *pcpd_last_error(void);              /* thread-local, library-owned */

/* ---- run-time specialisation of the sweep kernel -------
 * d and p are constants for the life of a handle, and the kernel's compare of the random planes with
 * the bits of T_d, T_p (C3) is cheaper when those bits are compile-time constants.  For handles with more
 * tile columns than that limit (smaller ones run column_kernel) the first pcpd_run of a handle therefore compiles the SAME device
 * source with T_d, T_p - and the schedule constants T_s, D, A and L - as template constants (NVRTC,
 * sm_100a; about a second, once per process, device and parameter set) and runs that kernel from then on.  Results are identical bit for bit.  If
 * libnvrtc cannot be loaded or the compilation fails, the handle keeps the built-in generic-threshold
 * CUDA kernel (this is not a CPU fallback) and pcpd_jit_message() says why.  Environment, read by
 * pcpd_create*: PCPD_JIT=0 never specialise; PCPD_JIT=force specialise at every problem size (test
 * hook); PCPD_NVRTC_PATH = full path of libnvrtc.so.12 if it is not on the loader path; tuning /
 * inspection hooks PCPD_JIT_NUD, PCPD_JIT_NUP (prefix lengths), PCPD_JIT_OPTS (extra NVRTC options),
 * PCPD_JIT_DUMP (file to keep the cubin in, for cuobjdump -sass).  Not used with
 * per-word-column probabilities (pcpd_create_scan), nor when d = 1 or p = 1.
 * pcpd_jit_state: 1 the handle's sweeps run the specialised kernel; 0 not tried (no sweep yet) or not
 * applicable; -1 tried and unavailable.  pcpd_jit_launch_count: specialised-kernel launches of this
 * process (also counted by pcpd_launch_count).  pcpd_jit_selftest: compile only - needs libnvrtc but no
 * device - sweep_warp_kernel<variant, ..., T_d, T_p> and return the cubin size; PCPD_ERR_DEVICE and the
 * compiler's message in pcpd_last_error() on failure. */
PCPD_API int pcpd_jit_state(const pcpd_t *h);
PCPD_API const char *pcpd_jit_message(void);
PCPD_API uint64_t pcpd_jit_launch_count(void);
PCPD_API int pcpd_jit_selftest(int variant, uint32_t T_d, uint32_t T_p, uint64_t *cubin_bytes);

/* ---- small and mid-size problems: one block per tile column -----------
 * With fewer tile columns ((L / T_s) * W) than the GPU has warp slots to fill, one warp per tile column leaves the
 * machine idle and each sweep is the latency of one warp's chain of D attempts.  Handles with at most 768 tile columns
 * (384 or 296 when the thresholds need few random planes) therefore run column_kernel: one block per tile column in which producer warps compute the state-independent part
 * of every attempt (MISC block, footprint position, the complete masks Dm and Pm) into a shared-memory ring and two
 * update warps - one per 32-bit half of the 64 replica lanes, which never interact - apply the attempts in order.
 * Same results bit for bit.  Environment, read by pcpd_create*: PCPD_SPLIT=0 never (the fused kernel at every size);
 * PCPD_SPLIT=column at every size (test hook); PCPD_COL_NPROD = producer warps per block (tuning).
 * pcpd_split_launch_count: column_kernel launches of this handle (1 per sweep; 0 = fused kernel). */
PCPD_API uint64_t pcpd_split_launch_count(const pcpd_t *h);

/* Number of kernels this library has launched so far in this process. */
PCPD_API uint64_t pcpd_launch_count(void);

/* ---- roofline microbenchmarks -----------------------
 * Runs `iters` dependent-chain iterations of one instruction mix on every SM
 * (2048 threads per SM, 8 independent chains per thread) and returns the achieved
 * rate in out_rate (thread-instructions per second, or Philox blocks per second
 * for kinds 3 and 7), timed with CUDA events, best of 3.
 * kind 0: LOP3 only; 1: IMAD.WIDE.U32 + LOP3 1:1 (a Philox round's mix; rate counts
 * both); 2: 32-bit IMAD only; 3: Philox-4x32-10 blocks; 4: LOP3 + 32-bit IMAD 1:1 on
 * independent chains (do the ALU and FMA pipes co-issue?); 5: IMAD.WIDE.U32 + 3 LOP3
 * (the sweep kernel's mix: bench.py's roofline peak); 6: IMAD.HI.U32 only;
 * 7: Philox with mul.hi + mad.lo written separately (ptxas fuses them back).
 * Kinds 8 .. 15 are the curve behind the roofline peak (rate = instructions as written):
 * 8: IMAD.WIDE.U32 only; 9: wide : LOP3 = 1 : 2; 10: 1 : 4; 11: wide + 32-bit IMAD 1 : 1;
 * 12: IADD3 only; 13: wide + 3 LOP3 of which two read ONE register (and an immediate);
 * 14: wide + LOP3 + 2 IADD3; 15: 2 wide : 5 LOP3 : 1 IMAD (the sweep kernel's own mix).
 * PCPD_ERR_ARG for another kind, iters == 0 or a NULL out pointer. */
PCPD_API int pcpd_microbench(int kind, uint32_t iters, double *out_rate);

#ifdef __cplusplus
}
#endif
#endif /* PCPD_H */
