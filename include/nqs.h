/*
 * nqs.h -- C ABI of the B200-native batched local-energy library (libnqs_b200.so).
 *
 * What it computes (citations: /root/reference/PAPER.md line numbers):
 *
 *   log psi(s) = sum_i a_i s_i + sum_j log cosh(b_j + sum_i W_ji s_i)       Eq. 38, :385-390
 *       complex-parameter (holomorphic, :299 option 1) Restricted Boltzmann Machine;
 *       j = 0..M-1 hidden units, i = 0..N-1 sites, W is [M,N] row-major (W[j*N+i]).
 *
 *   E_loc(s)   = sum_s' <s|H|s'> psi(s') / psi(s)                            Eq. 4, :63-68, :89
 *       for H = sum_t c_t P_t with P_t a product of at most two Pauli matrices on distinct
 *       sites ("branch-free" operators, :473; up to eight with the *_k entry points); the connected configurations s' and matrix
 *       elements <s|P_t|s'> are generated on the fly on the device (Eq. 39, :418-426;
 *       Algorithm 1 lines 6-8, :163-194; the four-call sequence at :464-469).
 *
 * Conventions: spins are int8 +1/-1, +1 = up = sigma^z eigenvalue +1.
 * Row convention for matrix elements: <s|X_k|s'> = 1, <s|Y_k|s'> = -i s_k, <s|Z_k|s> = s_k,
 * with s' = s with site k flipped for X and Y.  Terms reaching the same s' are summed; a
 * (summed) matrix element that is exactly zero contributes nothing (":458 non-zero matrix
 * elements").  Im log psi is defined mod 2 pi (sum over hidden units of an unwrapped phase).
 *
 * General rules for every entry point
 *   - Pointers named d_* are DEVICE pointers, h_* are HOST pointers.  The caller owns every
 *     buffer; the library never frees or retains caller memory.  Term arrays (h_sites,
 *     h_paulis, h_coeffs) are read before the call returns.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Device
 *     entry points are asynchronous on that stream and never synchronise the device.  Scratch
 *     memory (parameter tables, tanh(theta), packed GEMM operands) is taken in stream order from a
 *     memory pool the library owns (one per device, cudaMallocFromPoolAsync on `stream`) and
 *     returned to it on every exit path; freed scratch stays cached in that pool until
 *     nqs_release() trims it.  Global mutable state: that pool, the per-device record of kernel
 *     attributes, a cache of compiled Hamiltonians (at most 8, reference counted), the options of
 *     nqs_set_option and the profiling events -- all guarded by mutexes / atomics except the
 *     profiling helpers.
 *   - The entry points that take a term list (nqs_local_energy, nqs_local_energy_host,
 *     nqs_enumerate_connected) compile and upload the Hamiltonian on a cache miss; that upload is a
 *     pageable-memory copy in stream order (the runtime may synchronise `stream` once for it, and a
 *     miss cannot be captured into a CUDA graph).  A cache hit costs a key comparison and makes `stream`
 *     wait for the event that closed the upload (a no-op on the stream that uploaded).  An evicted
 *     Hamiltonian is freed in stream order after its most recent use on every stream that used it (one
 *     event per stream; an entry used from more than 16 streams is freed with a synchronising cudaFree).
 *   - *_host entry points take HOST buffers, copy them to the device, run the same kernels,
 *     copy the result back and synchronise before returning.
 *   - Return value: 0 (NQS_OK) or a negative NQS_ERR_* code; nqs_last_error() then returns a
 *     thread-local message.  No partial results are promised on error.  B == 0 is a no-op.
 *   - There is NO CPU fallback: without a usable CUDA device every compute call returns
 *     NQS_ERR_CUDA.
 *   - Spin values other than +1/-1 are undefined behaviour, unless the environment variable
 *     NQS_VALIDATE=1 is set (read at every call): then every entry point that takes device spins
 *     checks them first, synchronises `stream`, and returns NQS_ERR_INVALID_ARG if any value is not
 *     +1 or -1 (debug mode).  psi(s) = 0 or overflow follow IEEE (inf/NaN in the output), not an error.
 */
#ifndef NQS_B200_H
#define NQS_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct { float re, im; } nqs_c64; /* == complex64, interleaved */

enum { NQS_I = 0, NQS_X = 1, NQS_Y = 2, NQS_Z = 3 };

enum {
    NQS_OK = 0,
    NQS_ERR_INVALID_ARG = -1,  /* NULL pointer, negative size, N/M out of range            */
    NQS_ERR_INVALID_TERM = -2, /* site out of range, Pauli code > 3, same site twice,      */
                               /* non-identity Pauli on an unused (-1) slot                */
    NQS_ERR_CUDA = -3,         /* CUDA runtime error or no device                          */
    NQS_ERR_UNSUPPORTED = -4   /* shape outside what the kernels support                   */
};

/* Opaque compiled Hamiltonian (step a0 of DESIGN.md): terms grouped by flip set, diagonal
 * list, per-group matrix-element programs, uploaded to the device once. */
typedef struct nqs_hamiltonian nqs_hamiltonian;

/* ---------------------------------------------------------------------------------------
 * log psi(s) for a batch (Eq. 38).
 *   d_spins  [B,N] int8 row-major, values +1/-1            d_a [N], d_b [M], d_W [M,N] complex64
 *   d_logpsi [B]   complex64 out
 * ------------------------------------------------------------------------------------- */
int nqs_log_psi(const int8_t *d_spins, int64_t B, int32_t N, int32_t M, const nqs_c64 *d_a,
                const nqs_c64 *d_b, const nqs_c64 *d_W, nqs_c64 *d_logpsi, void *stream);

/* ---------------------------------------------------------------------------------------
 * E_loc(s) for a batch (Eq. 4; Algorithm 1 lines 6-8).
 *   T terms: h_sites [T,2] int32 (-1 = unused slot), h_paulis [T,2] uint8 (NQS_I..NQS_Z),
 *   h_coeffs [T] complex64.  Both slots unused / identity = constant term c * 1.
 *   d_eloc [B] complex64 out; d_logpsi [B] complex64 out or NULL.
 * Compiles (or fetches from an internal cache keyed by the term bytes) the Hamiltonian, then
 * behaves as nqs_local_energy_h.
 * ------------------------------------------------------------------------------------- */
int nqs_local_energy(const int8_t *d_spins, int64_t B, int32_t N, int32_t M, const nqs_c64 *d_a,
                     const nqs_c64 *d_b, const nqs_c64 *d_W, int32_t T, const int32_t *h_sites,
                     const uint8_t *h_paulis, const nqs_c64 *h_coeffs, nqs_c64 *d_eloc,
                     nqs_c64 *d_logpsi, void *stream);

/* Same with HOST buffers for everything (spins, parameters, outputs): H2D copies, kernels,
 * D2H copies, stream synchronise.  h_logpsi may be NULL.  Batches of more than ~47000 samples go through
 * the device in chunks of 37888 samples (B200) on two library-owned streams, so that the copy of chunk k + 1
 * overlaps the kernels of chunk k (pinned host buffers are needed for the overlap; pageable ones work,
 * serially).  Calls on the same device are serialised. */
int nqs_local_energy_host(const int8_t *h_spins, int64_t B, int32_t N, int32_t M, const nqs_c64 *h_a,
                          const nqs_c64 *h_b, const nqs_c64 *h_W, int32_t T, const int32_t *h_sites,
                          const uint8_t *h_paulis, const nqs_c64 *h_coeffs, nqs_c64 *h_eloc,
                          nqs_c64 *h_logpsi);

int nqs_log_psi_host(const int8_t *h_spins, int64_t B, int32_t N, int32_t M, const nqs_c64 *h_a,
                     const nqs_c64 *h_b, const nqs_c64 *h_W, nqs_c64 *h_logpsi);

/* ---------------------------------------------------------------------------------------
 * Compiled-Hamiltonian handle (static for a whole simulation; parameters change every step).
 * nqs_hamiltonian_create validates the terms (NQS_ERR_INVALID_TERM), groups them by flip set
 * (Eq. 39: all terms of a group reach the same s') and uploads the result to the current
 * device.  The handle is immutable and may be used from several streams.
 * ------------------------------------------------------------------------------------- */
int nqs_hamiltonian_create(int32_t N, int32_t T, const int32_t *h_sites, const uint8_t *h_paulis,
                           const nqs_c64 *h_coeffs, nqs_hamiltonian **out);
int nqs_hamiltonian_destroy(nqs_hamiltonian *h);

/* k-site Pauli strings ("tensor products of branch-free operators"): the same
 * with K slots per term -- h_sites [T,K] int32 (-1 = unused slot), h_paulis [T,K] uint8 -- 1 <= K <= 8, all sites of
 * a term distinct.  A term may carry any number of Z / I factors and at most FOUR X / Y factors (a flip set of m
 * sites costs 2^(m-1) table columns, one per pattern of relative signs; NQS_ERR_UNSUPPORTED beyond four).  Handles
 * made this way work with every *_h entry point; nqs_hamiltonian_info_k reports the flip sets as [G,4] (-1 padded).
 * nqs_local_energy_k is nqs_local_energy for such a term list. */
int nqs_hamiltonian_create_k(int32_t N, int32_t T, int32_t K, const int32_t *h_sites, const uint8_t *h_paulis,
                             const nqs_c64 *h_coeffs, nqs_hamiltonian **out);
int nqs_hamiltonian_compile_host_k(int32_t N, int32_t T, int32_t K, const int32_t *h_sites, const uint8_t *h_paulis,
                                   const nqs_c64 *h_coeffs, nqs_hamiltonian **out);
int nqs_hamiltonian_info_k(const nqs_hamiltonian *h, int32_t info[5], int32_t *flip_sites4);
int nqs_local_energy_k(const int8_t *d_spins, int64_t B, int32_t N, int32_t M, const nqs_c64 *d_a,
                       const nqs_c64 *d_b, const nqs_c64 *d_W, int32_t T, int32_t K, const int32_t *h_sites,
                       const uint8_t *h_paulis, const nqs_c64 *h_coeffs, nqs_c64 *d_eloc, nqs_c64 *d_logpsi,
                       void *stream);

/* Host-side description of the compiled form (no device work; usable without a GPU when the
 * handle was made with nqs_hamiltonian_compile_host):
 *   info[0] = G  number of flip groups (distinct non-empty flip sets)
 *   info[1] = C  number of table columns (1 per single-flip group, 1 or 2 per pair group)
 *   info[2] = number of diagonal terms (empty flip set)
 *   info[3] = number of terms in flip groups
 *   info[4] = N
 * flip_sites, if not NULL, receives [G,2] int32: the group's flip set (second = -1 if single),
 * in group order (order of first appearance in the term list). */
int nqs_hamiltonian_info(const nqs_hamiltonian *h, int32_t info[5], int32_t *flip_sites);

/* Host-only compile (validation + grouping, nothing uploaded): for tests of the host logic on
 * machines without a GPU.  A handle made this way is rejected by the compute entry points. */
int nqs_hamiltonian_compile_host(int32_t N, int32_t T, const int32_t *h_sites, const uint8_t *h_paulis,
                                 const nqs_c64 *h_coeffs, nqs_hamiltonian **out);

/* E_loc with a compiled handle.  The connected amplitudes (step a5) run on the tensor cores as a guarded
 * series (csrc/nqs_series.cuh) when B * columns * M >= 2^28 and N <= 2048; the guard -- a per-sample bound on the
 * series' own error against 0.5e-4 * max(1, |E_loc|) -- is evaluated on the device and, if any sample fails it,
 * the FP32 product-form kernel recomputes the call in the same stream (no host synchronisation either way). */
int nqs_local_energy_h(const nqs_hamiltonian *h, const int8_t *d_spins, int64_t B, int32_t M,
                       const nqs_c64 *d_a, const nqs_c64 *d_b, const nqs_c64 *d_W, nqs_c64 *d_eloc,
                       nqs_c64 *d_logpsi, void *stream);

/* ---------------------------------------------------------------------------------------
 * Options (process-wide, atomic; meant for tests and benchmarks -- the defaults are the product).
 *   NQS_OPT_A5_PATH     0 = automatic (above)          1 = FP32 product form only
 *                       2 = series + guard + fallback at ANY size
 *                       3 = series only: the guard is evaluated and recorded but nothing is recomputed
 *   NQS_OPT_THETA_PATH  0 = automatic (int8 tcgen05 kernel for N <= 512, else FP32 SIMT)   1 = FP32 SIMT only
 *   NQS_OPT_SMALL_PATH  0 = automatic: below the series' size threshold, when columns x M x 16 bytes of tables and the
 *                       per-sample state of >= 4 samples fit in 200 KB of shared memory, ONE kernel does the whole call
 *                       (csrc/nqs_small.cuh; theta summed in float32 from W split into two exact float32 levels, the
 *                       log cosh terms accumulated in float64)                               1 = never (multi-launch path)
 *   NQS_OPT_THETA_SPLIT 0 = automatic: on the series path the hidden units of a sample tile are split over 1, 2, 4 or 8
 *                       CTAs of the theta kernel, whichever needs the fewest waves of the 2 x SMs CTA slots (partial
 *                       log psi / row norms combined in a fixed order: deterministic)         1 = never split
 *   NQS_OPT_SERIES_WIDE 0 = automatic: more than 128 table columns are tiled in column tiles of up to 224 (the series
 *                       GEMM then makes two passes over the hidden units with one accumulator pair in TMEM at a time,
 *                       csrc/nqs_series.cuh) where that fits in shared memory           1 = tiles of <= 128 columns only;
 *                       the two give the same bits
 *   NQS_OPT_HOST_CHUNKS 0 = automatic: nqs_local_energy_host sends the batch through the device in chunks of 2 x SMs x 128
 *                       samples (whole waves of the kernels; at most 16 chunks, a short remainder joins the last),
 *                       copying chunk k + 1 while the kernels of chunk k run      1 .. 16 = that many equal chunks
 *   NQS_OPT_SERIES_LATCH 0 = automatic: with NQS_OPT_A5_PATH = 0 a Hamiltonian handle (or cached term list) remembers that
 *                       the guard refused its last series attempt: the result of every attempt lands in pinned host
 *                       memory and is read at the next call WITHOUT synchronising (so it may lag by the calls still in
 *                       flight).  After a refusal the next 8 calls with that handle run the product form alone -- no
 *                       series operands, GEMM or guard are enqueued -- then one call probes the series again; the skip
 *                       doubles up to 64 calls while the probes keep failing and returns to 8 once one passes.  The
 *                       latch is per handle, not per parameter set: calls that alternate between parameters inside and
 *                       outside the guard's window on ONE handle run mostly on the product form (slower, never less
 *                       accurate).                                                           1 = no latch: every large
 *                       call attempts the series (round-2 behaviour)
 * nqs_debug_last_a5 (synchronises `stream`; tests only; not meaningful while calls run concurrently on other
 * streams): out[0] = 1 if the most recent nqs_local_energy* call on this device attempted the series path, 2 if
 * it used the product form only, 3 if the single-launch kernel for small problems ran; out[1] = 1 if the guard failed; out[2] = samples over the guard threshold.
 * ------------------------------------------------------------------------------------- */
enum { NQS_OPT_A5_PATH = 0, NQS_OPT_THETA_PATH = 1, NQS_OPT_HOST_CHUNKS = 2, NQS_OPT_SMALL_PATH = 3, NQS_OPT_THETA_SPLIT = 4, NQS_OPT_SERIES_WIDE = 5, NQS_OPT_SERIES_LATCH = 6, NQS_OPT_COUNT = 7 };
int nqs_set_option(int32_t key, int32_t value);
int nqs_get_option(int32_t key, int32_t *value);
int nqs_debug_last_a5(int32_t out[3], void *stream);

/* ---------------------------------------------------------------------------------------
 * Test/debug entry (small inputs): materialise Eq. 39 -- the connected configurations and
 * summed matrix elements per flip group (PAPER.md:456-458 get_s_primes).  Slot 0 is the
 * diagonal (s' = s, element = sum of the diagonal terms), slot 1+g is flip group g (groups in
 * order of first appearance in the term list):
 *   d_sprime [B,G+1,N] int8, d_mel [B,G+1] complex64.  A zero element means "not connected".
 * *G_out (may be NULL) receives G.  A call with B = 0 only compiles the term list on the host and
 * reports G (no device needed), so that the caller can size the outputs.
 * nqs_enumerate_connected_h is the same with a compiled handle.
 * ------------------------------------------------------------------------------------- */
int nqs_enumerate_connected(const int8_t *d_spins, int64_t B, int32_t N, int32_t T, const int32_t *h_sites,
                            const uint8_t *h_paulis, const nqs_c64 *h_coeffs, int8_t *d_sprime,
                            nqs_c64 *d_mel, int32_t *G_out, void *stream);
int nqs_enumerate_connected_h(const nqs_hamiltonian *h, const int8_t *d_spins, int64_t B,
                              int8_t *d_sprime, nqs_c64 *d_mel, void *stream);

/* Optional per-kernel timing for benchmarks.  nqs_profile_enable(1) makes every following
 * nqs_local_energy* call record CUDA events on its stream around its kernels;
 * nqs_profile_last() waits for the most recent such call and returns the elapsed milliseconds of
 *   ms[0] parameter tables (a1; product-form tables and the series' T^k planes)
 *   ms[1] theta / log psi / tanh (a2, a3)             ms[2] series operand packing (t^k planes)
 *   ms[3] series GEMM + fused epilogue (a4, a5, a6)   ms[4] series guard / E_loc
 *   ms[5] product-form kernel (a4, a5; exits at once when the series passed its guard)
 *   ms[6] final reduction of the product form (a6) and bookkeeping
 * Segments of kernels that were not launched read ~0.  Not thread-safe; off by default. */
enum { NQS_PROFILE_SEGMENTS = 7 };
int nqs_profile_enable(int on);
int nqs_profile_last(float ms[NQS_PROFILE_SEGMENTS]);

/* ---------------------------------------------------------------------------------------
 * Batch statistics (Eq. 5; get_global_mean / get_global_variance, :511-515).
 *   d_x [B] complex64 (any local estimator, e.g. E_loc);  d_weights [B] float32 or NULL (= uniform;
 *   with w_b = p(s_b) over a full basis the mean is the exact expectation of Eq. 3).  Weights must be
 *   non-negative with a positive sum (otherwise the outputs are NaN, no error is raised).
 *   d_stats [4] float64 DEVICE out: Re mean, Im mean, variance <<|x - mean|^2>>, sum of weights.
 * Sums are accumulated in float64 in a fixed order (deterministic).  Asynchronous on `stream`.  B == 0 is a
 * no-op (d_stats is left untouched).
 * ------------------------------------------------------------------------------------- */
int nqs_energy_stats(const nqs_c64 *d_x, const float *d_weights, int64_t B, double *d_stats, void *stream);

/* ---------------------------------------------------------------------------------------
 * nqs_energy_stats for callers that are not able to allocate device memory (Eq. 5).
 *
 * Who this is for.  Every other device entry point takes its scratch memory from a pool the library grows with
 * the CUDA allocator.  That is not possible for a host program whose own allocator has already claimed (almost)
 * all of the device's memory -- the paper's own environment is the example: a JAX/XLA process reserves the whole
 * GPU at start-up unless told otherwise, and inside such a process a library-side allocation
 * simply fails with "out of memory" although the program has plenty of room in its own arena.  It is also not
 * acceptable in a sampling / optimisation loop with a latency bound, because an allocation that has to go to the
 * driver may stall the whole device, nor in a deployment where device memory is handed out by a budget the
 * library is not part of.  Such callers still own d_x, d_weights and d_stats (carved out of their arena) and
 * pass them in; what they can not provide for is memory the library would take behind their back.
 *
 * What it does.  Same arguments, same kernels, same launch geometry and therefore the same bits in d_stats as
 * nqs_energy_stats.  The difference is where the per-block partial sums live: in a fixed 8 KB array (256 records
 * of four float64 sums) that is part of the library image itself, so it exists on every GPU that loads the
 * library, from load until the process exits, and costs nothing at call time.  This entry point makes no call to
 * cudaMalloc / cudaFree, to the stream-ordered allocator or to any library routine that allocates, and does not
 * create the library's pool.
 *
 * Limit.  B <= NQS_STATS_STATIC_MAX_B (2^26 samples = 512 MiB of complex64 input, 64 times the largest batch the
 * paper uses, N_MC = 10^6 at PAPER.md:622).  A larger B returns NQS_ERR_UNSUPPORTED with a message that names the
 * limit; nothing is launched.  (The 256 records are filled by a strided loop, so the array itself does not grow
 * with B; the cap is the range this entry point is specified and tested for.)
 *
 * First call on a device.  The first call made while a given device is current looks up the array's address on
 * that device (cudaGetSymbolAddress) and remembers it; later calls on that device reuse it.  Make that first call
 * during set-up, before any stream capture is begun, with the device you mean to use already current.
 *
 * One array for everybody.  All calls on a device, from every stream and every thread, use the same 8 KB, and the
 * array keeps whatever the previous call left in it.  No clearing is needed: each call overwrites every record it
 * is going to read before it reads it.  But two calls whose kernels can run on the GPU at the same time (different
 * streams without an event between them, or two host threads on different streams) overwrite each other's partial
 * sums and both results are then garbage -- keep calls on a device in one stream, or order them with events.
 * Asynchronous on `stream`; B == 0 is a no-op; weights as in nqs_energy_stats.
 * ------------------------------------------------------------------------------------- */
#define NQS_STATS_STATIC_MAX_B (1ll << 26)
int nqs_energy_stats_static(const nqs_c64 *d_x, const float *d_weights, int64_t B, double *d_stats, void *stream);

/* ---------------------------------------------------------------------------------------
 * Force vector of the RBM (Eq. 16; energy gradient Eq. 7, :81-89):
 *   F_k = <<E_loc O_k^*>>^c = <<O_k^* E_loc>> - <<O_k^*>> <<E_loc>>,
 *   O_k(s) = d log psi(s) / d theta_k (Eq. 8, :93):  O_{a_i} = s_i, O_{b_j} = tanh theta_j,
 *   O_{W_ji} = tanh theta_j s_i  with theta_j = b_j + sum_i W_ji s_i.
 *   d_eloc [B] complex64 in (the local energies of the same batch); d_weights [B] float32 or NULL.
 *   d_F [N + M + M*N] complex64 out, ordered a (i), b (j), W (row-major j*N + i) like the inputs.
 *   d_stats [4] float64 device out or NULL: as nqs_energy_stats of d_eloc.
 * The contraction over the samples runs on the tensor cores as an exact int8 GEMM (28-bit
 * fixed-point split of conj(tanh theta) (E - mean) per hidden unit), so the result does not depend
 * on the summation order.  B <= 2^25.  Asynchronous on `stream`.
 * ------------------------------------------------------------------------------------- */
int nqs_forces(const int8_t *d_spins, int64_t B, int32_t N, int32_t M, const nqs_c64 *d_a,
               const nqs_c64 *d_b, const nqs_c64 *d_W, const nqs_c64 *d_eloc, const float *d_weights,
               nqs_c64 *d_F, double *d_stats, void *stream);

/* One VMC evaluation step (Algorithm 1 lines 6-9): nqs_local_energy_h followed by
 * nqs_forces on the same batch, with theta and tanh(theta) computed once and shared.  Arguments as in
 * those two calls; d_logpsi and d_stats may be NULL.  Results are identical to the two separate calls. */
int nqs_local_energy_forces_h(const nqs_hamiltonian *h, const int8_t *d_spins, int64_t B, int32_t M,
                              const nqs_c64 *d_a, const nqs_c64 *d_b, const nqs_c64 *d_W,
                              const float *d_weights, nqs_c64 *d_eloc, nqs_c64 *d_logpsi, nqs_c64 *d_F,
                              double *d_stats, void *stream);

/* ---------------------------------------------------------------------------------------
 * Quantum Fisher matrix of the RBM (Eq. 10-11; Algorithm 1 line 9; get_global_covariance, :515):
 *   S_{k,k'} = << O_k^* O_k' >>_c = sum_b w_b (O_k(s_b) - <O_k>)^* (O_k'(s_b) - <O_k'>) / sum_b w_b,
 *   <O_k> = sum_b w_b O_k(s_b) / sum_b w_b,   O_k as in nqs_forces, K = N + M + M*N parameters in the order a, b, W.
 *   d_weights [B] float32 or NULL (uniform), as in nqs_energy_stats.
 *   d_S [K,K] complex64 out, row-major (Hermitian, both triangles written);  d_Obar [K] complex64 out or NULL: <O_k>.
 * The contraction over the samples runs on the tensor cores: FP16 tcgen05 GEMM with FP32 accumulation of the
 * centred derivatives split error-free into two FP16 parts (22 bits); <O_k> comes from the exact int8 contraction
 * of nqs_forces.  Entry errors are of order 1e-6 sqrt(S_kk S_k'k') (float32 tanh, FP32 accumulation over B / 16
 * MMA steps).  K <= 8192 (NQS_ERR_UNSUPPORTED above: S would exceed 512 MB), B <= 2^25.  Asynchronous on `stream`.
 * nqs_vmc_step_h: nqs_local_energy_forces_h plus S and <O> of the same batch (Algorithm 1 lines 6-9 in one call),
 * theta / tanh(theta) computed once.  d_logpsi, d_Obar and d_stats may be NULL.
 * ------------------------------------------------------------------------------------- */
int nqs_fisher(const int8_t *d_spins, int64_t B, int32_t N, int32_t M, const nqs_c64 *d_a, const nqs_c64 *d_b,
               const nqs_c64 *d_W, const float *d_weights, nqs_c64 *d_S, nqs_c64 *d_Obar, void *stream);
int nqs_vmc_step_h(const nqs_hamiltonian *h, const int8_t *d_spins, int64_t B, int32_t M, const nqs_c64 *d_a,
                   const nqs_c64 *d_b, const nqs_c64 *d_W, const float *d_weights, nqs_c64 *d_eloc,
                   nqs_c64 *d_logpsi, nqs_c64 *d_F, nqs_c64 *d_S, nqs_c64 *d_Obar, double *d_stats, void *stream);

/* ---------------------------------------------------------------------------------------
 * Metropolis sampling of p(s) = |psi(s)|^2 / <psi|psi> with single-spin-flip
 * proposals, C independent chains advanced in lock-step (:490-494); one sweep = N steps (:341).
 *   d_spins    [C,N] int8 DEVICE in/out: the chains' states (start -> after S steps)
 *   d_sites    [S,C] int32 DEVICE: the site proposed to chain c at step t is d_sites[t*C + c] in [0,N)
 *   d_u        [S,C] float32 DEVICE, uniform in [0,1): the move is accepted iff
 *                    u < |psi(s')/psi(s)|^2      (u = 0 always accepts)
 *   d_accepted [C] int32 DEVICE out or NULL: accepted moves per chain
 * The random numbers are the caller's (e.g. torch.randint / torch.rand on the device), so a call is
 * a deterministic function of its inputs.  The acceptance test is evaluated in float32 (a decision
 * closer to a tie than ~1e-4 in log |ratio|^2 may differ from exact arithmetic).  The chain state is
 * exp(2 theta), recomputed from the spins every two sweeps (2 N steps) and updated in place by one
 * complex multiplication per hidden unit on each accepted move.  Valid for |Re theta| < 22: beyond that
 * |exp(2 theta) + 1|^2 leaves the float32 range, the log-ratio becomes NaN and the chain stops accepting; such a
 * chain is REPORTED, not silently frozen: d_accepted[c] = -1 (its spins are then meaningless).  A proposal with
 * psi(s') = 0 exactly (log-ratio -inf) is an ordinary rejection, not an overflow.  Sites outside
 * [0,N) are undefined behaviour.  S = 0 is a no-op.  Asynchronous.
 * NQS_ERR_UNSUPPORTED if one chain's state (8 M + N bytes) does not fit shared memory twice.
 * ------------------------------------------------------------------------------------- */
int nqs_metropolis(int8_t *d_spins, int64_t C, int32_t N, int32_t M, const nqs_c64 *d_a,
                   const nqs_c64 *d_b, const nqs_c64 *d_W, int32_t S, const int32_t *d_sites,
                   const float *d_u, int32_t *d_accepted, void *stream);

/* Test/debug variant: additionally writes d_decisions [S,C] uint8 DEVICE (may be NULL), 1 = the proposal of
 * step t to chain c was accepted -- the trace a test compares with the oracle's, decision by decision. */
int nqs_metropolis_trace(int8_t *d_spins, int64_t C, int32_t N, int32_t M, const nqs_c64 *d_a,
                         const nqs_c64 *d_b, const nqs_c64 *d_W, int32_t S, const int32_t *d_sites,
                         const float *d_u, int32_t *d_accepted, uint8_t *d_decisions, void *stream);

/* Shared-site variant: at step t EVERY chain proposes the same site d_sites[t] (d_sites [S] int32 DEVICE; d_u,
 * d_accepted, d_decisions as in nqs_metropolis_trace, d_decisions may be NULL).  Each chain is still a valid
 * single-spin-flip Metropolis chain of p(s) (its proposal sequence is a fixed, chain-independent schedule -- e.g. a
 * random permutation of the sites per sweep -- and its uniforms are its own).  The table rows exp(+-4W)[site] are
 * then fetched once per thread block and step instead of once per chain, and the chain state lives in registers:
 * several times the throughput of nqs_metropolis.  M <= 2048, and the block's shared memory -- 128 + 64 M_pad +
 * warps x N_pad + 12 N bytes, M_pad = M rounded up to 16 -- must fit 227 KB, i.e. N up to a few thousand sites
 * (NQS_ERR_UNSUPPORTED otherwise; nqs_metropolis has no such bound on N).  Same arithmetic,
 * acceptance rule, float32 caveat and theta refresh (every 2 N steps) as nqs_metropolis. */
int nqs_metropolis_shared(int8_t *d_spins, int64_t C, int32_t N, int32_t M, const nqs_c64 *d_a,
                          const nqs_c64 *d_b, const nqs_c64 *d_W, int32_t S, const int32_t *d_sites,
                          const float *d_u, int32_t *d_accepted, uint8_t *d_decisions, void *stream);

/* Pipe-rate micro-benchmark (the roofline is quoted against the nominal peak
 * AND a peak measured on the box).  Runs a register-only kernel (2 blocks of 320 threads per SM,
 * no memory traffic in the loop) `iters` iterations, best of 3 after one warm-up, on a private
 * stream; synchronous.  kind:
 *   0 scalar FFMA              (16 lane-FMAs per thread-iteration)
 *   1 FFMA2 (fma.rn.f32x2)     (16 lane-FMAs)
 *   2 the a5 inner-loop body, packed FFMA2 form, operands in registers (64 lane-FMAs)
 *   3 the same body as scalar FFMA (64 lane-FMAs)
 *   4 MUFU.EX2                 (8 lane-ops)
 * *lane_ops_per_s receives thread-level operations per second summed over the GPU (one FMA = one
 * operation); ms_out (may be NULL) the kernel time. */
int nqs_microbench(int32_t kind, int32_t iters, double *lane_ops_per_s, float *ms_out);

/* Number of kernels this library has launched in this process so far (all entry points, all streams). */
int nqs_launch_count(int64_t *out);

/* Thread-local message of the last error on this thread ("" if none). */
const char *nqs_last_error(void);

/* Drops the internal cache of compiled Hamiltonians and trims the library's scratch pools (device memory
 * returned to the driver once the work that used it has finished). */
int nqs_release(void);

/* "major.minor.patch sm_100a" */
const char *nqs_version(void);

#ifdef __cplusplus
}
#endif
#endif /* NQS_B200_H */
