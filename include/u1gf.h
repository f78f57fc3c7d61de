/* u1gf.h -- C-ABI boundary of libu1gf.so: B200-native (sm_100a) lattice-Landau-gauge relaxation and
 * Gribov-copy counting for compact U(1), the hot path of Mehta & Schroeck, "Enumerating Copies in the
 * First Gribov Region on the Lattice in up to four Dimensions" (arXiv:1403.0555).
 *
 * Citations are PAPER.md:L<line> (+ section / equation); R<k> are the readings listed in DESIGN.md section 3.
 *
 * Conventions common to every call
 *   - plain C, no exceptions cross the boundary.  Return value 0 = success, negative = error code below;
 *     u1gf_last_error() then returns a thread-local, NUL-terminated description valid until the next call.
 *   - "dev" pointers are CUDA device pointers owned by the CALLER (e.g. torch tensors); "host" pointers are
 *     ordinary host memory owned by the caller.  Only the orbit handle is library-owned.
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Device-pointer calls
 *     are asynchronous on that stream and never synchronise the device; `*_host` calls copy results back and
 *     return after the stream has drained.
 *   - there is NO CPU fallback: without a usable sm_100 device every compute call returns U1GF_ENODEV.
 *   - site index i = x0 + N0*(x1 + N1*(x2 + N2*x3)), periodic in every direction;
 *     link angle theta_{i,mu} at [i*d + mu]; complex numbers are interleaved (re, im) doubles.
 *   - gauge-transformed link U^g_{i,mu} = g_i U_{i,mu} conj(g_{i+mu}) (Eq. 5 convention, R1); the functional
 *     F[g] = sum_{i,mu} Re U^g_{i,mu} is MAXIMISED (Eq. 3, x_paper = 1 - F/(dV)).
 *   - per start, results are a pure function of (orbit, seed, start index, omega, eps, max_sweeps, check_every):
 *     no floating-point atomics, fixed reduction trees; independent of launch configuration and of which other
 *     starts run beside it.
 */
#ifndef U1GF_H
#define U1GF_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define U1GF_OK 0
#define U1GF_EINVAL (-1) /* bad argument (message says which) */
#define U1GF_ENODEV (-2) /* no CUDA device of compute capability 10.x */
#define U1GF_ECUDA (-3)  /* a CUDA runtime call failed (message carries cudaGetErrorString) */
#define U1GF_ENOMEM (-4) /* host or device allocation failed / workspace too small */

typedef struct u1gf_orbit u1gf_orbit; /* opaque, library-owned */

const char* u1gf_last_error(void);

/* Version of this ABI (2 = round 2: ensembles, pipeline, region bit 2; 3 = round 3: u1gf_paper_count_static and the
 * ensemble read-outs added, nothing removed or changed). */
int u1gf_abi_version(void);

/* ---------------------------------------------------------------------------------------------------------
 * a1  Orbit setup.  One gauge orbit = one link field on a periodic lattice.
 *   d           number of dimensions, 1..4 (the paper uses 2..4; d = 1 is accepted for the ring closed form)
 *   extents     host [d], each >= 2, V = prod extents <= 8192
 *   theta_host  host [V*d] link angles in radians, any range (only cos/sin are used)
 *   out         receives the handle.  U = (cos theta, sin theta) is evaluated on the host with libm and copied
 *               to the current CUDA device together with neighbour / update-phase tables.  Synchronous.
 * Update order (R3): sites are grouped into phases (parity, level) such that a phase contains no two
 * neighbouring sites; for all-even extents these are the two checkerboard colours of PAPER.md:L99.
 * ------------------------------------------------------------------------------------------------------- */
int u1gf_create_orbit(int d, const int32_t* extents, const double* theta_host, u1gf_orbit** out);
int u1gf_destroy_orbit(u1gf_orbit* o);
/* Volume V and dimension d of a handle (0 on NULL). */
int32_t u1gf_orbit_volume(const u1gf_orbit* o);
int32_t u1gf_orbit_dim(const u1gf_orbit* o);

/* ---------------------------------------------------------------------------------------------------------
 * a2-a6  Relaxation of a batch of random starts (Eq. 4-5; R2, R5, R6).
 * Start with index s: g_i = exp(i*pi*(2u-1)), u the 53-bit uniform of Philox4x32-10 with key (seed lo, seed hi)
 * and counter (i, s lo, s hi, 0) (PAPER.md:L121 names Philox).  Sweep: for each phase in order, every site of
 * the phase gets w_i = sum_mu [conj(U_{i,mu}) g_{i+mu} + U_{i-mu,mu} g_{i-mu}] (= conj K_i, Eq. 5),
 * g_i <- normalise((1-omega) g_i + omega w_i/|w_i|) (over-relaxation R2; omega = 1 is the paper's
 * algorithm); a site with |w_i|^2 < 1e-280 is left unchanged (R6).  After sweep t with t % check_every == 0 the
 * gauge precision vartheta = (1/V) sum_i Delta_i^2, Delta_i = Im(g_i conj w_i), is tested against eps (R5).
 *   seed, first_start, n_starts   start k uses index start_ids[k] if start_ids != NULL else first_start + k
 *   start_ids   dev [n_starts] or NULL
 *   omega       in [1, 2);  eps > 0;  max_sweeps >= 1;  check_every >= 1
 *   F_norm      dev [n]    F/(dV) of the final field
 *   sweeps      dev [n]    number of full sweeps performed
 *   status      dev [n]    bit0: max_sweeps reached without passing the test; bit1: an R6 skip occurred
 *   sig         dev [n*4]  canonical signature: g~_i = g_i conj(g_{V-1}) (angle at the last site (N,..,N) fixed to
 *                          zero); p_k = (1/V) sum_i (a_{k,i} Re g~_i + b_{k,i} Im g~_i), k = 0..3,
 *                          a, b in {+1,-1} from Philox key (0x51, 0) counter (i, k, 0, 1), bit 0 of words 0 / 1
 *   g_canon     dev [n*V*2] canonical fields g~, or NULL (16 GiB at 2^22 starts of 4^4: normally NULL, and only
 *               the representatives are re-relaxed with start_ids to obtain their fields)
 *   workspace   dev scratch of at least u1gf_relax_workspace_bytes(o, n_starts) bytes, 256-byte aligned; its
 *               contents are undefined afterwards.  Nothing is allocated inside the call.
 * Errors: EINVAL on NULL / out-of-range arguments, ENOMEM if workspace_bytes is too small, ECUDA on launch failure.
 * ------------------------------------------------------------------------------------------------------- */
size_t u1gf_relax_workspace_bytes(const u1gf_orbit* o, uint64_t n_starts);
int u1gf_relax_batch(const u1gf_orbit* o, uint64_t seed, uint64_t first_start, uint64_t n_starts,
                     const uint64_t* start_ids, double omega, double eps, int32_t max_sweeps, int32_t check_every,
                     double* F_norm, int32_t* sweeps, uint8_t* status, double* sig, double* g_canon,
                     void* workspace, size_t workspace_bytes, void* cuda_stream);
/* Same computation with HOST result arrays (and host start_ids or NULL): device buffers and workspace are
 * allocated inside, results copied back, stream drained before returning.  Any output pointer may be NULL. */
int u1gf_relax_batch_host(const u1gf_orbit* o, uint64_t seed, uint64_t first_start, uint64_t n_starts,
                          const uint64_t* start_ids_host, double omega, double eps, int32_t max_sweeps,
                          int32_t check_every, double* F_norm_host, int32_t* sweeps_host, uint8_t* status_host,
                          double* sig_host, double* g_canon_host);

/* Kernel selection for u1gf_relax_batch on this handle: 0 = automatic (specialised resident kernel when one
 * exists for the extents; the TMA-staged streamed kernel for 6^4 and 8^4; the streamed lane-per-start kernel for other
 * all-even lattices of 1024 sites and more and its phased variant for lattices with an odd extent of 64 sites and more;
 * else the generic one), 1 = force the generic kernel, 2 = force the streamed (plain loads) / phased lane-per-start
 * kernel, 3 = force the TMA-staged streamed kernel (6^4, 8^4 only; other extents fall back to the generic kernel).
 * Results per start are the same copies either way; kernels may differ in the last bits of F and, rarely, by a
 * sweep (R14). */
int u1gf_set_kernel(u1gf_orbit* o, int32_t which);
/* Name of the kernel u1gf_relax_batch will use for this handle (static string). */
const char* u1gf_kernel_name(const u1gf_orbit* o);

/* ---------------------------------------------------------------------------------------------------------
 * a7  First-Gribov-region test (R9).  For each configuration g (unit complex per site):
 * c_{i,mu} = Re(g_i U_{i,mu} conj g_{i+mu}); Faddeev-Popov operator = Hessian of -F,
 * (M v)_i = sum_mu [c_{i,mu}(v_i - v_{i+mu}) + c_{i-mu,mu}(v_i - v_{i-mu})]; lambda_1 = smallest eigenvalue of M on
 * the orthogonal complement of the constant vector (the global gauge zero mode), computed by a
 * batched matrix-free Lanczos iteration (one CTA per configuration).
 *   g           dev [.*V*2] configurations
 *   cfg_index   dev [n_cfg] int64 or NULL: configuration k is g[cfg_index[k]] (NULL: g[k]).  With it the fields of ALL
 *               starts, written once by u1gf_relax_batch(g_canon), serve the representatives without a gather or a
 *               second relaxation (the choice when most starts are their own copy: hot 4^4 and larger)
 *   tol_fp      region bits 0-1 = 1 if lambda_1 > tol_fp (inside), 2 if |lambda_1| <= tol_fp (marginal, "semi"definite),
 *               0 if lambda_1 < -tol_fp (outside); region bit 2 (value 4) is set when the iteration reached its cap of
 *               min(V-1, 512) steps with the Ritz residual bound still above 1e-10 (R16): lambda1 is then only an upper
 *               bound of the eigenvalue, and an "inside" verdict is not proven.  Lattices with V-1 <= 512 never get bit 2: a run
 *               that reaches k = V-1 has used up the whole space orthogonal to the constant mode and is taken as exact.
 *               That holds in exact arithmetic only (the iteration does not reorthogonalise); on such lattices lambda1
 *               has been within 1e-8 of the dense eigenvalue in every test, but the verdict is not proven by a bound
 *   lambda1     dev [n_cfg];  region dev [n_cfg];  n_in_region dev [1] = number of configurations with (region & 3) != 0
 *   lanczos_steps  dev [n_cfg] int32 or NULL: Lanczos steps taken per configuration
 * A converged relaxation can stop at a saddle it is still leaving (the stop rule tests the gradient only):
 * such copies come out with region 0 and are genuine -- DESIGN.md section 3, R17.
 * ------------------------------------------------------------------------------------------------------- */
int u1gf_check_fp(const u1gf_orbit* o, uint64_t n_cfg, const double* g, const int64_t* cfg_index, double tol_fp,
                  double* lambda1, uint8_t* region, int64_t* n_in_region, int32_t* lanczos_steps, void* cuda_stream);
int u1gf_check_fp_host(const u1gf_orbit* o, uint64_t n_cfg, const double* g_host, double tol_fp,
                       double* lambda1_host, uint8_t* region_host, int64_t* n_in_region_host);

/* ---------------------------------------------------------------------------------------------------------
 * a8  De-duplication and counting (PAPER.md:L129-135 sort the functional values and count distinct ones; L149
 * counts as a function of the number of samples; L167 histogram; R7, R8, R15).  Records with status bit0 set get
 * copy_id = -1.  The others are sorted by F/(dV) (ties by position), cut into maximal runs with adjacent gaps
 * <= tol_F; inside a run the unassigned record with the smallest position becomes a leader and takes every
 * unassigned record whose signature agrees within tol_sig (max norm), repeated until the run is used up.
 * Copies are numbered in order of first discovery (increasing leader position).
 *   F_norm dev [n], sig dev [n*4], status dev [n]
 *   copy_id      dev [n] int32
 *   n_distinct   dev [1] int64
 *   rep          dev [n] int64: rep[c] = position of the leader of copy c, c < n_distinct (rest undefined)
 *   multiplicity dev [n] int64: members of copy c
 *   hist         dev [nbins] int64 or NULL: histogram over nbins equal bins on [0,1] of F_norm[rep[c]] weighted by
 *                multiplicity[c]: bin b holds F/(dV) in [b/nbins, (b+1)/nbins), values outside [0,1] go to the end bins.
 *                The paper histograms the minimum value x = 1 - F/(dV) with bin width 1e-4: its bin j
 *                is bin nbins-1-j here (mirror image; the half-open ends swap sides)
 *   workspace    dev scratch >= u1gf_count_workspace_bytes(n), 256-byte aligned
 * ------------------------------------------------------------------------------------------------------- */
size_t u1gf_count_workspace_bytes(uint64_t n);
int u1gf_count_copies(uint64_t n, const double* F_norm, const double* sig, const uint8_t* status, double tol_F,
                      double tol_sig, int32_t* copy_id, int64_t* n_distinct, int64_t* rep, int64_t* multiplicity,
                      int64_t* hist, int32_t nbins, void* workspace, size_t workspace_bytes, void* cuda_stream);
int u1gf_count_copies_host(uint64_t n, const double* F_norm_host, const double* sig_host,
                           const uint8_t* status_host, double tol_F, double tol_sig, int32_t* copy_id_host,
                           int64_t* n_distinct_host, int64_t* rep_host, int64_t* multiplicity_host,
                           int64_t* hist_host, int32_t nbins);

/* ---------------------------------------------------------------------------------------------------------
 * Read-outs of the sorted samples.
 *
 * u1gf_discovery_curve: the paper plots the number of distinct minima found as a function of the number of samples
 * (Figs. 1-3).  With the copies numbered in order of first discovery (u1gf_count_copies),
 *   curve[k] = number of copies c < n_distinct whose leader position rep[c] is < 2^k,   k = 0 .. n_levels-1
 * i.e. the number of distinct copies among the first 2^k samples.  rep dev [n_distinct] int64 (as written by
 * u1gf_count_copies), curve dev [n_levels] int64, 1 <= n_levels <= 65.
 *
 * u1gf_paper_count: the paper's own count: the number of distinct integers
 * X = floor((1 - F_norm) * scale), scale = 1e8 in the paper, among the records with status bit0 clear.  It is
 * reported beside n_distinct of u1gf_count_copies (R7: such keys can merge distinct copies and split a copy that
 * straddles a key boundary).  F_norm dev [n], status dev [n], n_keys dev [1] int64, workspace dev scratch >=
 * u1gf_paper_count_workspace_bytes(n), 256-byte aligned.
 * Both calls are asynchronous on the stream, allocate nothing, and return U1GF_EINVAL on bad arguments.
 * ------------------------------------------------------------------------------------------------------- */
int u1gf_discovery_curve(uint64_t n_distinct, const int64_t* rep, int32_t n_levels, int64_t* curve, void* cuda_stream);
size_t u1gf_paper_count_workspace_bytes(uint64_t n);
int u1gf_paper_count(uint64_t n, const double* F_norm, const uint8_t* status, double scale, int64_t* n_keys,
                     void* workspace, size_t workspace_bytes, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------------------
 * u1gf_paper_count_static: u1gf_paper_count for callers that have no way to obtain device memory.
 *
 * Every other device-pointer call of this header wants a workspace from the caller, and the *_host calls allocate
 * one inside.  Neither works for code that was handed its input and output buffers by a host application and nothing
 * else: a plug-in inside a simulation whose driver carved up the whole of HBM at start-up and forbids (or would
 * fail) a later cudaMalloc; a measurement step inside a latency-critical loop, where cudaMalloc / cudaFree would
 * stall every stream of the device while they run; an embedding that may issue stream work only and has no
 * allocator of its own to ask.  For those, the scratch of this one call is built into the library: a fixed
 * 32 MiB array in device memory (`static __device__`, 256-byte aligned) that belongs to the library's device code.
 * Each GPU onto which that code is loaded holds those 32 MiB until the process exits, whether the call is ever made
 * or not.
 *
 *   n        number of records, 0 <= n <= U1GF_PAPER_COUNT_STATIC_MAX_N (2^20, one "mebisample" of PAPER.md:L131);
 *            a larger n is refused with U1GF_EINVAL and a message naming the limit -- use u1gf_paper_count then
 *   F_norm   dev [n], status dev [n], scale, n_keys dev [1] int64: exactly as u1gf_paper_count; the result is the same
 *            integer (same kernels, same sort, only the scratch differs).  Inputs and output stay the caller's.
 *   Set-up   the FIRST call on each device looks up where the array lives on that device (cudaGetSymbolAddress,
 *            return code checked, address kept per device ordinal).  That look-up can make the runtime load this
 *            library's device code onto the GPU, so make the first call on a device early -- with that device
 *            current, and before any stream capture is begun; n = 0 is enough (it does the set-up, zeroes n_keys and
 *            launches nothing else).  Later calls only enqueue a memset, two kernels and the radix sort on the stream.
 *   Allocation  none: no cudaMalloc, cudaFree or allocating library routine anywhere on this path, first call included
 *            (the sort gets its temporary storage from the array).
 *   Sharing  there is ONE array per GPU and every call uses it.  Calls on the same stream are ordered and safe.  Two
 *            calls that can overlap on the GPU (different streams without an event between them, or several host
 *            threads on different streams) race on it and return garbage counts -- serialise them.  The array keeps
 *            whatever the previous call left; the call relies on none of it (both key arrays are rewritten for all n
 *            records and the sort clears its own counters), and n_keys is zeroed on the stream first.
 * Errors: U1GF_EINVAL (NULL pointer, scale <= 0, n over the limit, device ordinal >= 64), U1GF_ENODEV, U1GF_ECUDA;
 *         U1GF_ENOMEM only if the sort asked for more temporary storage than the array leaves (not on sm_100a).
 * Asynchronous on the stream like the other device-pointer calls.
 * ------------------------------------------------------------------------------------------------------- */
#define U1GF_PAPER_COUNT_STATIC_MAX_N 1048576
int u1gf_paper_count_static(uint64_t n, const double* F_norm, const uint8_t* status, double scale, int64_t* n_keys,
                            void* cuda_stream);

/* ---------------------------------------------------------------------------------------------------------
 * The whole hot path in one call with HOST result buffers (what an application that keeps nothing on the device
 * calls, and what bench.py's `e2e` times): u1gf_relax_batch on all starts -> u1gf_count_copies -> the fields of the
 * representatives -> u1gf_check_fp.  Where those fields come from: normally the representatives are relaxed once more
 * with g_canon written (in chunks of 1 GiB of fields).  The handle remembers whether its last call found
 * n_distinct > n_starts/4 (a hot orbit: most starts are their own copy); if so, and n_starts*V*16 bytes are at most a
 * quarter of the device memory, the next call writes the fields of ALL starts in the first pass and hands
 * u1gf_check_fp cfg_index = rep, so nothing is relaxed twice.  Outputs are identical either way.
 * Intermediates never leave the device; device scratch comes from a
 * grow-only per-thread allocation that is kept between calls (u1gf_release_host_scratch frees it; the other *_host
 * calls use the same scratch).
 *   per start (host [n_starts] or NULL): F_norm, sweeps, status, sig [n*4], copy_id
 *   per copy  (host arrays of copy_capacity entries or NULL): rep (position of the leader), multiplicity, F_rep
 *             (F/(dV) of the leader), lambda1, region (as u1gf_check_fp); U1GF_ENOMEM if n_distinct > copy_capacity
 *             and any per-copy array is given
 *   n_distinct [1], n_in_region [1] (host, required); hist host [nbins] or NULL
 * ------------------------------------------------------------------------------------------------------- */
int u1gf_pipeline_host(const u1gf_orbit* o, uint64_t seed, uint64_t first_start, uint64_t n_starts, double omega,
                       double eps, int32_t max_sweeps, int32_t check_every, double tol_F, double tol_sig, double tol_fp,
                       int32_t nbins, double* F_norm_host, int32_t* sweeps_host, uint8_t* status_host, double* sig_host,
                       int32_t* copy_id_host, int64_t copy_capacity, int64_t* n_distinct_host, int64_t* rep_host,
                       int64_t* multiplicity_host, double* F_rep_host, double* lambda1_host, uint8_t* region_host,
                       int64_t* n_in_region_host, int64_t* hist_host);
int u1gf_release_host_scratch(void);

/* ---------------------------------------------------------------------------------------------------------
 * Ensembles: many gauge orbits of ONE lattice shape relaxed in ONE kernel launch.  The paper's
 * workload is an ensemble -- 100 orbits x 4 mebisamples per lattice size (Tab. I, Tab. III),
 * one lattice per thread block, grid over the samples (L121).
 *   u1gf_create_ensemble   theta_host [n_orbits][V*d] link angles, seeds_host [n_orbits] start seed of each orbit
 *                          (starts of orbit o are those of u1gf_relax_batch with seed seeds[o]).  Any lattice
 *                          u1gf_create_orbit accepts: shapes with a resident kernel (4x4, 8x8, 10x10, 4^3, 6^3, 2^4, 4^4)
 *                          run on it; every other shape (2x2, 6x6, 2^3, 8^3 of Tab. I / III, odd extents, ...) runs on
 *                          the generic kernel, one thread block per start with the grid over the starts of all orbits
 *                          (the paper's own mapping).  Synchronous.
 *   u1gf_ensemble_orbit    member k as an ordinary orbit handle (owned by the ensemble): for u1gf_check_fp and for
 *                          re-relaxing an orbit's representatives with u1gf_relax_batch(start_ids, g_canon)
 *   u1gf_relax_ensemble    every orbit runs the starts first_start + [0, n_starts_per_orbit); result k of orbit o is at
 *                          o * n_starts_per_orbit + k of F_norm / sweeps / status / sig [.*4] (device arrays of
 *                          n_orbits * n_starts_per_orbit entries).  Per start the results are those of
 *                          u1gf_relax_batch on the member orbit, with one exception on the shapes with a resident
 *                          kernel: a start that meets R6 (|w|^2 < 1e-280) comes back with status 3 instead of being
 *                          relaxed with the skip rule (the generic kernel applies the skip rule as always).
 *   u1gf_count_copies_ensemble   u1gf_count_copies per orbit on those arrays: copy ids, rep (positions) and
 *                          multiplicity are local to the orbit and stored at o * n_per_orbit; n_distinct dev
 *                          [n_orbits]; hist dev [n_orbits * nbins] or NULL; workspace >= u1gf_count_workspace_bytes(n_per_orbit):
 *                          one u1gf_count_copies after the other on the orbits' slices.  With a workspace of at least
 *                          u1gf_count_ensemble_onepass_workspace_bytes(n_orbits, n_per_orbit) bytes (0 = not available:
 *                          one orbit, or n_orbits * n_per_orbit >= 2^31) all orbits are de-duplicated in ONE pass instead --
 *                          records sorted by F, then stably by orbit index, runs cut at orbit boundaries -- with the same
 *                          outputs bit for bit and a fixed number of launches whatever n_orbits is
 * ------------------------------------------------------------------------------------------------------- */
typedef struct u1gf_ensemble u1gf_ensemble; /* opaque, library-owned */
int u1gf_create_ensemble(int d, const int32_t* extents, int32_t n_orbits, const double* theta_host,
                         const uint64_t* seeds_host, u1gf_ensemble** out);
int u1gf_destroy_ensemble(u1gf_ensemble* e);
int32_t u1gf_ensemble_size(const u1gf_ensemble* e);
const u1gf_orbit* u1gf_ensemble_orbit(const u1gf_ensemble* e, int32_t k);
size_t u1gf_relax_ensemble_workspace_bytes(const u1gf_ensemble* e, uint64_t n_starts_per_orbit);
int u1gf_relax_ensemble(const u1gf_ensemble* e, uint64_t first_start, uint64_t n_starts_per_orbit, double omega,
                        double eps, int32_t max_sweeps, int32_t check_every, double* F_norm, int32_t* sweeps,
                        uint8_t* status, double* sig, void* workspace, size_t workspace_bytes, void* cuda_stream);
size_t u1gf_count_ensemble_workspace_bytes(uint64_t n_per_orbit);
size_t u1gf_count_ensemble_onepass_workspace_bytes(int32_t n_orbits, uint64_t n_per_orbit);
int u1gf_count_copies_ensemble(int32_t n_orbits, uint64_t n_per_orbit, const double* F_norm, const double* sig,
                               const uint8_t* status, double tol_F, double tol_sig, int32_t* copy_id,
                               int64_t* n_distinct, int64_t* rep, int64_t* multiplicity, int64_t* hist, int32_t nbins,
                               void* workspace, size_t workspace_bytes, void* cuda_stream);

/* ---------------------------------------------------------------------------------------------------------
 * Ensemble read-outs: the quantities the paper tabulates and plots from an ensemble of orbits.
 * Inputs are the device arrays of u1gf_relax_ensemble / u1gf_count_copies_ensemble: F_norm [n_orbits*n_per_orbit],
 * rep / multiplicity [n_orbits*n_per_orbit] (entries c < n_distinct[o] of orbit o at o*n_per_orbit + c, rep local to the
 * orbit), n_distinct [n_orbits].  The paper's value of a minimum is x = 1 - F/(dV) (Eq. 3); its
 * "global minimum" of an orbit is the smallest x found there, x_g = 1 - max_c F_norm[rep[c]] (L169: "the smallest minimum
 * we find on each orbit").  All three calls are asynchronous on the stream, need no workspace and allocate nothing.
 *
 * u1gf_ensemble_stats     best_x dev [n_orbits]: x_g per orbit (NaN for an orbit without a converged start).
 *                         stats dev [8]: [0],[1] average and standard deviation over the orbits of n_distinct (Tab. I,
 *                         PAPER.md:L175-183); [2],[3] of x_g (Tab. III; orbits with NaN left out); [4],[5] of
 *                         n_in_region (dev [n_orbits] int64: copies inside the first Gribov region per orbit, L9/L50; NULL:
 *                         NaN); [6] orbits that entered [2],[3]; [7] n_orbits.  Standard deviation = sqrt(sum (v-mean)^2 /
 *                         (m-1)), 0 for m = 1 (reading R18: the paper prints "avg +- std" without a formula); sums run in
 *                         orbit order.
 * u1gf_relative_deviation_hist   (x_i - x_g)/x_g of every converged sample (Fig. 8): copy c of orbit o
 *                         puts multiplicity[c] samples into bin floor(dev / (dev_max/nbins)) of nbins equal bins on
 *                         [0, dev_max), larger values into the last bin.  counts dev [n_orbits*nbins] int64 per orbit;
 *                         n_converged dev [n_orbits] int64 = samples binned; avg dev [nbins] = the orbit average of
 *                         counts[o][b]/n_converged[o] ("subsequently, the data has been averaged over all orbits", L207)
 *                         over the n_orbits_used dev [1] orbits that have samples and x_g > 0 (the trivial orbit, x_g = 0,
 *                         has no relative deviation).  best_x: as written by u1gf_ensemble_stats.
 * u1gf_hist_ratio         ratio[b] = hist_big[b] / hist_small[b] for two histograms (int64 [nbins], e.g. `hist` of
 *                         u1gf_count_copies) of the same orbits from a larger and a smaller number of samples (PAPER.md:L167,
 *                         Fig. 5: 256 against 4 mebisamples in bins of 1e-4): +inf where only the larger run has entries,
 *                         NaN where neither has; n_only dev [2] int64 = number of bins only the larger / only the smaller
 *                         run fills (L167: "only very high-lying bins of the four mebisample run are empty while the
 *                         corresponding bins of the 256 mebisample run have entries").
 * Errors: U1GF_EINVAL on NULL arrays or sizes < 1, U1GF_ENODEV, U1GF_ECUDA.
 * ------------------------------------------------------------------------------------------------------- */
int u1gf_ensemble_stats(int32_t n_orbits, uint64_t n_per_orbit, const double* F_norm, const int64_t* rep,
                        const int64_t* n_distinct, const int64_t* n_in_region, double* best_x, double* stats,
                        void* cuda_stream);
int u1gf_relative_deviation_hist(int32_t n_orbits, uint64_t n_per_orbit, const double* F_norm, const int64_t* rep,
                                 const int64_t* multiplicity, const int64_t* n_distinct, const double* best_x, double dev_max,
                                 int32_t nbins, int64_t* counts, int64_t* n_converged, double* avg, int64_t* n_orbits_used,
                                 void* cuda_stream);
int u1gf_hist_ratio(int32_t nbins, const int64_t* hist_small, const int64_t* hist_big, double* ratio, int64_t* n_only,
                    void* cuda_stream);

/* ---------------------------------------------------------------------------------------------------------
 * Merging the copy tables of several start ranges (the paper runs 4 GPUs on independent samples,
 * PAPER.md:L121).  Each range was de-duplicated on its own; entry e of the concatenated tables is one copy of one
 * range: F_rep[e] = F/(dV) of its leader, sig_rep[e*4..], first_start[e] = GLOBAL start index of its leader,
 * multiplicity[e].  The entries are ordered by first_start (the discovery order of the whole job, L149) and clustered by
 * the copy identity of u1gf_count_copies (R7).  Outputs: merged_id[e] = merged copy of entry e, merged copies numbered
 * by increasing first discovery; n_merged dev [1]; merged_first_start / merged_multiplicity dev [m], the first n_merged
 * entries valid.  The global copy id of a start is merged_id[offset of its range + its local copy id].
 * Caveat: only the LEADERS of the ranges are clustered.  u1gf_count_copies on the undivided batch chains its F-runs
 * through every member (adjacent gaps <= tol_F); two leaders of one copy whose F differ by more than tol_F, bridged
 * there by other members, fall into different runs here and stay two merged copies.  The result equals the one-pass
 * count whenever the F spread inside a copy is below tol_F -- at the default tol_F = 1e-10 against a spread of about
 * 1e-13 after convergence to eps = 1e-13 that is the normal case; with a loose eps or a tight tol_F it is not guaranteed.
 * All arrays dev, int64 unless stated; workspace >= u1gf_merge_workspace_bytes(m), 256-byte aligned; asynchronous.
 * ------------------------------------------------------------------------------------------------------- */
size_t u1gf_merge_workspace_bytes(uint64_t m);
int u1gf_merge_copy_tables(uint64_t m, const double* F_rep, const double* sig_rep, const int64_t* first_start,
                           const int64_t* multiplicity, double tol_F, double tol_sig, int32_t* merged_id,
                           int64_t* n_merged, int64_t* merged_first_start, int64_t* merged_multiplicity,
                           void* workspace, size_t workspace_bytes, void* cuda_stream);


#ifdef __cplusplus
}
#endif
#endif /* U1GF_H */
