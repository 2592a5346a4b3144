/*
 * mfh.h -- C ABI of the B200-native block-procedural matrix-free Hamiltonian-vector product.
 *
 * phi = H psi for a dense D x D Hermitian H that is never materialised: for every block pair
 * (n,m) the block H^[n,m] is generated on the fly from a counter-based seed or streamed from an
 * HBM-resident cache, applied to psi^[m] and accumulated into phi^[n].
 *   PAPER.md = /root/reference/PAPER.md (arxiv/paper_2606_31598), cited "P:<line>".
 *   Block product                     P:107-116 Eq. 4-5;  P:143-147 Eq. 7
 *   apply_H_block(n,m,psi^[m])        P:135-141 Eq. 6
 *   Sources: seeded / fused action    P:153-157 Eq. 8;  P:171-175 Eq. 11
 *   Modes: full / partial cache       P:177-183;  P:431-446 Eq. 27
 *   Multi-vector Y = A X (R vectors)  P:212-230 Eq. 12-13
 *   Planner (analytic, measured)      P:258-296 Eq. 14-20;  P:298-360 Eq. 21-23
 *   Chebyshev propagator              P:705-721 Eq. 41-44
 * The entry rule, Philox4x32-10 + Box-Muller, the workloads and the tolerances come from
 * /root/repo/BASELINE.json; readings of silent points are listed in DESIGN.md.
 *
 * Conventions
 *   - Plain C, no torch types.  "dev" pointers are CUDA device pointers on the current device,
 *     "host" pointers are ordinary host memory.  `stream` is a cudaStream_t passed as void*
 *     (NULL = the legacy default stream).
 *   - Complex numbers are interleaved (re, im); MFH_C128 = 2 x double, MFH_C64 = 2 x float.
 *   - One vector: length D.  k vectors: row-major [D][k] (the k values of a row are contiguous).
 *   - All vectors are caller-owned and 16-byte aligned; phi must not alias psi.  The cache,
 *     partial-sum workspace and the Chebyshev / Lanczos scratch are library-owned (all allocated in
 *     mfh_plan, freed in mfh_destroy): after mfh_plan no entry point allocates device memory, so
 *     mfh_apply and the chained drivers can be captured in a CUDA graph without a warm-up call.
 *   - Devices: a handle lives on the CUDA device that was current in mfh_plan; every later call on it
 *     must be made with that device current (MFH_ERR_BAD_STATE otherwise).  One process per GPU or
 *     any number of devices per process both work: per-device kernel attributes are kept per handle.
 *   - Every function returns an int status (MFH_OK = 0); mfh_last_error() gives the message.
 *   - There is no CPU fallback: every compute entry point needs a CUDA device and fails with
 *     MFH_ERR_CUDA otherwise.
 */
#ifndef MFH_H
#define MFH_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define MFH_API __attribute__((visibility("default")))
#else
#define MFH_API
#endif

typedef struct mfh_handle_s* mfh_handle; /* opaque; library-owned until mfh_destroy */

enum { MFH_OK = 0, MFH_ERR_INVALID_ARG = 1, MFH_ERR_BAD_STATE = 2, MFH_ERR_OUT_OF_MEMORY = 3,
       MFH_ERR_CUDA = 4, MFH_ERR_NOT_CONVERGED = 5, MFH_ERR_UNSUPPORTED = 6 };
enum { MFH_C128 = 0, MFH_C64 = 1 };
enum { MFH_SRC_GUE = 0,           /* H = lambda * V(seed)                          configs 1,2,4,5 */
       MFH_SRC_DIAG_PLUS_GUE = 1, /* H_v = diag(h0(seed_h0)) + lambda_v * V(seed)  config 3        */
       MFH_SRC_ANALYTIC = 2,      /* H = lambda * F(theta), entries from a formula (Eq. 9): see
                                     mfh_set_source_params; seeds are ignored                       */
       MFH_SRC_EXTERNAL = 3       /* H = lambda * (blocks supplied by the caller, Eq. 10): see
                                     mfh_set_block; seeds are ignored                               */ };
enum { MFH_MODE_AUTO = 0, MFH_MODE_PROCEDURAL = 1, MFH_MODE_PARTIAL = 2, MFH_MODE_FULL = 3,
       /* Hermitian (canonical-pair) cache, Eq. 27: block (n,m), n <= m, is stored once
        * and used for phi^[n] += C psi^[m] and phi^[m] += C^dagger psi^[n]; as many pairs as the budget
        * allows (nearest block diagonals first), the rest is generated.  Half the memory of FULL.  One vector: every
        * loaded entry is used for both positions (half the bytes per apply as well).  k vectors (complex64, B % 128
        * == 0): a stored off-diagonal block is read ONCE per apply and serves both positions on the tensor cores (row
        * side from TMEM, column side with the block as shared-memory operand; half the bytes of FULL) -- when the
        * extra partial slots do not fit the budget, the mirrored position is served by a second, transposed read
        * instead (same bytes as FULL).  complex128 k-vector plans do not support the pair
        * cache. */
       MFH_MODE_PAIRS = 4 };

#define MFH_MAX_K 16       /* largest number of simultaneous vectors */
#define MFH_MIN_B 32       /* block size must be a multiple of this and divide D */
#define MFH_MAX_B 4096     /* largest block size (shared-memory column accumulators) */

/* Create a Hamiltonian description (host only; no device work, no allocation on the device).
 *   D        Hilbert-space dimension, 32 <= D <= 2^31, multiple of 32.
 *   B        block size b; multiple of 32 dividing D, <= MFH_MAX_B; 0 = planner picks.
 *   seed     64-bit seed of the GUE matrix V: entry (i,j), i<j, is (g1 + i g2)/sqrt(2D) with
 *            g1,g2 Box-Muller normals from Philox4x32-10(key=seed, ctr=(min(i,j),max(i,j),0,0));
 *            i>j is the conjugate; i==j is g1/sqrt(D), real (BASELINE.json configs[0]).
 *   lambda   coupling used when mfh_apply gets lambdas_host == NULL (1.0 for a plain GUE).
 *   seed_h0  seed of the diagonal H0 (uniform in (-1,1)); ignored for MFH_SRC_GUE.
 * Errors: MFH_ERR_INVALID_ARG for any violated constraint or unknown enum. */
MFH_API int mfh_create(mfh_handle* out, int64_t D, int32_t B, uint64_t seed, int32_t source_kind,
                       double lambda, int32_t dtype, uint64_t seed_h0);

/* Parameters of the analytic source (MFH_SRC_ANALYTIC; Eq. 9 "H^[n,m]_ab = f(n, m, a, b; theta) ... computed
 * when needed"; R22).  The paper names no f; this library provides one dense six-parameter family in
 * GLOBAL indices (partition invariant): a chain with power-law hopping, a Peierls phase and a quasi-periodic potential,
 *     H_ij = -t e^{+i phi} / (j - i)^alpha  (i < j),   H_ij = conj(H_ji)  (i > j),   H_ii = W cos(2 pi beta i + delta).
 * theta_host: 6 doubles (t, alpha, phi, W, beta, delta), all finite, alpha >= 0.  Call before mfh_plan (drops a
 * committed plan).  Every mode works (the cache is filled from the formula; the fused kernels evaluate it in
 * registers); k-vector plans use the CUDA-core kernels.  Errors: INVALID_ARG (NULL, non-finite, alpha < 0, handle
 * not created with MFH_SRC_ANALYTIC). */
MFH_API int mfh_set_source_params(mfh_handle h, const double* theta_host);

/* Externally stored blocks (MFH_SRC_EXTERNAL; Eq. 10 "H^[n,m] = D[key(n,m)] ... the block is loaded or
 * reconstructed only for the currently active part of the matrix-vector product").  Host memory reaches this GPU at
 * ~40 GB/s against 7 TB/s from HBM, so an external block is loaded ONCE into the HBM cache and
 * streamed from there: plan the handle with MFH_MODE_FULL (any dense operator, Hermitian or not; all N_blk^2 blocks)
 * or MFH_MODE_PAIRS (Hermitian operators; only the canonical blocks n <= m, used for both positions), then hand every
 * stored block over once:
 *   block      B x B complex of the handle's dtype, row-major, interleaved (re, im); host (pageable or pinned) or device
 *   is_device  0: host pointer, 1: device pointer
 * The copy is enqueued on `stream`; a host block is consumed before the call returns.  mfh_apply fails with
 * MFH_ERR_BAD_STATE until every stored block of the plan (of this rank, for a partitioned handle) has been set; a
 * block may be set again at any time (time-dependent operators).  Errors: INVALID_ARG (not an external handle, block
 * outside the plan's stored set, e.g. n > m in pairs mode), BAD_STATE (no plan), CUDA. */
MFH_API int mfh_set_block(mfh_handle h, int32_t n, int32_t m, const void* block, int32_t is_device, void* stream);

/* Analytic planner only (Algorithm 1; adaptive block size P:409-429; cache budget
 * Eq. 27).  Pure host arithmetic: needs no GPU, touches no handle.  Enumerates
 * mode x B candidates, rejects those with M_tot > alpha * hbm_free_bytes (Eq. 18, alpha = 0.9)
 * and ranks the rest by modelled seconds per job.  Writes a JSON record (chosen plan +
 * all candidates) to json_out (NUL-terminated, truncated to json_cap).
 *   mode  MFH_MODE_AUTO or a forced mode;  B  0 = enumerate, else forced.
 * Errors: MFH_ERR_INVALID_ARG; MFH_ERR_OUT_OF_MEMORY when no candidate fits. */
MFH_API int mfh_plan_analytic(int64_t D, int32_t dtype, int32_t k, int32_t mode, int32_t B,
                              int64_t n_applies_hint, int64_t hbm_free_bytes, char* json_out,
                              size_t json_cap);

/* Node-level analytic planner (Algorithm 1 with the task waves of Eq. 19; "parameter-parallel",
 * "row-parallel", "hybrid"; worked example P:765-779).  Pure host arithmetic.  n_tasks independent outer-loop jobs
 * (coupling values, ...) of n_applies_per_task applications of n_op dense operators on k vectors are spread over
 * n_gpus GPUs in groups of p_row GPUs (p_row = 1: parameter-parallel, p_row = n_gpus: row-parallel, between:
 * hybrid); inside a group the operator is partitioned with `scheme` (MFH_PART_ROWS / MFH_PART_PAIRS, see
 * mfh_set_partition).  For every p_row dividing n_gpus: C = n_gpus / p_row groups, W = ceil(n_tasks / C) waves
 * (Eq. 19), the best memory-feasible single-GPU plan of one rank of the group (Eq. 14-18 with alpha = 0.9 on
 * hbm_free_bytes_per_gpu, each operator getting 1/n_op of it), seconds per application = n_op x (local apply
 * + exchange of D k B_c bytes), score = W x n_applies_per_task x seconds per application (Eq. 22 with the model
 * time).  The JSON lists every p_row (feasible or not) and the chosen one (smallest score; ties -> smaller p_row).
 * Errors: INVALID_ARG; OUT_OF_MEMORY when no p_row has a feasible plan. */
MFH_API int mfh_plan_node_analytic(int64_t D, int32_t dtype, int32_t k, int32_t n_op, int64_t n_tasks, int32_t n_gpus,
                                   int64_t hbm_free_bytes_per_gpu, int32_t mode, int32_t B, int32_t scheme,
                                   int64_t n_applies_per_task, char* json_out, size_t json_cap);

/* Neural surrogate of the planner (host only; Eq. 24-26, Algorithm 3).  A one-hidden-layer
 * network on componentwise normalised plan features predicts the logarithm of the measured apply time:
 *     z = (x - mu) / sigma,   f(x) = tanh(z W1 + b1) W2 + b2   (Eq. 24),   t_NN(p) = exp(f(x(p)))   (Eq. 25),
 * trained by minimising the log-time mean-squared error (Eq. 26) over the records (x(p), t_mv(p)) the measured
 * planner produces; it only RANKS candidates, a local measurement of the top K_NN stays the decision rule.
 *   theta  = [mu (F) | sigma (F) | W1 (F x H, row-major) | b1 (H) | W2 (H) | b2], mfh_surrogate_theta_size doubles
 *   X      = [n][F] features (paper_2606_31598_b200/surrogate.py builds x(p) from a plan record), t_seconds > 0
 * mfh_surrogate_fit: mu, sigma from the data (sigma = 1 for constant features), seeded initial weights, `epochs`
 * full-batch Adam steps of size lr; *final_loss = Eq. 26 at the end.  mfh_surrogate_loss_grad: Eq. 26 and its
 * gradient with respect to [W1 | b1 | W2 | b2] (test export; grad_out may be NULL).  Errors: INVALID_ARG. */
/* The feature vector x(p) of a candidate plan, MFH_SURROGATE_FEATURES doubles written to x_out:
 *   (log D, log R, log N_blk, log b, log N_task, p_row, W(p), 1_full, 1_partial, 1_procedural, 1_pairs [this build's
 *    fourth storage mode], log F_mv, M_op/M_free, M_work/M_free, M_tot/M_free, 1_complex64, log GPU memory, log SMs)
 * from the plan's own numbers (the fields of a candidate record of mfh_plan / mfh_plan_analytic).  mode is the
 * candidate's committed mode (not AUTO).  Errors: INVALID_ARG. */
#define MFH_SURROGATE_FEATURES 18
MFH_API int mfh_surrogate_features(int64_t D, int32_t dtype, int32_t k, int32_t mode, int32_t B, double flops_per_apply,
                                   double cache_bytes, double work_bytes, double free_bytes, int64_t n_task, int32_t p_row,
                                   int64_t waves, double gpu_bytes, int32_t sms, double* x_out);
MFH_API int64_t mfh_surrogate_theta_size(int32_t n_features, int32_t hidden);
MFH_API int mfh_surrogate_fit(const double* X, const double* t_seconds, int64_t n, int32_t n_features, int32_t hidden,
                              int32_t epochs, double lr, uint64_t seed, double* theta_out, double* final_loss);
MFH_API int mfh_surrogate_predict(const double* theta, int32_t n_features, int32_t hidden, const double* X, int64_t n,
                                  double* t_pred_seconds);
MFH_API int mfh_surrogate_loss_grad(const double* theta, int32_t n_features, int32_t hidden, const double* X,
                                    const double* t_seconds, int64_t n, double* loss_out, double* grad_out);

/* Plan and commit: choose mode and B (analytic; measure != 0 additionally times the best
 * candidates on the device, Algorithm 2, R_warm = 1, R_bench = 3, K_bench <= 8), allocate the
 * cache and the workspace and fill the cache with the generator (one-time cost).
 *   k                 number of simultaneous vectors later passed to mfh_apply (1..MFH_MAX_K).
 *   n_applies_hint    expected number of applies R_H (amortises the cache fill); <= 0 means 1.
 *   hbm_budget_bytes  memory the plan may use; 0 = alpha * currently free device memory.
 *   json_out          optional (may be NULL) plan record, as for mfh_plan_analytic.
 * Synchronises `stream` before returning.  May be called again to re-plan.
 * Errors: INVALID_ARG, OUT_OF_MEMORY (nothing fits / allocation failed), CUDA. */
MFH_API int mfh_plan(mfh_handle h, int32_t mode, int32_t k, int64_t n_applies_hint,
                     int64_t hbm_budget_bytes, int32_t measure, void* stream, char* json_out,
                     size_t json_cap);

/* Algorithm 3, hybrid mode ("ranks the memory-feasible candidates by t_NN(p) W(p) ... a local measurement
 * remains the final decision rule"): as mfh_plan(MFH_MODE_AUTO, measure = 1), but the feasible candidates are ordered by
 * the surrogate's prediction t_NN = exp(f_theta(x(p))) (theta from mfh_surrogate_fit on MFH_SURROGATE_FEATURES
 * features) and only the k_nn best are committed and timed; the best measured one (Eq. 23) stays committed.  Each
 * candidate's memory is released before the next is tried.  The JSON record carries "planner":"hybrid" and every
 * candidate's "surrogate_apply_s".  Errors as mfh_plan; INVALID_ARG for theta == NULL, hidden < 1, k_nn < 1. */
MFH_API int mfh_plan_hybrid(mfh_handle h, const double* theta, int32_t hidden, int32_t k, int64_t n_applies_hint,
                            int64_t hbm_budget_bytes, int32_t k_nn, void* stream, char* json_out, size_t json_cap);

/* phi = H psi for k vectors (Eq. 7; Eq. 12 for k > 1), asynchronous on `stream`, no host
 * synchronisation, no allocation.  k must equal the k given to mfh_plan.
 *   psi_dev, phi_dev  device, [D][k] complex of the handle's dtype.
 *   lambdas_host      k doubles (host) or NULL = the handle's lambda for every vector.
 *   Result: phi[:,v] = h0 (.) psi[:,v] (only MFH_SRC_DIAG_PLUS_GUE) + lambda_v * V psi[:,v].
 * Errors: BAD_STATE before mfh_plan; INVALID_ARG (NULL pointers, k mismatch); CUDA. */
MFH_API int mfh_apply(mfh_handle h, const void* psi_dev, void* phi_dev, int32_t k,
                      const double* lambdas_host, void* stream);

/* Measurement export: mfh_apply with CUDA events recorded on `stream` around each of its launches;
 * synchronises `stream`.  ms_out (host, 4 floats) = milliseconds of { cached streaming kernel,
 * fused generate-and-apply kernel, reduce/epilogue kernel, whole apply } (0 for a kernel the plan
 * does not launch).  bench.py uses it for the per-kernel roofline. */
MFH_API int mfh_apply_timed(mfh_handle h, const void* psi_dev, void* phi_dev, int32_t k,
                            const double* lambdas_host, void* stream, float* ms_out);

/* Measurement export, in-pass: arm per-launch timing for the next n_applies calls of mfh_apply on this handle.  Each
 * of them records CUDA events on its stream before, between and after its launches -- no synchronisation, so the
 * applies run back to back exactly as in an untimed loop and the per-kernel durations come from the SAME pass as the
 * loop's own time.  mfh_timing_end synchronises `stream`, writes 4 floats per recorded apply to ms_out (layout as
 * mfh_apply_timed: cached, fused, reduce, whole apply), stores the number of recorded applies and disarms.
 * ms_out must hold 4 * n_applies floats.  Errors: INVALID_ARG, BAD_STATE (no plan), CUDA. */
MFH_API int mfh_timing_begin(mfh_handle h, int32_t n_applies);
MFH_API int mfh_timing_end(mfh_handle h, float* ms_out, int32_t* n_recorded, void* stream);

/* Allocation-free entry point: phi = lambda * V(seed) psi for ONE complex128 vector, V the seeded GUE operator of
 * mfh_create(kind = MFH_SRC_GUE) (Eq. 4-5; entries as BASELINE.json configs[0]), generated on the fly.  For
 * callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses that forbid it):
 * no handle and no plan; this call and everything below it calls no cudaMalloc, no cudaFree and no allocating library
 * routine.  Its scratch (generator table + 16 partial sums per row, added in a fixed order: deterministic, no atomics)
 * is ONE file-scope device array of 32 KB + 16 * MFH_STATIC_MAX_D * 16 B = 4.03 MB that every GPU which loads the
 * library holds until the process exits.
 *   D         matrix dimension: a multiple of 128, 128 <= D <= MFH_STATIC_MAX_D; a larger D is refused with
 *             MFH_ERR_INVALID_ARG and a message that names the limit (use mfh_create / mfh_plan / mfh_apply there)
 *   psi_dev   D complex128 (interleaved re, im), DEVICE pointer, 16-byte aligned, caller-owned, read only
 *   phi_dev   D complex128, DEVICE pointer, 16-byte aligned, caller-owned, overwritten; must not alias psi_dev
 *   stream    cudaStream_t of the CURRENT device (NULL = default stream); the call is asynchronous
 * The result equals mfh_apply on a procedural complex128 plan of the same (D, seed, lambda) up to the summation order
 * (<= 1e-11 relative L2, tests/test_zz_no_alloc.py).
 * SHARED STATE: all calls on one device use the same scratch array, which keeps the last call's contents (nothing in
 * it has to start at zero: every value a call reads it has written itself).  Calls that overlap on the GPU -- two
 * streams, or two host threads on different streams -- race on it: issue them on one stream or order them with events.
 * Host-side set-up is guarded by a mutex.  The first call on a device resolves the array's device address
 * (cudaGetSymbolAddress); a call whose D differs from the previous call's on that device re-uploads the 20 KB generator
 * table with a stream-ordered cudaMemcpyAsync from host memory.
 * Errors: MFH_ERR_INVALID_ARG (NULL / aliased pointers, D out of range or not a multiple of 128), MFH_ERR_UNSUPPORTED
 * (device ordinal >= 64), MFH_ERR_CUDA. */
#define MFH_STATIC_MAX_D 16384
MFH_API int mfh_apply_static(int64_t D, uint64_t seed, double lambda, const void* psi_dev, void* phi_dev, void* stream);

/* Same as mfh_apply but with HOST buffers: copies psi to the device, applies, copies phi back and
 * synchronises `stream` (the end-to-end call bench.py times).  Host buffers should be pinned. */
MFH_API int mfh_apply_host(mfh_handle h, const void* psi_host, void* phi_host, int32_t k,
                           const double* lambdas_host, void* stream);

/* out = exp(-i H t) psi by the Chebyshev expansion (Eq. 41-44), one vector (the handle must be
 * planned with k = 1; H uses the handle's lambda).  c = (e_max+e_min)/2, R = (e_max-e_min)/2,
 * a = R t; terms l = 0..K-1 with K = 1 + max{l : |J_l(a)| >= tol}; K-1 calls of the apply path.
 * Asynchronous on `stream` after the host-side Bessel table; *n_terms_out = K (may be NULL).
 * [e_min, e_max] must enclose the spectrum (for the GUE of this library: about +-2*lambda).
 * Errors: INVALID_ARG (e_max <= e_min, non-finite t, tol <= 0, k != 1); BAD_STATE; CUDA. */
MFH_API int mfh_chebyshev(mfh_handle h, const void* psi_dev, void* out_dev, double t, double e_min,
                          double e_max, double tol, int32_t* n_terms_out, void* stream);

/* Coupling scan with propagation (the paper's outer loop over coupling values, "independent outer-loop
 * parameters, such as coupling strengths", run here as k simultaneous columns of ONE k-vector plan, Eq. 12):
 *     out[:, v] = exp(-i H_v t) psi[:, v],   H_v = diag(h0) + lambda_v V   (MFH_SRC_DIAG_PLUS_GUE; lambda_v V otherwise),
 * all k columns with the same Chebyshev series (same bounds: [e_min, e_max] must enclose the spectrum of EVERY H_v, so
 * K is set by the widest one), each of the K-1 applies generating or reading every block once for all k columns.
 *   psi_dev, out_dev  [D][k] of the planned k;  lambdas_host  k doubles or NULL (the handle's lambda for all)
 * Errors as mfh_chebyshev. */
MFH_API int mfh_chebyshev_scan(mfh_handle h, const void* psi_dev, void* out_dev, double t, double e_min, double e_max,
                               double tol, const double* lambdas_host, int32_t* n_terms_out, void* stream);

/* out = exp(-beta (H - e_min)) psi, the imaginary-time (thermal / TPQ) Chebyshev filter the paper runs before its
 * real-time propagation ("the imaginary-time TPQ Chebyshev filter used order 80"; the series is not
 * printed there, R21).  Same recurrence as mfh_chebyshev (Eq. 41-43) with the modified-Bessel
 * coefficients of e^{-a x} = I_0(a) + 2 sum_l (-1)^l I_l(a) T_l(x), a = R beta, scaled by e^{-a}:
 *     out = sum_{l<K} (2 - delta_l0) (-1)^l [e^{-a} I_l(a)] T_l(H~) psi,   K = 1 + max{l : 2 e^{-a} I_l(a) >= tol},
 * so exp(-beta H) psi = exp(-beta e_min) * out and no factor exceeds 1.  beta >= 0, R beta <= 600.
 * *n_terms_out = K (may be NULL); K-1 applies of the planned path (k = 1).  Errors as mfh_chebyshev. */
MFH_API int mfh_chebyshev_imag(mfh_handle h, const void* psi_dev, void* out_dev, double beta, double e_min,
                               double e_max, double tol, int32_t* n_terms_out, void* stream);

/* Spectral bounds by matrix-free Lanczos ("matrix-free Lanczos iterations estimate spectral bounds
 * E_min and E_max"; --lanczos-m 40; reading R18).  m steps (capped at D) of the plain
 * three-term recurrence from v_1 = psi/||psi||, each step one apply of the planned path (k = 1) plus O(D)
 * vector kernels with the scalars kept on the device; theta_min, theta_max = extreme eigenvalues of the
 * tridiagonal T_m (host, Sturm bisection); with c, R the centre and half-width of [theta_min, theta_max]:
 *     *e_min = c - (1 + margin) R,   *e_max = c + (1 + margin) R        (Ritz values lie inside the spectrum).
 *   psi_dev              start vector (device, [D] complex), any non-zero norm; not modified
 *   alpha_host, beta_host  optional host arrays of m doubles receiving the recurrence coefficients
 * Synchronises `stream`.  Errors: INVALID_ARG, BAD_STATE (no plan), NOT_CONVERGED (breakdown), CUDA. */
MFH_API int mfh_lanczos_bounds(mfh_handle h, const void* psi_dev, int32_t m, double margin, double* e_min,
                               double* e_max, double* alpha_host, double* beta_host, void* stream);

/* n_steps successive propagations out = [exp(-i H tau)]^n_steps psi, each one Chebyshev expansion as in
 * mfh_chebyshev (the paper propagates N = 200 steps of tau).  out_dev must not alias psi_dev.
 * *n_terms_out = terms per step. */
MFH_API int mfh_chebyshev_steps(mfh_handle h, const void* psi_dev, void* out_dev, double tau, int32_t n_steps,
                                double e_min, double e_max, double tol, int32_t* n_terms_out, void* stream);

/* Distributed execution over `world` GPUs, one process and one handle per GPU (P:185-191 block-row
 * accumulation; P:461-469 row-parallel strategy; P:597-618 row distribution; R20, 6.10).  Call
 * before mfh_plan (drops a committed plan).  Every rank receives the FULL psi; after mfh_apply the ranks run
 * one exchange step of D * B_c bytes (linear in D), done by the caller (NCCL through torch.distributed
 * in paper_2606_31598_b200/distributed.py):
 *   MFH_PART_ROWS   the paper's scheme: rank r owns the block rows n_blk*r/world <= n < n_blk*(r+1)/world,
 *                   caches / generates only those and writes ONLY the rows of phi it owns (the other rows of
 *                   phi_dev are left untouched); exchange = all-gather of the segments.  No Hermitian reuse
 *                   across ranks: blocks whose mirror lies on another rank are generated one-sided.
 *   MFH_PART_PAIRS  the unordered block pairs {n,m} are dealt round-robin to the ranks (order: circular
 *                   distance d = 0..n_blk/2, then n); a rank owns both positions of its pairs, so every
 *                   Hermitian pair is generated or stored once in the whole job; mfh_apply writes a
 *                   full-length partial phi (the H0 term on the rank that owns block (n,n));
 *                   exchange = all-reduce (sum).
 *   MFH_PART_NONE   single GPU (world must be 1).
 * Block ownership is defined in block indices, so every rank must plan the SAME block size: with world > 1
 * mfh_plan refuses a handle created with B = 0 (MFH_ERR_INVALID_ARG) -- fix B in mfh_create on every rank
 * (paper_2606_31598_b200/distributed.py also compares the planned (B, n_blk, k) of all ranks).
 * mfh_chebyshev / mfh_chebyshev_steps / mfh_lanczos_bounds chain applies, so on a partitioned handle they
 * call the exchange hook registered with mfh_set_exchange after every apply (MFH_ERR_BAD_STATE if none).
 * Errors: INVALID_ARG (rank outside [0, world), world < 1, unknown scheme, world > 1 with MFH_PART_NONE). */
enum { MFH_PART_NONE = 0, MFH_PART_ROWS = 1, MFH_PART_PAIRS = 2 };
MFH_API int mfh_set_partition(mfh_handle h, int32_t rank, int32_t world, int32_t scheme);

/* Exchange hook of a partitioned handle: called on the host by the chained drivers right after an apply
 * has been enqueued, with the device vector the apply wrote (bytes = D * k * B_c) and the stream; it must
 * enqueue the all-gather (MFH_PART_ROWS) or all-reduce (MFH_PART_PAIRS) of that vector in stream order and
 * return 0.  The library itself contains no communication code.  fn = NULL removes the hook. */
typedef int (*mfh_exchange_fn)(void* user, void* phi_dev, size_t bytes, void* stream);
MFH_API int mfh_set_exchange(mfh_handle h, mfh_exchange_fn fn, void* user);

/* First block row and number of block rows that mfh_apply writes on this handle (after mfh_plan):
 * the owned slab for MFH_PART_ROWS, [0, n_blk) otherwise.  B_out receives the planned block size. */
MFH_API int mfh_get_partition_rows(mfh_handle h, int32_t* first_block_row, int32_t* n_block_rows, int32_t* B_out);

/* Free the handle and everything it owns.  NULL is accepted. */
MFH_API int mfh_destroy(mfh_handle h);

/* Thread-local message of the last failing call ("" if none). */
MFH_API const char* mfh_last_error(void);

/* JSON description of the committed plan (mode, B, cached blocks, bytes, launches per apply; "two_sided_pairs" /
 * "two_sided_stored_pairs": block pairs of a complex64 k-vector plan that are generated / read from the pair cache
 * ONCE for both positions by the two-sided tensor-core kernels). */
MFH_API int mfh_get_plan(mfh_handle h, char* json_out, size_t json_cap);

/* ---- system-bath Hamiltonian (the paper's own workload shape, R19) -------
 *     H = H_S (x) I_B + I_S (x) H_B + g A (x) B_1   on   w in C^{d_S} (x) C^{d_B}
 * with H_B, B_1 two dense d_B x d_B bath-side operators (seeded GUE, entry rule of mfh_create) applied
 * to R = d_S simultaneous state components (Eq. 12-13, n_op = 2).  The state is X[b][s], row-major
 * [d_B][d_S] complex of `dtype` (the k-vector layout with D = d_B, k = d_S); the result
 *     Y = H_B X + g (B_1 X) A^T + X H_S^T.
 *   HS_host, A_host   d_S x d_S Hermitian matrices, row-major interleaved complex doubles (host)
 *   d_S <= MFH_MAX_K; d_B, B as in mfh_create.  mfh_sb_plan plans both bath operators with k = d_S
 *   (cached blocks need B % 128 == 0) inside the budget (0 = 0.9 x free memory).
 * Errors as for mfh_create / mfh_plan / mfh_apply. */
typedef struct mfh_sb_s* mfh_sb_handle;
MFH_API int mfh_sb_create(mfh_sb_handle* out, int64_t d_B, int32_t d_S, int32_t B, uint64_t seed_HB, uint64_t seed_B1,
                          int32_t dtype, const double* HS_host, const double* A_host, double g);
MFH_API int mfh_sb_plan(mfh_sb_handle h, int32_t mode, int64_t n_applies_hint, int64_t hbm_budget_bytes, void* stream,
                        char* json_out, size_t json_cap);
MFH_API int mfh_sb_apply(mfh_sb_handle h, const void* x_dev, void* y_dev, void* stream);
MFH_API int mfh_sb_destroy(mfh_sb_handle h);

/* ---- test-only exports --------------------------------------------------------------------- */

/* Raw Philox4x32-10 words for n index pairs: key = seed, ctr = (min(i,j), max(i,j), stream_id, 0).
 * i_dev, j_dev: n uint32 (device); words_dev: 4n uint32 (device). */
MFH_API int mfh_debug_philox(uint64_t seed, uint32_t stream_id, const uint32_t* i_dev,
                             const uint32_t* j_dev, int64_t n, uint32_t* words_dev, void* stream);

/* Dense block H^[n,m] of V (lambda and H0 not applied) written row-major B x B complex of the
 * handle's dtype to block_dev -- the same generator the fused kernel and the cache fill use.
 * Needs B fixed (mfh_create with B != 0, or after mfh_plan). */
MFH_API int mfh_materialize_block(mfh_handle h, int32_t n, int32_t m, void* block_dev, void* stream);

/* Self-check exports (compute-sanitizer is not available on every machine; tests/test_gpu_selfcheck.py):
 *   mfh_debug_poison     fills the partial-sum workspace and the Chebyshev scratch with 0xFF bytes (NaN in both
 *                        precisions), asynchronously on `stream`: a kernel that reads a partial sum no kernel of the
 *                        same apply has written turns phi into NaN (the substitute for initcheck).
 *   mfh_debug_selfcheck  every library-owned plan buffer sits between two 4 KB guard bands filled with a byte pattern
 *                        at allocation; counts the guard bytes that no longer hold it (out-of-bounds writes; the
 *                        write side of memcheck).  Synchronises `stream`.
 * Errors: BAD_STATE (no plan), INVALID_ARG, CUDA. */
/* Test of the test: overwrites the guard byte right before (after = 0) or right after (after = 1) the buffer_index-th
 * library-owned buffer, as an out-of-bounds write would; mfh_debug_selfcheck must then report it. */
MFH_API int mfh_debug_corrupt_guard(mfh_handle h, int32_t buffer_index, int32_t after);
MFH_API int mfh_debug_poison(mfh_handle h, void* stream);
MFH_API int mfh_debug_selfcheck(mfh_handle h, int64_t* bad_guard_bytes, void* stream);

/* The Bessel table behind mfh_chebyshev (Jacobi-Anger coefficients, R7): J_l(x) for l = 0..l_max written to
 * out_host (l_max + 1 doubles, host), x >= 0, by Miller's downward recurrence normalised with
 * J_0 + 2 sum_j J_2j = 1 (valid for every x; host only, no GPU).  Errors: INVALID_ARG. */
MFH_API int mfh_debug_bessel_j(double x, int32_t l_max, double* out_host);

/* The H0 diagonal (D reals of the handle's real type) written to h0_dev. */
MFH_API int mfh_debug_h0(mfh_handle h, void* h0_dev, void* stream);

/* ---- measurement export --------------------------------------------------------------------- */

/* Instruction-mix ceiling of the fused generate-and-apply kernels: times a synthetic
 * kernel that issues, per unit, the same instruction counts as one generated entry -- no memory traffic,
 * four independent units in flight per thread -- and returns units per second (host double).
 *   MFH_MIX_C128_PAIR   14 32x32->64 multiplies + 26 ALU ops + 32 DFMA: one generated complex128 pair
 *                       {i,j} used for both phi_i and phi_j (2 matrix entries); of the 18 multiplies of a
 *                       Philox4x32-10 call the fused kernel shares 4 between the rows of a lane
 *   MFH_MIX_C64_ENTRY   14 multiplies + 20 ALU ops + 4 SFU ops + 11 FP32 ops: one generated complex64
 *                       entry whose multiply-accumulate runs on the tensor cores
 *   MFH_MIX_PHILOX      one full Philox call (18 multiplies, 18 xors);   MFH_MIX_DFMA31  the 32 FP64 operations alone
 * Component ceilings ("Philox-only, Philox+Box-Muller, MAC-only micro-kernels"), which call the
 * library's own generator functions (not typed-in instruction counts) in the fused kernel's shape -- 8 warps, 2 CTAs
 * per SM, 4 rows per lane -- and return generated PAIRS per second (one pair = two matrix entries with Hermitian reuse):
 *   MFH_COMP_PHILOX          pair_words() only, words xor-reduced
 *   MFH_COMP_PHILOX_BM_C128  + the FP64 Box-Muller of the complex128 kernels (tables in shared memory), entries summed
 *   MFH_COMP_MAC_C128        the two-sided multiply-accumulate alone (8 DFMA per pair, psi_j from shared memory, the
 *                            column accumulator rotated by shuffles) on entries that cost half an add each
 *   MFH_COMP_PHILOX_BM_C64 / MFH_COMP_MAC_C64   the same for the complex64 CUDA-core kernel (SFU Box-Muller, FFMA)
 * Pipe model (which instruction classes of the generator overlap on this GPU; units per second of the synthetic
 * kernel, one unit = the named instructions per lane):
 *   MFH_PIPE_WIDE16 (16 32x32->64 multiplies + 16 xors), MFH_PIPE_LOP32 (32 logic ops), MFH_PIPE_DFMA32 (32 DFMA with
 *   immediate operands), MFH_PIPE_DFMA32_REG3 (32 DFMA with three register operands), and the pairs
 *   MFH_PIPE_WIDE16_DFMA32, MFH_PIPE_LOP32_DFMA32, MFH_PIPE_WIDE16_LOP32: a pair that takes as long as the sum of
 *   its parts does not overlap.
 * FP64 multiply-accumulate streams of the cached complex128 k-vector kernel (units = DFMA thread instructions per
 * second): MFH_PIPE_CMAC_REGS -- the complex multiply-accumulate alone, psi values in registers, 16 DFMA in a row per
 * entry component (the ceiling of the pattern: every DFMA but the first of a run takes the entry from the operand
 * reuse cache); MFH_PIPE_CMAC_LDS -- that kernel's inner loop as written, entry and psi values from shared memory every
 * column (the ceiling of the loop).
 * Synchronises `stream`.  Errors: INVALID_ARG, CUDA. */
enum { MFH_MIX_C128_PAIR = 0, MFH_MIX_C64_ENTRY = 1, MFH_MIX_PHILOX = 2, MFH_MIX_DFMA31 = 3, MFH_COMP_PHILOX = 4,
       MFH_COMP_PHILOX_BM_C128 = 5, MFH_COMP_MAC_C128 = 6, MFH_COMP_PHILOX_BM_C64 = 7, MFH_COMP_MAC_C64 = 8,
       MFH_PIPE_WIDE16 = 9, MFH_PIPE_LOP32 = 10, MFH_PIPE_DFMA32 = 11, MFH_PIPE_DFMA32_REG3 = 12,
       MFH_PIPE_WIDE16_DFMA32 = 13, MFH_PIPE_LOP32_DFMA32 = 14, MFH_PIPE_WIDE16_LOP32 = 15,
       MFH_PIPE_CMAC_REGS = 16, MFH_PIPE_CMAC_LDS = 17 };
MFH_API int mfh_debug_pipe_rates(int32_t mix, double* units_per_s, void* stream);

/* Read-only HBM stream probe: times a kernel that reads `bytes` of buf_dev once (8 independent 128-bit
 * non-allocating loads per thread, grid = 8 CTAs per SM) and returns bytes per second (best of 3 after a
 * warm-up).  The roofline denominator for kernels that read a cached matrix once; a device-to-device copy
 * (MEASURED_PEAKS.json) also pays the write turn-around.  buf_dev: device, 16-byte aligned, >= 1 MiB and
 * larger than L2 for an HBM figure.  Synchronises `stream`.  Errors: INVALID_ARG, CUDA. */
MFH_API int mfh_debug_read_bandwidth(const void* buf_dev, size_t bytes, double* bytes_per_s, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* MFH_H */
