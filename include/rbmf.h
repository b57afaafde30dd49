/* rbmf.h -- C ABI of the B200-native reduced-basis hierarchical matched filter.
 *
 * The library implements the hot path of Dhurkunde, Fehrmann & Nitz, "A hierarchical approach to
 * matched filtering using a reduced basis" (arXiv:2110.13115; citations below are PAPER.md lines):
 *
 *   a1  g_k[j]      = s d[j] conj(b_k[j]),  j in band [j_low, N/2)
 *   a2  beta_k[n]   = sum_j g_k[j] exp(+2 pi i j n / N)                        (Eq. 6)
 *   a3  beta^avg_k[i] = (1/w) sum_{r<w} beta_k[i w + r]                        (Eq. 9)
 *   a4  R_t[i]      = (1/sigma_t) sum_k conj(c_tk) beta^avg_k[i]               (Eq. 7)
 *   a5  candidate (t,i)  iff |R_t[i]| >= thr_stage1
 *   a6  rho_t[i w + r] = (1/sigma_t) sum_k conj(c_tk) beta_k[i w + r], r < w, for every candidate;
 *       trigger iff |rho| >= thr_stage2
 *
 * with s = sqrt(2/N), d = unnormalised forward DFT of the whitened unit-variance strain, b_k orthonormal
 * over the band, c_tk the decomposition coefficients.  Every step runs in hand-written CUDA
 * kernels for sm_100a (a persistent, TMA-fed batched four-step Stockham FFT; a tcgen05/TMEM GEMM -- fp16 screen with a
 * derived error bound by default, split-bf16 on request -- with a fused threshold/compaction epilogue; a re-scoring
 * kernel that regroups the candidates by bin, scores them from a shared-memory copy of the bin's block of beta and
 * also confirms the screen's hits in fp32).  There is no CPU fallback.
 * Around that path: batches of segments and the step in front of the path (rbmf_filter_batch,
 * rbmf_prepare_strain), the paper's template routes as comparators (rbmf_filter_flat, RBMF_STAGE1_TEMPLATES), many
 * sub-banks against one strain (rbmf_bankset_*), and the preparation of a sub-bank (rbmf_prepare_basis / _coeffs).
 *
 * Conventions
 *  - "dev" pointers are CUDA device memory owned by the caller; "host" pointers are ordinary host memory.
 *  - The library never allocates or frees device memory: the caller provides one workspace
 *    (rbmf_workspace_bytes / rbmf_plan_set_workspace) that must outlive the plan's use.  The one entry point that
 *    needs neither plan nor workspace, rbmf_prepare_strain_static, works out of a fixed 12 MiB array that is part of
 *    the library image on every GPU (see its description below).
 *  - rbmf_set_basis / rbmf_set_coeffs copy and re-lay-out their inputs into the workspace; the caller's
 *    arrays may be freed after the stream has completed those calls.
 *  - All work is enqueued on the plan's stream (rbmf_set_stream; default: the legacy default stream) and
 *    is asynchronous unless stated.  No function throws or aborts; every one returns an rbmf_status.
 *  - complex64 = interleaved (re, im) float32, little endian.
 */
#ifndef RBMF_H
#define RBMF_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct rbmf_plan rbmf_plan; /* opaque */

/* One final trigger: a sample whose SNR modulus is above thr_stage2 inside a first-stage bin. */
typedef struct {
    int32_t template_id; /* row of the coefficient matrix                       */
    int32_t time_index;  /* sample n in [0, N)                                  */
    float snr_re;        /* complex SNR rho_t[n] (already divided by sigma_t)   */
    float snr_im;
} rbmf_trigger;

/* One first-stage candidate: a (template, bin) whose averaged SNR modulus is above thr_stage1. */
typedef struct {
    int32_t template_id;
    int32_t bin_index; /* i in [0, N/w): samples i w .. i w + w - 1            */
    float avg_re;      /* averaged complex SNR R_t[i]                         */
    float avg_im;
} rbmf_candidate;

typedef enum {
    RBMF_OK = 0,
    RBMF_ERR_ARG = -1,         /* bad argument (NULL, size, alignment, range)                          */
    RBMF_ERR_STATE = -2,       /* call order: workspace / basis / coefficients not set yet             */
    RBMF_ERR_CUDA = -3,        /* a CUDA runtime/driver call failed (rbmf_last_cuda_error has the code) */
    RBMF_ERR_OVERFLOW = -4,    /* more candidates or triggers than capacity; lists are truncated       */
    RBMF_ERR_UNSUPPORTED = -5  /* valid but not implemented for this size / device                     */
} rbmf_status;

/* Stage-1 reconstruction kernels (rbmf_plan_set_gemm_impl).  (Value 1 is not a product mode: it selects the
 * verification kernel of the diagnostics section at the end of this header and is accepted only through it.) */
typedef enum {
    RBMF_GEMM_TCGEN05 = 0, /* TMA + tcgen05.mma, bf16x3 split precision (fp32-equivalent) + TMEM epilogue          */
    RBMF_GEMM_SCREEN = 2   /* default: the same tensor-core kernel with ONE fp16 product per term and thr_stage1
                              lowered, per (bin, template block), by a derived bound of the fp16 error (operand
                              rounding is exact analysis; the tensor core's fp32 accumulation term is an assumption
                              verified on the device, largest observed error / bound 0.56), so its output is a
                              superset of the true candidates; kernel 3 then repeats the stage-1 test at
                              fp32 accuracy (the mean of the w fp32 samples it computes anyway is the averaged SNR of
                              Eq. 9) before scoring.  Same candidate and trigger sets as RBMF_GEMM_TCGEN05 up to
                              fp32 rounding at the threshold, one third of the tensor-core work.               */
} rbmf_gemm_impl;

/* Create a plan for segments of N samples (power of two, 2^10 <= N <= 2^24) at sampling rate fs [Hz],
 * lower cutoff f_low [Hz] (0 < f_low < fs/2), k basis vectors (multiple of 16, 16 <= k <= 1024) and T >= 1
 * templates.  Band = bins [ceil(f_low N / fs), N/2).  Host-only; no device work.  Defaults: w = 8,
 * max_candidates = max_triggers = 2^22.  *out is set to NULL on failure.  Segments longer than 2^20 samples are a
 * valid request that this build does not implement (the FFT is two passes of length <= 1024): RBMF_ERR_UNSUPPORTED. */
rbmf_status rbmf_plan_create(rbmf_plan** out, int64_t N, double fs, double f_low, int32_t k, int32_t T);

/* Stage-1 averaging window w of Eq. 9 (power of two, 1 <= w <= 32, N/w >= 128).  w = 1 is the flat search.
 * Must be called before rbmf_workspace_bytes / rbmf_plan_set_workspace. */
rbmf_status rbmf_plan_set_window(rbmf_plan* plan, int32_t w);

/* Capacity (entries) of the internal candidate list and of the caller's trigger array.  Must be called
 * before rbmf_workspace_bytes / rbmf_plan_set_workspace. */
rbmf_status rbmf_plan_set_capacity(rbmf_plan* plan, int64_t max_candidates, int64_t max_triggers);

/* Largest number of strain segments one rbmf_filter_batch call may take (default 1).  The paper filters a batch of
 * segments in parallel against the resident basis and coefficients; the workspace holds beta and the
 * beta^avg planes of max_batch segments.  max_batch * N must stay below 2^31 (a trigger's time_index counts samples
 * over the whole batch).  Must be called before rbmf_workspace_bytes / rbmf_plan_set_workspace. */
rbmf_status rbmf_plan_set_batch(rbmf_plan* plan, int32_t max_batch);

/* Select the stage-1 kernel (RBMF_GEMM_SCREEN, the default, or RBMF_GEMM_TCGEN05).  May be called at any time. */
rbmf_status rbmf_plan_set_gemm_impl(rbmf_plan* plan, int32_t impl);

/* Bytes of device workspace the plan needs (depends on N, k, T, w, capacities). */
rbmf_status rbmf_workspace_bytes(const rbmf_plan* plan, size_t* bytes);

/* Hand the plan its workspace: dev_ptr must be 1024-byte aligned device memory of >= rbmf_workspace_bytes.
 * Enqueues the initialisation of the plan's constant tables (twiddles) on the plan's stream.  Invalidates
 * any basis / coefficients set before. */
rbmf_status rbmf_plan_set_workspace(rbmf_plan* plan, void* dev_ptr, size_t bytes);

/* cudaStream_t to enqueue on (NULL = legacy default stream). */
rbmf_status rbmf_set_stream(rbmf_plan* plan, void* cuda_stream);

/* basis_dev: k x (N/2+1) complex64, row-major: b_k[j] (p~_k of PAPER.md:82), orthonormal over the band.
 * Values outside the band are ignored.  Copied (re-laid-out in the order the FFT reads it) into the workspace. */
rbmf_status rbmf_set_basis(rbmf_plan* plan, const void* basis_dev);

/* coeffs_dev: T x k complex64, row-major: c_tk, unconjugated.  sigma_dev: T float32 template
 * norms sigma_t > 0, or NULL => sigma_t = ||c_t||_2.  Copied (conjugated, scaled by 1/sigma_t, split into bf16
 * hi/lo planes) into the workspace.  A template whose sigma_t is not a positive finite number (or, with NULL, whose
 * coefficients are all zero) is disabled: it produces no candidates and no triggers. */
rbmf_status rbmf_set_coeffs(rbmf_plan* plan, const void* coeffs_dev, const float* sigma_dev);

/* Filter one segment.  strain_dev: (N/2+1) complex64, the unnormalised forward DFT of the whitened strain.
 * thr_stage1 > 0 applies to the modulus of the w-averaged SNR, thr_stage2 > 0 to the modulus of the SNR.
 * out_dev: array of max_triggers rbmf_trigger (unordered set on return).  n_out_dev: device int64 that
 * receives the TOTAL number of triggers found (may exceed max_triggers; then only max_triggers were written).
 * Enqueues only; results are valid once the stream has completed. */
rbmf_status rbmf_filter(rbmf_plan* plan, const void* strain_dev, float thr_stage1, float thr_stage2,
                        rbmf_trigger* out_dev, int64_t* n_out_dev);

/* The step in front of the path (PAPER.md:175 "FFT of the data", :177 division by sqrt(S_n)): forward real-to-complex
 * DFT of n_segments (<= max_batch) time series and whitening,
 *     strain_out[b][j] = inv_asd[j] * sum_n x[b][n] exp(-2 pi i j n / N),   j = 0 .. N/2,
 * i.e. exactly the array rbmf_filter / rbmf_filter_batch take.  x_dev: n_segments x N float32 (8-byte aligned);
 * inv_asd_dev: N/2+1 float32 = 1/sqrt(S_n(f_j)) in the caller's normalisation (such that the whitened series has unit
 * variance per sample), or NULL for data that is already white; strain_out_dev: n_segments x (N/2+1) complex64, must
 * not alias x_dev.  Enqueues three small kernels on the plan's stream (a four-step radix-2 FFT of the series packed
 * as N/2 complex values, then the real-input split); needs the workspace, not the basis or the coefficients. */
rbmf_status rbmf_prepare_strain(rbmf_plan* plan, const float* x_dev, const float* inv_asd_dev, int32_t n_segments,
                                void* strain_out_dev);

/* rbmf_prepare_strain for callers that cannot provide device memory: no plan, no workspace, and not one allocation
 * (no cudaMalloc / cudaFree / allocating library routine) inside the call.
 *
 * Who needs it.  Every other entry point works out of a workspace the caller allocates; rbmf_prepare_strain needs a
 * whole plan (sized for the filter) just to borrow 3 small scratch arrays from it.  Some users of the front end cannot
 * do that: a strain-conditioning stage that whitens data for several filter processes and owns no plan; a plug-in or
 * callback that runs inside another program's pipeline and is handed only its input and output buffers; a process in
 * which a framework's memory pool has already taken the whole GPU, so a raw cudaMalloc fails; a low-latency loop
 * (online searches use reduced-basis filtering; whitening dominates their latency) where cudaMalloc's device-wide synchronisation would
 * stall the filter streams running beside it.  For them the scratch (twiddle table, pass-1 intermediate, packed
 * spectrum) lives in a fixed array inside the library image: RBMF_STATIC_SCRATCH_BYTES (12 MiB) on EVERY GPU on which
 * the library's CUDA module gets loaded, from that load until the process exits, whether or not this call is used.
 *
 * The limit.  One call may transform at most RBMF_STATIC_MAX_SAMPLES = 2^20 samples in total: N a power of two,
 * 2^10 <= N <= 2^20, and n_segments * N <= 2^20 (e.g. one segment of 2^20, two of the Paper configuration's 2^19,
 * four of the paper's own 2^18 block).  More returns RBMF_ERR_UNSUPPORTED and launches nothing (N outside
 * [2^10, 2^24] or not a power of two: RBMF_ERR_ARG, as for rbmf_plan_create); split a larger batch into several
 * calls.  rbmf_prepare_strain_static_limits reports both numbers at run time (either pointer may be NULL).
 *
 * Arguments and result are those of rbmf_prepare_strain -- x_dev: n_segments x N float32 (8-byte aligned);
 * inv_asd_dev: N/2+1 float32 or NULL; strain_out_dev: n_segments x (N/2+1) complex64, 8-byte aligned, not aliasing
 * x_dev; all caller-owned device memory on the CURRENT device -- with N and the stream (cudaStream_t, NULL = legacy
 * default stream) given directly.  The output is bit-identical to rbmf_prepare_strain's (same kernels, same table).
 * Enqueues four kernels (the table for this N, two FFT passes, split + whitening) and returns; *cuda_error (may be
 * NULL) receives the cudaError_t when the status is RBMF_ERR_CUDA, else 0.
 *
 * First call on a device.  The first call made with a given device current looks up the array's address on that
 * device and sets the kernels' shared-memory attribute there (host-side work, once per device and process, guarded
 * by a mutex).  Make that first call during start-up, on the device in question, before any stream capture begins.
 *
 * Sharing.  All calls on one device use the SAME array, and it keeps what the last call left in it.  The call does
 * not rely on its contents (everything it reads it has written first, on its own stream, so nothing has to be
 * cleared), but two calls whose kernels can overlap on the GPU -- different streams without an event between them,
 * different host threads -- overwrite each other's table and intermediates and produce garbage without any error.
 * Run them on one stream, or order them with events.  Calls on different GPUs do not interact. */
#define RBMF_STATIC_MAX_SAMPLES (1 << 20)
#define RBMF_STATIC_SCRATCH_BYTES (3 * (RBMF_STATIC_MAX_SAMPLES / 2) * 8)
rbmf_status rbmf_prepare_strain_static(const float* x_dev, const float* inv_asd_dev, int64_t N, int32_t n_segments,
                                       void* strain_out_dev, void* cuda_stream, int32_t* cuda_error);
rbmf_status rbmf_prepare_strain_static_limits(int64_t* max_samples, size_t* scratch_bytes);

/* Filter n_segments (1 <= n_segments <= max_batch) segments at once ("filtering each segment in
 * parallel", basis and coefficients loaded once).  strain_dev: n_segments x (N/2+1) complex64, row-major, each row as
 * in rbmf_filter.  Steps a1-a3 run once per (segment, basis column) in ONE persistent launch (no launch gaps or
 * pipeline drains between segments); steps a4-a5 run as ONE contraction over the
 * n_segments * N/w bins of the batch (each coefficient tile is loaded once per batch); step a6 over all candidates.
 * Triggers carry the segment in the time index: time_index = segment * N + n, n in [0, N)  (rbmf_candidate:
 * bin_index = segment * N/w + i).  The result equals n_segments calls of rbmf_filter, segment by segment.
 * Other arguments, asynchrony and overflow behaviour as in rbmf_filter. */
rbmf_status rbmf_filter_batch(rbmf_plan* plan, const void* strain_dev, int32_t n_segments, float thr_stage1,
                              float thr_stage2, rbmf_trigger* out_dev, int64_t* n_out_dev);

/* End-to-end convenience with HOST buffers: copies the strain to the device, filters, waits, and copies
 * the triggers back.  strain_host: (N/2+1) complex64.  out_host: capacity_out entries (<= max_triggers).
 * *n_out_host = total found.  Synchronous.  Returns RBMF_ERR_OVERFLOW if either list overflowed. */
rbmf_status rbmf_filter_host(rbmf_plan* plan, const void* strain_host, float thr_stage1, float thr_stage2,
                             rbmf_trigger* out_host, int64_t capacity_out, int64_t* n_out_host);

/* rbmf_filter_host for a batch: strain_host is n_segments x (N/2+1) complex64; triggers as in rbmf_filter_batch. */
rbmf_status rbmf_filter_batch_host(rbmf_plan* plan, const void* strain_host, int32_t n_segments, float thr_stage1,
                                   float thr_stage2, rbmf_trigger* out_host, int64_t capacity_out,
                                   int64_t* n_out_host);

/* ---- The paper's template routes, as on-GPU comparators of the basis route ------
 * rbmf_plan_enable_template_routes(plan, slab): reserve workspace for them; slab = templates transformed per pass
 * (multiple of 4, <= 1024; 0 disables).  Before rbmf_workspace_bytes / rbmf_plan_set_workspace and after
 * rbmf_plan_set_window; needs w >= 2 and 2 N / w >= 1024 (RBMF_ERR_UNSUPPORTED otherwise).
 * rbmf_set_templates(plan, templates_dev, sigma_dev): templates_dev = T x (N/2+1) complex64, row-major, the filters
 * h_t[j] themselves (bank templates, or reconstructed ones sum_k c_tk b_k); values outside the band are ignored.  The
 * POINTER IS RETAINED (42 GB at T = 20000, N = 2^19: too large to copy): the array must stay valid and unchanged while
 * the template routes are used.  sigma_dev: T float32 norms (copied), or NULL => sigma_t = 1.
 * rbmf_filter_flat: the flat template method (PAPER.md:61-68; Eq. 13; the paper's cuFFT baseline, :338): one
 * full-length inverse FFT per template, rho_t[n] = (s / sigma_t) sum_j d[j] conj(h_t[j]) exp(2 pi i j n / N), and a
 * trigger for EVERY sample with |rho_t[n]| >= thr.  Needs no basis and no coefficients.  Outputs as in rbmf_filter.
 * rbmf_plan_set_stage1_route(plan, RBMF_STAGE1_TEMPLATES): rbmf_filter takes its first-stage candidates from the
 * paper's fast first stage by templates (Eq. 10-12: alias-folded spectrum + an inverse FFT of length N / w per
 * template) instead of the GEMM on the basis series; the second stage is unchanged (it re-scores from beta, so basis
 * and coefficients are still needed).  With h_t = sum_k c_tk b_k both routes define the same candidates (linearity,
 * PAPER.md:191, :218).  Single segments only (rbmf_filter_batch with n_segments > 1: RBMF_ERR_UNSUPPORTED). */
typedef enum { RBMF_STAGE1_BASIS = 0, RBMF_STAGE1_TEMPLATES = 1 } rbmf_stage1_route;
rbmf_status rbmf_plan_enable_template_routes(rbmf_plan* plan, int32_t slab);
rbmf_status rbmf_set_templates(rbmf_plan* plan, const void* templates_dev, const float* sigma_dev);
rbmf_status rbmf_plan_set_stage1_route(rbmf_plan* plan, int32_t route);
rbmf_status rbmf_filter_flat(rbmf_plan* plan, const void* strain_dev, float thr, rbmf_trigger* out_dev,
                             int64_t* n_out_dev);

/* ---- Many sub-banks against one strain (the bank is split into 64 sub-banks of 6250 templates, each
 * with its own basis P^m and coefficients D^m; Table I :154-165: p = 64 / 254 / 200 ...) -------------------------------
 * A bank set groups fully set-up plans (workspace, basis, coefficients) that agree on N, fs and f_low; k, T, w, list
 * capacities and the stage-1 kernel may differ per sub-bank.  rbmf_bankset_filter filters one strain segment against
 * all of them: the sub-banks are launched most-expensive-first (cost 8 T k N / w) round-robin on up to four internal
 * streams forked from / joined to `cuda_stream`, so the short kernels and the tails of one sub-bank overlap the next;
 * all sub-banks append to ONE trigger list out_dev (capacity max_triggers) through one shared position counter
 * n_out_dev (device int64: total found, may exceed max_triggers), with template_id = (sum of T of the sub-banks before
 * it in `plans`) + the template's row in its own sub-bank.  The result equals the union of rbmf_filter over the plans.
 * Ordering: every sub-bank's work starts after what has been enqueued so far on `cuda_stream` (the producer of the
 * strain) AND on that plan's own stream (rbmf_set_basis / rbmf_set_coeffs, an earlier rbmf_filter); `cuda_stream`
 * continues after all sub-banks.  The plans' own streams are NOT made to wait for the bank-set call: the plans must not
 * be used by other calls while a bank-set call is in flight; the set does not own them (destroy the set first).  rbmf_bankset_get_counts synchronises and returns per-sub-bank candidates / triggers (arrays of n_plans,
 * may be NULL) and the total; RBMF_ERR_OVERFLOW if a sub-bank's candidate list overflowed. */
typedef struct rbmf_bankset rbmf_bankset;
rbmf_status rbmf_bankset_create(rbmf_bankset** out, rbmf_plan* const* plans, int32_t n_plans);
rbmf_status rbmf_bankset_filter(rbmf_bankset* set, const void* strain_dev, float thr_stage1, float thr_stage2,
                                rbmf_trigger* out_dev, int64_t max_triggers, int64_t* n_out_dev, void* cuda_stream);
rbmf_status rbmf_bankset_get_counts(rbmf_bankset* set, int64_t* n_candidates, int64_t* n_triggers, int64_t* n_total);
rbmf_status rbmf_bankset_destroy(rbmf_bankset* set);

/* ---- Preparation on the GPU (amortised: once per sub-bank) --------------------------
 * No plan is needed.  templates_dev: n_templates x (N/2+1) complex64, row-major, the (whitened, unit-norm) templates of
 * a sub-bank "stored row-wise" (:152); only the band [ceil(f_low N / fs), N/2) is used.
 * rbmf_prepare_basis: the covariance matrix C = T T^H (n_templates <= 32768), its k leading eigenvectors by
 * `iterations` steps of block power iteration with re-orthonormalisation from seeded random start vectors (the paper
 * used Lanczos; any orthonormal basis of the leading subspace serves the path equally), and the basis
 * P = orth(V^H T): basis_out_dev = k x (N/2+1) complex64 with orthonormal rows over the band and zeros outside -- the
 * input of rbmf_set_basis.  eig_out_dev (k floats or NULL): estimates of the k leading eigenvalues of C (the squared
 * singular values of T).  workspace_dev: 16-byte aligned device memory of rbmf_prepare_basis_workspace_bytes.
 * rbmf_prepare_coeffs: the decomposition coefficients D = T P^H (:167-169), coeffs_out_dev = n_templates x k complex64
 * (c_tk, unconjugated: the input of rbmf_set_coeffs) and sigma_out_dev (n_templates floats or NULL) = ||c_t||_2.
 * fp32 arithmetic with fp64 accumulation across blocks of 512 terms; both calls only enqueue on cuda_stream.
 * Repeatability: the Gram-Schmidt dot products and norms of rbmf_prepare_basis are fp64 sums collected with atomics
 * from several thread blocks once a row is longer than 4096 entries, so two runs with the same seed agree to fp32
 * rounding (last-bit differences), not necessarily bit for bit; rbmf_prepare_coeffs is bit-reproducible. */
rbmf_status rbmf_prepare_basis_workspace_bytes(int32_t n_templates, int32_t k, size_t* bytes);
rbmf_status rbmf_prepare_basis(const void* templates_dev, int32_t n_templates, int64_t N, double fs, double f_low,
                               int32_t k, int32_t iterations, uint64_t seed, void* workspace_dev, size_t workspace_bytes,
                               void* basis_out_dev, float* eig_out_dev, void* cuda_stream);
rbmf_status rbmf_prepare_coeffs(const void* templates_dev, int32_t n_templates, const void* basis_dev, int32_t k,
                                int64_t N, double fs, double f_low, void* coeffs_out_dev, float* sigma_out_dev,
                                void* cuda_stream);

/* Counts of the last rbmf_filter (synchronises the stream).  RBMF_ERR_OVERFLOW if a capacity was exceeded
 * (in RBMF_GEMM_SCREEN mode the capacity max_candidates applies to the screened superset, see
 * rbmf_get_screened_count, while *n_candidates reports the candidates confirmed at fp32 accuracy). */
rbmf_status rbmf_get_counts(rbmf_plan* plan, int64_t* n_candidates, int64_t* n_triggers);

/* Number of entries kernel 2 asked to write to the stage-1 list in the last rbmf_filter (synchronises): the number
 * max_candidates must hold.  In RBMF_GEMM_SCREEN mode this is the screened superset (>= the confirmed candidates of
 * rbmf_get_counts); in RBMF_GEMM_TCGEN05 mode it equals *n_candidates. */
rbmf_status rbmf_get_screened_count(rbmf_plan* plan, int64_t* n_screened);

/* Copy up to `capacity` first-stage candidates of the last rbmf_filter to out_host (synchronises).
 * *n_out = total candidates found. */
rbmf_status rbmf_get_candidates(rbmf_plan* plan, rbmf_candidate* out_host, int64_t capacity, int64_t* n_out);

/* Read-only device views of internal arrays for diagnostics and parity tests (valid after rbmf_filter on the
 * plan's stream, until the next call), in the library's blocked layouts:
 *   which = 0: beta, complex64, [segment][k/4 chunks][N samples][4 columns]: beta_c[n] of segment b at
 *              ((b k/4 + c/4) N + n) 4 + c%4  (max_batch segments; a single-segment plan has b = 0 only);
 *   which = 1 / 2: beta^avg hi / lo plane, bfloat16, [ceil(k/32) K blocks][max_batch N/w bins][32 columns][re, im]
 *                  (value = hi + lo; columns >= k of the last block are zero).  In RBMF_GEMM_SCREEN mode plane 1
 *                  holds ONE float16 rounding of beta^avg in the same layout and plane 2 is stale.
 *   which = 3: the stage-1 list as kernel 2 wrote it (rbmf_candidate records, min(rbmf_get_screened_count,
 *              max_candidates) valid entries; *bytes = capacity in bytes).  In RBMF_GEMM_SCREEN mode avg_re/avg_im are
 *              the raw one-product fp16 tensor-core values R_16 the screen tested;
 *   which = 4: bin_norm, float32[max_batch N/w]: the upper bounds of ||beta^avg[i]||_2 the screen's error bound used;
 *   which = 5: tnorm_blk, float32[ceil(T/128)]: max_t ||c_t||_2 / sigma_t per block of 128 templates;
 *   which = 6: the final first-stage candidate list of the last rbmf_filter on the device (what rbmf_get_candidates
 *              copies; min(n_candidates, max_candidates) valid rbmf_candidate records; *bytes = capacity in bytes).
 * *dev_ptr receives the address, *bytes the size. */
rbmf_status rbmf_get_internal(rbmf_plan* plan, int32_t which, const void** dev_ptr, size_t* bytes);

/* Per-stage GPU time of the last rbmf_filter, in milliseconds (synchronises): ms[0] = a1-a3 (FFT stage),
 * ms[1] = a4-a5 (GEMM + threshold), ms[2] = a6 (stage 2), ms[3] = whole call.  Timing events are recorded
 * only after rbmf_plan_set_timing(plan, 1). */
rbmf_status rbmf_plan_set_timing(rbmf_plan* plan, int32_t enabled);
rbmf_status rbmf_get_stage_ms(rbmf_plan* plan, float ms[4]);
/* The same for an earlier call: the plan keeps the stage events of its last 64 timed calls, so a loop of up to 64
 * rbmf_filter calls can be enqueued WITHOUT a host round trip per call and its per-stage times read afterwards.
 * calls_back = 0 is the last call, 1 the one before, ... (RBMF_ERR_ARG beyond 63, RBMF_ERR_STATE beyond the number of
 * calls made since rbmf_plan_set_timing, which restarts the history).  Synchronises on the last call. */
rbmf_status rbmf_get_stage_ms_history(rbmf_plan* plan, int32_t calls_back, float ms[4]);

/* Number of kernels rbmf_filter launches for this plan's configuration. */
rbmf_status rbmf_launches_per_filter(const rbmf_plan* plan, int32_t* n);

rbmf_status rbmf_plan_destroy(rbmf_plan* plan);

const char* rbmf_status_string(rbmf_status status);
/* Last cudaError_t / CUresult seen by this plan (0 if none). */
int32_t rbmf_last_cuda_error(const rbmf_plan* plan);

/* ---- Diagnostics: test-only switches, not product modes -------------------------------------------------------
 * rbmf_diag_set(plan, option, value), any time after rbmf_plan_create:
 *   RBMF_DIAG_STAGE1_FP32_CHECK (value 0/1): run steps a4-a5 with a plain fp32 CUDA-core kernel on the bf16 hi + lo
 *       operands instead of the tensor-core kernel selected by rbmf_plan_set_gemm_impl (cross-check of the two
 *       tensor-core kernels against ordinary arithmetic; orders of magnitude slower);
 *   RBMF_DIAG_SINGLE_CTA_SCREEN (value 0/1): RBMF_GEMM_SCREEN uses its single-CTA kernel instead of the 2-CTA
 *       cluster kernel that multicasts the coefficient tile (the fallback for devices that cannot co-schedule
 *       clusters of 2); takes effect at the next rbmf_filter;
 *   RBMF_DIAG_STAGE2_PER_CANDIDATE (value 0/1): step a6 with the one-warp-per-candidate kernel (the fallback for
 *       w = 32 with k > 608, where one bin's block of beta does not fit in shared memory) instead of the kernel that
 *       regroups the candidates by bin.
 * Scheduling overrides (results are unchanged, only the order of the work; they replace the RBMF_FFT_SEG_MAJOR,
 * RBMF_FFT_LOOKAHEAD and RBMF_GEMM_GROUP environment variables of earlier builds -- the library reads no environment
 * variable any more); they take effect at the next rbmf_filter:
 *   RBMF_DIAG_FFT_CHUNK_MAJOR (value 0/1): a batch's FFT work runs basis-chunk-major (a chunk of 4 basis columns is
 *       read once for all segments) instead of segment-major, the measured-faster default;
 *   RBMF_DIAG_FFT_LOOKAHEAD (value 1..256, 0 = automatic): basis chunks whose first FFT pass may run ahead of the
 *       second pass in kernel 1's work queue (their intermediates must fit in L2);
 *   RBMF_DIAG_GEMM_GROUP (value >= 1, 0 = automatic): template blocks per raster group of kernel 2 (the group's
 *       coefficient tiles stay L2-resident while the beta^avg planes stream past once per group). */
typedef enum {
    RBMF_DIAG_STAGE1_FP32_CHECK = 1,
    RBMF_DIAG_SINGLE_CTA_SCREEN = 2,
    RBMF_DIAG_STAGE2_PER_CANDIDATE = 3,
    RBMF_DIAG_FFT_CHUNK_MAJOR = 4,
    RBMF_DIAG_FFT_LOOKAHEAD = 5,
    RBMF_DIAG_GEMM_GROUP = 6
} rbmf_diag_option;
rbmf_status rbmf_diag_set(rbmf_plan* plan, int32_t option, int32_t value);

#ifdef __cplusplus
}
#endif
#endif /* RBMF_H */
