/* nsgpu.h -- C ABI of the B200-native batched-likelihood + nested-slice-sampling library.
 *
 * Hot path of arXiv 2509.13307 (Lovick, Yallup, Piras, Spurio Mancini, Handley), cited as
 * P:L<line> of /root/reference/PAPER.md, with BASELINE.json north_star (BJ) for the kernel-level
 * definition.  Steps a1..a14 refer to SURVEY.md section 8(a) / DESIGN.md section 2.
 *
 * Conventions (all entry points)
 *  - Every call returns an nsgpu_status; nothing throws or aborts across this boundary.
 *    nsgpu_last_error(ctx) returns a ctx-owned, NUL-terminated description of the last failure.
 *  - "HOST" / "DEVICE" beside a pointer says where the memory lives.  DEVICE pointers are owned by
 *    the caller (e.g. torch tensors) and must be on the ctx's device; `stream` is a cudaStream_t
 *    passed as void* (NULL = the legacy default stream).  Calls taking a stream are asynchronous on
 *    it unless stated otherwise.
 *  - nsgpu_create copies every HOST input (the caller may free them on return) and owns all device
 *    workspaces until nsgpu_destroy.  Batch calls never allocate.  A ctx is not thread-safe.
 *  - Layouts are row-major and densely packed.  theta, u: float32; log L and all evidence
 *    quantities: float64 (reading P1: fp32 operands in the heavy stages, fp64 for the chi^2
 *    reduction, log L and every nested-sampling accumulator).
 *  - There is no CPU fallback anywhere: without a CUDA device nsgpu_create fails with NSGPU_ECUDA.
 */
#ifndef NSGPU_H
#define NSGPU_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__GNUC__)
#define NSGPU_API __attribute__((visibility("default")))
#else
#define NSGPU_API
#endif

typedef struct nsgpu_ctx nsgpu_ctx; /* opaque; one per (model, GPU) */

typedef enum {
  NSGPU_OK = 0,
  NSGPU_EINVAL = -1,  /* NULL pointer, bad enum, inconsistent sizes */
  NSGPU_ENOMEM = -2,  /* host or device allocation failed */
  NSGPU_ECUDA = -3,   /* a CUDA runtime/driver call failed (text in nsgpu_last_error) */
  NSGPU_ESHAPE = -4,  /* B > max_batch, n_live > max_batch, unsupported dimension */
  NSGPU_ENOTSPD = -5, /* Cholesky factor has a non-positive or non-finite diagonal */
  NSGPU_ENOCONV = -6  /* nsgpu_run hit max_iter before the termination criterion (result still filled) */
} nsgpu_status;

/* ---- prior (step a1; Table 1; reading N1) ------------------------------------------
 * The sampler works in the unit hypercube u in [0,1]^D; this table is the per-dimension transform
 *   kind 0 uniform : theta = p0 + (p1 - p0) u        (p0 = a, p1 = b)
 *   kind 1 gaussian: theta = p0 + p1 Phi^-1(u)       (p0 = mu, p1 = sigma)                      */
typedef struct {
  int32_t kind;
  double p0, p1;
} nsgpu_prior1d;

/* ---- one emulator (steps a2-a4; BJ: "dense layers with the gated activation
 * (beta + sigma(alpha x)(1 - beta)) x, then de-standardisation of log-spectra") ----------------
 * n_in -> n_hidden x width -> n_out.  All arrays HOST float32, copied at create.
 * W[l]: [fan_in][fan_out] row-major (y = x.W + b), l = 0..n_hidden; b[l]: [fan_out];
 * alpha[l], beta[l]: [width] per hidden layer (reading E1); inputs standardised (x - in_mean)/in_std;
 * output y = (h.W + b) * out_std + out_mean; out_kind 0: spectrum = y, 1: spectrum = 10^y (E2).   */
typedef struct {
  int32_t n_in, n_hidden, width, n_out, out_kind;
  const float* const* W;
  const float* const* b;
  const float* const* alpha;
  const float* const* beta;
  const float* in_mean;
  const float* in_std;
  const float* out_mean;
  const float* out_std;
} nsgpu_emulator;

/* ---- theory stage after the emulator(s) (steps a5-a9) ------------------------------------------
 * kind 0 identity     : model = theta                       (n_data = D; sampler validation, BJ cfg 0)
 * kind 1 emulator     : model = emulator 0 spectrum         (BJ cfg 0)
 * kind 2 cmb_binned   : s = [spectrum_0 | spectrum_1 | ...] / theta[cal_index]^2, model = Bin . s with
 *                       Bin a CSR matrix n_data x (n_emu * n_out)            (BJ cfg 1; readings C1-C3)
 * kind 3 shear_limber : eqs. A1-A4 on n_chi quadrature nodes evenly spaced in the scale
 *                       factor, the emulated log10 P(k, z) interpolated linearly in z and
 *                       log10 k, optional cubic z-spline n_z_emu -> n_z first (BJ cfg 3b)
 * kind 4 cmb_tt_cv   : the paper's own CMB likelihood: nu_l Chat_l / C_l ~ chi^2_{nu_l}, nu_l = 2 l + 1,
 *                       independently per multipole l = ell_min + i; emulator 0 gives C_l = 10^y (out_kind 1),
 *                       `data` holds the observed Chat_l > 0, n_data = n_out, `chol` is not used (may be NULL);
 *                       log L = sum_l log[(nu_l / C_l) f_chi2(nu_l Chat_l / C_l; nu_l)]
 * Emulator-input assembly (step a2): emulator input j < n_theta_in is theta[emu_in_idx[j]], or the
 * constant emu_in_const[j] where emu_in_idx[j] < 0; a shear emulator has n_in = n_theta_in + 1, its
 * last input being the redshift of the node.  Other kinds: n_in = n_theta_in.
 * All pointers HOST, copied at create.                                                            */
typedef struct {
  int32_t kind;
  int32_t n_theta_in;
  const int32_t* emu_in_idx;  /* [n_theta_in] */
  const double* emu_in_const; /* [n_theta_in] */
  /* kind 2 */
  const int32_t* bin_ptr; /* [n_data + 1] */
  const int32_t* bin_col; /* [nnz] */
  const float* bin_val;   /* [nnz] */
  int32_t cal_index;
  /* kind 4 */
  int32_t ell_min;
  /* kind 3 */
  int32_t n_z_emu, n_z, n_chi, n_k, n_ell, n_tomo;
  int32_t z_interp; /* 0: n_z == n_z_emu, no spline; 2: cubic not-a-knot spline n_z_emu -> n_z */
  double z_max, k_min, k_max;
  const double* ell;     /* [n_ell] multipoles the spectra are evaluated at (reading S7) */
  const double* nz_mean; /* [n_tomo] Gaussian n_i(z) means */
  double nz_sigma;
  /* where each physical parameter sits in theta (reading S2); < 0: w0 = -1, wa = 0, eta0 = 0.7 */
  int32_t idx_omega_b, idx_omega_cdm, idx_h, idx_w0, idx_wa, idx_eta0;
  int32_t idx_dz; /* first of n_tomo photo-z shifts */
  int32_t idx_ia; /* first of n_ia_terms n_tomo IA coefficients, bin-major (reading S2) */
  int32_t idx_m;  /* first of n_m_terms n_tomo shear-calibration coefficients, bin-major (S2) */
  /* coefficients per bin: A_i(z) = A_i0 + A_i1 x + A_i2 x^2 truncated after n_ia_terms in 1..3, m_i(l) = m_i0 +
   * m_i1 ln(l/550)/ln 30 after n_m_terms in 1..2.  (1, 1) is the paper's one amplitude and one bias per bin
   * (P:L344, L350); (3, 2) the BASELINE.json configs[2..4] layout.                                        */
  int32_t n_ia_terms, n_m_terms;
} nsgpu_theory;

/* flags for nsgpu_create */
#define NSGPU_MLP_AUTO 0u   /* tcgen05 tensor-core MLP where the shape allows it, SIMT otherwise */
#define NSGPU_MLP_SIMT 1u   /* fp32 CUDA-core MLP (on-device correctness reference) */
#define NSGPU_MLP_TC 2u     /* require the tcgen05 path (NSGPU_ESHAPE if width % 64 != 0) */
#define NSGPU_CHI2_STREAMED 8u /* chi^2 by the factor-streaming kernel (one CTA = all rows of 8..32 thetas) whatever n_data */
#define NSGPU_CHI2_TILED 16u   /* chi^2 by the tiled kernels (128-row blocks x 32..64 thetas) whatever n_data; default: n_data >= 512 */
#define NSGPU_MLP_CLUSTER 32u    /* tcgen05 GEMMs: CTA pairs that multicast the weight tiles, whatever the batch (default: large batches) */
#define NSGPU_MLP_NO_CLUSTER 64u /* ... never */
#define NSGPU_SHEAR_STREAM 4u /* kind 3: use the streaming projection kernels even where the grids fit shared memory */
#define NSGPU_MLP_FUSED 256u   /* tcgen05 path: one persistent kernel for all layers (CTA pairs own row blocks, activations in an
                                * L2-resident scratch) wherever the shape allows it (width 512, even n_hidden, n_in 6/7/9);
                                * bit-identical to the layered path; opt-in (measured no faster: profiles/r2_fused_mlp.md) */
#define NSGPU_MLP_LAYERED 512u /* one kernel per layer, activations through HBM (the default) */
#define NSGPU_MLP_FP64 1024u   /* precision study: CUDA-core MLP with fp64 activations and accumulation (fp32 weights as
                                * given, fp32 spectrum table); implies the SIMT path */
#define NSGPU_MLP_SPLIT4 2048u /* precision study: tcgen05 path with the fourth product lo.lo added (16 MMAs per k-block, not 12) */
#define NSGPU_NO_OVERLAP 4096u  /* kind 3: keep the theta-only half of the projection on the caller's stream (default: batches of
                                 * at most 1024 run it on a side stream, under the emulator kernels) */
#define NSGPU_NO_PDL 128u /* launch every kernel with plain stream ordering (default: the kernels of a likelihood call and of a
                            * slice-sampling round are chained by programmatic dependent launch) */

/* Create a context on CUDA device `device`.
 * data [n_data] and chol [n_data][n_data] (lower Cholesky factor of the data covariance, row-major,
 * upper triangle ignored; reading L2) are HOST float64.  max_batch bounds B of every batch call and
 * n_live/n_delete of the sampler calls.  Errors: EINVAL, ESHAPE, ENOTSPD, ENOMEM, ECUDA.           */
NSGPU_API nsgpu_status nsgpu_create(nsgpu_ctx** out, int32_t D, const nsgpu_prior1d* prior, int32_t n_emu,
                          const nsgpu_emulator* emu, const nsgpu_theory* theory, int32_t n_data,
                          const double* data, const double* chol, int32_t max_batch, int32_t device,
                          uint32_t flags);
NSGPU_API nsgpu_status nsgpu_destroy(nsgpu_ctx* ctx);
NSGPU_API const char* nsgpu_last_error(const nsgpu_ctx* ctx); /* ctx == NULL: error text of the last failed create */

/* a1: theta[B][D] = T(u[B][D]); DEVICE float32 both. */
NSGPU_API nsgpu_status nsgpu_prior_transform(nsgpu_ctx* ctx, const float* u, int32_t B, float* theta, void* stream);

/* a2-a10, the bulk likelihood evaluation: logL[B] (DEVICE float64) for theta[B][D] (DEVICE
 * float32, physical units).  theta outside the support of a uniform prior, or a non-finite model,
 * gives -inf, never NaN.  log L includes the Gaussian normalisation -1/2 ln det(2 pi C) (reading L1). */
NSGPU_API nsgpu_status nsgpu_loglike_batch(nsgpu_ctx* ctx, const float* theta, int32_t B, double* logL, void* stream);

/* Same computation with HOST buffers: copies theta to the device, evaluates, copies logL back and
 * returns when logL is valid (synchronous).  This is the end-to-end entry bench.py times.           */
NSGPU_API nsgpu_status nsgpu_loglike_batch_host(nsgpu_ctx* ctx, const float* theta_host, int32_t B, double* logL_host);

/* Stage taps for parity tests (DEVICE buffers).
 * emulate: spectrum of emulator `emu` for every theta: out [B][rows][n_out] float32, rows = n_z_emu
 *          for kind 3 and 1 otherwise; 10^y applied where out_kind = 1.
 * theory : model vectors [B][n_data] float64 (the input of the chi^2 stage).                        */
NSGPU_API nsgpu_status nsgpu_emulate_batch(nsgpu_ctx* ctx, int32_t emu, const float* theta, int32_t B, float* out, void* stream);
NSGPU_API nsgpu_status nsgpu_theory_batch(nsgpu_ctx* ctx, const float* theta, int32_t B, double* model, void* stream);

/* a11-a12 (+a14): evolve n_chains constrained slice-sampling chains (Neal 2003) for n_steps
 * moves each under log L > logL_star, started from rows start_idx[c] of the live set, directions drawn
 * from the live-set covariance (reading N3).  u_live [n_live][D] float32, logL_live [n_live] float64,
 * start_idx [n_chains] int32, u_out [n_chains][D] float32, logL_out [n_chains] float64: all DEVICE.
 * n_evals (HOST, optional): number of likelihood evaluations spent.  `iteration` and `seed` select the
 * Philox streams (reading N10).  Synchronises `stream` before returning.  Errors: EINVAL (NULL pointer, n_live < D + 1,
 * a start index outside [0, n_live)), ESHAPE (sizes above max_batch), ENOTSPD (live covariance not positive definite). */
NSGPU_API nsgpu_status nsgpu_slice_step(nsgpu_ctx* ctx, const float* u_live, const double* logL_live, int32_t n_live,
                              const int32_t* start_idx, int32_t n_chains, double logL_star, int32_t n_steps,
                              uint64_t seed, int32_t iteration, float* u_out, double* logL_out,
                              int64_t* n_evals, void* stream);

typedef struct {
  int32_t n_live, n_delete, n_steps; /* BJ cfg 4: 1000, 500, 5 D */
  double stop_frac;                  /* stop when Z_live / (Z + Z_live) < stop_frac (reading N7) */
  int64_t max_iter;
  uint64_t seed;
} nsgpu_run_opts;

typedef struct {
  double logZ, logZ_err, logZ_err_analytic, H; /* eq. 1; error bar per reading N9 */
  int64_t n_iter, n_dead, n_like_evals, n_rounds, n_failed_moves;
  double seconds; /* wall time of the run, host clock */
  double seconds_sampling, seconds_summary; /* ... split: the nested-sampling loop | final log Z, H, error bar, samples */
  int64_t n_nonfinite_rows; /* emulator rows whose output was not finite during this run (tcgen05 path: |h| >= 4094 overflows the
                             * fp16 activation planes).  Such proposals count as log L = -inf, i.e. as
                             * excluded prior volume: a non-zero value means log Z may be biased -- rerun with NSGPU_MLP_SIMT. */
} nsgpu_result;

/* a1-a14: the whole nested-sampling run.  Samples go to caller-allocated HOST buffers of
 * capacity `cap` rows (may be NULL with cap = 0): theta [cap][D] float32, logL [cap], logw [cap]
 * float64 with logw = log(L_i w_i / Z); *n_samples returns n_dead + n_live (the number
 * needed); min(cap, needed) rows are written.  Returns NSGPU_ENOCONV if max_iter was reached.
 * Blocking.  The run works on a non-blocking stream the context owns: a context is not thread-safe, but runs on
 * DIFFERENT contexts may be driven from different host threads at once and then share the GPU (a single run keeps
 * it only partly busy: batches of <= n_delete proposals); each returns exactly what it returns alone.        */
NSGPU_API nsgpu_status nsgpu_run(nsgpu_ctx* ctx, const nsgpu_run_opts* opts, nsgpu_result* res, float* theta_samples,
                       double* logL_samples, double* logw_samples, int64_t cap, int64_t* n_samples);

/* n_runs independent runs (seeds[r] replaces opts->seed) of the SAME model that share every likelihood batch: a single run
 * carries <= n_delete proposals per round and leaves the GPU half idle ("perfect scaling is hard to achieve"); here
 * the chains of all runs advance in the same rounds, each with its own L*, direction factor, Philox key and stopping test,
 * so res[r] (HOST [n_runs]) is exactly what nsgpu_run returns for seeds[r] (bit for bit; n_rounds and the wall times are
 * those of the shared loop).  Needs n_runs * n_delete <= max_batch.  Samples of run r: nsgpu_multi_samples (same buffers
 * and meaning as nsgpu_last_samples).  Returns NSGPU_ENOCONV if any run hit max_iter.  Blocking.                     */
NSGPU_API nsgpu_status nsgpu_run_multi(nsgpu_ctx* ctx, const nsgpu_run_opts* opts, int32_t n_runs, const uint64_t* seeds,
                                       nsgpu_result* res);
NSGPU_API nsgpu_status nsgpu_multi_samples(nsgpu_ctx* ctx, int32_t run, float* theta_samples, double* logL_samples,
                                           double* logw_samples, int64_t cap, int64_t* n_samples);

/* The error bar of log Z by 1000 simulated prior-volume sequences (reading N9) -- the same kernel and the
 * same arithmetic as the summary of nsgpu_run, but this entry point ALLOCATES NOTHING (no cudaMalloc / cudaFree, no
 * allocating library routine): for callers under CUDA graph capture, in tight serving loops, or in harnesses that forbid
 * allocation.  Its scratch (the dead sequence, the live block, the 1000 results) is a file-scope device array of
 * 1,048,576 + 16,384 + 1000 doubles = 8.1 MiB that every GPU loading the library holds until the process exits.
 * dead_logL [n_dead] (in deletion order), live_logL [n_live]: HOST float64; n_delete = points deleted per iteration
 * (point i had n_live - i mod n_delete live points); seed: the run's seed (same Philox streams as nsgpu_run, so for
 * the sequence of a finished run *logZ_err equals nsgpu_result.logZ_err).  *logZ_err HOST out; logZ_sims HOST [1000]
 * out or NULL.  Errors: EINVAL (NULL, sizes), ESHAPE when n_dead > 1,048,576 or n_live > 16,384.  Blocking (synchronises
 * `stream`).  All calls share the one array: calls that overlap on the GPU (two streams, two host threads) race. */
NSGPU_API nsgpu_status nsgpu_logz_error_noalloc(nsgpu_ctx* ctx, const double* dead_logL, int64_t n_dead,
                                                const double* live_logL, int32_t n_live, int32_t n_delete, uint64_t seed,
                                                double* logZ_err, double* logZ_sims, void* stream);

/* Multi-GPU nested sampling: one process per GPU, every rank holds the whole
 * live set and calls this with the same options.  Rank r evolves the chains nsgpu_shard_range gives it; the only
 * exchange of an iteration is an all-gather of the k new points, done through `allgather`: send and recv are DEVICE
 * pointers, every rank contributes bytes_per_rank bytes and receives world * bytes_per_rank bytes ordered by rank
 * (the layout of ncclAllGather); it must have completed, or be ordered on `stream`, when it returns; non-zero =
 * failure.  The Philox streams are keyed by the GLOBAL chain index, so the result does not depend on `world`:
 * every rank returns the same nsgpu_result, equal to nsgpu_run's.  n_like_evals is the total over ranks.         */
typedef int32_t (*nsgpu_allgather_fn)(void* user, const void* send, void* recv, int64_t bytes_per_rank, void* stream);
NSGPU_API nsgpu_status nsgpu_run_sharded(nsgpu_ctx* ctx, const nsgpu_run_opts* opts, int32_t rank, int32_t world,
                               nsgpu_allgather_fn allgather, void* user, nsgpu_result* res, float* theta_samples,
                               double* logL_samples, double* logw_samples, int64_t cap, int64_t* n_samples);
/* chains [*first, *first + *count) of n_chains belong to `rank`: contiguous blocks of ceil(n_chains / world). Host only. */
NSGPU_API void nsgpu_shard_range(int32_t n_chains, int32_t rank, int32_t world, int32_t* first, int32_t* count);

/* Samples of the last nsgpu_run on this ctx (kept until the next run or destroy): same buffers and
 * meaning as nsgpu_run's; *n_samples returns the number available; cap = 0 only queries the count. */
NSGPU_API nsgpu_status nsgpu_last_samples(nsgpu_ctx* ctx, float* theta_samples, double* logL_samples,
                                          double* logw_samples, int64_t cap, int64_t* n_samples);

/* a13 tap: delete the k lowest of logL_live [n_live] (DEVICE), accumulate the evidence starting from
 * (*logX, *logZ) (HOST in/out).  dead_idx [k] int32, logw [k] float64 (DEVICE out); *logL_star HOST. */
NSGPU_API nsgpu_status nsgpu_delete_lowest(nsgpu_ctx* ctx, const double* logL_live, int32_t n_live, int32_t k,
                                 double* logX, double* logZ, int32_t* dead_idx, double* logw,
                                 double* logL_star, void* stream);

/* a14 tap: lower Cholesky factor [D][D] (DEVICE float64) of the sample covariance of u_live + 1e-12 I. */
NSGPU_API nsgpu_status nsgpu_live_cholesky(nsgpu_ctx* ctx, const float* u_live, int32_t n_live, double* L_out, void* stream);

/* RNG tap: out[n][4] = Philox4x32-10(ctr[n][4], key[2]) (DEVICE uint32 in/out; key HOST). */
NSGPU_API nsgpu_status nsgpu_debug_philox(nsgpu_ctx* ctx, const uint32_t* ctr, int32_t n, const uint32_t* key, uint32_t* out, void* stream);

/* Per-stage device timing with CUDA events recorded on the caller's stream around the library's own
 * launches (for roofline accounting; off by default).  Stages: 0 first emulator layer (a2+a3),
 * 1 hidden-layer GEMMs (a3; the whole MLP when it is the fused kernel), 2 output-layer GEMM (a4), 3 shear projection
 * (a5-a8; without NSGPU_NO_OVERLAP only the half that reads the table: the theta-only half runs on a side stream under
 * the MLP stages), 4 CMB binning (a9),
 * 5 chi^2 (a10), 6 slice round + compaction (a11-a12), 7 identity/emulator copy.
 * nsgpu_stage_times synchronises the device, adds the elapsed times since the last call into
 * ms[8] / count[8] (HOST, overwritten) and resets the accumulators.                                 */
#define NSGPU_N_STAGES 8
NSGPU_API nsgpu_status nsgpu_set_profiling(nsgpu_ctx* ctx, int32_t on);
NSGPU_API nsgpu_status nsgpu_stage_times(nsgpu_ctx* ctx, double* ms, int64_t* count);

/* Counters of the last nsgpu_slice_step on this ctx (HOST out, either may be NULL): slice moves that reached the shrink
 * cap and stayed at their start point (reading N3: step-out cap 32, shrink cap 64), and likelihood rounds taken. */
NSGPU_API nsgpu_status nsgpu_sampler_counters(const nsgpu_ctx* ctx, int64_t* n_failed_moves, int64_t* n_rounds);

/* SM clock measured on the device between the steps of a timed region (bench.py's `clocks` record).  `mark` enqueues
 * on `stream` a tiny kernel whose blocks record the cycle counter and the global nanosecond timer of their SM (one
 * launch, ~3 us, nothing stays resident; at most 512 marks between reads).  `read` synchronises the device and returns,
 * for each pair of consecutive marks, the mean SM clock in MHz (cycles over time per SM, averaged over the SMs seen in
 * both) and the end time of the interval in ms since the first mark; HOST [cap], either may be NULL; it clears the marks. */
NSGPU_API nsgpu_status nsgpu_clock_mark(nsgpu_ctx* ctx, void* stream);
NSGPU_API nsgpu_status nsgpu_clock_marks_read(nsgpu_ctx* ctx, double* sm_mhz, double* t_ms, int32_t cap, int32_t* n_intervals);

/* Introspection: 0 = SIMT, 1 = tcgen05 for emulator `emu`; kernels launched since create. */
NSGPU_API int32_t nsgpu_mlp_path(const nsgpu_ctx* ctx, int32_t emu);
NSGPU_API int64_t nsgpu_launch_count(const nsgpu_ctx* ctx);
/* Emulator rows (tcgen05 path) whose output-layer accumulators were not finite since create (synchronises the device;
 * -1 on error).  The tcgen05 path carries hidden activations as fp16 hi/lo of 16 h, so |h| >= 4094 overflows (DESIGN.md
 * section 6); such rows, like rows of a non-finite theta, end as log L = -inf -- this counter makes that visible.
 * Trained weights that trip it should run with NSGPU_MLP_SIMT (fp32 activations).                                  */
NSGPU_API int64_t nsgpu_nonfinite_rows(nsgpu_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* NSGPU_H */
