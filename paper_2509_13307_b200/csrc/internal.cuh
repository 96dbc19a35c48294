// internal.cuh -- context layout and launch helpers shared by the nsgpu translation units.
// Not part of the public boundary (include/nsgpu.h is).
#pragma once

#include <cuda_runtime.h>
#include <cuda_fp16.h>
#include <nvtx3/nvToolsExt.h>
#include <stdint.h>

#include <algorithm>
#include <cstring>
#include <utility>
#include <map>
#include <string>
#include <vector>

#include "../../include/nsgpu.h"

#define NSGPU_MAX_LAYERS 8   // n_hidden + 1 <= 8
#define NSGPU_MAX_IN 16      // emulator inputs
#define NSGPU_MAX_TOMO 10
#define NSGPU_N_STAGES 8
#define NSGPU_MAX_D 64       // sampler dimension (one warp per chain, two dims per lane)

struct EmuDev {
  int n_in = 0, n_hidden = 0, width = 0, n_out = 0, out_kind = 0;
  float* W[NSGPU_MAX_LAYERS] = {};      // fp32 [fan_in][fan_out]
  float* b[NSGPU_MAX_LAYERS] = {};
  float* alpha[NSGPU_MAX_LAYERS] = {};
  float* beta[NSGPU_MAX_LAYERS] = {};
  float *in_mean = nullptr, *in_std = nullptr, *out_mean = nullptr, *out_std = nullptr, *out_zero = nullptr;
  int path = 0;                         // 0 SIMT, 1 tcgen05
  // tcgen05 path: weights of layers 1..n_hidden as fp16 hi/lo, [fan_out_padded][fan_in] (K-major),
  // scaled by 2^wexp[l] (see mlp_tc.cu)
  __half* Whi[NSGPU_MAX_LAYERS] = {};
  __half* Wlo[NSGPU_MAX_LAYERS] = {};
  float wscale_inv[NSGPU_MAX_LAYERS] = {};
  int n_out_pad = 0;
  void* tmaps = nullptr;                // host array of CUtensorMap (opaque here)
};

struct ShearDev {
  int n_z_emu = 0, n_z = 0, n_chi = 0, n_k = 0, n_ell = 0, n_tomo = 0, n_tap = 0;
  double z_max = 0, k_min = 0, k_max = 0, lk0 = 0, dlk = 0, da = 0, nz_sigma = 0;
  double *a_q = nullptr, *z_q = nullptr, *ln1pz = nullptr;   // [n_chi]
  double *lellh = nullptr, *lf = nullptr;                    // [n_ell] log10(ell + 1/2), ln(ell/550)/ln 30
  int* tap_start = nullptr;                // [n_chi] first emulator z node used by node q
  double* tap_w = nullptr;                 // [n_chi][n_tap] z-interpolation weights (spline folded in)
  double *ell = nullptr, *nz_mean = nullptr;
  double* mu_k = nullptr;                  // [n_k] emulator mu_out in fp64 (the spectrum table holds y - mu_out)
  double* aux = nullptr;                   // [max_batch][(3 + n_tomo) n_chi] hand-off between the two projection kernels
  double* pg = nullptr;                    // streaming path: [max_batch][n_ell][n_chi rounded up to even] P g_q
  int idx_omega_b = -1, idx_omega_cdm = -1, idx_h = -1, idx_w0 = -1, idx_wa = -1, idx_eta0 = -1;
  int idx_dz = -1, idx_ia = -1, idx_m = -1, n_ia_terms = 3, n_m_terms = 2;
  bool streaming = false;                  // chunked projection kernels (grids too large for the resident one, or forced)
};

struct SamplerDev;  // sampler.cu

struct nsgpu_ctx {
  int device = 0, D = 0, n_emu = 0, n_data = 0, max_batch = 0, kind = 0;
  uint32_t flags = 0;
  int rows_per_theta = 1;       // n_z_emu for shear, 1 otherwise
  int n_theta_in = 0;
  int sm_count = 148;
  // prior
  int* prior_kind = nullptr;
  double *prior_p0 = nullptr, *prior_p1 = nullptr;
  // emulator input assembly
  int* emu_in_idx = nullptr;
  double* emu_in_const = nullptr;
  float* z_emu = nullptr;       // [n_z_emu] emulator redshift nodes (fp32 inputs of the net)
  std::vector<EmuDev> emu;
  // cmb
  int *bin_ptr = nullptr, *bin_col = nullptr;
  float* bin_val = nullptr;
  int cal_index = -1, n_spec_cols = 0;
  ShearDev sh;
  // gaussian
  double* data = nullptr;       // [n_data]
  double* Linv = nullptr;       // [n_data][n_data] TRANSPOSE of the inverse Cholesky factor: LinvT[j][i], fp64
  int linv_ld = 0;              // row stride of Linv (doubles): >= n_data, 8 mod 16
  double log_norm = 0.0;
  double *tt_a = nullptr, *tt_b = nullptr, *tt_mu = nullptr;   // kind 4: (nu/2) ln 10 and nu Chat / 2 per multipole
  // workspaces
  void* act[2] = {nullptr, nullptr};   // [M_max][width] fp32 (SIMT) or 2 x fp16 (tcgen05)
  void* fused_scratch = nullptr;       // fused MLP kernel: per-cluster activation scratch (L2-resident), shared by the emulators
  float* spec = nullptr;               // [n_emu][M_max][spec_ld] de-standardised y (log10 where exp10)
  int spec_ld = 0;                     // row stride: n_out, rounded up to 4 floats for one-row-per-theta tables (16-byte stores)
  bool spec_kz = false;                // shear + tcgen05: per theta [n_k][n_z_emu] instead of [n_z_emu][n_k]
  double* model = nullptr;             // [max_batch][n_data]
  double* resid_t = nullptr;           // [n_data][max_batch rounded up to 64] model - data, transposed (chi^2 operand)
  double* chi2_part = nullptr;         // [row blocks of 128][max_batch rounded up to 64] partial sums of w^2
  float* theta_stage = nullptr;        // [max_batch][D] device staging for the host entry
  double* logL_stage = nullptr;
  float* theta_pinned = nullptr;       // pinned host staging
  double* logL_pinned = nullptr;
  SamplerDev* sampler = nullptr;
  void* probe = nullptr;               // clock probe state (probe.cu)
  cudaStream_t side_stream = nullptr;  // shear: the theta-only half of the projection runs here, under the emulator kernels
  cudaEvent_t ev_in = nullptr, ev_side = nullptr;
  cudaStream_t emu_stream[8] = {};     // kind 2: emulators 1.. run on streams of their own, concurrently with emulator 0
  cudaEvent_t emu_done[8] = {};
  std::string err;
  int64_t launches = 0;
  unsigned long long* nonfinite_rows = nullptr;   // device counter: emulator rows with non-finite output (tcgen05 path)
  // optional per-stage CUDA-event timing (nsgpu_set_profiling / nsgpu_stage_times)
  bool profiling = false;
  struct StageEv { int stage; cudaEvent_t a, b; };
  std::vector<StageEv> stage_events;
  std::vector<cudaEvent_t> event_pool;
  double stage_ms[NSGPU_N_STAGES] = {};
  int64_t stage_count[NSGPU_N_STAGES] = {};
};

// RAII stage timer: records an event pair on `st` around the enclosed launches when profiling is on, inside an NVTX range
// named after the stage (header-only NVTX3: a no-op unless a tool that collects NVTX is attached, e.g. `ncu --nvtx`)
static const char* const NSGPU_STAGE_NAMES[NSGPU_N_STAGES] = {"nsgpu:mlp_first", "nsgpu:mlp_hidden", "nsgpu:mlp_out", "nsgpu:shear_project",
                                                              "nsgpu:cmb_bin", "nsgpu:chi2", "nsgpu:slice_round", "nsgpu:copy_model"};
struct StageTimer {
  nsgpu_ctx* ctx; cudaStream_t st; int idx = -1;
  StageTimer(nsgpu_ctx* c, int stage, cudaStream_t s) : ctx(c), st(s) {
    if (!c->profiling || stage < 0) return;
    nvtxRangePushA(NSGPU_STAGE_NAMES[stage]);
    nsgpu_ctx::StageEv ev; ev.stage = stage;
    for (cudaEvent_t* e : {&ev.a, &ev.b}) {
      if (!c->event_pool.empty()) { *e = c->event_pool.back(); c->event_pool.pop_back(); }
      else cudaEventCreate(e);
    }
    cudaEventRecord(ev.a, s);
    c->stage_events.push_back(ev);
    idx = (int)c->stage_events.size() - 1;
  }
  ~StageTimer() { if (idx >= 0) { cudaEventRecord(ctx->stage_events[idx].b, st); nvtxRangePop(); } }
};

#define NSGPU_CUDA(call)                                                                  \
  do {                                                                                    \
    cudaError_t e_ = (call);                                                              \
    if (e_ != cudaSuccess) {                                                              \
      ctx->err = std::string(#call) + ": " + cudaGetErrorString(e_);                      \
      return NSGPU_ECUDA;                                                                 \
    }                                                                                     \
  } while (0)

// Raise a kernel's dynamic shared-memory limit to at least `bytes` on the context's device.
// cudaFuncAttributeMaxDynamicSharedMemorySize is a property of (function, device) shared by every context of the
// process, so the bookkeeping is process-wide, under a mutex, and the limit is only ever RAISED: a second context that
// needs less for the same kernel (another n_live, another grid) must not lower it under a live context, and two host
// threads driving two contexts must not interleave the set and the launch that relies on it.
cudaError_t nsgpu_raise_smem_limit(int device, const void* fn, size_t bytes);   // api.cu
template <class F>
inline cudaError_t nsgpu_ensure_smem(nsgpu_ctx* ctx, F* fn, size_t bytes) {
  return nsgpu_raise_smem_limit(ctx->device, reinterpret_cast<const void*>(fn), bytes);
}

#define NSGPU_LAUNCH_CHECK()                                                              \
  do {                                                                                    \
    ctx->launches++;                                                                      \
    cudaError_t e_ = cudaGetLastError();                                                  \
    if (e_ != cudaSuccess) {                                                              \
      ctx->err = std::string("kernel launch: ") + cudaGetErrorString(e_) + " at " +       \
                 __FILE__ + ":" + std::to_string(__LINE__);                               \
      return NSGPU_ECUDA;                                                                 \
    }                                                                                     \
  } while (0)

// ---- programmatic dependent launch (PDL) ------------------------------------------------------------------
// The kernels of one likelihood call / one slice-sampling round form a chain on one stream; a nested-sampling
// round is ~10 launches of 10-100 us each, so the drain-and-launch gap between two kernels is a visible share of
// it.  A kernel launched through launch_pdl may start (CTAs become resident as the predecessor's CTAs exit, and run
// their prologue: barrier init, TMEM allocation, staging of constants) while its predecessor is still running.
// Contract for every kernel launched this way: pdl_wait() before the FIRST access to anything an earlier kernel
// wrote (it returns once the predecessor grid has completed and its writes are visible), pdl_trigger() AFTER it.
// Because each kernel triggers only after its own wait, a kernel can overlap with its direct predecessor only:
// everything older is complete, so stream order is preserved transitively.  Kernels launched with <<<>>> keep
// plain stream ordering on both sides.
#ifdef __CUDACC__
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
#endif
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(const nsgpu_ctx* ctx, void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem,
                              cudaStream_t st, Args&&... args) {
  cudaLaunchConfig_t cfg;
  memset(&cfg, 0, sizeof(cfg));
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute attr[1];
  attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[0].val.programmaticStreamSerializationAllowed = (ctx->flags & NSGPU_NO_PDL) ? 0 : 1;
  cfg.attrs = attr; cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kern, KArgs(std::forward<Args>(args))...);
}

// stage entry points (one per translation unit); n_rows_dev != nullptr: only the first *n_rows_dev
// rows (theta) are live, B is then the launch bound
// spectrum output modes of the emulator forward pass
#define NSGPU_SPEC_EXP10 1   // write 10^y (emulate tap) instead of y
#define NSGPU_SPEC_NOMEAN 4  // write y - mu_out (the consumer adds mu_out in fp64)
#define NSGPU_SPEC_KZ 2      // shear only: table layout [theta][k][z] (z fastest) instead of [theta][z][k]
nsgpu_status mlp_forward_simt(nsgpu_ctx* ctx, int e, const float* theta, int B, const int* n_rows_dev,
                              float* spec_out, int ld_spec, int mode, cudaStream_t st);
nsgpu_status mlp_forward_tc(nsgpu_ctx* ctx, int e, const float* theta, int B, const int* n_rows_dev,
                            float* spec_out, int ld_spec, int mode, cudaStream_t st);
nsgpu_status mlp_tc_prepare(nsgpu_ctx* ctx, int e, const nsgpu_emulator* h);
void mlp_tc_release(nsgpu_ctx* ctx, int e);
nsgpu_status shear_project(nsgpu_ctx* ctx, const float* theta, int B, const int* n_rows_dev, cudaStream_t st, int phases = 3);
bool shear_has_split(const nsgpu_ctx* ctx);
size_t shear_resident_smem(const ShearDev& S);
nsgpu_status cmb_bin(nsgpu_ctx* ctx, const float* theta, int B, const int* n_rows_dev, cudaStream_t st);
nsgpu_status cmb_tt_loglike(nsgpu_ctx* ctx, const float* theta, int B, const int* n_rows_dev, double* logL, cudaStream_t st);
nsgpu_status copy_model(nsgpu_ctx* ctx, const float* theta, int B, const int* n_rows_dev, cudaStream_t st);
nsgpu_status chi2_loglike(nsgpu_ctx* ctx, const float* theta, int B, const int* n_rows_dev, double* logL,
                          cudaStream_t st);
nsgpu_status loglike_device(nsgpu_ctx* ctx, const float* theta, int B, const int* n_rows_dev, double* logL,
                            cudaStream_t st);
void nsgpu_probe_release(nsgpu_ctx* ctx);
nsgpu_status sampler_create(nsgpu_ctx* ctx);
void sampler_destroy(nsgpu_ctx* ctx);
