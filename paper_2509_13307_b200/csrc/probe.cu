// probe.cu -- SM clock measured ON the device between the steps of a timed region (bench.py's `clocks` record).
//
// nvidia-smi polls at >= 10-50 ms and reports the clock the driver last set, which says little about a 30 ms timed
// region under a power cap.  A clock MARK is a tiny kernel, ordered on the caller's stream like any other launch,
// whose blocks record the SM cycle counter (clock64) and the global nanosecond timer of the SM they land on; between
// two marks the mean SM clock is the cycle difference over the time difference, taken per SM (the cycle counters are
// per SM) and averaged over the SMs seen in both.  A mark costs one launch of ~3 us; nothing stays resident between
// marks.  (A resident sampling thread was tried first and rejected: the GEMM CTAs use the whole register file of an
// SM, so one resident warp displaced a CTA of the persistent grid and the hidden layers ran 75% slower.)
#include "internal.cuh"

namespace {

constexpr int MAX_MARKS = 512;
constexpr int MAX_SM = 256;

struct ProbeState {
  long long* dev = nullptr;   // [MAX_MARKS][MAX_SM][2] (clock64, globaltimer ns); clock 0 = SM not seen
  int n_marks = 0;
};

__global__ void clock_mark_kernel(long long* slot) {
  if (threadIdx.x != 0) return;
  unsigned smid;
  asm volatile("mov.u32 %0, %%smid;" : "=r"(smid));
  unsigned long long t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
  if (smid < MAX_SM) {
    slot[2 * smid] = clock64();
    slot[2 * smid + 1] = (long long)t;
  }
}

}  // namespace

extern "C" nsgpu_status nsgpu_clock_mark(nsgpu_ctx* ctx, void* stream) {
  if (!ctx) return NSGPU_EINVAL;
  NSGPU_CUDA(cudaSetDevice(ctx->device));
  ProbeState* P = reinterpret_cast<ProbeState*>(ctx->probe);
  if (!P) {
    P = new ProbeState();
    ctx->probe = P;
    NSGPU_CUDA(cudaMalloc((void**)&P->dev, sizeof(long long) * 2 * MAX_SM * MAX_MARKS));
  }
  if (P->n_marks >= MAX_MARKS) { ctx->err = "clock_mark: more than 512 marks since the last read"; return NSGPU_ESHAPE; }
  cudaStream_t st = (cudaStream_t)stream;
  long long* slot = P->dev + (size_t)P->n_marks * 2 * MAX_SM;
  NSGPU_CUDA(cudaMemsetAsync(slot, 0, sizeof(long long) * 2 * MAX_SM, st));
  clock_mark_kernel<<<2 * ctx->sm_count, 32, 0, st>>>(slot);
  cudaError_t e_ = cudaGetLastError();                      // not counted in ctx->launches: not part of the path
  if (e_ != cudaSuccess) { ctx->err = std::string("clock_mark: ") + cudaGetErrorString(e_); return NSGPU_ECUDA; }
  P->n_marks++;
  return NSGPU_OK;
}

extern "C" nsgpu_status nsgpu_clock_marks_read(nsgpu_ctx* ctx, double* sm_mhz, double* t_ms, int32_t cap, int32_t* n_intervals) {
  if (!ctx) return NSGPU_EINVAL;
  ProbeState* P = reinterpret_cast<ProbeState*>(ctx->probe);
  if (n_intervals) *n_intervals = 0;
  if (!P || P->n_marks < 2) { if (P) P->n_marks = 0; return NSGPU_OK; }
  NSGPU_CUDA(cudaSetDevice(ctx->device));
  NSGPU_CUDA(cudaDeviceSynchronize());
  const int n = P->n_marks;
  std::vector<long long> s((size_t)n * 2 * MAX_SM);
  NSGPU_CUDA(cudaMemcpy(s.data(), P->dev, sizeof(long long) * s.size(), cudaMemcpyDeviceToHost));
  P->n_marks = 0;
  if (n_intervals) *n_intervals = n - 1;
  double t_first = 0.0;
  for (int i = 0; i + 1 < n && i < cap; ++i) {
    const long long *a = &s[(size_t)i * 2 * MAX_SM], *b = &s[(size_t)(i + 1) * 2 * MAX_SM];
    double sum = 0.0, tend = 0.0, t0 = 0.0;
    int cnt = 0;
    for (int sm = 0; sm < MAX_SM; ++sm) {
      if (a[2 * sm] == 0 || b[2 * sm] == 0) continue;
      const double dt = (double)(b[2 * sm + 1] - a[2 * sm + 1]);
      if (dt <= 0.0) continue;
      sum += (double)(b[2 * sm] - a[2 * sm]) / dt * 1e3;
      tend += (double)b[2 * sm + 1];
      t0 += (double)a[2 * sm + 1];
      ++cnt;
    }
    if (i == 0) t_first = cnt ? t0 / cnt : 0.0;
    if (sm_mhz) sm_mhz[i] = cnt ? sum / cnt : 0.0;
    if (t_ms) t_ms[i] = cnt ? (tend / cnt - t_first) * 1e-6 : 0.0;
  }
  return NSGPU_OK;
}

void nsgpu_probe_release(nsgpu_ctx* ctx) {
  ProbeState* P = reinterpret_cast<ProbeState*>(ctx->probe);
  if (!P) return;
  cudaFree(P->dev);
  delete P;
  ctx->probe = nullptr;
}
