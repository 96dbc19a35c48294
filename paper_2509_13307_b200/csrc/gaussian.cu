// gaussian.cu -- step a10: Gaussian log-likelihood against a fixed dense covariance, and
// step a1: the prior transform (Table 1).
//
// log L = -1/2 sum w^2 - 1/2 ln det(2 pi C), w = L^-1 (model - d).  The whitening is a triangular
// solve against the Cholesky factor; because the factor is fixed for the life of the context its
// inverse (also lower triangular) is formed once, in fp64, at create, and the solve becomes the
// triangular product w = Linv r -- the limit of a blocked TRSM with pre-inverted diagonal blocks.
// Residuals, products and the sum of squares are fp64 (reading P1): n(n+1)/2 MAC per theta is three
// orders of magnitude below the emulator's work, and an fp32 whitening would eat the 1e-3 budget.
#include "internal.cuh"

namespace {

constexpr int TB = 16;   // thetas per CTA
constexpr int RG = 16;   // row groups per CTA (TB * RG = 256 threads)

__global__ void __launch_bounds__(TB* RG) chi2_kernel(const double* __restrict__ model,
                                                      const double* __restrict__ data,
                                                      const double* __restrict__ Linv, int n, int B,
                                                      const int* __restrict__ n_rows_dev,
                                                      const float* __restrict__ theta, int D,
                                                      const int* __restrict__ prior_kind,
                                                      const double* __restrict__ p0, const double* __restrict__ p1,
                                                      double log_norm, double* __restrict__ logL) {
  if (n_rows_dev) B = min(B, *n_rows_dev);
  const int b0 = blockIdx.x * TB;
  if (b0 >= B) return;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double* r = reinterpret_cast<double*>(smem_raw);       // [n][TB]
  double* part = r + (size_t)n * TB;                     // [RG][TB]
  const int lane = threadIdx.x % TB, grp = threadIdx.x / TB;
  // residuals, transposed into [j][theta] (coalesced global reads along j)
  for (int i = threadIdx.x; i < n * TB; i += blockDim.x) {
    const int t = i / n, j = i - t * n;
    const int b = b0 + t;
    r[(size_t)j * TB + t] = (b < B) ? model[(size_t)b * n + j] - data[j] : 0.0;
  }
  __syncthreads();
  double ss = 0.0;
  // rows are dealt round-robin to the row groups so the triangular work is balanced
  for (int i = grp; i < n; i += RG) {
    const double* Li = Linv + (size_t)i * n;
    double acc = 0.0;
    for (int j = 0; j <= i; ++j) acc = fma(__ldg(Li + j), r[(size_t)j * TB + lane], acc);
    ss = fma(acc, acc, ss);
  }
  part[grp * TB + lane] = ss;
  __syncthreads();
  if (grp == 0) {
    const int b = b0 + lane;
    if (b < B) {
      double chi2 = 0.0;
      for (int g = 0; g < RG; ++g) chi2 += part[g * TB + lane];
      double out = -0.5 * chi2 + log_norm;
      // support of the uniform priors (compared in the float32 theta arrives in) and finiteness
      bool ok = isfinite(out);
      for (int d = 0; d < D; ++d) {
        const float v = theta[(size_t)b * D + d];
        if (!isfinite(v)) ok = false;
        if (prior_kind[d] == 0 && (v < (float)p0[d] || v > (float)p1[d])) ok = false;
      }
      logL[b] = ok ? out : -INFINITY;
    }
  }
}

__global__ void prior_transform_kernel(const float* __restrict__ u, int B, int D,
                                       const int* __restrict__ kind, const double* __restrict__ p0,
                                       const double* __restrict__ p1, float* __restrict__ theta) {
  const size_t total = (size_t)B * D;
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
    const int d = (int)(i % D);
    const double x = (double)u[i];
    const double t = kind[d] == 0 ? p0[d] + (p1[d] - p0[d]) * x : p0[d] + p1[d] * normcdfinv(x);
    theta[i] = (float)t;
  }
}

}  // namespace

nsgpu_status chi2_loglike(nsgpu_ctx* ctx, const float* theta, int B, const int* n_rows_dev, double* logL,
                          cudaStream_t st) {
  if (B == 0) return NSGPU_OK;
  const int n = ctx->n_data;
  const size_t smem = ((size_t)n * TB + RG * TB) * sizeof(double);
  static size_t configured = 0;
  if (smem > configured) {
    NSGPU_CUDA(cudaFuncSetAttribute(chi2_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    configured = smem;
  }
  StageTimer tm(ctx, 5, st);
  chi2_kernel<<<(B + TB - 1) / TB, TB * RG, smem, st>>>(ctx->model, ctx->data, ctx->Linv, n, B, n_rows_dev, theta,
                                                         ctx->D, ctx->prior_kind, ctx->prior_p0, ctx->prior_p1,
                                                         ctx->log_norm, logL);
  NSGPU_LAUNCH_CHECK();
  return NSGPU_OK;
}

extern "C" nsgpu_status nsgpu_prior_transform(nsgpu_ctx* ctx, const float* u, int32_t B, float* theta, void* stream) {
  if (!ctx) return NSGPU_EINVAL;
  if (B < 0 || (B > 0 && (!u || !theta))) { ctx->err = "prior_transform: bad arguments"; return NSGPU_EINVAL; }
  if (B == 0) return NSGPU_OK;
  NSGPU_CUDA(cudaSetDevice(ctx->device));
  const size_t total = (size_t)B * ctx->D;
  const int blocks = (int)std::min<size_t>((total + 255) / 256, (size_t)ctx->sm_count * 8);
  prior_transform_kernel<<<blocks, 256, 0, (cudaStream_t)stream>>>(u, B, ctx->D, ctx->prior_kind, ctx->prior_p0,
                                                                   ctx->prior_p1, theta);
  NSGPU_LAUNCH_CHECK();
  return NSGPU_OK;
}
