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

constexpr int TB = 8;    // thetas per CTA: every inverse-factor element loaded from L2 is used TB times

// w = Linv r for TB thetas at once, one thread per PAIR of rows (t, n-1-t): the pair has n+1 non-zero
// columns whatever t is, so the triangular work is balanced across threads.  For a fixed column j the
// threads read LinvT[j][t] and LinvT[j][n-1-t] (coalesced) and the TB residuals r[j][.] (one broadcast
// shared-memory line).  fp64 throughout; chi^2 = sum over rows of w^2 by a block reduction.
__global__ void __launch_bounds__(512) chi2_kernel(const double* __restrict__ model, const double* __restrict__ data,
                                                    const double* __restrict__ LinvT, int n, int B,
                                                    const int* __restrict__ n_rows_dev, const float* __restrict__ theta,
                                                    int D, const int* __restrict__ prior_kind,
                                                    const double* __restrict__ p0, const double* __restrict__ p1,
                                                    double log_norm, double* __restrict__ logL) {
  if (n_rows_dev) B = min(B, *n_rows_dev);
  const int b0 = blockIdx.x * TB;
  if (b0 >= B) return;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double* r = reinterpret_cast<double*>(smem_raw);       // [n][TB]
  double* part = r + (size_t)n * TB;                     // [32][TB] per-warp partial chi^2
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarp = blockDim.x >> 5;
  // residuals, transposed into [j][theta] (coalesced global reads along j)
  for (int i = tid; i < n * TB; i += blockDim.x) {
    const int t = i / n, j = i - t * n;
    const int b = b0 + t;
    r[(size_t)j * TB + t] = (b < B) ? model[(size_t)b * n + j] - data[j] : 0.0;
  }
  __syncthreads();
  const int half = (n + 1) >> 1;
  const int ra = tid, rb = n - 1 - tid;                  // rows of this thread (ra <= rb); ra == rb for the middle row
  double wa[TB], wb[TB];
#pragma unroll
  for (int t = 0; t < TB; ++t) { wa[t] = 0.0; wb[t] = 0.0; }
  if (tid < half) {
    // columns j <= ra feed both rows; ra < j <= rb only the long row
    for (int j = 0; j <= ra; ++j) {
      const double la = LinvT[(size_t)j * n + ra], lb = LinvT[(size_t)j * n + rb];
      const double2* rj = reinterpret_cast<const double2*>(r + (size_t)j * TB);
#pragma unroll
      for (int t = 0; t < TB / 2; ++t) {
        const double2 v = rj[t];
        wa[2 * t] = fma(la, v.x, wa[2 * t]); wa[2 * t + 1] = fma(la, v.y, wa[2 * t + 1]);
        wb[2 * t] = fma(lb, v.x, wb[2 * t]); wb[2 * t + 1] = fma(lb, v.y, wb[2 * t + 1]);
      }
    }
    for (int j = ra + 1; j <= rb; ++j) {
      const double lb = LinvT[(size_t)j * n + rb];
      const double2* rj = reinterpret_cast<const double2*>(r + (size_t)j * TB);
#pragma unroll
      for (int t = 0; t < TB / 2; ++t) {
        const double2 v = rj[t];
        wb[2 * t] = fma(lb, v.x, wb[2 * t]); wb[2 * t + 1] = fma(lb, v.y, wb[2 * t + 1]);
      }
    }
  }
  const bool two = tid < half && ra != rb;
#pragma unroll
  for (int t = 0; t < TB; ++t) {
    double ss = (tid < half ? wb[t] * wb[t] : 0.0) + (two ? wa[t] * wa[t] : 0.0);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, o);
    if (lane == 0) part[warp * TB + t] = ss;
  }
  __syncthreads();
  if (tid < TB) {
    const int b = b0 + tid;
    if (b < B) {
      double chi2 = 0.0;
      for (int w = 0; w < nwarp; ++w) chi2 += part[w * TB + tid];
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
  const int threads = std::min(512, (((n + 1) / 2 + 31) / 32) * 32);
  if ((n + 1) / 2 > 512) { ctx->err = "chi2: n_data > 1024 not supported"; return NSGPU_ESHAPE; }
  const size_t smem = ((size_t)n * TB + 32 * TB) * sizeof(double);
  static size_t configured = 0;
  if (smem > configured) {
    NSGPU_CUDA(cudaFuncSetAttribute(chi2_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    configured = smem;
  }
  StageTimer tm(ctx, 5, st);
  chi2_kernel<<<(B + TB - 1) / TB, threads, smem, st>>>(ctx->model, ctx->data, ctx->Linv, n, B, n_rows_dev, theta,
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
