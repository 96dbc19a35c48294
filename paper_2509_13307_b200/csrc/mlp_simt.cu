// mlp_simt.cu -- CUDA-core emulator forward pass (steps a2-a4), in fp32 or -- NSGPU_MLP_FP64, for the precision study of
// SURVEY 8(f) #4 / P:L166 -- with fp64 activations and accumulation (fp32 weights, fp32 spectrum table).
//
// The on-device correctness reference for the tcgen05 path (mlp_tc.cu) and the path used for
// emulators whose width is not a multiple of 64 (toy-sized test networks).  One emulator evaluation
// (BJ north_star): x = (theta_emu[, z] - mu_in)/sigma_in; four hidden layers
// h <- (beta + sigma(alpha t)(1 - beta)) t with t = h.W + b; y = (h.W + b) sigma_out + mu_out.
#include "internal.cuh"

namespace {

__device__ __forceinline__ float gated_act(float t, float alpha, float beta) {
  // (beta + sigma(alpha t)(1 - beta)) t, sigma(s) = 1/(1+e^-s): e^-s -> inf gives 0, -> 0 gives 1
  float sg = 1.0f / (1.0f + expf(-alpha * t));
  return (beta + sg * (1.0f - beta)) * t;
}
__device__ __forceinline__ double gated_act(double t, double alpha, double beta) {
  double sg = 1.0 / (1.0 + exp(-alpha * t));
  return (beta + sg * (1.0 - beta)) * t;
}
__device__ __forceinline__ float fma_t(float a, float b, float c) { return fmaf(a, b, c); }
__device__ __forceinline__ double fma_t(double a, double b, double c) { return fma(a, b, c); }

// a2 + first hidden layer: gathers the emulator inputs from theta (or constants), appends z_m for
// shear, standardises, applies layer 0.  One thread per (row, neuron); neurons are the fast index.
template <class T>
__global__ void mlp_first_layer_simt(const float* __restrict__ theta, int D, int rows_per_theta,
                                     int M, const int* __restrict__ n_rows_dev,
                                     const int* __restrict__ emu_in_idx, const double* __restrict__ emu_in_const,
                                     int n_theta_in, const float* __restrict__ z_emu, int n_in,
                                     const float* __restrict__ in_mean, const float* __restrict__ in_std,
                                     const float* __restrict__ W, const float* __restrict__ b,
                                     const float* __restrict__ alpha, const float* __restrict__ beta,
                                     int width, T* __restrict__ out) {
  int m = blockIdx.x;
  if (n_rows_dev && m >= (*n_rows_dev) * rows_per_theta) return;
  if (m >= M) return;
  int th = m / rows_per_theta, zi = m - th * rows_per_theta;
  __shared__ T x[NSGPU_MAX_IN];
  if (threadIdx.x < n_in) {
    int i = threadIdx.x;
    T v;
    if (i < n_theta_in) {
      int src = emu_in_idx[i];
      v = src >= 0 ? (T)theta[(size_t)th * D + src] : (T)(float)emu_in_const[i];
    } else {
      v = (T)z_emu[zi];
    }
    x[i] = (v - (T)in_mean[i]) / (T)in_std[i];
  }
  __syncthreads();
  for (int j = blockIdx.y * blockDim.x + threadIdx.x; j < width; j += gridDim.y * blockDim.x) {
    T t = (T)b[j];
    for (int i = 0; i < n_in; ++i) t = fma_t(x[i], (T)W[(size_t)i * width + j], t);
    out[(size_t)m * width + j] = gated_act(t, (T)alpha[j], (T)beta[j]);
  }
}

// C[M][N] = epi(A[M][K] . W[K][N] + b): 64x64 tile, 16-deep k-slab, 256 threads, 4x4 per thread.
// EPI 0: gated activation (hidden layer); EPI 1: y = t sigma_out + mu_out, optionally 10^y.
template <int EPI, class T, class TO>
__global__ void __launch_bounds__(256) gemm_simt(const T* __restrict__ A, const float* __restrict__ W,
                                                 const float* __restrict__ bias, const float* __restrict__ p0,
                                                 const float* __restrict__ p1, int M, int N, int K,
                                                 const int* __restrict__ n_rows_dev, int rows_per_theta,
                                                 int apply_exp10, TO* __restrict__ C, int ldc) {
  if (n_rows_dev) M = min(M, (*n_rows_dev) * rows_per_theta);
  const int m0 = blockIdx.x * 64, n0 = blockIdx.y * 64;
  if (m0 >= M) return;
  __shared__ T As[16][64 + 4];
  __shared__ T Ws[16][64 + 4];
  const int tx = threadIdx.x % 16, ty = threadIdx.x / 16;
  T acc[4][4] = {};
  for (int k0 = 0; k0 < K; k0 += 16) {
    for (int i = threadIdx.x; i < 64 * 16; i += 256) {
      int r = i / 16, c = i % 16;              // A tile: 64 rows x 16 k
      int gm = m0 + r, gk = k0 + c;
      As[c][r] = (gm < M && gk < K) ? A[(size_t)gm * K + gk] : (T)0;
      int kr = i / 64, nc = i % 64;            // W tile: 16 k x 64 cols
      int gk2 = k0 + kr, gn = n0 + nc;
      Ws[kr][nc] = (gk2 < K && gn < N) ? (T)W[(size_t)gk2 * N + gn] : (T)0;
    }
    __syncthreads();
#pragma unroll
    for (int kk = 0; kk < 16; ++kk) {
      T a[4], w[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) a[i] = As[kk][ty * 4 + i];
#pragma unroll
      for (int j = 0; j < 4; ++j) w[j] = Ws[kk][tx * 4 + j];
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = fma_t(a[i], w[j], acc[i][j]);
    }
    __syncthreads();
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    int gm = m0 + ty * 4 + i;
    if (gm >= M) continue;
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      int gn = n0 + tx * 4 + j;
      if (gn >= N) continue;
      T t = acc[i][j] + (T)bias[gn];
      T v;
      if (EPI == 0) {
        v = gated_act(t, (T)p0[gn], (T)p1[gn]);
      } else {
        v = fma_t(t, (T)p0[gn], (T)p1[gn]);    // p0 = sigma_out, p1 = mu_out
        if (apply_exp10) v = (T)exp10((double)v);
      }
      C[(size_t)gm * ldc + gn] = (TO)v;
    }
  }
}

}  // namespace

template <class T>
static nsgpu_status forward_simt(nsgpu_ctx* ctx, int e, const float* theta, int B, const int* n_rows_dev, float* spec_out,
                                 int ld_spec, int mode, cudaStream_t st) {
  const bool apply_exp10 = (mode & NSGPU_SPEC_EXP10) != 0;
  const EmuDev& E = ctx->emu[e];
  const int rpt = ctx->rows_per_theta;
  const int M = B * rpt;
  if (M == 0) return NSGPU_OK;
  T* cur = (T*)ctx->act[0];
  T* nxt = (T*)ctx->act[1];
  {
    StageTimer tm(ctx, 0, st);
    dim3 grid(M, (E.width + 127) / 128);
    mlp_first_layer_simt<T><<<grid, 128, 0, st>>>(theta, ctx->D, rpt, M, n_rows_dev, ctx->emu_in_idx,
                                                  ctx->emu_in_const, ctx->n_theta_in, ctx->z_emu, E.n_in,
                                                  E.in_mean, E.in_std, E.W[0], E.b[0], E.alpha[0], E.beta[0],
                                                  E.width, cur);
    NSGPU_LAUNCH_CHECK();
  }
  for (int l = 1; l < E.n_hidden; ++l) {
    StageTimer tm(ctx, 1, st);
    dim3 grid((M + 63) / 64, (E.width + 63) / 64);
    gemm_simt<0, T, T><<<grid, 256, 0, st>>>(cur, E.W[l], E.b[l], E.alpha[l], E.beta[l], M, E.width, E.width,
                                             n_rows_dev, rpt, 0, nxt, E.width);
    NSGPU_LAUNCH_CHECK();
    T* t = cur; cur = nxt; nxt = t;
  }
  {
    StageTimer tm(ctx, 2, st);
    dim3 grid((M + 63) / 64, (E.n_out + 63) / 64);
    gemm_simt<1, T, float><<<grid, 256, 0, st>>>(cur, E.W[E.n_hidden], E.b[E.n_hidden], E.out_std,
                                                 (mode & NSGPU_SPEC_NOMEAN) ? E.out_zero : E.out_mean, M,
                                                 E.n_out, E.width, n_rows_dev, rpt, apply_exp10 ? 1 : 0, spec_out, ld_spec);
    NSGPU_LAUNCH_CHECK();
  }
  return NSGPU_OK;
}

nsgpu_status mlp_forward_simt(nsgpu_ctx* ctx, int e, const float* theta, int B, const int* n_rows_dev,
                              float* spec_out, int ld_spec, int mode, cudaStream_t st) {
  return (ctx->flags & NSGPU_MLP_FP64) ? forward_simt<double>(ctx, e, theta, B, n_rows_dev, spec_out, ld_spec, mode, st)
                                       : forward_simt<float>(ctx, e, theta, B, n_rows_dev, spec_out, ld_spec, mode, st);
}
