// mlp_tc.cu -- emulator MLP on the 5th-generation tensor cores (steps a2-a4).
//
// One emulator evaluation (BJ north_star): x = (theta_emu[, z] - mu_in)/sigma_in; hidden
// layers h <- (beta + sigma(alpha t)(1 - beta)) t with t = h.W + b; y = (h.W + b) sigma_out + mu_out.
//
// Precision (reading P1): the 1e-4 relative tolerance on 10^y rules out single-pass
// TF32 (rms 7e-4).  Every GEMM operand is split into two fp16 numbers, x = hi + lo (22 significant
// bits), and the product is three kind::f16 MMA passes  hi.hi + lo.hi + hi.lo  accumulated in fp32 in
// TMEM -- the accuracy of 3xTF32 at twice its tensor rate.  Weights are split once at create (scaled by
// a power of two so that hi and lo are normal fp16 numbers); activations are split in the epilogue of
// the layer that produces them (scaled by 16) and travel to the next layer as fp16 hi/lo planes.
//
// Activation planes live in HBM in the tensor core's own canonical (no-swizzle, K-major) operand
// layout, [M/128 tiles][K/8 pieces][128 rows][8 halves]: a 128-row x 64-column k-block of A is 16 KB
// contiguous (one cp.async.bulk per plane, no tensor map), and the epilogue -- where a thread owns a
// ROW of the accumulator -- writes 16-byte pieces that are contiguous across the lanes of a warp.
//
// Kernel: persistent, one CTA per SM: epilogue warps + 1 TMA producer warp + 1 MMA warp.  Tile 128 rows
// x BLOCK_N columns; K in blocks of 64; per k-block the producer brings four tiles (A_hi, A_lo by bulk
// copy; W_hi, W_lo by tiled TMA with 128-byte swizzle) and the MMA thread issues 12 tcgen05.mma into a
// fresh TMEM partial (two partial buffers); the epilogue warps sum the partials in registers.
#include <cuda.h>

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>

#include "internal.cuh"
#include "tc_ptx.cuh"

namespace {

constexpr int BLOCK_M = 128;
// fp16 elements per k-block: a template parameter of the GEMM (64: two smem stages of 96 KB for 256-column tiles,
// 128-byte-swizzled weight rows; 32: four stages of 48 KB, 64-byte swizzle).
constexpr int PIECE_HALVES = BLOCK_M * 8;      // one 16-byte piece of every row of a tile: 2 KB
constexpr float ACT_SCALE = 16.0f;             // activations are stored as fp16 hi/lo of 16 h
constexpr int SMEM_BUDGET = 225 * 1024;
// tcgen05.mma adds into its fp32 TMEM accumulator with truncation toward zero (measured): every
// accumulating MMA shrinks the accumulator by U[0,1) ulp.  Measured on one K = 512 layer with everything else exact
// (profiles/r2_truncation_model.md): relative bias -c x (number of accumulations a contribution sits through), with
// c = 3.2e-8 (0.54 x 2^-24) for sums of mixed sign and 4.9e-8 (0.82 x 2^-24) for sums of one sign, the same for
// partials of 1, 2, 4 and 8 k-blocks; symmetric under a sign flip of the weights (toward zero, not toward -inf).
// A partial of n k-blocks of s = BK/16 k-steps is 3 s n MMAs in the order (2 s corrections, s hi.hi) per k-block;
// the hi.hi group j of k-block i is issued at step 3 s i + 2 s + j and is part of the accumulator at the
// 3 s n - (3 s i + 2 s + j) later accumulations: 1.5 s n - s + 0.5 on average.  The mean of that bias is undone by one
// factor folded into the epilogue scale (fp32, so a whole number of 2^-23); what is left is < 5e-8 per layer of slope
// and the spread of the counts around their mean times the (random-signed) differences between the k-blocks'
// contributions (rms 2.5e-7 |t| for 64 columns per partial, 4.6e-7 for 128: measured).
constexpr double TRUNC_C = 3.2e-8;
inline float trunc_comp(int K, int bk, int kpp) {
  if (const char* ev = getenv("NSGPU_TRUNC_ULPS")) return 1.0f + (float)(atof(ev) / 8388608.0);   // kernel A/B runs
  const int k_blocks = K / bk, st = bk / 16;
  double wsum = 0.0;
  for (int kb0 = 0; kb0 < k_blocks; kb0 += kpp) {
    const int n = std::min(kpp, k_blocks - kb0);
    wsum += n * (1.5 * st * n - st + 0.5);
  }
  const double ulps = std::nearbyint(TRUNC_C * (wsum / k_blocks) * 8388608.0);   // in units of 2^-23
  return 1.0f + (float)(ulps / 8388608.0);
}

__host__ __device__ constexpr int a_tile_bytes(int bk) { return BLOCK_M * bk * 2; }   // bk / 8 pieces x (128 rows x 16 bytes)
__host__ __device__ constexpr int stage_bytes(int block_n, int bk) { return 2 * a_tile_bytes(bk) + 2 * block_n * bk * 2; }
__host__ __device__ constexpr int num_stages(int block_n, int bk) {
  int s = (SMEM_BUDGET - 1024 - 10 * 1024) / stage_bytes(block_n, bk);   // 1 KB alignment slack, 10 KB params + barriers
  return s > 8 ? 8 : s;
}

struct GemmArgs {
  int M_host;                 // rows to process (upper bound when n_rows_dev != nullptr)
  const int* n_rows_dev;      // live thetas (device) or nullptr
  int rows_per_theta;
  int K;                      // fan-in (multiple of 64)
  int kpp;                    // k-blocks accumulated in TMEM per partial (1, 2, 4 ...; see mlp_gemm_tc)
  int split4;                 // precision study: also issue the lo.lo product (NSGPU_MLP_SPLIT4)
  int N_pad;                  // padded fan-out (multiple of BLOCK_N)
  int n_valid;                // true fan-out
  const __half *a_hi, *a_lo;  // input planes, canonical layout, K columns
  const float4* p_hidden;     // [N_pad] {bias, -alpha log2 e, 16 beta, 16 (1 - beta)}
  const float2* p_out;        // [N_pad] {cscale sigma_out, b sigma_out + mu_out}
  const float4* p_out4;       // [N_pad/2] the same for column pairs: {s1_0, s1_1, s0_0, s0_1}
  float cscale;               // 2^-(wexp + 4): undoes the operand scalings
  __half *out_hi, *out_lo;    // next layer's planes (canonical layout, ld_out columns)
  int ld_out;
  float* out_f32;             // output layer
  int ld_f32;                 // out_mode 0: y[m][n] at m ld_f32 + n
  int out_mode;               // out_mode 1: y at theta(m) (n_valid rpt) + n rpt + z(m)  ([theta][n][z], z fastest)
  int apply_exp10;
  unsigned long long* nonfinite;   // output layer: rows whose accumulators are not finite (see nsgpu_nonfinite_rows)
};

__device__ __forceinline__ float ex2_approx(float x) { float y; asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }
__device__ __forceinline__ float rcp_approx(float x) { float y; asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x)); return y; }

// 16 (beta + sigma(alpha t)(1 - beta)) t with p = {., -alpha log2 e, 16 beta, 16 (1 - beta)};
// sigma(s) = 1/(1 + 2^(-s log2 e)): 2^x -> inf gives 0, -> 0 gives 1 (no NaN path)
__device__ __forceinline__ float gated_act16(float t, const float4& p) {
  const float sg = rcp_approx(1.0f + ex2_approx(p.y * t));
  return fmaf(sg, p.w, p.z) * t;
}

// packed fp32x2 arithmetic (sm_100: FFMA2 / FMUL2 / FADD2 halve the FMA-pipe instruction count)
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk2(float a, float b) { f32x2 r; asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(a), "f"(b)); return r; }
__device__ __forceinline__ void upk2(f32x2 v, float& a, float& b) { asm("mov.b64 {%0, %1}, %2;" : "=f"(a), "=f"(b) : "l"(v)); }
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) { f32x2 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) { f32x2 d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b) { f32x2 d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }

// Two columns of the hidden-layer epilogue at once: t = acc cs + bias; 16 (beta + sigma(alpha t)(1 - beta)) t;
// hi/lo fp16 split.  pa = {bias0, bias1, a2_0, a2_1}, pb = {16 beta0, 16 beta1, 16 (1-beta0), 16 (1-beta1)}.
__device__ __forceinline__ void act_split_pair(f32x2 acc, f32x2 cs2, const float4& pa, const float4& pb, uint32_t& hi,
                                               uint32_t& lo) {
  const f32x2 t = fma2(acc, cs2, pk2(pa.x, pa.y));
  float s0, s1;
  upk2(mul2(pk2(pa.z, pa.w), t), s0, s1);
  // sigma = 1/(1 + 2^(-alpha t log2 e)): 2 MUFU ops per column.  (A Newton reciprocal on the FMA pipe was
  // measured no faster: the epilogue is issue-bound, not MUFU-bound.)
  const float e0 = ex2_approx(s0), e1 = ex2_approx(s1);
  float d0, d1;
  upk2(add2(pk2(e0, e1), pk2(1.0f, 1.0f)), d0, d1);
  const f32x2 sg = pk2(rcp_approx(d0), rcp_approx(d1));
  const f32x2 o = mul2(fma2(sg, pk2(pb.z, pb.w), pk2(pb.x, pb.y)), t);
  float o0, o1;
  upk2(o, o0, o1);
  const __half2 h = __floats2half2_rn(o0, o1);
  const float2 hf = __half22float2(h);
  float l0, l1;
  upk2(fma2(pk2(hf.x, hf.y), pk2(-1.0f, -1.0f), o), l0, l1);
  const __half2 l = __floats2half2_rn(l0, l1);
  hi = *reinterpret_cast<const uint32_t*>(&h);
  lo = *reinterpret_cast<const uint32_t*>(&l);
}

// x -> (hi, lo) fp16 pair planes, two elements at a time
__device__ __forceinline__ void split2(float a, float b, uint32_t& hi, uint32_t& lo) {
  const __half2 h = __floats2half2_rn(a, b);
  const float2 hf = __half22float2(h);
  const __half2 l = __floats2half2_rn(a - hf.x, b - hf.y);
  hi = *reinterpret_cast<const uint32_t*>(&h);
  lo = *reinterpret_cast<const uint32_t*>(&l);
}

// a2 + first hidden layer (K = n_in <= 16: CUDA cores), output as the canonical fp16 hi/lo planes of
// 16 h.  One CTA per 128-row tile; lane = row, each warp walks 16-byte pieces (8 neurons) so that a
// warp's stores are 512 contiguous bytes.  W0 and the activation parameters are staged in shared memory.
template <int NIN>
__global__ void __launch_bounds__(256) mlp_first_layer_tc(const float* __restrict__ theta, int D, int rows_per_theta,
                                                          int M, const int* __restrict__ n_rows_dev,
                                                          const int* __restrict__ emu_in_idx,
                                                          const double* __restrict__ emu_in_const, int n_theta_in,
                                                          const float* __restrict__ z_emu, int n_in,
                                                          const float* __restrict__ in_mean,
                                                          const float* __restrict__ in_std, const float* __restrict__ W,
                                                          const float4* __restrict__ params, int width, int split,
                                                          __half* __restrict__ out_hi, __half* __restrict__ out_lo) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float4* sp = reinterpret_cast<float4*>(smem_raw);          // [width]
  float* sW = reinterpret_cast<float*>(sp + width);          // [n_in][width]
  // Columns this CTA needs: all of them, or -- small batches, where the host launches one CTA per (tile, 1/split of
  // the pieces) and staging 26 KB of constants per CTA was most of its life -- only those of its own part.
  int col0 = 0, col1 = width;
  if (split > 1 && (int)gridDim.x >= ((M + BLOCK_M - 1) / BLOCK_M) * split) {   // M: the launch bound, so one item per CTA
    const int n_pieces_ = width >> 3, ppi_ = (n_pieces_ + split - 1) / split, part_ = blockIdx.x % split;
    col0 = min(8 * part_ * ppi_, width);
    col1 = min(8 * (part_ + 1) * ppi_, width);
  }
  for (int i = (col0 >> 1) + threadIdx.x; i < (col1 >> 1); i += blockDim.x) {   // two columns per entry pair (see act_split_pair)
    const float4 c0 = params[2 * i], c1 = params[2 * i + 1];
    sp[2 * i] = make_float4(c0.x, c1.x, c0.y, c1.y);
    sp[2 * i + 1] = make_float4(c0.z, c1.z, c0.w, c1.w);
  }
  {
    const int nc = col1 - col0;
    for (int i = threadIdx.x; i < n_in * nc; i += blockDim.x) {
      const int c = i / nc, j = col0 + (i - c * nc);
      sW[c * width + j] = W[c * width + j];
    }
  }
  pdl_wait();                                                // constants staged above; theta and the row count below (launch_pdl contract)
  pdl_trigger();
  if (n_rows_dev) M = min(M, (*n_rows_dev) * rows_per_theta);
  __syncthreads();
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int r = (warp & 3) * 32 + lane;                      // row within the tile
  const int n_pieces = width >> 3;
  const int ppi = (n_pieces + split - 1) / split;      // pieces per work item
  const int half = (ppi + 1) >> 1;                           // ... per warp group
  const int n_items = ((M + BLOCK_M - 1) / BLOCK_M) * split;
  const f32x2 one2 = pk2(1.0f, 1.0f);
  // a work item is (128-row tile, 1/split of its pieces); the host launches one CTA per item.  split = 1 for large
  // batches (measured: finer items only add input gathers there), 4 when whole tiles would leave SMs idle.
  for (int item = blockIdx.x; item < n_items; item += gridDim.x) {
    const int tile = item / split, part = item - tile * split;
    const int m0 = tile * BLOCK_M;
    const int m = min(m0 + r, M - 1);
    const int th = m / rows_per_theta, zi = m - th * rows_per_theta;
    f32x2 x2[NIN];                                          // NIN = n_in at compile time: no predicated-off work
#pragma unroll
    for (int c = 0; c < NIN; ++c) {
      float v;
      if (c < n_theta_in) {
        const int src = emu_in_idx[c];
        v = src >= 0 ? theta[(size_t)th * D + src] : (float)emu_in_const[c];
      } else {
        v = z_emu[zi];
      }
      v = (v - in_mean[c]) / in_std[c];
      x2[c] = pk2(v, v);
    }
    const int p_begin = part * ppi + (warp >> 2) * half;
    const int p_end = min(min(p_begin + half, (part + 1) * ppi), n_pieces);
    const size_t tile_base = (size_t)tile * ((size_t)BLOCK_M * width) + (size_t)r * 8;
    for (int p = p_begin; p < p_end; ++p) {
      uint32_t hi[4], lo[4];
      f32x2 t[4] = {0ull, 0ull, 0ull, 0ull};                    // 8 neurons of this piece, bias added in the epilogue
#pragma unroll
      for (int c = 0; c < NIN; ++c) {
        const float4 wlo = *reinterpret_cast<const float4*>(sW + c * width + 8 * p);
        const float4 whi = *reinterpret_cast<const float4*>(sW + c * width + 8 * p + 4);
        t[0] = fma2(x2[c], pk2(wlo.x, wlo.y), t[0]); t[1] = fma2(x2[c], pk2(wlo.z, wlo.w), t[1]);
        t[2] = fma2(x2[c], pk2(whi.x, whi.y), t[2]); t[3] = fma2(x2[c], pk2(whi.z, whi.w), t[3]);
      }
#pragma unroll
      for (int jj = 0; jj < 4; ++jj) act_split_pair(t[jj], one2, sp[8 * p + 2 * jj], sp[8 * p + 2 * jj + 1], hi[jj], lo[jj]);
      if (m0 + r < M) {
        const size_t o = tile_base + (size_t)p * PIECE_HALVES;
        *reinterpret_cast<uint4*>(out_hi + o) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
        *reinterpret_cast<uint4*>(out_lo + o) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
      }
    }
  }
}

// Store under a predicate, never a branch.  The [theta][k][z] table epilogue does 2 x 56 guarded stores per thread and tile;
// whether the compiler predicates them or builds a convergence region around each one is a heuristic that flipped with
// unrelated changes to the kernel this round (output layer 0.289 -> 0.338 ms on c3a with identical arithmetic, found by
// bisecting against the round-1 build and diffing the SASS); with the predicate written out: 0.303 ms.
__device__ __forceinline__ void st_global_if(float* p, float v, bool ok) {
  asm volatile("{\n.reg .pred q;\nsetp.ne.b32 q, %2, 0;\n@q st.global.f32 [%0], %1;\n}" ::"l"(p), "f"(v), "r"((int)ok) : "memory");
}

// Epilogue of NP column pairs (pairs P0 .. P0+NP-1 of the thread's CPT/2; a[i] is pair P0 + i) of one accumulator
// row: EPI 0 bias + gated activation + hi/lo split into the next layer's canonical planes; EPI 1 de-standardised
// fp32 output (row-major, or [theta][n][z] for the shear table).
struct TileRef { int m_blk, n0, r_in, row; bool row_ok; };
// OUT_MODE >= 0 fixes g.out_mode at compile time and drops the 10^y code (the fused kernel: half the epilogue code, and
// no exp10f inlined 200 times -- its emulate tap applies 10^y in a pass of its own)
template <int EPI, int P0, int NP, int OUT_MODE = -1>
__device__ __forceinline__ void epi_pairs(const f32x2* a, const TileRef& t, const GemmArgs& g, const float* params) {
  static_assert(P0 % 4 == 0 && NP % 4 == 0, "whole 16-byte pieces");
  const int n0 = t.n0 + 2 * P0;                                  // first column of this slice
  if (EPI == 0) {
    const float4* p = reinterpret_cast<const float4*>(params) + n0;
    const f32x2 cs2 = pk2(g.cscale, g.cscale);
    // canonical layout: piece n0/8 + c of this tile, 16 bytes per row: lanes are contiguous
    const size_t o = (size_t)t.m_blk * ((size_t)BLOCK_M * g.ld_out) + (size_t)(n0 >> 3) * PIECE_HALVES + (size_t)t.r_in * 8;
    __half* dh = g.out_hi + o;
    __half* dl = g.out_lo + o;
#pragma unroll
    for (int c = 0; c < NP / 4; ++c) {
      uint32_t hi[4], lo[4];
#pragma unroll
      for (int j = 0; j < 4; ++j) act_split_pair(a[4 * c + j], cs2, p[8 * c + 2 * j], p[8 * c + 2 * j + 1], hi[j], lo[j]);
      // No row test: the planes are allocated in whole 128-row tiles, so the rows past M of the last tile are
      // stored too (finite values nobody reads).  A test here makes every 8-column piece a basic block of its own
      // and the MUFU / conversion chains of different pieces can no longer be interleaved.
      *reinterpret_cast<uint4*>(dh + (size_t)c * PIECE_HALVES) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
      *reinterpret_cast<uint4*>(dl + (size_t)c * PIECE_HALVES) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
    }
  } else {
    const float4* p4 = g.p_out4 + (n0 >> 1);                       // warp-uniform addresses: L1 broadcast
    const int rr = t.row_ok ? t.row : 0;
    const bool exp10_on = OUT_MODE < 0 && g.apply_exp10;
    if (OUT_MODE < 0 ? g.out_mode == 1 : OUT_MODE == 1) {
      // [theta][n][z] with z fastest: consecutive rows (lanes) of one theta are contiguous
      const int th = rr / g.rows_per_theta, zi = rr - th * g.rows_per_theta;
      float* dst = g.out_f32 + (size_t)th * ((size_t)g.n_valid * g.rows_per_theta) + zi;
#pragma unroll
      for (int j = 0; j < NP; ++j) {                               // two columns per step: one 16-byte parameter load, one FFMA2
        const float4 pj = __ldg(p4 + j);                           // {s1_0, s1_1, s0_0, s0_1}
        float y0, y1;
        upk2(fma2(a[j], pk2(pj.x, pj.y), pk2(pj.z, pj.w)), y0, y1);
        if (exp10_on) { y0 = exp10f(y0); y1 = exp10f(y1); }
        const int n = n0 + 2 * j;
        st_global_if(dst + (size_t)n * g.rows_per_theta, y0, t.row_ok && n < g.n_valid);
        st_global_if(dst + (size_t)(n + 1) * g.rows_per_theta, y1, t.row_ok && n + 1 < g.n_valid);
      }
    } else {
      float* dst = g.out_f32 + (size_t)rr * g.ld_f32 + n0;
      const bool vec = (g.ld_f32 & 3) == 0;
#pragma unroll
      for (int c = 0; c < NP / 2; ++c) {
        float y[4];
        const float4 pa = __ldg(p4 + 2 * c), pb = __ldg(p4 + 2 * c + 1);
        upk2(fma2(a[2 * c], pk2(pa.x, pa.y), pk2(pa.z, pa.w)), y[0], y[1]);
        upk2(fma2(a[2 * c + 1], pk2(pb.x, pb.y), pk2(pb.z, pb.w)), y[2], y[3]);
        if (exp10_on) {
#pragma unroll
          for (int j = 0; j < 4; ++j) y[j] = exp10f(y[j]);
        }
        if (t.row_ok) {
          if (vec && n0 + 4 * c + 4 <= g.n_valid) {
            reinterpret_cast<float4*>(dst)[c] = make_float4(y[0], y[1], y[2], y[3]);
          } else {
#pragma unroll
            for (int j = 0; j < 4; ++j)
              if (n0 + 4 * c + j < g.n_valid) dst[4 * c + j] = y[j];
          }
        }
      }
    }
  }
}

// C[M][N] = epi(A[M][K] . W[N][K]^T) with A, W as fp16 hi/lo planes (three MMA passes).
// EPI 0: hidden layer -> next layer's hi/lo planes; EPI 1: output layer -> fp32 y (optionally 10^y).
//
// Accumulation ("tensor-core accumulator truncation"): tcgen05.mma adds into its
// fp32 TMEM accumulator with truncation, which over a K = 512 chain of 96 instructions shrinks every
// output by ~2e-6 -- a coherent error the 1e-3 log L tolerance cannot absorb.  So the tensor core
// only ever accumulates ONE k-block (64 inputs: 8 small correction MMAs first, then the 4 hi.hi MMAs)
// into a fresh TMEM partial; the epilogue warps pull each partial into registers (tcgen05.ld) and do
// the cross-k-block summation in round-to-nearest fp32 there, while the MMA thread fills the other
// partial buffer.  Bias, activation, hi/lo split and the global stores then run from registers.
constexpr int EPI_WARPS = 8;                         // 2 per TMEM lane quarter, each half of the tile's columns
constexpr int GEMM_THREADS = 384;                    // warpgroups 0-1 epilogue; warpgroup 2: TMA producer, MMA issuer, 2 idle
constexpr int DEFER_PAIRS = 32;                      // 64 columns of a finished tile wait in registers (see below)
//
// Weight multicast (CS > 1): with one CTA per SM and 96 KB of operands per k-block, a hidden layer pulls
// 768 KB per tile from L2 -- 44 B/clk/SM at the measured tile time, which IS the chip's L2 -> SM throughput
// (~6300 B/clk over 148 SMs), and two thirds of it are weight tiles that every CTA working on the same column
// block reads again.  So CS CTAs of a thread-block cluster take CS consecutive row blocks of the SAME column
// block in lock step; each loads 1/CS of the W_hi / W_lo tile and multicasts it into the shared memory of all
// of them (96 -> 64 KB of L2 reads per CTA and k-block for CS = 2).  A stage may be refilled
// only when every CTA of the cluster has consumed it: the MMA commit that frees it is multicast as well and the
// `empty` barriers count CS arrivals.  The MMA / TMEM / epilogue side is unchanged.
template <int BLOCK_N, int EPI, int CS = 1, int BK = 64>
__global__ void __launch_bounds__(GEMM_THREADS, 1) mlp_gemm_tc(const __grid_constant__ CUtensorMap tm_whi,
                                                               const __grid_constant__ CUtensorMap tm_wlo, GemmArgs g) {
  constexpr int STAGES = num_stages(BLOCK_N, BK);
  constexpr int STAGE = stage_bytes(BLOCK_N, BK);
  constexpr int A_TILE_BYTES = a_tile_bytes(BK);
  constexpr int B_TILE_BYTES = BLOCK_N * BK * 2;
  constexpr int CPT = BLOCK_N / (EPI_WARPS / 4);                 // columns per epilogue thread
  constexpr int LDC = (CPT % 16 == 0) ? 16 : 8;                  // columns per tcgen05.ld
  constexpr int NPB = BLOCK_N <= 128 ? 4 : 2;                    // TMEM partial buffers (ring)
  constexpr int PB_COLS = 512 / NPB;
  constexpr uint32_t IDESC = tc::idesc_f16_f32(BLOCK_M, BLOCK_N);
  static_assert(STAGES >= 2, "need at least two smem stages");
  static_assert(BLOCK_N % 32 == 0 && BLOCK_N >= 32 && BLOCK_N <= 256 && CPT % 8 == 0, "UMMA N for M = 128; CPT multiple of 8");

  extern __shared__ unsigned char smem_dyn[];
  const uint32_t base = (tc::smem_u32(smem_dyn) + 1023u) & ~1023u;       // SWIZZLE_128B tiles: 1024-byte aligned
  unsigned char* base_ptr = smem_dyn + (base - tc::smem_u32(smem_dyn));
  const uint32_t bars = base + STAGES * STAGE;                            // full[S], empty[S], pfull[2], pempty[2]
  const uint32_t full0 = bars, empty0 = bars + 8 * STAGES, pfull0 = bars + 16 * STAGES, pempty0 = pfull0 + 32;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(base_ptr + STAGES * STAGE + 16 * STAGES + 64);
  float* params = reinterpret_cast<float*>(base_ptr + STAGES * STAGE + 16 * STAGES + 80);   // 16-byte aligned

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    for (int s = 0; s < STAGES; ++s) { tc::mbar_init(full0 + 8 * s, 1); tc::mbar_init(empty0 + 8 * s, CS); }
    for (int b = 0; b < NPB; ++b) { tc::mbar_init(pfull0 + 8 * b, 1); tc::mbar_init(pempty0 + 8 * b, EPI_WARPS); }
    tc::fence_barrier_init();
  }
  if (warp == EPI_WARPS + 1) tc::tmem_alloc(tc::smem_u32(tmem_slot), 512);
  if (warp == EPI_WARPS && lane == 0) { tc::prefetch_tmap(&tm_whi); tc::prefetch_tmap(&tm_wlo); }
  if (EPI == 0) {   // hidden layers: N_pad <= 512 -> 8 KB of per-column parameters staged once
    for (int i = threadIdx.x; i < g.N_pad / 2; i += blockDim.x) {   // two columns per entry pair (see act_split_pair)
      const float4 c0 = g.p_hidden[2 * i], c1 = g.p_hidden[2 * i + 1];
      reinterpret_cast<float4*>(params)[2 * i] = make_float4(c0.x, c1.x, c0.y, c1.y);
      reinterpret_cast<float4*>(params)[2 * i + 1] = make_float4(c0.z, c1.z, c0.w, c1.w);
    }
  }
  // everything above touches only constants and this CTA's own shared memory / TMEM: it may run while the previous
  // layer is still finishing (launch_pdl contract); the activations and the row count are read below
  pdl_wait();
  pdl_trigger();
  tc::fence_before_sync();
  __syncthreads();
  if (CS > 1) tc::cluster_sync();        // every CTA's barriers exist before a peer's multicast or commit reaches them
  tc::fence_after_sync();
  const uint32_t tmem_base = *tmem_slot;
  int M = g.M_host;
  if (g.n_rows_dev) M = min(M, (*g.n_rows_dev) * g.rows_per_theta);
  const int n_blocks = g.N_pad / BLOCK_N;
  const int m_blocks = (M + BLOCK_M - 1) / BLOCK_M;
  // work items: (group of CS row blocks, column block); CTA `crank` of a cluster takes row block CS grp + crank
  // (clamped: the spare CTA of a ragged last group repeats the last row block and stores the same values)
  const int crank = CS > 1 ? (int)tc::cluster_ctarank() : 0;
  const int num_tiles = ((m_blocks + CS - 1) / CS) * n_blocks;
  const int tile0 = blockIdx.x / CS, tile_step = gridDim.x / CS;
  constexpr uint16_t CMASK = (uint16_t)((1u << CS) - 1u);
  constexpr int W_SUB_BYTES = B_TILE_BYTES / CS;                 // this CTA's share of a weight tile
  const int k_blocks = g.K / BK;
  const int kpp = g.kpp;

  // registers: 384 x 168 at launch -> 232 for the epilogue warpgroups (accumulators + deferred columns), 40 for the rest
  if (warp >= EPI_WARPS) {
    asm volatile("setmaxnreg.dec.sync.aligned.u32 40;");
  if (warp == EPI_WARPS) {
    // ===== TMA producer =====
    if (lane == 0) {
      uint32_t stage = 0, phase = 0;
      for (int tile = tile0; tile < num_tiles; tile += tile_step) {
        const int m_grp = tile / n_blocks, n_blk = tile - m_grp * n_blocks;
        const int m_blk = min(m_grp * CS + crank, m_blocks - 1);
        // this tile's A rows: k-block kb is the 16 KB starting at piece 8 kb
        const size_t a_tile = (size_t)m_blk * ((size_t)BLOCK_M * g.K);
        for (int kb = 0; kb < k_blocks; ++kb) {
          tc::mbar_wait(empty0 + 8 * stage, phase ^ 1);
          const uint32_t s0 = base + stage * STAGE, fb = full0 + 8 * stage;
          tc::mbar_arrive_expect_tx(fb, STAGE);
          const size_t a_off = a_tile + (size_t)kb * (BK / 8) * PIECE_HALVES;
          tc::bulk_load(s0, g.a_hi + a_off, A_TILE_BYTES, fb);
          tc::bulk_load(s0 + A_TILE_BYTES, g.a_lo + a_off, A_TILE_BYTES, fb);
          if (CS == 1) {
            tc::tma_load_2d(s0 + 2 * A_TILE_BYTES, &tm_whi, kb * BK, n_blk * BLOCK_N, fb);
            tc::tma_load_2d(s0 + 2 * A_TILE_BYTES + B_TILE_BYTES, &tm_wlo, kb * BK, n_blk * BLOCK_N, fb);
          } else {   // tensor maps with boxes of BLOCK_N / CS rows
            const int wrow = n_blk * BLOCK_N + crank * (BLOCK_N / CS);
            tc::tma_load_2d_mc(s0 + 2 * A_TILE_BYTES + crank * W_SUB_BYTES, &tm_whi, kb * BK, wrow, fb, CMASK);
            tc::tma_load_2d_mc(s0 + 2 * A_TILE_BYTES + B_TILE_BYTES + crank * W_SUB_BYTES, &tm_wlo, kb * BK, wrow, fb, CMASK);
          }
          if (++stage == STAGES) { stage = 0; phase ^= 1; }
        }
      }
    }
  } else if (warp == EPI_WARPS + 1) {
    // ===== MMA issuer (one thread): one fresh TMEM partial per k-block =====
    if (lane == 0) {
      uint32_t stage = 0, phase = 0, pcount = 0;
      for (int tile = tile0; tile < num_tiles; tile += tile_step) {
        for (int kb0 = 0; kb0 < k_blocks; kb0 += kpp, ++pcount) {
          const uint32_t pb = pcount % NPB, pphase = (pcount / NPB) & 1;
          tc::mbar_wait(pempty0 + 8 * pb, pphase ^ 1);          // the epilogue has pulled this partial
          const uint32_t d_tmem = tmem_base + pb * PB_COLS;
          const int kb1 = min(kb0 + kpp, k_blocks);
          for (int kb = kb0; kb < kb1; ++kb) {
            tc::mbar_wait(full0 + 8 * stage, phase);
            tc::fence_after_sync();
            const uint32_t s0 = base + stage * STAGE;
            // A: canonical no-swizzle K-major tile -- 16-byte pieces 2048 bytes apart along K (leading
            // byte offset), 8-row groups 128 bytes apart along M (stride byte offset); one MMA consumes
            // two pieces (K = 16).  W: rows of BK halves, 128- or 64-byte swizzle, 32 bytes per MMA.
            const uint64_t a_hi = tc::smem_desc_nosw(s0, 2048, 128), a_lo = tc::smem_desc_nosw(s0 + A_TILE_BYTES, 2048, 128);
            const uint64_t b_hi = BK == 64 ? tc::smem_desc_sw128(s0 + 2 * A_TILE_BYTES) : tc::smem_desc_sw64(s0 + 2 * A_TILE_BYTES);
            const uint64_t b_lo = BK == 64 ? tc::smem_desc_sw128(s0 + 2 * A_TILE_BYTES + B_TILE_BYTES)
                                           : tc::smem_desc_sw64(s0 + 2 * A_TILE_BYTES + B_TILE_BYTES);
            // Corrections first (in the first k-block of a partial the accumulator is still ~2^-11 of its final
            // size), hi.hi last.
            if (g.split4) {
#pragma unroll
              for (int k = 0; k < BK / 16; ++k)
                tc::mma_f16_ss(d_tmem, a_lo + (uint64_t)(256 * k), b_lo + (uint64_t)(2 * k), IDESC, (k != 0) | (kb != kb0));
            }
#pragma unroll
            for (int k = 0; k < BK / 16; ++k) {
              const uint64_t adv_a = (uint64_t)(256 * k), adv_b = (uint64_t)(2 * k);
              tc::mma_f16_ss(d_tmem, a_lo + adv_a, b_hi + adv_b, IDESC, (k != 0) | (kb != kb0) | (g.split4 != 0));
              tc::mma_f16_ss(d_tmem, a_hi + adv_a, b_lo + adv_b, IDESC, 1);
            }
#pragma unroll
            for (int k = 0; k < BK / 16; ++k) {
              const uint64_t adv_a = (uint64_t)(256 * k), adv_b = (uint64_t)(2 * k);
              tc::mma_f16_ss(d_tmem, a_hi + adv_a, b_hi + adv_b, IDESC, 1);
            }
            if (CS == 1) tc::mma_commit(empty0 + 8 * stage);      // smem slot free when these MMAs retire
            else tc::mma_commit_mc(empty0 + 8 * stage, CMASK);    // ... in every CTA that multicasts into it
            if (++stage == STAGES) { stage = 0; phase ^= 1; }
          }
          tc::mma_commit(pfull0 + 8 * pb);                        // partial complete
        }
      }
    }
  }
  } else {
    asm volatile("setmaxnreg.inc.sync.aligned.u32 232;");
    // ===== epilogue warps: TMEM lanes 32 (warp % 4) .., columns CPT (warp / 4) .. =====
    // The accumulators of a tile live in registers, so its epilogue can overlap only the two k-blocks of the next
    // tile that the partial ring holds.  To shorten that critical section the last DEFP column pairs of a finished
    // tile are parked in spare registers and processed, 16 columns at a time, in the idle slots after the next
    // tile's first drains.
    constexpr int NPAIR = CPT / 2;
    constexpr int DEFP = (NPAIR >= 48) ? (EPI == 0 ? DEFER_PAIRS : DEFER_PAIRS - 8) : 0;   // the output epilogue needs more temporaries
    constexpr int IMM = NPAIR - DEFP, NCH = DEFP / 8;
    const int q = warp & 3, hcol = warp >> 2;
    uint32_t pcount = 0;
    f32x2 prev[DEFP > 0 ? DEFP : 1];
    TileRef pt = {0, 0, 0, 0, false};
    int pdone = NCH;                                            // deferred chunks already processed (NCH: none pending)
#define NSGPU_CHUNK_CASE(i) \
  if ((c_) == (i) && DEFP > 8 * (i)) epi_pairs<EPI, IMM + (DEFP > 8 * (i) ? 8 * (i) : 0), 8>(prev + (DEFP > 8 * (i) ? 8 * (i) : 0), pt, g, params)
#define NSGPU_RUN_CHUNK(c)                                                          \
  do {                                                                              \
    const int c_ = (c);                                                             \
    NSGPU_CHUNK_CASE(0); NSGPU_CHUNK_CASE(1); NSGPU_CHUNK_CASE(2); NSGPU_CHUNK_CASE(3); NSGPU_CHUNK_CASE(4); NSGPU_CHUNK_CASE(5); \
  } while (0)
    for (int tile = tile0; tile < num_tiles; tile += tile_step) {
      const int m_grp = tile / n_blocks, n_blk = tile - m_grp * n_blocks;
      const int m_blk = min(m_grp * CS + crank, m_blocks - 1);
      f32x2 acc[NPAIR];
      for (int kb = 0; kb < k_blocks; kb += kpp, ++pcount) {
        const uint32_t pb = pcount % NPB, pphase = (pcount / NPB) & 1;
        tc::mbar_wait(pfull0 + 8 * pb, pphase);
        tc::fence_after_sync();
        const uint32_t t_src = tmem_base + pb * PB_COLS + ((uint32_t)(q * 32) << 16) + hcol * CPT;
        // Two tcgen05.ld in flight per wait: the drain of a partial is a chain of load round trips on the tile's
        // critical path (one load per wait: hidden GEMMs 6% slower); four would not leave registers for the deferral.
        constexpr int NLD = CPT / LDC, DB = 2;
#pragma unroll
        for (int c0 = 0; c0 < NLD; c0 += DB) {
          uint32_t r[DB][LDC];
#pragma unroll
          for (int b = 0; b < DB; ++b)
            if (c0 + b < NLD) tc::tmem_ld_cols(t_src + LDC * (c0 + b), r[b]);
          tc::tmem_ld_wait();
#pragma unroll
          for (int b = 0; b < DB; ++b) {
            if (c0 + b >= NLD) continue;
            const int c = c0 + b;
            if (kb == 0) {
#pragma unroll
              for (int j = 0; j < LDC / 2; ++j) acc[(LDC / 2) * c + j] = pk2(__uint_as_float(r[b][2 * j]), __uint_as_float(r[b][2 * j + 1]));
            } else {
#pragma unroll
              for (int j = 0; j < LDC / 2; ++j)
                acc[(LDC / 2) * c + j] = add2(acc[(LDC / 2) * c + j], pk2(__uint_as_float(r[b][2 * j]), __uint_as_float(r[b][2 * j + 1])));
            }
          }
        }
        tc::fence_before_sync();
        __syncwarp();
        if (lane == 0) tc::mbar_arrive(pempty0 + 8 * pb);
        if (DEFP > 0 && pdone < NCH && (kb >= 1 || kpp > 1)) { NSGPU_RUN_CHUNK(pdone); ++pdone; }
      }
      while (DEFP > 0 && pdone < NCH) { NSGPU_RUN_CHUNK(pdone); ++pdone; }   // short K: not enough idle slots
      const int r_in = q * 32 + lane;
      const TileRef ct = {m_blk, n_blk * BLOCK_N + hcol * CPT, r_in, m_blk * BLOCK_M + r_in, m_blk * BLOCK_M + r_in < M};
      if (EPI == 1 && n_blk == 0 && hcol == 0 && ct.row_ok) {
        // Hidden activations travel as fp16 hi/lo of 16 h: |h| >= 4094 overflows to inf, the next layer turns that into
        // NaN for the whole row, and chi^2 maps it to log L = -inf.  Count such rows so that this is never silent.
        float v0, v1;
        upk2(acc[0], v0, v1);
        if (!(fabsf(v0) <= 3.0e38f)) atomicAdd(g.nonfinite, 1ull);
      }
      epi_pairs<EPI, 0, IMM>(acc, ct, g, params);
      if (DEFP > 0) {
#pragma unroll
        for (int i = 0; i < DEFP; ++i) prev[i] = acc[IMM + i];
        pt = ct;
        pdone = 0;
      }
    }
    while (DEFP > 0 && pdone < NCH) { NSGPU_RUN_CHUNK(pdone); ++pdone; }
#undef NSGPU_RUN_CHUNK
#undef NSGPU_CHUNK_CASE
  }
  tc::fence_before_sync();
  __syncthreads();
  if (CS > 1) tc::cluster_sync();        // no CTA leaves while a peer can still write into its shared memory
  if (warp == EPI_WARPS + 1) tc::tmem_dealloc(tmem_base, 512);
}

// =====================================================================================================
// Fused multi-layer kernel: a CTA pair owns 128-row blocks through ALL layers ("fused MLP").
//
// The layered path launches one kernel per layer and round-trips every activation plane through HBM (2 KB per row and
// layer each way: 2.5 GB of the 3.85 GB a c3a step moved in round 1) and pays a launch boundary per layer (40% of a
// nested-sampling round at B ~ 300-500).  Here a cluster of two CTAs takes row blocks cl, cl + NC, ... and carries
// each of them from theta to the spectrum table: CTA `crank` computes column half `crank` of every hidden layer (the
// first one on the CUDA cores, the others on the tensor cores exactly as mlp_gemm_tc does: same k-block order, same
// partials, same epilogue arithmetic, so the results are bit-identical to the layered path) and every second column
// block of the output layer.  Activations live in a per-cluster scratch in global memory -- two slots (row blocks in
// flight) x two buffers (layer in / layer out) x 256 KB, 74 MB for 74 clusters -- that is rewritten for every row block
// and therefore stays in the 126 MB L2.  Layers are separated by an mbarrier both CTAs arrive on (`ready[slot]`), not
// by a grid-wide barrier.  Two row blocks are interleaved (A1 B1 A2 B2 ...): the epilogue of (A, l) runs while the
// tensor core works on (B, l), and (A, l + 1) starts as soon as both halves of (A, l) are stored.
//
// ready[slot] completes once per (group, layer 0 .. n_layers-1) after 2 x 8 warp arrivals (both CTAs' epilogue warps,
// each after its last store of that layer's output, fence.proxy.async, release at cluster scope); the TMA producer
// waits for it (acquire at cluster scope) before the first bulk copy of the next layer's A operand.  The first layer
// of the NEXT group is computed by the epilogue warps in the gaps between TMEM drains, after ready[slot] has
// completed for layer n_layers-1 of the current group (the last reader of that buffer, in both CTAs).
// =====================================================================================================
constexpr int FUSED_BN_H = 256;
constexpr int FUSED_STAGES = 2;
constexpr int FUSED_STAGE = stage_bytes(256, 64);       // 96 KB: room for the widest tile (output tiles use less)
constexpr int FUSED_MAX_GEMM = 6;                       // GEMM layers (n_hidden) the argument block holds
constexpr int FL_UNIT_PIECES = 4;                       // first layer: 16-byte pieces per work unit and warp
constexpr int FL_UNITS = 16 / FL_UNIT_PIECES;           // a warp owns 16 of the CTA's 32 pieces

struct FusedArgs {
  int M_host;
  const int* n_rows_dev;
  int rows_per_theta;
  int n_layers;               // GEMM layers = n_hidden: layers 1 .. n_layers-1 hidden, layer n_layers the output
  // first layer (a2 + layer 0)
  const float* theta; int D; const int* emu_in_idx; const double* emu_in_const; int n_theta_in; const float* z_emu;
  const float* in_mean; const float* in_std; const float* W0;
  const float4* p_hidden[FUSED_MAX_GEMM];   // per-column parameters of layers 0 .. n_layers-1 (global, [512])
  float cscale[FUSED_MAX_GEMM + 1];         // GEMM layer l = 1 .. n_layers
  // output layer
  const float4* p_out4; int n_blocks_out; int n_valid;
  float* out_f32; int ld_f32; int out_mode; int apply_exp10;
  unsigned long long* nonfinite;
  __half* scratch;            // [clusters][2 slots][2 buffers][hi, lo][128 x 512]
};
struct FusedMaps { CUtensorMap hi[FUSED_MAX_GEMM], lo[FUSED_MAX_GEMM]; };   // index l - 1 for GEMM layer l

// One unit of the first layer for row block `rb`: FL_UNIT_PIECES 16-byte pieces (8 neurons each) of this warp's share of
// the CTA's column half, for the 32 rows of the warp's quarter.  Same arithmetic, in the same order, as
// mlp_first_layer_tc.
template <int NIN>
__device__ __forceinline__ void fused_first_layer_unit(const FusedArgs& f, int rb, int unit, int M, int crank, int warp, int lane,
                                                       const float* sW0, const float4* sp0, __half* out_hi, __half* out_lo) {
  const int r = (warp & 3) * 32 + lane;
  const int m = min(rb * BLOCK_M + r, M - 1);
  const int th = m / f.rows_per_theta, zi = m - th * f.rows_per_theta;
  f32x2 x2[NIN];
#pragma unroll
  for (int c = 0; c < NIN; ++c) {
    float v;
    if (c < f.n_theta_in) {
      const int src = f.emu_in_idx[c];
      v = src >= 0 ? f.theta[(size_t)th * f.D + src] : (float)f.emu_in_const[c];
    } else {
      v = f.z_emu[zi];
    }
    v = (v - f.in_mean[c]) / f.in_std[c];
    x2[c] = pk2(v, v);
  }
  const f32x2 one2 = pk2(1.0f, 1.0f);
  const int p_first = (warp >> 2) * 16 + unit * FL_UNIT_PIECES;            // piece within the CTA's half (0 .. 31)
#pragma unroll 1
  for (int pp = 0; pp < FL_UNIT_PIECES; ++pp) {
    const int p = p_first + pp;
    uint32_t hi[4], lo[4];
    f32x2 t[4] = {0ull, 0ull, 0ull, 0ull};
#pragma unroll
    for (int c = 0; c < NIN; ++c) {
      const float4 wlo = *reinterpret_cast<const float4*>(sW0 + c * FUSED_BN_H + 8 * p);
      const float4 whi = *reinterpret_cast<const float4*>(sW0 + c * FUSED_BN_H + 8 * p + 4);
      t[0] = fma2(x2[c], pk2(wlo.x, wlo.y), t[0]); t[1] = fma2(x2[c], pk2(wlo.z, wlo.w), t[1]);
      t[2] = fma2(x2[c], pk2(whi.x, whi.y), t[2]); t[3] = fma2(x2[c], pk2(whi.z, whi.w), t[3]);
    }
#pragma unroll
    for (int jj = 0; jj < 4; ++jj) act_split_pair(t[jj], one2, sp0[8 * p + 2 * jj], sp0[8 * p + 2 * jj + 1], hi[jj], lo[jj]);
    const size_t o = (size_t)(32 * crank + p) * PIECE_HALVES + (size_t)r * 8;
    *reinterpret_cast<uint4*>(out_hi + o) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
    *reinterpret_cast<uint4*>(out_lo + o) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
  }
}


struct FusedCtx {             // what the epilogue helpers of mlp_fused_tc need besides the tile state
  uint32_t ready0;
  int lane, warp, crank, cl, NC, nl, M;
  __half* scr;
  const float* sW0;
  const float4* sparams;
};

// this warp's stores of one layer of one row block are done: arrive on ready[slot] of both CTAs
__device__ __forceinline__ void fused_signal_ready(const FusedCtx& fc, int slot) {
  tc::fence_proxy_async_all();
  __syncwarp();
  if (fc.lane == 0) { tc::mbar_arrive_cluster(fc.ready0 + 8 * slot, 0); tc::mbar_arrive_cluster(fc.ready0 + 8 * slot, 1); }
}

// First layer of the row block of group g that goes into slot s (this CTA's column half, this warp's share).  Called only
// where no accumulators are live: before the first tile, and at the end of a tile.
template <int NIN>
__device__ __forceinline__ void fused_run_first_layer(const FusedArgs& f, const FusedCtx& fc, int s, int g) {
  constexpr size_t PLANE = (size_t)BLOCK_M * 2 * FUSED_BN_H;
  if (g > 0)      // buffer 0 of the slot was last read by layer nl - 1 of group g - 1, in both CTAs
    tc::mbar_wait_cluster(fc.ready0 + 8 * s, (uint32_t)(((g - 1) * fc.nl + fc.nl - 1) & 1));
  __half* o_hi = fc.scr + (size_t)(s * 2) * (2 * PLANE);
#pragma unroll 1
  for (int u = 0; u < FL_UNITS; ++u)
    fused_first_layer_unit<NIN>(f, fc.cl + (2 * g + s) * fc.NC, u, fc.M, fc.crank, fc.warp, fc.lane, fc.sW0, fc.sparams, o_hi, o_hi + PLANE);
  fused_signal_ready(fc, s);
}

__global__ void exp10_inplace_kernel(float* y, size_t n) {
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) y[i] = exp10f(y[i]);
}

template <int BN_O, int NIN, int OUT_MODE>
__global__ void __launch_bounds__(GEMM_THREADS, 1) mlp_fused_tc(const __grid_constant__ FusedMaps tm, const FusedArgs f) {
  constexpr int BK = 64, A_TILE_BYTES = a_tile_bytes(BK);
  constexpr int STAGES = FUSED_STAGES, STAGE = FUSED_STAGE;
  constexpr int WIDTH = 2 * FUSED_BN_H;
  constexpr int NPB = 2, PB_COLS = 256;
  constexpr uint32_t IDESC_H = tc::idesc_f16_f32(BLOCK_M, FUSED_BN_H), IDESC_O = tc::idesc_f16_f32(BLOCK_M, BN_O);
  constexpr size_t PLANE = (size_t)BLOCK_M * WIDTH;            // halves per plane of a row block
  static_assert(BN_O % 32 == 0 && BN_O <= 256, "output tile width");

  extern __shared__ unsigned char smem_dyn[];
  const uint32_t base = (tc::smem_u32(smem_dyn) + 1023u) & ~1023u;
  unsigned char* base_ptr = smem_dyn + (base - tc::smem_u32(smem_dyn));
  const uint32_t bars = base + STAGES * STAGE;
  const uint32_t full0 = bars, empty0 = bars + 16, pfull0 = bars + 32, pempty0 = bars + 48, ready0 = bars + 64;
  uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(base_ptr + STAGES * STAGE + 96);
  float4* sparams = reinterpret_cast<float4*>(base_ptr + STAGES * STAGE + 128);      // [n_layers][256] (layer 0 first)
  float* sW0 = reinterpret_cast<float*>(sparams + f.n_layers * FUSED_BN_H);          // [NIN][256]

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int crank = (int)tc::cluster_ctarank();
  const int c0 = crank * FUSED_BN_H;                               // first column of this CTA's half of a hidden layer
  if (threadIdx.x == 0) {
    for (int s = 0; s < STAGES; ++s) { tc::mbar_init(full0 + 8 * s, 1); tc::mbar_init(empty0 + 8 * s, 1); }
    for (int b = 0; b < NPB; ++b) { tc::mbar_init(pfull0 + 8 * b, 1); tc::mbar_init(pempty0 + 8 * b, EPI_WARPS); }
    for (int s = 0; s < 2; ++s) tc::mbar_init(ready0 + 8 * s, 2 * EPI_WARPS);
    tc::fence_barrier_init();
  }
  if (warp == EPI_WARPS + 1) tc::tmem_alloc(tc::smem_u32(tmem_slot), 512);
  if (warp == EPI_WARPS && lane == 0)
    for (int l = 0; l < f.n_layers; ++l) { tc::prefetch_tmap(&tm.hi[l]); tc::prefetch_tmap(&tm.lo[l]); }
  // constants: the per-column parameters of this CTA's half of every hidden layer, and its half of W0
  for (int l = 0; l < f.n_layers; ++l)
    for (int i = threadIdx.x; i < FUSED_BN_H / 2; i += blockDim.x) {
      const float4 a = f.p_hidden[l][c0 + 2 * i], b = f.p_hidden[l][c0 + 2 * i + 1];
      sparams[l * FUSED_BN_H + 2 * i] = make_float4(a.x, b.x, a.y, b.y);
      sparams[l * FUSED_BN_H + 2 * i + 1] = make_float4(a.z, b.z, a.w, b.w);
    }
  for (int i = threadIdx.x; i < NIN * FUSED_BN_H; i += blockDim.x) {
    const int c = i / FUSED_BN_H, j = i - c * FUSED_BN_H;
    sW0[i] = f.W0[c * WIDTH + c0 + j];
  }
  pdl_wait();
  pdl_trigger();
  tc::fence_before_sync();
  __syncthreads();
  tc::cluster_sync();          // both CTAs' barriers exist before the peer's first arrive reaches them
  tc::fence_after_sync();
  const uint32_t tmem_base = *tmem_slot;
  int M = f.M_host;
  if (f.n_rows_dev) M = min(M, (*f.n_rows_dev) * f.rows_per_theta);
  const int m_blocks = (M + BLOCK_M - 1) / BLOCK_M;
  const int cl = blockIdx.x >> 1, NC = gridDim.x >> 1;
  const int n_rb = cl < m_blocks ? (m_blocks - cl + NC - 1) / NC : 0;   // row blocks cl, cl + NC, ... of this cluster
  const int n_groups = (n_rb + 1) >> 1;
  const int nl = f.n_layers;
  __half* const scr = f.scratch + (size_t)cl * (8 * PLANE);            // [slot][buffer][hi, lo][PLANE]
  auto buf_hi = [&](int slot, int b) -> __half* { return scr + (size_t)(slot * 2 + b) * (2 * PLANE); };

  if (warp >= EPI_WARPS) {
    // registers: the producer and MMA threads walk a five-deep loop nest with 64-bit descriptors and pointers: with the 40
    // registers mlp_gemm_tc leaves them they spilled into local memory on the MMA issue path (ncu: 1.2 M local loads per
    // launch from single lanes).  56 here, 224 for the epilogue warps: what the third warpgroup gives up ((168 - 56) x 128
    // registers) is exactly what the two epilogue warpgroups take ((224 - 168) x 256); asking for more never returns.
    asm volatile("setmaxnreg.dec.sync.aligned.u32 56;");
    if (warp == EPI_WARPS) {
      // ===== TMA producer =====
      if (lane == 0) {
        uint32_t stage = 0, phase = 0;
        for (int g = 0; g < n_groups; ++g) {
          const int ns = min(2, n_rb - 2 * g);
          for (int l = 1; l <= nl; ++l)
            for (int s = 0; s < ns; ++s) {
              const bool is_out = l == nl;
              const int n_nb = is_out ? f.n_blocks_out : 2, bn = is_out ? BN_O : FUSED_BN_H;
              // layer l - 1 of this row block is complete in both CTAs (completion g nl + l - 1 of ready[s])
              tc::mbar_wait_cluster(ready0 + 8 * s, (uint32_t)((g * nl + l - 1) & 1));
              tc::fence_proxy_async_all();
              const __half* a_hi = buf_hi(s, (l - 1) & 1);
              const __half* a_lo = a_hi + PLANE;
              const uint32_t bytes = 2 * A_TILE_BYTES + 2 * bn * 128;
              for (int nb = crank; nb < n_nb; nb += 2)
#pragma unroll 1
                for (int kb = 0; kb < WIDTH / BK; ++kb) {
                  tc::mbar_wait(empty0 + 8 * stage, phase ^ 1);
                  const uint32_t s0 = base + stage * STAGE, fb = full0 + 8 * stage;
                  tc::mbar_arrive_expect_tx(fb, bytes);
                  const size_t a_off = (size_t)kb * 8 * PIECE_HALVES;
                  tc::bulk_load(s0, a_hi + a_off, A_TILE_BYTES, fb);
                  tc::bulk_load(s0 + A_TILE_BYTES, a_lo + a_off, A_TILE_BYTES, fb);
                  tc::tma_load_2d(s0 + 2 * A_TILE_BYTES, &tm.hi[l - 1], kb * BK, nb * bn, fb);
                  tc::tma_load_2d(s0 + 2 * A_TILE_BYTES + bn * 128, &tm.lo[l - 1], kb * BK, nb * bn, fb);
                  if (++stage == STAGES) { stage = 0; phase ^= 1; }
                }
            }
        }
      }
    } else if (warp == EPI_WARPS + 1) {
      // ===== MMA issuer: one fresh TMEM partial per k-block, as in mlp_gemm_tc =====
      if (lane == 0) {
        uint32_t stage = 0, phase = 0, pcount = 0;
        for (int g = 0; g < n_groups; ++g) {
          const int ns = min(2, n_rb - 2 * g);
          for (int l = 1; l <= nl; ++l)
            for (int s = 0; s < ns; ++s) {
              const bool is_out = l == nl;
              const int n_nb = is_out ? f.n_blocks_out : 2, bn = is_out ? BN_O : FUSED_BN_H;
              const uint32_t idesc = is_out ? IDESC_O : IDESC_H;
              for (int nb = crank; nb < n_nb; nb += 2)
#pragma unroll 1
                for (int kb = 0; kb < WIDTH / BK; ++kb, ++pcount) {
                  const uint32_t pb = pcount % NPB, pphase = (pcount / NPB) & 1;
                  tc::mbar_wait(pempty0 + 8 * pb, pphase ^ 1);
                  tc::mbar_wait(full0 + 8 * stage, phase);
                  tc::fence_after_sync();
                  const uint32_t d_tmem = tmem_base + pb * PB_COLS;
                  const uint32_t s0 = base + stage * STAGE;
                  const uint64_t a_hi = tc::smem_desc_nosw(s0, 2048, 128), a_lo = tc::smem_desc_nosw(s0 + A_TILE_BYTES, 2048, 128);
                  const uint64_t b_hi = tc::smem_desc_sw128(s0 + 2 * A_TILE_BYTES);
                  const uint64_t b_lo = tc::smem_desc_sw128(s0 + 2 * A_TILE_BYTES + bn * 128);
#pragma unroll
                  for (int k = 0; k < BK / 16; ++k) {
                    const uint64_t adv_a = (uint64_t)(256 * k), adv_b = (uint64_t)(2 * k);
                    tc::mma_f16_ss(d_tmem, a_lo + adv_a, b_hi + adv_b, idesc, k != 0);
                    tc::mma_f16_ss(d_tmem, a_hi + adv_a, b_lo + adv_b, idesc, 1);
                  }
#pragma unroll
                  for (int k = 0; k < BK / 16; ++k) {
                    const uint64_t adv_a = (uint64_t)(256 * k), adv_b = (uint64_t)(2 * k);
                    tc::mma_f16_ss(d_tmem, a_hi + adv_a, b_hi + adv_b, idesc, 1);
                  }
                  tc::mma_commit(empty0 + 8 * stage);
                  tc::mma_commit(pfull0 + 8 * pb);
                  if (++stage == STAGES) { stage = 0; phase ^= 1; }
                }
            }
        }
      }
    }
  } else {
    asm volatile("setmaxnreg.inc.sync.aligned.u32 224;");
    // ===== epilogue warps: drains + epilogues of the GEMM tiles, and the first layer of the row blocks to come =====
    const int q = warp & 3, hcol = warp >> 2;
    const int r_in = q * 32 + lane;
    uint32_t pcount = 0;
    int armed[2] = {-1, -1};                       // group whose first layer may be computed into slot s (-1: none)
    FusedCtx fc;
    fc.ready0 = ready0; fc.lane = lane; fc.warp = warp; fc.crank = crank; fc.cl = cl; fc.NC = NC; fc.nl = nl; fc.M = M;
    fc.scr = scr; fc.sW0 = sW0; fc.sparams = sparams;
    if (n_rb > 0) fused_run_first_layer<NIN>(f, fc, 0, 0);
    if (n_rb > 1) fused_run_first_layer<NIN>(f, fc, 1, 0);

// One GEMM tile on the epilogue side: pull the eight k-block partials out of TMEM into registers (round-to-nearest
// sums), then bias + activation + split (hidden) or de-standardisation (output) and the stores.  No deferred columns
// here (mlp_gemm_tc parks the last 64 of a tile): the next layer of this row block waits for exactly these stores.
#define NSGPU_FUSED_TILE(EPI_, BN_, PARAMS_, CS_, OHI_, OLO_, TREF_, SLOT_)                                          \
  do {                                                                                                              \
    constexpr int CPT = BN_ / (EPI_WARPS / 4), NPAIR = CPT / 2, LDC = (CPT % 16 == 0) ? 16 : 8;                     \
    _Pragma("unroll 1") for (int kb = 0; kb < WIDTH / BK; ++kb, ++pcount) {                                         \
      const uint32_t pb = pcount % NPB, pphase = (pcount / NPB) & 1;                                                \
      tc::mbar_wait(pfull0 + 8 * pb, pphase);                                                                       \
      tc::fence_after_sync();                                                                                       \
      const uint32_t t_src = tmem_base + pb * PB_COLS + ((uint32_t)(q * 32) << 16) + hcol * CPT;                    \
      constexpr int NLD = CPT / LDC, DB = 2;                                                                        \
      _Pragma("unroll") for (int c0_ = 0; c0_ < NLD; c0_ += DB) {                                                   \
        uint32_t r[DB][LDC];                                                                                        \
        _Pragma("unroll") for (int b = 0; b < DB; ++b)                                                              \
          if (c0_ + b < NLD) tc::tmem_ld_cols(t_src + LDC * (c0_ + b), r[b]);                                       \
        tc::tmem_ld_wait();                                                                                         \
        _Pragma("unroll") for (int b = 0; b < DB; ++b) {                                                            \
          if (c0_ + b >= NLD) continue;                                                                             \
          const int c = c0_ + b;                                                                                    \
          if (kb == 0) {                                                                                            \
            _Pragma("unroll") for (int j = 0; j < LDC / 2; ++j)                                                     \
              acc[(LDC / 2) * c + j] = pk2(__uint_as_float(r[b][2 * j]), __uint_as_float(r[b][2 * j + 1]));         \
          } else {                                                                                                  \
            _Pragma("unroll") for (int j = 0; j < LDC / 2; ++j)                                                     \
              acc[(LDC / 2) * c + j] = add2(acc[(LDC / 2) * c + j], pk2(__uint_as_float(r[b][2 * j]), __uint_as_float(r[b][2 * j + 1]))); \
          }                                                                                                         \
        }                                                                                                           \
      }                                                                                                             \
      tc::fence_before_sync();                                                                                      \
      __syncwarp();                                                                                                 \
      if (lane == 0) tc::mbar_arrive(pempty0 + 8 * pb);                                                             \
    }                                                                                                               \
    const TileRef ct = TREF_;                                                                                       \
    GemmArgs g_;                                                                                                    \
    g_.rows_per_theta = f.rows_per_theta; g_.n_valid = f.n_valid; g_.p_out4 = f.p_out4; g_.ld_out = WIDTH;          \
    g_.out_f32 = f.out_f32; g_.ld_f32 = f.ld_f32; g_.out_mode = OUT_MODE; g_.apply_exp10 = 0;                       \
    g_.cscale = CS_; g_.out_hi = OHI_; g_.out_lo = OLO_;                                                            \
    if (EPI_ == 1 && ct.n0 == 0 && ct.row_ok) {                                                                     \
      float v0, v1;                                                                                                 \
      upk2(acc[0], v0, v1);                                                                                         \
      if (!(fabsf(v0) <= 3.0e38f)) atomicAdd(f.nonfinite, 1ull);                                                    \
    }                                                                                                               \
    epi_pairs<EPI_, 0, NPAIR, OUT_MODE>(acc, ct, g_, PARAMS_);                                                      \
    if (EPI_ == 0) fused_signal_ready(fc, SLOT_);                                                                   \
    /* first layer of the row block that takes a slot next, armed by an EARLIER tile */                            \
    _Pragma("unroll") for (int s_ = 0; s_ < 2; ++s_)                                                                \
      if (armed[s_] >= 0) { fused_run_first_layer<NIN>(f, fc, s_, armed[s_]); armed[s_] = -1; }                     \
  } while (0)

    f32x2 acc[FUSED_BN_H / 4];                     // one accumulator row segment: 128 columns (hidden), BN_O / 2 (output)
    for (int g = 0; g < n_groups; ++g) {
      const int ns = min(2, n_rb - 2 * g);
      for (int l = 1; l <= nl; ++l)
        for (int s = 0; s < ns; ++s) {
          const int rb = cl + (2 * g + s) * NC;
          if (l < nl) {
            __half* o_hi = buf_hi(s, l & 1);
            __half* o_lo = o_hi + PLANE;
            const float* prm = reinterpret_cast<const float*>(sparams + l * FUSED_BN_H) - 4 * c0;
            // hidden tile: m_blk 0 (the scratch holds one row block), columns c0 + hcol CPT ..
            NSGPU_FUSED_TILE(0, FUSED_BN_H, prm, f.cscale[l], o_hi, o_lo,
                             (TileRef{0, c0 + hcol * CPT, r_in, rb * BLOCK_M + r_in, rb * BLOCK_M + r_in < M}), s);
            // the first layer of the row block that takes this slot next may start once layer nl - 1 here is done
            if (l == nl - 1 && 2 * (g + 1) + s < n_rb) armed[s] = g + 1;
          } else {
            for (int nb = crank; nb < f.n_blocks_out; nb += 2)
              NSGPU_FUSED_TILE(1, BN_O, nullptr, f.cscale[l], nullptr, nullptr,
                               (TileRef{rb, nb * BN_O + hcol * CPT, r_in, rb * BLOCK_M + r_in, rb * BLOCK_M + r_in < M}), s);
          }
        }
    }
#undef NSGPU_FUSED_TILE
  }
  tc::fence_before_sync();
  __syncthreads();
  tc::cluster_sync();
  if (warp == EPI_WARPS + 1) tc::tmem_dealloc(tmem_base, 512);
}

}  // namespace

// ---------------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------------
namespace {

struct TcLayer {
  int K = 0, N_pad = 0, n_valid = 0, block_n = 0, wexp = 0;
  __half *Whi = nullptr, *Wlo = nullptr;     // [N_pad][K] K-major, scaled by 2^wexp
  float4* p_hidden = nullptr;                // layers 0 .. n_hidden-1
  float2 *p_out = nullptr, *p_out_nm = nullptr;     // output layer (with / without mu_out)
  float4 *p_out4 = nullptr, *p_out4_nm = nullptr;
  CUtensorMap tm_whi, tm_wlo;                // box = block_n rows
  CUtensorMap tm_whi_s[2], tm_wlo_s[2];      // hidden layers: boxes of 128 and 64 rows for small batches
  bool has_s[2] = {false, false};
  CUtensorMap tm_whi_c, tm_wlo_c;            // boxes of block_n / 2 rows: one CTA's multicast share of a tile
  bool has_c = false;
};

struct TcState {
  std::vector<TcLayer> layers;               // index = layer 0 .. n_hidden (layer 0 uses p_hidden only)
  __half* act[2][2] = {};                    // [buffer][hi, lo] canonical-layout planes
  void* own_act[2] = {nullptr, nullptr};     // emulators 1.. own their activation buffers (emulator 0 uses ctx->act)
  size_t M_pad = 0;
  bool fused_ok = false;                     // shapes the fused multi-layer kernel takes (mlp_fused_tc)
  FusedMaps fmaps;
  // k-block (64 or 32 columns) and k-blocks per TMEM partial.  Measured (profiles/r2_gemm_pipeline_ab.md): four stages of
  // 32 columns are no faster than two of 64 (the kernel is bound by the chip's power cap, not by operand latency), and
  // every further k-block in a partial costs precision (more truncating accumulations) for 3-5% of time.  NSGPU_BK /
  // NSGPU_KPP override them for kernel A/B runs.
  int bk = 64;
  int kpp = 1;
};

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = (EncodeTiledFn)p;
  }
  return fn;
}

// fp16 [rows][cols] row-major, box = box_rows x bk columns (128 or 64 bytes) with the swizzle of that width, OOB -> 0
bool make_tmap(CUtensorMap* tm, const void* ptr, size_t rows, size_t cols, int box_rows, int bk) {
  EncodeTiledFn fn = encode_fn();
  if (!fn) return false;
  const cuuint64_t dims[2] = {(cuuint64_t)cols, (cuuint64_t)rows};
  const cuuint64_t strides[1] = {(cuuint64_t)cols * sizeof(__half)};
  const cuuint32_t box[2] = {(cuuint32_t)bk, (cuuint32_t)box_rows};
  const cuuint32_t estr[2] = {1, 1};
  return fn(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 2, const_cast<void*>(ptr), dims, strides, box, estr,
            CU_TENSOR_MAP_INTERLEAVE_NONE, bk == 64 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_64B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

int pick_block_n(int n, bool hidden) {
  if (hidden) return n % 256 == 0 ? 256 : (n % 128 == 0 ? 128 : 64);   // 128 (4 TMEM partials) measured no faster than 256
  const int cand[4] = {256, 224, 128, 64};
  int best = 64, best_pad = 1 << 30;
  for (int c : cand) {
    const int pad = (n + c - 1) / c * c;
    if (pad < best_pad) { best_pad = pad; best = c; }
  }
  return best;
}

template <int BN, int EPI, int BK>
nsgpu_status launch_gemm(nsgpu_ctx* ctx, const CUtensorMap& whi, const CUtensorMap& wlo, const GemmArgs& g, cudaStream_t st) {
  const int smem = num_stages(BN, BK) * stage_bytes(BN, BK) + 16 * num_stages(BN, BK) + 128 + (EPI == 0 ? 16 * g.N_pad : 0) + 1024;
  NSGPU_CUDA(nsgpu_ensure_smem(ctx, mlp_gemm_tc<BN, EPI, 1, BK>, SMEM_BUDGET));
  const int tiles = ((g.M_host + BLOCK_M - 1) / BLOCK_M) * (g.N_pad / BN);
  const int grid = std::min(tiles, ctx->sm_count);
  NSGPU_CUDA(launch_pdl(ctx, mlp_gemm_tc<BN, EPI, 1, BK>, dim3(grid), dim3(GEMM_THREADS), smem, st, whi, wlo, g));
  NSGPU_LAUNCH_CHECK();
  return NSGPU_OK;
}

// Clusters of CS CTAs that share the weight tiles (whi / wlo: tensor maps with boxes of BN / CS rows).
template <int BN, int EPI, int CS, int BK>
nsgpu_status launch_gemm_cluster(nsgpu_ctx* ctx, const CUtensorMap& whi, const CUtensorMap& wlo, const GemmArgs& g,
                                 cudaStream_t st) {
  const int smem = num_stages(BN, BK) * stage_bytes(BN, BK) + 16 * num_stages(BN, BK) + 128 + (EPI == 0 ? 16 * g.N_pad : 0) + 1024;
  NSGPU_CUDA(nsgpu_ensure_smem(ctx, mlp_gemm_tc<BN, EPI, CS, BK>, SMEM_BUDGET));
  const int m_blocks = (g.M_host + BLOCK_M - 1) / BLOCK_M;
  const int items = ((m_blocks + CS - 1) / CS) * (g.N_pad / BN);
  const int clusters = std::min(items, ctx->sm_count / CS);
  cudaLaunchConfig_t cfg;
  memset(&cfg, 0, sizeof(cfg));
  cfg.gridDim = dim3(clusters * CS);
  cfg.blockDim = dim3(GEMM_THREADS);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[2];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = CS; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
  attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;   // see launch_pdl
  attr[1].val.programmaticStreamSerializationAllowed = (ctx->flags & NSGPU_NO_PDL) ? 0 : 1;
  cfg.attrs = attr;
  cfg.numAttrs = 2;
  if (CS > 2) {   // clusters of more than two CTAs do not fit every SM (GPC sizes): a persistent grid must not exceed what is co-resident
    static int max_clusters = -1;
    if (max_clusters < 0) {
      int n = 0;
      if (cudaOccupancyMaxActiveClusters(&n, mlp_gemm_tc<BN, EPI, CS, BK>, &cfg) != cudaSuccess || n < 1) n = ctx->sm_count / CS;
      max_clusters = n;
      if (getenv("NSGPU_VERBOSE")) fprintf(stderr, "nsgpu: clusters of %d: %d co-resident\n", CS, n);
    }
    cfg.gridDim = dim3(std::min(clusters, max_clusters) * CS);
  }
  NSGPU_CUDA(cudaLaunchKernelEx(&cfg, mlp_gemm_tc<BN, EPI, CS, BK>, whi, wlo, g));
  NSGPU_LAUNCH_CHECK();
  return NSGPU_OK;
}

template <int EPI, int BK>
nsgpu_status dispatch_gemm_bk(nsgpu_ctx* ctx, const TcLayer& L, const GemmArgs& g, cudaStream_t st) {
  // Small batches (few 128-row blocks): narrower tiles so that the grid still covers the SMs.
  if (EPI == 0 && (ctx->flags & NSGPU_MLP_CLUSTER) == 0) {
    const int m_blocks = (g.M_host + BLOCK_M - 1) / BLOCK_M;
    int bn = L.block_n;
    while (bn > 64 && m_blocks * (g.N_pad / bn) < ctx->sm_count && L.has_s[bn == 256 ? 0 : 1]) bn >>= 1;
    if (bn != L.block_n) {
      const int i = bn == 128 ? 0 : 1;
      return bn == 128 ? launch_gemm<128, EPI, BK>(ctx, L.tm_whi_s[i], L.tm_wlo_s[i], g, st)
                       : launch_gemm<64, EPI, BK>(ctx, L.tm_whi_s[i], L.tm_wlo_s[i], g, st);
    }
  }
  // Large batches: CTA pairs share the weight tiles (see mlp_gemm_tc).  Clusters of 4 were measured 50% slower than
  // pairs (the lock step of four CTAs costs more than the L2 reads it saves).
  if (L.has_c && (L.block_n == 256 || L.block_n == 224)) {
    const int m_blocks_all = (g.M_host + BLOCK_M - 1) / BLOCK_M;
    bool pair = m_blocks_all * (g.N_pad / L.block_n) >= 2 * ctx->sm_count;
    if (ctx->flags & NSGPU_MLP_NO_CLUSTER) pair = false;
    if (ctx->flags & NSGPU_MLP_CLUSTER) pair = true;
    // kernel A/B runs (NSGPU_CS4): hidden layers in clusters of 4 (each CTA loads a quarter of the weight tile: the 64-row maps)
    static const bool cs4 = getenv("NSGPU_CS4") != nullptr;
    if (pair && cs4 && EPI == 0 && L.block_n == 256 && L.has_s[1])
      return launch_gemm_cluster<256, EPI, 4, BK>(ctx, L.tm_whi_s[1], L.tm_wlo_s[1], g, st);
    if (pair) return L.block_n == 256 ? launch_gemm_cluster<256, EPI, 2, BK>(ctx, L.tm_whi_c, L.tm_wlo_c, g, st)
                                      : launch_gemm_cluster<224, EPI, 2, BK>(ctx, L.tm_whi_c, L.tm_wlo_c, g, st);
  }
  switch (L.block_n) {
    case 256: return launch_gemm<256, EPI, BK>(ctx, L.tm_whi, L.tm_wlo, g, st);
    case 224: return launch_gemm<224, EPI, BK>(ctx, L.tm_whi, L.tm_wlo, g, st);
    case 128: return launch_gemm<128, EPI, BK>(ctx, L.tm_whi, L.tm_wlo, g, st);
    default: return launch_gemm<64, EPI, BK>(ctx, L.tm_whi, L.tm_wlo, g, st);
  }
}

template <int EPI>
nsgpu_status dispatch_gemm(nsgpu_ctx* ctx, const TcLayer& L, const GemmArgs& g, int bk, cudaStream_t st) {
  return bk == 64 ? dispatch_gemm_bk<EPI, 64>(ctx, L, g, st) : dispatch_gemm_bk<EPI, 32>(ctx, L, g, st);
}

}  // namespace

nsgpu_status mlp_tc_prepare(nsgpu_ctx* ctx, int e, const nsgpu_emulator* h) {
  EmuDev& E = ctx->emu[e];
  if (!encode_fn()) { ctx->err = "cuTensorMapEncodeTiled not available from the driver"; return NSGPU_ECUDA; }
  TcState* T = new TcState();
  E.tmaps = T;
  const int width = h->width, nh = h->n_hidden;
  const size_t M_max = (size_t)ctx->max_batch * ctx->rows_per_theta;
  const size_t M_pad = (M_max + BLOCK_M - 1) / BLOCK_M * BLOCK_M;       // api.cu sizes ctx->act for this
  T->M_pad = M_pad;
  if (const char* ev = getenv("NSGPU_BK")) T->bk = atoi(ev) == 64 ? 64 : 32;
  if (const char* ev = getenv("NSGPU_KPP")) T->kpp = std::min(std::max(atoi(ev), 1), 16);
  T->layers.resize(nh + 1);
  const float log2e = 1.4426950408889634f;
  for (int l = 0; l <= nh; ++l) {
    TcLayer& L = T->layers[l];
    const bool hidden = l < nh;
    L.K = l == 0 ? h->n_in : width;
    L.n_valid = hidden ? width : h->n_out;
    L.block_n = pick_block_n(L.n_valid, hidden);
    L.N_pad = (L.n_valid + L.block_n - 1) / L.block_n * L.block_n;
    if (l >= 1) {
      // W[l] is [K][n_valid] row-major at the ABI; the tensor core wants K-major [N_pad][K].
      const float* W = h->W[l];
      float wmax = 0.f;
      for (size_t i = 0; i < (size_t)L.K * L.n_valid; ++i) wmax = std::max(wmax, fabsf(W[i]));
      L.wexp = wmax > 0.f ? (int)floorf(log2f(4096.0f / wmax)) : 0;
      L.wexp = std::min(std::max(L.wexp, -8), 24);
      const float sc = ldexpf(1.0f, L.wexp);
      std::vector<__half> hi((size_t)L.N_pad * L.K, __float2half_rn(0.f)), lo(hi);
      for (int k = 0; k < L.K; ++k)
        for (int n = 0; n < L.n_valid; ++n) {
          const float w = W[(size_t)k * L.n_valid + n] * sc;
          const __half wh = __float2half_rn(w);
          hi[(size_t)n * L.K + k] = wh;
          lo[(size_t)n * L.K + k] = __float2half_rn(w - __half2float(wh));
        }
      NSGPU_CUDA(cudaMalloc((void**)&L.Whi, hi.size() * sizeof(__half)));
      NSGPU_CUDA(cudaMalloc((void**)&L.Wlo, lo.size() * sizeof(__half)));
      NSGPU_CUDA(cudaMemcpy(L.Whi, hi.data(), hi.size() * sizeof(__half), cudaMemcpyHostToDevice));
      NSGPU_CUDA(cudaMemcpy(L.Wlo, lo.data(), lo.size() * sizeof(__half), cudaMemcpyHostToDevice));
      if (!make_tmap(&L.tm_whi, L.Whi, L.N_pad, L.K, L.block_n, T->bk) || !make_tmap(&L.tm_wlo, L.Wlo, L.N_pad, L.K, L.block_n, T->bk)) {
        ctx->err = "cuTensorMapEncodeTiled failed for a weight plane";
        return NSGPU_ECUDA;
      }
      if (L.block_n == 256 || L.block_n == 224)     // multicast shares: boxes of block_n / 2 rows
        L.has_c = make_tmap(&L.tm_whi_c, L.Whi, L.N_pad, L.K, L.block_n / 2, T->bk) && make_tmap(&L.tm_wlo_c, L.Wlo, L.N_pad, L.K, L.block_n / 2, T->bk);
      if (hidden) {   // narrower boxes over the same planes (N_pad = width is a multiple of 64)
        const int bs[2] = {128, 64};
        for (int i = 0; i < 2; ++i)
          L.has_s[i] = bs[i] < L.block_n && L.N_pad % bs[i] == 0 && make_tmap(&L.tm_whi_s[i], L.Whi, L.N_pad, L.K, bs[i], T->bk) &&
                       make_tmap(&L.tm_wlo_s[i], L.Wlo, L.N_pad, L.K, bs[i], T->bk);
      }
    }
    if (hidden) {
      std::vector<float4> p(L.N_pad, make_float4(0.f, 0.f, 0.f, 0.f));
      for (int n = 0; n < width; ++n) {
        const float be = h->beta[l][n];
        p[n] = make_float4(h->b[l][n], -h->alpha[l][n] * log2e, ACT_SCALE * be, ACT_SCALE * (1.0f - be));
      }
      NSGPU_CUDA(cudaMalloc((void**)&L.p_hidden, p.size() * sizeof(float4)));
      NSGPU_CUDA(cudaMemcpy(L.p_hidden, p.data(), p.size() * sizeof(float4), cudaMemcpyHostToDevice));
    } else {
      const float cs = ldexpf(1.0f, -(L.wexp + 4)) * trunc_comp(L.K, T->bk, T->kpp);
      // two parameter sets: with mu_out folded in, and without (NSGPU_SPEC_NOMEAN: the consumer adds mu_out
      // in fp64, so that the fp32 table carries only the O(sigma_out) deviation)
      for (int nomean = 0; nomean < 2; ++nomean) {
        std::vector<float2> p(L.N_pad, make_float2(0.f, 0.f));
        for (int n = 0; n < h->n_out; ++n)
          p[n] = make_float2(cs * h->out_std[n], h->b[l][n] * h->out_std[n] + (nomean ? 0.0f : h->out_mean[n]));
        std::vector<float4> p4(L.N_pad / 2);
        for (int n = 0; n < L.N_pad / 2; ++n) p4[n] = make_float4(p[2 * n].x, p[2 * n + 1].x, p[2 * n].y, p[2 * n + 1].y);
        float2** d2 = nomean ? &L.p_out_nm : &L.p_out;
        float4** d4 = nomean ? &L.p_out4_nm : &L.p_out4;
        NSGPU_CUDA(cudaMalloc((void**)d2, p.size() * sizeof(float2)));
        NSGPU_CUDA(cudaMemcpy(*d2, p.data(), p.size() * sizeof(float2), cudaMemcpyHostToDevice));
        NSGPU_CUDA(cudaMalloc((void**)d4, p4.size() * sizeof(float4)));
        NSGPU_CUDA(cudaMemcpy(*d4, p4.data(), p4.size() * sizeof(float4), cudaMemcpyHostToDevice));
      }
    }
  }
  // fused multi-layer kernel: width 512 (one 256-column tile per CTA of a pair), an even number of GEMM layers, the
  // input counts the BASELINE configurations use, output tiles of 224 or 256 columns, default k-block / partial sizes
  {
    const TcLayer& Lo = T->layers[nh];
    T->fused_ok = width == 2 * FUSED_BN_H && nh % 2 == 0 && nh >= 2 && nh <= FUSED_MAX_GEMM && T->bk == 64 && T->kpp == 1 &&
                  (h->n_in == 6 || h->n_in == 7 || h->n_in == 9) && (Lo.block_n == 224 || Lo.block_n == 256);
    if (T->fused_ok) {
      for (int l = 1; l <= nh; ++l) { T->fmaps.hi[l - 1] = T->layers[l].tm_whi; T->fmaps.lo[l - 1] = T->layers[l].tm_wlo; }
      if (!ctx->fused_scratch) {
        const size_t bytes = (size_t)(ctx->sm_count / 2) * 8 * BLOCK_M * width * sizeof(__half);   // 1 MB per cluster
        NSGPU_CUDA(cudaMalloc(&ctx->fused_scratch, bytes));
        NSGPU_CUDA(cudaMemset(ctx->fused_scratch, 0, bytes));
      }
    }
  }
  for (int i = 0; i < 2; ++i) {
    // emulator 0 ping-pongs through the context's buffers; further emulators (kind 2: TT, TE, EE) get buffers of their own so
    // that the emulators of one likelihood call can run concurrently on separate streams (api.cu run_emulators)
    void* base = ctx->act[i];
    if (e > 0) {
      NSGPU_CUDA(cudaMalloc(&T->own_act[i], M_pad * width * 2 * sizeof(__half)));
      base = T->own_act[i];
    }
    T->act[i][0] = reinterpret_cast<__half*>(base);
    T->act[i][1] = T->act[i][0] + M_pad * width;
    // rows past the live ones are read by the last tile of a batch (results discarded): keep them finite
    NSGPU_CUDA(cudaMemset(base, 0, M_pad * width * 2 * sizeof(__half)));
  }
  return NSGPU_OK;
}

void mlp_tc_release(nsgpu_ctx* ctx, int e) {
  TcState* T = reinterpret_cast<TcState*>(ctx->emu[e].tmaps);
  if (!T) return;
  cudaFree(T->own_act[0]); cudaFree(T->own_act[1]);
  for (TcLayer& L : T->layers) { cudaFree(L.Whi); cudaFree(L.Wlo); cudaFree(L.p_hidden); cudaFree(L.p_out); cudaFree(L.p_out4); cudaFree(L.p_out_nm); cudaFree(L.p_out4_nm); }
  delete T;
  ctx->emu[e].tmaps = nullptr;
}


namespace {

// The fused kernel is OPT-IN (NSGPU_MLP_FUSED).  Measured on B200, c3a (profiles/r2_fused_mlp.md): bit-identical to the
// layered path and half its DRAM traffic, but not faster -- MLP 1.48 vs 1.29 ms at B = 4096 (96 KB of L2 reads per
// k-block and CTA without weight multicast, against 64 KB: the L2 -> SM limit; no deferred epilogue), equal at B = 512,
// 9% better at B = 256, and 2% slower inside a nested-sampling run (rounds of ~300 proposals).
bool use_fused(const nsgpu_ctx* ctx, const TcState* T, int M) {
  (void)M;
  return T->fused_ok && (ctx->flags & NSGPU_MLP_FUSED) != 0 && (ctx->flags & (NSGPU_MLP_LAYERED | NSGPU_MLP_SPLIT4)) == 0;
}

template <int BN_O, int NIN, int OUT_MODE>
nsgpu_status launch_fused(nsgpu_ctx* ctx, const TcState* T, const FusedArgs& f, int smem, cudaStream_t st) {
  NSGPU_CUDA(nsgpu_ensure_smem(ctx, mlp_fused_tc<BN_O, NIN, OUT_MODE>, (size_t)smem));
  const int m_blocks = (f.M_host + BLOCK_M - 1) / BLOCK_M;
  const int clusters = std::min(m_blocks, ctx->sm_count / 2);
  cudaLaunchConfig_t cfg;
  memset(&cfg, 0, sizeof(cfg));
  cfg.gridDim = dim3(clusters * 2);
  cfg.blockDim = dim3(GEMM_THREADS);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = st;
  cudaLaunchAttribute attr[2];
  attr[0].id = cudaLaunchAttributeClusterDimension;
  attr[0].val.clusterDim.x = 2; attr[0].val.clusterDim.y = 1; attr[0].val.clusterDim.z = 1;
  attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  attr[1].val.programmaticStreamSerializationAllowed = (ctx->flags & NSGPU_NO_PDL) ? 0 : 1;
  cfg.attrs = attr;
  cfg.numAttrs = 2;
  NSGPU_CUDA(cudaLaunchKernelEx(&cfg, mlp_fused_tc<BN_O, NIN, OUT_MODE>, T->fmaps, f));
  NSGPU_LAUNCH_CHECK();
  return NSGPU_OK;
}

nsgpu_status mlp_forward_fused(nsgpu_ctx* ctx, const EmuDev& E, TcState* T, const float* theta, int M, const int* n_rows_dev,
                               float* spec_out, int ld_spec, int mode, cudaStream_t st) {
  const int nh = E.n_hidden;
  FusedArgs f;
  memset(&f, 0, sizeof(f));
  f.M_host = M; f.n_rows_dev = n_rows_dev; f.rows_per_theta = ctx->rows_per_theta; f.n_layers = nh;
  f.theta = theta; f.D = ctx->D; f.emu_in_idx = ctx->emu_in_idx; f.emu_in_const = ctx->emu_in_const;
  f.n_theta_in = ctx->n_theta_in; f.z_emu = ctx->z_emu; f.in_mean = E.in_mean; f.in_std = E.in_std; f.W0 = E.W[0];
  for (int l = 0; l < nh; ++l) f.p_hidden[l] = T->layers[l].p_hidden;
  for (int l = 1; l <= nh; ++l) f.cscale[l] = ldexpf(1.0f, -(T->layers[l].wexp + 4)) * trunc_comp(T->layers[l].K, T->bk, T->kpp);
  const TcLayer& Lo = T->layers[nh];
  f.p_out4 = (mode & NSGPU_SPEC_NOMEAN) ? Lo.p_out4_nm : Lo.p_out4;
  f.n_blocks_out = Lo.N_pad / Lo.block_n; f.n_valid = Lo.n_valid;
  f.out_f32 = spec_out; f.ld_f32 = ld_spec; f.out_mode = (mode & NSGPU_SPEC_KZ) ? 1 : 0; f.apply_exp10 = (mode & NSGPU_SPEC_EXP10) ? 1 : 0;
  f.nonfinite = ctx->nonfinite_rows;
  f.scratch = reinterpret_cast<__half*>(ctx->fused_scratch);
  const int smem = FUSED_STAGES * FUSED_STAGE + 128 + nh * FUSED_BN_H * (int)sizeof(float4) + E.n_in * FUSED_BN_H * (int)sizeof(float) + 1024;
  nsgpu_status rs = NSGPU_ESHAPE;
  {
    StageTimer tm(ctx, 1, st);                     // the whole MLP is one launch: booked under the hidden-layer stage
#define NSGPU_FUSED_CASE(BN_, NIN_)                                                                       \
  if (Lo.block_n == BN_ && E.n_in == NIN_)                                                                \
    rs = f.out_mode ? launch_fused<BN_, NIN_, 1>(ctx, T, f, smem, st) : launch_fused<BN_, NIN_, 0>(ctx, T, f, smem, st)
    NSGPU_FUSED_CASE(224, 6); NSGPU_FUSED_CASE(224, 7); NSGPU_FUSED_CASE(224, 9);
    NSGPU_FUSED_CASE(256, 6); NSGPU_FUSED_CASE(256, 7); NSGPU_FUSED_CASE(256, 9);
#undef NSGPU_FUSED_CASE
  }
  if (rs != NSGPU_OK) return rs;
  if (mode & NSGPU_SPEC_EXP10) {                   // emulate tap: 10^y as a pass of its own (same exp10f, same bits)
    const size_t n = (size_t)M * ld_spec;
    exp10_inplace_kernel<<<(unsigned)std::min<size_t>((n + 255) / 256, 65535), 256, 0, st>>>(spec_out, n);
    NSGPU_LAUNCH_CHECK();
  }
  return NSGPU_OK;
}

}  // namespace

nsgpu_status mlp_forward_tc(nsgpu_ctx* ctx, int e, const float* theta, int B, const int* n_rows_dev, float* spec_out,
                            int ld_spec, int mode, cudaStream_t st) {
  const EmuDev& E = ctx->emu[e];
  TcState* T = reinterpret_cast<TcState*>(E.tmaps);
  const int rpt = ctx->rows_per_theta;
  const int M = B * rpt;
  if (M == 0) return NSGPU_OK;
  if (use_fused(ctx, T, M)) return mlp_forward_fused(ctx, E, T, theta, M, n_rows_dev, spec_out, ld_spec, mode, st);
  int cur = 0;
  {
    StageTimer tm(ctx, 0, st);
    const size_t smem = (size_t)E.width * sizeof(float4) + (size_t)E.n_in * E.width * sizeof(float);
    const int fl_tiles = (M + BLOCK_M - 1) / BLOCK_M;
    const int fl_split = fl_tiles >= 4 * ctx->sm_count ? 1 : 4;
    const int fl_grid = fl_tiles * fl_split;
#define NSGPU_FL(N_) case N_: NSGPU_CUDA(launch_pdl(ctx, mlp_first_layer_tc<N_>, dim3(fl_grid), dim3(256), smem, st, ARGS_)); break;
#define ARGS_ theta, ctx->D, rpt, M, n_rows_dev, ctx->emu_in_idx,                                                                       ctx->emu_in_const, ctx->n_theta_in, ctx->z_emu,                                                                       E.n_in, E.in_mean, E.in_std, E.W[0],                                                                       T->layers[0].p_hidden, E.width, fl_split, T->act[0][0],                                                                       T->act[0][1]
    switch (E.n_in) {
      NSGPU_FL(1) NSGPU_FL(2) NSGPU_FL(3) NSGPU_FL(4) NSGPU_FL(5) NSGPU_FL(6) NSGPU_FL(7) NSGPU_FL(8)
      NSGPU_FL(9) NSGPU_FL(10) NSGPU_FL(11) NSGPU_FL(12) NSGPU_FL(13) NSGPU_FL(14) NSGPU_FL(15) NSGPU_FL(16)
      default: ctx->err = "emulator n_in > 16"; return NSGPU_ESHAPE;
    }
#undef ARGS_
#undef NSGPU_FL
    NSGPU_LAUNCH_CHECK();
  }
  for (int l = 1; l <= E.n_hidden; ++l) {
    const TcLayer& L = T->layers[l];
    const bool hidden = l < E.n_hidden;
    GemmArgs g;
    memset(&g, 0, sizeof(g));
    g.M_host = M; g.n_rows_dev = n_rows_dev; g.rows_per_theta = rpt; g.K = L.K; g.N_pad = L.N_pad; g.n_valid = L.n_valid;
    g.p_hidden = L.p_hidden; g.p_out = (mode & NSGPU_SPEC_NOMEAN) ? L.p_out_nm : L.p_out; g.p_out4 = (mode & NSGPU_SPEC_NOMEAN) ? L.p_out4_nm : L.p_out4; g.cscale = ldexpf(1.0f, -(L.wexp + 4)) * trunc_comp(L.K, T->bk, T->kpp); g.kpp = T->kpp; g.split4 = (ctx->flags & NSGPU_MLP_SPLIT4) ? 1 : 0;
    g.a_hi = T->act[cur][0]; g.a_lo = T->act[cur][1];
    g.out_hi = T->act[cur ^ 1][0]; g.out_lo = T->act[cur ^ 1][1]; g.ld_out = E.width;
    g.out_f32 = spec_out; g.ld_f32 = ld_spec; g.apply_exp10 = (mode & NSGPU_SPEC_EXP10) ? 1 : 0;
    g.out_mode = (mode & NSGPU_SPEC_KZ) ? 1 : 0;
    g.nonfinite = ctx->nonfinite_rows;
    StageTimer tm(ctx, hidden ? 1 : 2, st);
    nsgpu_status s = hidden ? dispatch_gemm<0>(ctx, L, g, T->bk, st) : dispatch_gemm<1>(ctx, L, g, T->bk, st);
    if (s != NSGPU_OK) return s;
    cur ^= 1;
  }
  return NSGPU_OK;
}
