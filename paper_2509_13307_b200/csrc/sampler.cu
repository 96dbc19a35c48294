// sampler.cu -- nested sampling with batch deletion and constrained slice sampling (steps a11-a14).
//
// P:L50  "iteratively replaces the point with the lowest likelihood ... evidence accumulated as a sum of
//         likelihood values weighted by successively smaller prior volumes"
// P:L52  slice sampling (Neal 2003) under a hard likelihood constraint, as in Nested Slice Sampling
// P:L62  "selecting k live points with the lowest likelihoods ... evolving them ... in parallel"
// The paper gives prose only; the choices it leaves open are DESIGN.md readings N1-N10.
//
// Design (differs from the paper's vmapped lock-step while-loops, "perfect scaling is hard to
// achieve"): every chain is a resumable state machine owned by one warp (lanes hold the dimensions,
// so the per-chain state lives in registers while the warp runs).  One ROUND = every unfinished chain
// advances until it has exactly one in-box proposal that needs a likelihood (out-of-box proposals
// are rejected on the spot and cost nothing), the proposals are compacted into a dense batch, the
// bulk likelihood runs once on that batch, and the next round consumes the results.  Chains never
// wait for each other inside a slice move.
#include <math.h>
#include <string.h>

#include <algorithm>
#include <chrono>

#include "internal.cuh"

#define MAX_STEP_OUT 32
#define MAX_SHRINK 64
#define BRACKET_W 2.0
#define MAX_LIVE 16384

struct SamplerDev {
  int cap = 0;   // max chains / live points
  cudaStream_t run_stream = nullptr;   // nsgpu_run's own non-blocking stream: runs on different contexts overlap on the GPU
  int rounds_needed = 0, rounds_n_steps = -1;   // rounds the last evolve() took (for that n_steps): sizes the next first burst
  int64_t last_failed_moves = 0;                // slice moves of the last nsgpu_slice_step that hit the shrink cap
  // chain state (SoA)
  float *x0 = nullptr, *dir = nullptr, *xprop = nullptr, *theta_chain = nullptr;   // [cap][D]
  double *l = nullptr, *r = nullptr, *t = nullptr, *logL0 = nullptr;
  int *phase = nullptr, *cnt = nullptr, *step = nullptr, *pending = nullptr, *finished = nullptr, *need = nullptr;
  unsigned* rng_j = nullptr;
  int *row_of_chain = nullptr, *start_idx = nullptr;
  // batch
  float* theta_prop = nullptr;   // [cap][D]
  double* logL_prop = nullptr;   // [cap]
  // scalars: [0] n_active, [1] n_finished, [2] n_fails
  int* counters = nullptr;
  unsigned long long* n_evals = nullptr;
  double* scal = nullptr;        // [0] logL_star, [1] logX, [2] logZ, [3] logZ_live, [4] stop flag
  double* Lsig = nullptr;        // [D][D] lower Cholesky of the live covariance
  // live set and per-iteration outputs (nsgpu_run)
  float* u_live = nullptr;       // [cap][D]
  double* logL_live = nullptr;
  int *dead_idx = nullptr, *surv_idx = nullptr;
  double* logw = nullptr;
  float* u_out = nullptr;
  double* logL_out = nullptr;
  // host mirrors
  int* h_counters = nullptr;           // pinned [4]
  unsigned long long* h_evals = nullptr;
  double* h_scal = nullptr;            // pinned [8]
  // samples of the last nsgpu_run (host): theta [n][D], logL [n], logw [n]
  std::vector<float> last_theta;
  std::vector<double> last_logL, last_logw;
  struct SampleSet { std::vector<float> theta; std::vector<double> logL, logw; };
  std::vector<SampleSet> multi;        // samples of the runs of the last nsgpu_run_multi
};

namespace {

// ---------------- Philox4x32-10 (Salmon et al. 2011), device side ---------------------------------
__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint2 k) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const unsigned hi0 = __umulhi(0xD2511F53u, c.x), lo0 = 0xD2511F53u * c.x;
    const unsigned hi1 = __umulhi(0xCD9E8D57u, c.z), lo1 = 0xCD9E8D57u * c.z;
    c = make_uint4(hi1 ^ c.y ^ k.x, lo1, hi0 ^ c.w ^ k.y, lo0);
    k.x += 0x9E3779B9u;
    k.y += 0xBB67AE85u;
  }
  return c;
}
__device__ __forceinline__ double u01(unsigned x) { return ((double)x + 0.5) * (1.0 / 4294967296.0); }

struct Stream {   // reading N10: block j of (seed, chain, iteration, tag) = philox(ctr=(j,chain,iteration,tag), key=seed)
  uint2 key;
  unsigned chain, iteration, tag;
  __device__ uint4 block(unsigned j) const { return philox4x32_10(make_uint4(j, chain, iteration, tag), key); }
  __device__ double uniform(unsigned j) const { return u01(block(j).x); }
  __device__ double normal(unsigned j0, int i) const {   // i-th normal of a run starting at block j0
    const uint4 w = block(j0 + (unsigned)(i >> 2));
    const int e = i & 3;
    const unsigned a = (e < 2) ? w.x : w.z, b = (e < 2) ? w.y : w.w;
    const double rr = sqrt(-2.0 * log(u01(a))), ang = 6.283185307179586 * u01(b);
    return (e & 1) ? rr * sin(ang) : rr * cos(ang);
  }
};

__global__ void philox_kernel(const uint4* ctr, int n, uint2 key, uint4* out) {
  int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) out[i] = philox4x32_10(ctr[i], key);
}

__device__ __forceinline__ double transform1(int kind, double p0, double p1, double u) {
  return kind == 0 ? p0 + (p1 - p0) * u : p0 + p1 * normcdfinv(u);
}

enum { P_NEW = 0, P_OUT_L = 1, P_OUT_R = 2, P_SHRINK = 3 };

struct RoundArgs {
  int n_chains, D, n_steps;
  int chain0;              // global id of this launch's chain 0 (sharded runs: the Philox streams are per GLOBAL chain)
  uint2 key;
  unsigned iteration;
  const double* scal;      // [0] = logL_star
  const double* Lsig;
  const int* prior_kind;
  const double *p0, *p1;
  float *x0, *dir, *xprop, *theta_chain;
  double *l, *r, *t, *logL0;
  int *phase, *cnt, *step, *pending, *finished, *need;
  unsigned* rng_j;
  const int* row_of_chain;
  const double* logL_prop;
  int* counters;
  float* u_out;
  double* logL_out;
  // several runs of one model sharing every round (nsgpu_run_multi): chain c belongs to run c / n_per_run and is its chain
  // c % n_per_run; per run: scal + 8 run (L*), Lsig + D D run, keys[run], iters[run], counters evals[run] / fails[run].
  // n_per_run = 0: one run, the scalar fields above.
  int n_per_run;
  const uint2* keys;
  const unsigned* iters;
  unsigned long long* run_evals;
  int* run_fails;
};

// a11 + a12: one warp per chain; consume last round's likelihood, advance the slice state machine to the
// next proposal that needs a likelihood.  Phase transitions are taken from the state as it was when the
// result was requested: a chain consumes exactly one likelihood result per round.
__global__ void __launch_bounds__(128) slice_round_kernel(RoundArgs a) {
  extern __shared__ double sL[];   // [D][D] direction factor of the run this block's first chain belongs to
  pdl_wait();      // logL_prop comes from the likelihood kernels of the previous round (launch_pdl contract)
  pdl_trigger();
  const int D = a.D;
  // A kernel of 500 warps on 148 SMs is pure latency: the D-step product L_Sigma z read its factor from global memory with
  // a dependent load per step (~39 L2 round trips in series for every new slice; ncu: 24 us per round).  Stage the factor
  // once per block (coalesced, one round trip); the accumulation order below is unchanged.
  const int c_first = min((int)((blockIdx.x * blockDim.x) >> 5), a.n_chains - 1);
  const int run_blk = a.n_per_run ? c_first / a.n_per_run : 0;
  {
    // sixteen loads in flight per thread before the first store: one L2 round trip for D <= 45, two for D = 64 (a plain
    // load-store loop was twelve round trips in series: the ncu source page had 69% of this kernel's samples on it)
    const double* src = a.Lsig + (size_t)run_blk * D * D;
    const int n = D * D;
    for (int i0 = threadIdx.x; i0 < n; i0 += 16 * blockDim.x) {
      double v[16];
#pragma unroll
      for (int u = 0; u < 16; ++u) { const int i = i0 + u * blockDim.x; v[u] = i < n ? src[i] : 0.0; }
#pragma unroll
      for (int u = 0; u < 16; ++u) { const int i = i0 + u * blockDim.x; if (i < n) sL[i] = v[u]; }
    }
  }
  __syncthreads();
  const int c = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (c >= a.n_chains) return;
  if (a.finished[c]) { if (lane == 0) a.need[c] = 0; return; }
  const int d0 = lane, d1 = lane + 32;
  const bool v0 = d0 < D, v1 = d1 < D;
  const size_t base = (size_t)c * D;
  float xa = v0 ? a.x0[base + d0] : 0.f, xb = v1 ? a.x0[base + d1] : 0.f;
  float da = v0 ? a.dir[base + d0] : 0.f, db = v1 ? a.dir[base + d1] : 0.f;
  float pa = v0 ? a.xprop[base + d0] : 0.f, pb = v1 ? a.xprop[base + d1] : 0.f;
  double l = a.l[c], r = a.r[c], t = a.t[c], logL0 = a.logL0[c];
  int phase = a.phase[c], cnt = a.cnt[c], step = a.step[c];
  unsigned j = a.rng_j[c];
  const int run = a.n_per_run ? c / a.n_per_run : 0;
  const int lc = c - run * a.n_per_run;                          // chain index within its run (= c for one run)
  const double Lstar = a.scal[8 * run];
  const double* Lsig = run == run_blk ? sL : a.Lsig + (size_t)run * D * D;   // a block that straddles two runs: the other run reads global
  Stream S{a.n_per_run ? a.keys[run] : a.key, (unsigned)(a.chain0 + lc), a.n_per_run ? a.iters[run] : a.iteration, 0u};
  bool inside = false;
  double val = 0.0;
  if (a.pending[c]) {
    val = a.logL_prop[a.row_of_chain[c]];
    inside = val > Lstar;                       // strict (reading N5); -inf and NaN compare false
  }
  int fails = 0;
  bool emit = false, done = false;
  while (true) {
    double tp = 0.0;
    bool propose = false;
    if (phase == P_OUT_L) {
      if (inside) { l -= BRACKET_W; ++cnt; if (cnt < MAX_STEP_OUT) { tp = l; propose = true; } }
      if (!propose) { cnt = 0; phase = P_OUT_R; tp = r; propose = true; }
    } else if (phase == P_OUT_R) {
      if (inside) { r += BRACKET_W; ++cnt; if (cnt < MAX_STEP_OUT) { tp = r; propose = true; } }
      if (!propose) { cnt = 0; phase = P_SHRINK; t = l + (r - l) * S.uniform(j++); tp = t; propose = true; }
    } else if (phase == P_SHRINK) {
      if (inside) {
        xa = pa; xb = pb; logL0 = val; ++step; phase = P_NEW;
      } else {
        if (t < 0.0) l = t; else r = t;
        ++cnt;
        if (cnt < MAX_SHRINK) { t = l + (r - l) * S.uniform(j++); tp = t; propose = true; }
        else { ++fails; ++step; phase = P_NEW; }
      }
    }
    if (phase == P_NEW && !propose) {
      if (step >= a.n_steps) { done = true; break; }
      // direction d = L_sigma z / ||z|| (reading N3)
      const double za = v0 ? S.normal(j, d0) : 0.0, zb = v1 ? S.normal(j, d1) : 0.0;
      j += (unsigned)((D + 3) >> 2);
      double nn = za * za + zb * zb;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) nn += __shfl_xor_sync(0xffffffffu, nn, o);
      double acca = 0.0, accb = 0.0;
      for (int jj = 0; jj < D; ++jj) {
        const double zj = __shfl_sync(0xffffffffu, jj < 32 ? za : zb, jj & 31);
        if (v0 && jj <= d0) acca += Lsig[(size_t)d0 * D + jj] * zj;
        if (v1 && jj <= d1) accb += Lsig[(size_t)d1 * D + jj] * zj;
      }
      const double inv = 1.0 / sqrt(nn);
      da = (float)(acca * inv); db = (float)(accb * inv);
      l = -BRACKET_W * S.uniform(j++);
      r = l + BRACKET_W;
      cnt = 0; phase = P_OUT_L; tp = l; propose = true;
    }
    // propose x0 + tp d; out-of-box is rejected here without a likelihood call
    pa = (float)((double)xa + tp * (double)da);
    pb = (float)((double)xb + tp * (double)db);
    const bool ok = (!v0 || (pa >= 0.f && pa <= 1.f)) && (!v1 || (pb >= 0.f && pb <= 1.f));
    if (__all_sync(0xffffffffu, ok)) { emit = true; break; }
    inside = false;
  }
  if (v0) { a.x0[base + d0] = xa; a.dir[base + d0] = da; a.xprop[base + d0] = pa; }
  if (v1) { a.x0[base + d1] = xb; a.dir[base + d1] = db; a.xprop[base + d1] = pb; }
  if (emit) {
    if (v0) a.theta_chain[base + d0] = (float)transform1(a.prior_kind[d0], a.p0[d0], a.p1[d0], (double)pa);
    if (v1) a.theta_chain[base + d1] = (float)transform1(a.prior_kind[d1], a.p0[d1], a.p1[d1], (double)pb);
  }
  if (done) {
    if (v0) a.u_out[base + d0] = xa;
    if (v1) a.u_out[base + d1] = xb;
  }
  if (lane == 0) {
    a.l[c] = l; a.r[c] = r; a.t[c] = t; a.logL0[c] = logL0;
    a.phase[c] = phase; a.cnt[c] = cnt; a.step[c] = step; a.rng_j[c] = j;
    a.pending[c] = emit ? 1 : 0;
    a.need[c] = emit ? 1 : 0;
    if (a.n_per_run) {
      if (emit) atomicAdd(&a.run_evals[run], 1ull);
      if (fails) atomicAdd(&a.run_fails[run], fails);
    }
    if (fails) atomicAdd(&a.counters[2], fails);
    if (done) { a.finished[c] = 1; a.logL_out[c] = logL0; atomicAdd(&a.counters[1], 1); }
  }
}

// block-wide exclusive scan of one int per thread (1024 threads)
__device__ int block_excl_scan_int(int v, int* wsum, int* total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  int inc = v;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { int t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
  if (lane == 31) wsum[warp] = inc;
  __syncthreads();
  if (warp == 0) {
    int w = wsum[lane], winc = w;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { int t = __shfl_up_sync(0xffffffffu, winc, o); if (lane >= o) winc += t; }
    wsum[lane] = winc - w;
    if (lane == 31) *total = winc;
  }
  __syncthreads();
  const int out = wsum[warp] + inc - v;
  __syncthreads();
  return out;
}

// compaction of the proposals that need a likelihood into a dense batch (deterministic: chain order).  Every CTA repeats
// the (cheap) scan of the flags into shared memory; CTA 0 publishes the rows and the count; the rows are then copied by all
// CTAs, one warp per chain (a single CTA walking all n_chains D floats through dependent loads took 12.7 us per round).
__global__ void __launch_bounds__(1024) compact_kernel(int n_chains, int D, const int* __restrict__ need,
                                                        int* __restrict__ row_of_chain,
                                                        const float* __restrict__ theta_chain,
                                                        float* __restrict__ theta_prop, int* counters,
                                                        unsigned long long* n_evals) {
  extern __shared__ int srow[];   // [n_chains]
  __shared__ int wsum[32];
  __shared__ int total;
  int carry = 0;
  pdl_wait();
  pdl_trigger();
  for (int base = 0; base < n_chains; base += blockDim.x) {
    const int c = base + threadIdx.x;
    const int f = (c < n_chains) ? need[c] : 0;
    const int ex = block_excl_scan_int(f, wsum, &total);
    if (c < n_chains) srow[c] = f ? carry + ex : -1;
    carry += total;
    __syncthreads();
  }
  if (blockIdx.x == 0) {
    for (int c = threadIdx.x; c < n_chains; c += blockDim.x) row_of_chain[c] = srow[c];
    if (threadIdx.x == 0) { counters[0] = carry; *n_evals += (unsigned long long)carry; }
  }
  const int lane = threadIdx.x & 31;
  const int gw = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), nw = gridDim.x * (blockDim.x >> 5);
  for (int c = gw; c < n_chains; c += nw) {
    const int row = srow[c];
    if (row < 0) continue;
    for (int d = lane; d < D; d += 32) theta_prop[(size_t)row * D + d] = theta_chain[(size_t)c * D + d];
  }
}

__global__ void chain_init_kernel(int n_chains, int chain0, int D, uint2 key, unsigned iteration, const int* __restrict__ surv_idx,
                                  int n_surv, const int* __restrict__ start_in, int* __restrict__ start_idx,
                                  const float* __restrict__ u_live, const double* __restrict__ logL_live,
                                  float* x0, double* logL0, int* phase, int* cnt, int* step, int* pending,
                                  int* finished, int* need, unsigned* rng_j, int n_live, double* scal) {
  const int c = blockIdx.x * blockDim.x + threadIdx.x;
  if (c >= n_chains) return;
  int s;
  if (start_in) {
    s = start_in[c];
    if (s < 0 || s >= n_live) { scal[6] = 1.0; s = min(max(s, 0), n_live - 1); }   // caller's index out of range: flagged, clamped
  } else {   // reading N4: uniform with replacement from the survivors; Stream(seed, c, iteration, tag 1)
    Stream S{key, (unsigned)(chain0 + c), iteration, 1u};
    int pick = (int)(S.uniform(0) * n_surv);
    s = surv_idx[min(pick, n_surv - 1)];
  }
  start_idx[c] = s;
  for (int d = 0; d < D; ++d) x0[(size_t)c * D + d] = u_live[(size_t)s * D + d];
  logL0[c] = logL_live[s];
  phase[c] = P_NEW; cnt[c] = 0; step[c] = 0; pending[c] = 0; finished[c] = 0; need[c] = 0; rng_j[c] = 0;
}

// a14: sample covariance of the live set in u-space + 1e-12 I, lower Cholesky factor; one CTA
// `status` (may be NULL): set to 1 when a pivot is not positive (fewer than D + 1 distinct live points, or non-finite
// coordinates): the factor is then unusable and the host returns NSGPU_ENOTSPD instead of sampling NaN directions.
__global__ void __launch_bounds__(256) live_cholesky_kernel(const float* __restrict__ u, int n, int D, double* __restrict__ L,
                                                            double* __restrict__ status) {
  __shared__ double mean[NSGPU_MAX_D];
  __shared__ double cov[NSGPU_MAX_D * NSGPU_MAX_D];
  for (int d = threadIdx.x; d < D; d += blockDim.x) {
    double s = 0.0;
    for (int i = 0; i < n; ++i) s += (double)u[(size_t)i * D + d];
    mean[d] = s / n;
  }
  __syncthreads();
  for (int e = threadIdx.x; e < D * D; e += blockDim.x) {
    const int r = e / D, cidx = e - r * D;
    if (cidx > r) { cov[e] = 0.0; continue; }
    double s = 0.0;
    for (int i = 0; i < n; ++i) s += ((double)u[(size_t)i * D + r] - mean[r]) * ((double)u[(size_t)i * D + cidx] - mean[cidx]);
    cov[e] = s / (n - 1) + (r == cidx ? 1e-12 : 0.0);
  }
  __syncthreads();
  // column Cholesky; D <= 64, one warp-synchronous pass per column by the whole block
  for (int k = 0; k < D; ++k) {
    if (threadIdx.x == 0) {
      const double piv = cov[k * D + k];
      if (!(piv > 0.0) && status) *status = 1.0;
      cov[k * D + k] = sqrt(piv);
    }
    __syncthreads();
    for (int i = k + 1 + threadIdx.x; i < D; i += blockDim.x) cov[i * D + k] /= cov[k * D + k];
    __syncthreads();
    for (int e = threadIdx.x; e < D * D; e += blockDim.x) {
      const int i = e / D, jj = e - i * D;
      if (jj > k && jj <= i) cov[i * D + jj] -= cov[i * D + k] * cov[jj * D + k];
    }
    __syncthreads();
  }
  for (int e = threadIdx.x; e < D * D; e += blockDim.x) L[e] = cov[e];
}

// a13: delete the k lowest live points, accumulate the evidence.  One CTA of 1024 threads.
// Total order by (logL, index) via a bitonic sort in shared memory (reading N5); volumes by a prefix
// sum of -1/n_j and the weights folded into log Z by a block log-sum-exp (reading N6).
__global__ void __launch_bounds__(1024) delete_lowest_kernel(const double* __restrict__ logL, int n, int k,
                                                              double* __restrict__ scal, int* __restrict__ dead_idx,
                                                              int* __restrict__ surv_idx, double* __restrict__ logw) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  int np2 = 1;
  while (np2 < n) np2 <<= 1;
  double* key = reinterpret_cast<double*>(smem_raw);   // [np2]
  int* idx = reinterpret_cast<int*>(key + np2);        // [np2]
  __shared__ double red[32];
  __shared__ double wsum[33];
  __shared__ int isum[32];
  __shared__ int itot;
  for (int i = threadIdx.x; i < np2; i += blockDim.x) {
    key[i] = i < n ? logL[i] : INFINITY;
    idx[i] = i < n ? i : 0x7fffffff;
  }
  __syncthreads();
  for (int size = 2; size <= np2; size <<= 1)
    for (int stride = size >> 1; stride > 0; stride >>= 1) {
      for (int i = threadIdx.x; i < np2; i += blockDim.x) {
        const int p = i ^ stride;
        if (p > i) {
          const bool up = (i & size) == 0;
          const double a = key[i], b = key[p];
          const int ia = idx[i], ib = idx[p];
          const bool gt = (a > b) || (a == b && ia > ib) || (a != a && b == b);
          if (gt == up) { key[i] = b; key[p] = a; idx[i] = ib; idx[p] = ia; }
        }
      }
      __syncthreads();
    }
  const double logX0 = scal[1], logZ0 = scal[2];
  // prefix sum of 1/n_j (exclusive) -> log X_{j-1}; terms l_j + log w_j
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  double carry = 0.0, mx = -INFINITY;
  for (int base = 0; base < k; base += blockDim.x) {
    const int jj = base + threadIdx.x;
    const double nj = (double)(n - jj);
    const double v = jj < k ? 1.0 / nj : 0.0;
    double inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { double tt = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += tt; }
    if (lane == 31) wsum[warp] = inc;
    __syncthreads();
    if (warp == 0) {
      double w = wsum[lane], winc = w;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) { double tt = __shfl_up_sync(0xffffffffu, winc, o); if (lane >= o) winc += tt; }
      wsum[lane] = winc - w;
      if (lane == 31) wsum[32] = winc;
    }
    __syncthreads();
    if (jj < k) {
      const double logX_prev = logX0 - (carry + wsum[warp] + inc - v);
      const double lw = logX_prev + log(-expm1(-1.0 / nj));
      logw[jj] = lw;
      dead_idx[jj] = idx[jj];
      mx = fmax(mx, key[jj] + lw);
    }
    carry += wsum[32];
    __syncthreads();
  }
  // block log-sum-exp of the k terms together with the running log Z
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
  if (lane == 0) red[warp] = mx;
  __syncthreads();
  if (warp == 0) {
    double m = red[lane];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
    if (lane == 0) red[0] = fmax(m, logZ0);
  }
  __syncthreads();
  const double M = red[0];
  __syncthreads();
  double se = 0.0;
  for (int jj = threadIdx.x; jj < k; jj += blockDim.x) se += exp(key[jj] + logw[jj] - M);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) se += __shfl_xor_sync(0xffffffffu, se, o);
  if (lane == 0) red[warp] = se;
  __syncthreads();
  if (threadIdx.x == 0) {
    double tot = 0.0;
    for (int w = 0; w < 32; ++w) tot += red[w];
    if (logZ0 > -INFINITY) tot += exp(logZ0 - M);
    scal[2] = (M > -INFINITY) ? M + log(tot) : -INFINITY;
    scal[1] = logX0 - carry;
    scal[0] = key[k - 1];                                   // L* = largest deleted
  }
  __syncthreads();
  // survivors in index order: mark the dead, scan the flags
  int* deadflag = idx;                                        // reuse after copying the dead indices out
  __syncthreads();
  for (int i = threadIdx.x; i < np2; i += blockDim.x) deadflag[i] = 0;
  __syncthreads();
  for (int jj = threadIdx.x; jj < k; jj += blockDim.x) deadflag[dead_idx[jj]] = 1;
  __syncthreads();
  int icarry = 0;
  for (int base = 0; base < n; base += blockDim.x) {
    const int i = base + threadIdx.x;
    const int f = (i < n && !deadflag[i]) ? 1 : 0;
    const int ex = block_excl_scan_int(f, isum, &itot);
    if (f) surv_idx[icarry + ex] = i;
    icarry += itot;
    __syncthreads();
  }
}

__global__ void replace_kernel(int k, int D, const int* __restrict__ dead_idx, const float* __restrict__ u_out,
                               const double* __restrict__ logL_out, float* u_live, double* logL_live) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= k * D) return;
  const int c = i / D, d = i - c * D;
  u_live[(size_t)dead_idx[c] * D + d] = u_out[i];
  if (d == 0) logL_live[dead_idx[c]] = logL_out[c];
}

__global__ void gather_rows_kernel(int k, int D, const int* __restrict__ rows, const float* __restrict__ src_u,
                                   const double* __restrict__ src_l, float* dst_u, double* dst_l) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= k * D) return;
  const int c = i / D, d = i - c * D;
  dst_u[i] = src_u[(size_t)rows[c] * D + d];
  if (d == 0) dst_l[c] = src_l[rows[c]];
}

// termination test (reading N7): logZ_live = logsumexp(l_live) - ln n + logX
__global__ void __launch_bounds__(1024) live_evidence_kernel(const double* __restrict__ logL, int n, double log_stop,
                                                              double* scal) {
  __shared__ double red[32];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  double mx = -INFINITY;
  for (int i = threadIdx.x; i < n; i += blockDim.x) mx = fmax(mx, logL[i]);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
  if (lane == 0) red[warp] = mx;
  __syncthreads();
  if (warp == 0) {
    double m = red[lane];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmax(m, __shfl_xor_sync(0xffffffffu, m, o));
    if (lane == 0) red[0] = m;
  }
  __syncthreads();
  const double M = red[0];
  __syncthreads();
  double se = 0.0;
  for (int i = threadIdx.x; i < n; i += blockDim.x) se += exp(logL[i] - M);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) se += __shfl_xor_sync(0xffffffffu, se, o);
  if (lane == 0) red[warp] = se;
  __syncthreads();
  if (threadIdx.x == 0) {
    double tot = 0.0;
    for (int w = 0; w < 32; ++w) tot += red[w];
    const double lzl = M + log(tot) - log((double)n) + scal[1];
    const double lz = scal[2];
    const double hi = fmax(lz, lzl), lo = fmin(lz, lzl);
    const double both = hi + log1p(exp(lo - hi));
    scal[3] = lzl;
    scal[4] = (lzl - both < log_stop) ? 1.0 : 0.0;
  }
}

__global__ void init_live_kernel(int n, int D, uint2 key, float* u) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n * D) return;
  const int p = i / D, d = i - p * D;
  Stream S{key, (unsigned)p, 0u, 2u};     // point p: D uniforms from blocks 0..D-1, word 0
  u[i] = (float)S.uniform((unsigned)d);
}

// Error bar of log Z by simulated prior volumes (reading N9; Skilling 2006): sequence m redraws every
// shrinkage factor t_i = U^{1/n_i} over the recorded dead points (n_i = n - i mod k: batch deletion) and recomputes
// log Z = logsumexp_i [l_i + log X_{i-1} + log(1 - t_i)] with the live points at X_final / n.  One CTA per sequence:
// tiles of 1024 dead points, the running log X by a block prefix sum, an online log-sum-exp per thread joined at the end.
// Uniforms: Philox stream (seed; block i/4, sequence m, tag 3), word i mod 4 (reading N10).
__global__ void __launch_bounds__(256) evidence_error_kernel(const double* __restrict__ dead_logL, long long nd, int n, int k,
                                                             const double* __restrict__ live_logL, uint2 key,
                                                             double* __restrict__ zs) {
  __shared__ double wsum[8], red_m[8], red_s[8];
  const unsigned m = blockIdx.x;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  double carry = 0.0, mx = -INFINITY, se = 0.0;
  auto add_term = [&](double term) {
    if (!(term > -INFINITY)) return;
    if (term > mx) { se = se * exp(mx - term) + 1.0; mx = term; }
    else se += exp(term - mx);
  };
  for (long long base = 0; base < nd; base += 1024) {
    const long long i0 = base + 4 * threadIdx.x;
    const unsigned long long blk = (unsigned long long)i0 >> 2;
    const uint4 w = philox4x32_10(make_uint4((unsigned)blk, m, (unsigned)(blk >> 32), 3u), key);
    const unsigned ww[4] = {w.x, w.y, w.z, w.w};
    double lt[4], tot = 0.0;
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      const long long i = i0 + e;
      lt[e] = i < nd ? log(u01(ww[e])) / (double)(n - (int)(i % k)) : 0.0;
      tot += lt[e];
    }
    double inc = tot;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const double t = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += t; }
    if (lane == 31) wsum[warp] = inc;
    __syncthreads();
    double woff = 0.0, tile = 0.0;
#pragma unroll
    for (int q = 0; q < 8; ++q) { if (q < warp) woff += wsum[q]; tile += wsum[q]; }
    double lx = carry + woff + inc - tot;           // log X before this thread's first point
#pragma unroll
    for (int e = 0; e < 4; ++e) {
      const long long i = i0 + e;
      if (i < nd) { add_term(dead_logL[i] + lx + log(-expm1(lt[e]))); lx += lt[e]; }
    }
    carry += tile;
    __syncthreads();
  }
  const double lw_live = carry - log((double)n);
  for (int i = threadIdx.x; i < n; i += blockDim.x) add_term(live_logL[i] + lw_live);
  // join the per-thread (max, sum) pairs
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    const double om = __shfl_xor_sync(0xffffffffu, mx, o), os = __shfl_xor_sync(0xffffffffu, se, o);
    const double nm = fmax(mx, om);
    se = (mx > -INFINITY ? se * exp(mx - nm) : 0.0) + (om > -INFINITY ? os * exp(om - nm) : 0.0);
    mx = nm;
  }
  if (lane == 0) { red_m[warp] = mx; red_s[warp] = se; }
  __syncthreads();
  if (threadIdx.x == 0) {
    double M = -INFINITY, S = 0.0;
    for (int q = 0; q < 8; ++q) M = fmax(M, red_m[q]);
    for (int q = 0; q < 8; ++q) if (red_m[q] > -INFINITY) S += red_s[q] * exp(red_m[q] - M);
    zs[m] = M > -INFINITY ? M + log(S) : -INFINITY;
  }
}

}  // namespace

// ---------------------------------------------------------------------------------------------------
nsgpu_status sampler_create(nsgpu_ctx* ctx) {
  SamplerDev* S = new SamplerDev();
  ctx->sampler = S;
  NSGPU_CUDA(cudaStreamCreateWithFlags(&S->run_stream, cudaStreamNonBlocking));
  const size_t cap = ctx->max_batch, D = ctx->D;
  S->cap = (int)cap;
#define A(p, T, n) NSGPU_CUDA(cudaMalloc((void**)&S->p, sizeof(T) * (n)))
  A(x0, float, cap * D); A(dir, float, cap * D); A(xprop, float, cap * D); A(theta_chain, float, cap * D);
  A(l, double, cap); A(r, double, cap); A(t, double, cap); A(logL0, double, cap);
  A(phase, int, cap); A(cnt, int, cap); A(step, int, cap); A(pending, int, cap); A(finished, int, cap); A(need, int, cap);
  A(rng_j, unsigned, cap); A(row_of_chain, int, cap); A(start_idx, int, cap);
  A(theta_prop, float, cap * D); A(logL_prop, double, cap);
  A(counters, int, 4); A(n_evals, unsigned long long, 1); A(scal, double, 8); A(Lsig, double, D * D);
  A(u_live, float, cap * D); A(logL_live, double, cap); A(dead_idx, int, cap); A(surv_idx, int, cap);
  A(logw, double, cap); A(u_out, float, cap * D); A(logL_out, double, cap);
#undef A
  NSGPU_CUDA(cudaMallocHost((void**)&S->h_counters, 4 * sizeof(int)));
  NSGPU_CUDA(cudaMallocHost((void**)&S->h_evals, sizeof(unsigned long long)));
  NSGPU_CUDA(cudaMallocHost((void**)&S->h_scal, 8 * sizeof(double)));
  NSGPU_CUDA(cudaMemset(S->xprop, 0, sizeof(float) * cap * D));
  NSGPU_CUDA(cudaMemset(S->dir, 0, sizeof(float) * cap * D));
  return NSGPU_OK;
}

void sampler_destroy(nsgpu_ctx* ctx) {
  SamplerDev* S = ctx->sampler;
  if (!S) return;
  void* ptrs[] = {S->x0, S->dir, S->xprop, S->theta_chain, S->l, S->r, S->t, S->logL0, S->phase, S->cnt, S->step,
                  S->pending, S->finished, S->need, S->rng_j, S->row_of_chain, S->start_idx, S->theta_prop,
                  S->logL_prop, S->counters, S->n_evals, S->scal, S->Lsig, S->u_live, S->logL_live, S->dead_idx,
                  S->surv_idx, S->logw, S->u_out, S->logL_out};
  for (void* p : ptrs) cudaFree(p);
  if (S->run_stream) cudaStreamDestroy(S->run_stream);
  cudaFreeHost(S->h_counters); cudaFreeHost(S->h_evals); cudaFreeHost(S->h_scal);
  delete S;
  ctx->sampler = nullptr;
}

static nsgpu_status launch_live_cholesky(nsgpu_ctx* ctx, const float* u_live, int n_live, double* L, double* status,
                                         cudaStream_t st) {
  live_cholesky_kernel<<<1, 256, 0, st>>>(u_live, n_live, ctx->D, L, status);
  NSGPU_LAUNCH_CHECK();
  return NSGPU_OK;
}

static nsgpu_status launch_delete(nsgpu_ctx* ctx, const double* logL, int n, int k, cudaStream_t st, double* scal = nullptr,
                                  int* dead_idx = nullptr, int* surv_idx = nullptr, double* logw = nullptr) {
  SamplerDev* S = ctx->sampler;
  if (!scal) { scal = S->scal; dead_idx = S->dead_idx; surv_idx = S->surv_idx; logw = S->logw; }
  int np2 = 1;
  while (np2 < n) np2 <<= 1;
  const size_t smem = (size_t)np2 * (sizeof(double) + sizeof(int));
  NSGPU_CUDA(nsgpu_ensure_smem(ctx, delete_lowest_kernel, smem));
  delete_lowest_kernel<<<1, 1024, smem, st>>>(logL, n, k, scal, dead_idx, surv_idx, logw);
  NSGPU_LAUNCH_CHECK();
  return NSGPU_OK;
}

// Evolve n_chains chains to completion.  Chains were initialised by chain_init_kernel; Lsig and scal[0]
// (L*) are set.  Host reads the finished-counter after batches of rounds (one small D2H per batch).
struct MultiArgs {           // device arrays of nsgpu_run_multi (see RoundArgs)
  int n_per_run, n_target;   // chains per run; chains that will finish (active runs x n_per_run)
  const uint2* keys; const unsigned* iters; unsigned long long* run_evals; int* run_fails; const double* scal; const double* Lsig;
};

static nsgpu_status evolve(nsgpu_ctx* ctx, int n_chains, int chain0, int n_steps, uint64_t seed, int iteration, cudaStream_t st,
                           int64_t* rounds_out, const MultiArgs* multi = nullptr) {
  SamplerDev* S = ctx->sampler;
  RoundArgs a;
  a.n_chains = n_chains; a.D = ctx->D; a.n_steps = n_steps; a.chain0 = chain0;
  a.key = make_uint2((unsigned)(seed & 0xffffffffu), (unsigned)(seed >> 32));
  a.iteration = (unsigned)iteration;
  a.scal = S->scal; a.Lsig = S->Lsig; a.prior_kind = ctx->prior_kind; a.p0 = ctx->prior_p0; a.p1 = ctx->prior_p1;
  a.x0 = S->x0; a.dir = S->dir; a.xprop = S->xprop; a.theta_chain = S->theta_chain;
  a.l = S->l; a.r = S->r; a.t = S->t; a.logL0 = S->logL0;
  a.phase = S->phase; a.cnt = S->cnt; a.step = S->step; a.pending = S->pending; a.finished = S->finished; a.need = S->need;
  a.rng_j = S->rng_j; a.row_of_chain = S->row_of_chain; a.logL_prop = S->logL_prop; a.counters = S->counters;
  a.u_out = S->u_out; a.logL_out = S->logL_out;
  a.n_per_run = 0; a.keys = nullptr; a.iters = nullptr; a.run_evals = nullptr; a.run_fails = nullptr;
  if (multi) { a.n_per_run = multi->n_per_run; a.keys = multi->keys; a.iters = multi->iters; a.run_evals = multi->run_evals;
               a.run_fails = multi->run_fails; a.scal = multi->scal; a.Lsig = multi->Lsig; }
  const int n_target = multi ? multi->n_target : n_chains;
  NSGPU_CUDA(cudaMemsetAsync(S->counters, 0, 4 * sizeof(int), st));
  const int blocks = (n_chains * 32 + 127) / 128;
  const int compact_ctas = std::min(std::max((n_chains + 31) / 32, 1), 16);   // 32 warps each: one chain row per warp up to 512 chains
  if (n_chains > 51200) { ctx->err = "sampler: more than 51200 chains in one round (the compaction keeps its row table in shared memory)"; return NSGPU_ESHAPE; }
  if (sizeof(int) * (size_t)n_chains > 48 * 1024) NSGPU_CUDA(nsgpu_ensure_smem(ctx, compact_kernel, sizeof(int) * (size_t)n_chains));
  int64_t rounds = 0;
  // Rounds are launched in bursts and the finished-counter is read after each burst (one small D2H).  A round
  // after the last chain has finished is a dozen empty launches, a check is a pipeline drain: the first burst
  // runs up to just short of what the previous call on this context needed (n_steps to start with: no chain
  // can finish earlier), then short bursts until every chain is done.
  int burst = std::max(8, (S->rounds_needed > 0 && S->rounds_n_steps == n_steps) ? S->rounds_needed - 24 : n_steps);
  while (true) {
    for (int i = 0; i < burst; ++i) {
      {
      StageTimer tm(ctx, 6, st);
      NSGPU_CUDA(launch_pdl(ctx, slice_round_kernel, dim3(blocks), dim3(128), sizeof(double) * ctx->D * ctx->D, st, a));
      NSGPU_LAUNCH_CHECK();
      NSGPU_CUDA(launch_pdl(ctx, compact_kernel, dim3(compact_ctas), dim3(1024), sizeof(int) * n_chains, st, n_chains, ctx->D, S->need,
                            S->row_of_chain, S->theta_chain, S->theta_prop, S->counters, S->n_evals));
      NSGPU_LAUNCH_CHECK();
      }
      nsgpu_status s = loglike_device(ctx, S->theta_prop, n_chains, S->counters, S->logL_prop, st);
      if (s != NSGPU_OK) return s;
      ++rounds;
    }
    NSGPU_CUDA(cudaMemcpyAsync(S->h_counters, S->counters, 4 * sizeof(int), cudaMemcpyDeviceToHost, st));
    NSGPU_CUDA(cudaStreamSynchronize(st));
    if (S->h_counters[1] >= n_target) break;
    burst = 16;
    if (rounds > (int64_t)n_steps * (MAX_STEP_OUT * 2 + MAX_SHRINK + 4) + 16) {
      ctx->err = "slice sampling: chains did not finish (internal error)";
      return NSGPU_ECUDA;
    }
  }
  S->rounds_needed = (int)std::min<int64_t>(rounds, 1 << 30);
  S->rounds_n_steps = n_steps;
  if (rounds_out) *rounds_out += rounds;
  return NSGPU_OK;
}

static nsgpu_status check_sampler_args(nsgpu_ctx* ctx, int n_live, int n_chains) {
  if (!ctx) return NSGPU_EINVAL;
  if (n_live < 2 || n_chains < 1) { ctx->err = "sampler: n_live >= 2 and n_chains >= 1 required"; return NSGPU_EINVAL; }
  if (n_live > ctx->max_batch || n_chains > ctx->max_batch || n_live > MAX_LIVE) {
    ctx->err = "sampler: n_live / n_chains exceed max_batch (or 16384)";
    return NSGPU_ESHAPE;
  }
  cudaError_t e = cudaSetDevice(ctx->device);
  if (e != cudaSuccess) { ctx->err = cudaGetErrorString(e); return NSGPU_ECUDA; }
  return NSGPU_OK;
}

extern "C" nsgpu_status nsgpu_slice_step(nsgpu_ctx* ctx, const float* u_live, const double* logL_live, int32_t n_live,
                                         const int32_t* start_idx, int32_t n_chains, double logL_star, int32_t n_steps,
                                         uint64_t seed, int32_t iteration, float* u_out, double* logL_out,
                                         int64_t* n_evals, void* stream) {
  nsgpu_status s = check_sampler_args(ctx, n_live, n_chains);
  if (s != NSGPU_OK) return s;
  if (!u_live || !logL_live || !start_idx || !u_out || !logL_out || n_steps < 0) { ctx->err = "slice_step: bad arguments"; return NSGPU_EINVAL; }
  SamplerDev* S = ctx->sampler;
  cudaStream_t st = (cudaStream_t)stream;
  const int D = ctx->D;
  if (n_live < D + 1) { ctx->err = "slice_step: the live covariance needs n_live >= D + 1"; return NSGPU_EINVAL; }
  for (int i = 0; i < 8; ++i) S->h_scal[i] = 0.0;
  S->h_scal[0] = logL_star;                       // [5] Cholesky status, [6] start-index status: cleared
  NSGPU_CUDA(cudaMemcpyAsync(S->scal, S->h_scal, 8 * sizeof(double), cudaMemcpyHostToDevice, st));
  s = launch_live_cholesky(ctx, u_live, n_live, S->Lsig, S->scal + 5, st);
  if (s != NSGPU_OK) return s;
  NSGPU_CUDA(cudaMemsetAsync(S->n_evals, 0, sizeof(unsigned long long), st));
  const uint2 key = make_uint2((unsigned)(seed & 0xffffffffu), (unsigned)(seed >> 32));
  chain_init_kernel<<<(n_chains + 127) / 128, 128, 0, st>>>(n_chains, 0, D, key, (unsigned)iteration, nullptr, 0, start_idx,
                                                            S->start_idx, u_live, logL_live, S->x0, S->logL0, S->phase,
                                                            S->cnt, S->step, S->pending, S->finished, S->need, S->rng_j, n_live, S->scal);
  NSGPU_LAUNCH_CHECK();
  s = evolve(ctx, n_chains, 0, n_steps, seed, iteration, st, nullptr);
  if (s != NSGPU_OK) return s;
  NSGPU_CUDA(cudaMemcpyAsync(u_out, S->u_out, sizeof(float) * (size_t)n_chains * D, cudaMemcpyDeviceToDevice, st));
  NSGPU_CUDA(cudaMemcpyAsync(logL_out, S->logL_out, sizeof(double) * (size_t)n_chains, cudaMemcpyDeviceToDevice, st));
  NSGPU_CUDA(cudaMemcpyAsync(S->h_evals, S->n_evals, sizeof(unsigned long long), cudaMemcpyDeviceToHost, st));
  NSGPU_CUDA(cudaMemcpyAsync(S->h_scal, S->scal, 8 * sizeof(double), cudaMemcpyDeviceToHost, st));
  NSGPU_CUDA(cudaStreamSynchronize(st));
  if (n_evals) *n_evals = (int64_t)*S->h_evals;
  S->last_failed_moves = S->h_counters[2];
  if (S->h_scal[6] != 0.0) { ctx->err = "slice_step: start_idx out of [0, n_live)"; return NSGPU_EINVAL; }
  if (S->h_scal[5] != 0.0) { ctx->err = "slice_step: live-set covariance is not positive definite"; return NSGPU_ENOTSPD; }
  return NSGPU_OK;
}

extern "C" nsgpu_status nsgpu_sampler_counters(const nsgpu_ctx* ctx, int64_t* n_failed_moves, int64_t* n_rounds) {
  if (!ctx || !ctx->sampler) return NSGPU_EINVAL;
  if (n_failed_moves) *n_failed_moves = ctx->sampler->last_failed_moves;
  if (n_rounds) *n_rounds = ctx->sampler->rounds_needed;
  return NSGPU_OK;
}

extern "C" nsgpu_status nsgpu_delete_lowest(nsgpu_ctx* ctx, const double* logL_live, int32_t n_live, int32_t k,
                                            double* logX, double* logZ, int32_t* dead_idx, double* logw,
                                            double* logL_star, void* stream) {
  nsgpu_status s = check_sampler_args(ctx, n_live, k);
  if (s != NSGPU_OK) return s;
  if (!logL_live || !logX || !logZ || !dead_idx || !logw || !logL_star || k >= n_live) { ctx->err = "delete_lowest: bad arguments"; return NSGPU_EINVAL; }
  SamplerDev* S = ctx->sampler;
  cudaStream_t st = (cudaStream_t)stream;
  S->h_scal[0] = 0.0; S->h_scal[1] = *logX; S->h_scal[2] = *logZ;
  NSGPU_CUDA(cudaMemcpyAsync(S->scal, S->h_scal, 3 * sizeof(double), cudaMemcpyHostToDevice, st));
  s = launch_delete(ctx, logL_live, n_live, k, st);
  if (s != NSGPU_OK) return s;
  NSGPU_CUDA(cudaMemcpyAsync(dead_idx, S->dead_idx, sizeof(int) * (size_t)k, cudaMemcpyDeviceToDevice, st));
  NSGPU_CUDA(cudaMemcpyAsync(logw, S->logw, sizeof(double) * (size_t)k, cudaMemcpyDeviceToDevice, st));
  NSGPU_CUDA(cudaMemcpyAsync(S->h_scal, S->scal, 3 * sizeof(double), cudaMemcpyDeviceToHost, st));
  NSGPU_CUDA(cudaStreamSynchronize(st));
  *logL_star = S->h_scal[0]; *logX = S->h_scal[1]; *logZ = S->h_scal[2];
  return NSGPU_OK;
}

extern "C" nsgpu_status nsgpu_live_cholesky(nsgpu_ctx* ctx, const float* u_live, int32_t n_live, double* L_out, void* stream) {
  nsgpu_status s = check_sampler_args(ctx, n_live, 1);
  if (s != NSGPU_OK) return s;
  if (!u_live || !L_out) { ctx->err = "live_cholesky: NULL pointer"; return NSGPU_EINVAL; }
  return launch_live_cholesky(ctx, u_live, n_live, L_out, nullptr, (cudaStream_t)stream);
}

extern "C" nsgpu_status nsgpu_debug_philox(nsgpu_ctx* ctx, const uint32_t* ctr, int32_t n, const uint32_t* key,
                                           uint32_t* out, void* stream) {
  if (!ctx) return NSGPU_EINVAL;
  if (n < 0 || (n > 0 && (!ctr || !key || !out))) { ctx->err = "debug_philox: bad arguments"; return NSGPU_EINVAL; }
  if (n == 0) return NSGPU_OK;
  NSGPU_CUDA(cudaSetDevice(ctx->device));
  philox_kernel<<<(n + 255) / 256, 256, 0, (cudaStream_t)stream>>>((const uint4*)ctr, n, make_uint2(key[0], key[1]), (uint4*)out);
  NSGPU_LAUNCH_CHECK();
  return NSGPU_OK;
}

extern "C" nsgpu_status nsgpu_last_samples(nsgpu_ctx* ctx, float* theta_samples, double* logL_samples,
                                           double* logw_samples, int64_t cap, int64_t* n_samples) {
  if (!ctx) return NSGPU_EINVAL;
  SamplerDev* S = ctx->sampler;
  const int64_t ntot = (int64_t)S->last_logL.size();
  if (n_samples) *n_samples = ntot;
  if (cap <= 0) return NSGPU_OK;
  if (!theta_samples || !logL_samples || !logw_samples) { ctx->err = "last_samples: NULL buffer"; return NSGPU_EINVAL; }
  const size_t nw = (size_t)std::min<int64_t>(cap, ntot);
  memcpy(theta_samples, S->last_theta.data(), sizeof(float) * nw * ctx->D);
  memcpy(logL_samples, S->last_logL.data(), sizeof(double) * nw);
  memcpy(logw_samples, S->last_logw.data(), sizeof(double) * nw);
  return NSGPU_OK;
}

// ---------------------------------------------------------------------------------------------------
// nsgpu_run: the outer loop.  Host code only schedules kernels and reads one flag per
// iteration; all arithmetic on the live set happens in the kernels above.  The final summary (total
// log Z with the live points, H, error bar by simulated volumes -- reading N9) is fp64 host arithmetic
// over the recorded (logL, n_j) sequence.
// ---------------------------------------------------------------------------------------------------
extern "C" void nsgpu_shard_range(int32_t n_chains, int32_t rank, int32_t world, int32_t* first, int32_t* count) {
  const int per = world > 0 ? (n_chains + world - 1) / world : n_chains;
  const int c0 = std::min(n_chains, rank * per);
  if (first) *first = c0;
  if (count) *count = std::max(0, std::min(n_chains, c0 + per) - c0);
}

// Final summary of one run (host arithmetic over the recorded sequence, reading N8/N9): total log Z with the live points,
// H, error bar by simulated volumes (evidence_error_kernel) and by the analytic formula, weighted samples theta = T(u).
static nsgpu_status summarize_run(nsgpu_ctx* ctx, int n, int k, uint2 key, double logX, const std::vector<float>& dead_u,
                                  const std::vector<double>& dead_logL, const std::vector<double>& dead_logw,
                                  const std::vector<float>& live_u, const std::vector<double>& live_l,
                                  const double* d_live_logL, cudaStream_t st, nsgpu_result* res, std::vector<float>& out_theta,
                                  std::vector<double>& out_logL, std::vector<double>& out_logw) {
  SamplerDev* S = ctx->sampler;
  const int D = ctx->D;
  nsgpu_status s = NSGPU_OK;
  const size_t nd = dead_logL.size(), ntot = nd + n;
  std::vector<double> all_l(ntot), all_w(ntot);
  for (size_t i = 0; i < nd; ++i) { all_l[i] = dead_logL[i]; all_w[i] = dead_logw[i]; }
  for (int i = 0; i < n; ++i) { all_l[nd + i] = live_l[i]; all_w[nd + i] = logX - log((double)n); }   // reading N8
  auto logsumexp = [](const std::vector<double>& v) -> double {
    double mx = -INFINITY;
    for (double x : v) mx = std::max(mx, x);
    if (!(mx > -INFINITY)) return (double)-INFINITY;
    double sacc = 0.0;
    for (double x : v) sacc += exp(x - mx);
    return mx + log(sacc);
  };
  std::vector<double> terms(ntot);
  for (size_t i = 0; i < ntot; ++i) terms[i] = all_l[i] + all_w[i];
  const double logZ = logsumexp(terms);
  double H = 0.0;
  for (size_t i = 0; i < ntot; ++i) {
    const double p = exp(terms[i] - logZ);
    if (p > 0.0) H += p * (all_l[i] - logZ);
  }
  // error bar: redraw the volume sequence M = 1000 times with t_j = U^{1/n_j} (Skilling 2006) -- one CTA per
  // sequence (evidence_error_kernel); the host only takes the standard deviation of the 1000 results.  (Round 1 did
  // this in a single-threaded host loop of 1000 x n_dead log/expm1/exp calls: 3.4 s for a c4 run.)
  double err_sim = 0.0;
  {
    const int M = 1000;
    double *d_dead = nullptr, *d_zs = nullptr;
    NSGPU_CUDA(cudaMalloc((void**)&d_dead, sizeof(double) * std::max<size_t>(nd, 1)));
    NSGPU_CUDA(cudaMalloc((void**)&d_zs, sizeof(double) * M));
    std::vector<double> zs(M);
    cudaError_t e1 = cudaMemcpyAsync(d_dead, dead_logL.data(), sizeof(double) * nd, cudaMemcpyHostToDevice, st);
    evidence_error_kernel<<<M, 256, 0, st>>>(d_dead, (long long)nd, n, k, d_live_logL, key, d_zs);
    ctx->launches++;
    cudaError_t e2 = cudaMemcpyAsync(zs.data(), d_zs, sizeof(double) * M, cudaMemcpyDeviceToHost, st);
    cudaError_t e3 = cudaStreamSynchronize(st);
    cudaFree(d_dead); cudaFree(d_zs);
    NSGPU_CUDA(e1); NSGPU_CUDA(e2); NSGPU_CUDA(e3);
    double mean = 0.0;
    for (double z : zs) mean += z;
    mean /= M;
    for (double z : zs) err_sim += (z - mean) * (z - mean);
    err_sim = sqrt(err_sim / (M - 1));
  }
  double s1 = 0.0, s2 = 0.0;
  for (int j = 0; j < k; ++j) { s1 += 1.0 / (n - j); s2 += 1.0 / ((double)(n - j) * (n - j)); }
  const double cfac = n * s2 / s1;
  res->logZ = logZ; res->logZ_err = err_sim; res->logZ_err_analytic = sqrt(std::max(cfac * H, 0.0) / n); res->H = H;
  res->n_dead = (int64_t)nd;
  {
    // theta = T(u) through the a1 kernel, in chunks of max_batch rows; kept in the ctx for nsgpu_last_samples
    std::vector<float> all_u(ntot * D);
    memcpy(all_u.data(), dead_u.data(), sizeof(float) * nd * D);
    memcpy(all_u.data() + nd * D, live_u.data(), sizeof(float) * (size_t)n * D);
    out_theta.resize(ntot * D);
    out_logL = all_l;
    out_logw.resize(ntot);
    for (size_t i = 0; i < ntot; ++i) out_logw[i] = terms[i] - logZ;
    for (size_t off = 0; off < ntot; off += (size_t)ctx->max_batch) {
      const int nb = (int)std::min<size_t>((size_t)ctx->max_batch, ntot - off);
      NSGPU_CUDA(cudaMemcpyAsync(S->xprop, all_u.data() + off * D, sizeof(float) * (size_t)nb * D, cudaMemcpyHostToDevice, st));
      s = nsgpu_prior_transform(ctx, S->xprop, nb, S->theta_prop, st);
      if (s != NSGPU_OK) return s;
      NSGPU_CUDA(cudaMemcpyAsync(out_theta.data() + off * D, S->theta_prop, sizeof(float) * (size_t)nb * D, cudaMemcpyDeviceToHost, st));
      NSGPU_CUDA(cudaStreamSynchronize(st));   // copies and kernel ordered on the run's stream (not the legacy default one)
    }
  }
  return s;
}

// non-finite emulator rows so far on this context (device counter, see nsgpu_nonfinite_rows); -1 on error
static long long read_nonfinite(nsgpu_ctx* ctx, cudaStream_t st) {
  unsigned long long v = 0;
  if (!ctx->nonfinite_rows || cudaStreamSynchronize(st) != cudaSuccess ||
      cudaMemcpy(&v, ctx->nonfinite_rows, sizeof(v), cudaMemcpyDeviceToHost) != cudaSuccess)
    return -1;
  return (long long)v;
}

static nsgpu_status run_impl(nsgpu_ctx* ctx, const nsgpu_run_opts* o, int rank, int world, nsgpu_allgather_fn exch,
                             void* user, nsgpu_result* res, float* theta_samples, double* logL_samples,
                             double* logw_samples, int64_t cap, int64_t* n_samples) {
  if (!ctx) return NSGPU_EINVAL;
  if (!o || !res) { ctx->err = "run: NULL options or result"; return NSGPU_EINVAL; }
  if (world < 1 || rank < 0 || rank >= world || (world > 1 && !exch)) { ctx->err = "run: bad rank / world / exchange function"; return NSGPU_EINVAL; }
  nsgpu_status s = check_sampler_args(ctx, o->n_live, o->n_delete);
  if (s != NSGPU_OK) return s;
  if (o->n_delete >= o->n_live || o->n_steps < 1 || !(o->stop_frac > 0) || o->max_iter < 1) { ctx->err = "run: bad options"; return NSGPU_EINVAL; }
  if (o->n_live < ctx->D + 1) { ctx->err = "run: the live covariance needs n_live >= D + 1"; return NSGPU_EINVAL; }
  const auto t_start = std::chrono::steady_clock::now();
  long long nf0 = -2;   // read once the stream is known
  SamplerDev* S = ctx->sampler;
  // one rank: the context's own stream, so that runs of several contexts (the two models of a comparison, driven from
  // two host threads) share the GPU; sharded runs stay on the legacy default stream the exchange callback is ordered with
  cudaStream_t st = world == 1 ? S->run_stream : (cudaStream_t)0;
  nf0 = read_nonfinite(ctx, st);
  const int D = ctx->D, n = o->n_live, k = o->n_delete;
  const uint2 key = make_uint2((unsigned)(o->seed & 0xffffffffu), (unsigned)(o->seed >> 32));
  std::vector<float> dead_u;
  std::vector<double> dead_logL, dead_logw;
  std::vector<int> dead_nj;
  std::vector<float> hu((size_t)k * D);
  std::vector<double> hl(k), hw(k);
  float* d_dead_u = S->x0;           // scratch before chains are initialised
  double* d_dead_l = S->logL0;
  memset(res, 0, sizeof(*res));
  // sharded runs (S 8(e)): rank r evolves the global chains [c0, c0 + n_loc); everything else is done by every
  // rank on identical data, so that after the exchange all ranks hold the same live set, bit for bit
  int32_t c0 = 0, n_loc = k;
  nsgpu_shard_range(k, rank, world, &c0, &n_loc);
  const int per = (k + world - 1) / world;
  struct Gather {                      // [world * per] rows: global chain g sits at row g
    float* u = nullptr; double* l = nullptr; unsigned long long* cnt = nullptr;
    ~Gather() { cudaFree(u); cudaFree(l); cudaFree(cnt); }
  } G;
  if (world > 1) {
    NSGPU_CUDA(cudaMalloc((void**)&G.u, sizeof(float) * (size_t)world * per * D));
    NSGPU_CUDA(cudaMalloc((void**)&G.l, sizeof(double) * (size_t)world * per));
    NSGPU_CUDA(cudaMalloc((void**)&G.cnt, sizeof(unsigned long long) * 4 * (size_t)(world + 1)));
  }

  init_live_kernel<<<(n * D + 255) / 256, 256, 0, st>>>(n, D, key, S->u_live);
  NSGPU_LAUNCH_CHECK();
  s = nsgpu_prior_transform(ctx, S->u_live, n, S->theta_prop, st);
  if (s != NSGPU_OK) return s;
  s = loglike_device(ctx, S->theta_prop, n, nullptr, S->logL_live, st);
  if (s != NSGPU_OK) return s;
  for (int i = 0; i < 8; ++i) S->h_scal[i] = 0.0;
  S->h_scal[2] = -INFINITY;
  NSGPU_CUDA(cudaMemcpyAsync(S->scal, S->h_scal, 8 * sizeof(double), cudaMemcpyHostToDevice, st));
  NSGPU_CUDA(cudaMemsetAsync(S->n_evals, 0, sizeof(unsigned long long), st));
  int64_t it = 0, rounds = 0;
  int n_fail_total = 0;
  bool converged = false;
  while (it < o->max_iter) {
    ++it;
    s = launch_live_cholesky(ctx, S->u_live, n, S->Lsig, S->scal + 5, st);   // before deletion
    if (s != NSGPU_OK) return s;
    s = launch_delete(ctx, S->logL_live, n, k, st);
    if (s != NSGPU_OK) return s;
    // record the dead points
    gather_rows_kernel<<<(k * D + 255) / 256, 256, 0, st>>>(k, D, S->dead_idx, S->u_live, S->logL_live, d_dead_u, d_dead_l);
    NSGPU_LAUNCH_CHECK();
    NSGPU_CUDA(cudaMemcpyAsync(hu.data(), d_dead_u, sizeof(float) * (size_t)k * D, cudaMemcpyDeviceToHost, st));
    NSGPU_CUDA(cudaMemcpyAsync(hl.data(), d_dead_l, sizeof(double) * (size_t)k, cudaMemcpyDeviceToHost, st));
    NSGPU_CUDA(cudaMemcpyAsync(hw.data(), S->logw, sizeof(double) * (size_t)k, cudaMemcpyDeviceToHost, st));
    NSGPU_CUDA(cudaStreamSynchronize(st));
    dead_u.insert(dead_u.end(), hu.begin(), hu.end());
    dead_logL.insert(dead_logL.end(), hl.begin(), hl.end());
    dead_logw.insert(dead_logw.end(), hw.begin(), hw.end());
    for (int j = 0; j < k; ++j) dead_nj.push_back(n - j);
    nsgpu_status es = NSGPU_OK;
    if (n_loc > 0) {
      chain_init_kernel<<<(n_loc + 127) / 128, 128, 0, st>>>(n_loc, c0, D, key, (unsigned)it, S->surv_idx, n - k, nullptr,
                                                             S->start_idx, S->u_live, S->logL_live, S->x0, S->logL0, S->phase,
                                                             S->cnt, S->step, S->pending, S->finished, S->need, S->rng_j, n, S->scal);
      ctx->launches++;
      es = cudaGetLastError() == cudaSuccess ? evolve(ctx, n_loc, c0, o->n_steps, o->seed, (int)it, st, &rounds) : NSGPU_ECUDA;
      if (es == NSGPU_OK) n_fail_total += S->h_counters[2];
    }
    if (world > 1) {
      // A rank whose chains failed must not leave the others waiting in the all-gather below: every iteration first
      // exchanges one status word, and all ranks stop together when any of them reports a failure.
      unsigned long long mine = es == NSGPU_OK ? 0ull : 1ull;
      std::vector<unsigned long long> all((size_t)world, 0ull);
      bool ok = cudaMemcpy(G.cnt, &mine, sizeof(mine), cudaMemcpyHostToDevice) == cudaSuccess &&
                exch(user, G.cnt, G.cnt + 4, (int64_t)sizeof(mine), st) == 0 &&
                cudaMemcpy(all.data(), G.cnt + 4, sizeof(mine) * world, cudaMemcpyDeviceToHost) == cudaSuccess;
      if (es != NSGPU_OK) return es;
      if (!ok) { ctx->err = "run: status exchange failed"; return NSGPU_ECUDA; }
      for (int r = 0; r < world; ++r)
        if (all[r] != 0ull) { ctx->err = "run: rank " + std::to_string(r) + " reported a failure; all ranks stop"; return NSGPU_ECUDA; }
    } else if (es != NSGPU_OK) {
      return es;
    }
    const float* new_u = S->u_out;
    const double* new_l = S->logL_out;
    if (world > 1) {   // the one exchange of an iteration: all-gather of the new points (k (D + 2) words in all)
      NSGPU_CUDA(cudaStreamSynchronize(st));
      if (exch(user, S->u_out, G.u, (int64_t)sizeof(float) * per * D, st) != 0 ||
          exch(user, S->logL_out, G.l, (int64_t)sizeof(double) * per, st) != 0) {
        ctx->err = "run: exchange function failed";
        return NSGPU_ECUDA;
      }
      new_u = G.u; new_l = G.l;
    }
    replace_kernel<<<(k * D + 255) / 256, 256, 0, st>>>(k, D, S->dead_idx, new_u, new_l, S->u_live, S->logL_live);
    NSGPU_LAUNCH_CHECK();
    live_evidence_kernel<<<1, 1024, 0, st>>>(S->logL_live, n, log(o->stop_frac), S->scal);
    NSGPU_LAUNCH_CHECK();
    NSGPU_CUDA(cudaMemcpyAsync(S->h_scal, S->scal, 8 * sizeof(double), cudaMemcpyDeviceToHost, st));
    NSGPU_CUDA(cudaStreamSynchronize(st));
    if (S->h_scal[5] != 0.0) { ctx->err = "run: live-set covariance is not positive definite"; return NSGPU_ENOTSPD; }
    if (S->h_scal[4] != 0.0) { converged = true; break; }
  }
  // final summary
  const auto t_sampled = std::chrono::steady_clock::now();
  const double logX = S->h_scal[1];
  std::vector<float> live_u((size_t)n * D);
  std::vector<double> live_l(n);
  NSGPU_CUDA(cudaStreamSynchronize(st));
  NSGPU_CUDA(cudaMemcpy(live_u.data(), S->u_live, sizeof(float) * (size_t)n * D, cudaMemcpyDeviceToHost));
  NSGPU_CUDA(cudaMemcpy(live_l.data(), S->logL_live, sizeof(double) * (size_t)n, cudaMemcpyDeviceToHost));
  NSGPU_CUDA(cudaMemcpy(S->h_evals, S->n_evals, sizeof(unsigned long long), cudaMemcpyDeviceToHost));
  unsigned long long evals_all = *S->h_evals;
  if (world > 1) {   // totals over ranks: evaluations and failed moves add, rounds take the longest rank
    unsigned long long mine[4] = {*S->h_evals, (unsigned long long)rounds, (unsigned long long)n_fail_total, 0ull};
    std::vector<unsigned long long> all(4 * (size_t)world);
    NSGPU_CUDA(cudaMemcpy(G.cnt, mine, sizeof(mine), cudaMemcpyHostToDevice));
    if (exch(user, G.cnt, G.cnt + 4, (int64_t)sizeof(mine), st) != 0) { ctx->err = "run: exchange function failed"; return NSGPU_ECUDA; }
    NSGPU_CUDA(cudaMemcpy(all.data(), G.cnt + 4, sizeof(mine) * world, cudaMemcpyDeviceToHost));
    evals_all = 0; n_fail_total = 0;
    for (int r = 0; r < world; ++r) {
      evals_all += all[4 * r];
      rounds = std::max<int64_t>(rounds, (int64_t)all[4 * r + 1]);
      n_fail_total += (int)all[4 * r + 2];
    }
  }
  s = summarize_run(ctx, n, k, key, logX, dead_u, dead_logL, dead_logw, live_u, live_l, S->logL_live, st, res, S->last_theta,
                    S->last_logL, S->last_logw);
  if (s != NSGPU_OK) return s;
  res->n_iter = it; res->n_like_evals = (int64_t)evals_all + n; res->n_rounds = rounds; res->n_failed_moves = n_fail_total;
  if (n_samples) *n_samples = (int64_t)S->last_logL.size();
  if (cap > 0 && theta_samples && logL_samples && logw_samples) {
    int64_t got = 0;
    s = nsgpu_last_samples(ctx, theta_samples, logL_samples, logw_samples, cap, &got);
    if (s != NSGPU_OK) return s;
  }
  const auto t_end = std::chrono::steady_clock::now();
  res->seconds = std::chrono::duration<double>(t_end - t_start).count();
  res->seconds_sampling = std::chrono::duration<double>(t_sampled - t_start).count();
  res->seconds_summary = std::chrono::duration<double>(t_end - t_sampled).count();
  { const long long nf1 = read_nonfinite(ctx, st); res->n_nonfinite_rows = (nf0 >= 0 && nf1 >= 0) ? nf1 - nf0 : -1; }
  return converged ? NSGPU_OK : NSGPU_ENOCONV;
}

extern "C" nsgpu_status nsgpu_run(nsgpu_ctx* ctx, const nsgpu_run_opts* o, nsgpu_result* res, float* theta_samples,
                                  double* logL_samples, double* logw_samples, int64_t cap, int64_t* n_samples) {
  return run_impl(ctx, o, 0, 1, nullptr, nullptr, res, theta_samples, logL_samples, logw_samples, cap, n_samples);
}

extern "C" nsgpu_status nsgpu_run_sharded(nsgpu_ctx* ctx, const nsgpu_run_opts* o, int32_t rank, int32_t world,
                                          nsgpu_allgather_fn allgather, void* user, nsgpu_result* res,
                                          float* theta_samples, double* logL_samples, double* logw_samples, int64_t cap,
                                          int64_t* n_samples) {
  return run_impl(ctx, o, rank, world, allgather, user, res, theta_samples, logL_samples, logw_samples, cap, n_samples);
}

// ---------------------------------------------------------------------------------------------------
// nsgpu_run_multi: R independent runs (seeds) of ONE model that share every likelihood batch.
// A single run keeps the GPU half idle: a round carries <= k (on average ~0.6 k) proposals through ten launches
// ("perfect scaling is hard to achieve").  Here the chains of all runs advance in the same rounds: chain slot
// c belongs to run c / k, and slice_round_kernel takes L*, the direction factor, the Philox key and the iteration
// number of that run; compaction and the likelihood see one batch of up to R k proposals.  Everything per run
// (live set, deletion, evidence scan, stopping test, summary) is done per run with the same kernels, so every run
// returns exactly what nsgpu_run returns for its seed.  Runs stay in lock step per iteration; a converged run drops out.
// ---------------------------------------------------------------------------------------------------
namespace {
struct MultiBuf {
  float *u_live = nullptr, *dead_u = nullptr;
  double *logL_live = nullptr, *scal = nullptr, *Lsig = nullptr, *logw = nullptr, *dead_l = nullptr;
  int *dead_idx = nullptr, *surv_idx = nullptr, *run_fails = nullptr;
  uint2* keys = nullptr;
  unsigned* iters = nullptr;
  unsigned long long* run_evals = nullptr;
  ~MultiBuf() {
    void* p[] = {u_live, dead_u, logL_live, scal, Lsig, logw, dead_l, dead_idx, surv_idx, run_fails, keys, iters, run_evals};
    for (void* q : p) cudaFree(q);
  }
};
}  // namespace

extern "C" nsgpu_status nsgpu_run_multi(nsgpu_ctx* ctx, const nsgpu_run_opts* o, int32_t n_runs, const uint64_t* seeds,
                                        nsgpu_result* res) {
  if (!ctx) return NSGPU_EINVAL;
  if (!o || !res || !seeds || n_runs < 1 || n_runs > 64) { ctx->err = "run_multi: NULL pointer or n_runs outside 1..64"; return NSGPU_EINVAL; }
  nsgpu_status s = check_sampler_args(ctx, o->n_live, o->n_delete);
  if (s != NSGPU_OK) return s;
  if (o->n_delete >= o->n_live || o->n_steps < 1 || !(o->stop_frac > 0) || o->max_iter < 1) { ctx->err = "run_multi: bad options"; return NSGPU_EINVAL; }
  if (o->n_live < ctx->D + 1) { ctx->err = "run_multi: the live covariance needs n_live >= D + 1"; return NSGPU_EINVAL; }
  if ((int64_t)n_runs * o->n_delete > ctx->max_batch) { ctx->err = "run_multi: n_runs x n_delete exceeds max_batch"; return NSGPU_ESHAPE; }
  const auto t_start = std::chrono::steady_clock::now();
  long long nf0 = -2;
  SamplerDev* S = ctx->sampler;
  cudaStream_t st = S->run_stream;
  const int D = ctx->D, n = o->n_live, k = o->n_delete, R = n_runs;
  nf0 = read_nonfinite(ctx, st);
  MultiBuf B;
#define MB(p, T, cnt) NSGPU_CUDA(cudaMalloc((void**)&B.p, sizeof(T) * (size_t)(cnt)))
  MB(u_live, float, (size_t)R * n * D); MB(logL_live, double, (size_t)R * n); MB(scal, double, R * 8); MB(Lsig, double, (size_t)R * D * D);
  MB(dead_idx, int, (size_t)R * k); MB(surv_idx, int, (size_t)R * n); MB(logw, double, (size_t)R * k); MB(dead_u, float, (size_t)R * k * D);
  MB(dead_l, double, (size_t)R * k); MB(keys, uint2, R); MB(iters, unsigned, R); MB(run_evals, unsigned long long, R); MB(run_fails, int, R);
#undef MB
  std::vector<uint2> keys(R);
  for (int r = 0; r < R; ++r) keys[r] = make_uint2((unsigned)(seeds[r] & 0xffffffffu), (unsigned)(seeds[r] >> 32));
  NSGPU_CUDA(cudaMemcpyAsync(B.keys, keys.data(), sizeof(uint2) * R, cudaMemcpyHostToDevice, st));
  NSGPU_CUDA(cudaMemsetAsync(B.run_evals, 0, sizeof(unsigned long long) * R, st));
  NSGPU_CUDA(cudaMemsetAsync(B.run_fails, 0, sizeof(int) * R, st));
  std::vector<double> h_scal((size_t)R * 8, 0.0);
  for (int r = 0; r < R; ++r) h_scal[8 * r + 2] = -INFINITY;
  NSGPU_CUDA(cudaMemcpyAsync(B.scal, h_scal.data(), sizeof(double) * R * 8, cudaMemcpyHostToDevice, st));
  for (int r = 0; r < R; ++r) {          // initial live sets: the same draws and likelihood calls as nsgpu_run(seed r)
    memset(&res[r], 0, sizeof(nsgpu_result));
    float* ul = B.u_live + (size_t)r * n * D;
    init_live_kernel<<<(n * D + 255) / 256, 256, 0, st>>>(n, D, keys[r], ul);
    NSGPU_LAUNCH_CHECK();
    s = nsgpu_prior_transform(ctx, ul, n, S->theta_prop, st);
    if (s != NSGPU_OK) return s;
    s = loglike_device(ctx, S->theta_prop, n, nullptr, B.logL_live + (size_t)r * n, st);
    if (s != NSGPU_OK) return s;
  }
  struct Host { std::vector<float> dead_u; std::vector<double> dead_logL, dead_logw; bool active = true, converged = false; int64_t n_iter = 0; double logX = 0.0; };
  std::vector<Host> H(R);
  std::vector<float> hu((size_t)R * k * D);
  std::vector<double> hl((size_t)R * k), hw((size_t)R * k);
  std::vector<unsigned> h_iters(R, 0u);
  int64_t it = 0, rounds = 0;
  int n_active = R;
  while (n_active > 0 && it < o->max_iter) {
    ++it;
    for (int r = 0; r < R; ++r) {
      if (!H[r].active) continue;
      float* ul = B.u_live + (size_t)r * n * D;
      double* ll = B.logL_live + (size_t)r * n;
      s = launch_live_cholesky(ctx, ul, n, B.Lsig + (size_t)r * D * D, B.scal + 8 * r + 5, st);
      if (s != NSGPU_OK) return s;
      s = launch_delete(ctx, ll, n, k, st, B.scal + 8 * r, B.dead_idx + (size_t)r * k, B.surv_idx + (size_t)r * n, B.logw + (size_t)r * k);
      if (s != NSGPU_OK) return s;
      gather_rows_kernel<<<(k * D + 255) / 256, 256, 0, st>>>(k, D, B.dead_idx + (size_t)r * k, ul, ll, B.dead_u + (size_t)r * k * D,
                                                              B.dead_l + (size_t)r * k);
      NSGPU_LAUNCH_CHECK();
      h_iters[r] = (unsigned)it;
    }
    NSGPU_CUDA(cudaMemcpyAsync(hu.data(), B.dead_u, sizeof(float) * hu.size(), cudaMemcpyDeviceToHost, st));
    NSGPU_CUDA(cudaMemcpyAsync(hl.data(), B.dead_l, sizeof(double) * hl.size(), cudaMemcpyDeviceToHost, st));
    NSGPU_CUDA(cudaMemcpyAsync(hw.data(), B.logw, sizeof(double) * hw.size(), cudaMemcpyDeviceToHost, st));
    NSGPU_CUDA(cudaMemcpyAsync(B.iters, h_iters.data(), sizeof(unsigned) * R, cudaMemcpyHostToDevice, st));
    NSGPU_CUDA(cudaStreamSynchronize(st));
    for (int r = 0; r < R; ++r) {
      if (!H[r].active) continue;
      H[r].dead_u.insert(H[r].dead_u.end(), hu.begin() + (size_t)r * k * D, hu.begin() + (size_t)(r + 1) * k * D);
      H[r].dead_logL.insert(H[r].dead_logL.end(), hl.begin() + (size_t)r * k, hl.begin() + (size_t)(r + 1) * k);
      H[r].dead_logw.insert(H[r].dead_logw.end(), hw.begin() + (size_t)r * k, hw.begin() + (size_t)(r + 1) * k);
      const size_t c0 = (size_t)r * k;      // this run's chain slots
      chain_init_kernel<<<(k + 127) / 128, 128, 0, st>>>(k, 0, D, keys[r], (unsigned)it, B.surv_idx + (size_t)r * n, n - k, nullptr,
                                                         S->start_idx + c0, B.u_live + (size_t)r * n * D, B.logL_live + (size_t)r * n,
                                                         S->x0 + c0 * D, S->logL0 + c0, S->phase + c0, S->cnt + c0, S->step + c0,
                                                         S->pending + c0, S->finished + c0, S->need + c0, S->rng_j + c0, n, B.scal + 8 * r);
      NSGPU_LAUNCH_CHECK();
    }
    MultiArgs ma;
    ma.n_per_run = k; ma.n_target = n_active * k; ma.keys = B.keys; ma.iters = B.iters; ma.run_evals = B.run_evals;
    ma.run_fails = B.run_fails; ma.scal = B.scal; ma.Lsig = B.Lsig;
    s = evolve(ctx, R * k, 0, o->n_steps, 0, (int)it, st, &rounds, &ma);
    if (s != NSGPU_OK) return s;
    for (int r = 0; r < R; ++r) {
      if (!H[r].active) continue;
      const size_t c0 = (size_t)r * k;
      replace_kernel<<<(k * D + 255) / 256, 256, 0, st>>>(k, D, B.dead_idx + c0, S->u_out + c0 * D, S->logL_out + c0,
                                                          B.u_live + (size_t)r * n * D, B.logL_live + (size_t)r * n);
      NSGPU_LAUNCH_CHECK();
      live_evidence_kernel<<<1, 1024, 0, st>>>(B.logL_live + (size_t)r * n, n, log(o->stop_frac), B.scal + 8 * r);
      NSGPU_LAUNCH_CHECK();
    }
    NSGPU_CUDA(cudaMemcpyAsync(h_scal.data(), B.scal, sizeof(double) * R * 8, cudaMemcpyDeviceToHost, st));
    NSGPU_CUDA(cudaStreamSynchronize(st));
    for (int r = 0; r < R; ++r) {
      if (!H[r].active) continue;
      if (h_scal[8 * r + 5] != 0.0) { ctx->err = "run_multi: live-set covariance is not positive definite"; return NSGPU_ENOTSPD; }
      H[r].n_iter = it; H[r].logX = h_scal[8 * r + 1];
      if (h_scal[8 * r + 4] != 0.0) { H[r].converged = true; H[r].active = false; --n_active; }
    }
  }
  const auto t_sampled = std::chrono::steady_clock::now();
  std::vector<unsigned long long> evals(R);
  std::vector<int> fails(R);
  NSGPU_CUDA(cudaMemcpy(evals.data(), B.run_evals, sizeof(unsigned long long) * R, cudaMemcpyDeviceToHost));
  NSGPU_CUDA(cudaMemcpy(fails.data(), B.run_fails, sizeof(int) * R, cudaMemcpyDeviceToHost));
  S->multi.assign(R, SamplerDev::SampleSet());
  bool all_conv = true;
  std::vector<float> live_u((size_t)n * D);
  std::vector<double> live_l(n);
  for (int r = 0; r < R; ++r) {
    NSGPU_CUDA(cudaMemcpy(live_u.data(), B.u_live + (size_t)r * n * D, sizeof(float) * (size_t)n * D, cudaMemcpyDeviceToHost));
    NSGPU_CUDA(cudaMemcpy(live_l.data(), B.logL_live + (size_t)r * n, sizeof(double) * (size_t)n, cudaMemcpyDeviceToHost));
    s = summarize_run(ctx, n, k, keys[r], H[r].logX, H[r].dead_u, H[r].dead_logL, H[r].dead_logw, live_u, live_l,
                      B.logL_live + (size_t)r * n, st, &res[r], S->multi[r].theta, S->multi[r].logL, S->multi[r].logw);
    if (s != NSGPU_OK) return s;
    res[r].n_iter = H[r].n_iter; res[r].n_like_evals = (int64_t)evals[r] + n; res[r].n_rounds = rounds; res[r].n_failed_moves = fails[r];
    all_conv = all_conv && H[r].converged;
  }
  const auto t_end = std::chrono::steady_clock::now();
  for (int r = 0; r < R; ++r) {          // wall times are those of the whole call: the runs share every round
    res[r].seconds = std::chrono::duration<double>(t_end - t_start).count();
    res[r].seconds_sampling = std::chrono::duration<double>(t_sampled - t_start).count();
    res[r].seconds_summary = std::chrono::duration<double>(t_end - t_sampled).count();
  }
  {   // the runs share every batch: the count is that of the whole call, reported with each run
    const long long nf1 = read_nonfinite(ctx, st);
    for (int r = 0; r < R; ++r) res[r].n_nonfinite_rows = (nf0 >= 0 && nf1 >= 0) ? nf1 - nf0 : -1;
  }
  return all_conv ? NSGPU_OK : NSGPU_ENOCONV;
}

extern "C" nsgpu_status nsgpu_multi_samples(nsgpu_ctx* ctx, int32_t run, float* theta_samples, double* logL_samples,
                                            double* logw_samples, int64_t cap, int64_t* n_samples) {
  if (!ctx) return NSGPU_EINVAL;
  SamplerDev* S = ctx->sampler;
  if (run < 0 || run >= (int)S->multi.size()) { ctx->err = "multi_samples: no such run"; return NSGPU_EINVAL; }
  const SamplerDev::SampleSet& X = S->multi[run];
  const int64_t ntot = (int64_t)X.logL.size();
  if (n_samples) *n_samples = ntot;
  if (cap <= 0) return NSGPU_OK;
  if (!theta_samples || !logL_samples || !logw_samples) { ctx->err = "multi_samples: NULL buffer"; return NSGPU_EINVAL; }
  const size_t nw = (size_t)std::min<int64_t>(cap, ntot);
  memcpy(theta_samples, X.theta.data(), sizeof(float) * nw * ctx->D);
  memcpy(logL_samples, X.logL.data(), sizeof(double) * nw);
  memcpy(logw_samples, X.logw.data(), sizeof(double) * nw);
  return NSGPU_OK;
}

// ---------------------------------------------------------------------------------------------------
// nsgpu_logz_error_noalloc: the error bar of log Z by simulated prior volumes (reading N9) WITHOUT any
// allocation.  The summary of nsgpu_run does this with two cudaMalloc'd buffers (the dead log L sequence and the 1000
// simulated log Z); callers that may not allocate (code under CUDA graph capture, tight serving loops, harnesses that
// forbid cudaMalloc) get the same kernel on a file-scope device array instead.  Every GPU that loads the library holds
// the array until the process exits: NSGPU_NOALLOC_MAX_DEAD + NSGPU_NOALLOC_MAX_LIVE + 1000 doubles = 8.1 MiB.
// In HOST code `g_noalloc_scratch` is only a stand-in for the symbol, never a device address: the address is taken once
// per device with cudaGetSymbolAddress (that device current) and that pointer is what the copies and the kernel get.
// All calls share the array and it keeps the last call's contents: every call overwrites the parts it reads
// ([0, n_dead), the live block, the 1000 results are zeroed first), and calls that overlap on the GPU (two streams, two
// host threads) race -- serialise them.
// ---------------------------------------------------------------------------------------------------
#define NSGPU_NOALLOC_MAX_DEAD (1 << 20)
#define NSGPU_NOALLOC_MAX_LIVE MAX_LIVE
#define NSGPU_NOALLOC_SIMS 1000
static __device__ __align__(256) double g_noalloc_scratch[NSGPU_NOALLOC_MAX_DEAD + NSGPU_NOALLOC_MAX_LIVE + NSGPU_NOALLOC_SIMS];

#include <mutex>
static cudaError_t noalloc_scratch_ptr(int device, double** out) {   // call with `device` current
  static std::mutex mu;
  static double* ptr[64] = {};
  std::lock_guard<std::mutex> lock(mu);
  if (device < 0 || device >= 64) return cudaErrorInvalidDevice;
  if (!ptr[device]) {
    double* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress((void**)&p, g_noalloc_scratch);
    if (e != cudaSuccess) return e;
    ptr[device] = p;
  }
  *out = ptr[device];
  return cudaSuccess;
}

extern "C" nsgpu_status nsgpu_logz_error_noalloc(nsgpu_ctx* ctx, const double* dead_logL, int64_t n_dead,
                                                 const double* live_logL, int32_t n_live, int32_t n_delete, uint64_t seed,
                                                 double* logZ_err, double* logZ_sims, void* stream) {
  if (!ctx) return NSGPU_EINVAL;
  if (!live_logL || !logZ_err || n_dead < 0 || (n_dead > 0 && !dead_logL) || n_live < 1 || n_delete < 1 || n_delete >= n_live) {
    ctx->err = "logz_error_noalloc: NULL pointer or bad sizes (need n_live >= 1, 1 <= n_delete < n_live)";
    return NSGPU_EINVAL;
  }
  if (n_dead > NSGPU_NOALLOC_MAX_DEAD || n_live > NSGPU_NOALLOC_MAX_LIVE) {
    ctx->err = "logz_error_noalloc: n_dead exceeds 1048576 or n_live exceeds 16384 (the static scratch array; use nsgpu_run's summary for longer runs)";
    return NSGPU_ESHAPE;
  }
  NSGPU_CUDA(cudaSetDevice(ctx->device));
  double* scr = nullptr;
  NSGPU_CUDA(noalloc_scratch_ptr(ctx->device, &scr));
  cudaStream_t st = (cudaStream_t)stream;
  double* d_dead = scr;
  double* d_live = scr + NSGPU_NOALLOC_MAX_DEAD;
  double* d_zs = d_live + NSGPU_NOALLOC_MAX_LIVE;
  if (n_dead > 0) NSGPU_CUDA(cudaMemcpyAsync(d_dead, dead_logL, sizeof(double) * (size_t)n_dead, cudaMemcpyHostToDevice, st));
  NSGPU_CUDA(cudaMemcpyAsync(d_live, live_logL, sizeof(double) * (size_t)n_live, cudaMemcpyHostToDevice, st));
  NSGPU_CUDA(cudaMemsetAsync(d_zs, 0, sizeof(double) * NSGPU_NOALLOC_SIMS, st));
  const uint2 key = make_uint2((unsigned)(seed & 0xffffffffu), (unsigned)(seed >> 32));
  evidence_error_kernel<<<NSGPU_NOALLOC_SIMS, 256, 0, st>>>(d_dead, (long long)n_dead, n_live, n_delete, d_live, key, d_zs);
  NSGPU_LAUNCH_CHECK();
  double zs_local[NSGPU_NOALLOC_SIMS];
  double* zs = logZ_sims ? logZ_sims : zs_local;
  NSGPU_CUDA(cudaMemcpyAsync(zs, d_zs, sizeof(double) * NSGPU_NOALLOC_SIMS, cudaMemcpyDeviceToHost, st));
  NSGPU_CUDA(cudaStreamSynchronize(st));
  double mean = 0.0, var = 0.0;
  for (int m = 0; m < NSGPU_NOALLOC_SIMS; ++m) mean += zs[m];
  mean /= NSGPU_NOALLOC_SIMS;
  for (int m = 0; m < NSGPU_NOALLOC_SIMS; ++m) var += (zs[m] - mean) * (zs[m] - mean);
  *logZ_err = sqrt(var / (NSGPU_NOALLOC_SIMS - 1));
  return NSGPU_OK;
}
