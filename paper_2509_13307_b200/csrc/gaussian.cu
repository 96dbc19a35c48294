// gaussian.cu -- step a10: Gaussian log-likelihood against a fixed dense covariance, and
// step a1: the prior transform (Table 1).
//
// log L = -1/2 sum w^2 - 1/2 ln det(2 pi C), w = L^-1 (model - d).  The whitening is a triangular
// solve against the Cholesky factor; because the factor is fixed for the life of the context its
// inverse (also lower triangular) is formed once, in fp64, at create, and the solve becomes the
// triangular product w = Linv r -- the limit of a blocked TRSM with pre-inverted diagonal blocks.
// Residuals, products and the sum of squares are fp64 (reading P1): n(n+1)/2 MAC per theta is three
// orders of magnitude below the emulator's work, and an fp32 whitening would eat the 1e-3 budget.
// Two kernels: chi2_kernel streams the factor through every CTA (n_data < 512); chi2_tile_kernel is a blocked
// triangular product on the fp64 tensor cores (larger data vectors).
#include "internal.cuh"
#include "tc_ptx.cuh"

namespace {


// w = Linv r for TB thetas at once.  A thread owns a PAIR of rows (t, n-1-t) -- n+1 non-zero columns
// whatever t is, so the triangular work is balanced -- and TG of the CTA's TB thetas.  The factor is
// streamed through shared memory in chunks of CH columns (LinvT rows, contiguous in memory) by bulk
// asynchronous copies, double buffered: thread 0 starts chunk c+1 while the CTA multiplies chunk c.
// The column index is uniform across a warp, so the residuals r[j][.] are one broadcast line of
// shared memory (a per-lane column made every load a 26-way bank conflict) and the factor elements
// S[j][row] are conflict-free; LinvT is stored as a full matrix whose upper part is zero, so lanes for
// which column j lies above their row just add 0.  Only the part of a chunk that can be non-zero is
// copied (rows i >= first column of the chunk: half the factor on average; LinvT rows have an even stride
// so that every such piece is 16-byte aligned); rows above it are masked, never read.
// fp64 throughout; chi^2 = sum over rows of w^2.
template <int TB, int TG, int MAXT>
__global__ void __launch_bounds__(MAXT) chi2_kernel(const double* __restrict__ model, const double* __restrict__ data,
                                                     const double* __restrict__ LinvT, int n, int ns, int B, int RT, int CH,
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
  constexpr int NBUF = 4;                                // factor chunks in flight: copy latency, not bandwidth, bounds a CTA
  unsigned long long* bars = reinterpret_cast<unsigned long long*>(part + 32 * TB);   // full[NBUF], empty[NBUF]
  const uint32_t full0 = tc::smem_u32(bars), empty0 = full0 + 8 * NBUF;
  double* S = reinterpret_cast<double*>(bars + 2 * NBUF);  // [NBUF][CH][ns], 16-byte aligned (n TB even)
  // ns: row stride of LinvT (even).  chunk c -> buffer: columns j0 .. j0 + jn, rows j0 .. ns of each (one bulk copy per column)
  const bool tri = ns >= 512;                               // short rows: one copy of whole rows is cheaper to issue
  auto load_chunk = [&](int c, int buf) {
    const int j0 = c * CH, jn = min(CH, n - j0);
    if (!tri) {
      const uint32_t bytes = (uint32_t)jn * ns * 8u;
      tc::mbar_arrive_expect_tx(full0 + 8 * buf, bytes);
      tc::bulk_load(tc::smem_u32(S + (size_t)buf * CH * ns), LinvT + (size_t)j0 * ns, bytes, full0 + 8 * buf);
      return;
    }
    const uint32_t bytes = (uint32_t)(ns - j0) * 8u;
    tc::mbar_arrive_expect_tx(full0 + 8 * buf, bytes * jn);
    for (int jj = 0; jj < jn; ++jj)
      tc::bulk_load(tc::smem_u32(S + ((size_t)buf * CH + jj) * ns + j0), LinvT + (size_t)(j0 + jj) * ns + j0, bytes,
                    full0 + 8 * buf);
  };
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarp = blockDim.x >> 5;
  const int n_chunks = (n + CH - 1) / CH;
  if (tid == 0) {
    for (int b = 0; b < NBUF; ++b) { tc::mbar_init(full0 + 8 * b, 1); tc::mbar_init(empty0 + 8 * b, nwarp); }
    tc::fence_barrier_init();
    for (int c = 0; c < NBUF - 1 && c < n_chunks; ++c) load_chunk(c, c);   // prologue: NBUF-1 chunks in flight
  }
  // residuals, transposed into [j][theta] (coalesced global reads along j)
  for (int i = tid; i < n * TB; i += blockDim.x) {
    const int t = i / n, j = i - t * n;
    const int b = b0 + t;
    r[(size_t)j * TB + t] = (b < B) ? model[(size_t)b * n + j] - data[j] : 0.0;
  }
  __syncthreads();
  const int half = (n + 1) >> 1;
  const int rt = tid % RT, grp = tid / RT;               // RT is a multiple of 32: a warp has one group
  const int ra = rt, rb = n - 1 - rt;                    // rows of this thread (ra <= rb); equal for the middle row
  const double* rg = r + grp * TG;                       // this group's thetas
  const int rt0 = rt & ~31;                              // first row-pair of this warp
  const int ja_end = min(rt0 + 31, half - 1);            // last column any lane's short row needs
  const int jb_end = n - 1 - rt0;                        // last column any lane's long row needs
  const int ia = min(ra, n - 1), ib = max(rb, 0);        // clamp the idle lanes of the last warp
  double wa[TG], wb[TG];
#pragma unroll
  for (int t = 0; t < TG; ++t) { wa[t] = 0.0; wb[t] = 0.0; }
  for (int c = 0; c < n_chunks; ++c) {
    const int buf = c % NBUF;
    if (tid == 0 && c + NBUF - 1 < n_chunks) {             // refill the buffer chunk c-1 used
      const int cn = c + NBUF - 1, nb = cn % NBUF;
      if (c >= 1) tc::mbar_wait(empty0 + 8 * nb, ((c - 1) / NBUF) & 1);
      load_chunk(cn, nb);
    }
    tc::mbar_wait(full0 + 8 * buf, (c / NBUF) & 1);
    const double* Sb = S + (size_t)buf * CH * ns;
    const int j0 = c * CH, jn = min(CH, n - j0);
    const bool has_a = ia >= j0, has_b = ib >= j0;           // rows above the chunk were not copied
    if (j0 <= jb_end) {
#pragma unroll 4
      for (int jj = 0; jj < jn; ++jj) {
        const int j = j0 + jj;
        const double lb = has_b ? Sb[(size_t)jj * ns + ib] : 0.0;
        double v[TG];
#pragma unroll
        for (int t = 0; t < TG; ++t) v[t] = rg[(size_t)j * TB + t];
#pragma unroll
        for (int t = 0; t < TG; ++t) wb[t] = fma(lb, v[t], wb[t]);
        if (j <= ja_end) {                                   // warp-uniform: the short rows end early
          const double la = has_a ? Sb[(size_t)jj * ns + ia] : 0.0;
#pragma unroll
          for (int t = 0; t < TG; ++t) wa[t] = fma(la, v[t], wa[t]);
        }
      }
    }
    __syncwarp();
    if (lane == 0) tc::mbar_arrive(empty0 + 8 * buf);
  }
  const bool one = rt < half, two = one && ra != rb;
#pragma unroll
  for (int t = 0; t < TG; ++t) {
    double ss = (one ? wb[t] * wb[t] : 0.0) + (two ? wa[t] * wa[t] : 0.0);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, o);
    if (lane == 0) part[(warp % (RT >> 5)) * TB + grp * TG + t] = ss;   // one slot per (row-warp, theta)
  }
  __syncthreads();
  if (tid < TB) {
    const int b = b0 + tid;
    if (b < B) {
      double chi2 = 0.0;
      for (int w = 0; w < (RT >> 5); ++w) chi2 += part[w * TB + tid];
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

// ---- the same streaming scheme on the fp64 tensor cores (n_data < 512) ---------------------------------------
// One CTA = all rows of 8 NTL thetas; the factor is streamed in chunks of CH columns as above, but the product is
// DMMA (m8n8k4): a warp owns the pair of 8-row tiles (w, MT-1-w) -- balanced triangular work as with the row pairs
// -- times NTL 8-theta tiles.  Per 4 columns: 2 A fragments, NTL B fragments, up to 2 NTL DMMAs of 256 FMA.
// LinvT rows are padded to a stride of 8 mod 16 doubles, in global memory too (fragment loads cover every bank
// twice; a chunk is one contiguous bulk copy).
__device__ __forceinline__ void dmma_8x8x4_s(double (&d)[2], double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
               : "+d"(d[0]), "+d"(d[1]) : "d"(a), "d"(b));
}
template <int NTL, int MAXT, int NBUF>
__global__ void __launch_bounds__(MAXT) chi2_mma_kernel(const double* __restrict__ model, const double* __restrict__ data,
                                                         const double* __restrict__ LinvT, int n, int B, int CH, int nsp,
                                                         const int* __restrict__ n_rows_dev, const float* __restrict__ theta,
                                                         int D, const int* __restrict__ prior_kind,
                                                         const double* __restrict__ p0, const double* __restrict__ p1,
                                                         double log_norm, double* __restrict__ logL) {
  constexpr int TB = 8 * NTL, TBP = TB + 8;               // NBUF chunks of the factor in flight
  pdl_wait();      // launch_pdl contract: the row count and the model vectors come from earlier kernels
  pdl_trigger();
  if (n_rows_dev) B = min(B, *n_rows_dev);
  const int b0 = blockIdx.x * TB;
  if (b0 >= B) return;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int n4 = (n + 3) & ~3;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarp = blockDim.x >> 5;
  double* r = reinterpret_cast<double*>(smem_raw);        // [n4][TBP] residuals, rows n .. n4-1 zero
  double* part = r + (size_t)n4 * TBP;                    // [nwarp][TB]
  unsigned long long* bars = reinterpret_cast<unsigned long long*>(part + (size_t)nwarp * TB);   // full[NBUF], empty[NBUF]
  int* bad = reinterpret_cast<int*>(bars + 2 * NBUF);     // [TB] theta outside the prior support / not finite
  double* S = reinterpret_cast<double*>(bad + TB);        // [NBUF][CH][nsp]
  const uint32_t full0 = tc::smem_u32(bars), empty0 = full0 + 8 * NBUF;
  const int n_chunks = (n + CH - 1) / CH;
  // LinvT rows have the same (padded) stride in global memory, so a chunk of CH columns is ONE contiguous bulk
  // copy.  (Copying only the rows below the chunk's first column halves the bytes but takes one copy per
  // column: measured slower, 0.060 vs 0.050 ms at B = 4096 -- small copies are bound by their number.)
  auto load_chunk = [&](int c, int buf) {                 // whole warp 0
    if (lane == 0) {
      const int j0 = c * CH, jn = min(CH, n - j0);
      const uint32_t bytes = (uint32_t)jn * nsp * 8u;
      tc::mbar_arrive_expect_tx(full0 + 8 * buf, bytes);
      tc::bulk_load(tc::smem_u32(S + (size_t)buf * CH * nsp), LinvT + (size_t)j0 * nsp, bytes, full0 + 8 * buf);
    }
  };
  if (tid == 0) {
    for (int b = 0; b < NBUF; ++b) { tc::mbar_init(full0 + 8 * b, 1); tc::mbar_init(empty0 + 8 * b, nwarp); }
    tc::fence_barrier_init();
  }
  __syncwarp();
  if (warp == 0)                                          // the first chunks travel while the residuals are formed
    for (int c = 0; c < NBUF - 1 && c < n_chunks; ++c) load_chunk(c, c);
  // residuals, transposed into [j][theta]: four independent loads in flight per thread (the loop is bound by the
  // latency of the model reads, not by their number)
  const int n_res = n4 * TB;
  for (int i0 = tid; i0 < n_res; i0 += 4 * blockDim.x) {
    double mv[4];
    int jj[4], tt[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      const int i = i0 + u * blockDim.x;
      const int t = i / n4, j = i - t * n4;
      const int b = b0 + t;
      tt[u] = t; jj[u] = j;
      mv[u] = (i < n_res && b < B && j < n) ? __ldg(model + (size_t)b * n + j) - __ldg(data + j) : 0.0;
    }
#pragma unroll
    for (int u = 0; u < 4; ++u)
      if (i0 + u * blockDim.x < n_res) r[(size_t)jj[u] * TBP + tt[u]] = mv[u];
  }
  // prior support and finiteness of theta (compared in the float32 theta arrives in): all threads, one flag per theta
  if (tid < TB) bad[tid] = 0;
  __syncthreads();
  for (int i = tid; i < TB * D; i += blockDim.x) {
    const int t = i / D, d = i - t * D;
    if (b0 + t < B) {
      const float v = __ldg(theta + (size_t)(b0 + t) * D + d);
      if (!isfinite(v) || (prior_kind[d] == 0 && (v < (float)p0[d] || v > (float)p1[d]))) bad[t] = 1;
    }
  }
  const int MT = (n + 7) >> 3;
  const int mtA = warp, mtB = MT - 1 - warp;              // short and long 8-row tiles of this warp
  const bool hasB = mtB >= mtA, hasA = mtA < mtB;         // the middle tile of an odd count is B alone
  const int fk = lane & 3, fr = lane >> 2;
  const int rowA = 8 * mtA + fr, rowB = 8 * mtB + fr;
  double accA[NTL][2], accB[NTL][2];
#pragma unroll
  for (int t = 0; t < NTL; ++t) { accA[t][0] = accA[t][1] = 0.0; accB[t][0] = accB[t][1] = 0.0; }
  for (int c = 0; c < n_chunks; ++c) {
    const int buf = c % NBUF;
    if (warp == 0 && c + NBUF - 1 < n_chunks) {
      const int cn = c + NBUF - 1, nb = cn % NBUF;
      if (c >= 1 && lane == 0) tc::mbar_wait(empty0 + 8 * nb, ((c - 1) / NBUF) & 1);
      __syncwarp();
      load_chunk(cn, nb);
    }
    tc::mbar_wait(full0 + 8 * buf, (c / NBUF) & 1);
    const int j0 = c * CH;
    if (hasB && j0 <= 8 * mtB + 7) {                      // warp-uniform: the chunk reaches this warp's long tile
      const double* Sb = S + (size_t)buf * CH * nsp;
      for (int k4 = 0; k4 < CH; k4 += 4) {
        const int jb = j0 + k4;
        if (jb >= n || jb > 8 * mtB + 7) break;
        const int jj = k4 + fk;
        const bool in = j0 + jj < n;                      // columns past n in the last chunk were not copied
        const double* rj = r + (size_t)(j0 + jj) * TBP + fr;
        double v[NTL];
#pragma unroll
        for (int t = 0; t < NTL; ++t) v[t] = rj[8 * t];   // rows n .. n4-1 of r are zero
        const double b_ = in ? Sb[(size_t)jj * nsp + rowB] : 0.0;     // rows up to 8 MT - 1 < nsp; past n: the stride's zero padding
#pragma unroll
        for (int t = 0; t < NTL; ++t) dmma_8x8x4_s(accB[t], b_, v[t]);
        if (hasA && jb <= 8 * mtA + 7) {                  // warp-uniform: the short tile ends early
          const double a_ = in ? Sb[(size_t)jj * nsp + rowA] : 0.0;
#pragma unroll
          for (int t = 0; t < NTL; ++t) dmma_8x8x4_s(accA[t], a_, v[t]);
        }
      }
    }
    __syncwarp();
    if (lane == 0) tc::mbar_arrive(empty0 + 8 * buf);
  }
  // sum of w^2 over this warp's rows per theta (lanes with equal fk hold the same two thetas), then over warps
#pragma unroll
  for (int t = 0; t < NTL; ++t)
#pragma unroll
    for (int e = 0; e < 2; ++e) {
      double ss = ((hasB && rowB < n) ? accB[t][e] * accB[t][e] : 0.0) + ((hasA && rowA < n) ? accA[t][e] * accA[t][e] : 0.0);
      ss += __shfl_xor_sync(0xffffffffu, ss, 4);
      ss += __shfl_xor_sync(0xffffffffu, ss, 8);
      ss += __shfl_xor_sync(0xffffffffu, ss, 16);
      if (fr == 0) part[(size_t)warp * TB + 8 * t + 2 * fk + e] = ss;
    }
  __syncthreads();
  if (tid < TB) {
    const int b = b0 + tid;
    if (b < B) {
      double chi2 = 0.0;
      for (int w = 0; w < nwarp; ++w) chi2 += part[(size_t)w * TB + tid];
      const double out = -0.5 * chi2 + log_norm;
      logL[b] = (isfinite(out) && !bad[tid]) ? out : -INFINITY;
    }
  }
}

// ---- tiled whitening: W = Linv R as a blocked triangular product ------------------------------------------
// For many thetas at once the kernel above streams the whole factor through every CTA (n^2/2 doubles per
// 8 thetas), which is what bounds it for n ~ 1000.  Here a CTA owns a 128-row block of Linv and TG*8 thetas:
// the factor crosses L2 -> shared memory once per 64 thetas.  Operands: LinvT (column j contiguous over rows)
// and the residuals transposed to [n][batch] so that both tiles of a k-step are contiguous pieces moved by
// bulk asynchronous copies through a ring of stages.  The product itself runs on the fp64 tensor cores (DMMA).
// Partial sums of w^2 per (row block, theta) are joined in a fixed order by chi2_finalize_kernel.
constexpr int CT_ROWS = 128, CT_KC = 8, CT_NBUF = 4, CT_WARPS = 8;

__global__ void residual_transpose_kernel(const double* __restrict__ model, const double* __restrict__ data, int n, int B,
                                          const int* __restrict__ n_rows_dev, size_t ldr, double* __restrict__ rt) {
  __shared__ double tile[32][33];
  pdl_wait();      // launch_pdl contract
  pdl_trigger();
  const int live = n_rows_dev ? min(B, *n_rows_dev) : B;
  const int j0 = blockIdx.x * 32, b0 = blockIdx.y * 32;
  if (b0 >= ((live + 63) & ~63)) return;
  for (int y = threadIdx.y; y < 32; y += blockDim.y) {
    const int b = b0 + y, j = j0 + threadIdx.x;
    tile[y][threadIdx.x] = (b < live && j < n) ? model[(size_t)b * n + j] - data[j] : 0.0;
  }
  __syncthreads();
  for (int y = threadIdx.y; y < 32; y += blockDim.y) {
    const int j = j0 + y, b = b0 + threadIdx.x;
    if (j < n) rt[(size_t)j * ldr + b] = tile[threadIdx.x][y];
  }
}

// D (8x8) += A (8x4, row) . B (4x8, col) on the fp64 tensor cores.  Fragments (PTX ISA, mma.m8n8k4 .f64): lane l holds
// A[l >> 2][l & 3], B[l & 3][l >> 2] and D[l >> 2][2 (l & 3) + {0, 1}].
__device__ __forceinline__ void dmma_8x8x4(double (&d)[2], double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
               : "+d"(d[0]), "+d"(d[1]) : "d"(a), "d"(b));
}

// TG = thetas per CTA / 8 (8: 64 thetas, 4: 32).  A warp owns 16 rows (two 8-row MMA tiles) and all the CTA's thetas:
// per 4 columns of the factor it loads 2 A and TG B fragments and issues 2 TG DMMAs (256 FMA each) -- an eighth of
// the instructions of the scalar formulation, which ran at half the fp64 rate for instruction overhead alone.  The
// tile rows are padded by 8 doubles so that a fragment load (4 columns x 8 rows) covers every bank exactly twice.
template <int TG>
__global__ void __launch_bounds__(CT_WARPS * 32, 2) chi2_tile_kernel(const double* __restrict__ LinvT,
                                                                     const double* __restrict__ rt, int n, int ns, int B,
                                                                     const int* __restrict__ n_rows_dev, size_t ldr,
                                                                     int n_tb, double* __restrict__ part) {
  constexpr int TBLK = 8 * TG;                            // thetas per CTA
  constexpr int LDL = CT_ROWS + 8, LDR = TBLK + 8;        // padded tile rows (stride = 8 mod 16 doubles)
  pdl_wait();      // launch_pdl contract
  pdl_trigger();
  const int live = n_rows_dev ? min(B, *n_rows_dev) : B;
  const int n_rb = (n + CT_ROWS - 1) / CT_ROWS;
  const int rb = n_rb - 1 - blockIdx.x / n_tb;            // longest row blocks first
  const int b0 = (blockIdx.x % n_tb) * TBLK;
  if (b0 >= live) return;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  typedef double LTile[CT_KC][LDL];
  typedef double RTile[CT_KC][LDR];
  LTile* Ls = reinterpret_cast<LTile*>(smem_raw);                                   // [CT_NBUF]
  RTile* Rs = reinterpret_cast<RTile*>(smem_raw + sizeof(LTile) * CT_NBUF);         // [CT_NBUF]
  unsigned long long* bars = reinterpret_cast<unsigned long long*>(smem_raw + (sizeof(LTile) + sizeof(RTile)) * CT_NBUF);
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int i0 = rb * CT_ROWS;                            // ns: row stride of LinvT (multiple of 8)
  const int rows = min(CT_ROWS, ns - i0);                 // even: ns and i0 are
  const int K = min(i0 + CT_ROWS, n);                     // columns 0 .. K-1 reach this row block
  const int n_steps = (K + CT_KC - 1) / CT_KC;
  const uint32_t full0 = tc::smem_u32(bars), empty0 = full0 + 8 * CT_NBUF;
  // one k-step = 2 CT_KC small copies: issued by the lanes of warp 0 in parallel (a single thread issuing them one
  // after the other put ~1000 clk per step on the critical path of its warp)
  auto load_step = [&](int s, int buf) {                 // whole warp 0
    const int j0 = s * CT_KC, jn = min(CT_KC, K - j0);
    if (lane == 0) tc::mbar_arrive_expect_tx(full0 + 8 * buf, (uint32_t)jn * (uint32_t)(rows * 8 + TBLK * 8));
    __syncwarp();
    if (lane < jn)
      tc::bulk_load(tc::smem_u32(&Ls[buf][lane][0]), LinvT + (size_t)(j0 + lane) * ns + i0, (uint32_t)rows * 8u, full0 + 8 * buf);
    else if (lane >= 16 && lane - 16 < jn)
      tc::bulk_load(tc::smem_u32(&Rs[buf][lane - 16][0]), rt + (size_t)(j0 + lane - 16) * ldr + b0, TBLK * 8u, full0 + 8 * buf);
  };
  static_assert(CT_KC <= 16 && CT_KC % 4 == 0 && CT_ROWS == 16 * CT_WARPS, "one lane per copy; whole MMA k-steps; 16 rows per warp");
  if (tid == 0) {
    for (int b = 0; b < CT_NBUF; ++b) { tc::mbar_init(full0 + 8 * b, 1); tc::mbar_init(empty0 + 8 * b, CT_WARPS); }
    tc::fence_barrier_init();
  }
  __syncthreads();
  if (warp == 0)
    for (int s = 0; s < CT_NBUF - 1 && s < n_steps; ++s) load_step(s, s);
  double acc[2][TG][2];
#pragma unroll
  for (int m = 0; m < 2; ++m)
#pragma unroll
    for (int t = 0; t < TG; ++t) { acc[m][t][0] = 0.0; acc[m][t][1] = 0.0; }
  const int fk = lane & 3, fr = lane >> 2;               // fragment coordinates of this lane
  for (int s = 0; s < n_steps; ++s) {
    const int buf = s % CT_NBUF;
    if (warp == 0 && s + CT_NBUF - 1 < n_steps) {
      const int sn = s + CT_NBUF - 1, nb = sn % CT_NBUF;
      if (s >= 1 && lane == 0) tc::mbar_wait(empty0 + 8 * nb, ((s - 1) / CT_NBUF) & 1);
      __syncwarp();
      load_step(sn, nb);
    }
    tc::mbar_wait(full0 + 8 * buf, (s / CT_NBUF) & 1);
    const int jn = min(CT_KC, K - s * CT_KC);
#pragma unroll
    for (int ks = 0; ks < CT_KC / 4; ++ks) {
      const int jj = 4 * ks + fk;
      const bool in = jj < jn;                            // columns past K in the last step were not copied
      double a[2], v[TG];
#pragma unroll
      for (int m = 0; m < 2; ++m) a[m] = in ? Ls[buf][jj][16 * warp + 8 * m + fr] : 0.0;
#pragma unroll
      for (int t = 0; t < TG; ++t) v[t] = in ? Rs[buf][jj][8 * t + fr] : 0.0;
#pragma unroll
      for (int m = 0; m < 2; ++m)
#pragma unroll
        for (int t = 0; t < TG; ++t) dmma_8x8x4(acc[m][t], a[m], v[t]);
    }
    __syncwarp();
    if (lane == 0) tc::mbar_arrive(empty0 + 8 * buf);
  }
  // sum of w^2 over this warp's 16 rows for each theta (lanes with equal fk hold the same two thetas of a tile),
  // then over the 8 warps through shared memory in a fixed order
  __syncthreads();                                       // every warp is done with the ring: reuse it
  double* red = reinterpret_cast<double*>(smem_raw);     // [CT_WARPS][TBLK]
#pragma unroll
  for (int t = 0; t < TG; ++t)
#pragma unroll
    for (int e = 0; e < 2; ++e) {
      double ss = 0.0;
#pragma unroll
      for (int m = 0; m < 2; ++m) {
        const bool ok = i0 + 16 * warp + 8 * m + fr < n;  // rows past n hold stale tiles
        ss += ok ? acc[m][t][e] * acc[m][t][e] : 0.0;
      }
      ss += __shfl_xor_sync(0xffffffffu, ss, 4);
      ss += __shfl_xor_sync(0xffffffffu, ss, 8);
      ss += __shfl_xor_sync(0xffffffffu, ss, 16);
      if (fr == 0) red[warp * TBLK + 8 * t + 2 * fk + e] = ss;
    }
  __syncthreads();
  if (tid < TBLK) {
    double ss = 0.0;
#pragma unroll
    for (int w = 0; w < CT_WARPS; ++w) ss += red[w * TBLK + tid];
    part[(size_t)rb * ldr + b0 + tid] = ss;
  }
}

__global__ void chi2_finalize_kernel(const double* __restrict__ part, int n_rb, size_t ldr, int B,
                                     const int* __restrict__ n_rows_dev, const float* __restrict__ theta, int D,
                                     const int* __restrict__ prior_kind, const double* __restrict__ p0,
                                     const double* __restrict__ p1, double log_norm, double* __restrict__ logL) {
  pdl_wait();      // launch_pdl contract
  pdl_trigger();
  if (n_rows_dev) B = min(B, *n_rows_dev);
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= B) return;
  double chi2 = 0.0;
  for (int rb = 0; rb < n_rb; ++rb) chi2 += part[(size_t)rb * ldr + b];
  const double out = -0.5 * chi2 + log_norm;
  bool ok = isfinite(out);
  for (int d = 0; d < D; ++d) {
    const float v = theta[(size_t)b * D + d];
    if (!isfinite(v)) ok = false;
    if (prior_kind[d] == 0 && (v < (float)p0[d] || v > (float)p1[d])) ok = false;
  }
  logL[b] = ok ? out : -INFINITY;
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
  // n >= 512: tiled path (transposed residuals, blocked triangular product on the fp64 tensor cores, fixed-order
  // join).  Measured at B = 4096: n = 1100 0.25 vs 1.03 ms, n = 613 0.12 vs 0.25 ms; n = 300 0.073 vs 0.064 ms
  // (three launches and short k loops), so small problems stay on the single streaming kernel below.
  const bool tiled = (ctx->flags & NSGPU_CHI2_TILED) ? true : ((ctx->flags & NSGPU_CHI2_STREAMED) ? false : n >= 512);
  if (ctx->resid_t && tiled) {
    const size_t ldr = ((size_t)ctx->max_batch + 63) & ~(size_t)63;
    const int n_rb = (n + CT_ROWS - 1) / CT_ROWS;
    StageTimer tm(ctx, 5, st);
    dim3 tg((n + 31) / 32, (((B + 63) & ~63) + 31) / 32);
    NSGPU_CUDA(launch_pdl(ctx, residual_transpose_kernel, tg, dim3(32, 8), 0, st, ctx->model, ctx->data, n, B, n_rows_dev, ldr, ctx->resid_t));
    NSGPU_LAUNCH_CHECK();
    // 64 thetas per CTA; 32 when that would leave SMs idle (the nested-sampling rounds)
    const bool small = (size_t)n_rb * ((B + 63) / 64) < (size_t)ctx->sm_count;
    const int tblk = small ? 32 : 64, n_tb = (B + tblk - 1) / tblk;
    const size_t smem_t = (size_t)CT_NBUF * CT_KC * (CT_ROWS + 8 + tblk + 8) * sizeof(double) + 2 * CT_NBUF * 8;
    NSGPU_CUDA(nsgpu_ensure_smem(ctx, chi2_tile_kernel<8>, smem_t));
    NSGPU_CUDA(nsgpu_ensure_smem(ctx, chi2_tile_kernel<4>, smem_t));
    if (small) NSGPU_CUDA(launch_pdl(ctx, chi2_tile_kernel<4>, dim3(n_rb * n_tb), dim3(CT_WARPS * 32), smem_t, st, ctx->Linv, ctx->resid_t, n, ctx->linv_ld, B, n_rows_dev, ldr, n_tb, ctx->chi2_part));
    else NSGPU_CUDA(launch_pdl(ctx, chi2_tile_kernel<8>, dim3(n_rb * n_tb), dim3(CT_WARPS * 32), smem_t, st, ctx->Linv, ctx->resid_t, n, ctx->linv_ld, B, n_rows_dev, ldr, n_tb, ctx->chi2_part));
    NSGPU_LAUNCH_CHECK();
    NSGPU_CUDA(launch_pdl(ctx, chi2_finalize_kernel, dim3((B + 127) / 128), dim3(128), 0, st, ctx->chi2_part, n_rb, ldr, B, n_rows_dev, theta, ctx->D,
                          ctx->prior_kind, ctx->prior_p0, ctx->prior_p1, ctx->log_norm, logL));
    NSGPU_LAUNCH_CHECK();
    return NSGPU_OK;
  }
  if ((ctx->flags & NSGPU_CHI2_STREAMED) == 0 && n < 512 && n >= 8) {
    // tensor-core streaming kernel: 32 thetas per CTA, fewer when the grid would not cover the SMs
    int ntl = 4;
    while (ntl > 1 && (B + 8 * ntl - 1) / (8 * ntl) < ctx->sm_count / 2) ntl >>= 1;
    const int MT = (n + 7) / 8, warps = (MT + 1) / 2, threads = 32 * warps;
    const int nsp = ctx->linv_ld;                                             // 8 mod 16 doubles, >= n rounded up to 8
    const int n4 = (n + 3) & ~3, TBP = 8 * ntl + 8;
    const size_t smem_fixed = ((size_t)n4 * TBP + (size_t)warps * 8 * ntl + 16 + 16) * sizeof(double);   // + up to 2 x 8 mbarriers + 8 ntl prior flags
    int CH = (int)((100 * 1024 / 4) / ((size_t)nsp * 8));
    CH = std::max(4, std::min(16, CH & ~3));
    // small batches are bound by the latency of the chunk ring, not by arithmetic: eight chunks in flight when
    // the (then small) residual block leaves room
    const int nbuf = (ntl <= 2 && smem_fixed + 8 * (size_t)CH * nsp * sizeof(double) <= 200 * 1024) ? 8 : 4;
    const size_t smem = smem_fixed + (size_t)nbuf * CH * nsp * sizeof(double);
    if (smem <= 220 * 1024) {
      StageTimer tm(ctx, 5, st);
      const int grid = (B + 8 * ntl - 1) / (8 * ntl);
#define NSGPU_CHI2_MMA(NTL_, MAXT_, NBUF_)                                                                            \
  do {                                                                                                                \
    NSGPU_CUDA(nsgpu_ensure_smem(ctx, chi2_mma_kernel<NTL_, MAXT_, NBUF_>, 220 * 1024));                               \
    NSGPU_CUDA(launch_pdl(ctx, chi2_mma_kernel<NTL_, MAXT_, NBUF_>, dim3(grid), dim3(threads), smem, st, ctx->model, ctx->data, ctx->Linv, \
                          n, B, CH, nsp, n_rows_dev, theta, ctx->D, ctx->prior_kind, ctx->prior_p0, ctx->prior_p1,     \
                          ctx->log_norm, logL));                                                                        \
  } while (0)
#define NSGPU_CHI2_MMA_T(MAXT_)                                                                                       \
  do {                                                                                                                \
    if (ntl == 4) NSGPU_CHI2_MMA(4, MAXT_, 4);                                                                         \
    else if (ntl == 2 && nbuf == 8) NSGPU_CHI2_MMA(2, MAXT_, 8);                                                       \
    else if (ntl == 2) NSGPU_CHI2_MMA(2, MAXT_, 4);                                                                    \
    else if (nbuf == 8) NSGPU_CHI2_MMA(1, MAXT_, 8);                                                                   \
    else NSGPU_CHI2_MMA(1, MAXT_, 4);                                                                                  \
  } while (0)
      if (threads <= 640) NSGPU_CHI2_MMA_T(640); else NSGPU_CHI2_MMA_T(1024);
#undef NSGPU_CHI2_MMA_T
#undef NSGPU_CHI2_MMA
      NSGPU_LAUNCH_CHECK();
      return NSGPU_OK;
    }
  }
  const int RT = (((n + 1) / 2 + 31) / 32) * 32;        // row-pair threads, whole warps
  if (RT > 1024) { ctx->err = "chi2: n_data > 2048 not supported"; return NSGPU_ESHAPE; }
  // G thread groups per CTA, TG thetas per thread, TB = G TG thetas per CTA.  Large batches: TG = 8 (each
  // factor element read from shared memory feeds 8 FMAs).  Small batches (the nested-sampling rounds):
  // fewer thetas per CTA so that the grid still covers the SMs.
  const int groups = RT <= 160 ? 4 : (RT <= 320 ? 2 : 1);
  int tg = 8;
  while (tg > 2 && groups > 1 && (B + groups * tg - 1) / (groups * tg) < ctx->sm_count / 2) tg >>= 1;
  const int TBv = groups * tg;
  // chunk of CH factor columns per buffer: four buffers within ~100 KB, CH even
  const size_t ns = (size_t)ctx->linv_ld;
  const size_t smem_fixed = ((size_t)n * TBv + 32 * TBv + 8) * sizeof(double);
  int CH = (int)((100 * 1024 / 4) / (ns * 8));
  CH = std::max(2, std::min(16, CH & ~1));
  if (CH < 4 && smem_fixed + 4 * 4 * ns * sizeof(double) <= 216 * 1024) CH = 4;   // large n: use what is left
  const size_t smem = smem_fixed + 4 * (size_t)CH * ns * sizeof(double);
  if (smem > 220 * 1024) { ctx->err = "chi2: tiles exceed shared memory"; return NSGPU_ESHAPE; }
  StageTimer tm(ctx, 5, st);
  const int grid = (B + TBv - 1) / TBv, threads = groups * RT;
#define NSGPU_CHI2_ARGS ctx->model, ctx->data, ctx->Linv, n, (int)ns, B, RT, CH, n_rows_dev, theta, ctx->D, ctx->prior_kind, ctx->prior_p0, ctx->prior_p1, ctx->log_norm, logL
#define NSGPU_CHI2_LAUNCH(TB_, TG_, MAXT_)                                                                        \
  do {                                                                                                            \
    NSGPU_CUDA(nsgpu_ensure_smem(ctx, chi2_kernel<TB_, TG_, MAXT_>, 220 * 1024));                                   \
    chi2_kernel<TB_, TG_, MAXT_><<<grid, threads, smem, st>>>(NSGPU_CHI2_ARGS);                                   \
  } while (0)
  if (groups == 4 && tg == 8) NSGPU_CHI2_LAUNCH(32, 8, 640);
  else if (groups == 4 && tg == 4) NSGPU_CHI2_LAUNCH(16, 4, 640);
  else if (groups == 4) NSGPU_CHI2_LAUNCH(8, 2, 640);
  else if (groups == 2 && tg == 8) NSGPU_CHI2_LAUNCH(16, 8, 640);
  else if (groups == 2 && tg == 4) NSGPU_CHI2_LAUNCH(8, 4, 640);
  else if (groups == 2) NSGPU_CHI2_LAUNCH(4, 2, 640);
  else if (threads <= 640) NSGPU_CHI2_LAUNCH(8, 8, 640);
  else NSGPU_CHI2_LAUNCH(8, 8, 1024);
#undef NSGPU_CHI2_LAUNCH
#undef NSGPU_CHI2_ARGS
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
