// theory.cu -- from emulated log-spectra to the model vector (steps a5-a9).
//
// shear_project : per theta, background (a6), windows (a7), z/k interpolation of the emulated
//                 log10 P(k,z) table staged in shared memory and the extended-Limber sums reduced over
//                 the chi-quadrature nodes with warp shuffles (a5, a8)  [P:L330-353 eqs. A1-A4; P:L359]
// cmb_bin       : 10^y / linear, / A_cal^2, CSR binning (a9)            [BJ cfg 1; readings C1-C3]
// copy_model    : identity / emulator-only theories (BJ cfg 0)
//
// HBM-bound stages: the only large read is the spectrum table written by the emulator (84 KB per
// theta for c2/c3a).  All arithmetic here is fp64 -- it is ~0.15 MFLOP per theta against 100 MFLOP in
// the emulator, and the absolute log L tolerance leaves no room for fp32 round-off downstream of
// the network.  The oracle sums the four terms of eq. A1 separately; this kernel
// projects the factored form (W^gamma + W^I)_i (W^gamma + W^I)_j once.
#include "internal.cuh"

namespace {

constexpr double C_OVER_H0 = 2997.92458;   // Mpc/h
constexpr double C1_RHOCR = 0.0138768;     // reading S12

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// In-place exclusive prefix sum of arr[0..n) (or suffix sum when `reverse`) by the whole block.
// wsum: shared scratch of 33 doubles.
__device__ void block_scan_exclusive(double* arr, int n, bool reverse, double* wsum) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
  double carry = 0.0;
  for (int base = 0; base < n; base += blockDim.x) {
    int i = base + threadIdx.x;
    int idx = reverse ? n - 1 - i : i;
    double v = (i < n) ? arr[idx] : 0.0;
    double inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      double t = __shfl_up_sync(0xffffffffu, inc, o);
      if (lane >= o) inc += t;
    }
    if (lane == 31) wsum[warp] = inc;
    __syncthreads();
    if (warp == 0) {
      double w = (lane < nwarp) ? wsum[lane] : 0.0;
      double winc = w;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        double t = __shfl_up_sync(0xffffffffu, winc, o);
        if (lane >= o) winc += t;
      }
      if (lane < nwarp) wsum[lane] = winc - w;      // exclusive warp offsets
      if (lane == nwarp - 1) wsum[32] = winc;       // chunk total
    }
    __syncthreads();
    if (i < n) arr[idx] = carry + wsum[warp] + inc - v;
    carry += wsum[32];
    __syncthreads();
  }
}

struct ShearArgs {
  int n_z_emu, n_chi, n_k, n_ell, n_tomo, n_tap;
  double k_min, k_max, lk0, dlk, da, nz_sigma;
  const double *a_q, *z_q, *tap_w, *ell, *nz_mean;
  const int* tap_start;
  int idx_omega_b, idx_omega_cdm, idx_h, idx_w0, idx_wa, idx_eta0, idx_dz, idx_ia, idx_m;
};

__global__ void __launch_bounds__(256) shear_project_kernel(const float* __restrict__ theta, int D,
                                                            const int* __restrict__ n_rows_dev,
                                                            const float* __restrict__ spec, ShearArgs A,
                                                            double* __restrict__ model, int n_data) {
  const int b = blockIdx.x;
  if (n_rows_dev && b >= *n_rows_dev) return;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int nq = A.n_chi, nt = A.n_tomo;
  double* chi = reinterpret_cast<double*>(smem_raw);   // [nq]
  double* Eq = chi + nq;                               // [nq]
  double* Dq = Eq + nq;                                // [nq]
  double* gq = Dq + nq;                                // [nq]   dchi / chi^2
  double* s0 = gq + nq;                                // [nq]   scratch (suffix sum A)
  double* s1 = s0 + nq;                                // [nq]   scratch (suffix sum B)
  double* Wt = s1 + nq;                                // [nt][nq] total window
  double* Pg = Wt + (size_t)nt * nq;                   // [n_ell][nq]
  double* wsum = Pg + (size_t)A.n_ell * nq;            // [33]
  const size_t n_dbl = ((size_t)nq * (6 + nt + A.n_ell) + 34 + 1) & ~(size_t)1;   // keep the table 16-byte aligned
  float* table = reinterpret_cast<float*>(chi + n_dbl);  // [n_z_emu][n_k]

  const float* th = theta + (size_t)b * D;
  // stage this theta's log10 P table (the kernel's only large HBM read)
  {
    const float* src = spec + (size_t)b * A.n_z_emu * A.n_k;
    const int n = A.n_z_emu * A.n_k;
    if ((n & 3) == 0 && ((reinterpret_cast<uintptr_t>(src) & 15) == 0)) {
      const float4* s4 = reinterpret_cast<const float4*>(src);
      float4* d4 = reinterpret_cast<float4*>(table);
      for (int i = threadIdx.x; i < n / 4; i += blockDim.x) d4[i] = __ldg(s4 + i);
    } else {
      for (int i = threadIdx.x; i < n; i += blockDim.x) table[i] = __ldg(src + i);
    }
  }
  const double ob = th[A.idx_omega_b], oc = th[A.idx_omega_cdm], h = th[A.idx_h];
  const double Om = (ob + oc) / (h * h);
  const double w0 = A.idx_w0 >= 0 ? (double)th[A.idx_w0] : -1.0;
  const double wa = A.idx_wa >= 0 ? (double)th[A.idx_wa] : 0.0;
  const double eta0 = A.idx_eta0 >= 0 ? (double)th[A.idx_eta0] : 0.7;
  const double gam = 0.55 + 0.05 * (1.0 + w0 + 0.5 * wa);

  // a6: E_q, f_q da -> chi (exclusive scan + half cell), growth exponent -> ln D
  for (int q = threadIdx.x; q < nq; q += blockDim.x) {
    const double a = A.a_q[q], z = A.z_q[q];
    const double E2 = Om * (1.0 + z) * (1.0 + z) * (1.0 + z) +
                      (1.0 - Om) * pow(1.0 + z, 3.0 * (1.0 + w0 + wa)) * exp(-3.0 * wa * z / (1.0 + z));
    const double E = sqrt(E2);
    Eq[q] = E;
    const double f = 1.0 / (a * a * E);
    gq[q] = f * A.da;                                         // f_q da
    const double Om_a = Om / (a * a * a) / E2;
    s1[q] = pow(Om_a, gam) * A.da / a;                        // growth integrand
    chi[q] = gq[q];
    Dq[q] = s1[q];
  }
  __syncthreads();
  block_scan_exclusive(chi, nq, false, wsum);
  block_scan_exclusive(Dq, nq, false, wsum);
  for (int q = threadIdx.x; q < nq; q += blockDim.x) {
    const double c = C_OVER_H0 * (chi[q] + 0.5 * gq[q]);
    chi[q] = c;
    Dq[q] = exp(-(Dq[q] + 0.5 * s1[q]));
    gq[q] = C_OVER_H0 * gq[q] / (c * c);                      // dchi_q / chi_q^2
  }
  __syncthreads();

  // a7: per tomographic bin, n_i(z - dz_i), W^gamma by two suffix sums (A - chi B), W^I, total
  const double norm = 1.0 / (A.nz_sigma * 2.5066282746310002);   // 1/(sigma sqrt(2 pi))
  for (int i = 0; i < nt; ++i) {
    const double mu = A.nz_mean[i] + (double)th[A.idx_dz + i];
    const double A0 = th[A.idx_ia + 3 * i], A1 = th[A.idx_ia + 3 * i + 1], A2 = th[A.idx_ia + 3 * i + 2];
    for (int q = threadIdx.x; q < nq; q += blockDim.x) {
      const double z = A.z_q[q], a = A.a_q[q];
      const double u = (z - mu) / A.nz_sigma;
      const double nz = exp(-0.5 * u * u) * norm;
      const double w = nz * A.da / (a * a);                   // n_i(z_q) dz_q
      s0[q] = w;
      s1[q] = w / chi[q];
      const double x = (1.0 + z) / 1.62 - 1.0;
      const double Aia = A0 + A1 * x + A2 * x * x;
      Wt[(size_t)i * nq + q] = -Aia * C1_RHOCR * Om / Dq[q] * nz * Eq[q] / C_OVER_H0;   // W^I (eq. A4)
    }
    __syncthreads();
    block_scan_exclusive(s0, nq, true, wsum);
    block_scan_exclusive(s1, nq, true, wsum);
    for (int q = threadIdx.x; q < nq; q += blockDim.x) {
      const double wg = 1.5 * Om / (C_OVER_H0 * C_OVER_H0) * (1.0 + A.z_q[q]) * chi[q] * (s0[q] - chi[q] * s1[q]);
      Wt[(size_t)i * nq + q] += wg;                           // + W^gamma (eq. A3)
    }
    __syncthreads();
  }

  // a5 + a8 (lookup): P(k = (ell+1/2)/chi_q, z_q) g_q for every (ell, q)
  const int n_lookup = A.n_ell * nq;
  for (int it = threadIdx.x; it < n_lookup; it += blockDim.x) {
    const int bl = it / nq, q = it - bl * nq;
    const double k = (A.ell[bl] + 0.5) / chi[q];
    double P = 0.0;
    if (k >= A.k_min && k <= A.k_max) {
      const double x = log10(k);
      int j = (int)floor((x - A.lk0) / A.dlk);
      j = min(max(j, 0), A.n_k - 2);
      const double s = (x - (A.lk0 + j * A.dlk)) / A.dlk;
      const int m0 = A.tap_start[q];
      const double* tw = A.tap_w + (size_t)q * A.n_tap;
      double lo = 0.0, hi = 0.0;
      for (int t = 0; t < A.n_tap; ++t) {
        const float* row = table + (size_t)(m0 + t) * A.n_k + j;
        lo += tw[t] * (double)row[0];
        hi += tw[t] * (double)row[1];
      }
      double y = (1.0 - s) * lo + s * hi;
      y -= (eta0 - 0.7) * 0.1 * k * k / (k * k + 1.0);
      P = exp10(y);
    }
    Pg[it] = P * gq[q];
  }
  __syncthreads();

  // a8 (sum): C_ij(ell) = sum_q Wt_i Wt_j Pg; one warp per output, lanes stride q, shuffle reduce
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nwarp = blockDim.x >> 5;
  const int n_pairs = nt * (nt + 1) / 2;
  for (int o = warp; o < n_pairs * A.n_ell; o += nwarp) {
    const int p = o / A.n_ell, bl = o - p * A.n_ell;
    int i = 0, rem = p;                                        // pair p -> (i <= j), row-major upper
    while (rem >= nt - i) { rem -= nt - i; ++i; }
    const int j = i + rem;
    const double* wi = Wt + (size_t)i * nq;
    const double* wj = Wt + (size_t)j * nq;
    const double* pg = Pg + (size_t)bl * nq;
    double acc = 0.0;
    for (int q = lane; q < nq; q += 32) acc += wi[q] * wj[q] * pg[q];
    acc = warp_sum(acc);
    if (lane == 0) {
      const double lf = log(A.ell[bl] / 550.0) / 3.4011973816621555;   // ln(ell/550)/ln 30
      const double mi = (double)th[A.idx_m + 2 * i] + (double)th[A.idx_m + 2 * i + 1] * lf;
      const double mj = (double)th[A.idx_m + 2 * j] + (double)th[A.idx_m + 2 * j + 1] * lf;
      model[(size_t)b * n_data + o] = (1.0 + mi) * (1.0 + mj) * acc;
    }
  }
}

// a9: one CTA per theta.  Stage the n_emu spectra in shared memory (coalesced, 10^y applied once per
// multipole, / A_cal^2), then one thread per bin walks its CSR row.
__global__ void __launch_bounds__(256) cmb_bin_kernel(const float* __restrict__ theta, int D,
                                                      const int* __restrict__ n_rows_dev,
                                                      const float* __restrict__ spec, int n_emu, int n_out,
                                                      size_t emu_stride, unsigned exp10_mask, int cal_index,
                                                      const int* __restrict__ bin_ptr,
                                                      const int* __restrict__ bin_col,
                                                      const float* __restrict__ bin_val, int n_data,
                                                      double* __restrict__ model) {
  const int b = blockIdx.x;
  if (n_rows_dev && b >= *n_rows_dev) return;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  double* s = reinterpret_cast<double*>(smem_raw);   // [n_emu * n_out]
  const double acal = theta[(size_t)b * D + cal_index];
  const double inv = 1.0 / (acal * acal);
  for (int e = 0; e < n_emu; ++e) {
    const float* src = spec + e * emu_stride + (size_t)b * n_out;
    const bool ex = (exp10_mask >> e) & 1u;
    for (int i = threadIdx.x; i < n_out; i += blockDim.x) {
      const double y = (double)__ldg(src + i);
      s[e * n_out + i] = (ex ? exp10(y) : y) * inv;
    }
  }
  __syncthreads();
  for (int r = threadIdx.x; r < n_data; r += blockDim.x) {
    double acc = 0.0;
    for (int e = bin_ptr[r]; e < bin_ptr[r + 1]; ++e) acc += (double)bin_val[e] * s[bin_col[e]];
    model[(size_t)b * n_data + r] = acc;
  }
}

// kind 0: model = theta; kind 1: model = spectrum of emulator 0 (10^y where out_kind = 1)
__global__ void copy_model_kernel(const float* __restrict__ src, int n, int B, const int* __restrict__ n_rows_dev,
                                  int apply_exp10, double* __restrict__ model) {
  if (n_rows_dev) B = min(B, *n_rows_dev);
  const size_t total = (size_t)B * n;
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
    const double y = (double)src[i];
    model[i] = apply_exp10 ? exp10(y) : y;
  }
}

}  // namespace

static size_t shear_smem_bytes(const ShearDev& S) {
  size_t d = ((size_t)S.n_chi * (6 + S.n_tomo + S.n_ell) + 34 + 1) & ~(size_t)1;
  return d * sizeof(double) + (size_t)S.n_z_emu * S.n_k * sizeof(float) + 16;
}

nsgpu_status shear_project(nsgpu_ctx* ctx, const float* theta, int B, const int* n_rows_dev, cudaStream_t st) {
  if (B == 0) return NSGPU_OK;
  const ShearDev& S = ctx->sh;
  ShearArgs A;
  A.n_z_emu = S.n_z_emu; A.n_chi = S.n_chi; A.n_k = S.n_k; A.n_ell = S.n_ell; A.n_tomo = S.n_tomo; A.n_tap = S.n_tap;
  A.k_min = S.k_min; A.k_max = S.k_max; A.lk0 = S.lk0; A.dlk = S.dlk; A.da = S.da; A.nz_sigma = S.nz_sigma;
  A.a_q = S.a_q; A.z_q = S.z_q; A.tap_w = S.tap_w; A.ell = S.ell; A.nz_mean = S.nz_mean; A.tap_start = S.tap_start;
  A.idx_omega_b = S.idx_omega_b; A.idx_omega_cdm = S.idx_omega_cdm; A.idx_h = S.idx_h; A.idx_w0 = S.idx_w0;
  A.idx_wa = S.idx_wa; A.idx_eta0 = S.idx_eta0; A.idx_dz = S.idx_dz; A.idx_ia = S.idx_ia; A.idx_m = S.idx_m;
  const size_t smem = shear_smem_bytes(S);
  static size_t configured = 0;
  if (smem > configured) {
    NSGPU_CUDA(cudaFuncSetAttribute(shear_project_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    configured = smem;
  }
  StageTimer tm(ctx, 3, st);
  shear_project_kernel<<<B, 256, smem, st>>>(theta, ctx->D, n_rows_dev, ctx->spec, A, ctx->model, ctx->n_data);
  NSGPU_LAUNCH_CHECK();
  return NSGPU_OK;
}

nsgpu_status cmb_bin(nsgpu_ctx* ctx, const float* theta, int B, const int* n_rows_dev, cudaStream_t st) {
  if (B == 0) return NSGPU_OK;
  const int n_out = ctx->emu[0].n_out;
  unsigned mask = 0;
  for (int e = 0; e < ctx->n_emu; ++e) mask |= (ctx->emu[e].out_kind == 1 ? 1u : 0u) << e;
  const size_t smem = (size_t)ctx->n_emu * n_out * sizeof(double);
  static size_t configured = 0;
  if (smem > configured) {
    NSGPU_CUDA(cudaFuncSetAttribute(cmb_bin_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    configured = smem;
  }
  const size_t emu_stride = (size_t)ctx->max_batch * ctx->rows_per_theta * n_out;
  StageTimer tm(ctx, 4, st);
  cmb_bin_kernel<<<B, 256, smem, st>>>(theta, ctx->D, n_rows_dev, ctx->spec, ctx->n_emu, n_out, emu_stride, mask,
                                       ctx->cal_index, ctx->bin_ptr, ctx->bin_col, ctx->bin_val, ctx->n_data,
                                       ctx->model);
  NSGPU_LAUNCH_CHECK();
  return NSGPU_OK;
}

nsgpu_status copy_model(nsgpu_ctx* ctx, const float* theta, int B, const int* n_rows_dev, cudaStream_t st) {
  if (B == 0) return NSGPU_OK;
  const bool ident = ctx->kind == 0;
  const float* src = ident ? theta : ctx->spec;
  const int n = ctx->n_data;
  const int ex = (!ident && ctx->emu[0].out_kind == 1) ? 1 : 0;
  int blocks = (int)std::min<size_t>(((size_t)B * n + 255) / 256, 148 * 8);
  StageTimer tm(ctx, 7, st);
  copy_model_kernel<<<blocks, 256, 0, st>>>(src, n, B, n_rows_dev, ex, ctx->model);
  NSGPU_LAUNCH_CHECK();
  return NSGPU_OK;
}
