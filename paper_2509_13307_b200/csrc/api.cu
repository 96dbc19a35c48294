// api.cu -- context life cycle and the likelihood entry points of include/nsgpu.h.
#include <math.h>
#include <string.h>

#include <algorithm>
#include <new>

#include "internal.cuh"

#include <mutex>

static thread_local std::string g_create_error;

cudaError_t nsgpu_raise_smem_limit(int device, const void* fn, size_t bytes) {
  static std::mutex mu;
  static std::map<std::pair<int, const void*>, size_t> limit;   // (device, kernel) -> bytes opted in so far
  std::lock_guard<std::mutex> lock(mu);
  size_t& cur = limit[std::make_pair(device, fn)];
  if (bytes <= cur) return cudaSuccess;
  const cudaError_t e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
  if (e == cudaSuccess) cur = bytes;
  return e;
}

namespace {

template <class T>
cudaError_t upload(T** dst, const T* src, size_t n) {
  *dst = nullptr;
  if (n == 0) return cudaSuccess;
  cudaError_t e = cudaMalloc((void**)dst, n * sizeof(T));
  if (e != cudaSuccess) return e;
  return cudaMemcpy(*dst, src, n * sizeof(T), cudaMemcpyHostToDevice);
}

// Cubic not-a-knot spline operator: S[e][m] = value at xe[e] of the spline through the unit data e_m
// on nodes x[0..n).  Dense Gaussian elimination with partial pivoting for the second derivatives.
void spline_matrix(const std::vector<double>& x, const std::vector<double>& xe, std::vector<double>& S) {
  const int n = (int)x.size(), ne = (int)xe.size();
  std::vector<double> h(n - 1);
  for (int i = 0; i + 1 < n; ++i) h[i] = x[i + 1] - x[i];
  // A M = R Y  with Y = identity: solve for M as an n x n matrix (column m = second derivs for e_m)
  std::vector<double> A((size_t)n * n, 0.0), R((size_t)n * n, 0.0);
  A[0 * n + 0] = h[1]; A[0 * n + 1] = -(h[0] + h[1]); A[0 * n + 2] = h[0];
  A[(size_t)(n - 1) * n + n - 3] = h[n - 2];
  A[(size_t)(n - 1) * n + n - 2] = -(h[n - 3] + h[n - 2]);
  A[(size_t)(n - 1) * n + n - 1] = h[n - 3];
  for (int i = 1; i + 1 < n; ++i) {
    A[(size_t)i * n + i - 1] = h[i - 1];
    A[(size_t)i * n + i] = 2.0 * (h[i - 1] + h[i]);
    A[(size_t)i * n + i + 1] = h[i];
    R[(size_t)i * n + i - 1] += 6.0 / h[i - 1];
    R[(size_t)i * n + i] += -6.0 / h[i - 1] - 6.0 / h[i];
    R[(size_t)i * n + i + 1] += 6.0 / h[i];
  }
  for (int c = 0; c < n; ++c) {
    int piv = c;
    for (int r = c + 1; r < n; ++r)
      if (fabs(A[(size_t)r * n + c]) > fabs(A[(size_t)piv * n + c])) piv = r;
    if (piv != c)
      for (int k = 0; k < n; ++k) {
        std::swap(A[(size_t)c * n + k], A[(size_t)piv * n + k]);
        std::swap(R[(size_t)c * n + k], R[(size_t)piv * n + k]);
      }
    for (int r = c + 1; r < n; ++r) {
      const double f = A[(size_t)r * n + c] / A[(size_t)c * n + c];
      if (f == 0.0) continue;
      for (int k = c; k < n; ++k) A[(size_t)r * n + k] -= f * A[(size_t)c * n + k];
      for (int k = 0; k < n; ++k) R[(size_t)r * n + k] -= f * R[(size_t)c * n + k];
    }
  }
  std::vector<double> M((size_t)n * n);
  for (int r = n - 1; r >= 0; --r)
    for (int k = 0; k < n; ++k) {
      double s = R[(size_t)r * n + k];
      for (int c = r + 1; c < n; ++c) s -= A[(size_t)r * n + c] * M[(size_t)c * n + k];
      M[(size_t)r * n + k] = s / A[(size_t)r * n + r];
    }
  S.assign((size_t)ne * n, 0.0);
  for (int e = 0; e < ne; ++e) {
    int i = 0;
    while (i < n - 2 && xe[e] >= x[i + 1]) ++i;
    const double hl = h[i], t0 = x[i + 1] - xe[e], t1 = xe[e] - x[i];
    for (int m = 0; m < n; ++m) {
      double v = (M[(size_t)i * n + m] * t0 * t0 * t0 + M[(size_t)(i + 1) * n + m] * t1 * t1 * t1) / (6.0 * hl);
      v += (-M[(size_t)i * n + m] * hl / 6.0) * t0 + (-M[(size_t)(i + 1) * n + m] * hl / 6.0) * t1;
      if (m == i) v += t0 / hl;
      if (m == i + 1) v += t1 / hl;
      S[(size_t)e * n + m] = v;
    }
  }
}

nsgpu_status build_shear(nsgpu_ctx* ctx, const nsgpu_theory* t) {
  ShearDev& S = ctx->sh;
  if (t->n_z_emu < 2 || t->n_z < 2 || t->n_chi < 1 || t->n_k < 2 || t->n_ell < 1 || t->n_tomo < 1 ||
      t->n_tomo > NSGPU_MAX_TOMO || !t->ell || !t->nz_mean || !(t->z_max > 0) || !(t->k_min > 0) ||
      !(t->k_max > t->k_min) || !(t->nz_sigma > 0)) {
    ctx->err = "shear theory: bad grid sizes or NULL arrays";
    return NSGPU_EINVAL;
  }
  if (t->z_interp == 0 && t->n_z != t->n_z_emu) { ctx->err = "z_interp = 0 needs n_z == n_z_emu"; return NSGPU_EINVAL; }
  if (t->z_interp != 0 && t->z_interp != 2) { ctx->err = "z_interp must be 0 or 2"; return NSGPU_EINVAL; }
  if (t->z_interp == 2 && t->n_z_emu < 4) { ctx->err = "cubic z-spline needs n_z_emu >= 4"; return NSGPU_EINVAL; }
  const int idx[] = {t->idx_omega_b, t->idx_omega_cdm, t->idx_h, t->idx_dz, t->idx_ia, t->idx_m};
  for (int v : idx)
    if (v < 0 || v >= ctx->D) { ctx->err = "shear theory: parameter index out of range"; return NSGPU_EINVAL; }
  if (t->n_ia_terms < 1 || t->n_ia_terms > 3 || t->n_m_terms < 1 || t->n_m_terms > 2) {
    ctx->err = "shear theory: n_ia_terms must be 1..3 and n_m_terms 1..2";
    return NSGPU_EINVAL;
  }
  if (t->idx_dz + t->n_tomo > ctx->D || t->idx_ia + t->n_ia_terms * t->n_tomo > ctx->D ||
      t->idx_m + t->n_m_terms * t->n_tomo > ctx->D ||
      t->idx_w0 >= ctx->D || t->idx_wa >= ctx->D || t->idx_eta0 >= ctx->D) {
    ctx->err = "shear theory: parameter block exceeds D";
    return NSGPU_EINVAL;
  }
  S.n_z_emu = t->n_z_emu; S.n_z = t->n_z; S.n_chi = t->n_chi; S.n_k = t->n_k; S.n_ell = t->n_ell; S.n_tomo = t->n_tomo;
  S.z_max = t->z_max; S.k_min = t->k_min; S.k_max = t->k_max; S.nz_sigma = t->nz_sigma;
  S.lk0 = log10(t->k_min);
  S.dlk = (log10(t->k_max) - log10(t->k_min)) / (t->n_k - 1);
  S.idx_omega_b = t->idx_omega_b; S.idx_omega_cdm = t->idx_omega_cdm; S.idx_h = t->idx_h; S.idx_w0 = t->idx_w0;
  S.idx_wa = t->idx_wa; S.idx_eta0 = t->idx_eta0; S.idx_dz = t->idx_dz; S.idx_ia = t->idx_ia; S.idx_m = t->idx_m;
  S.n_ia_terms = t->n_ia_terms; S.n_m_terms = t->n_m_terms;
  // quadrature nodes: midpoints of n_chi equal cells in the scale factor, a = 1 .. 1/(1+z_max) (S3)
  const double a_min = 1.0 / (1.0 + t->z_max);
  S.da = (1.0 - a_min) / t->n_chi;
  std::vector<double> a_q(t->n_chi), z_q(t->n_chi);
  for (int q = 0; q < t->n_chi; ++q) { a_q[q] = 1.0 - (q + 0.5) * S.da; z_q[q] = 1.0 / a_q[q] - 1.0; }
  // z-interpolation taps over the emulator nodes: linear between Limber nodes, composed with
  // the cubic spline n_z_emu -> n_z when requested (BJ cfg 3b).  Both are constant matrices.
  std::vector<double> ze(t->n_z_emu), zl(t->n_z);
  for (int m = 0; m < t->n_z_emu; ++m) ze[m] = m * t->z_max / (t->n_z_emu - 1);
  for (int m = 0; m < t->n_z; ++m) zl[m] = m * t->z_max / (t->n_z - 1);
  const double dzl = zl[1] - zl[0];
  std::vector<int> tap_start(t->n_chi);
  std::vector<double> tap_w;
  if (t->z_interp == 0) {
    S.n_tap = 2;
    tap_w.assign((size_t)t->n_chi * 2, 0.0);
    for (int q = 0; q < t->n_chi; ++q) {
      int m = (int)floor(z_q[q] / dzl);
      m = std::min(std::max(m, 0), t->n_z - 2);
      const double tt = (z_q[q] - zl[m]) / dzl;
      tap_start[q] = m;
      tap_w[(size_t)q * 2] = 1.0 - tt;
      tap_w[(size_t)q * 2 + 1] = tt;
    }
  } else {
    S.n_tap = t->n_z_emu;
    std::vector<double> Sm;
    spline_matrix(ze, zl, Sm);
    tap_w.assign((size_t)t->n_chi * S.n_tap, 0.0);
    for (int q = 0; q < t->n_chi; ++q) {
      int m = (int)floor(z_q[q] / dzl);
      m = std::min(std::max(m, 0), t->n_z - 2);
      const double tt = (z_q[q] - zl[m]) / dzl;
      tap_start[q] = 0;
      for (int k = 0; k < S.n_tap; ++k)
        tap_w[(size_t)q * S.n_tap + k] = (1.0 - tt) * Sm[(size_t)m * S.n_tap + k] + tt * Sm[(size_t)(m + 1) * S.n_tap + k];
    }
  }
  std::vector<float> zef(t->n_z_emu);
  for (int m = 0; m < t->n_z_emu; ++m) zef[m] = (float)ze[m];
  NSGPU_CUDA(upload(&S.a_q, a_q.data(), a_q.size()));
  NSGPU_CUDA(upload(&S.z_q, z_q.data(), z_q.size()));
  {
    std::vector<double> ln1pz(t->n_chi), lellh(t->n_ell), lf(t->n_ell);
    for (int q = 0; q < t->n_chi; ++q) ln1pz[q] = log1p(z_q[q]);
    for (int b = 0; b < t->n_ell; ++b) { lellh[b] = log10(t->ell[b] + 0.5); lf[b] = log(t->ell[b] / 550.0) / log(30.0); }
    NSGPU_CUDA(upload(&S.ln1pz, ln1pz.data(), ln1pz.size()));
    NSGPU_CUDA(upload(&S.lellh, lellh.data(), lellh.size()));
    NSGPU_CUDA(upload(&S.lf, lf.data(), lf.size()));
  }
  NSGPU_CUDA(upload(&S.tap_start, tap_start.data(), tap_start.size()));
  NSGPU_CUDA(upload(&S.tap_w, tap_w.data(), tap_w.size()));
  NSGPU_CUDA(upload(&S.ell, t->ell, (size_t)t->n_ell));
  NSGPU_CUDA(upload(&S.nz_mean, t->nz_mean, (size_t)t->n_tomo));
  NSGPU_CUDA(upload(&ctx->z_emu, zef.data(), zef.size()));
  {   // rows of n_chi rounded up to even (the streaming kernels bulk-copy row pieces); padding stays zero
    const size_t aux_bytes = (size_t)ctx->max_batch * (3 + t->n_tomo) * ((t->n_chi + 1) & ~1) * sizeof(double);
    NSGPU_CUDA(cudaMalloc((void**)&S.aux, aux_bytes));
    NSGPU_CUDA(cudaMemset(S.aux, 0, aux_bytes));
  }
  // the resident projection keeps a theta's table and scratch in shared memory (two CTAs per SM); larger
  // grids -- the paper's 1025 nodes and 10 bins -- take the streaming kernels
  S.streaming = (ctx->flags & NSGPU_SHEAR_STREAM) != 0 || shear_resident_smem(S) > 113 * 1024;
  if (S.streaming) {
    const size_t pg_bytes = (size_t)ctx->max_batch * t->n_ell * ((t->n_chi + 1) & ~1) * sizeof(double);
    NSGPU_CUDA(cudaMalloc((void**)&S.pg, pg_bytes));
    NSGPU_CUDA(cudaMemset(S.pg, 0, pg_bytes));
  }
  return NSGPU_OK;
}

nsgpu_status create_impl(nsgpu_ctx* ctx, int32_t D, const nsgpu_prior1d* prior, int32_t n_emu,
                         const nsgpu_emulator* emu, const nsgpu_theory* th, int32_t n_data, const double* data,
                         const double* chol, int32_t max_batch, int32_t device, uint32_t flags) {
  if (D < 1 || D > NSGPU_MAX_D) { ctx->err = "D must be in [1, 64]"; return NSGPU_ESHAPE; }
  if (!prior || !th || !data || (!chol && th->kind != 4) || n_data < 1 || max_batch < 1 || n_emu < 0 || (n_emu > 0 && !emu)) {
    ctx->err = "create: NULL pointer or non-positive size";
    return NSGPU_EINVAL;
  }
  if (th->kind < 0 || th->kind > 4) { ctx->err = "unknown theory kind"; return NSGPU_EINVAL; }
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
    ctx->err = "no CUDA device: nsgpu has no CPU fallback";
    return NSGPU_ECUDA;
  }
  if (device < 0 || device >= ndev) { ctx->err = "device index out of range"; return NSGPU_EINVAL; }
  NSGPU_CUDA(cudaSetDevice(device));
  ctx->device = device; ctx->D = D; ctx->n_emu = n_emu; ctx->n_data = n_data; ctx->max_batch = max_batch;
  ctx->kind = th->kind; ctx->flags = flags;
  cudaDeviceProp prop;
  NSGPU_CUDA(cudaGetDeviceProperties(&prop, device));
  ctx->sm_count = prop.multiProcessorCount;

  // prior table
  std::vector<int> pk(D);
  std::vector<double> p0(D), p1(D);
  for (int d = 0; d < D; ++d) {
    pk[d] = prior[d].kind; p0[d] = prior[d].p0; p1[d] = prior[d].p1;
    if (pk[d] != 0 && pk[d] != 1) { ctx->err = "prior kind must be 0 or 1"; return NSGPU_EINVAL; }
    if ((pk[d] == 0 && !(p1[d] > p0[d])) || (pk[d] == 1 && !(p1[d] > 0))) { ctx->err = "degenerate prior"; return NSGPU_EINVAL; }
  }
  NSGPU_CUDA(upload(&ctx->prior_kind, pk.data(), (size_t)D));
  NSGPU_CUDA(upload(&ctx->prior_p0, p0.data(), (size_t)D));
  NSGPU_CUDA(upload(&ctx->prior_p1, p1.data(), (size_t)D));

  // theory-dependent shape checks
  const int need_emu = th->kind == 0 ? 0 : (th->kind == 2 ? -1 : 1);   // kinds 1, 3, 4: exactly one emulator
  if (need_emu == 0 && n_data != D) { ctx->err = "identity theory needs n_data == D"; return NSGPU_ESHAPE; }
  if (need_emu == 1 && n_emu != 1) { ctx->err = "this theory kind takes exactly one emulator"; return NSGPU_EINVAL; }
  if (need_emu == -1 && (n_emu < 1 || n_emu > 8)) { ctx->err = "cmb_binned takes 1..8 emulators"; return NSGPU_EINVAL; }
  ctx->rows_per_theta = th->kind == 3 ? th->n_z_emu : 1;
  if (th->kind != 0) {
    ctx->n_theta_in = th->n_theta_in;
    if (th->n_theta_in < 1 || th->n_theta_in > NSGPU_MAX_IN - 1 || !th->emu_in_idx || !th->emu_in_const) {
      ctx->err = "bad emulator-input map";
      return NSGPU_EINVAL;
    }
    for (int j = 0; j < th->n_theta_in; ++j)
      if (th->emu_in_idx[j] >= D) { ctx->err = "emu_in_idx out of range"; return NSGPU_EINVAL; }
    NSGPU_CUDA(upload(&ctx->emu_in_idx, th->emu_in_idx, (size_t)th->n_theta_in));
    NSGPU_CUDA(upload(&ctx->emu_in_const, th->emu_in_const, (size_t)th->n_theta_in));
  }
  if (th->kind == 3) {
    nsgpu_status s = build_shear(ctx, th);
    if (s != NSGPU_OK) return s;
    if (n_data != th->n_tomo * (th->n_tomo + 1) / 2 * th->n_ell) { ctx->err = "shear: n_data != n_pairs * n_ell"; return NSGPU_ESHAPE; }
  }

  // emulators
  ctx->emu.resize(n_emu);
  int width_max = 0;
  for (int e = 0; e < n_emu; ++e) {
    const nsgpu_emulator& h = emu[e];
    EmuDev& E = ctx->emu[e];
    if (h.n_hidden < 1 || h.n_hidden + 1 > NSGPU_MAX_LAYERS || h.width < 1 || h.n_out < 1 || !h.W || !h.b || !h.alpha ||
        !h.beta || !h.in_mean || !h.in_std || !h.out_mean || !h.out_std) {
      ctx->err = "emulator: bad sizes or NULL arrays";
      return NSGPU_EINVAL;
    }
    const int want_in = ctx->n_theta_in + (th->kind == 3 ? 1 : 0);
    if (h.n_in != want_in) { ctx->err = "emulator n_in does not match the input map"; return NSGPU_ESHAPE; }
    if (e > 0 && (h.n_out != emu[0].n_out)) { ctx->err = "all emulators must share n_out"; return NSGPU_ESHAPE; }
    E.n_in = h.n_in; E.n_hidden = h.n_hidden; E.width = h.width; E.n_out = h.n_out; E.out_kind = h.out_kind;
    width_max = std::max(width_max, h.width);
    for (int l = 0; l <= h.n_hidden; ++l) {
      const size_t fi = l == 0 ? h.n_in : h.width, fo = l == h.n_hidden ? h.n_out : h.width;
      if (!h.W[l] || !h.b[l]) { ctx->err = "emulator: NULL layer"; return NSGPU_EINVAL; }
      NSGPU_CUDA(upload(&E.W[l], h.W[l], fi * fo));
      NSGPU_CUDA(upload(&E.b[l], h.b[l], fo));
      if (l < h.n_hidden) {
        NSGPU_CUDA(upload(&E.alpha[l], h.alpha[l], (size_t)h.width));
        NSGPU_CUDA(upload(&E.beta[l], h.beta[l], (size_t)h.width));
      }
    }
    NSGPU_CUDA(upload(&E.in_mean, h.in_mean, (size_t)h.n_in));
    NSGPU_CUDA(upload(&E.in_std, h.in_std, (size_t)h.n_in));
    NSGPU_CUDA(upload(&E.out_mean, h.out_mean, (size_t)h.n_out));
    { std::vector<float> z((size_t)h.n_out, 0.0f); NSGPU_CUDA(upload(&E.out_zero, z.data(), z.size())); }
    NSGPU_CUDA(upload(&E.out_std, h.out_std, (size_t)h.n_out));
  }
  if ((th->kind == 1 || th->kind == 4) && emu[0].n_out != n_data) { ctx->err = "emulator theory needs n_out == n_data"; return NSGPU_ESHAPE; }
  if (th->kind == 4 && (emu[0].out_kind != 1 || th->ell_min < 0)) { ctx->err = "cmb_tt_cv needs an exp10 emulator and ell_min >= 0"; return NSGPU_EINVAL; }
  if (th->kind == 3 && emu[0].n_out != th->n_k) { ctx->err = "shear: emulator n_out != n_k"; return NSGPU_ESHAPE; }
  if (th->kind == 3) {
    std::vector<double> mu((size_t)th->n_k);
    for (int i = 0; i < th->n_k; ++i) mu[i] = (double)emu[0].out_mean[i];
    NSGPU_CUDA(upload(&ctx->sh.mu_k, mu.data(), mu.size()));
  }
  if (th->kind == 2) {
    if (!th->bin_ptr || !th->bin_col || !th->bin_val || th->cal_index < 0 || th->cal_index >= D) {
      ctx->err = "cmb_binned: NULL binning matrix or bad cal_index";
      return NSGPU_EINVAL;
    }
    const int nnz = th->bin_ptr[n_data];
    ctx->n_spec_cols = n_emu * emu[0].n_out;
    for (int i = 0; i < nnz; ++i)
      if (th->bin_col[i] < 0 || th->bin_col[i] >= ctx->n_spec_cols) { ctx->err = "bin_col out of range"; return NSGPU_EINVAL; }
    NSGPU_CUDA(upload(&ctx->bin_ptr, th->bin_ptr, (size_t)n_data + 1));
    NSGPU_CUDA(upload(&ctx->bin_col, th->bin_col, (size_t)nnz));
    NSGPU_CUDA(upload(&ctx->bin_val, th->bin_val, (size_t)nnz));
    ctx->cal_index = th->cal_index;
  }

  if (th->kind == 4) {
    // cosmic-variance TT likelihood: log p_l = const_l - (nu/2) ln C_l - nu Chat_l / (2 C_l) with ln C = y ln 10.
    // Per multipole the kernel needs a_l = (nu/2) ln 10 and b_l = nu Chat_l / 2; the constants are summed here in fp64.
    const size_t n = n_data;
    std::vector<double> ta(n), tb(n);
    double cst = 0.0;
    for (size_t i = 0; i < n; ++i) {
      const double nu = 2.0 * (th->ell_min + (double)i) + 1.0, ch = data[i];
      if (!(ch > 0.0) || !std::isfinite(ch)) { ctx->err = "cmb_tt_cv: observed spectrum must be positive"; return NSGPU_EINVAL; }
      ta[i] = 0.5 * nu * log(10.0);
      tb[i] = 0.5 * nu * ch;
      cst += log(nu) + (0.5 * nu - 1.0) * (log(nu) + log(ch)) - 0.5 * nu * log(2.0) - lgamma(0.5 * nu);
    }
    ctx->log_norm = cst;
    NSGPU_CUDA(upload(&ctx->tt_a, ta.data(), n));
    NSGPU_CUDA(upload(&ctx->tt_b, tb.data(), n));
    { std::vector<double> mu(n); for (size_t i = 0; i < n; ++i) mu[i] = (double)emu[0].out_mean[i]; NSGPU_CUDA(upload(&ctx->tt_mu, mu.data(), n)); }
    NSGPU_CUDA(upload(&ctx->data, data, n));
  } else {
  // Gaussian: invert the Cholesky factor once (forward substitution on the identity, fp64)
  {
    const size_t n = n_data;
    double logdet = 0.0;
    for (size_t i = 0; i < n; ++i) {
      const double d = chol[i * n + i];
      if (!(d > 0.0) || !std::isfinite(d)) { ctx->err = "Cholesky factor: non-positive diagonal"; return NSGPU_ENOTSPD; }
      logdet += log(d);
    }
    ctx->log_norm = -0.5 * ((double)n * log(2.0 * M_PI) + 2.0 * logdet);
    std::vector<double> Linv(n * n, 0.0);
    for (size_t c = 0; c < n; ++c) {           // column c of the inverse
      Linv[c * n + c] = 1.0 / chol[c * n + c];
      for (size_t i = c + 1; i < n; ++i) {
        double s = 0.0;
        for (size_t j = c; j < i; ++j) s += chol[i * n + j] * Linv[j * n + c];
        Linv[i * n + c] = -s / chol[i * n + i];
      }
    }
    // stored transposed: LinvT[j][i] = Linv[i][j] (non-zero for i >= j), so that for a fixed column j the
    // rows i are contiguous -- coalesced for the row-per-thread chi^2 kernel
    // row stride: smallest >= n that is 8 mod 16 doubles -- 16-byte aligned pieces for the bulk copies, and a
    // tensor-core fragment load (4 columns x 8 rows) from a tile with this stride covers every bank exactly twice
    const size_t ns = n + ((8 + 16 - n % 16) % 16);
    ctx->linv_ld = (int)ns;
    std::vector<double> LinvT(n * ns, 0.0);
    for (size_t i = 0; i < n; ++i)
      for (size_t j = 0; j <= i; ++j) LinvT[j * ns + i] = Linv[i * n + j];
    NSGPU_CUDA(upload(&ctx->Linv, LinvT.data(), n * ns));
    NSGPU_CUDA(upload(&ctx->data, data, n));
  }
  }

  // workspaces
  const size_t M_max = (size_t)max_batch * ctx->rows_per_theta;
  if (n_emu > 0) {
    // fp32 [M][width] (SIMT) or two fp16 planes in 128-row tiles (tcgen05): pad M to a multiple of 128
    const size_t act_bytes = ((M_max + 127) / 128 * 128) * (size_t)width_max * ((flags & NSGPU_MLP_FP64) ? sizeof(double) : sizeof(float));
    NSGPU_CUDA(cudaMalloc(&ctx->act[0], act_bytes));
    NSGPU_CUDA(cudaMalloc(&ctx->act[1], act_bytes));
    ctx->spec_ld = th->kind == 3 ? emu[0].n_out : (emu[0].n_out + 3) & ~3;
    NSGPU_CUDA(cudaMalloc((void**)&ctx->spec, (size_t)n_emu * M_max * ctx->spec_ld * sizeof(float)));
  }
  NSGPU_CUDA(cudaMalloc((void**)&ctx->model, (size_t)max_batch * n_data * sizeof(double)));
  if (th->kind != 4) {   // chi^2 workspaces: transposed residuals [n_data][batch rounded up to 64], partial sums per row block
    const size_t bp = ((size_t)max_batch + 63) & ~(size_t)63;
    NSGPU_CUDA(cudaMalloc((void**)&ctx->resid_t, (size_t)n_data * bp * sizeof(double)));
    NSGPU_CUDA(cudaMalloc((void**)&ctx->chi2_part, (size_t)((n_data + 127) / 128) * bp * sizeof(double)));
  }
  NSGPU_CUDA(cudaMalloc((void**)&ctx->theta_stage, (size_t)max_batch * D * sizeof(float)));
  NSGPU_CUDA(cudaMalloc((void**)&ctx->logL_stage, (size_t)max_batch * sizeof(double)));
  NSGPU_CUDA(cudaMallocHost((void**)&ctx->theta_pinned, (size_t)max_batch * D * sizeof(float)));
  NSGPU_CUDA(cudaMallocHost((void**)&ctx->logL_pinned, (size_t)max_batch * sizeof(double)));

  NSGPU_CUDA(cudaMalloc((void**)&ctx->nonfinite_rows, sizeof(unsigned long long)));
  NSGPU_CUDA(cudaMemset(ctx->nonfinite_rows, 0, sizeof(unsigned long long)));
  if (th->kind == 3) {
    NSGPU_CUDA(cudaStreamCreateWithFlags(&ctx->side_stream, cudaStreamNonBlocking));
    NSGPU_CUDA(cudaEventCreateWithFlags(&ctx->ev_in, cudaEventDisableTiming));
    NSGPU_CUDA(cudaEventCreateWithFlags(&ctx->ev_side, cudaEventDisableTiming));
  }
  for (int e = 1; e < n_emu && e < 8; ++e) {
    NSGPU_CUDA(cudaStreamCreateWithFlags(&ctx->emu_stream[e], cudaStreamNonBlocking));
    NSGPU_CUDA(cudaEventCreateWithFlags(&ctx->emu_done[e], cudaEventDisableTiming));
  }
  // MLP path selection
  for (int e = 0; e < n_emu; ++e) {
    EmuDev& E = ctx->emu[e];
    const bool tc_ok = (E.width % 64 == 0) && E.width >= 64 && E.width <= 512 && prop.major == 10;
    if ((flags & 3u) == NSGPU_MLP_TC && !tc_ok) {
      ctx->err = "NSGPU_MLP_TC: tcgen05 path needs width % 64 == 0, 64 <= width <= 512 and an sm_100 device";
      return NSGPU_ESHAPE;
    }
    E.path = ((flags & 3u) != NSGPU_MLP_SIMT && (flags & NSGPU_MLP_FP64) == 0 && tc_ok) ? 1 : 0;
    if (E.path == 1) {
      nsgpu_status s = mlp_tc_prepare(ctx, e, &emu[e]);
      if (s != NSGPU_OK) return s;
    }
  }
  // the tcgen05 output layer writes the shear table as [theta][k][z] (coalesced for a row-per-thread epilogue)
  ctx->spec_kz = th->kind == 3 && n_emu == 1 && ctx->emu[0].path == 1;
  return sampler_create(ctx);
}

}  // namespace

extern "C" nsgpu_status nsgpu_create(nsgpu_ctx** out, int32_t D, const nsgpu_prior1d* prior, int32_t n_emu,
                                     const nsgpu_emulator* emu, const nsgpu_theory* theory, int32_t n_data,
                                     const double* data, const double* chol, int32_t max_batch, int32_t device,
                                     uint32_t flags) {
  if (!out) { g_create_error = "create: out is NULL"; return NSGPU_EINVAL; }
  *out = nullptr;
  nsgpu_ctx* ctx = new (std::nothrow) nsgpu_ctx();
  if (!ctx) { g_create_error = "create: out of host memory"; return NSGPU_ENOMEM; }
  nsgpu_status s;
  try {
    s = create_impl(ctx, D, prior, n_emu, emu, theory, n_data, data, chol, max_batch, device, flags);
  } catch (const std::bad_alloc&) {
    ctx->err = "create: out of host memory";
    s = NSGPU_ENOMEM;
  }
  if (s != NSGPU_OK) {
    if (s == NSGPU_ECUDA && ctx->err.find("out of memory") != std::string::npos) s = NSGPU_ENOMEM;
    g_create_error = ctx->err;
    nsgpu_destroy(ctx);
    return s;
  }
  *out = ctx;
  return NSGPU_OK;
}

extern "C" nsgpu_status nsgpu_destroy(nsgpu_ctx* ctx) {
  if (!ctx) return NSGPU_EINVAL;
  cudaSetDevice(ctx->device);
  nsgpu_probe_release(ctx);
  cudaDeviceSynchronize();
  sampler_destroy(ctx);
  if (ctx->side_stream) cudaStreamDestroy(ctx->side_stream);
  for (int e = 0; e < 8; ++e) { if (ctx->emu_stream[e]) cudaStreamDestroy(ctx->emu_stream[e]); if (ctx->emu_done[e]) cudaEventDestroy(ctx->emu_done[e]); }
  if (ctx->ev_in) cudaEventDestroy(ctx->ev_in);
  if (ctx->ev_side) cudaEventDestroy(ctx->ev_side);
  for (auto& ev : ctx->stage_events) { cudaEventDestroy(ev.a); cudaEventDestroy(ev.b); }
  for (cudaEvent_t ev : ctx->event_pool) cudaEventDestroy(ev);
  for (size_t e = 0; e < ctx->emu.size(); ++e) {
    EmuDev& E = ctx->emu[e];
    mlp_tc_release(ctx, (int)e);
    for (int l = 0; l < NSGPU_MAX_LAYERS; ++l) { cudaFree(E.W[l]); cudaFree(E.b[l]); cudaFree(E.alpha[l]); cudaFree(E.beta[l]); }
    cudaFree(E.in_mean); cudaFree(E.in_std); cudaFree(E.out_mean); cudaFree(E.out_std); cudaFree(E.out_zero);
  }
  cudaFree(ctx->prior_kind); cudaFree(ctx->prior_p0); cudaFree(ctx->prior_p1);
  cudaFree(ctx->emu_in_idx); cudaFree(ctx->emu_in_const); cudaFree(ctx->z_emu);
  cudaFree(ctx->bin_ptr); cudaFree(ctx->bin_col); cudaFree(ctx->bin_val);
  ShearDev& S = ctx->sh;
  cudaFree(S.aux); cudaFree(S.pg); cudaFree(S.mu_k); cudaFree(S.a_q); cudaFree(S.z_q); cudaFree(S.ln1pz); cudaFree(S.lellh); cudaFree(S.lf); cudaFree(S.tap_start); cudaFree(S.tap_w); cudaFree(S.ell); cudaFree(S.nz_mean);
  cudaFree(ctx->data); cudaFree(ctx->Linv); cudaFree(ctx->tt_a); cudaFree(ctx->tt_b); cudaFree(ctx->tt_mu);
  cudaFree(ctx->act[0]); cudaFree(ctx->act[1]); cudaFree(ctx->fused_scratch); cudaFree(ctx->spec); cudaFree(ctx->model); cudaFree(ctx->resid_t); cudaFree(ctx->chi2_part);
  cudaFree(ctx->theta_stage); cudaFree(ctx->logL_stage); cudaFree(ctx->nonfinite_rows);
  cudaFreeHost(ctx->theta_pinned); cudaFreeHost(ctx->logL_pinned);
  cudaGetLastError();
  delete ctx;
  return NSGPU_OK;
}

extern "C" const char* nsgpu_last_error(const nsgpu_ctx* ctx) { return ctx ? ctx->err.c_str() : g_create_error.c_str(); }

extern "C" int32_t nsgpu_mlp_path(const nsgpu_ctx* ctx, int32_t emu) {
  if (!ctx || emu < 0 || emu >= ctx->n_emu) return -1;
  return ctx->emu[emu].path;
}

extern "C" nsgpu_status nsgpu_set_profiling(nsgpu_ctx* ctx, int32_t on) {
  if (!ctx) return NSGPU_EINVAL;
  ctx->profiling = on != 0;
  if (ctx->profiling) {   // events for ~200 steps up front: creating them inside a timed region showed up as host hiccups
    NSGPU_CUDA(cudaSetDevice(ctx->device));
    while (ctx->event_pool.size() < 4096) {
      cudaEvent_t e;
      NSGPU_CUDA(cudaEventCreate(&e));
      ctx->event_pool.push_back(e);
    }
  }
  return NSGPU_OK;
}

extern "C" nsgpu_status nsgpu_stage_times(nsgpu_ctx* ctx, double* ms, int64_t* count) {
  if (!ctx || !ms || !count) return NSGPU_EINVAL;
  NSGPU_CUDA(cudaSetDevice(ctx->device));
  NSGPU_CUDA(cudaDeviceSynchronize());
  for (auto& ev : ctx->stage_events) {
    float t = 0.f;
    if (cudaEventElapsedTime(&t, ev.a, ev.b) == cudaSuccess) { ctx->stage_ms[ev.stage] += t; ctx->stage_count[ev.stage]++; }
    ctx->event_pool.push_back(ev.a);
    ctx->event_pool.push_back(ev.b);
  }
  ctx->stage_events.clear();
  for (int i = 0; i < NSGPU_N_STAGES; ++i) {
    ms[i] = ctx->stage_ms[i]; count[i] = ctx->stage_count[i];
    ctx->stage_ms[i] = 0.0; ctx->stage_count[i] = 0;
  }
  return NSGPU_OK;
}

extern "C" int64_t nsgpu_launch_count(const nsgpu_ctx* ctx) { return ctx ? ctx->launches : -1; }

extern "C" int64_t nsgpu_nonfinite_rows(nsgpu_ctx* ctx) {
  if (!ctx || !ctx->nonfinite_rows) return -1;
  unsigned long long v = 0;
  if (cudaSetDevice(ctx->device) != cudaSuccess || cudaDeviceSynchronize() != cudaSuccess ||
      cudaMemcpy(&v, ctx->nonfinite_rows, sizeof(v), cudaMemcpyDeviceToHost) != cudaSuccess)
    return -1;
  return (int64_t)v;
}

static nsgpu_status run_emulators(nsgpu_ctx* ctx, const float* theta, int B, const int* n_rows_dev, cudaStream_t st) {
  const size_t stride = (size_t)ctx->max_batch * ctx->rows_per_theta * ctx->spec_ld;
  // Several emulators (c1: TT, TE, EE at one row per theta: hidden GEMMs of 64 tiles on 148 SMs) run concurrently: fork after
  // theta is ready, emulator e on its own stream and activation buffers, join before the consumer.
  bool conc = ctx->n_emu > 1 && ctx->emu_stream[1] != nullptr && (ctx->flags & (NSGPU_NO_OVERLAP | NSGPU_MLP_FUSED)) == 0;
  for (int e = 0; e < ctx->n_emu && conc; ++e) conc = ctx->emu[e].path == 1;
  if (conc) {
    if (!ctx->ev_in) NSGPU_CUDA(cudaEventCreateWithFlags(&ctx->ev_in, cudaEventDisableTiming));
    NSGPU_CUDA(cudaEventRecord(ctx->ev_in, st));
    const int mode = ctx->kind == 4 ? NSGPU_SPEC_NOMEAN : 0;
    for (int e = 0; e < ctx->n_emu; ++e) {
      cudaStream_t se = e == 0 ? st : ctx->emu_stream[e];
      if (e > 0) NSGPU_CUDA(cudaStreamWaitEvent(se, ctx->ev_in, 0));
      nsgpu_status s = mlp_forward_tc(ctx, e, theta, B, n_rows_dev, ctx->spec + e * stride, ctx->spec_ld, mode, se);
      if (s != NSGPU_OK) return s;
      if (e > 0) NSGPU_CUDA(cudaEventRecord(ctx->emu_done[e], se));
    }
    for (int e = 1; e < ctx->n_emu; ++e) NSGPU_CUDA(cudaStreamWaitEvent(st, ctx->emu_done[e], 0));
    return NSGPU_OK;
  }
  for (int e = 0; e < ctx->n_emu; ++e) {
    float* out = ctx->spec + e * stride;
    // kinds 3 and 4: the fp32 table carries only the O(sigma_out) deviation y - mu_out; the consumer adds mu_out in fp64
    const int mode = (ctx->spec_kz ? NSGPU_SPEC_KZ : 0) | ((ctx->kind == 4 || ctx->kind == 3) ? NSGPU_SPEC_NOMEAN : 0);
    nsgpu_status s = ctx->emu[e].path == 1 ? mlp_forward_tc(ctx, e, theta, B, n_rows_dev, out, ctx->spec_ld, mode, st)
                                           : mlp_forward_simt(ctx, e, theta, B, n_rows_dev, out, ctx->spec_ld, mode & NSGPU_SPEC_NOMEAN, st);
    if (s != NSGPU_OK) return s;
  }
  return NSGPU_OK;
}

static nsgpu_status theory_device(nsgpu_ctx* ctx, const float* theta, int B, const int* n_rows_dev, cudaStream_t st) {
  // Shear: background and windows (a6-a7) depend on theta only, so they run on a side stream while the emulator
  // kernels (tensor-bound; the fp64 pipe is idle) work on `st`: theta is ready at ev_in, the table half waits for
  // ev_side.  The next call's ev_in is recorded after this call's table half, which orders the reuse of `aux`.
  // Measured (c3a, one B200): at B = 512 and inside nested-sampling rounds (~300 proposals) the step is 2% shorter; at
  // B = 4096 the GEMMs fill every SM, the side kernel only takes from them what it gains (hidden layers +0.04 ms, projection
  // -0.04 ms) and the extra events make the host side jittery -- so only batches of at most 1024 take the side stream.
  const bool overlap = ctx->kind == 3 && ctx->side_stream && B > 0 && B <= 1024 && (ctx->flags & NSGPU_NO_OVERLAP) == 0 &&
                       shear_has_split(ctx);
  if (overlap) {
    NSGPU_CUDA(cudaEventRecord(ctx->ev_in, st));
    NSGPU_CUDA(cudaStreamWaitEvent(ctx->side_stream, ctx->ev_in, 0));
    nsgpu_status s1 = shear_project(ctx, theta, B, n_rows_dev, ctx->side_stream, 1);
    if (s1 != NSGPU_OK) return s1;
    NSGPU_CUDA(cudaEventRecord(ctx->ev_side, ctx->side_stream));
  }
  nsgpu_status s = run_emulators(ctx, theta, B, n_rows_dev, st);
  if (s != NSGPU_OK) return s;
  if (overlap) {
    NSGPU_CUDA(cudaStreamWaitEvent(st, ctx->ev_side, 0));
    return shear_project(ctx, theta, B, n_rows_dev, st, 2);
  }
  switch (ctx->kind) {
    case 0:
    case 1:
    case 4: return copy_model(ctx, theta, B, n_rows_dev, st);
    case 2: return cmb_bin(ctx, theta, B, n_rows_dev, st);
    default: return shear_project(ctx, theta, B, n_rows_dev, st);
  }
}

nsgpu_status loglike_device(nsgpu_ctx* ctx, const float* theta, int B, const int* n_rows_dev, double* logL,
                            cudaStream_t st) {
  if (ctx->kind == 4) {   // the per-multipole likelihood reads the emulated log-spectrum directly
    nsgpu_status s4 = run_emulators(ctx, theta, B, n_rows_dev, st);
    if (s4 != NSGPU_OK) return s4;
    return cmb_tt_loglike(ctx, theta, B, n_rows_dev, logL, st);
  }
  nsgpu_status s = theory_device(ctx, theta, B, n_rows_dev, st);
  if (s != NSGPU_OK) return s;
  return chi2_loglike(ctx, theta, B, n_rows_dev, logL, st);
}

static nsgpu_status check_batch(nsgpu_ctx* ctx, const void* a, const void* b, int32_t B) {
  if (!ctx) return NSGPU_EINVAL;
  if (B < 0 || (B > 0 && (!a || !b))) { ctx->err = "batch call: NULL pointer or negative B"; return NSGPU_EINVAL; }
  if (B > ctx->max_batch) { ctx->err = "batch call: B exceeds max_batch"; return NSGPU_ESHAPE; }
  cudaError_t e = cudaSetDevice(ctx->device);
  if (e != cudaSuccess) { ctx->err = cudaGetErrorString(e); return NSGPU_ECUDA; }
  return NSGPU_OK;
}

extern "C" nsgpu_status nsgpu_loglike_batch(nsgpu_ctx* ctx, const float* theta, int32_t B, double* logL, void* stream) {
  nsgpu_status s = check_batch(ctx, theta, logL, B);
  if (s != NSGPU_OK || B == 0) return s;
  return loglike_device(ctx, theta, B, nullptr, logL, (cudaStream_t)stream);
}

extern "C" nsgpu_status nsgpu_loglike_batch_host(nsgpu_ctx* ctx, const float* theta_host, int32_t B, double* logL_host) {
  nsgpu_status s = check_batch(ctx, theta_host, logL_host, B);
  if (s != NSGPU_OK || B == 0) return s;
  cudaStream_t st = 0;
  memcpy(ctx->theta_pinned, theta_host, (size_t)B * ctx->D * sizeof(float));
  NSGPU_CUDA(cudaMemcpyAsync(ctx->theta_stage, ctx->theta_pinned, (size_t)B * ctx->D * sizeof(float),
                             cudaMemcpyHostToDevice, st));
  s = loglike_device(ctx, ctx->theta_stage, B, nullptr, ctx->logL_stage, st);
  if (s != NSGPU_OK) return s;
  NSGPU_CUDA(cudaMemcpyAsync(ctx->logL_pinned, ctx->logL_stage, (size_t)B * sizeof(double), cudaMemcpyDeviceToHost, st));
  NSGPU_CUDA(cudaStreamSynchronize(st));
  memcpy(logL_host, ctx->logL_pinned, (size_t)B * sizeof(double));
  return NSGPU_OK;
}

extern "C" nsgpu_status nsgpu_emulate_batch(nsgpu_ctx* ctx, int32_t e, const float* theta, int32_t B, float* out, void* stream) {
  nsgpu_status s = check_batch(ctx, theta, out, B);
  if (s != NSGPU_OK || B == 0) return s;
  if (e < 0 || e >= ctx->n_emu) { ctx->err = "emulate: emulator index out of range"; return NSGPU_EINVAL; }
  const bool ex = ctx->emu[e].out_kind == 1;
  const int mode = ex ? NSGPU_SPEC_EXP10 : 0;
  return ctx->emu[e].path == 1 ? mlp_forward_tc(ctx, e, theta, B, nullptr, out, ctx->emu[e].n_out, mode, (cudaStream_t)stream)
                               : mlp_forward_simt(ctx, e, theta, B, nullptr, out, ctx->emu[e].n_out, mode, (cudaStream_t)stream);
}

extern "C" nsgpu_status nsgpu_theory_batch(nsgpu_ctx* ctx, const float* theta, int32_t B, double* model, void* stream) {
  nsgpu_status s = check_batch(ctx, theta, model, B);
  if (s != NSGPU_OK || B == 0) return s;
  s = theory_device(ctx, theta, B, nullptr, (cudaStream_t)stream);
  if (s != NSGPU_OK) return s;
  NSGPU_CUDA(cudaMemcpyAsync(model, ctx->model, (size_t)B * ctx->n_data * sizeof(double), cudaMemcpyDeviceToDevice,
                             (cudaStream_t)stream));
  return NSGPU_OK;
}
