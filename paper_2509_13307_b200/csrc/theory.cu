// theory.cu -- from emulated log-spectra to the model vector (steps a5-a9).
//
// shear_project : per theta, background (a6), windows (a7), z/k interpolation of the emulated
//                 log10 P(k,z) table staged in shared memory and the extended-Limber sums reduced over
//                 the chi-quadrature nodes with warp shuffles (a5, a8)  [P:L330-353 eqs. A1-A4; P:L359]
// shear_windows, shear_power, shear_limber : the same for grids that do not fit shared memory (the paper's
//                 1025 nodes x 10 bins): windows with the bins scanned in groups, lookups against the table in
//                 place, Limber product on the fp64 tensor cores over chunks of the quadrature axis
// cmb_bin       : 10^y / linear, / A_cal^2, CSR binning (a9)            [BJ cfg 1; readings C1-C3]
// cmb_tt        : the paper's cosmic-variance TT likelihood
// copy_model    : identity / emulator-only theories (BJ cfg 0)
//
// HBM-bound stages: the only large read is the spectrum table written by the emulator (84 KB per
// theta for c2/c3a).  All arithmetic here is fp64 -- it is ~0.15 MFLOP per theta against 100 MFLOP in
// the emulator, and the absolute log L tolerance leaves no room for fp32 round-off downstream of
// the network.  The oracle sums the four terms of eq. A1 separately; this kernel
// projects the factored form (W^gamma + W^I)_i (W^gamma + W^I)_j once.
#include <math_constants.h>

#include "internal.cuh"
#include "tc_ptx.cuh"

namespace {

constexpr double C_OVER_H0 = 2997.92458;   // Mpc/h
constexpr double C1_RHOCR = 0.0138768;     // reading S12

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// exp(x) in fp64 for |x| < 700: n = rint(x log2 e), r = x - n ln 2 (two-constant reduction), degree-11
// Taylor polynomial on |r| <= 0.347 (truncation 0.347^12/12! = 6e-15), scaled by 2^n through the exponent
// field.  A third of the instructions of the library routine; the projection spends most of its
// arithmetic in 2^y and Gaussian evaluations.
__device__ __forceinline__ double exp_fast(double x) {
  if (x < -700.0) return 0.0;
  if (x > 709.0) return CUDART_INF;                      // past the exponent range: overflow, not garbage
  const double n = rint(x * 1.4426950408889634);
  double r = fma(n, -6.93147180369123816490e-01, x);
  r = fma(n, -1.90821492927058770002e-10, r);
  // Estrin evaluation of sum_{i<=11} r^i / i!: dependency depth 4 instead of the 11 of Horner's rule (the
  // lookups are latency-bound: 16 warps per SM)
  const double r2 = r * r, r4 = r2 * r2, r8 = r4 * r4;
  const double a0 = fma(r, 1.0, 1.0);
  const double a1 = fma(r, 1.6666666666666666e-01, 0.5);
  const double a2 = fma(r, 8.333333333333333e-03, 4.1666666666666664e-02);
  const double a3 = fma(r, 1.984126984126984e-04, 1.3888888888888889e-03);
  const double a4 = fma(r, 2.7557319223985893e-06, 2.48015873015873e-05);
  const double a5 = fma(r, 2.505210838544172e-08, 2.755731922398589e-07);
  const double b0 = fma(a1, r2, a0), b1 = fma(a3, r2, a2), b2 = fma(a5, r2, a4);
  const double p = fma(b2, r8, fma(b1, r4, b0));
  const int e = (int)n;
  return __hiloint2double(__double2hiint(p) + (e << 20), __double2loint(p));
}

// 1/x in fp64 for normal positive x: fp32 reciprocal seed, two Newton steps (relative error < 1e-15)
__device__ __forceinline__ double rcp_fast(double x) {
  double r = (double)__frcp_rn((float)x);
  r = fma(r, fma(-x, r, 1.0), r);
  r = fma(r, fma(-x, r, 1.0), r);
  return r;
}

// Exclusive prefix (or suffix, when `reverse`) sum of arr[0..n) in place by ONE warp: each lane sums a
// contiguous chunk, a shuffle scan carries across lanes.  No block-level synchronisation inside.
__device__ void warp_scan_exclusive(double* arr, int n, bool reverse, int lane) {
  const int per = (n + 31) >> 5;
  const int b0 = lane * per, b1 = min(b0 + per, n);
  double local = 0.0;
  for (int i = b0; i < b1; ++i) local += arr[reverse ? n - 1 - i : i];
  double inc = local;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const double t = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += t;
  }
  double run = inc - local;
  for (int i = b0; i < b1; ++i) {
    const int idx = reverse ? n - 1 - i : i;
    const double v = arr[idx];
    arr[idx] = run;
    run += v;
  }
}

// D (8x8) += A (8x4, row-major) . B (4x8, column-major) on the fp64 tensor cores
__device__ __forceinline__ void dmma_8x8x4(double (&d)[2], double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0, %1}, {%2}, {%3}, {%0, %1};"
               : "+d"(d[0]), "+d"(d[1]) : "d"(a), "d"(b));
}

struct ShearArgs {
  int n_z_emu, n_chi, n_k, n_ell, n_tomo, n_tap;
  int sz, sk;   // table strides: element (z node m, k node j) at m sz + j sk
  double k_min, k_max, lk0, dlk, da, nz_sigma;
  const double* mu_k;          // [n_k] mu_out of the emulator in fp64: the fp32 table holds y - mu_out
  const double *a_q, *z_q, *ln1pz, *tap_w, *ell, *lellh, *lf, *nz_mean;
  const int* tap_start;
  int idx_omega_b, idx_omega_cdm, idx_h, idx_w0, idx_wa, idx_eta0, idx_dz, idx_ia, idx_m, n_ia_terms, n_m_terms;
};

// One CTA per theta.  Thread 0 starts a bulk asynchronous copy (TMA, cp.async.bulk) of this theta's
// log10 P table into shared memory -- the kernel's only large HBM read -- and the CTA computes the
// background and the windows (which do not need the table) while it lands.
//
// PHASE 0: everything in one launch (fallback for grids whose scratch arrays are not 16-byte sized).
// PHASE 1: background + windows only (a6, a7), no table: many CTAs per SM; writes gq, log10 chi, 1/chi and the
//          total windows to `aux` [(3 + n_tomo) n_chi doubles per theta].
// PHASE 2: table + aux by bulk copy, then lookups and Limber sums (a5, a8).  Splitting takes the serial,
//          table-free prologue out of the kernel whose occupancy the 84 KB table pins at two CTAs per SM.
constexpr int SHEAR_THREADS = 256;
template <int PHASE>
__global__ void __launch_bounds__(SHEAR_THREADS, 2) shear_project_kernel(const float* __restrict__ theta, int D,
                                                                         const int* __restrict__ n_rows_dev,
                                                                         const float* __restrict__ spec, ShearArgs A,
                                                                         double* __restrict__ aux,
                                                                         double* __restrict__ model, int n_data) {
  const int b = blockIdx.x;
  pdl_wait();      // launch_pdl contract: the row count, the table and aux come from earlier kernels
  pdl_trigger();
  if (n_rows_dev && b >= *n_rows_dev) return;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int nq = A.n_chi, nt = A.n_tomo, nqp = nq | 1;
  const int n_scr = max(2 * nt, A.n_ell);
  double* chi = reinterpret_cast<double*>(smem_raw);   // [nq]
  double* Eq = chi + nq;                               // [nq]
  double* Dq = Eq + nq;                                // [nq]
  double* gq = Dq + nq;                                // [nq]   dchi / chi^2
  double* hs = gq + nq;                                // [nq]   half-cell terms, then log10 chi
  double* ichi = hs + nq;                              // [nq]   1 / chi
  double* Wt = ichi + nq;                              // [nt][nq] total window
  double* scr = Wt + (size_t)nt * nq;                  // [n_scr][nqp]: scan arrays, then Pg[n_ell][nqp]
  const int n_tap_s = A.n_tap <= 4 ? A.n_tap : 0;      // few taps: the z-interpolation weights are staged too
  double* c_ell = scr + (size_t)n_scr * nqp;           // [n_ell] ell + 1/2
  double* c_lell = c_ell + A.n_ell;                    // [n_ell] log10(ell + 1/2)
  double* c_tw = c_lell + A.n_ell;                     // [nq][n_tap_s]
  int* c_ts = reinterpret_cast<int*>(c_tw + (size_t)nq * n_tap_s);   // [nq] first tap row
  size_t n_dbl = (size_t)nq * (6 + nt) + (size_t)n_scr * nqp + 2 * A.n_ell + (size_t)nq * n_tap_s + (nq + 1) / 2 + 2;
  n_dbl = (n_dbl + 1) & ~(size_t)1;
  unsigned long long* bar = reinterpret_cast<unsigned long long*>(chi + n_dbl - 2);   // 8-byte mbarrier
  float* table = reinterpret_cast<float*>(chi + n_dbl);   // [n_z_emu][n_k], 16-byte aligned

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarp = blockDim.x >> 5;
  const unsigned nq_magic = 0xFFFFFFFFu / (unsigned)nq + 1u;    // it / nq == umulhi(it, magic) for it < 2^16
  const float* th = theta + (size_t)b * D;
  const float* src = spec + (size_t)b * A.n_z_emu * A.n_k;
  const unsigned table_bytes = (unsigned)(A.n_z_emu * A.n_k) * 4u;
  const bool bulk = (table_bytes & 15u) == 0 && ((reinterpret_cast<uintptr_t>(src) & 15) == 0);
  const unsigned bar_s = (unsigned)__cvta_generic_to_shared(bar);
  const unsigned aux_bytes = (unsigned)((3 + nt) * nq) * 8u;   // gq, hs, ichi, Wt are contiguous in shared memory
  const double* aux_b = aux + (size_t)b * (3 + nt) * nq;
  if (PHASE != 1) {
    if (bulk) {
      if (tid == 0) {
        const unsigned total = table_bytes + (PHASE == 2 ? aux_bytes : 0u);
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(bar_s) : "memory");
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("{\n.reg .b64 st;\nmbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1;\n}" ::"r"(bar_s), "r"(total) : "memory");
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                     ::"r"((unsigned)__cvta_generic_to_shared(table)), "l"(src), "r"(table_bytes), "r"(bar_s) : "memory");
        if (PHASE == 2)
          asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                       ::"r"((unsigned)__cvta_generic_to_shared(gq)), "l"(aux_b), "r"(aux_bytes), "r"(bar_s) : "memory");
      }
    } else {
      for (int i = tid; i < A.n_z_emu * A.n_k; i += blockDim.x) table[i] = __ldg(src + i);
    }
    if (PHASE == 2) __syncthreads();   // the mbarrier is initialised before anyone polls it
  }
  if (PHASE != 1) {   // small constant tables of the lookups (published by the __syncthreads below / in the phases)
    for (int i = tid; i < A.n_ell; i += blockDim.x) { c_ell[i] = A.ell[i] + 0.5; c_lell[i] = A.lellh[i]; }
    for (int i = tid; i < nq; i += blockDim.x) c_ts[i] = A.tap_start[i];
    for (int i = tid; i < nq * n_tap_s; i += blockDim.x) c_tw[i] = A.tap_w[i];
  }
  const double ob = th[A.idx_omega_b], oc = th[A.idx_omega_cdm], h = th[A.idx_h];
  const double Om = (ob + oc) / (h * h);
  const double w0 = A.idx_w0 >= 0 ? (double)th[A.idx_w0] : -1.0;
  const double wa = A.idx_wa >= 0 ? (double)th[A.idx_wa] : 0.0;
  const double eta0 = A.idx_eta0 >= 0 ? (double)th[A.idx_eta0] : 0.7;
  const double gam = 0.55 + 0.05 * (1.0 + w0 + 0.5 * wa);
  const double de_exp = 3.0 * (1.0 + w0 + wa);

  if (PHASE != 2) {
  // a6: E_q; f_q da and the growth integrand go to the scan arrays
  double* sc_f = scr;
  double* sc_g = scr + nqp;
  for (int q = tid; q < nq; q += blockDim.x) {
    const double a = A.a_q[q], z = A.z_q[q], opz = 1.0 + z;
    // reciprocals by rcp_fast (1e-15): an fp64 division is ~30 instructions
    const double E2 = Om * opz * opz * opz + (1.0 - Om) * exp_fast(de_exp * A.ln1pz[q] - 3.0 * wa * z * rcp_fast(opz));
    const double E = sqrt(E2);
    Eq[q] = E;
    const double ia_ = rcp_fast(a);
    const double fda = A.da * rcp_fast(a * a * E);
    const double Om_a = Om * rcp_fast(a * a * a * E2);
    const double gi = exp_fast(gam * log(Om_a)) * A.da * ia_;
    gq[q] = fda;
    hs[q] = gi;
    sc_f[q] = fda;
    sc_g[q] = gi;
  }
  __syncthreads();
  if (warp == 0) warp_scan_exclusive(sc_f, nq, false, lane);
  else if (warp == 1) warp_scan_exclusive(sc_g, nq, false, lane);
  __syncthreads();
  for (int q = tid; q < nq; q += blockDim.x) {
    const double c = C_OVER_H0 * (sc_f[q] + 0.5 * gq[q]);
    const double ic = rcp_fast(c);
    chi[q] = c;
    ichi[q] = ic;
    Dq[q] = exp_fast(sc_g[q] + 0.5 * hs[q]);                  // 1 / D_q
    gq[q] = C_OVER_H0 * gq[q] * ic * ic;                      // dchi_q / chi_q^2
  }
  __syncthreads();

  // a7: n_i(z - dz_i); W^I; the two suffix sums of W^gamma = A - chi B for all bins at once
  const double inv_sig = 1.0 / A.nz_sigma;
  const double norm = inv_sig / 2.5066282746310002;              // 1/(sigma sqrt(2 pi))
  const double wg_fac = 1.5 * Om / (C_OVER_H0 * C_OVER_H0);
  for (int it = tid; it < nt * nq; it += blockDim.x) {
    const int i = (int)__umulhi((unsigned)it, nq_magic), q = it - i * nq;
    const double mu = A.nz_mean[i] + (double)th[A.idx_dz + i];
    const float* ia = th + A.idx_ia + A.n_ia_terms * i;
    const double A0 = ia[0], A1 = A.n_ia_terms > 1 ? (double)ia[1] : 0.0, A2 = A.n_ia_terms > 2 ? (double)ia[2] : 0.0;
    const double z = A.z_q[q];
    const double u = (z - mu) * inv_sig;
    const double nz = exp_fast(-0.5 * u * u) * norm;
    const double w = nz * A.da * (1.0 + z) * (1.0 + z);       // n_i(z_q) dz_q, dz = da / a^2
    scr[(size_t)(2 * i) * nqp + q] = w;
    scr[(size_t)(2 * i + 1) * nqp + q] = w * ichi[q];
    const double x = fma(1.0 + z, 1.0 / 1.62, -1.0);          // a multiply: an fp64 division is ~30 instructions
    const double Aia = A0 + A1 * x + A2 * x * x;
    Wt[(size_t)i * nq + q] = -Aia * (C1_RHOCR / C_OVER_H0) * Om * Dq[q] * nz * Eq[q];   // W^I (eq. A4); Dq holds 1/D
  }
  __syncthreads();
  for (int c = warp; c < 2 * nt; c += nwarp) warp_scan_exclusive(scr + (size_t)c * nqp, nq, true, lane);
  __syncthreads();
  for (int it = tid; it < nt * nq; it += blockDim.x) {
    const int i = (int)__umulhi((unsigned)it, nq_magic), q = it - i * nq;
    const double s0 = scr[(size_t)(2 * i) * nqp + q], s1 = scr[(size_t)(2 * i + 1) * nqp + q];
    const double wg = wg_fac * (1.0 + A.z_q[q]) * chi[q] * (s0 - chi[q] * s1);
    Wt[(size_t)i * nq + q] += wg;                             // + W^gamma (eq. A3)
    if (i == 0) hs[q] = log10(chi[q]);
  }
  __syncthreads();
  if (PHASE == 1) {   // hand gq, log10 chi, 1/chi and the windows to the table kernel
    for (int i = tid; i < (3 + nt) * nq; i += blockDim.x) aux[(size_t)b * (3 + nt) * nq + i] = gq[i];
    return;
  }
  }   // PHASE != 2
  if (PHASE == 2) __syncthreads();   // constant tables staged
  if (bulk) {   // the table (and aux) have landed?
    unsigned ok = 0;
    while (!ok)
      asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0;\nselp.u32 %0, 1, 0, p;\n}"
                   : "=r"(ok) : "r"(bar_s) : "memory");
  }

  // a5 + a8 (lookup): P(k = (ell+1/2)/chi_q, z_q) g_q for every (ell, q); log10 k = log10(ell+1/2) - log10 chi
  double* Pg = scr;                                           // [n_ell][nqp]
  const double inv_dlk = 1.0 / A.dlk, bar_amp = (eta0 - 0.7) * 0.1;
  const bool vec_taps = A.sz == 1 && A.n_tap == A.n_z_emu && (A.n_tap & 3) == 0 && bulk;   // tap_start == 0 for all q
  // Work item = (quadrature node q, group of 4 ell): the per-node quantities (1/chi, log10 chi, g_q, the z taps)
  // are loaded once and serve four lookups; consecutive lanes have consecutive q.
  const int n_lg4 = (A.n_ell + 3) >> 2;
  for (int item = tid; item < n_lg4 * nq; item += blockDim.x) {
    const int lg = (int)__umulhi((unsigned)item, nq_magic), q = item - lg * nq;
    const double ic = ichi[q], lc = hs[q], g_q = gq[q];
    const int m0 = c_ts[q];
    const double* tw = n_tap_s ? c_tw + (size_t)q * A.n_tap : A.tap_w + (size_t)q * A.n_tap;
    const double tw0 = tw[0], tw1 = A.n_tap > 1 ? tw[1] : 0.0;
    const float* col0 = table + (size_t)m0 * A.sz;             // two-tap fast path: rows m0, m0 + 1
#pragma unroll 2
    for (int u = 0; u < 4; ++u) {
      const int bl = 4 * lg + u;
      if (bl >= A.n_ell) break;
      const double k = c_ell[bl] * ic;
      double P = 0.0;
      if (k >= A.k_min && k <= A.k_max) {
        const double x = c_lell[bl] - lc;
        int j = (int)floor((x - A.lk0) * inv_dlk);
        j = min(max(j, 0), A.n_k - 2);
        const double s = (x - (A.lk0 + j * A.dlk)) * inv_dlk;
        double lo = 0.0, hi = 0.0;
        if (vec_taps) {
          // [k][z] table, taps = all emulator nodes (spline folded in): the taps of one k are contiguous
          const float4* r0 = reinterpret_cast<const float4*>(table + (size_t)j * A.sk);
          const float4* r1 = reinterpret_cast<const float4*>(table + (size_t)(j + 1) * A.sk);
          const double2* tw2 = reinterpret_cast<const double2*>(tw);
          for (int t4 = 0; t4 < A.n_tap / 4; ++t4) {
            const float4 a = r0[t4], c = r1[t4];
            const double2 w01 = __ldg(tw2 + 2 * t4), w23 = __ldg(tw2 + 2 * t4 + 1);
            lo = fma(w01.x, (double)a.x, lo); lo = fma(w01.y, (double)a.y, lo);
            lo = fma(w23.x, (double)a.z, lo); lo = fma(w23.y, (double)a.w, lo);
            hi = fma(w01.x, (double)c.x, hi); hi = fma(w01.y, (double)c.y, hi);
            hi = fma(w23.x, (double)c.z, hi); hi = fma(w23.y, (double)c.w, hi);
          }
        } else if (A.n_tap == 2) {
          const float* r0 = col0 + (size_t)j * A.sk;
          lo = fma(tw1, (double)r0[A.sz], tw0 * (double)r0[0]);
          hi = fma(tw1, (double)r0[A.sk + A.sz], tw0 * (double)r0[A.sk]);
        } else {
          for (int t = 0; t < A.n_tap; ++t) {
            const float* row = table + (size_t)(m0 + t) * A.sz + (size_t)j * A.sk;
            const double w = tw[t];
            lo = fma(w, (double)row[0], lo);
            hi = fma(w, (double)row[A.sk], hi);
          }
        }
        double y = fma(s, hi - lo, lo);
        const double mu0 = __ldg(A.mu_k + j);                  // the table holds the deviation from mu_out(k): add it in fp64
        y += fma(s, __ldg(A.mu_k + j + 1) - mu0, mu0);
        const double k2 = k * k;
        y -= bar_amp * k2 * rcp_fast(k2 + 1.0);
        P = exp_fast(y * 2.302585092994046);
      }
      Pg[(size_t)bl * nqp + q] = P * g_q;
    }
  }
  __syncthreads();

  // a8 (sum): C_ij(ell) = sum_q Wt_i Wt_j Pg is a [pairs][q] x [q][ell] product: fp64 tensor cores (mma.m8n8k4.f64;
  // fragments: lane l holds A[l >> 2][l & 3], B[l & 3][l >> 2], D[l >> 2][2 (l & 3) + {0, 1}]).  A warp owns two
  // 8-pair tiles x all 8-ell tiles and every KS-th 4-node k-step; the A element W_i W_j is formed on the fly by
  // the lane that needs it.  The k-slices are joined through shared memory in a fixed order.  Falls back to the scalar loop below for more than 32 multipoles.
  const int n_pairs = nt * (nt + 1) / 2;
  const int MT = (n_pairs + 7) >> 3, NT = (A.n_ell + 7) >> 3;
  const int MP = (MT + 1) >> 1;
  if (NT <= 4 && MP <= nwarp && (size_t)(nwarp / MP) * MT * 8 * NT * 8 <= n_dbl + (size_t)A.n_z_emu * A.n_k / 2) {
    const int KS = nwarp / MP, mp = warp / KS, kslice = warp - mp * KS;
    const bool active = mp < MP;
    const int fk = lane & 3, fr = lane >> 2;
    const double *wi[2], *wj[2];
    bool row_ok[2];
#pragma unroll
    for (int m = 0; m < 2; ++m) {
      const int p = (2 * mp + m) * 8 + fr;
      int i = 0, j = 0;
      row_ok[m] = active && p < n_pairs;
      if (row_ok[m]) {
        int rem = p;
        while (rem >= nt - i) { rem -= nt - i; ++i; }
        j = i + rem;
      }
      wi[m] = Wt + (size_t)i * nq;
      wj[m] = Wt + (size_t)j * nq;
    }
    const bool two = active && 2 * mp + 1 < MT;
    double acc[2][4][2];
#pragma unroll
    for (int m = 0; m < 2; ++m)
#pragma unroll
      for (int t = 0; t < 4; ++t) { acc[m][t][0] = 0.0; acc[m][t][1] = 0.0; }
    if (active) {
      for (int q0 = 4 * kslice; q0 < nq; q0 += 4 * KS) {
        const int q = q0 + fk;
        const bool in = q < nq;                                // ragged last k-step
        const double a0 = (in && row_ok[0]) ? wi[0][q] * wj[0][q] : 0.0;
        const double a1 = (in && row_ok[1]) ? wi[1][q] * wj[1][q] : 0.0;
#pragma unroll
        for (int t = 0; t < 4; ++t) {
          if (t < NT) {
            const int bl = 8 * t + fr;
            const double bv = (in && bl < A.n_ell) ? Pg[(size_t)bl * nqp + q] : 0.0;
            dmma_8x8x4(acc[0][t], a0, bv);
            if (two) dmma_8x8x4(acc[1][t], a1, bv);
          }
        }
      }
    }
    __syncthreads();                                           // every warp is done with Wt and Pg: reuse the CTA's shared memory
    double* red = chi;                                         // [KS][MT * 8][NT * 8]
    const int ldc = NT * 8;
    if (active) {
#pragma unroll
      for (int m = 0; m < 2; ++m) {
        if (m == 1 && !two) break;
        const int row = (2 * mp + m) * 8 + fr;
#pragma unroll
        for (int t = 0; t < 4; ++t)
          if (t < NT) {
            double* dst = red + ((size_t)kslice * MT * 8 + row) * ldc + 8 * t + 2 * fk;
            dst[0] = acc[m][t][0]; dst[1] = acc[m][t][1];
          }
      }
    }
    __syncthreads();
    for (int o = tid; o < n_pairs * A.n_ell; o += blockDim.x) {
      const int p = o / A.n_ell, bl = o - p * A.n_ell;
      double v = 0.0;
      for (int k = 0; k < KS; ++k) v += red[((size_t)k * MT * 8 + p) * ldc + bl];
      int i = 0, rem = p;
      while (rem >= nt - i) { rem -= nt - i; ++i; }
      const int j = i + rem;
      const double lf = A.lf[bl];                              // ln(ell/550)/ln 30
      const float* mpi = th + A.idx_m + A.n_m_terms * i;
      const float* mpj = th + A.idx_m + A.n_m_terms * j;
      const double mi = (double)mpi[0] + (A.n_m_terms > 1 ? (double)mpi[1] * lf : 0.0);
      const double mj = (double)mpj[0] + (A.n_m_terms > 1 ? (double)mpj[1] * lf : 0.0);
      model[(size_t)b * n_data + o] = (1.0 + mi) * (1.0 + mj) * v;
    }
    return;
  }
  // a8 (sum): C_ij(ell) = sum_q Wt_i Wt_j Pg.  Work item = (pair, group of 4 ell); 4 adjacent lanes share
  // an item and split the q range, so the window product is formed once per 4 outputs; a 2-step shuffle
  // reduction joins the four partial sums.
  const int n_lg = (A.n_ell + 3) >> 2, n_items = n_pairs * n_lg;
  const int part = tid & 3;
  for (int item0 = 0; item0 < n_items; item0 += blockDim.x >> 2) {
    const int item = item0 + (tid >> 2);
    const bool live = item < n_items;
    const int p = live ? item / n_lg : 0, lg = live ? item - p * n_lg : 0;
    int i = 0, rem = p;                                        // pair p -> (i <= j), row-major upper
    while (rem >= nt - i) { rem -= nt - i; ++i; }
    const int j = i + rem;
    const double* wi = Wt + (size_t)i * nq;
    const double* wj = Wt + (size_t)j * nq;
    const int l0 = 4 * lg;
    const double* pg0 = Pg + (size_t)min(l0, A.n_ell - 1) * nqp;
    const double* pg1 = Pg + (size_t)min(l0 + 1, A.n_ell - 1) * nqp;
    const double* pg2 = Pg + (size_t)min(l0 + 2, A.n_ell - 1) * nqp;
    const double* pg3 = Pg + (size_t)min(l0 + 3, A.n_ell - 1) * nqp;
    double a0 = 0.0, a1 = 0.0, a2 = 0.0, a3 = 0.0;
    if (live)
      for (int q = part; q < nq; q += 4) {
        const double ww = wi[q] * wj[q];
        a0 = fma(ww, pg0[q], a0); a1 = fma(ww, pg1[q], a1); a2 = fma(ww, pg2[q], a2); a3 = fma(ww, pg3[q], a3);
      }
#pragma unroll
    for (int o = 1; o < 4; o <<= 1) {
      a0 += __shfl_xor_sync(0xffffffffu, a0, o); a1 += __shfl_xor_sync(0xffffffffu, a1, o);
      a2 += __shfl_xor_sync(0xffffffffu, a2, o); a3 += __shfl_xor_sync(0xffffffffu, a3, o);
    }
    const int bl = l0 + part;                                  // lane `part` writes ell l0 + part
    if (live && bl < A.n_ell) {
      const double acc = part == 0 ? a0 : (part == 1 ? a1 : (part == 2 ? a2 : a3));
      const double lf = A.lf[bl];                              // ln(ell/550)/ln 30
      const float* mpi = th + A.idx_m + A.n_m_terms * i;
      const float* mpj = th + A.idx_m + A.n_m_terms * j;
      const double mi = (double)mpi[0] + (A.n_m_terms > 1 ? (double)mpi[1] * lf : 0.0);
      const double mj = (double)mpj[0] + (A.n_m_terms > 1 ? (double)mpj[1] * lf : 0.0);
      model[(size_t)b * n_data + (size_t)p * A.n_ell + bl] = (1.0 + mi) * (1.0 + mj) * acc;
    }
  }
}

// ---- streaming projection (any grid size) --------------------------------------------------------------
// The resident kernel above keeps the whole log10 P table and all scratch arrays of a theta in shared
// memory: that caps it at ~50 z nodes x 420 k and ~100 quadrature nodes.  The paper's own grid is 1025
// nodes and 10 bins: the two kernels below do the same arithmetic with shared memory that
// does not grow with the table -- the table is read in place (each lookup touches two 32-byte sectors; the
// lanes of a warp hold consecutive quadrature nodes, whose taps are neighbours in the [k][z] layout), and
// the quadrature axis is walked in chunks.

// a6 + a7 for any n_chi: background and total windows to `aux` ([theta][(3 + n_tomo) n_chi]: g_q, log10 chi,
// 1/chi, W_i).  The suffix scans of the shear windows run G bins at a time so that shared memory is
// (4 + 2 G) n_chi doubles.
constexpr int WIN_G = 4, WIN_Q = 5;   // bins per scan pass; quadrature nodes per thread
__global__ void __launch_bounds__(256) shear_windows_kernel(const float* __restrict__ theta, int D,
                                                            const int* __restrict__ n_rows_dev, ShearArgs A, int G,
                                                            double* __restrict__ aux) {
  pdl_wait();      // launch_pdl contract
  pdl_trigger();
  const int b = blockIdx.x;
  if (n_rows_dev && b >= *n_rows_dev) return;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int nq = A.n_chi, nt = A.n_tomo, nqp = nq | 1;
  double* chi = reinterpret_cast<double*>(smem_raw);   // [nqp] f_q da first, then chi_q
  double* Eq = chi + nqp;
  double* iD = Eq + nqp;                               // growth integrand first, then 1 / D_q
  double* ichi = iD + nqp;
  double* scr = ichi + nqp;                            // [2 G][nqp] scan arrays
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarp = blockDim.x >> 5;
  const float* th = theta + (size_t)b * D;
  const int nqs = (nq + 1) & ~1;                       // row stride of `aux` here: even, rows are bulk-copied in chunks
  double* aux_b = aux + (size_t)b * (3 + nt) * nqs;
  const double ob = th[A.idx_omega_b], oc = th[A.idx_omega_cdm], h = th[A.idx_h];
  const double Om = (ob + oc) / (h * h);
  const double w0 = A.idx_w0 >= 0 ? (double)th[A.idx_w0] : -1.0;
  const double wa = A.idx_wa >= 0 ? (double)th[A.idx_wa] : 0.0;
  const double gam = 0.55 + 0.05 * (1.0 + w0 + 0.5 * wa);
  const double de_exp = 3.0 * (1.0 + w0 + wa);
  for (int q = tid; q < nq; q += blockDim.x) {
    const double a = A.a_q[q], z = A.z_q[q], opz = 1.0 + z;
    const double E2 = Om * opz * opz * opz + (1.0 - Om) * exp_fast(de_exp * A.ln1pz[q] - 3.0 * wa * z * rcp_fast(opz));
    const double E = sqrt(E2);
    const double fda = A.da * rcp_fast(a * a * E);
    const double gi = exp_fast(gam * log(Om * rcp_fast(a * a * a * E2))) * A.da * rcp_fast(a);
    Eq[q] = E; chi[q] = fda; iD[q] = gi;
    scr[q] = fda; scr[nqp + q] = gi;
  }
  __syncthreads();
  if (warp == 0) warp_scan_exclusive(scr, nq, false, lane);
  else if (warp == 1) warp_scan_exclusive(scr + nqp, nq, false, lane);
  __syncthreads();
  for (int q = tid; q < nq; q += blockDim.x) {
    const double fda = chi[q];
    const double c = C_OVER_H0 * (scr[q] + 0.5 * fda);
    const double ic = rcp_fast(c);
    chi[q] = c;
    ichi[q] = ic;
    iD[q] = exp_fast(scr[nqp + q] + 0.5 * iD[q]);
    aux_b[q] = C_OVER_H0 * fda * ic * ic;               // g_q = dchi_q / chi_q^2
    aux_b[nqs + q] = log10(c);
    aux_b[2 * nqs + q] = ic;
  }
  __syncthreads();
  const double inv_sig = 1.0 / A.nz_sigma;
  const double norm = inv_sig / 2.5066282746310002;
  const double wg_fac = 1.5 * Om / (C_OVER_H0 * C_OVER_H0);
  double* Wt = aux_b + 3 * (size_t)nqs;
  // A thread owns up to WIN_Q quadrature nodes (tid, tid + blockDim, ...) and walks the G bins of a pass for each:
  // no index division, one base pointer per bin; the W^I of its (bin, node) items stay in registers across the scans,
  // so each window is written once.
  for (int i0 = 0; i0 < nt; i0 += G) {
    const int g = min(G, nt - i0);
    double wI[WIN_G][WIN_Q];
#pragma unroll
    for (int ii = 0; ii < WIN_G; ++ii) {
      if (ii < g) {
        const int i = i0 + ii;
        const double mu = A.nz_mean[i] + (double)th[A.idx_dz + i];
        const float* ia = th + A.idx_ia + A.n_ia_terms * i;
        const double A0 = ia[0], A1 = A.n_ia_terms > 1 ? (double)ia[1] : 0.0, A2 = A.n_ia_terms > 2 ? (double)ia[2] : 0.0;
        double* s0 = scr + (size_t)(2 * ii) * nqp;
        double* s1 = s0 + nqp;
#pragma unroll
        for (int s = 0; s < WIN_Q; ++s) {
          const int q = tid + s * (int)blockDim.x;
          wI[ii][s] = 0.0;
          if (q < nq) {
            const double z = A.z_q[q], opz = 1.0 + z;
            const double u = (z - mu) * inv_sig;
            const double nz = exp_fast(-0.5 * u * u) * norm;
            const double w = nz * A.da * opz * opz;                    // n_i(z_q) dz_q, dz = da / a^2
            s0[q] = w;
            s1[q] = w * ichi[q];
            const double x = fma(opz, 1.0 / 1.62, -1.0);               // a multiply: an fp64 division is ~30 instructions
            const double Aia = A0 + A1 * x + A2 * x * x;
            wI[ii][s] = -Aia * (C1_RHOCR / C_OVER_H0) * Om * iD[q] * nz * Eq[q];   // W^I (eq. A4)
          }
        }
      }
    }
    __syncthreads();
    for (int c = warp; c < 2 * g; c += nwarp) warp_scan_exclusive(scr + (size_t)c * nqp, nq, true, lane);
    __syncthreads();
#pragma unroll
    for (int ii = 0; ii < WIN_G; ++ii) {
      if (ii < g) {
        const double* s0 = scr + (size_t)(2 * ii) * nqp;
        const double* s1 = s0 + nqp;
        double* wt = Wt + (size_t)(i0 + ii) * nqs;
#pragma unroll
        for (int s = 0; s < WIN_Q; ++s) {
          const int q = tid + s * (int)blockDim.x;
          if (q < nq)
            wt[q] = wI[ii][s] + wg_fac * (1.0 + A.z_q[q]) * chi[q] * (s0[q] - chi[q] * s1[q]);   // + W^gamma (eq. A3)
        }
      }
    }
    __syncthreads();
  }
}

// a5 + a8 (lookup) for any grid: P(k = (ell + 1/2)/chi_q, z_q) g_q for every (ell, q) to `pg` ([theta][ell][nq2],
// nq2 = n_chi rounded up to even).  One thread per (q, group of 4 ell), consecutive lanes = consecutive q; the
// table is read in place: no shared memory, so the SM holds 2048 threads and the L2 latency of the 16 loads
// each thread has in flight is covered.
__global__ void __launch_bounds__(256) shear_power_kernel(const float* __restrict__ theta, int D,
                                                          const int* __restrict__ n_rows_dev,
                                                          const float* __restrict__ spec, ShearArgs A,
                                                          const double* __restrict__ aux, int blocks_per_theta,
                                                          double* __restrict__ pg) {
  pdl_wait();      // launch_pdl contract
  pdl_trigger();
  const int b = blockIdx.x / blocks_per_theta, blk = blockIdx.x - b * blocks_per_theta;
  if (n_rows_dev && b >= *n_rows_dev) return;
  const int nq = A.n_chi, nq2 = (nq + 1) & ~1, n_lg4 = (A.n_ell + 3) >> 2;
  const int it = blk * blockDim.x + threadIdx.x;
  if (it >= n_lg4 * nq) return;
  const int lg = it / nq, q = it - lg * nq;
  const float* th = theta + (size_t)b * D;
  const float* table = spec + (size_t)b * A.n_z_emu * A.n_k;
  const double* aux_b = aux + (size_t)b * (3 + A.n_tomo) * nq2;
  double* out = pg + (size_t)b * A.n_ell * nq2 + q;
  const double eta0 = A.idx_eta0 >= 0 ? (double)th[A.idx_eta0] : 0.7;
  const double inv_dlk = 1.0 / A.dlk, bar_amp = (eta0 - 0.7) * 0.1;
  const double g_q = aux_b[q], lc = aux_b[nq2 + q], ic = aux_b[2 * nq2 + q];
  const double* tw = A.tap_w + (size_t)q * A.n_tap;
  const float* col0 = table + (size_t)A.tap_start[q] * A.sz;
  const int l0 = 4 * lg, nl = min(4, A.n_ell - l0);
  double kk[4], ss[4], mu[4];
  const float* r0[4];
  bool ok[4];
#pragma unroll
  for (int u = 0; u < 4; ++u) {
    const int bl = min(l0 + u, A.n_ell - 1);
    kk[u] = (A.ell[bl] + 0.5) * ic;
    ok[u] = u < nl && kk[u] >= A.k_min && kk[u] <= A.k_max;
    const double x = A.lellh[bl] - lc;
    int j = (int)floor((x - A.lk0) * inv_dlk);
    j = min(max(j, 0), A.n_k - 2);
    ss[u] = (x - (A.lk0 + j * A.dlk)) * inv_dlk;
    r0[u] = col0 + (size_t)j * A.sk;
    const double mu0 = __ldg(A.mu_k + j);                      // the table holds the deviation from mu_out(k)
    mu[u] = fma(ss[u], __ldg(A.mu_k + j + 1) - mu0, mu0);
  }
  double lo[4], hi[4];
  if (A.n_tap == 2) {
    float f[4][4];
#pragma unroll
    for (int u = 0; u < 4; ++u) {   // all 16 loads are issued before the first use
      f[u][0] = __ldg(r0[u]); f[u][1] = __ldg(r0[u] + A.sz); f[u][2] = __ldg(r0[u] + A.sk); f[u][3] = __ldg(r0[u] + A.sk + A.sz);
    }
    const double tw0 = tw[0], tw1 = tw[1];
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      lo[u] = fma(tw1, (double)f[u][1], tw0 * (double)f[u][0]);
      hi[u] = fma(tw1, (double)f[u][3], tw0 * (double)f[u][2]);
    }
  } else {
#pragma unroll
    for (int u = 0; u < 4; ++u) { lo[u] = 0.0; hi[u] = 0.0; }
    for (int t = 0; t < A.n_tap; ++t) {
      const double w = tw[t];
#pragma unroll
      for (int u = 0; u < 4; ++u) {
        lo[u] = fma(w, (double)__ldg(r0[u] + (size_t)t * A.sz), lo[u]);
        hi[u] = fma(w, (double)__ldg(r0[u] + (size_t)t * A.sz + A.sk), hi[u]);
      }
    }
  }
#pragma unroll
  for (int u = 0; u < 4; ++u) {
    if (u >= nl) break;
    double P = 0.0;
    if (ok[u]) {
      double y = fma(ss[u], hi[u] - lo[u], lo[u]) + mu[u];
      const double k2 = kk[u] * kk[u];
      const float k2f = (float)k2;                     // |bar_amp| <= 0.03: fp32 is 3e-9 of log10 P here
      y -= bar_amp * (double)__fdividef(k2f, k2f + 1.0f);
      P = exp_fast(y * 2.302585092994046);
    }
    out[(size_t)(l0 + u) * nq2] = P * g_q;
  }
}

// a8 (sum) for any grid: C_ij(ell) = sum_q W_i W_j (P g)_q is, per theta, the product of WW [pairs][q] with
// (P g)^T [q][ell] (55 x 1025 by 1025 x 20 for the paper's grid): a dense fp64 contraction, done on the fp64 tensor
// cores (mma.m8n8k4.f64).  Fragments: lane l holds A[l >> 2][l & 3] (pair, node), B[l & 3][l >> 2] (node, ell) and
// D[l >> 2][2 (l & 3) + {0, 1}].  The A element W_i W_j is formed on the fly by the one lane that needs it (two
// shared-memory loads and a DMUL), so the pair products never exist in memory.  A warp owns two 8-pair tiles x all
// ell tiles and a slice of the 4-node k-steps of each chunk; chunks of QC nodes of W and P g are staged by 8-byte
// cp.async into a double buffer, one chunk ahead.  Row stride = 4 mod 16 doubles: a fragment load (8 rows x 4
// consecutive nodes) covers every bank exactly twice.
constexpr int LIMBER_THREADS = 256;
constexpr int LIMBER_QC = 64;                 // quadrature nodes per chunk
constexpr int LIMBER_LD = LIMBER_QC + 4;      // row stride of the staged chunks
constexpr int LIMBER_MAX_NT = 4;              // ell tiles of 8: n_ell <= 32
template <int NT>
__global__ void __launch_bounds__(LIMBER_THREADS, 3) shear_limber_kernel(const float* __restrict__ theta, int D,
                                                                         const int* __restrict__ n_rows_dev, ShearArgs A,
                                                                         const double* __restrict__ aux,
                                                                         const double* __restrict__ pg_all,
                                                                         double* __restrict__ model, int n_data) {
  pdl_wait();      // launch_pdl contract
  pdl_trigger();
  const int b = blockIdx.x;
  if (n_rows_dev && b >= *n_rows_dev) return;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int nq = A.n_chi, nq2 = (nq + 1) & ~1, nt = A.n_tomo;
  const int n_pairs = nt * (nt + 1) / 2;
  const int MT = (n_pairs + 7) >> 3;                                   // 8-row MMA tiles; NT 8-column tiles (template)
  const int MP = (MT + 1) >> 1, KS = (LIMBER_THREADS / 32) / MP;       // m-tile pairs; k-slices (warps per pair)
  const int w_rows = nt + 1, p_rows = NT * 8;                          // + one zero row for the padding pairs
  const size_t buf_doubles = (size_t)(w_rows + p_rows) * LIMBER_LD;
  double* sm = reinterpret_cast<double*>(smem_raw);                    // two buffers of [w_rows + p_rows][LD]
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const float* th = theta + (size_t)b * D;
  const double* w_b = aux + ((size_t)b * (3 + nt) + 3) * nq2;
  const double* pg_b = pg_all + (size_t)b * A.n_ell * nq2;
  for (int i = tid; i < 2 * (int)buf_doubles; i += blockDim.x) sm[i] = 0.0;   // padding rows and columns stay zero

  // this warp's tiles and this lane's fragment rows
  const int mp = warp / KS, kslice = warp - mp * KS;
  const bool active = mp < MP;
  const int fk = lane & 3, fr = lane >> 2;
  int wi_off[2], wj_off[2];                                            // row offsets of W_i, W_j for the lane's two pairs
#pragma unroll
  for (int m = 0; m < 2; ++m) {
    const int p = (2 * mp + m) * 8 + fr;
    int i = nt, j = nt;                                                // the zero row
    if (active && p < n_pairs) {
      i = 0;
      int rem = p;
      while (rem >= nt - i) { rem -= nt - i; ++i; }
      j = i + rem;
    }
    wi_off[m] = i * LIMBER_LD + fk;
    wj_off[m] = j * LIMBER_LD + fk;
  }
  const bool two = active && 2 * mp + 1 < MT;                          // the last pair of tiles may be a single tile
  double acc[2][NT][2];
#pragma unroll
  for (int m = 0; m < 2; ++m)
#pragma unroll
    for (int t = 0; t < NT; ++t) { acc[m][t][0] = 0.0; acc[m][t][1] = 0.0; }

  // chunk c of the windows and of P g goes to buffer c & 1: one bulk asynchronous copy per row (512 bytes), issued by
  // the lanes of warp 0 in parallel, completion on the buffer's mbarrier; one chunk ahead of the arithmetic.
  // (`aux` and `pg` rows have even strides and a zeroed padding element, so every piece is 16-byte sized and aligned.)
  const int n_chunks = (nq + LIMBER_QC - 1) / LIMBER_QC;
  const int n_rows_st = nt + A.n_ell;
  unsigned long long* bars = reinterpret_cast<unsigned long long*>(sm + 2 * buf_doubles);   // full[2]
  const uint32_t full0 = (uint32_t)__cvta_generic_to_shared(bars);
  auto stage = [&](int c) {                              // all threads
    const int q0 = c * LIMBER_QC, cnt = min(LIMBER_QC, nq2 - q0);      // even
    double* Wb = sm + (size_t)(c & 1) * buf_doubles;
    double* Pb = Wb + (size_t)w_rows * LIMBER_LD;
    if (cnt < LIMBER_QC)                                 // ragged last chunk: clear what the copies do not cover
      for (int i = tid; i < n_rows_st * (LIMBER_QC - cnt); i += blockDim.x) {
        const int r = i / (LIMBER_QC - cnt), qq = cnt + i - r * (LIMBER_QC - cnt);
        (r < nt ? Wb + (size_t)r * LIMBER_LD : Pb + (size_t)(r - nt) * LIMBER_LD)[qq] = 0.0;
      }
    if (warp == 0) {
      const uint32_t bar = full0 + 8 * (c & 1);
      if (lane == 0)
        asm volatile("{\n.reg .b64 st;\nmbarrier.arrive.expect_tx.shared::cta.b64 st, [%0], %1;\n}" ::"r"(bar), "r"((uint32_t)(n_rows_st * cnt * 8)) : "memory");
      __syncwarp();
      for (int r = lane; r < n_rows_st; r += 32) {
        double* dst = r < nt ? Wb + (size_t)r * LIMBER_LD : Pb + (size_t)(r - nt) * LIMBER_LD;
        const double* src = (r < nt ? w_b + (size_t)r * nq2 : pg_b + (size_t)(r - nt) * nq2) + q0;
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                     ::"r"((uint32_t)__cvta_generic_to_shared(dst)), "l"(src), "r"((uint32_t)(cnt * 8)), "r"(bar) : "memory");
      }
    }
  };
  if (tid == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(full0) : "memory");
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(full0 + 8) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();                                       // zero fill done, barriers initialised
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic-proxy zero fill before async-proxy writes
  stage(0);
  for (int c = 0; c < n_chunks; ++c) {
    tc::mbar_wait(full0 + 8 * (c & 1), (c >> 1) & 1);     // chunk c has landed (bounded wait: traps instead of hanging)
    __syncthreads();                                     // everyone is done with chunk c - 1: its buffer may be refilled
    if (c + 1 < n_chunks) stage(c + 1);                  // overlaps the arithmetic below
    if (active) {
      const double* Wb = sm + (size_t)(c & 1) * buf_doubles;
      const double* Pb = Wb + (size_t)w_rows * LIMBER_LD + (size_t)fr * LIMBER_LD + fk;
      const double *wi0 = Wb + wi_off[0], *wj0 = Wb + wj_off[0], *wi1 = Wb + wi_off[1], *wj1 = Wb + wj_off[1];
      if (two) {
#pragma unroll 4
        for (int q = 4 * kslice; q < LIMBER_QC; q += 4 * KS) {
          const double a0 = wi0[q] * wj0[q], a1 = wi1[q] * wj1[q];
#pragma unroll
          for (int t = 0; t < NT; ++t) {
            const double bv = Pb[8 * t * LIMBER_LD + q];
            dmma_8x8x4(acc[0][t], a0, bv);
            dmma_8x8x4(acc[1][t], a1, bv);
          }
        }
      } else {
#pragma unroll 4
        for (int q = 4 * kslice; q < LIMBER_QC; q += 4 * KS) {
          const double a0 = wi0[q] * wj0[q];
#pragma unroll
          for (int t = 0; t < NT; ++t) dmma_8x8x4(acc[0][t], a0, Pb[8 * t * LIMBER_LD + q]);
        }
      }
    }
  }
  // join the k-slices in a fixed order through shared memory (the chunk buffers are free after the barrier), apply
  // the shear-calibration factors and write the model
  __syncthreads();
  const int ldc = NT * 8;
  double* red = sm;                                      // [KS][MT * 8][NT * 8]
  if (active) {
#pragma unroll
    for (int m = 0; m < 2; ++m) {
      if (m == 1 && !two) break;
      const int row = (2 * mp + m) * 8 + fr;
#pragma unroll
      for (int t = 0; t < NT; ++t) {
        double* dst = red + ((size_t)kslice * MT * 8 + row) * ldc + 8 * t + 2 * fk;
        dst[0] = acc[m][t][0]; dst[1] = acc[m][t][1];
      }
    }
  }
  __syncthreads();
  for (int o = tid; o < n_pairs * A.n_ell; o += blockDim.x) {
    const int p = o / A.n_ell, bl = o - p * A.n_ell;
    double v = 0.0;
    for (int k = 0; k < KS; ++k) v += red[((size_t)k * MT * 8 + p) * ldc + bl];
    int i = 0, rem = p;
    while (rem >= nt - i) { rem -= nt - i; ++i; }
    const int j = i + rem;
    const double lf = A.lf[bl];
    const float* mpi = th + A.idx_m + A.n_m_terms * i;
    const float* mpj = th + A.idx_m + A.n_m_terms * j;
    const double mi = (double)mpi[0] + (A.n_m_terms > 1 ? (double)mpi[1] * lf : 0.0);
    const double mj = (double)mpj[0] + (A.n_m_terms > 1 ? (double)mpj[1] * lf : 0.0);
    model[(size_t)b * n_data + o] = (1.0 + mi) * (1.0 + mj) * v;
  }
}

// a9: model[b][r] = sum_e Bin[r][e] s_b[col_e] / A_cal^2, s = 10^y (or y) of the three emulated spectra.  One thread
// per (bin r, block of CB_T thetas): a CSR entry is read once and serves CB_T thetas; for a fixed theta the lanes
// of a warp (adjacent bins) read adjacent runs of the spectrum row and write adjacent model entries.  No shared
// memory: 2048 threads per SM cover the load latency.  fp64 from the table value onward.
constexpr int CB_T = 8;
__global__ void __launch_bounds__(128) cmb_bin_kernel(const float* __restrict__ theta, int D, int B,
                                                      const int* __restrict__ n_rows_dev,
                                                      const float* __restrict__ spec, int n_emu, int n_out, int ld,
                                                      size_t emu_stride, unsigned exp10_mask, int cal_index,
                                                      const int* __restrict__ bin_ptr,
                                                      const int* __restrict__ bin_col,
                                                      const float* __restrict__ bin_val, int n_data,
                                                      double* __restrict__ model) {
  pdl_wait();      // launch_pdl contract
  pdl_trigger();
  if (n_rows_dev) B = min(B, *n_rows_dev);
  const int b0 = blockIdx.y * CB_T;
  if (b0 >= B) return;
  const int r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= n_data) return;
  const int nb = min(CB_T, B - b0);
  double acc[CB_T];
#pragma unroll
  for (int t = 0; t < CB_T; ++t) acc[t] = 0.0;
  const int e1 = bin_ptr[r + 1];
  for (int e = bin_ptr[r]; e < e1; ++e) {
    const int col = bin_col[e];
    const double v = (double)bin_val[e];
    const int em = col / n_out;                          // which emulator's spectrum
    const float* src = spec + em * emu_stride + (size_t)b0 * ld + (col - em * n_out);
    const bool ex = (exp10_mask >> em) & 1u;
    float y[CB_T];
#pragma unroll
    for (int t = 0; t < CB_T; ++t) y[t] = __ldg(src + (size_t)min(t, nb - 1) * ld);
#pragma unroll
    for (int t = 0; t < CB_T; ++t) {
      const double sv = ex ? exp_fast((double)y[t] * 2.302585092994046) : (double)y[t];
      acc[t] = fma(v, sv, acc[t]);
    }
  }
#pragma unroll
  for (int t = 0; t < CB_T; ++t)
    if (t < nb) {
      const double acal = theta[(size_t)(b0 + t) * D + cal_index];
      model[(size_t)(b0 + t) * n_data + r] = acc[t] / (acal * acal);
    }
}

// kind 4: log L = const - sum_l [ a_l y_l + b_l 10^(-y_l) ], y = emulated log10 C_l.  One CTA per theta,
// fp64 terms and reduction; reads 4 n_out bytes per theta (HBM-bound), writes log L directly.
__global__ void __launch_bounds__(128) cmb_tt_kernel(const float* __restrict__ theta, int D, int B,
                                                     const int* __restrict__ n_rows_dev, const float* __restrict__ spec,
                                                     int n, int ld, const double* __restrict__ ta, const double* __restrict__ tb,
                                                     const double* __restrict__ mu, double cst, const int* __restrict__ prior_kind,
                                                     const double* __restrict__ p0, const double* __restrict__ p1,
                                                     double* __restrict__ logL) {
  pdl_wait();      // launch_pdl contract
  pdl_trigger();
  const int b = blockIdx.x;
  if (n_rows_dev) B = min(B, *n_rows_dev);
  if (b >= B) return;
  __shared__ double red[4];
  const float* y = spec + (size_t)b * ld;
  double acc = 0.0;
  for (int i = threadIdx.x; i < n; i += blockDim.x) {
    const double yi = (double)__ldg(y + i) + mu[i];            // the table holds y - mu_out (fp32), mu_out added in fp64
    acc += fma(ta[i], yi, tb[i] * exp_fast(-2.302585092994046 * yi));
  }
  acc = warp_sum(acc);
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
  __syncthreads();
  if (threadIdx.x == 0) {
    double out = cst - (red[0] + red[1] + red[2] + red[3]);
    bool ok = isfinite(out);
    for (int d = 0; d < D; ++d) {
      const float v = theta[(size_t)b * D + d];
      if (!isfinite(v)) ok = false;
      if (prior_kind[d] == 0 && (v < (float)p0[d] || v > (float)p1[d])) ok = false;
    }
    logL[b] = ok ? out : -INFINITY;
  }
}

// kind 0: model = theta; kind 1: model = spectrum of emulator 0 (10^y where out_kind = 1)
__global__ void copy_model_kernel(const float* __restrict__ src, int n, int ld, int B, const int* __restrict__ n_rows_dev,
                                  int apply_exp10, const double* __restrict__ mu, double* __restrict__ model) {
  pdl_wait();      // launch_pdl contract
  pdl_trigger();
  if (n_rows_dev) B = min(B, *n_rows_dev);
  const size_t total = (size_t)B * n;
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
    const size_t b = i / n, j = i - b * n;
    const double y = (double)src[b * ld + j] + (mu ? mu[j] : 0.0);
    model[i] = apply_exp10 ? exp10(y) : y;
  }
}

}  // namespace

static size_t shear_smem_bytes(const ShearDev& S) {
  const size_t nqp = (size_t)S.n_chi | 1, n_scr = (size_t)std::max(2 * S.n_tomo, S.n_ell);
  const size_t n_tap_s = S.n_tap <= 4 ? S.n_tap : 0;
  size_t d = (size_t)S.n_chi * (6 + S.n_tomo) + n_scr * nqp + 2 * S.n_ell + (size_t)S.n_chi * n_tap_s + (S.n_chi + 1) / 2 + 2;
  d = (d + 1) & ~(size_t)1;
  return d * sizeof(double) + (size_t)S.n_z_emu * S.n_k * sizeof(float) + 16;
}

// `phases`: 1 = the theta-only half (background, windows -> aux), 2 = the half that reads the emulated table, 3 = both.
// api.cu runs phase 1 on a side stream under the emulator kernels (its inputs do not depend on them).
nsgpu_status shear_project(nsgpu_ctx* ctx, const float* theta, int B, const int* n_rows_dev, cudaStream_t st, int phases) {
  if (B == 0) return NSGPU_OK;
  const ShearDev& S = ctx->sh;
  ShearArgs A;
  A.n_z_emu = S.n_z_emu; A.n_chi = S.n_chi; A.n_k = S.n_k; A.n_ell = S.n_ell; A.n_tomo = S.n_tomo; A.n_tap = S.n_tap;
  A.sz = ctx->spec_kz ? 1 : S.n_k; A.sk = ctx->spec_kz ? S.n_z_emu : 1;
  A.k_min = S.k_min; A.k_max = S.k_max; A.lk0 = S.lk0; A.dlk = S.dlk; A.da = S.da; A.nz_sigma = S.nz_sigma;
  A.mu_k = S.mu_k;
  A.a_q = S.a_q; A.z_q = S.z_q; A.ln1pz = S.ln1pz; A.tap_w = S.tap_w; A.ell = S.ell; A.lellh = S.lellh; A.lf = S.lf;
  A.nz_mean = S.nz_mean; A.tap_start = S.tap_start;
  A.idx_omega_b = S.idx_omega_b; A.idx_omega_cdm = S.idx_omega_cdm; A.idx_h = S.idx_h; A.idx_w0 = S.idx_w0;
  A.idx_wa = S.idx_wa; A.idx_eta0 = S.idx_eta0; A.idx_dz = S.idx_dz; A.idx_ia = S.idx_ia; A.idx_m = S.idx_m;
  A.n_ia_terms = S.n_ia_terms; A.n_m_terms = S.n_m_terms;
  // stage 3 is the half that reads the table (the HBM-roofline kernel); the theta-only half is timed with it only when it
  // runs on the same stream -- on the side stream it sits under the MLP stages
  StageTimer tm(ctx, (phases & 2) ? 3 : -1, st);
  if (S.streaming) {
    const size_t nqp = (size_t)S.n_chi | 1;
    // bins per scan pass: as many as keep the windows kernel at three CTAs per SM
    const int win_threads = S.n_chi > 256 ? 256 : 128;
    int G = std::min(S.n_tomo, WIN_G);
    while (G > 1 && (4 + 2 * (size_t)G) * nqp * sizeof(double) > 72 * 1024) --G;
    const size_t smem_w = (4 + 2 * (size_t)G) * nqp * sizeof(double);
    const int n_pairs = S.n_tomo * (S.n_tomo + 1) / 2, MT = (n_pairs + 7) / 8, NT = (S.n_ell + 7) / 8;
    const int MP = (MT + 1) / 2;
    if (MP > LIMBER_THREADS / 32 || NT > LIMBER_MAX_NT || smem_w > 220 * 1024 || S.n_chi > win_threads * WIN_Q) {
      ctx->err = "shear: n_tomo, n_ell (> 32) or n_chi too large for the streaming projection";
      return NSGPU_ESHAPE;
    }
    const int KS = (LIMBER_THREADS / 32) / MP;
    const size_t smem_l = std::max((size_t)2 * (S.n_tomo + 1 + NT * 8) * LIMBER_LD + 2, (size_t)KS * MT * 8 * NT * 8) * sizeof(double);
    if (phases & 1) {
      NSGPU_CUDA(nsgpu_ensure_smem(ctx, shear_windows_kernel, smem_w));
      NSGPU_CUDA(launch_pdl(ctx, shear_windows_kernel, dim3(B), dim3(win_threads), smem_w, st, theta, ctx->D, n_rows_dev, A, G, S.aux));
      NSGPU_LAUNCH_CHECK();
    }
    if (!(phases & 2)) return NSGPU_OK;
    const int bpt = (((S.n_ell + 3) / 4) * S.n_chi + 255) / 256;
    NSGPU_CUDA(launch_pdl(ctx, shear_power_kernel, dim3((unsigned)((size_t)B * bpt)), dim3(256), 0, st, theta, ctx->D, n_rows_dev, ctx->spec, A, S.aux, bpt, S.pg));
    NSGPU_LAUNCH_CHECK();
#define NSGPU_LIMBER(NT_)                                                                                              \
  case NT_:                                                                                                           \
    NSGPU_CUDA(nsgpu_ensure_smem(ctx, shear_limber_kernel<NT_>, smem_l));                                              \
    NSGPU_CUDA(launch_pdl(ctx, shear_limber_kernel<NT_>, dim3(B), dim3(LIMBER_THREADS), smem_l, st, theta, ctx->D, n_rows_dev, A, S.aux, S.pg, ctx->model, ctx->n_data)); \
    break;
    switch (NT) { NSGPU_LIMBER(1) NSGPU_LIMBER(2) NSGPU_LIMBER(3) NSGPU_LIMBER(4) }
#undef NSGPU_LIMBER
    NSGPU_LAUNCH_CHECK();
    return NSGPU_OK;
  }
  const size_t smem = shear_smem_bytes(S);
  const size_t smem1 = smem - (size_t)S.n_z_emu * S.n_k * sizeof(float);       // phase 1 stages no table
  NSGPU_CUDA(nsgpu_ensure_smem(ctx, shear_project_kernel<0>, smem));
  NSGPU_CUDA(nsgpu_ensure_smem(ctx, shear_project_kernel<1>, smem));
  NSGPU_CUDA(nsgpu_ensure_smem(ctx, shear_project_kernel<2>, smem));
  // the two-kernel split needs 16-byte sized / aligned pieces for the bulk copies
  const bool split = ((size_t)S.n_z_emu * S.n_k * 4) % 16 == 0 && ((size_t)(3 + S.n_tomo) * S.n_chi * 8) % 16 == 0 &&
                     ((size_t)3 * S.n_chi * 8) % 16 == 0 && S.aux != nullptr;
  if (split) {
    if (phases & 1) {
      NSGPU_CUDA(launch_pdl(ctx, shear_project_kernel<1>, dim3(B), dim3(128), smem1, st, theta, ctx->D, n_rows_dev, ctx->spec, A, S.aux, ctx->model, ctx->n_data));
      NSGPU_LAUNCH_CHECK();
    }
    if (!(phases & 2)) return NSGPU_OK;
    NSGPU_CUDA(launch_pdl(ctx, shear_project_kernel<2>, dim3(B), dim3(SHEAR_THREADS), smem, st, theta, ctx->D, n_rows_dev, ctx->spec, A, S.aux, ctx->model, ctx->n_data));
  } else {
    if (!(phases & 2)) return NSGPU_OK;          // no split possible: everything in phase 2
    NSGPU_CUDA(launch_pdl(ctx, shear_project_kernel<0>, dim3(B), dim3(SHEAR_THREADS), smem, st, theta, ctx->D, n_rows_dev, ctx->spec, A, S.aux, ctx->model, ctx->n_data));
  }
  NSGPU_LAUNCH_CHECK();
  return NSGPU_OK;
}

// shared memory of the resident projection; the caller switches to the streaming kernels when it does not fit
size_t shear_resident_smem(const ShearDev& S) { return shear_smem_bytes(S); }

// can the theta-only half run as a launch of its own? (streaming kernels: always; resident: when the bulk-copy pieces align)
bool shear_has_split(const nsgpu_ctx* ctx) {
  const ShearDev& S = ctx->sh;
  if (S.streaming) return true;
  return ((size_t)S.n_z_emu * S.n_k * 4) % 16 == 0 && ((size_t)(3 + S.n_tomo) * S.n_chi * 8) % 16 == 0 &&
         ((size_t)3 * S.n_chi * 8) % 16 == 0 && S.aux != nullptr;
}

nsgpu_status cmb_bin(nsgpu_ctx* ctx, const float* theta, int B, const int* n_rows_dev, cudaStream_t st) {
  if (B == 0) return NSGPU_OK;
  const int n_out = ctx->emu[0].n_out;
  unsigned mask = 0;
  for (int e = 0; e < ctx->n_emu; ++e) mask |= (ctx->emu[e].out_kind == 1 ? 1u : 0u) << e;
  const size_t emu_stride = (size_t)ctx->max_batch * ctx->rows_per_theta * ctx->spec_ld;
  StageTimer tm(ctx, 4, st);
  dim3 grid((ctx->n_data + 127) / 128, (B + CB_T - 1) / CB_T);
  NSGPU_CUDA(launch_pdl(ctx, cmb_bin_kernel, grid, dim3(128), 0, st, theta, ctx->D, B, n_rows_dev, ctx->spec, ctx->n_emu, n_out, ctx->spec_ld,
                        emu_stride, mask, ctx->cal_index, ctx->bin_ptr, ctx->bin_col, ctx->bin_val, ctx->n_data, ctx->model));
  NSGPU_LAUNCH_CHECK();
  return NSGPU_OK;
}

nsgpu_status cmb_tt_loglike(nsgpu_ctx* ctx, const float* theta, int B, const int* n_rows_dev, double* logL, cudaStream_t st) {
  if (B == 0) return NSGPU_OK;
  StageTimer tm(ctx, 4, st);
  NSGPU_CUDA(launch_pdl(ctx, cmb_tt_kernel, dim3(B), dim3(128), 0, st, theta, ctx->D, B, n_rows_dev, ctx->spec, ctx->n_data, ctx->spec_ld, ctx->tt_a,
                        ctx->tt_b, ctx->tt_mu, ctx->log_norm, ctx->prior_kind, ctx->prior_p0, ctx->prior_p1, logL));
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
  NSGPU_CUDA(launch_pdl(ctx, copy_model_kernel, dim3(blocks), dim3(256), 0, st, src, n, ident ? n : ctx->spec_ld, B, n_rows_dev, ex,
                        ctx->kind == 4 ? ctx->tt_mu : (const double*)nullptr, ctx->model));
  NSGPU_LAUNCH_CHECK();
  return NSGPU_OK;
}
