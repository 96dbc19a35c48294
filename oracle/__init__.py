"""fp64 CPU oracle for the nsgpu hot path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain, slow, obviously-correct numpy/fp64 restatement of what the hot path computes,
written from /root/reference/PAPER.md (arXiv 2509.13307; cited below as P:L<line>) and the
readings listed in DESIGN.md (section "Readings of the paper").  It shares no code with the CUDA
path under `paper_2509_13307_b200/csrc/` and never imports the package's binding; the only
common module is `paper_2509_13307_b200/workloads.py` (seeded inputs, no method arithmetic),
whose objects are consumed here by attribute access only.

Only `tests/`, `__graft_entry__.smoke()` and the `cpu_baseline` / `--impl reference` legs of
`bench.py` may import this package.

Parity pins (tests/test_oracle_*.py, `-m "not gpu"`):
  emulator.mlp_forward   hand-computed 2-3-2 net; beta=1 / alpha=0 linear collapses; ReLU limit
  shear.*                EdS closed forms for chi, D; single-plane lensing kernel; power-law Limber
                         closed form; eq. A1 four-term sum == factored form; spline vs scipy + cubics
  cmb.*                  sigma_out=0 => 10^mu_out exactly; uniform-bin averages of constants
  gaussian.*             C=I, diagonal C, r = L e_j, 3x3 explicit inverse, log det vs eigenvalues
  prior.*                Phi^-1 against erfinv; uniform end points
  philox.*               Random123 known-answer vectors
  nested.*               constant-likelihood log Z, hand-computed 4-live/2-delete weights,
                         closed-form Gaussian-in-box log Z and H, slice-step uniformity (KS)
Parity UNPINNED (nothing but GPU == oracle fixes them):
  the invented nuisance extensions of reading S2 (A_{i,1}, A_{i,2}, m_{i,1}) and the baryon
  template of reading S21 -- they reduce to the paper's model when those coefficients are 0,
  which is tested; config-4 log Z has no closed form.
"""
