"""CMB-like binned theory vector (step a9; BASELINE.json configs[1]; readings C1-C3):
s = [10^y_TT, y_TE, 10^y_EE] / A_cal^2, model = Bin . s with a block-diagonal CSR binning matrix.
(The paper's own CMB likelihood, is a different, cosmic-variance form: DESIGN.md "Next".)"""
import numpy as np


def model_vector(th, theta, spectra):
    """theta: one row; spectra: list of emulated spectra (already 10^y where out_kind = exp10),
    each [n_out]. Returns model[n_data]."""
    s = np.concatenate([np.asarray(x, np.float64) for x in spectra])
    a_cal = float(theta[th.cal_index])
    s = s / (a_cal * a_cal)
    n_data = len(th.bin_ptr) - 1
    out = np.zeros(n_data)
    for r in range(n_data):
        acc = 0.0
        for e in range(th.bin_ptr[r], th.bin_ptr[r + 1]):
            acc += float(th.bin_val[e]) * s[th.bin_col[e]]
        out[r] = acc
    return out
