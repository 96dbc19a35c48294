"""CosmoPower-style MLP emulator forward pass (steps a2-a4).

The paper only names the emulator; BASELINE.json north_star fixes the form:
dense layers with the gated activation (beta + sigma(alpha x)(1 - beta)) x, per-neuron alpha,
beta (reading E1), standardised inputs and de-standardised log-spectra (reading E2)."""
import numpy as np


def sigmoid(t):
    """overflow-safe logistic function."""
    out = np.empty_like(t)
    pos = t >= 0
    out[pos] = 1.0 / (1.0 + np.exp(-t[pos]))
    e = np.exp(t[~pos])
    out[~pos] = e / (1.0 + e)
    return out


def activation(t, alpha, beta):
    return (beta + (1.0 - beta) * sigmoid(alpha * t)) * t


def mlp_raw(emu, X):
    """X: [M, n_in] raw inputs. Returns the de-standardised output y [M, n_out] BEFORE out_kind."""
    f64 = lambda a: np.asarray(a, dtype=np.float64)
    x = (f64(X) - f64(emu.in_mean)) / f64(emu.in_std)
    for l in range(emu.n_hidden):
        t = x @ f64(emu.W[l]) + f64(emu.b[l])
        x = activation(t, f64(emu.alpha[l]), f64(emu.beta[l]))
    y = x @ f64(emu.W[emu.n_hidden]) + f64(emu.b[emu.n_hidden])
    return y * f64(emu.out_std) + f64(emu.out_mean)


def mlp_forward(emu, X):
    """Emulated spectrum: y for out_kind 0 (linear), 10^y for out_kind 1 (exp10)."""
    y = mlp_raw(emu, X)
    return np.power(10.0, y) if emu.out_kind == 1 else y


def mlp_forward_loops(emu, x_row):
    """Triple-loop restatement for ONE input row (pure Python, tiny nets only): the brute-force
    pin of mlp_raw's matmul form."""
    import math
    x = [(float(x_row[i]) - float(emu.in_mean[i])) / float(emu.in_std[i]) for i in range(emu.n_in)]
    for l in range(emu.n_hidden + 1):
        W, b = emu.W[l], emu.b[l]
        out = []
        for j in range(W.shape[1]):
            s = float(b[j])
            for i in range(W.shape[0]):
                s += x[i] * float(W[i, j])
            if l < emu.n_hidden:
                a, be = float(emu.alpha[l][j]), float(emu.beta[l][j])
                sg = 1.0 / (1.0 + math.exp(-a * s)) if a * s >= 0 else math.exp(a * s) / (1.0 + math.exp(a * s))
                s = (be + (1.0 - be) * sg) * s
            out.append(s)
        x = out
    return [x[j] * float(emu.out_std[j]) + float(emu.out_mean[j]) for j in range(emu.n_out)]
