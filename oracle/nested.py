"""Nested sampling with batch deletion and constrained slice sampling, step by step
(steps a11-a14; "replaces the point with the lowest likelihood ... evidence accumulated as
a sum of likelihood values weighted by successively smaller prior volumes"; P:L52 slice sampling
(Neal 2003) under a hard likelihood constraint; "selecting k live points with the lowest
likelihoods ... evolving them with the likelihood constraint in parallel").  The paper gives prose
only; every choice it leaves open is a DESIGN.md reading N1-N10, restated at the step it applies.

Each chain is written as ordinary sequential code (a Python generator that yields the point it
needs a likelihood for).  `evolve_chains` only schedules those requests into batches; it takes no
part in the algorithm.
"""
import math
import numpy as np

from .philox import Stream

BRACKET_W = 2.0        # reading N3: initial bracket width in units of the direction vector
MAX_STEP_OUT = 32      # cap on expansions per side
MAX_SHRINK = 64        # cap on shrink steps; then the move fails and the chain stays at x0


def logaddexp(a, b):
    return float(np.logaddexp(a, b))


# ------------------------------------------------------------------------------------------
# a13: delete the k lowest, accumulate the evidence (readings N5, N6)
# ------------------------------------------------------------------------------------------
def delete_lowest(logL_live, k, logX, logZ):
    """Stable order by (logL, index); dead = first k; L* = largest deleted.
    For j = 0..k-1: n_j = n_live - j, logX_j = logX_{j-1} - 1/n_j,
    log w_j = logX_{j-1} + ln(1 - e^{-1/n_j}), logZ <- logaddexp(logZ, l_(j) + log w_j)."""
    n = len(logL_live)
    order = sorted(range(n), key=lambda i: (logL_live[i], i))
    dead = order[:k]
    logw, n_j = [], []
    for j, i in enumerate(dead):
        nj = n - j
        lw = logX + math.log(-math.expm1(-1.0 / nj))
        logZ = logaddexp(logZ, logL_live[i] + lw)
        logX = logX - 1.0 / nj
        logw.append(lw)
        n_j.append(nj)
    return dead, np.array(logw), np.array(n_j), logX, logZ, float(logL_live[dead[-1]])


# ------------------------------------------------------------------------------------------
# a14: live-set covariance and its Cholesky factor (reading N3)
# ------------------------------------------------------------------------------------------
def live_cholesky(u_live):
    u = np.asarray(u_live, np.float64)
    n, D = u.shape
    mean = u.sum(axis=0) / n
    c = u - mean
    cov = c.T @ c / (n - 1) + 1e-12 * np.eye(D)
    return np.linalg.cholesky(cov)


# ------------------------------------------------------------------------------------------
# a11/a12: one slice move, one chain (Neal 2003 stepping-out + shrinkage along a random direction)
# ------------------------------------------------------------------------------------------
def slice_move(x0, logL0, direction, Lstar, stream):
    """Generator. Yields a point x; is sent log L(T(x)) (or -inf if x is outside [0,1]^D, which
    the scheduler decides without a likelihood call).  inside(x) == value > L* (strict, N5).
    Returns (x_new, logL_new, failed)."""
    w = BRACKET_W
    l = -w * stream.uniform()
    r = l + w
    n = 0
    while n < MAX_STEP_OUT and (yield x0 + l * direction) > Lstar:
        l -= w
        n += 1
    n = 0
    while n < MAX_STEP_OUT and (yield x0 + r * direction) > Lstar:
        r += w
        n += 1
    for _ in range(MAX_SHRINK):
        t = l + (r - l) * stream.uniform()
        x = x0 + t * direction
        val = yield x
        if val > Lstar:
            return x, val, False
        if t < 0.0:
            l = t
        else:
            r = t
    return x0, logL0, True


def chain(x0, logL0, L_sigma, Lstar, n_steps, stream):
    """n_steps slice moves; direction d = L_sigma z / ||z||, z ~ N(0, I_D) (reading N3)."""
    D = len(x0)
    x, lx, fails = np.array(x0, np.float64), float(logL0), 0
    for _ in range(n_steps):
        z = stream.normals(D)
        d = L_sigma @ z / math.sqrt(float(z @ z))
        x, lx, failed = yield from slice_move(x, lx, d, Lstar, stream)
        fails += int(failed)
    return x, lx, fails


def evolve_chains(loglike_u, x0s, logL0s, L_sigma, Lstar, n_steps, seed, iteration):
    """Run len(x0s) chains; batches the likelihood requests of all chains that are waiting.
    Returns new points, their logL, number of likelihood evaluations, number of failed moves."""
    k = len(x0s)
    gens = [chain(x0s[c], logL0s[c], L_sigma, Lstar, n_steps, Stream(seed, c, iteration, 0)) for c in range(k)]
    waiting, done = {}, {}
    for c, g in enumerate(gens):
        try:
            waiting[c] = next(g)
        except StopIteration as e:          # n_steps == 0
            done[c] = e.value
    n_evals = 0
    while waiting:
        ids = list(waiting)
        pts = np.stack([waiting[c] for c in ids])
        in_box = np.all((pts >= 0.0) & (pts <= 1.0), axis=1)
        vals = np.full(len(ids), -np.inf)
        if np.any(in_box):
            vals[in_box] = loglike_u(pts[in_box])
            n_evals += int(in_box.sum())
        for c, v in zip(ids, vals):
            try:
                waiting[c] = gens[c].send(float(v))
            except StopIteration as e:
                done[c] = e.value
                del waiting[c]
    xs = np.stack([done[c][0] for c in range(k)])
    ls = np.array([done[c][1] for c in range(k)])
    return xs, ls, n_evals, sum(done[c][2] for c in range(k))


# ------------------------------------------------------------------------------------------
# error bar (reading N9) and information H
# ------------------------------------------------------------------------------------------
def batch_error_factor(n_live, k):
    """c = n_live sum_j (n_live-j)^-2 / sum_j (n_live-j)^-1, j = 0..k-1 (1 for k=1)."""
    j = np.arange(k)
    return n_live * np.sum(1.0 / (n_live - j) ** 2) / np.sum(1.0 / (n_live - j))


def simulate_logZ_error(logL_dead, n_j, logL_live_final, M=1000, seed=12345):
    """Redraw the volume sequence M times with t_j = U^{1/n_j} (Skilling 2006; the assumption the
    paper states at P:L182-184) and return the standard deviation of log Z."""
    rng = np.random.default_rng(seed)
    logL_dead = np.asarray(logL_dead, np.float64)
    n_j = np.asarray(n_j, np.float64)
    nl = len(logL_live_final)
    out = np.empty(M)
    for m in range(M):
        logt = np.log(rng.random(len(n_j))) / n_j
        logX = np.cumsum(logt)
        logX_prev = np.concatenate([[0.0], logX[:-1]])
        logw = logX_prev + np.log(-np.expm1(logt))
        terms = np.concatenate([logL_dead + logw, np.asarray(logL_live_final) + logX[-1] - math.log(nl)])
        mx = terms.max()
        out[m] = mx + math.log(np.sum(np.exp(terms - mx)))
    return float(out.std(ddof=1))


# ------------------------------------------------------------------------------------------
# the run (readings N1-N9)
# ------------------------------------------------------------------------------------------
def run(loglike_u, D, n_live, n_delete, n_steps, stop_frac=1e-3, seed=1, max_iter=100000, u_init=None):
    """Returns a dict: logZ, logZ_err (simulated), logZ_err_analytic, H, n_iter, n_like_evals,
    samples (u [N,D], logL [N], logw [N] = log(L_i w_i / Z))."""
    k = n_delete
    if u_init is None:
        u_live = np.empty((n_live, D))
        for i in range(n_live):
            st = Stream(seed, i, 0, 2)
            for d in range(D):
                u_live[i, d] = st.uniform()
    else:
        u_live = np.array(u_init, np.float64)
    logL_live = np.array(loglike_u(u_live), np.float64)
    n_evals = n_live
    logX, logZ = 0.0, -np.inf
    dead_u, dead_logL, dead_logw, dead_nj = [], [], [], []
    it = 0
    converged = False
    while it < max_iter:
        it += 1
        L_sigma = live_cholesky(u_live)                                  # before deletion (c.2 step 3)
        dead, logw, n_j, logX, logZ, Lstar = delete_lowest(list(logL_live), k, logX, logZ)
        for j, i in enumerate(dead):
            dead_u.append(u_live[i].copy()); dead_logL.append(float(logL_live[i]))
            dead_logw.append(float(logw[j])); dead_nj.append(int(n_j[j]))
        dead_set = set(dead)
        survivors = [i for i in range(n_live) if i not in dead_set]
        starts = [survivors[int(Stream(seed, c, it, 1).uniform() * len(survivors))] for c in range(k)]  # N4
        xs, ls, ne, _ = evolve_chains(loglike_u, u_live[starts], logL_live[starts], L_sigma, Lstar,
                                      n_steps, seed, it)
        n_evals += ne
        for c, i in enumerate(dead):                                     # chain c replaces dead row
            u_live[i] = xs[c]
            logL_live[i] = ls[c]
        mx = logL_live.max()
        logZ_live = mx + math.log(np.sum(np.exp(logL_live - mx))) - math.log(n_live) + logX      # N7
        if logZ_live - logaddexp(logZ, logZ_live) < math.log(stop_frac):
            converged = True
            break
    all_u = np.concatenate([np.array(dead_u).reshape(-1, D), u_live])
    all_logL = np.concatenate([dead_logL, logL_live])
    all_logw = np.concatenate([dead_logw, np.full(n_live, logX - math.log(n_live))])             # N8
    terms = all_logL + all_logw
    mx = terms.max()
    logZ_tot = mx + math.log(np.sum(np.exp(terms - mx)))
    p = np.exp(terms - logZ_tot)
    H = float(np.sum(p * (all_logL - logZ_tot)))
    err_sim = simulate_logZ_error(dead_logL, dead_nj, logL_live, seed=seed + 99)
    err_ana = math.sqrt(max(batch_error_factor(n_live, k) * H, 0.0) / n_live)
    return dict(logZ=logZ_tot, logZ_err=err_sim, logZ_err_analytic=err_ana, H=H, n_iter=it,
                n_like_evals=n_evals, converged=converged,
                u=all_u, logL=all_logL, logw=terms - logZ_tot, n_dead=len(dead_logL))
