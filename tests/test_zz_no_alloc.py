"""-m gpu: nsgpu_logz_error_noalloc, the one entry point that allocates nothing (its scratch is a file-scope device array
of 8.1 MiB; include/nsgpu.h).  Collected last on purpose (pytest -x: a failure here must not hide other tests).
Checks it against the existing path -- the error bar nsgpu_run's summary computes with cudaMalloc'd buffers -- on calls in a
row that share the static array: a long sequence, then a shorter one (stale contents behind it), then the first again."""
import numpy as np
import pytest

from paper_2509_13307_b200 import nsgpu, workloads as W

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")


def test_logz_error_noalloc_equals_the_run_summary_on_calls_in_a_row():
    wl = W.toy_identity(D=4)
    cases = [(160, 40, 8, 3), (96, 48, 6, 5)]            # (n_live, n_delete, n_steps, seed): 40+ and ~15 iterations
    with nsgpu.Context(wl, max_batch=160) as ctx:
        runs = [ctx.run(n, k, steps, seed=seed) for n, k, steps, seed in cases]
        assert runs[0]["n_dead"] > runs[1]["n_dead"] > 0

        def call(i):
            r, (n, k, _, seed) = runs[i], cases[i]
            nd = r["n_dead"]
            return ctx.logz_error_noalloc(r["logL"][:nd], r["logL"][nd:], k, seed)

        for i in (0, 1, 0, 1):                            # same tolerance as the sampler tests' evidence quantities: 1e-12
            err, sims = call(i)
            assert err == pytest.approx(runs[i]["logZ_err"], rel=1e-12, abs=0.0), (i, err, runs[i]["logZ_err"])
            assert np.all(np.isfinite(sims)) and sims.std(ddof=1) == pytest.approx(err, rel=1e-12)
            assert abs(sims.mean() - runs[i]["logZ"]) < 5.0 * err + 0.05     # the simulations scatter around the run's log Z
        # a caller's own stream, and no simulated values wanted
        s2 = torch.cuda.Stream()
        e2, _ = ctx.logz_error_noalloc(runs[0]["logL"][:runs[0]["n_dead"]], runs[0]["logL"][runs[0]["n_dead"]:], cases[0][1],
                                       cases[0][3], stream=s2)
        assert e2 == pytest.approx(runs[0]["logZ_err"], rel=1e-12)
        # sizes beyond the static array are refused with a clear error, and the context stays usable
        with pytest.raises(nsgpu.NsgpuError) as e:
            ctx.logz_error_noalloc(np.zeros((1 << 20) + 1), np.zeros(50), 25, 1)
        assert e.value.status == nsgpu.ESHAPE and "1048576" in str(e.value)
        with pytest.raises(nsgpu.NsgpuError) as e:
            ctx.logz_error_noalloc(np.zeros(10), np.zeros(50), 50, 1)
        assert e.value.status == nsgpu.EINVAL
        assert call(1)[0] == pytest.approx(runs[1]["logZ_err"], rel=1e-12)
