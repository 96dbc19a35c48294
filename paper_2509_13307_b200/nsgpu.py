"""Thin ctypes binding over the C-ABI library (include/nsgpu.h).  Argument marshalling only:
every step of the path runs in the CUDA kernels of libnsgpu.so.  torch is used for device memory
and streams.  There is no CPU fallback: if the library is missing or no CUDA device exists, calls
raise.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("NSGPU_LIB") or os.path.join(_HERE, "lib", "libnsgpu.so")   # NSGPU_LIB: another build of the library (kernel A/B runs)

OK, EINVAL, ENOMEM, ECUDA, ESHAPE, ENOTSPD, ENOCONV = 0, -1, -2, -3, -4, -5, -6
STATUS_NAMES = {0: "NSGPU_OK", -1: "NSGPU_EINVAL", -2: "NSGPU_ENOMEM", -3: "NSGPU_ECUDA",
                -4: "NSGPU_ESHAPE", -5: "NSGPU_ENOTSPD", -6: "NSGPU_ENOCONV"}
MLP_AUTO, MLP_SIMT, MLP_TC = 0, 1, 2
CHI2_STREAMED, CHI2_TILED = 8, 16   # OR into `mlp`: force one of the two chi^2 kernels (default: tiled for n_data >= 512)
MLP_CLUSTER, MLP_NO_CLUSTER = 32, 64   # OR into `mlp`: weight-multicast CTA pairs always / never (default: large batches)
SHEAR_STREAM = 4          # OR into `mlp`: streaming projection kernels even for grids that fit shared memory
MLP_FUSED, MLP_LAYERED = 256, 512   # OR into `mlp`: fused multi-layer tcgen05 kernel where the shape allows (opt-in) / layered (default)
MLP_FP64, MLP_SPLIT4 = 1024, 2048   # OR into `mlp`: precision-study modes (fp64 CUDA-core emulator; 4-product tcgen05 split)
NO_OVERLAP = 4096         # OR into `mlp`: no side stream for the theta-only half of the shear projection
NO_PDL = 128              # OR into `mlp`: plain stream ordering between kernels (default: programmatic dependent launch)

EXPORTS = ["nsgpu_create", "nsgpu_destroy", "nsgpu_last_error", "nsgpu_prior_transform",
           "nsgpu_loglike_batch", "nsgpu_loglike_batch_host", "nsgpu_emulate_batch", "nsgpu_theory_batch",
           "nsgpu_slice_step", "nsgpu_run", "nsgpu_last_samples", "nsgpu_delete_lowest", "nsgpu_live_cholesky",
           "nsgpu_debug_philox", "nsgpu_set_profiling", "nsgpu_stage_times", "nsgpu_mlp_path", "nsgpu_launch_count",
           "nsgpu_run_sharded", "nsgpu_shard_range", "nsgpu_sampler_counters", "nsgpu_nonfinite_rows",
           "nsgpu_clock_mark", "nsgpu_clock_marks_read", "nsgpu_run_multi", "nsgpu_multi_samples", "nsgpu_logz_error_noalloc"]


class NsgpuError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"{STATUS_NAMES.get(status, status)}: {msg}")
        self.status = status


class _Prior1d(C.Structure):
    _fields_ = [("kind", C.c_int32), ("p0", C.c_double), ("p1", C.c_double)]


_pf = C.POINTER(C.c_float)
_pd = C.POINTER(C.c_double)
_pi = C.POINTER(C.c_int32)


class _Emulator(C.Structure):
    _fields_ = [("n_in", C.c_int32), ("n_hidden", C.c_int32), ("width", C.c_int32), ("n_out", C.c_int32),
                ("out_kind", C.c_int32), ("W", C.POINTER(_pf)), ("b", C.POINTER(_pf)), ("alpha", C.POINTER(_pf)),
                ("beta", C.POINTER(_pf)), ("in_mean", _pf), ("in_std", _pf), ("out_mean", _pf), ("out_std", _pf)]


class _Theory(C.Structure):
    _fields_ = [("kind", C.c_int32), ("n_theta_in", C.c_int32), ("emu_in_idx", _pi), ("emu_in_const", _pd),
                ("bin_ptr", _pi), ("bin_col", _pi), ("bin_val", _pf), ("cal_index", C.c_int32), ("ell_min", C.c_int32),
                ("n_z_emu", C.c_int32), ("n_z", C.c_int32), ("n_chi", C.c_int32), ("n_k", C.c_int32),
                ("n_ell", C.c_int32), ("n_tomo", C.c_int32), ("z_interp", C.c_int32),
                ("z_max", C.c_double), ("k_min", C.c_double), ("k_max", C.c_double),
                ("ell", _pd), ("nz_mean", _pd), ("nz_sigma", C.c_double),
                ("idx_omega_b", C.c_int32), ("idx_omega_cdm", C.c_int32), ("idx_h", C.c_int32),
                ("idx_w0", C.c_int32), ("idx_wa", C.c_int32), ("idx_eta0", C.c_int32),
                ("idx_dz", C.c_int32), ("idx_ia", C.c_int32), ("idx_m", C.c_int32),
                ("n_ia_terms", C.c_int32), ("n_m_terms", C.c_int32)]


class _RunOpts(C.Structure):
    _fields_ = [("n_live", C.c_int32), ("n_delete", C.c_int32), ("n_steps", C.c_int32), ("stop_frac", C.c_double),
                ("max_iter", C.c_int64), ("seed", C.c_uint64)]


class _Result(C.Structure):
    _fields_ = [("logZ", C.c_double), ("logZ_err", C.c_double), ("logZ_err_analytic", C.c_double), ("H", C.c_double),
                ("n_iter", C.c_int64), ("n_dead", C.c_int64), ("n_like_evals", C.c_int64), ("n_rounds", C.c_int64),
                ("n_failed_moves", C.c_int64), ("seconds", C.c_double), ("seconds_sampling", C.c_double),
                ("seconds_summary", C.c_double), ("n_nonfinite_rows", C.c_int64)]


# int32 allgather(void* user, const void* send, void* recv, int64 bytes_per_rank, void* stream)  (include/nsgpu.h)
ALLGATHER_FN = C.CFUNCTYPE(C.c_int32, C.c_void_p, C.c_void_p, C.c_void_p, C.c_int64, C.c_void_p)

_lib = None


def lib():
    """Load libnsgpu.so (fails loudly when it has not been built: `python -m paper_2509_13307_b200.build`)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} not found: build it with `python -m paper_2509_13307_b200.build` "
                          "(nsgpu has no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp = C.c_void_p
    L.nsgpu_create.restype = C.c_int
    L.nsgpu_create.argtypes = [C.POINTER(vp), C.c_int32, C.POINTER(_Prior1d), C.c_int32, C.POINTER(_Emulator),
                               C.POINTER(_Theory), C.c_int32, _pd, _pd, C.c_int32, C.c_int32, C.c_uint32]
    L.nsgpu_destroy.restype = C.c_int
    L.nsgpu_destroy.argtypes = [vp]
    L.nsgpu_last_error.restype = C.c_char_p
    L.nsgpu_last_error.argtypes = [vp]
    L.nsgpu_prior_transform.restype = C.c_int
    L.nsgpu_prior_transform.argtypes = [vp, vp, C.c_int32, vp, vp]
    L.nsgpu_loglike_batch.restype = C.c_int
    L.nsgpu_loglike_batch.argtypes = [vp, vp, C.c_int32, vp, vp]
    L.nsgpu_loglike_batch_host.restype = C.c_int
    L.nsgpu_loglike_batch_host.argtypes = [vp, vp, C.c_int32, vp]
    L.nsgpu_emulate_batch.restype = C.c_int
    L.nsgpu_emulate_batch.argtypes = [vp, C.c_int32, vp, C.c_int32, vp, vp]
    L.nsgpu_theory_batch.restype = C.c_int
    L.nsgpu_theory_batch.argtypes = [vp, vp, C.c_int32, vp, vp]
    L.nsgpu_slice_step.restype = C.c_int
    L.nsgpu_slice_step.argtypes = [vp, vp, vp, C.c_int32, vp, C.c_int32, C.c_double, C.c_int32, C.c_uint64, C.c_int32,
                                   vp, vp, C.POINTER(C.c_int64), vp]
    L.nsgpu_run.restype = C.c_int
    L.nsgpu_run.argtypes = [vp, C.POINTER(_RunOpts), C.POINTER(_Result), vp, vp, vp, C.c_int64, C.POINTER(C.c_int64)]
    L.nsgpu_run_sharded.restype = C.c_int
    L.nsgpu_run_sharded.argtypes = [vp, C.POINTER(_RunOpts), C.c_int32, C.c_int32, ALLGATHER_FN, vp, C.POINTER(_Result),
                                    vp, vp, vp, C.c_int64, C.POINTER(C.c_int64)]
    L.nsgpu_sampler_counters.restype = C.c_int
    L.nsgpu_sampler_counters.argtypes = [vp, C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
    L.nsgpu_run_multi.restype = C.c_int
    L.nsgpu_run_multi.argtypes = [vp, C.POINTER(_RunOpts), C.c_int32, C.POINTER(C.c_uint64), C.POINTER(_Result)]
    L.nsgpu_multi_samples.restype = C.c_int
    L.nsgpu_multi_samples.argtypes = [vp, C.c_int32, vp, vp, vp, C.c_int64, C.POINTER(C.c_int64)]
    L.nsgpu_logz_error_noalloc.restype = C.c_int
    L.nsgpu_logz_error_noalloc.argtypes = [vp, _pd, C.c_int64, _pd, C.c_int32, C.c_int32, C.c_uint64, _pd, _pd, vp]
    L.nsgpu_clock_mark.restype = C.c_int
    L.nsgpu_clock_mark.argtypes = [vp, vp]
    L.nsgpu_clock_marks_read.restype = C.c_int
    L.nsgpu_clock_marks_read.argtypes = [vp, _pd, _pd, C.c_int32, C.POINTER(C.c_int32)]
    L.nsgpu_nonfinite_rows.restype = C.c_int64
    L.nsgpu_nonfinite_rows.argtypes = [vp]
    L.nsgpu_shard_range.restype = None
    L.nsgpu_shard_range.argtypes = [C.c_int32, C.c_int32, C.c_int32, C.POINTER(C.c_int32), C.POINTER(C.c_int32)]
    L.nsgpu_last_samples.restype = C.c_int
    L.nsgpu_last_samples.argtypes = [vp, vp, vp, vp, C.c_int64, C.POINTER(C.c_int64)]
    L.nsgpu_delete_lowest.restype = C.c_int
    L.nsgpu_delete_lowest.argtypes = [vp, vp, C.c_int32, C.c_int32, _pd, _pd, vp, vp, _pd, vp]
    L.nsgpu_live_cholesky.restype = C.c_int
    L.nsgpu_live_cholesky.argtypes = [vp, vp, C.c_int32, vp, vp]
    L.nsgpu_debug_philox.restype = C.c_int
    L.nsgpu_debug_philox.argtypes = [vp, vp, C.c_int32, C.POINTER(C.c_uint32), vp, vp]
    L.nsgpu_set_profiling.restype = C.c_int
    L.nsgpu_set_profiling.argtypes = [vp, C.c_int32]
    L.nsgpu_stage_times.restype = C.c_int
    L.nsgpu_stage_times.argtypes = [vp, _pd, C.POINTER(C.c_int64)]
    L.nsgpu_mlp_path.restype = C.c_int32
    L.nsgpu_mlp_path.argtypes = [vp, C.c_int32]
    L.nsgpu_launch_count.restype = C.c_int64
    L.nsgpu_launch_count.argtypes = [vp]
    _lib = L
    return L


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _ptr(a, typ):
    return a.ctypes.data_as(typ)


def _stream_ptr(stream=None):
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def shard_range(n_chains, rank, world):
    """(first, count) of the chains rank `rank` of `world` evolves (nsgpu_shard_range; host only)."""
    a, b = C.c_int32(0), C.c_int32(0)
    lib().nsgpu_shard_range(int(n_chains), int(rank), int(world), C.byref(a), C.byref(b))
    return a.value, b.value


class _RawBuffer:
    """a device (or host) pointer as a flat uint8 array for torch (zero copy)"""

    def __init__(self, ptr, nbytes, cuda):
        iface = {"shape": (int(nbytes),), "typestr": "|u1", "data": (int(ptr), False), "version": 2 if cuda else 3, "strides": None}
        if cuda:
            self.__cuda_array_interface__ = iface
        else:
            self.__array_interface__ = iface


def torch_allgather(device=None, group=None):
    """The exchange step of nsgpu_run_sharded on torch.distributed: `all_gather_into_tensor` straight on the
    library's buffers (NCCL for device pointers; `device=None` treats them as host pointers, for gloo tests).
    Returns a Python callable with the nsgpu_allgather_fn signature."""
    import torch
    import torch.distributed as dist

    def cb(user, send, recv, nbytes, stream):
        try:
            world = dist.get_world_size(group)
            if device is None:
                s = torch.from_numpy(np.asarray(_RawBuffer(send, nbytes, False)))
                r = torch.from_numpy(np.asarray(_RawBuffer(recv, nbytes * world, False)))
            else:
                s = torch.as_tensor(_RawBuffer(send, nbytes, True), device=f"cuda:{device}")
                r = torch.as_tensor(_RawBuffer(recv, nbytes * world, True), device=f"cuda:{device}")
            dist.all_gather_into_tensor(r, s, group=group)
            if device is not None:
                torch.cuda.synchronize(device)
            return 0
        except Exception as e:          # never let an exception cross the C boundary
            import sys
            print(f"nsgpu allgather failed: {e!r}", file=sys.stderr)
            return 1

    return cb


class Context:
    """nsgpu_create / nsgpu_destroy wrapper.  `wl` is a `workloads.Workload` with data and chol attached."""

    def __init__(self, wl, max_batch: int, device: int = 0, mlp: int = MLP_AUTO):
        L = lib()
        if wl.data is None or (wl.chol is None and wl.theory.kind != 4):
            raise ValueError("workload has no data vector / Cholesky factor attached")
        self._keep = []           # host arrays must outlive nsgpu_create only, kept anyway for clarity
        keep = self._keep.append
        D = wl.D
        prior = (_Prior1d * D)()
        for d in range(D):
            prior[d].kind, prior[d].p0, prior[d].p1 = int(wl.prior_kind[d]), float(wl.prior_p0[d]), float(wl.prior_p1[d])
        n_emu = len(wl.emulators)
        emus = (_Emulator * max(n_emu, 1))()
        for e, em in enumerate(wl.emulators):
            def arr_of(lst):
                arrs = [_f32(a) for a in lst]
                keep(arrs)
                ptrs = (_pf * len(arrs))(*[_ptr(a, _pf) for a in arrs])
                keep(ptrs)
                return ptrs
            x = emus[e]
            x.n_in, x.n_hidden, x.width, x.n_out, x.out_kind = em.n_in, em.n_hidden, em.width, em.n_out, em.out_kind
            x.W, x.b, x.alpha, x.beta = arr_of(em.W), arr_of(em.b), arr_of(em.alpha), arr_of(em.beta)
            for name in ("in_mean", "in_std", "out_mean", "out_std"):
                a = _f32(getattr(em, name)); keep(a)
                setattr(x, name, _ptr(a, _pf))
        th = wl.theory
        t = _Theory()
        t.kind = th.kind
        idx = np.ascontiguousarray(th.emu_in_idx, np.int32); cst = np.ascontiguousarray(th.emu_in_const, np.float64)
        keep(idx); keep(cst)
        t.n_theta_in = len(idx)
        t.emu_in_idx, t.emu_in_const = _ptr(idx, _pi), _ptr(cst, _pd)
        t.cal_index = th.cal_index
        t.ell_min = int(getattr(th, "ell_min", 2))
        if th.kind == 2:
            bp, bc, bv = (np.ascontiguousarray(th.bin_ptr, np.int32), np.ascontiguousarray(th.bin_col, np.int32),
                          _f32(th.bin_val))
            keep(bp); keep(bc); keep(bv)
            t.bin_ptr, t.bin_col, t.bin_val = _ptr(bp, _pi), _ptr(bc, _pi), _ptr(bv, _pf)
        if th.kind == 3:
            for name in ("n_z_emu", "n_z", "n_chi", "n_k", "n_ell", "n_tomo", "z_interp", "idx_omega_b", "idx_omega_cdm",
                         "idx_h", "idx_w0", "idx_wa", "idx_eta0", "idx_dz", "idx_ia", "idx_m", "n_ia_terms", "n_m_terms"):
                setattr(t, name, int(getattr(th, name)))
            t.z_max, t.k_min, t.k_max, t.nz_sigma = float(th.z_max), float(th.k_min), float(th.k_max), float(th.nz_sigma)
            ell = np.ascontiguousarray(th.ell, np.float64); nzm = np.ascontiguousarray(th.nz_mean, np.float64)
            keep(ell); keep(nzm)
            t.ell, t.nz_mean = _ptr(ell, _pd), _ptr(nzm, _pd)
        data = np.ascontiguousarray(wl.data, np.float64)
        chol = np.ascontiguousarray(wl.chol, np.float64) if wl.chol is not None else None
        self._h = C.c_void_p()
        self.D, self.n_data, self.max_batch, self.device = D, wl.n_data, int(max_batch), int(device)
        self.rows = th.n_z_emu if th.kind == 3 else 1
        self.n_out = wl.emulators[0].n_out if n_emu else 0
        st = L.nsgpu_create(C.byref(self._h), D, prior, n_emu, emus, C.byref(t), wl.n_data, _ptr(data, _pd),
                            _ptr(chol, _pd) if chol is not None else None, int(max_batch), int(device), int(mlp))
        if st != OK:
            msg = L.nsgpu_last_error(None)
            self._h = C.c_void_p()
            raise NsgpuError(st, msg.decode() if msg else "")

    # -- helpers ---------------------------------------------------------------------------------
    def _check(self, st, allow=()):
        if st != OK and st not in allow:
            msg = lib().nsgpu_last_error(self._h)
            raise NsgpuError(st, msg.decode() if msg else "")
        return st

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            lib().nsgpu_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def _dev(self):
        import torch
        return torch.device("cuda", self.device)

    @staticmethod
    def _p(t):
        return C.c_void_p(t.data_ptr())

    def _theta_arg(self, theta):
        import torch
        assert theta.is_cuda and theta.dtype == torch.float32 and theta.is_contiguous() and theta.shape[-1] == self.D
        return theta

    # -- entry points (same names as the C ABI, minus the prefix) ------------------------------------
    def prior_transform(self, u, stream=None):
        import torch
        u = self._theta_arg(u)
        out = torch.empty_like(u)
        self._check(lib().nsgpu_prior_transform(self._h, self._p(u), u.shape[0], self._p(out), _stream_ptr(stream)))
        return out

    def loglike_batch(self, theta, out=None, stream=None):
        import torch
        theta = self._theta_arg(theta)
        B = theta.shape[0]
        if out is None:
            out = torch.empty(B, dtype=torch.float64, device=theta.device)
        self._check(lib().nsgpu_loglike_batch(self._h, self._p(theta), B, self._p(out), _stream_ptr(stream)))
        return out

    def loglike_batch_host(self, theta_host: np.ndarray, out: Optional[np.ndarray] = None) -> np.ndarray:
        theta_host = _f32(theta_host)
        B = theta_host.shape[0]
        if out is None:
            out = np.empty(B, np.float64)
        self._check(lib().nsgpu_loglike_batch_host(self._h, theta_host.ctypes.data_as(C.c_void_p), B,
                                                   out.ctypes.data_as(C.c_void_p)))
        return out

    def emulate_batch(self, theta, emu=0, stream=None):
        import torch
        theta = self._theta_arg(theta)
        B = theta.shape[0]
        out = torch.empty((B, self.rows, self.n_out), dtype=torch.float32, device=theta.device)
        self._check(lib().nsgpu_emulate_batch(self._h, emu, self._p(theta), B, self._p(out), _stream_ptr(stream)))
        return out

    def theory_batch(self, theta, stream=None):
        import torch
        theta = self._theta_arg(theta)
        B = theta.shape[0]
        out = torch.empty((B, self.n_data), dtype=torch.float64, device=theta.device)
        self._check(lib().nsgpu_theory_batch(self._h, self._p(theta), B, self._p(out), _stream_ptr(stream)))
        return out

    def slice_step(self, u_live, logL_live, start_idx, logL_star, n_steps, seed=1, iteration=1, stream=None):
        import torch
        u_live = self._theta_arg(u_live)
        assert logL_live.dtype == torch.float64 and start_idx.dtype == torch.int32
        n_live, n_chains = u_live.shape[0], start_idx.shape[0]
        u_out = torch.empty((n_chains, self.D), dtype=torch.float32, device=u_live.device)
        l_out = torch.empty(n_chains, dtype=torch.float64, device=u_live.device)
        ne = C.c_int64(0)
        self._check(lib().nsgpu_slice_step(self._h, self._p(u_live), self._p(logL_live), n_live, self._p(start_idx),
                                           n_chains, float(logL_star), int(n_steps), int(seed), int(iteration),
                                           self._p(u_out), self._p(l_out), C.byref(ne), _stream_ptr(stream)))
        return u_out, l_out, ne.value

    def sampler_counters(self):
        """(n_failed_moves, n_rounds) of the last slice_step on this context."""
        a, b = C.c_int64(0), C.c_int64(0)
        self._check(lib().nsgpu_sampler_counters(self._h, C.byref(a), C.byref(b)))
        return a.value, b.value

    def delete_lowest(self, logL_live, k, logX=0.0, logZ=-np.inf, stream=None):
        import torch
        n = logL_live.shape[0]
        dead = torch.empty(k, dtype=torch.int32, device=logL_live.device)
        logw = torch.empty(k, dtype=torch.float64, device=logL_live.device)
        lx, lz, ls = C.c_double(logX), C.c_double(logZ), C.c_double(0.0)
        self._check(lib().nsgpu_delete_lowest(self._h, self._p(logL_live), n, k, C.byref(lx), C.byref(lz), self._p(dead),
                                              self._p(logw), C.byref(ls), _stream_ptr(stream)))
        return dead, logw, lx.value, lz.value, ls.value

    def live_cholesky(self, u_live, stream=None):
        import torch
        u_live = self._theta_arg(u_live)
        out = torch.empty((self.D, self.D), dtype=torch.float64, device=u_live.device)
        self._check(lib().nsgpu_live_cholesky(self._h, self._p(u_live), u_live.shape[0], self._p(out), _stream_ptr(stream)))
        return out

    def debug_philox(self, ctr, key, stream=None):
        import torch
        assert ctr.dtype == torch.int32 or ctr.dtype == torch.uint32
        n = ctr.shape[0]
        out = torch.empty_like(ctr)
        k = (C.c_uint32 * 2)(int(key[0]), int(key[1]))
        self._check(lib().nsgpu_debug_philox(self._h, self._p(ctr), n, k, self._p(out), _stream_ptr(stream)))
        return out

    def run(self, n_live, n_delete, n_steps, stop_frac=1e-3, max_iter=100000, seed=1, return_samples=True):
        """nsgpu_run -> dict(logZ, logZ_err, logZ_err_analytic, H, n_iter, n_dead, n_like_evals, n_rounds,
        n_failed_moves, seconds, converged[, theta, logL, logw])."""
        o = _RunOpts(int(n_live), int(n_delete), int(n_steps), float(stop_frac), int(max_iter), int(seed))
        r = _Result()
        ns = C.c_int64(0)
        st = self._check(lib().nsgpu_run(self._h, C.byref(o), C.byref(r), None, None, None, 0, C.byref(ns)),
                         allow=(ENOCONV,))
        out = {f: getattr(r, f) for f, _ in _Result._fields_}
        out["converged"] = st == OK
        if return_samples:
            n = ns.value
            th = np.empty((n, self.D), np.float32); ll = np.empty(n, np.float64); lw = np.empty(n, np.float64)
            self._check(lib().nsgpu_last_samples(self._h, th.ctypes.data_as(C.c_void_p), ll.ctypes.data_as(C.c_void_p),
                                                 lw.ctypes.data_as(C.c_void_p), n, C.byref(ns)))
            out.update(theta=th, logL=ll, logw=lw, n_samples=n)
        return out

    def run_multi(self, n_live, n_delete, n_steps, seeds, stop_frac=1e-3, max_iter=100000, return_samples=True):
        """nsgpu_run_multi: one dict per seed, each equal to `run(..., seed=s)`; the runs share every likelihood batch."""
        seeds = [int(x) for x in seeds]
        R = len(seeds)
        o = _RunOpts(int(n_live), int(n_delete), int(n_steps), float(stop_frac), int(max_iter), 0)
        res = (_Result * R)()
        sd = (C.c_uint64 * R)(*seeds)
        st = self._check(lib().nsgpu_run_multi(self._h, C.byref(o), R, sd, res), allow=(ENOCONV,))
        outs = []
        for r in range(R):
            out = {f: getattr(res[r], f) for f, _ in _Result._fields_}
            out["seed"] = seeds[r]
            out["converged"] = st == OK or out["n_iter"] < int(max_iter)
            if return_samples:
                ns = C.c_int64(0)
                self._check(lib().nsgpu_multi_samples(self._h, r, None, None, None, 0, C.byref(ns)))
                n = ns.value
                th = np.empty((n, self.D), np.float32); ll = np.empty(n, np.float64); lw = np.empty(n, np.float64)
                self._check(lib().nsgpu_multi_samples(self._h, r, th.ctypes.data_as(C.c_void_p), ll.ctypes.data_as(C.c_void_p),
                                                      lw.ctypes.data_as(C.c_void_p), n, C.byref(ns)))
                out.update(theta=th, logL=ll, logw=lw, n_samples=n)
            outs.append(out)
        return outs

    def logz_error_noalloc(self, dead_logL, live_logL, n_delete, seed, stream=None):
        """nsgpu_logz_error_noalloc -> (logZ_err, the 1000 simulated log Z); host arrays in, nothing allocated on the GPU."""
        dead = np.ascontiguousarray(dead_logL, np.float64); live = np.ascontiguousarray(live_logL, np.float64)
        err = C.c_double(0.0); sims = np.zeros(1000, np.float64)
        self._check(lib().nsgpu_logz_error_noalloc(self._h, _ptr(dead, _pd), int(dead.shape[0]), _ptr(live, _pd), int(live.shape[0]),
                                                   int(n_delete), int(seed), C.byref(err), _ptr(sims, _pd), _stream_ptr(stream)))
        return err.value, sims

    def run_sharded(self, n_live, n_delete, n_steps, stop_frac=1e-3, max_iter=100000, seed=1, rank=None, world=None,
                    allgather=None, return_samples=True):
        """nsgpu_run_sharded: the same run with the k chains of an iteration split over `world` processes (one GPU
        each, every rank calls this with the same arguments).  `allgather` defaults to torch.distributed
        (`torch_allgather`, NCCL on device buffers); every rank gets the same result as `run`."""
        import torch.distributed as dist
        if rank is None:
            rank, world = dist.get_rank(), dist.get_world_size()
        cb = allgather if allgather is not None else torch_allgather(self.device)
        fn = ALLGATHER_FN(cb)
        o = _RunOpts(int(n_live), int(n_delete), int(n_steps), float(stop_frac), int(max_iter), int(seed))
        r = _Result()
        ns = C.c_int64(0)
        st = self._check(lib().nsgpu_run_sharded(self._h, C.byref(o), int(rank), int(world), fn, None, C.byref(r),
                                                 None, None, None, 0, C.byref(ns)), allow=(ENOCONV,))
        out = {f: getattr(r, f) for f, _ in _Result._fields_}
        out["converged"] = st == OK
        if return_samples:
            n = ns.value
            th = np.empty((n, self.D), np.float32); ll = np.empty(n, np.float64); lw = np.empty(n, np.float64)
            self._check(lib().nsgpu_last_samples(self._h, th.ctypes.data_as(C.c_void_p), ll.ctypes.data_as(C.c_void_p),
                                                 lw.ctypes.data_as(C.c_void_p), n, C.byref(ns)))
            out.update(theta=th, logL=ll, logw=lw, n_samples=n)
        return out

    STAGES = ["mlp_first", "mlp_hidden", "mlp_out", "shear_project", "cmb_bin", "chi2", "slice_round", "copy_model"]

    def set_profiling(self, on: bool):
        self._check(lib().nsgpu_set_profiling(self._h, 1 if on else 0))

    def stage_times(self):
        """{stage: (total_ms, launches_timed)} since the last call (synchronises the device)."""
        ms = (C.c_double * 8)(); cnt = (C.c_int64 * 8)()
        self._check(lib().nsgpu_stage_times(self._h, ms, cnt))
        return {n: (ms[i], cnt[i]) for i, n in enumerate(self.STAGES)}

    def mlp_path(self, emu=0):
        return lib().nsgpu_mlp_path(self._h, emu)

    def clock_mark(self, stream=None):
        """enqueue a clock mark on the stream (see nsgpu_clock_mark)"""
        self._check(lib().nsgpu_clock_mark(self._h, _stream_ptr(stream)))

    def clock_marks_read(self):
        """(sm_mhz, t_ms) for each interval between consecutive marks; clears the marks."""
        mhz = np.zeros(512, np.float64); t = np.zeros(512, np.float64); n = C.c_int32(0)
        self._check(lib().nsgpu_clock_marks_read(self._h, _ptr(mhz, _pd), _ptr(t, _pd), 512, C.byref(n)))
        return mhz[:n.value], t[:n.value]

    def nonfinite_rows(self):
        return lib().nsgpu_nonfinite_rows(self._h)

    def launch_count(self):
        return lib().nsgpu_launch_count(self._h)
