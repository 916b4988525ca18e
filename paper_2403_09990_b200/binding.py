"""Thin ctypes binding over libclosure_b200.so (include/closure.h): argument marshalling only.

Every step of the path runs inside the library's CUDA kernels / host miniball; torch is used
for device memory and streams.  There is no CPU fallback: if the shared library is missing or
cannot be loaded, importing the entry points raises.
"""
from __future__ import annotations

import ctypes
import os
from ctypes import (POINTER, Structure, byref, c_char_p, c_double, c_int, c_longlong, c_ubyte,
                    c_ulonglong, c_void_p)

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libclosure_b200.so")

OK, EINVAL, EINIT, ENOINIT, ECUDA, ENOMEM, EUNSUPPORTED, ETOOLARGE = 0, -1, -2, -3, -4, -5, -6, -7
COMPACT_STATIC_MAX = 8388608

EXPORTS = [
    "closure_default_params", "closure_create", "closure_set_params", "closure_set_pivot", "closure_set_init",
    "closure_sample_range", "closure_sample", "closure_sample_batch", "closure_compact", "closure_compact_static", "closure_megb",
    "closure_init_sample", "closure_init_from_trials", "closure_run", "closure_enable_stats", "closure_get_stats", "closure_alu_peak", "closure_miniball_host",
    "closure_last_error", "closure_strerror", "closure_abi_version", "closure_destroy",
]


class ClosureParams(Structure):
    _fields_ = [("mode", c_int), ("n_p", c_int), ("n_p_star", c_int), ("n_t", c_int),
                ("omega0", c_double), ("v0", c_double), ("gamma", c_double), ("t_p", c_double),
                ("theta_p", c_double), ("precision", c_int), ("flags", c_int)]


class MegbResult(Structure):
    _fields_ = [("R", c_double * 9), ("t", c_double * 3), ("rot_radius", c_double),
                ("trans_radius", c_double), ("rot_support", c_longlong * 5),
                ("trans_support", c_longlong * 4), ("n_rot_support", c_int), ("n_trans_support", c_int),
                ("host_seconds", c_double), ("d2h_bytes", c_double), ("max_pivot_seconds", c_double),
                ("pivots", c_int), ("pad_", c_int), ("prepare_seconds", c_double)]


class Stats(Structure):
    _fields_ = [("perturb_pairs", c_ulonglong), ("ladder_pairs", c_ulonglong),
                ("perturb_setups", c_ulonglong), ("ladder_setups", c_ulonglong),
                ("accepted_steps", c_ulonglong), ("walker_steps", c_ulonglong),
                ("perturb_pairs_f32", c_ulonglong), ("ladder_pairs_f32", c_ulonglong),
                ("fallback_steps", c_ulonglong), ("verified_rungs", c_ulonglong),
                ("setup_cycles", c_ulonglong), ("total_cycles", c_ulonglong),
                ("threshold_probes", c_ulonglong), ("survivors", c_ulonglong), ("reserved_", c_ulonglong),
                ("threshold_failures", c_ulonglong)]


class ClosureError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"closure status {status}: {message}")
        self.status = status


_lib = None


def load_library():
    """Load libclosure_b200.so; fail loudly if it has not been built (no fallback)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            f"{LIB_PATH} is missing: build it with `python -m paper_2403_09990_b200.build` "
            "(nvcc, sm_100a).  There is no CPU fallback.")
    L = ctypes.CDLL(LIB_PATH)
    L.closure_default_params.argtypes = [c_int, POINTER(ClosureParams)]
    L.closure_create.argtypes = [c_int, POINTER(c_double), c_int, POINTER(c_double), POINTER(c_double),
                                 POINTER(ClosureParams), POINTER(c_void_p)]
    L.closure_set_params.argtypes = [c_void_p, POINTER(ClosureParams)]
    L.closure_set_pivot.argtypes = [c_void_p, POINTER(c_double)]
    L.closure_set_init.argtypes = [c_void_p, POINTER(c_double), c_int, POINTER(c_double)]
    L.closure_sample_range.argtypes = [c_void_p, c_longlong, c_longlong, c_int, c_ulonglong, c_void_p,
                                       c_void_p, c_void_p, c_void_p]
    L.closure_sample.argtypes = [c_void_p, c_longlong, c_int, c_ulonglong, c_void_p, c_void_p, c_void_p]
    L.closure_sample_batch.argtypes = [POINTER(c_void_p), c_int, c_longlong, c_int, POINTER(c_ulonglong),
                                       c_void_p, c_void_p, c_void_p]
    L.closure_compact.argtypes = [c_void_p, c_void_p, c_void_p, c_longlong, c_void_p, c_void_p, c_void_p]
    L.closure_compact_static.argtypes = [c_void_p, c_void_p, c_longlong, c_void_p, c_void_p, c_void_p]
    L.closure_megb.argtypes = [c_void_p, c_void_p, c_longlong, POINTER(MegbResult), c_void_p]
    L.closure_run.argtypes = [c_void_p, c_longlong, c_int, c_ulonglong, POINTER(MegbResult),
                              POINTER(c_longlong), c_void_p]
    L.closure_enable_stats.argtypes = [c_void_p, c_int]
    L.closure_get_stats.argtypes = [c_void_p, POINTER(Stats)]
    L.closure_alu_peak.argtypes = [c_int, POINTER(c_double), POINTER(c_double), c_void_p]
    L.closure_init_sample.argtypes = [c_void_p, c_longlong, c_longlong, c_ulonglong, c_void_p, c_void_p, c_void_p]
    L.closure_init_from_trials.argtypes = [c_void_p, c_longlong, c_ulonglong, c_int, POINTER(c_int), c_void_p]
    L.closure_miniball_host.argtypes = [POINTER(c_double), c_longlong, c_int, POINTER(c_double),
                                        POINTER(c_double), POINTER(c_longlong), POINTER(c_int)]
    L.closure_last_error.argtypes = [c_void_p]
    L.closure_last_error.restype = c_char_p
    L.closure_strerror.argtypes = [c_int]
    L.closure_strerror.restype = c_char_p
    L.closure_abi_version.restype = c_int
    L.closure_destroy.argtypes = [c_void_p]
    L.closure_destroy.restype = None
    _lib = L
    return L


def _dp(a: np.ndarray):
    return a.ctypes.data_as(POINTER(c_double))


def _stream_ptr(stream) -> c_void_p:
    if stream is None:
        import torch
        stream = torch.cuda.current_stream()
    return c_void_p(int(getattr(stream, "cuda_stream", stream)))


def make_params(p) -> ClosureParams:
    """From any object with the paper's parameter names (e.g. instances.WalkParams)."""
    return ClosureParams(int(p.mode), int(p.n_p), int(p.n_p_star), int(p.n_t), float(p.omega0),
                         float(p.v0), float(p.gamma), float(p.t_p), float(p.theta_p),
                         int(getattr(p, "precision", 64)), int(getattr(p, "flags", 0)))


def closure_default_params(residual_type: int) -> ClosureParams:
    p = ClosureParams()
    rc = load_library().closure_default_params(residual_type, byref(p))
    if rc != OK:
        raise ClosureError(rc, closure_strerror(rc))
    return p


def closure_strerror(status: int) -> str:
    return load_library().closure_strerror(status).decode()


def closure_abi_version() -> int:
    return load_library().closure_abi_version()


def closure_alu_peak(precision: int = 64, stream=None) -> tuple[float, float]:
    f, s = c_double(0), c_double(0)
    rc = load_library().closure_alu_peak(precision, byref(f), byref(s), _stream_ptr(stream))
    if rc != OK:
        raise ClosureError(rc, closure_strerror(rc))
    return f.value, s.value


def closure_miniball_host(points) -> tuple[np.ndarray, float, np.ndarray]:
    """Host-only Gaertner miniball of an (n, d) array, d <= 4 -> (center, radius, support)."""
    pts = np.ascontiguousarray(points, dtype=np.float64)
    n, d = pts.shape
    c = np.zeros(d)
    r = c_double(0)
    sup = np.zeros(5, dtype=np.int64)
    ns = c_int(0)
    rc = load_library().closure_miniball_host(_dp(pts), n, d, _dp(c), byref(r),
                                              sup.ctypes.data_as(POINTER(c_longlong)), byref(ns))
    if rc != OK:
        raise ClosureError(rc, closure_strerror(rc))
    return c, r.value, sup[:ns.value].copy()


def _as_dict(r: MegbResult) -> dict:
    return dict(R=np.array(r.R).reshape(3, 3), t=np.array(r.t), rot_radius=r.rot_radius,
                trans_radius=r.trans_radius, rot_support=np.array(r.rot_support[:r.n_rot_support]),
                trans_support=np.array(r.trans_support[:r.n_trans_support]), host_seconds=r.host_seconds,
                d2h_bytes=int(r.d2h_bytes), max_pivot_seconds=r.max_pivot_seconds, pivots=int(r.pivots),
                prepare_seconds=r.prepare_seconds)


class Closure:
    """Owns one closure_t handle; methods carry the C entry points' names."""

    def __init__(self, residual_type: int, measurements, betas, intrinsics=None, params=None):
        L = load_library()
        meas = np.ascontiguousarray(measurements, dtype=np.float64)
        bet = np.ascontiguousarray(betas, dtype=np.float64).reshape(-1)
        K = None if intrinsics is None else np.ascontiguousarray(intrinsics, dtype=np.float64)
        P = params if isinstance(params, ClosureParams) else (
            closure_default_params(residual_type) if params is None else make_params(params))
        self._h = c_void_p()
        self.residual_type = residual_type
        self.n = int(meas.shape[0]) if meas.ndim == 2 else 0
        rc = L.closure_create(residual_type, _dp(meas), self.n, _dp(bet), None if K is None else _dp(K),
                              byref(P), byref(self._h))
        if rc != OK:
            self._h = c_void_p()
            raise ClosureError(rc, closure_strerror(rc))
        self.params = P
        self.mean_pose = None

    @classmethod
    def closure_create(cls, inst, params=None) -> "Closure":
        """From an instances.Instance-like object."""
        return cls(inst.residual_type, inst.measurements, inst.betas, inst.intrinsics,
                   inst.params if params is None else params)

    def _check(self, rc: int):
        if rc != OK:
            msg = load_library().closure_last_error(self._h).decode() or closure_strerror(rc)
            raise ClosureError(rc, msg)

    def closure_set_params(self, params):
        P = params if isinstance(params, ClosureParams) else make_params(params)
        self._check(load_library().closure_set_params(self._h, byref(P)))
        self.params = P

    def closure_set_pivot(self, pivot):
        c = np.ascontiguousarray(pivot, dtype=np.float64).reshape(3)
        self._check(load_library().closure_set_pivot(self._h, _dp(c)))

    def closure_set_init(self, poses) -> np.ndarray:
        S0 = np.ascontiguousarray(poses, dtype=np.float64).reshape(-1, 12)
        mean = np.zeros(12)
        self._check(load_library().closure_set_init(self._h, _dp(S0), S0.shape[0], _dp(mean)))
        self.mean_pose = (mean[:9].reshape(3, 3).copy(), mean[9:].copy())
        return mean

    def closure_init_sample(self, num_trials: int, seed: int, out_poses=None, out_ok=None, stream=None, *,
                            trial_begin: int = 0):
        """Step I trials -> (poses (T,12) f64 cuda tensor, ok (T,) u8 cuda tensor)."""
        import torch
        dev = torch.device("cuda")
        if out_poses is None:
            out_poses = torch.empty((num_trials, 12), dtype=torch.float64, device=dev)
        if out_ok is None:
            out_ok = torch.empty((num_trials,), dtype=torch.uint8, device=dev)
        self._check(load_library().closure_init_sample(
            self._h, trial_begin, num_trials, seed, c_void_p(out_poses.data_ptr()), c_void_p(out_ok.data_ptr()),
            _stream_ptr(stream)))
        return out_poses, out_ok

    def closure_init_from_trials(self, num_trials: int, seed: int, max_poses: int = 128, stream=None) -> int:
        """Step I end to end (trials, compaction, closure_set_init) -> |S_0|."""
        n0 = c_int(0)
        self._check(load_library().closure_init_from_trials(self._h, num_trials, seed, max_poses, byref(n0),
                                                            _stream_ptr(stream)))
        return int(n0.value)

    def closure_sample(self, num_walkers: int, num_steps: int, seed: int, out_samples=None,
                       out_on_boundary=None, stream=None, *, walker_begin: int = 0, trace: bool = False):
        """-> (samples (W,12) f64 cuda tensor, on_boundary (W,) u8 cuda tensor[, trace (W,S) i32])."""
        import torch
        dev = torch.device("cuda")
        if out_samples is None:
            out_samples = torch.empty((num_walkers, 12), dtype=torch.float64, device=dev)
        if out_on_boundary is None:
            out_on_boundary = torch.empty((num_walkers,), dtype=torch.uint8, device=dev)
        tr = torch.zeros((num_walkers, num_steps), dtype=torch.int32, device=dev) if trace else None
        self._check(load_library().closure_sample_range(
            self._h, walker_begin, num_walkers, num_steps, seed, c_void_p(out_samples.data_ptr()),
            c_void_p(out_on_boundary.data_ptr()), c_void_p(tr.data_ptr()) if trace else None,
            _stream_ptr(stream)))
        return (out_samples, out_on_boundary, tr) if trace else (out_samples, out_on_boundary)

    def closure_compact(self, samples, flags, out_compacted=None, out_count=None, stream=None):
        import torch
        n = int(flags.shape[0])
        if out_compacted is None:
            out_compacted = torch.empty((max(n, 1), 12), dtype=torch.float64, device=samples.device)
        if out_count is None:
            out_count = torch.zeros((1,), dtype=torch.int64, device=samples.device)
        self._check(load_library().closure_compact(
            self._h, c_void_p(samples.data_ptr()), c_void_p(flags.data_ptr()), n,
            c_void_p(out_compacted.data_ptr()), c_void_p(out_count.data_ptr()), _stream_ptr(stream)))
        return out_compacted, out_count

    def closure_megb(self, samples, count: int | None = None, stream=None) -> dict:
        r = MegbResult()
        cnt = int(samples.shape[0]) if count is None else int(count)
        self._check(load_library().closure_megb(self._h, c_void_p(samples.data_ptr()), cnt, byref(r),
                                                _stream_ptr(stream)))
        return _as_dict(r)

    def closure_run(self, num_walkers: int, num_steps: int, seed: int, stream=None) -> dict:
        r = MegbResult()
        cnt = c_longlong(0)
        self._check(load_library().closure_run(self._h, num_walkers, num_steps, seed, byref(r), byref(cnt),
                                               _stream_ptr(stream)))
        out = _as_dict(r)
        out["count"] = cnt.value
        return out

    def closure_enable_stats(self, on: bool = True):
        self._check(load_library().closure_enable_stats(self._h, int(on)))

    def closure_get_stats(self) -> dict:
        s = Stats()
        self._check(load_library().closure_get_stats(self._h, byref(s)))
        return {k: int(getattr(s, k)) for k, _ in Stats._fields_}

    def closure_destroy(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            load_library().closure_destroy(self._h)
            self._h = c_void_p()

    def __del__(self):
        try:
            self.closure_destroy()
        except Exception:
            pass


def closure_compact_static(samples, flags, out_compacted, out_count, stream=None):
    """closure_compact on the library's static scratch: allocates nothing (the caller passes every buffer), at most
    COMPACT_STATIC_MAX records; calls on one device must not overlap."""
    rc = load_library().closure_compact_static(c_void_p(samples.data_ptr()), c_void_p(flags.data_ptr()), int(flags.shape[0]),
                                               c_void_p(out_compacted.data_ptr()), c_void_p(out_count.data_ptr()),
                                               _stream_ptr(stream))
    if rc != OK:
        raise ClosureError(rc, closure_strerror(rc))
    return out_compacted, out_count


def closure_sample_batch(handles: list[Closure], walkers_per_instance: int, num_steps: int, seeds,
                         out_samples=None, out_on_boundary=None, stream=None):
    import torch
    nb = len(handles)
    dev = torch.device("cuda")
    if out_samples is None:
        out_samples = torch.empty((nb, walkers_per_instance, 12), dtype=torch.float64, device=dev)
    if out_on_boundary is None:
        out_on_boundary = torch.empty((nb, walkers_per_instance), dtype=torch.uint8, device=dev)
    hs = (c_void_p * nb)(*[h._h.value for h in handles])
    sd = (c_ulonglong * nb)(*[int(s) for s in seeds])
    rc = load_library().closure_sample_batch(hs, nb, walkers_per_instance, num_steps, sd,
                                             c_void_p(out_samples.data_ptr()),
                                             c_void_p(out_on_boundary.data_ptr()), _stream_ptr(stream))
    handles[0]._check(rc)
    return out_samples, out_on_boundary
