"""CPU oracle for the CLOSURE boundary walk + miniball (arXiv 2403.09990).

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only ``tests/``, ``__graft_entry__.smoke()`` and
the ``cpu_baseline`` / ``--impl reference`` legs of ``bench.py`` may import this package.
It imports nothing from ``paper_2403_09990_b200`` and the CUDA path imports nothing from
here.  Instances are passed in as plain arrays (any object with ``residual_type``,
``measurements``, ``betas``, ``intrinsics`` works).

The arithmetic lives in ``closure_oracle.c`` / ``miniball_oracle.c`` (plain C99, fp64, one
pose evaluation at a time, citing PAPER.md line by line); this file only builds them with
gcc and marshals numpy arrays through ctypes.  The one numeric step done here is the mean
rotation ``proj_SO(3)(sum R_j)`` (Alg. 2 l.3), through numpy's SVD.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from ctypes import POINTER, c_double, c_int, c_int32, c_int64, c_ubyte, c_uint32, c_uint64

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_BUILD = os.path.join(_HERE, "_build")
_LIB_PATH = os.path.join(_BUILD, "liboracle.so")
_SOURCES = [os.path.join(_HERE, "closure_oracle.c"), os.path.join(_HERE, "miniball_oracle.c")]
_lib = None


class _Params(ctypes.Structure):
    _fields_ = [("mode", c_int), ("n_p", c_int), ("n_p_star", c_int), ("n_t", c_int),
                ("omega0", c_double), ("v0", c_double), ("gamma", c_double),
                ("t_p", c_double), ("theta_p", c_double), ("vel_scale", c_double * 9), ("pivot", c_double * 3)]


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (no FMA contraction, no fast-math)."""
    os.makedirs(_BUILD, exist_ok=True)
    stale = force or not os.path.exists(_LIB_PATH) or any(
        os.path.getmtime(s) > os.path.getmtime(_LIB_PATH) for s in _SOURCES)
    if stale:
        tmp = _LIB_PATH + f".{os.getpid()}.tmp"
        cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-ffp-contract=off", "-fno-fast-math",
               "-shared", "-fPIC", "-o", tmp] + _SOURCES + ["-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB_PATH)
    return _LIB_PATH


def _dp(a):
    return a.ctypes.data_as(POINTER(c_double))


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        L.ora_u32_to_pm1.restype = c_double
        L.ora_u32_to_pm1.argtypes = [c_uint32]
        L.ora_residual_sq.restype = c_double
        L.ora_margin.restype = c_double
        L.ora_in_purse.restype = c_int
        L.ora_num_constraints.restype = c_int
        L.ora_walk.restype = c_int
        L.ora_compact.restype = c_int64
        L.ora_meb_brute.restype = c_int
        L.ora_meb_welzl.restype = c_int
        L.ora_megb.restype = c_int
        _lib = L
    return _lib


def _f64(a, shape=None):
    a = np.ascontiguousarray(np.asarray(a, dtype=np.float64))
    if shape is not None:
        a = a.reshape(shape)
    return a


def _inst_arrays(inst):
    meas = _f64(inst.measurements)
    betas = _f64(inst.betas).reshape(-1)
    K = _f64(inst.intrinsics if inst.intrinsics is not None else np.zeros(4)).reshape(4)
    n = meas.shape[0]
    assert betas.shape[0] == lib().ora_num_constraints(int(inst.residual_type), n)
    return int(inst.residual_type), n, meas, betas, K


# ------------------------------------------------------------------ primitives

def philox4x32_10(ctr, key) -> np.ndarray:
    c = np.asarray(ctr, dtype=np.uint32).copy()
    k = np.asarray(key, dtype=np.uint32).copy()
    out = np.zeros(4, dtype=np.uint32)
    lib().ora_philox4x32_10(c.ctypes.data_as(POINTER(c_uint32)), k.ctypes.data_as(POINTER(c_uint32)),
                            out.ctypes.data_as(POINTER(c_uint32)))
    return out


def u32_to_pm1(x: int) -> float:
    return float(lib().ora_u32_to_pm1(c_uint32(int(x))))


def exp_so3(phi) -> np.ndarray:
    p = _f64(phi, 3)
    R = np.zeros(9)
    lib().ora_exp_so3(_dp(p), _dp(R))
    return R.reshape(3, 3)


def residual_sq(inst, c: int, R, t) -> float:
    ty, n, meas, betas, K = _inst_arrays(inst)
    R = _f64(R, 9); t = _f64(t, 3)
    return float(lib().ora_residual_sq(c_int(ty), c_int(c), _dp(meas), _dp(K), _dp(R), _dp(t)))


def in_purse(inst, R, t) -> bool:
    ty, n, meas, betas, K = _inst_arrays(inst)
    R = _f64(R, 9); t = _f64(t, 3)
    return bool(lib().ora_in_purse(c_int(ty), c_int(n), _dp(meas), _dp(betas), _dp(K), _dp(R), _dp(t)))


def margin(inst, R, t) -> float:
    ty, n, meas, betas, K = _inst_arrays(inst)
    R = _f64(R, 9); t = _f64(t, 3)
    return float(lib().ora_margin(c_int(ty), c_int(n), _dp(meas), _dp(betas), _dp(K), _dp(R), _dp(t)))


def mean_pose(S0) -> tuple[np.ndarray, np.ndarray]:
    """R_bar = proj_SO(3)(sum_j R_j), t_bar = mean t_j (Alg. 2 l.3-4)."""
    S0 = _f64(S0).reshape(-1, 12)
    M = S0[:, :9].reshape(-1, 3, 3).sum(axis=0)
    U, _, Vt = np.linalg.svd(M)
    D = np.diag([1.0, 1.0, float(np.sign(np.linalg.det(U @ Vt)))])
    return U @ D @ Vt, S0[:, 9:].mean(axis=0)


def pca_velocity_scale(S0) -> np.ndarray:
    """S = sqrtm(Cov(S_t0)) / sqrt(lambda_max): the centre velocity is rescaled by the relative spread of the
    initial translations along their principal axes ("rescale the center velocity based
    on the expansion of S_t0 on 3 PCA weights"; R-23).  Identity for fewer than two poses or no spread."""
    t = _f64(S0).reshape(-1, 12)[:, 9:]
    if t.shape[0] < 2:
        return np.eye(3)
    d = t - t.mean(axis=0)
    C = d.T @ d / t.shape[0]
    lam, U = np.linalg.eigh(C)
    lam = np.clip(lam, 0.0, None)
    if not lam.max() > 0.0:
        return np.eye(3)
    return (U * np.sqrt(lam / lam.max())) @ U.T


# ------------------------------------------------------------------ the walk

def walk(inst, params, S0, walker_ids, n_steps: int, seed: int, *, trace: bool = False,
         n_threads: int = 1, mean=None):
    """Run Alg. 2 / Alg. A8 for the listed walkers.

    Returns (samples (W,12), on_boundary (W,) uint8[, trace (W,S) int32, slack (W,S) f64]).
    """
    ty, n, meas, betas, K = _inst_arrays(inst)
    S0 = _f64(S0).reshape(-1, 12)
    Rbar, tbar = mean_pose(S0) if mean is None else mean
    Rbar = _f64(Rbar, 9); tbar = _f64(tbar, 3)
    ids = np.ascontiguousarray(np.asarray(walker_ids, dtype=np.int64)).reshape(-1)
    W = ids.shape[0]
    # flag 64 = CLOSURE_FLAG_PCA_VELOCITY: the PCA normalisation of the centre velocity (R-23)
    scale = pca_velocity_scale(S0) if (int(getattr(params, "flags", 0)) & 64) else np.eye(3)
    P = _Params(int(params.mode), int(params.n_p), int(params.n_p_star), int(params.n_t),
                float(params.omega0), float(params.v0), float(params.gamma),
                float(params.t_p), float(params.theta_p), (c_double * 9)(*scale.reshape(9)),
                (c_double * 3)(*[float(x) for x in getattr(params, "pivot", (0.0, 0.0, 0.0))]))
    samples = np.zeros((W, 12))
    flags = np.zeros(W, dtype=np.uint8)
    tr = np.zeros((W, n_steps), dtype=np.int32) if trace else None
    sl = np.zeros((W, n_steps)) if trace else None
    rc = lib().ora_walk(
        c_int(ty), c_int(n), _dp(meas), _dp(betas), _dp(K), ctypes.byref(P), _dp(S0),
        c_int(S0.shape[0]), _dp(Rbar), _dp(tbar), ids.ctypes.data_as(POINTER(c_int64)), c_int64(W),
        c_int(n_steps), c_uint64(seed), _dp(samples), flags.ctypes.data_as(POINTER(c_ubyte)),
        tr.ctypes.data_as(POINTER(c_int32)) if trace else None,
        _dp(sl) if trace else None, c_int(n_threads))
    if rc != 0:
        raise ValueError("ora_walk: bad arguments")
    return (samples, flags, tr, sl) if trace else (samples, flags)


def compact(samples, flags):
    samples = _f64(samples).reshape(-1, 12)
    flags = np.ascontiguousarray(np.asarray(flags, dtype=np.uint8))
    out = np.zeros_like(samples)
    cnt = lib().ora_compact(_dp(samples), flags.ctypes.data_as(POINTER(c_ubyte)),
                            c_int64(samples.shape[0]), _dp(out))
    return out[:cnt]


# ------------------------------------------------------------------ miniball / MEGB

def _meb(fn, pts, *extra):
    pts = _f64(pts)
    n, d = pts.shape
    c = np.zeros(d); r = c_double(0.0)
    sup = np.zeros(d + 1, dtype=np.int64); ns = c_int(0)
    rc = fn(_dp(pts), c_int64(n), c_int(d), *extra, _dp(c), ctypes.byref(r),
            sup.ctypes.data_as(POINTER(c_int64)), ctypes.byref(ns))
    if rc != 0:
        raise ValueError("miniball oracle failed")
    return c, r.value, sup[:ns.value].copy()


def meb_brute(pts):
    return _meb(lib().ora_meb_brute, pts)


def meb_welzl(pts, shuffle_seed: int = 1):
    pts = _f64(pts)
    n, d = pts.shape
    c = np.zeros(d); r = c_double(0.0)
    sup = np.zeros(d + 1, dtype=np.int64); ns = c_int(0)
    rc = lib().ora_meb_welzl(_dp(pts), c_int64(n), c_int(d), c_uint64(shuffle_seed), _dp(c),
                             ctypes.byref(r), sup.ctypes.data_as(POINTER(c_int64)), ctypes.byref(ns),
                             c_int(d + 1))
    if rc != 0:
        raise ValueError("miniball oracle failed")
    return c, r.value, sup[:ns.value].copy()


def megb(samples, Rbar):
    """-> dict(R (3,3), t (3,), rot_radius [rad], trans_radius, rot_support, trans_support)."""
    samples = _f64(samples).reshape(-1, 12)
    Rbar = _f64(Rbar, 9)
    out = np.zeros(14)
    rs = np.zeros(5, dtype=np.int64); ts = np.zeros(4, dtype=np.int64)
    nrs = c_int(0); nts = c_int(0)
    rc = lib().ora_megb(_dp(samples), c_int64(samples.shape[0]), _dp(Rbar), _dp(out),
                        rs.ctypes.data_as(POINTER(c_int64)), ctypes.byref(nrs),
                        ts.ctypes.data_as(POINTER(c_int64)), ctypes.byref(nts))
    if rc != 0:
        raise ValueError("ora_megb failed")
    return dict(R=out[:9].reshape(3, 3).copy(), t=out[9:12].copy(), rot_radius=float(out[12]),
                trans_radius=float(out[13]), rot_support=rs[:nrs.value].copy(),
                trans_support=ts[:nts.value].copy())
