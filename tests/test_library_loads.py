"""-m "not gpu": the C-ABI library builds, loads and exports every symbol include/closure.h
declares; compute entry points fail loudly without a device (no CPU fallback)."""
import os
import re

import numpy as np
import pytest

from paper_2403_09990_b200 import binding as B
from paper_2403_09990_b200 import build as build_mod
from paper_2403_09990_b200 import instances as I

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    build_mod.build_library()
    return B.load_library()


def test_every_declared_symbol_is_exported(lib):
    header = open(os.path.join(ROOT, "include", "closure.h")).read()
    declared = set(re.findall(r"\b(closure_[a-z_]+)\s*\(", header))
    declared -= {"closure_s"}
    assert declared == set(B.EXPORTS), declared ^ set(B.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name
    assert B.closure_abi_version() == 2


def test_default_params_and_strerror(lib):
    p = B.closure_default_params(I.REG_3D3D)
    assert (p.n_p, p.n_p_star, p.n_t, p.gamma, p.omega0, p.t_p) == (150, 10, 15, 0.5, 0.5, 0.1)
    p = B.closure_default_params(I.REPROJ_2D3D)
    assert (p.omega0, p.v0, p.theta_p) == (1.0, 2.0, 0.2)
    assert B.closure_default_params(I.POSE_REG).n_t == 10
    with pytest.raises(B.ClosureError):
        B.closure_default_params(99)
    assert "PURSE" in B.closure_strerror(B.EINIT)


def test_invalid_arguments_rejected_before_any_cuda_call(lib):
    inst = I.make_instance(1)
    for mutate in ("beta", "nan", "type", "kstar"):
        it = I.make_instance(1)
        params = None
        ty = it.residual_type
        if mutate == "beta":
            it.betas = it.betas.copy(); it.betas[3] = 0.0
        elif mutate == "nan":
            it.measurements = it.measurements.copy(); it.measurements[0, 0] = np.inf
        elif mutate == "type":
            ty = 7
        else:
            params = I.WalkParams(n_p=5, n_p_star=6)
        with pytest.raises(B.ClosureError) as e:
            B.Closure(ty, it.measurements, it.betas, it.intrinsics, it.params if params is None else params)
        assert e.value.status == B.EINVAL
    with pytest.raises(B.ClosureError) as e:
        B.Closure(inst.residual_type, inst.measurements, inst.betas, None, I.WalkParams(n_p=50, n_p_star=21))
    assert e.value.status == B.EUNSUPPORTED


def test_no_cpu_fallback(lib):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    inst = I.make_instance(1)
    with pytest.raises(B.ClosureError) as e:
        B.Closure.closure_create(inst)
    assert e.value.status == B.ECUDA


def test_host_miniball_against_oracle_definition(lib):
    """Host logic of closure_megb: the library's Gaertner solver vs the oracle's enumeration
    of the definition (tiny inputs) and vs Welzl (larger clouds, cospherical quaternions)."""
    import oracle
    rng = np.random.default_rng(0)
    for k in range(60):
        d = int(rng.integers(1, 5))
        n = int(rng.integers(1, 11))
        pts = rng.standard_normal((n, d)) * rng.uniform(0.01, 3.0, size=d)
        c, r, s = B.closure_miniball_host(pts)
        cb, rb, sb = oracle.meb_brute(pts)
        assert abs(r - rb) <= 1e-12 * max(rb, 1e-300) and np.allclose(c, cb, atol=1e-11)
        assert set(s) == set(sb)
    q = rng.standard_normal((50000, 4)) * 0.05 + np.array([1.0, 0, 0, 0])
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    c, r, s = B.closure_miniball_host(q)
    co, ro, so = oracle.meb_welzl(q)
    assert abs(r - ro) <= 1e-12 * ro and set(s) == set(so)
    assert B.closure_miniball_host(np.ones((5, 3)))[1] == 0.0
    with pytest.raises(B.ClosureError):
        B.closure_miniball_host(np.zeros((3, 5)))


def test_bench_traffic_lookup_is_keyed_to_sources_and_launch_size():
    """bench.py's `roofline.traffic` comes from committed ncu captures: an entry counts only for the sources it was taken
    on and for the very launch it was taken on (walkers, iterations, instances); anything else reads as null."""
    import bench
    from paper_2403_09990_b200 import instances as I
    assert bench.NCU_TRAFFIC_BYTES, "profiles/ncu_traffic.json missing or unreadable"
    h = bench._csrc_hash()
    for key, e in bench.NCU_TRAFFIC_BYTES.items():
        workload, mode, precision = key.split("/")
        cfg = int(workload[1])
        inst = I.make_instance(cfg)
        assert inst.name == workload
        # every entry states the full-size launch of its config
        assert (e["walkers"], e["iterations"], e["instances"]) == (inst.num_walkers, inst.num_steps, inst.batch)
        assert e["bytes"] == e["read"] + e["write"]
        got = bench._traffic(workload, mode, int(precision), e["walkers"], e["iterations"], e["instances"])
        assert got == (e["bytes"] if e["csrc_hash"] == h else None)
        assert bench._traffic(workload, mode, int(precision), e["walkers"] // 2, e["iterations"], e["instances"]) is None
        assert bench._traffic(workload, mode, int(precision), e["walkers"], e["iterations"] + 1, e["instances"]) is None
    assert bench._traffic("C9_nothing", "rot", 64, 1, 1, 1) is None
