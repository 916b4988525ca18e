"""-m gpu: compaction kernel (bit-exact against the oracle's stable filter), closure_megb
(radii within 1e-9 relative of the oracle's Welzl solver), batch launch, API errors."""
import numpy as np
import pytest

import oracle
from paper_2403_09990_b200 import binding as B
from paper_2403_09990_b200 import instances as I
from tests.gpu_common import gpu_walk

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def handle():
    inst = I.make_instance(1)
    h = B.Closure.closure_create(inst)
    h.closure_set_init(I.make_init_poses(inst, 16))
    yield h
    h.closure_destroy()


@pytest.mark.parametrize("n,frac", [(0, 0.5), (1, 1.0), (1, 0.0), (7, 0.5), (2047, 0.3), (2048, 1.0), (2049, 0.9),
                                    (65536, 0.97), (100003, 0.01), (1 << 20, 0.5), (300000, 0.0), (300000, 1.0)])
def test_compaction_bit_exact(handle, n, frac):
    import torch
    rng = np.random.default_rng(n + int(frac * 100))
    smp = rng.standard_normal((n, 12))
    flags = (rng.uniform(size=n) < frac).astype(np.uint8)
    if n > 3:
        flags[1] = 255 if frac > 0 else 0      # any non-zero byte counts as set
    d_s = torch.from_numpy(smp).cuda()
    d_f = torch.from_numpy(flags).cuda()
    out, cnt = handle.closure_compact(d_s, d_f)
    torch.cuda.synchronize()
    expect = oracle.compact(smp, flags)
    assert int(cnt.item()) == expect.shape[0]
    assert np.array_equal(out.cpu().numpy()[:expect.shape[0]], expect)


def test_compaction_unaligned_flag_pointer(handle):
    import torch
    rng = np.random.default_rng(5)
    n = 5000
    smp = rng.standard_normal((n, 12))
    flags = (rng.uniform(size=n + 3) < 0.5).astype(np.uint8)
    d_s = torch.from_numpy(smp).cuda()
    d_f = torch.from_numpy(flags).cuda()[3:]
    out, cnt = handle.closure_compact(d_s, d_f)
    expect = oracle.compact(smp, flags[3:])
    assert int(cnt.item()) == expect.shape[0]
    assert np.array_equal(out.cpu().numpy()[:expect.shape[0]], expect)


@pytest.mark.parametrize("config", [1, 3, 4])
def test_megb_matches_oracle(config):
    import torch
    inst = I.make_instance(config)
    S0 = I.make_init_poses(inst, 64)
    h = B.Closure.closure_create(inst)
    try:
        h.closure_set_init(S0)
        smp, flag = h.closure_sample(2048, 60, 5)
        comp, cnt = h.closure_compact(smp, flag)
        count = int(cnt.item())
        res = h.closure_megb(comp, count)
        host = comp.cpu().numpy()[:count]
    finally:
        h.closure_destroy()
    Rbar, _ = oracle.mean_pose(S0)
    ref = oracle.megb(host, Rbar)
    assert abs(res["rot_radius"] - ref["rot_radius"]) <= 1e-9 * ref["rot_radius"]
    assert abs(res["trans_radius"] - ref["trans_radius"]) <= 1e-9 * ref["trans_radius"]
    assert np.allclose(res["R"], ref["R"], atol=1e-9) and np.allclose(res["t"], ref["t"], atol=1e-9)
    assert set(res["rot_support"]) == set(ref["rot_support"])
    assert set(res["trans_support"]) == set(ref["trans_support"])
    # the library's mean pose (Newton polar factor) against the oracle's (SVD)
    assert np.allclose(h.mean_pose[0], Rbar, atol=1e-13)


def test_megb_on_random_clouds(handle):
    """Solver-only check on clouds that did not come from the walk (anisotropic, duplicates)."""
    import torch
    from scipy.spatial.transform import Rotation
    rng = np.random.default_rng(2)
    for n in (1, 2, 3, 50, 20000):
        rot = Rotation.from_rotvec(rng.standard_normal((n, 3)) * [0.3, 0.05, 0.01]).as_matrix()
        smp = np.concatenate([rot.reshape(n, 9), rng.standard_normal((n, 3)) * [1.0, 0.1, 3.0]], 1)
        if n >= 50:
            smp[10] = smp[11]
        res = handle.closure_megb(torch.from_numpy(smp).cuda(), n)
        ref = oracle.megb(smp, handle.mean_pose[0])
        assert abs(res["rot_radius"] - ref["rot_radius"]) <= 1e-9 * max(ref["rot_radius"], 1e-30) + 1e-15
        assert abs(res["trans_radius"] - ref["trans_radius"]) <= 1e-9 * ref["trans_radius"] + 1e-300


def test_run_whole_path_matches_stagewise():
    inst = I.make_instance(1)
    S0 = I.make_init_poses(inst, 32)
    h = B.Closure.closure_create(inst)
    try:
        h.closure_set_init(S0)
        whole = h.closure_run(1000, 50, 9)
        smp, flag = h.closure_sample(1000, 50, 9)
        comp, cnt = h.closure_compact(smp, flag)
        stage = h.closure_megb(comp, int(cnt.item()))
    finally:
        h.closure_destroy()
    assert whole["count"] == int(cnt.item())
    assert whole["rot_radius"] == stage["rot_radius"] and whole["trans_radius"] == stage["trans_radius"]


def test_batch_launch_equals_single_launches():
    import torch
    insts = [I.make_custom_reg(n, 300 + n) for n in (5, 12, 9)]
    P = insts[0].params
    hs = []
    try:
        for it in insts:
            h = B.Closure.closure_create(it, P)
            h.closure_set_init(I.make_init_poses(it, 8))
            hs.append(h)
        seeds = [11, 12, 13]
        bs, bf = B.closure_sample_batch(hs, 200, 15, seeds)
        torch.cuda.synchronize()
        for b, h in enumerate(hs):
            s, f = h.closure_sample(200, 15, seeds[b])
            assert torch.equal(s, bs[b]) and torch.equal(f, bf[b])
    finally:
        for h in hs:
            h.closure_destroy()


def test_statistics_counters():
    inst = I.make_instance(1)
    h = B.Closure.closure_create(inst)
    try:
        h.closure_set_init(I.make_init_poses(inst, 8))
        h.closure_enable_stats(True)
        s1, f1 = h.closure_sample(256, 10, 3)
        st = h.closure_get_stats()
        h.closure_enable_stats(False)
        s2, f2 = h.closure_sample(256, 10, 3)
        import torch
        assert torch.equal(s1, s2) and torch.equal(f1, f2)          # counting changes no result
    finally:
        h.closure_destroy()
    assert st["walker_steps"] == 2560
    assert st["perturb_pairs_f32"] + st["perturb_pairs"] >= 2560 * 150 * inst.n     # every pair screened or exact
    assert st["perturb_pairs"] < 2560 * 150 * inst.n // 4                              # few re-evaluated in fp64
    assert 0 < st["ladder_pairs_f32"] <= 2560 * 150 * inst.n
    assert st["accepted_steps"] <= 2560 and st["fallback_steps"] < 256


def test_api_errors():
    inst = I.make_instance(1)
    bad = I.make_instance(1)
    bad.betas = bad.betas.copy()
    bad.betas[0] = -1.0
    with pytest.raises(B.ClosureError) as e:
        B.Closure.closure_create(bad)
    assert e.value.status == B.EINVAL
    h = B.Closure.closure_create(inst)
    try:
        with pytest.raises(B.ClosureError) as e:
            h.closure_sample(10, 1, 1)
        assert e.value.status == B.ENOINIT
        outside = I.make_init_poses(inst, 4)
        outside[2, 9:] += 5.0
        with pytest.raises(B.ClosureError) as e:
            h.closure_set_init(outside)
        assert e.value.status == B.EINIT and "2" in str(e.value)
        P = B.make_params(inst.params)
        P.n_p_star = P.n_p + 1
        with pytest.raises(B.ClosureError) as e:
            h.closure_set_params(P)
        assert e.value.status == B.EINVAL
        nan = I.make_init_poses(inst, 4)
        nan[0, 0] = np.nan
        with pytest.raises(B.ClosureError):
            h.closure_set_init(nan)
    finally:
        h.closure_destroy()


def test_alu_peak_is_plausible():
    f64, _ = B.closure_alu_peak(64)
    f32, _ = B.closure_alu_peak(32)
    assert 1e13 < f64 < 6e13 and 3e13 < f32 < 1.6e14
    ph, _ = B.closure_alu_peak(4)                     # Philox4x32-10 calls per second
    assert 1e11 < ph < 5e12


@pytest.mark.parametrize("config,walkers", [(1, 6000), (3, 20000), (4, 70000)])
def test_device_side_megb_equals_host_side_and_oracle(config, walkers):
    """closure_megb keeps clouds of >= 4096 samples on the device (embedding pass + one max-reduction per
    miniball pivot); CLOSURE_FLAG_HOST_MEGB = 8 forces the host path.  Same pivots, same support sets, radii
    equal to the last bit or two; both within 1e-9 of the oracle's Welzl solver."""
    import copy
    inst = I.make_instance(config)
    S0 = I.make_init_poses(inst, 64)
    res = {}
    for name, flags in (("device", 0), ("host", 8)):
        P = copy.copy(inst.params)
        P.flags = flags
        h = B.Closure.closure_create(inst, P)
        try:
            h.closure_set_init(S0)
            smp, flag = h.closure_sample(walkers, 40, 5)
            comp, cnt = h.closure_compact(smp, flag)
            count = int(cnt.item())
            assert count >= 4096
            res[name] = h.closure_megb(comp, count)
            host = comp.cpu().numpy()[:count]
        finally:
            h.closure_destroy()
    d, hst = res["device"], res["host"]
    assert set(d["rot_support"]) == set(hst["rot_support"]) and set(d["trans_support"]) == set(hst["trans_support"])
    assert abs(d["rot_radius"] - hst["rot_radius"]) <= 1e-13 * hst["rot_radius"]
    assert abs(d["trans_radius"] - hst["trans_radius"]) <= 1e-13 * hst["trans_radius"]
    ref = oracle.megb(host, oracle.mean_pose(S0)[0])
    assert abs(d["rot_radius"] - ref["rot_radius"]) <= 1e-9 * ref["rot_radius"]
    assert abs(d["trans_radius"] - ref["trans_radius"]) <= 1e-9 * ref["trans_radius"]
    assert np.allclose(d["R"], ref["R"], atol=1e-9) and np.allclose(d["t"], ref["t"], atol=1e-9)
