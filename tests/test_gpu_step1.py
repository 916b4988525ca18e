"""-m gpu: Step I on the device (closure_init_sample / closure_init_from_trials) against oracle/step1.py,
trial by trial.  Candidate poses within 1e-9; the accept decision identical except where the oracle's
constraint margin of that candidate is below 1e-9 (the Newton polar factor and numpy's SVD agree to ~1e-14)."""
import numpy as np
import pytest

import oracle
from oracle import step1
from paper_2403_09990_b200 import binding as B
from paper_2403_09990_b200 import instances as I

pytestmark = pytest.mark.gpu


def _gpu_trials(inst, T, seed, begin=0):
    import torch
    h = B.Closure.closure_create(inst)
    try:
        poses, ok = h.closure_init_sample(T, seed, trial_begin=begin)
        torch.cuda.synchronize()
        return poses.cpu().numpy(), ok.cpu().numpy()
    finally:
        h.closure_destroy()


def _candidate(inst, seed, k):
    meas = np.asarray(inst.measurements)
    if inst.residual_type == I.REG_3D3D:
        idx = list(step1.triplet(seed, k, inst.n))
        return step1.arun(meas[idx, 0:3], meas[idx, 3:6])
    return step1.convex_pose(meas, step1.convex_weights(seed, k, inst.n))


def _compare(inst, T, seed, begin=0):
    g_poses, g_ok = _gpu_trials(inst, T, seed, begin)
    o_poses, o_ok = step1.init_sample(inst, T, seed, trial_begin=begin)
    near = 0
    for q in range(T):
        if g_ok[q] != o_ok[q]:
            cand = _candidate(inst, seed, begin + q)
            assert cand is not None, f"trial {begin + q}: degenerate for the oracle, accepted by the GPU"
            m = oracle.margin(inst, cand[0].reshape(9), cand[1])
            assert abs(m) < 1e-9, f"trial {begin + q}: accept decision differs with oracle margin {m:.3e}"
            near += 1
            continue
        if o_ok[q]:
            err = np.abs(g_poses[q] - o_poses[q])
            assert np.all(err <= 1e-9 * np.abs(o_poses[q]) + 1e-12), f"trial {begin + q}: pose differs by {err.max():.2e}"
        else:
            assert np.all(g_poses[q] == 0.0)
    assert near <= max(1, T // 200)
    return g_ok


@pytest.mark.parametrize("config,T", [(1, 2000), (2, 2000), (4, 1500), (5, 600)])
def test_trials_match_oracle(config, T):
    inst = I.make_instance(config)
    ok = _compare(inst, T, 11)
    assert ok.mean() > 0.1


def test_split_form_ragged_sizes_replay_and_high_trial_index():
    sp = I.to_split(I.make_instance(4))
    _compare(sp, 300, 5)
    inst = I.make_instance(1)
    for T in (1, 127, 129):
        _compare(inst, T, 2)
    full = _gpu_trials(inst, 400, 9)
    part = _gpu_trials(inst, 100, 9, begin=150)
    assert np.array_equal(full[0][150:250], part[0]) and np.array_equal(full[1][150:250], part[1])
    other = _gpu_trials(inst, 400, 10)
    assert not np.array_equal(full[0], other[0])
    _compare(inst, 64, 9, begin=(1 << 32) + 7)               # high counter word
    custom = I.make_custom_reg(3, 77)                        # the only triplet there is
    _compare(custom, 50, 1)


def test_init_from_trials_feeds_the_walk():
    import torch
    inst = I.make_instance(2)
    h = B.Closure.closure_create(inst)
    try:
        n0 = h.closure_init_from_trials(1000, 21, max_poses=100)
        assert n0 == 100
        poses, ok = h.closure_init_sample(1000, 21)
        kept = poses.cpu().numpy()[ok.cpu().numpy().astype(bool)][:100]
        smp, flag = h.closure_sample(256, 0, 1)                 # zero iterations return S_0[w mod n0]
        torch.cuda.synchronize()
        assert np.array_equal(smp.cpu().numpy(), kept[np.arange(256) % 100])
        res = h.closure_run(2048, 60, 3)
        assert res["count"] > 1800 and res["rot_radius"] > 0 and res["trans_radius"] > 0
    finally:
        h.closure_destroy()


def _compare_p3p(inst, T, seed, begin=0):
    """Ex.1 (R-24).  The oracle takes the roots of the quartic from numpy's companion-matrix
    eigenvalues, the kernel isolates them by bisection; both polish the depths by Newton on the distance
    equations, so well-conditioned trials agree to ~1e-12.  A trial the oracle flags as ill-conditioned (nearly
    double root, nearly singular Jacobian: the SET of solutions is not stable under rounding) is not compared;
    an accept decision may differ only where some candidate's oracle margin is below 1e-9."""
    g_poses, g_ok = _gpu_trials(inst, T, seed, begin)
    o_poses, o_ok = step1.init_sample(inst, T, seed, trial_begin=begin)
    skipped = near = 0
    for q in range(T):
        sols, ill, _ = step1.p3p_trial(inst, seed, begin + q)
        if ill:
            skipped += 1
            continue
        if g_ok[q] != o_ok[q]:
            ms = [abs(oracle.margin(inst, R.reshape(9), t)) for _, R, t in sols]
            assert ms and min(ms) < 1e-9, f"trial {begin + q}: accept decision differs, oracle margins {ms}"
            near += 1
            continue
        if o_ok[q]:
            err = np.abs(g_poses[q] - o_poses[q])
            assert np.all(err <= 1e-9 * np.abs(o_poses[q]) + 1e-11), f"trial {begin + q}: pose differs by {err.max():.2e}"
        else:
            assert np.all(g_poses[q] == 0.0)
    assert skipped <= max(2, T // 50), f"{skipped} of {T} trials ill-conditioned"
    assert near <= max(1, T // 200)
    return g_ok


def test_p3p_trials_match_oracle():
    inst = I.make_instance(3)
    ok = _compare_p3p(inst, 3000, 11)
    assert ok.mean() > 0.02                                       # ~5 % of the trials land inside the PURSE
    for T in (1, 127, 129):
        _compare_p3p(inst, T, 2)
    _compare_p3p(inst, 64, 9, begin=(1 << 32) + 7)               # high counter word
    full = _gpu_trials(inst, 400, 9)
    part = _gpu_trials(inst, 100, 9, begin=150)
    assert np.array_equal(full[0][150:250], part[0]) and np.array_equal(full[1][150:250], part[1])


def test_p3p_trials_with_elliptic_bounds_match_oracle():
    """Ex.1 with Lambda_i != I: the 2D points are uniform in the ellipses, the PURSE test uses the ellipse norm."""
    ell = I.to_ellipsoidal(I.make_instance(3), 2)
    ok = _compare_p3p(ell, 1500, 19)
    assert ok.mean() > 0.02


def test_p3p_candidates_reproject_onto_the_sampled_pixels_and_feed_the_walk():
    """Property at any size: an accepted pose maps the three selected 3D points onto the three sampled pixels
    (each within its own ellipse), and satisfies every constraint of the instance."""
    import torch
    inst = I.make_instance(3)
    T, seed = 20000, 5
    poses, ok = _gpu_trials(inst, T, seed)
    meas, K = np.asarray(inst.measurements), np.asarray(inst.intrinsics).reshape(4)
    acc = np.nonzero(ok)[0]
    assert acc.size > 400
    for q in acc[:300]:
        R, t = poses[q, :9].reshape(3, 3), poses[q, 9:]
        assert oracle.margin(inst, poses[q, :9], t) >= -1e-9
        _, _, (idx, ys) = step1.p3p_trial(inst, seed, int(q))
        for i, y in zip(idx, ys):
            pc = R @ meas[i, 2:5] + t
            px = np.array([K[0] * pc[0] / pc[2] + K[2], K[1] * pc[1] / pc[2] + K[3]])
            assert np.abs(px - np.array(y)).max() < 1e-7
    h = B.Closure.closure_create(inst)
    try:
        n0 = h.closure_init_from_trials(4000, 21, max_poses=100)
        assert n0 == 100
        res = h.closure_run(4096, 60, 3)
        assert res["count"] > 3500 and res["rot_radius"] > 0 and res["trans_radius"] > 0
        torch.cuda.synchronize()
    finally:
        h.closure_destroy()


def test_step1_errors():
    h = B.Closure.closure_create(I.make_custom_reg(2, 5))
    try:
        with pytest.raises(B.ClosureError) as e:
            h.closure_init_sample(10, 1)
        assert e.value.status == B.EINVAL
    finally:
        h.closure_destroy()
    tight = I.make_instance(2)
    tight.betas = tight.betas * 1e-6                              # nothing can satisfy this
    h = B.Closure.closure_create(tight)
    try:
        with pytest.raises(B.ClosureError) as e:
            h.closure_init_from_trials(200, 1)
        assert e.value.status == B.EINIT
    finally:
        h.closure_destroy()
