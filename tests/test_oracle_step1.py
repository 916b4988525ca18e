"""Pins of the Step I oracle (oracle/step1.py): Arun's method, the RANSAG triplets and the convex-combination
sampler, against closed forms, a library routine and brute-force perturbation -- not against itself."""
import numpy as np
import pytest
from scipy.spatial.transform import Rotation

import oracle
from oracle import step1
from paper_2403_09990_b200 import instances as I


def _rand_rot(rng):
    return Rotation.from_quat(rng.standard_normal(4)).as_matrix()


def test_arun_recovers_a_noiseless_rigid_motion():
    rng = np.random.default_rng(0)
    for _ in range(20):
        R, t = _rand_rot(rng), rng.uniform(-1, 1, 3)
        a = rng.uniform(-1, 1, (3, 3))
        b = a @ R.T + t
        Rh, th = step1.arun(a, b)
        assert np.allclose(Rh, R, atol=1e-12) and np.allclose(th, t, atol=1e-12)
        assert abs(np.linalg.det(Rh) - 1.0) < 1e-12


def test_arun_is_the_least_squares_rotation_with_noise_and_equals_scipy():
    rng = np.random.default_rng(1)
    for _ in range(20):
        R, t = _rand_rot(rng), rng.uniform(-1, 1, 3)
        a = rng.uniform(-1, 1, (3, 3))
        b = a @ R.T + t + 0.05 * rng.standard_normal((3, 3))
        Rh, th = step1.arun(a, b)
        assert abs(np.linalg.det(Rh) - 1.0) < 1e-12 and np.allclose(Rh @ Rh.T, np.eye(3), atol=1e-12)
        cost = lambda Rr, tt: float(((b - a @ Rr.T - tt) ** 2).sum())
        c0 = cost(Rh, th)
        for _ in range(50):                                   # no nearby rigid motion does better
            dR = Rotation.from_rotvec(1e-3 * rng.standard_normal(3)).as_matrix()
            assert cost(dR @ Rh, th + 1e-3 * rng.standard_normal(3)) >= c0 - 1e-12
        # library routine: Kabsch on the centred vectors
        ref, _ = Rotation.align_vectors(b - b.mean(0), a - a.mean(0))
        assert np.allclose(ref.as_matrix(), Rh, atol=1e-9)
        assert np.allclose(th, b.mean(0) - Rh @ a.mean(0), atol=1e-13)   # optimal t given R


def test_arun_rejects_collinear_triplets_and_handles_the_reflection_case():
    a = np.array([[0.0, 0, 0], [1, 1, 1], [2, 2, 2]])
    assert step1.arun(a, a) is None
    # a planar triplet whose unconstrained orthogonal fit is a reflection: the guard must return det = +1
    a = np.array([[1.0, 0, 0], [0, 1, 0], [-1, -1, 0]])
    b = a * np.array([1.0, -1.0, 1.0])                      # mirrored in the plane
    Rh, _ = step1.arun(a, b)
    assert abs(np.linalg.det(Rh) - 1.0) < 1e-12
    assert np.allclose(Rh @ a.T, b.T, atol=1e-12)           # a 180-degree turn about x does it


def test_triplets_are_distinct_uniform_and_replayable():
    n = 7
    seen = np.zeros((n, n, n), dtype=int)
    for k in range(4000):
        i = step1.triplet(5, k, n)
        assert len(set(i)) == 3 and all(0 <= v < n for v in i)
        seen[i] += 1
    assert step1.triplet(5, 17, n) == step1.triplet(5, 17, n) != step1.triplet(6, 17, n)
    counts = seen[seen > 0]
    assert counts.size == n * (n - 1) * (n - 2)              # every ordered triple occurs
    assert counts.min() > 5 and counts.max() < 45            # about 4000 / 210 = 19 each
    assert step1.triplet(1, (1 << 32) + 3, 50) != step1.triplet(1, 3, 50)   # high counter word is used


def test_convex_weights_and_pose():
    inst = I.make_instance(4)
    meas = np.asarray(inst.measurements)
    for k in range(20):
        w = step1.convex_weights(9, k, inst.n)
        assert np.all(w > 0) and abs(w.sum() - 1.0) < 1e-14
        R, t = step1.convex_pose(meas, w)
        assert np.allclose(R @ R.T, np.eye(3), atol=1e-12) and abs(np.linalg.det(R) - 1) < 1e-12
        lo, hi = meas[:, 9:12].min(0), meas[:, 9:12].max(0)
        assert np.all(t >= lo - 1e-15) and np.all(t <= hi + 1e-15)        # inside the hull's bounding box
        M = sum(w[i] * meas[i, :9].reshape(3, 3) for i in range(inst.n))
        d0 = np.linalg.norm(R - M)
        rng = np.random.default_rng(k)
        for _ in range(30):                                  # nearest rotation in the Frobenius norm
            dR = Rotation.from_rotvec(1e-3 * rng.standard_normal(3)).as_matrix()
            assert np.linalg.norm(dR @ R - M) >= d0 - 1e-13
    one = np.zeros(inst.n); one[3] = 1.0
    R, t = step1.convex_pose(meas, one)                      # a vertex of the simplex is the hypothesis itself
    assert np.allclose(R.reshape(9), meas[3, :9], atol=1e-12) and np.allclose(t, meas[3, 9:12])


@pytest.mark.parametrize("config", [1, 2, 4, 5])
def test_init_sample_yields_poses_inside_the_purse(config):
    inst = I.make_instance(config)
    poses, ok = step1.init_sample(inst, 300, 11)
    assert ok.sum() >= 3, "no trial produced a pose inside the PURSE"
    for q in np.nonzero(ok)[0]:
        assert oracle.in_purse(inst, poses[q, :9], poses[q, 9:])
        R = poses[q, :9].reshape(3, 3)
        assert np.allclose(R @ R.T, np.eye(3), atol=1e-12)
    assert np.all(poses[ok == 0] == 0.0)
    p2, ok2 = step1.init_sample(inst, 10, 11, trial_begin=100)             # any trial replays alone
    assert np.array_equal(p2, poses[100:110]) and np.array_equal(ok2, ok[100:110])
    # the generating pose is near the accepted ones (they all lie in the same small set)
    assert np.abs(poses[ok == 1][:, 9:] - inst.t_gt).max() < 0.5


def test_split_form_and_unsupported_residual():
    sp = I.to_split(I.make_instance(4))
    poses, ok = step1.init_sample(sp, 100, 3)
    for q in np.nonzero(ok)[0]:
        assert oracle.in_purse(sp, poses[q, :9], poses[q, 9:])
    with pytest.raises(ValueError):
        step1.init_sample(I.make_instance(3), 4, 1)
