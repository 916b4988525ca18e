"""Pins for the oracle's primitives: Philox, uniform map, Exp, residuals, PURSE membership.

Each test checks the oracle against something fixed OUTSIDE it: published vectors, a
library routine (scipy), a closed form, or a hand-worked value.
"""
import os

import numpy as np
import pytest
from scipy.linalg import expm
from scipy.spatial.transform import Rotation

import oracle
from paper_2403_09990_b200 import instances as I


class _Inst:
    def __init__(self, ty, meas, betas, K=None):
        self.residual_type = ty
        self.measurements = np.atleast_2d(np.asarray(meas, dtype=float))
        self.betas = np.asarray(betas, dtype=float)
        self.intrinsics = None if K is None else np.asarray(K, dtype=float)


def _skew(p):
    return np.array([[0, -p[2], p[1]], [p[2], 0, -p[0]], [-p[1], p[0], 0]])


def test_philox_known_answers(golden_dir):
    rows = [l.split() for l in open(os.path.join(golden_dir, "philox4x32_10_kat.txt"))
            if l.strip() and not l.startswith("#")]
    assert len(rows) == 3
    for r in rows:
        v = [int(x, 16) for x in r]
        out = oracle.philox4x32_10(v[0:4], v[4:6])
        assert [int(x) for x in out] == v[6:10]


def test_philox_counter_sensitivity():
    # every counter word and key word must matter (a dropped word would collide)
    base = oracle.philox4x32_10([1, 2, 3, 4], [5, 6])
    for pos in range(4):
        c = [1, 2, 3, 4]
        c[pos] += 1
        assert not np.array_equal(oracle.philox4x32_10(c, [5, 6]), base)
    assert not np.array_equal(oracle.philox4x32_10([1, 2, 3, 4], [6, 6]), base)
    assert not np.array_equal(oracle.philox4x32_10([1, 2, 3, 4], [5, 7]), base)


def test_uniform_map_is_exact_and_symmetric():
    assert oracle.u32_to_pm1(0) == 2.0 ** -32 - 1.0
    assert oracle.u32_to_pm1(2 ** 32 - 1) == 1.0 - 2.0 ** -32
    assert oracle.u32_to_pm1(2 ** 31) == 2.0 ** -32
    for x in (0, 1, 12345, 2 ** 31 - 1, 2 ** 32 - 2):
        assert oracle.u32_to_pm1(x) == -oracle.u32_to_pm1(2 ** 32 - 1 - x)
        assert -1.0 < oracle.u32_to_pm1(x) < 1.0


@pytest.mark.parametrize("phi", [[0.3, -0.2, 0.5], [1e-3, 2e-3, -1e-3], [2.0, 1.0, -2.0],
                                 [0.0, 0.0, 0.0], [3e-5, -4e-5, 1e-5]])
def test_exp_against_library_and_identities(phi):
    phi = np.array(phi)
    R = oracle.exp_so3(phi)
    K = np.array([[0, -phi[2], phi[1]], [phi[2], 0, -phi[0]], [-phi[1], phi[0], 0]])
    assert np.allclose(R, expm(K), atol=1e-14, rtol=0)                     # matrix exponential
    assert np.allclose(R, Rotation.from_rotvec(phi).as_matrix(), atol=1e-14, rtol=0)
    assert np.allclose(R.T @ R, np.eye(3), atol=1e-14)
    assert abs(np.linalg.det(R) - 1.0) < 1e-14
    assert np.allclose(R @ phi, phi, atol=1e-15)
    assert abs(np.trace(R) - (1 + 2 * np.cos(np.linalg.norm(phi)))) < 1e-14


def test_exp_series_branch_is_continuous():
    u = np.array([1.0, 2.0, -2.0]) / 3.0
    lo, hi = oracle.exp_so3(0.999999e-4 * u), oracle.exp_so3(1.000001e-4 * u)
    assert np.allclose(lo, expm(_skew(0.999999e-4 * u)), atol=1e-15, rtol=0)
    assert np.allclose(hi, expm(_skew(1.000001e-4 * u)), atol=1e-15, rtol=0)
    assert np.abs(lo - hi).max() < 3e-10


def test_registration_residual_hand_values():
    Rz = np.array([[0.0, -1, 0], [1, 0, 0], [0, 0, 1]])                    # +90 deg about z
    t = np.array([0.5, -0.25, 2.0])
    # R a = (0,1,0); b = R a + t  -> zero residual.  A transposed R would give 4.
    inst = _Inst(I.REG_3D3D, [[1, 0, 0, 0.5, 0.75, 2.0]], [0.1])
    assert oracle.residual_sq(inst, 0, Rz, t) == 0.0
    assert oracle.residual_sq(inst, 0, Rz.T, t) == 4.0
    inst = _Inst(I.REG_3D3D, [[1, 2, 3, 1, 2, 4]], [1.0])
    assert oracle.residual_sq(inst, 0, np.eye(3), np.zeros(3)) == 1.0
    assert oracle.in_purse(inst, np.eye(3), np.zeros(3))                   # on the boundary: <=
    assert oracle.margin(inst, np.eye(3), np.zeros(3)) == 0.0
    assert not oracle.in_purse(inst, np.eye(3), np.array([0, 0, -1e-9]))
    # sign of t: b - (Ra + t)
    assert oracle.residual_sq(inst, 0, np.eye(3), np.array([0, 0, 1.0])) == 0.0


def test_reprojection_residual_hand_values():
    K = [500.0, 400.0, 320.0, 240.0]
    # point on the optical axis projects to the principal point
    inst = _Inst(I.REPROJ_2D3D, [[323.0, 244.0, 0, 0, 0]], [6.0], K)
    assert oracle.residual_sq(inst, 0, np.eye(3), np.array([0, 0, 1.0])) == 25.0
    assert oracle.in_purse(inst, np.eye(3), np.array([0, 0, 1.0]))
    # p = (0.2, -0.1, 2) -> u = 500*0.1+320 = 370, v = 400*(-0.05)+240 = 220
    inst = _Inst(I.REPROJ_2D3D, [[370.0, 220.0, 0.2, -0.1, 0.5]], [1.0], K)
    assert abs(oracle.residual_sq(inst, 0, np.eye(3), np.array([0, 0, 1.5]))) < 1e-24
    # rotation acts on Z before translation: R = Rz(90): Z=(0.2,-0.1,.5) -> (0.1,0.2,.5)
    Rz = np.array([[0.0, -1, 0], [1, 0, 0], [0, 0, 1]])
    sq = oracle.residual_sq(inst, 0, Rz, np.array([0, 0, 1.5]))
    assert abs(sq - ((370 - (500 * 0.05 + 320)) ** 2 + (220 - (400 * 0.1 + 240)) ** 2)) < 1e-9
    # cheirality (reading R-10): depth <= 0 is a violation with infinite norm
    assert oracle.residual_sq(inst, 0, np.eye(3), np.array([0, 0, -0.5])) == np.inf
    assert not oracle.in_purse(inst, np.eye(3), np.array([0, 0, -0.5]))
    assert oracle.margin(inst, np.eye(3), np.array([0, 0, -0.5])) == -np.inf


def test_pose_regression_frobenius_is_geodesic_ball():
    # ||R - R_i||_F^2 = 8 sin^2(theta/2): Ex.3's rotation constraint is a geodesic ball
    # (PAPER.md:193).  theta = geodesic angle between R and R_i.
    rng = np.random.default_rng(3)
    for _ in range(5):
        Ri = I.haar_rotation(rng)
        w = rng.standard_normal(3)
        w *= rng.uniform(0.01, 1.0) / np.linalg.norm(w)
        R = Ri @ Rotation.from_rotvec(w).as_matrix()
        theta = np.linalg.norm(w)
        ti = rng.standard_normal(3)
        t = ti + np.array([0.03, -0.04, 0.12])
        row = np.concatenate([Ri.reshape(9), ti])
        stacked = _Inst(I.POSE_REG, [row], [1.0])
        assert abs(oracle.residual_sq(stacked, 0, R, t) - (8 * np.sin(theta / 2) ** 2 + 0.13 ** 2)) < 1e-13
        split = _Inst(I.POSE_REG_SPLIT, [row], [1.0, 1.0])
        assert abs(oracle.residual_sq(split, 0, R, t) - 8 * np.sin(theta / 2) ** 2) < 1e-13
        assert abs(oracle.residual_sq(split, 1, R, t) - 0.13 ** 2) < 1e-15
        # boundary angle of the split rotation constraint: 2 asin(beta / (2 sqrt 2))
        beta_r = 0.2
        th_b = 2 * np.arcsin(beta_r / (2 * np.sqrt(2)))
        sp = _Inst(I.POSE_REG_SPLIT, [row], [beta_r, 10.0])
        u = w / np.linalg.norm(w)
        assert oracle.in_purse(sp, Ri @ Rotation.from_rotvec((th_b - 1e-9) * u).as_matrix(), ti)
        assert not oracle.in_purse(sp, Ri @ Rotation.from_rotvec((th_b + 1e-9) * u).as_matrix(), ti)


@pytest.mark.parametrize("config", [1, 2, 3, 4, 5])
def test_generating_pose_and_init_set_inside_purse(config):
    """Construction pin (PURSE definition): noise radius < beta puts the
    generating pose inside S with margin >= beta - noise radius, and S_0 is inside S."""
    inst = I.make_instance(config)
    m = oracle.margin(inst, inst.R_gt, inst.t_gt)
    assert m >= float(np.min(inst.betas - inst.noise_radius)) - 1e-12
    assert oracle.in_purse(inst, inst.R_gt, inst.t_gt)
    S0 = I.make_init_poses(inst, 128)
    assert all(oracle.in_purse(inst, s[:9], s[9:]) for s in S0)
    # a pose far away is outside
    assert not oracle.in_purse(inst, inst.R_gt, inst.t_gt + 10.0)
    if config == 4:
        sp = I.to_split(inst)
        assert all(oracle.in_purse(sp, s[:9], s[9:]) for s in I.make_init_poses(sp, 64))


def test_margin_is_min_over_constraints_and_matches_numpy():
    inst = I.make_instance(2)
    rng = np.random.default_rng(0)
    R = Rotation.from_rotvec(0.02 * rng.standard_normal(3)).as_matrix() @ inst.R_gt
    t = inst.t_gt + 0.01 * rng.standard_normal(3)
    a, b = inst.measurements[:, :3], inst.measurements[:, 3:]
    norms = np.linalg.norm(b - (a @ R.T + t), axis=1)
    assert abs(oracle.margin(inst, R, t) - np.min(inst.betas - norms)) < 1e-14
    assert oracle.in_purse(inst, R, t) == bool(np.all(norms <= inst.betas))


def test_mean_pose_is_projection_onto_so3():
    rng = np.random.default_rng(5)
    R0 = I.haar_rotation(rng)
    S0 = np.zeros((40, 12))
    for s in range(40):
        S0[s, :9] = (Rotation.from_rotvec(0.1 * rng.standard_normal(3)).as_matrix() @ R0).reshape(9)
        S0[s, 9:] = rng.standard_normal(3)
    Rbar, tbar = oracle.mean_pose(S0)
    assert np.allclose(Rbar.T @ Rbar, np.eye(3), atol=1e-14) and np.linalg.det(Rbar) > 0
    assert np.allclose(tbar, S0[:, 9:].mean(0))
    # nearest rotation in Frobenius norm: no nearby rotation does better
    M = S0[:, :9].reshape(-1, 3, 3).sum(0)
    best = np.linalg.norm(M - 40 * Rbar)
    for _ in range(50):
        Rn = Rotation.from_rotvec(1e-3 * rng.standard_normal(3)).as_matrix() @ Rbar
        assert np.linalg.norm(M - 40 * Rn) >= best - 1e-12
    assert Rotation.from_matrix(Rbar @ R0.T).magnitude() < 0.1
