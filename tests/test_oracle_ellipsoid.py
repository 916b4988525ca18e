"""Pins of the oracle's ellipse / ellipsoid residuals (eq. (6) with a general Lambda_i, PAPER.md:58, 179-191;
SURVEY.md NEXT-4) against what the mathematics fixes: Lambda = I is the ball form bit for bit, Lambda = s^2 I is
the ball form with beta / s, a general Lambda is the plain norm of the Cholesky-whitened residual, and a
frozen-rotation walk of a single constraint ends on the ellipsoid itself."""
import copy

import numpy as np
import pytest

import oracle
from paper_2403_09990_b200 import instances as I


def _with_lambda(inst, lam_rows):
    head = 6 if inst.residual_type == I.REG_3D3D else 5
    out = copy.copy(inst)
    out.residual_type = I.REG_3D3D_ELL if inst.residual_type == I.REG_3D3D else I.REPROJ_2D3D_ELL
    out.measurements = np.concatenate([np.asarray(inst.measurements)[:, :head], lam_rows], axis=1)
    return out


@pytest.mark.parametrize("config", [1, 3])
def test_identity_lambda_is_the_ball_form_bit_for_bit(config):
    inst = I.make_instance(config)
    d = 3 if config == 1 else 2
    ell = _with_lambda(inst, np.tile(np.eye(d).reshape(-1), (inst.n, 1)))
    S0 = I.make_init_poses(inst, 8)
    P = copy.copy(inst.params); P.n_p = 10; P.n_p_star = 2; P.n_t = 6
    a = oracle.walk(inst, P, S0, np.arange(24), 8, 3, trace=True)
    b = oracle.walk(ell, P, S0, np.arange(24), 8, 3, trace=True)
    assert np.array_equal(a[0], b[0]) and np.array_equal(a[2], b[2])


@pytest.mark.parametrize("config", [1, 3])
def test_scaled_identity_is_the_ball_form_with_a_scaled_bound(config):
    inst = I.make_instance(config)
    d = 3 if config == 1 else 2
    s = 1.7
    ell = _with_lambda(inst, np.tile((s * s * np.eye(d)).reshape(-1), (inst.n, 1)))
    ball = copy.copy(inst); ball.betas = inst.betas / s
    rng = np.random.default_rng(0)
    for _ in range(20):
        pose = I.make_init_poses(inst, 2, seed=int(rng.integers(1 << 30)))[1]
        pose[9:] += rng.normal(scale=0.02 if config == 1 else 0.002, size=3)
        R, t = pose[:9], pose[9:]
        for c in range(inst.n):
            assert abs(oracle.residual_sq(ell, c, R, t) - s * s * oracle.residual_sq(inst, c, R, t)) <= \
                1e-13 * s * s * oracle.residual_sq(inst, c, R, t)
        assert abs(oracle.margin(ell, R, t) - s * oracle.margin(ball, R, t)) < 1e-12 * max(1.0, float(np.max(inst.betas)))
        if abs(oracle.margin(ball, R, t)) > 1e-9:
            assert oracle.in_purse(ell, R, t) == oracle.in_purse(ball, R, t)


@pytest.mark.parametrize("config", [1, 3])
def test_general_lambda_is_the_norm_of_the_cholesky_whitened_residual(config):
    """||g||_Lambda^2 = g^T Lambda g = ||L^T g||^2 with Lambda = L L^T (numpy's Cholesky), g from numpy."""
    inst = I.make_instance(config)
    ell = I.to_ellipsoidal(inst, 4)
    m = np.asarray(ell.measurements)
    rng = np.random.default_rng(1)
    for _ in range(10):
        pose = I.make_init_poses(inst, 2, seed=int(rng.integers(1 << 30)))[1]
        R, t = pose[:9].reshape(3, 3), pose[9:]
        for c in range(inst.n):
            if config == 1:
                g = m[c, 3:6] - (R @ m[c, 0:3] + t)
                Lam = m[c, 6:15].reshape(3, 3)
            else:
                p = R @ m[c, 2:5] + t
                K = np.asarray(inst.intrinsics)
                g = m[c, 0:2] - np.array([K[0] * p[0] / p[2] + K[2], K[1] * p[1] / p[2] + K[3]])
                Lam = m[c, 5:9].reshape(2, 2)
            assert np.array_equal(Lam, Lam.T) and np.all(np.linalg.eigvalsh(Lam) > 0)
            L = np.linalg.cholesky(Lam)
            want = float(np.sum((L.T @ g) ** 2))
            assert abs(oracle.residual_sq(ell, c, pose[:9], t) - want) <= 1e-12 * want + 1e-300
        # looser than the ball (lambda <= 1): the ball form's S_0 stays inside
        assert oracle.in_purse(ell, pose[:9], t)
    # an anisotropic bound must bite somewhere the ball does not: scale a pose out along the weakest axis
    assert any(abs(oracle.margin(ell, p[:9], p[9:]) - oracle.margin(inst, p[:9], p[9:])) > 1e-6
               for p in I.make_init_poses(inst, 8))


def test_single_ellipsoid_samples_lie_on_the_ellipsoid():
    """One 3D-3D constraint, rotation frozen (theta_p = 0): S_t is the ellipsoid (t - q)^T Lambda (t - q) <= beta^2
    about q = b - R a; walkers stop within one last ladder step of its surface, and the MEB of the samples is the
    ball of the longest semi-axis beta / sqrt(lambda_min)."""
    base = I.make_custom_reg(1, 21, beta=0.1, noise=0.02)
    Q, _ = np.linalg.qr(np.random.default_rng(2).standard_normal((3, 3)))
    lam = np.array([1.0, 0.49, 0.25])
    Lam = (Q * lam) @ Q.T
    Lam = 0.5 * (Lam + Lam.T)
    ell = _with_lambda(base, Lam.reshape(1, 9))
    P = I.WalkParams(mode=I.MODE_TRANS, n_p=2, n_p_star=1, n_t=16, v0=0.08, theta_p=0.0)
    S0 = np.concatenate([base.R_gt.reshape(9), base.t_gt])[None, :]
    smp, hit = oracle.walk(ell, P, S0, np.arange(400), 40, 3)
    q = base.measurements[0, 3:] - base.R_gt @ base.measurements[0, :3]
    dlt = smp[:, 9:] - q
    val = np.sqrt(np.einsum("ni,ij,nj->n", dlt, Lam, dlt))
    assert np.all(val <= 0.1 * (1 + 1e-12))
    assert np.all(val >= 0.1 - P.v0 * 0.5 ** 15 - 1e-12)                 # sqrt(lambda_max) = 1: the step bounds the gap
    assert hit.all()
    c, rad, _ = oracle.meb_welzl(smp[:, 9:])
    assert rad <= 0.1 / np.sqrt(lam.min()) + 1e-12 and rad > 0.9 * 0.1 / np.sqrt(lam.min())
    # the extent along each principal axis is that axis' semi-length
    ext = np.abs(dlt @ Q).max(axis=0)
    assert np.all(ext <= 0.1 / np.sqrt(lam) + 1e-12) and np.all(ext > 0.8 * 0.1 / np.sqrt(lam))
