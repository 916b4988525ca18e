"""Seeded synthetic PURSE instances shaped like the paper's workloads.

This module is the ONE piece shared by the CUDA path and the CPU oracle: it only
draws inputs.  It holds none of the method's arithmetic (no residual, no PURSE
membership test, no exponential-map walk step, no random-walk RNG): rotations are
built from quaternions, noise is drawn in balls/discs, and the initial pose set
``S_0`` is made feasible *by construction* (triangle-inequality radii, below), not
by evaluating the constraints.

Shapes follow BASELINE.json's five configs, which stand in for the paper's
datasets (LM-O: N~10 2D-3D keypoints; 3DMatch: N=50 3D-3D matches,
PAPER.md:349; LM: 10 pose hypotheses).  The datasets themselves are
not used anywhere.  Walk parameters are the paper's where units carry over
 and SURVEY.md section 8(d)'s where they do not.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

# residual types / modes: numeric values match include/closure.h
REPROJ_2D3D = 1
REG_3D3D = 2
POSE_REG = 3
POSE_REG_SPLIT = 4
REG_3D3D_ELL = 5
REPROJ_2D3D_ELL = 6
MODE_ROT = 0
MODE_TRANS = 1


@dataclass
class WalkParams:
    """The paper's simulation-parameter tuple P."""
    mode: int = MODE_ROT
    n_p: int = 150          # N_P
    n_p_star: int = 10      # N_P*
    n_t: int = 15           # N_T
    omega0: float = 0.5
    v0: float = 0.0
    gamma: float = 0.5
    t_p: float = 0.1
    theta_p: float = 0.0    # the paper's R_p
    flags: int = 0          # include/closure.h CLOSURE_FLAG_* (1 = plain fp64 kernel only)
    pivot: tuple = (0.0, 0.0, 0.0)   # body pivot of update_rotation (closure_set_pivot; R-1)


@dataclass
class Instance:
    name: str
    residual_type: int
    n: int
    measurements: np.ndarray          # (n, row) float64, row layout per include/closure.h
    betas: np.ndarray                 # (n,) or (2n,) for POSE_REG_SPLIT
    intrinsics: np.ndarray | None     # (fx, fy, cx, cy) or None
    R_gt: np.ndarray                  # generating pose (inside the PURSE by construction)
    t_gt: np.ndarray
    noise_radius: np.ndarray          # per-constraint bound on the generated noise norm
    params: WalkParams
    num_walkers: int
    num_steps: int
    batch: int = 1
    seed: int = 0
    extra: dict = field(default_factory=dict)


def _unit_quat_to_matrix(q: np.ndarray) -> np.ndarray:
    w, x, y, z = q
    return np.array([
        [1 - 2 * (y * y + z * z), 2 * (x * y - z * w), 2 * (x * z + y * w)],
        [2 * (x * y + z * w), 1 - 2 * (x * x + z * z), 2 * (y * z - x * w)],
        [2 * (x * z - y * w), 2 * (y * z + x * w), 1 - 2 * (x * x + y * y)],
    ])


def haar_rotation(rng: np.random.Generator) -> np.ndarray:
    """Haar-uniform rotation: normalised Gaussian 4-vector read as a quaternion."""
    q = rng.standard_normal(4)
    return _unit_quat_to_matrix(q / np.linalg.norm(q))


def rotation_from_axis_angle(axis: np.ndarray, angle: float) -> np.ndarray:
    axis = np.asarray(axis, dtype=np.float64)
    nrm = np.linalg.norm(axis)
    if nrm == 0.0 or angle == 0.0:
        return np.eye(3)
    a = axis / nrm
    h = 0.5 * angle
    return _unit_quat_to_matrix(np.concatenate(([np.cos(h)], np.sin(h) * a)))


def uniform_in_ball(rng: np.random.Generator, radius: float, dim: int = 3) -> np.ndarray:
    """Uniform in volume (dim=3) / area (dim=2)."""
    v = rng.standard_normal(dim)
    v /= np.linalg.norm(v)
    return v * radius * rng.uniform() ** (1.0 / dim)


# ----------------------------------------------------------------------------- configs

def _make_reg(rng, n, noise_small, beta_small, frac_large=0.0, noise_large=0.0, beta_large=0.0):
    a = rng.uniform(-1.0, 1.0, size=(n, 3))
    R = haar_rotation(rng)
    t = rng.uniform(-1.0, 1.0, size=3)
    betas = np.full(n, beta_small)
    radius = np.full(n, noise_small)
    if frac_large > 0.0:
        n_large = int(round(frac_large * n))
        idx = rng.permutation(n)[:n_large]
        betas[idx] = beta_large
        radius[idx] = noise_large
    b = np.empty_like(a)
    for i in range(n):
        b[i] = R @ a[i] + t + uniform_in_ball(rng, radius[i], 3)
    meas = np.concatenate([a, b], axis=1)            # row [a(3) b(3)]
    return meas, betas, radius, R, t


def _make_reproj(rng, n):
    """2D-3D keypoints of BASELINE config 3: pinhole 572.4 / 325.3 / 242.0, Z_i ~ U[-0.1, 0.1]^3 m, depth 0.8-1.2 m, pixel noise
    uniform in a disc of 5 px.  The projection here only GENERATES the measurements."""
    K = np.array([572.4, 572.4, 325.3, 242.0])
    Z = rng.uniform(-0.1, 0.1, size=(n, 3))
    R = haar_rotation(rng)
    t = np.array([rng.uniform(-0.1, 0.1), rng.uniform(-0.1, 0.1), rng.uniform(0.8, 1.2)])
    z = np.empty((n, 2))
    for i in range(n):
        p = R @ Z[i] + t
        z[i] = np.array([K[0] * p[0] / p[2] + K[2], K[1] * p[1] / p[2] + K[3]]) \
            + uniform_in_ball(rng, 5.0, 2)
    return np.concatenate([z, Z], axis=1), K, R, t        # row [z(2) Z(3)]


def make_instance(config: int, instance_index: int = 0, *, num_walkers: int | None = None,
                  num_steps: int | None = None) -> Instance:
    """BASELINE.json configs C1..C5 (1-based).  Instance seed = 1000*config + index."""
    seed = 1000 * config + instance_index
    rng = np.random.default_rng(seed)
    if config == 1:
        meas, betas, rad, R, t = _make_reg(rng, 10, 0.05, 0.1)
        inst = Instance("C1_reg_n10", REG_3D3D, 10, meas, betas, None, R, t, rad,
                        WalkParams(omega0=0.5, t_p=0.1), 1024, 200)
    elif config == 2:
        meas, betas, rad, R, t = _make_reg(rng, 50, 0.05, 0.1, 0.2, 0.1, 0.2)
        inst = Instance("C2_reg_n50", REG_3D3D, 50, meas, betas, None, R, t, rad,
                        WalkParams(omega0=0.5, t_p=0.1), 65536, 1000)
    elif config == 3:
        n = 8
        meas, K, R, t = _make_reproj(rng, n)
        inst = Instance("C3_reproj_n8", REPROJ_2D3D, n, meas, np.full(n, 8.0), K, R, t,
                        np.full(n, 5.0),
                        WalkParams(omega0=1.0, v0=2.0, theta_p=0.2, t_p=0.01), 262144, 1000)
    elif config == 4:
        n = 10
        R = haar_rotation(rng)
        t = rng.uniform(-1.0, 1.0, size=3)
        meas = np.empty((n, 12))
        for i in range(n):
            w = uniform_in_ball(rng, 0.05, 3)
            Ri = R @ rotation_from_axis_angle(w, float(np.linalg.norm(w)))
            ti = t + uniform_in_ball(rng, 0.01, 3)
            meas[i, :9] = Ri.reshape(9)              # row [R_i (9, row-major) t_i (3)]
            meas[i, 9:] = ti
        # ||R - R_i||_F = 2 sqrt(2) sin(theta/2) <= sqrt(2) * 0.05 ; ||t - t_i|| <= 0.01
        rad = np.full(n, float(np.hypot(np.sqrt(2.0) * 0.05, 0.01)))
        inst = Instance("C4_posereg_n10", POSE_REG, n, meas, np.full(n, 0.12), None, R, t, rad,
                        WalkParams(omega0=0.5, t_p=0.1, n_t=10), 262144, 2000)
    elif config == 5:
        meas, betas, rad, R, t = _make_reg(rng, 200, 0.02, 0.05)
        # smallest setting of the paper's own ablation grid; SURVEY.md 8(d)
        inst = Instance("C5_reg_n200", REG_3D3D, 200, meas, betas, None, R, t, rad,
                        WalkParams(omega0=0.5, t_p=0.05, n_p=20, n_p_star=2, n_t=5),
                        65536, 2000, batch=64)
    else:
        raise ValueError(f"unknown config {config}")
    inst.seed = seed
    if num_walkers is not None:
        inst.num_walkers = num_walkers
    if num_steps is not None:
        inst.num_steps = num_steps
    return inst


def make_custom_reg(n: int, seed: int, *, noise: float = 0.05, beta: float = 0.1,
                    distinct_betas: bool = False) -> Instance:
    """Free-size registration instance for tests (ragged N, every beta different, ...)."""
    rng = np.random.default_rng(seed)
    meas, betas, rad, R, t = _make_reg(rng, n, noise, beta)
    if distinct_betas:
        betas = betas * (1.0 + 0.5 * rng.uniform(size=n))
    inst = Instance(f"reg_n{n}_s{seed}", REG_3D3D, n, meas, betas, None, R, t, rad,
                    WalkParams(omega0=0.5, t_p=beta), 256, 50)
    inst.seed = seed
    return inst


def make_custom_reproj(n: int, seed: int, *, beta: float = 8.0) -> Instance:
    """Free-size reprojection instance for tests (a table longer than C3's 8 keypoints)."""
    rng = np.random.default_rng(seed)
    meas, K, R, t = _make_reproj(rng, n)
    inst = Instance(f"reproj_n{n}_s{seed}", REPROJ_2D3D, n, meas, np.full(n, beta), K, R, t, np.full(n, 5.0),
                    WalkParams(omega0=1.0, v0=2.0, theta_p=0.2, t_p=0.01), 256, 50)
    inst.seed = seed
    return inst


def to_ellipsoidal(inst: Instance, seed: int = 0, lam_min: float = 0.35) -> Instance:
    """Ellipse / ellipsoid form of a REPROJ_2D3D / REG_3D3D instance (eq. (6) with a general Lambda_i,
    PAPER.md:58, 179-191): Lambda_i = Q_i diag(lambda) Q_i^T with a random rotation Q_i and eigenvalues uniform in
    [lam_min, 1].  lambda <= 1 makes every constraint looser than its ball, so the generating pose and every
    S_0 drawn for the ball form stay inside."""
    rng = np.random.default_rng(9_000_000 + seed + inst.seed)
    if inst.residual_type == REG_3D3D:
        d, ty, head = 3, REG_3D3D_ELL, 6
    elif inst.residual_type == REPROJ_2D3D:
        d, ty, head = 2, REPROJ_2D3D_ELL, 5
    else:
        raise ValueError("ellipsoidal bounds exist for the residuals with point measurements")
    lam = np.empty((inst.n, d * d))
    for i in range(inst.n):
        Q, _ = np.linalg.qr(rng.standard_normal((d, d)))
        L = (Q * rng.uniform(lam_min, 1.0, d)) @ Q.T
        lam[i] = (0.5 * (L + L.T)).reshape(-1)                      # exactly symmetric
    meas = np.concatenate([np.asarray(inst.measurements)[:, :head], lam], axis=1)
    out = Instance(inst.name + "_ell", ty, inst.n, meas, np.array(inst.betas, copy=True), inst.intrinsics,
                   inst.R_gt, inst.t_gt, inst.noise_radius, inst.params, inst.num_walkers, inst.num_steps)
    out.seed = inst.seed
    return out


def to_split(inst: Instance, beta_r: float = 0.11, beta_t: float = 0.03) -> Instance:
    """PURSEreg form of a POSE_REG instance: two bounds per hypothesis."""
    assert inst.residual_type == POSE_REG
    betas = np.empty(2 * inst.n)
    betas[0::2] = beta_r
    betas[1::2] = beta_t
    out = Instance(inst.name + "_split", POSE_REG_SPLIT, inst.n, inst.measurements.copy(), betas,
                   None, inst.R_gt, inst.t_gt,
                   np.stack([np.full(inst.n, np.sqrt(2.0) * 0.05), np.full(inst.n, 0.01)], 1).reshape(-1),
                   inst.params, inst.num_walkers, inst.num_steps)
    out.seed = inst.seed
    return out


# ----------------------------------------------------------------------------- S_0

def _safe_radii(inst: Instance) -> tuple[float, float]:
    """Rotation angle / translation radius about the generating pose that keep every
    constraint satisfied by the triangle inequality alone (no residual is evaluated).

    slack_i = beta_i - noise_radius_i > 0 is known from how the instance was drawn.
    """
    m = inst.measurements
    if inst.residual_type in (REG_3D3D, REG_3D3D_ELL):        # Lambda <= I: the ball form is the tighter one
        slack = float(np.min(inst.betas - inst.noise_radius))
        lever = float(np.max(np.linalg.norm(m[:, :3], axis=1)))
        # |Exp(phi) R a - R a| <= phi |a| ; residual moves by at most phi*lever + |dt|
        return 0.45 * slack / lever, 0.45 * slack
    if inst.residual_type == POSE_REG:
        slack = float(np.min(inst.betas - inst.noise_radius))
        # stacked vector moves by sqrt(2 phi^2 + |dt|^2)
        return 0.6 * slack / np.sqrt(2.0), 0.6 * slack
    if inst.residual_type == POSE_REG_SPLIT:
        sl = inst.betas - inst.noise_radius
        return 0.9 * float(np.min(sl[0::2])) / np.sqrt(2.0), 0.9 * float(np.min(sl[1::2]))
    if inst.residual_type in (REPROJ_2D3D, REPROJ_2D3D_ELL):
        slack = float(np.min(inst.betas - inst.noise_radius))         # pixels
        fx, fy = float(inst.intrinsics[0]), float(inst.intrinsics[1])
        lever = float(np.max(np.linalg.norm(m[:, 2:5], axis=1)))
        depth_min = float(inst.t_gt[2]) - lever
        lateral = float(np.max(np.abs(inst.t_gt[:2]))) + lever
        # |d pixel| <= sqrt(2) * f * eps / depth * (1 + lateral/depth), eps = |dp|, with 2x margin
        gain = np.sqrt(2.0) * max(fx, fy) / (0.9 * depth_min) * (1.0 + lateral / (0.9 * depth_min))
        eps = 0.45 * slack / gain
        return 0.5 * eps / lever, 0.5 * eps
    raise ValueError("bad residual type")


def make_init_poses(inst: Instance, n0: int = 128, seed: int | None = None) -> np.ndarray:
    """S_0: (n0, 12) rows [R row-major (9), t (3)], element 0 = generating pose.

    Stands in for Step I (RANSAG / convex-combination sampler),
    which is off the hot path.  |S_0| ~ 100 is the paper's typical size.
    """
    rng = np.random.default_rng((inst.seed if seed is None else seed) + 7_000_000)
    phi_max, dt_max = _safe_radii(inst)
    out = np.empty((n0, 12))
    out[0, :9] = inst.R_gt.reshape(9)
    out[0, 9:] = inst.t_gt
    for s in range(1, n0):
        axis = rng.standard_normal(3)
        Rp = rotation_from_axis_angle(axis, phi_max * rng.uniform())
        out[s, :9] = (Rp @ inst.R_gt).reshape(9)
        out[s, 9:] = inst.t_gt + uniform_in_ball(rng, dt_max, 3)
    return out
