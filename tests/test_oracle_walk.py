"""Pins for the oracle's walk (Alg. 2 / Alg. A8).

What fixes the expected values here is outside oracle/closure_oracle.c:
  * closed-form ray exits from an intersection of Euclidean balls (rotation frozen,
    PURSE3D3D) and the exactly predictable greedy ladder sum;
  * the sphere / geodesic-ball geometry of N=1 instances;
  * invariants the paper states (feasibility PAPER.md:334, independence of walks PAPER.md:336);
  * a second, numpy/scipy re-statement of ONE iteration built only from pinned primitives;
  * a brute-force grid over SE(3) on a tiny instance (Prop. 4).
"""
import copy

import numpy as np
import pytest
from scipy import stats
from scipy.spatial.transform import Rotation

import oracle
from paper_2403_09990_b200 import instances as I


def _reg_instance(n, seed, beta=0.1, noise=0.05):
    return I.make_custom_reg(n, seed, noise=noise, beta=beta)


def _single_pose(inst):
    return np.concatenate([inst.R_gt.reshape(9), inst.t_gt])[None, :]


# ----------------------------------------------------------------------------- closed form

def test_frozen_rotation_walk_hits_closed_form_ray_exit():
    """TRANS mode with theta_p = 0 on Ex.2: S_t|R = intersection of balls B(b_i - R a_i, beta_i).
    A walker moves along a fixed ray; it must stop at the greedy ladder sum below the exit."""
    inst = _reg_instance(6, 11)
    S0 = _single_pose(inst)                      # |S_0| = 1 -> direction term is zero (R-3)
    P = I.WalkParams(mode=I.MODE_TRANS, n_p=4, n_p_star=2, n_t=12, v0=0.05, gamma=0.5, theta_p=0.0)
    steps = 40
    smp, hit, tr, _ = oracle.walk(inst, P, S0, np.arange(64), steps, 7, trace=True)
    a, b = inst.measurements[:, :3], inst.measurements[:, 3:]
    q = b - a @ inst.R_gt.T
    checked = 0
    for w in range(64):
        assert np.array_equal(smp[w, :9], S0[0, :9])             # rotation never changes
        move = smp[w, 9:] - inst.t_gt
        L = np.linalg.norm(move)
        assert L > 0
        d = move / L
        e = q - inst.t_gt
        de = e @ d
        Lstar = np.min(de + np.sqrt(de ** 2 - np.sum(e * e, 1) + inst.betas ** 2))
        s_star = Lstar / P.v0                                    # |v| = v0 exactly (unit vector)
        s, m_list = 0.0, []
        for _ in range(steps):                                   # greedy ladder, scalars only
            m0 = 0
            for m in range(1, P.n_t + 1):
                if s + P.gamma ** (m - 1) <= s_star:
                    m0 = m
                    break
            if m0:
                s += P.gamma ** (m0 - 1)
            m_list.append(m0)
        near_tie = any(abs(s_ + P.gamma ** (m - 1) - s_star) < 1e-9
                       for s_ in [s] for m in range(1, P.n_t + 1))
        if near_tie:
            continue
        checked += 1
        assert abs(L / P.v0 - s) < 1e-10
        assert 0 <= s_star - s < P.gamma ** (P.n_t - 1) * 1.0000001
        assert list(tr[w] & 255) == m_list
        assert hit[w] == (1 if any(m != 1 for m in m_list) else 0)
    assert checked >= 60


def test_random_unit_vector_is_uniform_on_sphere():
    """R-4: with huge beta the first step is always taken in full: t_1 - t_0 = v0 * v~."""
    inst = _reg_instance(3, 5, beta=100.0)
    P = I.WalkParams(mode=I.MODE_TRANS, n_p=1, n_p_star=1, n_t=1, v0=2.0, theta_p=0.0)
    n = 8192
    smp, hit = oracle.walk(inst, P, _single_pose(inst), np.arange(n), 1, 99)
    u = (smp[:, 9:] - inst.t_gt) / P.v0
    assert np.allclose(np.linalg.norm(u, axis=1), 1.0, atol=1e-14)
    assert not hit.any()
    assert np.linalg.norm(u.mean(0)) < 4.0 / np.sqrt(3 * n) * np.sqrt(3)
    assert np.allclose(u.T @ u / n, np.eye(3) / 3, atol=0.02)
    for c in range(3):                                           # Archimedes: each coordinate uniform
        assert stats.kstest(u[:, c], stats.uniform(-1, 2).cdf).pvalue > 1e-3
    az = np.arctan2(u[:, 1], u[:, 0])
    assert stats.kstest(az, stats.uniform(-np.pi, 2 * np.pi).cdf).pvalue > 1e-3


def test_single_constraint_registration_samples_lie_on_sphere():
    inst = _reg_instance(1, 21, beta=0.1, noise=0.03)
    P = I.WalkParams(mode=I.MODE_TRANS, n_p=2, n_p_star=1, n_t=14, v0=0.08, theta_p=0.0)
    smp, hit = oracle.walk(inst, P, _single_pose(inst), np.arange(256), 30, 3)
    qc = inst.measurements[0, 3:] - inst.R_gt @ inst.measurements[0, :3]
    r = np.linalg.norm(smp[:, 9:] - qc, axis=1)
    assert np.all(r <= 0.1 + 1e-15) and np.all(r >= 0.1 - P.v0 * 0.5 ** 13 - 1e-12)
    assert hit.all()
    c, rad, _ = oracle.meb_welzl(smp[:, 9:])
    assert rad <= 0.1 + 1e-12 and rad > 0.97 * 0.1
    assert np.linalg.norm(c - qc) < 0.01


def test_single_hypothesis_split_rotation_ball():
    """PURSEreg with N=1: S_R is the geodesic ball of angle 2 asin(beta_R / (2 sqrt 2)) about R_1."""
    base = I.make_instance(4)
    sp = I.to_split(base, beta_r=0.2, beta_t=0.05)
    sp.n = 1
    sp.measurements = sp.measurements[:1]
    sp.betas = sp.betas[:2]
    R1 = sp.measurements[0, :9].reshape(3, 3)
    S0 = np.concatenate([R1.reshape(9), sp.measurements[0, 9:]])[None, :]
    P = I.WalkParams(mode=I.MODE_ROT, n_p=2, n_p_star=1, n_t=14, omega0=0.3, t_p=0.0)
    smp, hit = oracle.walk(sp, P, S0, np.arange(256), 30, 4)
    th_b = 2 * np.arcsin(0.2 / (2 * np.sqrt(2)))
    ang = np.array([Rotation.from_matrix(s[:9].reshape(3, 3) @ R1.T).magnitude() for s in smp])
    assert np.all(ang <= th_b + 1e-12) and np.all(ang >= th_b - 0.3 * 0.5 ** 13 - 1e-9)
    g = oracle.megb(smp, R1)
    assert g["rot_radius"] <= th_b + 1e-9 and g["rot_radius"] > 0.97 * th_b
    assert Rotation.from_matrix(g["R"] @ R1.T).magnitude() < 0.1 * th_b
    assert g["trans_radius"] < 1e-15


# ----------------------------------------------------------------------------- one iteration, restated

def _xi(seed, w, s, j, tag):
    x = oracle.philox4x32_10([w & 0xFFFFFFFF, s, j, tag | ((w >> 32) << 8)],
                             [seed & 0xFFFFFFFF, seed >> 32])
    return x


def _np_norms(inst, R, t):
    m, ty = inst.measurements, inst.residual_type
    if ty == I.REG_3D3D:
        return np.linalg.norm(m[:, 3:] - (m[:, :3] @ R.T + t), axis=1)
    if ty == I.REPROJ_2D3D:
        p = m[:, 2:5] @ R.T + t
        K = inst.intrinsics
        uv = np.stack([K[0] * p[:, 0] / p[:, 2] + K[2], K[1] * p[:, 1] / p[:, 2] + K[3]], 1)
        nr = np.linalg.norm(m[:, :2] - uv, axis=1)
        return np.where(p[:, 2] > 0, nr, np.inf)
    dR = np.linalg.norm(R.reshape(1, 9) - m[:, :9], axis=1)
    dt = np.linalg.norm(t - m[:, 9:], axis=1)
    if ty == I.POSE_REG:
        return np.hypot(dR, dt)
    return np.stack([dR, dt], 1).reshape(-1)


def _np_walk(inst, P, S0, w, steps, seed):
    """numpy/scipy re-statement of Alg. 2 / A8 for one walker (uses only Philox words)."""
    Rbar, tbar = oracle.mean_pose(S0)
    R = S0[w % len(S0), :9].reshape(3, 3).copy()
    t = S0[w % len(S0), 9:].copy()
    x = _xi(seed, w, 0, 0, 0)
    z = oracle.u32_to_pm1(int(x[0])); ph = np.pi * (oracle.u32_to_pm1(int(x[1])) + 1)
    ut = np.array([np.sqrt(1 - z * z) * np.cos(ph), np.sqrt(1 - z * z) * np.sin(ph), z])
    if P.mode == I.MODE_ROT:
        rv = Rotation.from_matrix(R @ Rbar.T).as_rotvec()
        th = np.linalg.norm(rv)
        u = rv / th if th >= 1e-12 else np.zeros(3)
        vel = P.omega0 * (u + ut)
    else:
        dv = t - tbar
        nd = np.linalg.norm(dv)
        vel = P.v0 * ((dv / nd if nd >= 1e-12 else np.zeros(3)) + ut)
    codes = []
    for s in range(1, steps + 1):
        poses, d = [], []
        for j in range(P.n_p):
            xs = _xi(seed, w, s, j, 1)
            xi = np.array([oracle.u32_to_pm1(int(xs[c])) for c in range(3)])
            if P.mode == I.MODE_ROT:
                poses.append((R, t + P.t_p * xi))
            else:
                poses.append((Rotation.from_rotvec(P.theta_p * xi).as_matrix() @ R, t))
            d.append(np.min(inst.betas - _np_norms(inst, *poses[-1])))
        order = sorted(range(P.n_p), key=lambda j: (-d[j], j))[:P.n_p_star]
        code = 0
        for m in range(1, P.n_t + 1):
            dT = P.gamma ** (m - 1)
            for j in order:
                Rj, tj = poses[j]
                if P.mode == I.MODE_ROT:
                    cand = (Rotation.from_rotvec(dT * vel).as_matrix() @ Rj, tj)
                else:
                    cand = (Rj, tj + dT * vel)
                if np.all(_np_norms(inst, *cand) <= inst.betas):
                    R, t = cand
                    code = m | (j << 8)
                    break
            if code:
                break
        codes.append(code)
    return R, t, codes


def _cases():
    c1 = I.make_instance(1)
    c3 = I.make_instance(3)
    c4 = I.make_instance(4)
    out = [("reg_rot", c1, c1.params),
           ("reg_trans", c1, I.WalkParams(mode=I.MODE_TRANS, v0=0.1, theta_p=0.02, n_p=30, n_p_star=4, n_t=8)),
           ("reproj_rot", c3, c3.params),
           ("reproj_trans", c3, I.WalkParams(mode=I.MODE_TRANS, v0=0.02, theta_p=0.01, n_p=30, n_p_star=4, n_t=8)),
           ("posereg_rot", c4, c4.params),
           ("split_rot", I.to_split(c4), c4.params),
           ("split_trans", I.to_split(c4), I.WalkParams(mode=I.MODE_TRANS, v0=0.02, theta_p=0.02, n_p=20, n_p_star=3, n_t=8))]
    return out


@pytest.mark.parametrize("name,inst,P", _cases(), ids=[c[0] for c in _cases()])
def test_walk_matches_numpy_restatement(name, inst, P):
    P = copy.copy(P)
    P.n_p = min(P.n_p, 40)
    P.n_p_star = min(P.n_p_star, 5)
    S0 = I.make_init_poses(inst, 16)
    ids = np.array([0, 5, 17, (1 << 32) + 5])
    steps = 6
    smp, hit, tr, sl = oracle.walk(inst, P, S0, ids, steps, 42, trace=True)
    for q, w in enumerate(ids):
        R, t, codes = _np_walk(inst, P, S0, int(w), steps, 42)
        if sl[q].min() < 1e-9:
            continue
        assert list(tr[q]) == codes
        assert np.allclose(smp[q, :9].reshape(3, 3), R, atol=1e-12, rtol=0)
        assert np.allclose(smp[q, 9:], t, atol=1e-12, rtol=0)
        assert hit[q] == int(any((c & 255) != 1 for c in codes))
    # the high counter word matters: walker 2^32+5 is not walker 5
    assert not np.array_equal(smp[1], smp[3])


# ----------------------------------------------------------------------------- invariants

@pytest.mark.parametrize("name,inst,P", _cases(), ids=[c[0] for c in _cases()])
def test_samples_feasible_replayable_and_flag_consistent(name, inst, P):
    S0 = I.make_init_poses(inst, 32)
    ids = np.arange(48)
    smp, hit, tr, sl = oracle.walk(inst, P, S0, ids, 25, 1234, trace=True, n_threads=4)
    for s in smp:                                                 # PAPER.md:334 "still in S"
        assert oracle.in_purse(inst, s[:9], s[9:])
        R = s[:9].reshape(3, 3)
        assert np.allclose(R.T @ R, np.eye(3), atol=1e-12)
    # replay of a single walker, alone, single-threaded (counter-based RNG)
    for w in (0, 13, 47):
        s1, h1 = oracle.walk(inst, P, S0, [w], 25, 1234)
        assert np.array_equal(s1[0], smp[w]) and h1[0] == hit[w]
    # flag = some iteration did not take the full step
    assert np.array_equal(hit, np.any((tr & 255) != 1, axis=1).astype(np.uint8))
    # another seed gives another cloud
    smp2, _ = oracle.walk(inst, P, S0, ids, 25, 1235)
    assert not np.array_equal(smp, smp2)
    # prefix property: running fewer iterations gives the earlier state of the same walk
    s_short, _ = oracle.walk(inst, P, S0, [3], 10, 1234)
    s_long, _, tr_long, _ = oracle.walk(inst, P, S0, [3], 25, 1234, trace=True)
    if np.all(tr_long[0, 10:] == 0):
        assert np.array_equal(s_short[0], s_long[0])


def test_constraint_permutation_leaves_walk_unchanged():
    inst = I.make_instance(2)
    S0 = I.make_init_poses(inst, 8)
    smp, hit = oracle.walk(inst, inst.params, S0, np.arange(6), 12, 5)
    perm = np.random.default_rng(0).permutation(inst.n)
    inst2 = copy.copy(inst)
    inst2.measurements = inst.measurements[perm]
    inst2.betas = inst.betas[perm]
    smp2, hit2 = oracle.walk(inst2, inst.params, S0, np.arange(6), 12, 5)
    assert np.array_equal(smp, smp2) and np.array_equal(hit, hit2)


def test_bad_parameters_rejected():
    inst = I.make_instance(1)
    S0 = I.make_init_poses(inst, 4)
    P = copy.copy(inst.params)
    P.n_p_star = P.n_p + 1
    with pytest.raises(ValueError):
        oracle.walk(inst, P, S0, [0], 1, 1)


# ----------------------------------------------------------------------------- extent vs brute force

def test_sampled_extent_agrees_with_dense_grid():
    """Tiny Ex.2 instance: feasible nodes of a dense grid over SE(3) vs the sampled cloud.
    Prop. 4: radius of any subset <= true radius (up to the grid diagonal);
    plausibility floor 0.85 (the paper's worst reported average eta is 0.914)."""
    inst = _reg_instance(5, 77, beta=0.06, noise=0.03)
    a, b = inst.measurements[:, :3], inst.measurements[:, 3:]
    S0 = I.make_init_poses(inst, 64)
    P = I.WalkParams(mode=I.MODE_ROT, n_p=60, n_p_star=6, n_t=12, omega0=0.3, t_p=0.03)
    smp, hit = oracle.walk(inst, P, S0, np.arange(768), 25, 9, n_threads=8)
    g = oracle.megb(smp, inst.R_gt)                       # rotation-boundary sampler (Alg. 2)
    Pt = I.WalkParams(mode=I.MODE_TRANS, n_p=60, n_p_star=6, n_t=12, v0=0.05, theta_p=0.05)
    smp_t, _ = oracle.walk(inst, Pt, S0, np.arange(768), 25, 9, n_threads=8)
    gt = oracle.megb(smp_t, inst.R_gt)                    # translation-boundary sampler (Alg. A8)

    # grid over rotation vectors (left-multiplied onto R_gt) x translations
    nr, nt = 19, 17
    hr, ht = 0.12, 0.07
    axis_r = np.linspace(-hr, hr, nr)
    axis_t = np.linspace(-ht, ht, nt)
    rv = np.stack(np.meshgrid(axis_r, axis_r, axis_r, indexing="ij"), -1).reshape(-1, 3)
    tv = np.stack(np.meshgrid(axis_t, axis_t, axis_t, indexing="ij"), -1).reshape(-1, 3) + inst.t_gt
    Rs = Rotation.from_rotvec(rv).as_matrix() @ inst.R_gt                 # (nr^3, 3, 3)
    rot_ok = np.zeros(len(rv), bool)
    trans_ok = np.zeros(len(tv), bool)
    for c0 in range(0, len(rv), 256):
        Rc = Rs[c0:c0 + 256]
        q = b[None] - np.einsum("rij,nj->rni", Rc, a)                     # (r, N, 3)
        d2 = ((tv[None, :, None, :] - q[:, None, :, :]) ** 2).sum(-1)     # (r, T, N)
        ok = np.all(d2 <= inst.betas[None, None, :] ** 2, axis=2)         # (r, T)
        rot_ok[c0:c0 + 256] = ok.any(1)
        trans_ok |= ok.any(0)
    # grid must contain the set strictly inside its box
    assert not rot_ok.reshape(nr, nr, nr)[[0, -1]].any() and not trans_ok.reshape(nt, nt, nt)[[0, -1]].any()
    grid_poses = np.zeros((int(rot_ok.sum()), 12))
    grid_poses[:, :9] = Rs[rot_ok].reshape(-1, 9)
    D_grid = oracle.megb(grid_poses, inst.R_gt)["rot_radius"]
    _, d_grid, _ = oracle.meb_welzl(tv[trans_ok])
    h_R = np.sqrt(3) * (axis_r[1] - axis_r[0])
    h_t = np.sqrt(3) * (axis_t[1] - axis_t[0])
    for res in (g, gt):                                   # any subset of S: never larger
        assert res["rot_radius"] <= D_grid + h_R
        assert res["trans_radius"] <= d_grid + h_t
    assert g["rot_radius"] >= 0.85 * D_grid               # each sampler on the set it targets
    assert gt["trans_radius"] >= 0.85 * d_grid


# ------------------------------------------------------------------ PCA normalisation of the centre velocity (R-23)
def test_pca_velocity_scale_closed_forms():
    """S = sqrtm(Cov) / sqrt(lambda_max): exact on a cloud with a known covariance."""
    from scipy.spatial.transform import Rotation
    Q = Rotation.from_rotvec([0.3, -0.7, 0.2]).as_matrix()
    sig = np.array([3.0, 1.0, 0.1])
    # +-sigma_k along each principal axis: covariance Q diag(sigma^2) Q^T / 3 exactly
    pts = np.concatenate([+sig[k] * Q[:, k][None, :] for k in range(3)] + [-sig[k] * Q[:, k][None, :] for k in range(3)])
    S0 = np.zeros((6, 12)); S0[:, :9] = np.eye(3).reshape(9); S0[:, 9:] = pts + np.array([5.0, -2.0, 1.0])
    S = oracle.pca_velocity_scale(S0)
    assert np.allclose(S, Q @ np.diag(sig / sig.max()) @ Q.T, atol=1e-13)
    assert np.allclose(S, S.T) and np.allclose(S @ Q[:, 0], Q[:, 0])            # longest axis kept, others shrunk
    iso = S0.copy(); iso[:, 9:] = np.concatenate([np.eye(3), -np.eye(3)])
    assert np.allclose(oracle.pca_velocity_scale(iso), np.eye(3), atol=1e-14)   # no anisotropy, no rescaling
    assert np.array_equal(oracle.pca_velocity_scale(S0[:1]), np.eye(3))        # a single pose has no spread


def test_pca_velocity_changes_only_the_direction_of_travel():
    """Rotation frozen (theta_p = 0): the walker moves along its velocity; with the flag the displacement is
    parallel to S times the unflagged displacement direction, and an isotropic S_0 changes nothing."""
    import copy
    inst = I.make_instance(1)
    S0 = I.make_init_poses(inst, 32)
    S0[:, 9] = inst.t_gt[0] + (S0[:, 9] - inst.t_gt[0]) * 0.05                  # squeeze the cloud along x
    P = copy.copy(inst.params); P.mode = I.MODE_TRANS; P.theta_p = 0.0; P.v0 = 0.02; P.n_p = 4; P.n_p_star = 1; P.n_t = 12
    Pf = copy.copy(P); Pf.flags = 64
    ids = np.arange(40)
    a, _ = oracle.walk(inst, P, S0, ids, 1, 3)
    b, _ = oracle.walk(inst, Pf, S0, ids, 1, 3)
    S = oracle.pca_velocity_scale(S0)
    assert S[0, 0] < 0.5                                                         # x is the thin direction
    moved = 0
    for w in ids:
        t0 = S0[w % 32, 9:]
        da, db = a[w, 9:] - t0, b[w, 9:] - t0
        if np.linalg.norm(da) > 1e-6 and np.linalg.norm(db) > 1e-6:
            moved += 1
            assert np.linalg.norm(np.cross(S @ da, db)) <= 1e-9 * np.linalg.norm(S @ da) * np.linalg.norm(db)
    assert moved > 10


# ----------------------------------------------------------------------------- body pivot of update_rotation (R-1)

def _shifted(inst, c):
    """The same problem with source points a - c: pose (R, tau = t + R c) there is pose (R, t) here."""
    out = copy.copy(inst)
    meas = np.array(inst.measurements, dtype=np.float64, copy=True)
    lo = 0 if inst.residual_type == I.REG_3D3D else 2
    meas[:, lo:lo + 3] -= c
    out.measurements = meas
    return out


@pytest.mark.parametrize("config", [1, 3])
def test_body_pivot_keeps_the_pivot_point_fixed_and_equals_the_recentred_problem(config):
    """update_rotation about a body point c ("object movement"; R-1): (a) pivot 0 is the
    default walk bit for bit; (b) an accepted step leaves the image of c where the perturbed pose had it,
    R' c + t' = R* c + t_j; (c) the walk equals the pivot-free walk of the problem re-centred at c
    (source points a - c, translations tau = t + R c), mapped back by t = tau - R c."""
    inst = I.make_instance(config)
    S0 = I.make_init_poses(inst, 16)
    P = copy.copy(inst.params); P.n_p = 12; P.n_p_star = 3; P.n_t = 8
    c = np.array([0.3, -0.2, 0.45])
    Pc = copy.copy(P); Pc.pivot = tuple(c)
    P0 = copy.copy(P); P0.pivot = (0.0, 0.0, 0.0)
    ids = np.arange(48)
    base = oracle.walk(inst, P, S0, ids, 6, 5, trace=True)
    zero = oracle.walk(inst, P0, S0, ids, 6, 5, trace=True)
    assert np.array_equal(base[0], zero[0]) and np.array_equal(base[2], zero[2])            # (a)

    one, _, tr, _ = oracle.walk(inst, Pc, S0, ids, 1, 5, trace=True)                         # (b)
    moved = 0
    for w in ids:
        m0, j0 = int(tr[w, 0]) & 0xFF, int(tr[w, 0]) >> 8
        R0, t0 = S0[w % 16, :9].reshape(3, 3), S0[w % 16, 9:]
        R1, t1 = one[w, :9].reshape(3, 3), one[w, 9:]
        if m0 == 0:
            assert np.array_equal(one[w], S0[w % 16])
            continue
        x = oracle.philox4x32_10([w, 1, j0, 1], [5, 0])
        tj = t0 + P.t_p * np.array([oracle.u32_to_pm1(int(x[r])) for r in range(3)])
        assert np.abs((R1 @ c + t1) - (R0 @ c + tj)).max() < 1e-12
        assert np.abs(R1 - R0).max() > 1e-6                                                  # it did rotate
        moved += 1
    assert moved > 20

    sh = _shifted(inst, c)                                                                   # (c)
    S0s = S0.copy()
    S0s[:, 9:] += S0[:, :9].reshape(-1, 3, 3) @ c
    a_smp, a_flag, a_tr, a_sl = oracle.walk(inst, Pc, S0, ids, 6, 5, trace=True)
    b_smp, b_flag, b_tr, b_sl = oracle.walk(sh, P0, S0s, ids, 6, 5, trace=True)
    same = 0
    for w in ids:
        if not np.array_equal(a_tr[w], b_tr[w]):
            first = int(np.argmax(a_tr[w] != b_tr[w]))
            assert min(a_sl[w, first], b_sl[w, first]) < 1e-9                               # a near-tie only
            continue
        back = b_smp[w].copy()
        back[9:] -= b_smp[w, :9].reshape(3, 3) @ c
        assert np.abs(back - a_smp[w]).max() < 1e-11 and a_flag[w] == b_flag[w]
        same += 1
    assert same >= 46
    assert np.abs(a_smp - base[0]).max() > 1e-3                                              # and it is a different walk
