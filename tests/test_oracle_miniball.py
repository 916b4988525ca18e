"""Pins for the oracle's miniball / MEGB (Step III).

The minimum enclosing ball is unique: closed forms, the definition by
enumeration, and invariances fix it without reference to any implementation.
"""
import numpy as np
import pytest
from scipy.spatial.transform import Rotation

import oracle


def test_two_points():
    c, r, sup = oracle.meb_brute(np.array([[0.0, 0, 0], [2.0, 0, 0]]))
    assert np.allclose(c, [1, 0, 0]) and abs(r - 1.0) < 1e-15 and set(sup) == {0, 1}
    c, r, sup = oracle.meb_welzl(np.array([[0.0, 0, 0], [2.0, 0, 0]]))
    assert np.allclose(c, [1, 0, 0]) and abs(r - 1.0) < 1e-15 and set(sup) == {0, 1}


def test_single_and_duplicate_points():
    c, r, _ = oracle.meb_welzl(np.array([[1.0, 2, 3]]))
    assert np.allclose(c, [1, 2, 3]) and r == 0.0
    c, r, _ = oracle.meb_welzl(np.tile([[1.0, 2, 3, 4]], (7, 1)))
    assert np.allclose(c, [1, 2, 3, 4]) and r == 0.0


@pytest.mark.parametrize("d", [3, 4])
def test_regular_simplex(d):
    # vertices e_k of the standard simplex in R^(d+1) are equidistant; project to R^d by
    # dropping the barycentre direction (QR) -> regular simplex with circumradius sqrt(d/(d+1))
    E = np.eye(d + 1) - 1.0 / (d + 1)
    Q, _ = np.linalg.qr(E[:, :d])
    P = E @ Q                                              # (d+1, d) coordinates
    c, r, sup = oracle.meb_welzl(P + 3.0)
    assert abs(r - np.sqrt(d / (d + 1.0))) < 1e-14
    assert np.allclose(c, 3.0, atol=1e-14) and len(sup) == d + 1
    cb, rb, _ = oracle.meb_brute(P + 3.0)
    assert abs(rb - r) < 1e-14 and np.allclose(cb, c, atol=1e-14)


@pytest.mark.parametrize("d", [2, 3, 4])
def test_points_on_known_sphere_plus_interior(d):
    rng = np.random.default_rng(d)
    # antipodal pairs guarantee the known sphere is the MEB
    v = rng.standard_normal((20, d))
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    pts = np.concatenate([v, -v[:3], 0.7 * rng.uniform(-1, 1, (200, d)) / np.sqrt(d)]) * 2.5 + 1.0
    c, r, _ = oracle.meb_welzl(rng.permutation(pts))
    assert abs(r - 2.5) < 1e-13 and np.allclose(c, 1.0, atol=1e-13)


@pytest.mark.parametrize("d,n,seed", [(3, 9, 0), (3, 12, 1), (4, 8, 2), (4, 11, 3), (2, 12, 4)])
def test_welzl_equals_definition_on_tiny_inputs(d, n, seed):
    rng = np.random.default_rng(seed)
    pts = rng.standard_normal((n, d))
    cb, rb, sb = oracle.meb_brute(pts)
    for sh in range(4):
        c, r, s = oracle.meb_welzl(pts, shuffle_seed=sh)
        assert abs(r - rb) < 1e-13 and np.allclose(c, cb, atol=1e-13)
        assert set(s) == set(sb)
    dist = np.linalg.norm(pts - cb, axis=1)
    assert np.all(dist <= rb * (1 + 1e-12)) and np.sum(np.abs(dist - rb) < 1e-12) >= 2


def test_invariances_and_monotonicity():
    rng = np.random.default_rng(10)
    pts = rng.standard_normal((500, 4)) * [1.0, 0.3, 2.0, 0.1]
    c, r, _ = oracle.meb_welzl(pts)
    assert np.all(np.linalg.norm(pts - c, axis=1) <= r * (1 + 1e-12))
    c2, r2, _ = oracle.meb_welzl(rng.permutation(pts), shuffle_seed=5)
    assert abs(r - r2) < 1e-13 and np.allclose(c, c2, atol=1e-12)
    Q, _ = np.linalg.qr(rng.standard_normal((4, 4)))
    shift = np.array([5.0, -3, 2, 1])
    c3, r3, _ = oracle.meb_welzl(pts @ Q.T + shift)
    assert abs(r - r3) < 1e-12 and np.allclose(c3, Q @ c + shift, atol=1e-12)
    # Prop. 4: the ball of a subset is never larger
    for k in (5, 50, 250):
        assert oracle.meb_welzl(pts[:k])[1] <= r + 1e-13


def test_cospherical_quaternion_cloud():
    """All quaternions lie on the unit 3-sphere (degenerate for naive solvers)."""
    rng = np.random.default_rng(4)
    R0 = Rotation.random(random_state=1)
    cloud = (Rotation.from_rotvec(0.2 * rng.uniform(-1, 1, (3000, 3))) * R0).as_quat()  # xyzw
    q = cloud[:, [3, 0, 1, 2]]
    q *= np.sign(q @ q[0])[:, None]
    c, r, sup = oracle.meb_welzl(q)
    d = np.linalg.norm(q - c, axis=1)
    assert np.all(d <= r * (1 + 1e-12)) and 2 <= len(sup) <= 5
    h = np.linalg.norm(c)
    assert abs(h * h + r * r - 1.0) < 1e-12                 # centre of a cap: h^2 + r^2 = 1 (R-16)


def test_quaternion_roundtrip_and_sign():
    L = oracle.lib()
    import ctypes
    rng = np.random.default_rng(0)
    for k in range(50):
        rot = Rotation.random(random_state=k) if k else Rotation.from_rotvec([np.pi - 1e-9, 0, 0])
        R = np.ascontiguousarray(rot.as_matrix().reshape(9))
        q = np.zeros(4); R2 = np.zeros(9)
        L.ora_quat_from_rotation(R.ctypes.data_as(ctypes.POINTER(ctypes.c_double)),
                                 q.ctypes.data_as(ctypes.POINTER(ctypes.c_double)))
        L.ora_rotation_from_quat(q.ctypes.data_as(ctypes.POINTER(ctypes.c_double)),
                                 R2.ctypes.data_as(ctypes.POINTER(ctypes.c_double)))
        assert np.allclose(R, R2, atol=1e-14) and abs(np.linalg.norm(q) - 1) < 1e-15
        ref = rot.as_quat()[[3, 0, 1, 2]]
        assert min(np.linalg.norm(q - ref), np.linalg.norm(q + ref)) < 1e-14


def test_megb_geodesic_ball_of_known_radius():
    """Rotations at geodesic angle exactly alpha from C in antipodal direction pairs, plus
    interior ones: MEGB = (C, alpha); translations on a sphere of radius rho about c."""
    rng = np.random.default_rng(8)
    C = Rotation.random(random_state=3)
    alpha, rho = 0.3, 0.07
    c = np.array([0.5, -1.0, 2.0])
    dirs = rng.standard_normal((15, 3))
    dirs /= np.linalg.norm(dirs, axis=1, keepdims=True)
    dirs = np.concatenate([dirs, -dirs])
    rots = [Rotation.from_rotvec(alpha * u) * C for u in dirs] + \
           [Rotation.from_rotvec(alpha * rng.uniform(0, 0.9) * u) * C for u in dirs]
    ts = [c + rho * u for u in dirs] + [c + rho * 0.5 * u for u in dirs]
    samples = np.array([np.concatenate([r.as_matrix().reshape(9), t]) for r, t in zip(rots, ts)])
    g = oracle.megb(samples, C.as_matrix())
    assert abs(g["rot_radius"] - alpha) < 1e-12
    assert abs(g["trans_radius"] - rho) < 1e-13
    assert Rotation.from_matrix(g["R"] @ C.as_matrix().T).magnitude() < 1e-12
    assert np.allclose(g["t"], c, atol=1e-13)
    # geodesic distance of every sample to the centre is within the radius
    for r in rots:
        ang = np.arccos(np.clip((np.trace(g["R"].T @ r.as_matrix()) - 1) / 2, -1, 1))
        assert ang <= g["rot_radius"] + 1e-7
    assert all(i < len(dirs) for i in g["rot_support"]) and all(i < len(dirs) for i in g["trans_support"])
    # sign alignment (R-15): a reference on the far side of the double cover changes nothing
    g2 = oracle.megb(samples, (Rotation.from_rotvec([0, 0, 0.2]) * C).as_matrix())
    assert abs(g2["rot_radius"] - alpha) < 1e-12


def test_compact_is_stable_filter():
    rng = np.random.default_rng(1)
    s = rng.standard_normal((100, 12))
    f = (rng.uniform(size=100) < 0.4).astype(np.uint8)
    out = oracle.compact(s, f)
    assert np.array_equal(out, s[f.astype(bool)])
    assert oracle.compact(s, np.zeros(100, np.uint8)).shape == (0, 12)
