"""CPU oracle for Step I of CLOSURE, "initialize starting poses", Ex.2 and Ex.3.

TEST INFRASTRUCTURE, NOT THE PRODUCT (see oracle/__init__.py).  Plain numpy, fp64, one trial at a time.

Ex.2: "In each RANSAG trial, we randomly select 3 pairs of corresponding points, and apply
Arun's Method [6] to compute a candidate pose s.  We put s into S_0 if s satisfies (PURSE3D3D)."
Ex.3: "In each trial, we randomly generate a convex combination of 10 pose hypotheses to
compute a candidate pose s.  We put s into S_0 if s satisfies (PURSEreg)."

The paper fixes neither the random numbers nor how rotations are combined; R-21 / R-22:
* random words of trial k: Philox4x32-10, counter (k_lo32, c, 0, tag | k_hi32 << 8), key = seed;
  tag 2 = triplet (c = 0), tag 3 = weights (word 4c + l of the stream feeds hypothesis 4c + l);
* triplet: i1 = x0 mod N, i2 = x1 mod (N-1), i3 = x2 mod (N-2), each skipping the indices already taken
  (three distinct correspondences); a triplet whose source or target triangle has a normal shorter than
  1e-8 is degenerate and the trial is rejected;
* Arun's method = least-squares rigid fit: H = sum (a_k - a_bar)(b_k - b_bar)^T = U S V^T,
  R = V diag(1, 1, det(V U^T)) U^T, t = b_bar - R a_bar (the determinant guard is Arun's own remedy for
  the reflection case, which is the generic case for three points: H has rank 2);
* convex combination: u_i = (x_i + 1/2) 2^-32, w_i = u_i / sum u, R = proj_SO(3)(sum w_i R_i) as in
  Alg. 2 l.3, t = sum w_i t_i; rejected if sum w_i R_i has no positive determinant;
* a candidate enters S_0 iff it satisfies the PURSE (squared form, R-9).
"""
from __future__ import annotations

import numpy as np

import oracle

TAG_TRIPLET, TAG_WEIGHTS = 2, 3
REPROJ_2D3D, REG_3D3D, POSE_REG, POSE_REG_SPLIT = 1, 2, 3, 4


def trial_words(seed: int, k: int, c: int, tag: int) -> np.ndarray:
    ctr = [k & 0xFFFFFFFF, c, 0, tag | (((k >> 32) & 0xFFFFFF) << 8)]
    return oracle.philox4x32_10(ctr, [seed & 0xFFFFFFFF, (seed >> 32) & 0xFFFFFFFF])


def triplet(seed: int, k: int, n: int) -> tuple[int, int, int]:
    x = trial_words(seed, k, 0, TAG_TRIPLET)
    i1 = int(x[0]) % n
    i2 = int(x[1]) % (n - 1)
    if i2 >= i1:
        i2 += 1
    i3 = int(x[2]) % (n - 2)
    for taken in sorted((i1, i2)):
        if i3 >= taken:
            i3 += 1
    return i1, i2, i3


def arun(a: np.ndarray, b: np.ndarray):
    """Least-squares (R, t) with b_k ~ R a_k + t (Arun, Huang, Blostein 1987).  None if degenerate."""
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    abar, bbar = a.mean(axis=0), b.mean(axis=0)
    ac, bc = a - abar, b - bbar
    if a.shape[0] == 3:
        if np.linalg.norm(np.cross(ac[0], ac[1])) < 1e-8 or np.linalg.norm(np.cross(bc[0], bc[1])) < 1e-8:
            return None
    H = ac.T @ bc
    U, _, Vt = np.linalg.svd(H)
    V = Vt.T
    D = np.diag([1.0, 1.0, float(np.sign(np.linalg.det(V @ U.T)))])
    R = V @ D @ U.T
    return R, bbar - R @ abar


def convex_weights(seed: int, k: int, n: int) -> np.ndarray:
    u = np.empty(n)
    for c in range((n + 3) // 4):
        x = trial_words(seed, k, c, TAG_WEIGHTS)
        for l in range(4):
            if 4 * c + l < n:
                u[4 * c + l] = (float(x[l]) + 0.5) * 2.0 ** -32
    s = 0.0
    for i in range(n):                      # left to right
        s += u[i]
    return u / s


def convex_pose(meas: np.ndarray, w: np.ndarray):
    M = np.zeros((3, 3))
    t = np.zeros(3)
    for i in range(meas.shape[0]):
        M += w[i] * meas[i, :9].reshape(3, 3)
        t += w[i] * meas[i, 9:12]
    if not np.linalg.det(M) > 0.0:
        return None
    U, _, Vt = np.linalg.svd(M)
    return U @ Vt, t                        # det M > 0  =>  U V^T is the nearest rotation


def init_sample(inst, num_trials: int, seed: int, trial_begin: int = 0):
    """-> poses (num_trials, 12) (zeros where rejected), ok (num_trials,) uint8, in trial order."""
    ty = int(inst.residual_type)
    meas = np.asarray(inst.measurements, dtype=np.float64)
    n = meas.shape[0]
    poses = np.zeros((num_trials, 12))
    ok = np.zeros(num_trials, dtype=np.uint8)
    for q in range(num_trials):
        k = trial_begin + q
        if ty == REG_3D3D:
            if n < 3:
                raise ValueError("RANSAG needs at least 3 correspondences")
            idx = list(triplet(seed, k, n))
            cand = arun(meas[idx, 0:3], meas[idx, 3:6])
        elif ty in (POSE_REG, POSE_REG_SPLIT):
            cand = convex_pose(meas, convex_weights(seed, k, n))
        else:
            raise ValueError("Step I for the reprojection residual needs a P3P solver (not built)")
        if cand is None:
            continue
        R, t = cand
        if oracle.in_purse(inst, R.reshape(9), t):
            poses[q, :9] = R.reshape(9)
            poses[q, 9:] = t
            ok[q] = 1
    return poses, ok
