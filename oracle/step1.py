"""CPU oracle for Step I of CLOSURE, "initialize starting poses", Ex.1, Ex.2 and Ex.3.

TEST INFRASTRUCTURE, NOT THE PRODUCT (see oracle/__init__.py).  Plain numpy, fp64, one trial at a time.

Ex.1: "In each RANSAG trial, we randomly select 3 constraints (i.e., 3 ellipses in Fig. 3(a)) and
find a 2D point in each constraint.  We then apply the perspective-3-point (P3P) minimal solver [22] to obtain a
candidate pose s.  We add s into the set S_0 if s satisfies (PURSE2D3D)."
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

Ex.1, R-24 (the paper names a P3P solver [22] and says nothing else):
* the three constraints: the triplet rule above (tag 2);
* "a 2D point in each constraint": y_l = z_l + beta_l e_l with e_l uniform in the unit disc, drawn by rejection from
  the square: Philox counter (k_lo32, l, a, 4 | k_hi32 << 8) for attempt a = 0..7 gives two candidate points
  (xi(x0), xi(x1)) and (xi(x2), xi(x3)), xi as in R-5; the first with e0^2 + e1^2 <= 1 is taken (centre of the disc if
  all 16 fail, probability 2e-11);
* P3P = the classical distance formulation (Grunert 1841; Haralick et al. 1994 review it): unit bearings f_l of the
  y_l, depths d_l > 0 with |d_i f_i - d_j f_j|^2 = |Z_i - Z_j|^2.  With d_2 = u d_1, d_3 = v d_1 the three equations
  reduce to a quartic in v (derivation at `p3p_quartic`); every positive real root with u > 0 gives depths, polished
  by three Newton steps on the three distance equations, and the pose is the rigid fit (Arun, exact for a congruent
  triangle) of Z_l -> d_l f_l;
* ellipse form (Lambda_i != I): y_l = z_l + beta_l L^-T e_l with Lambda_l = L L^T (Cholesky), uniform in the ellipse;
* up to four poses per trial: they are tried in ascending order of d_1 and the first that satisfies
  (PURSE2D3D) enters S_0 (one pose per trial).
"""
from __future__ import annotations

import numpy as np

import oracle

TAG_TRIPLET, TAG_WEIGHTS, TAG_DISC = 2, 3, 4
REPROJ_2D3D, REG_3D3D, POSE_REG, POSE_REG_SPLIT, REG_3D3D_ELL, REPROJ_2D3D_ELL = 1, 2, 3, 4, 5, 6


def trial_words(seed: int, k: int, c: int, tag: int, a: int = 0) -> np.ndarray:
    ctr = [k & 0xFFFFFFFF, c, a, tag | (((k >> 32) & 0xFFFFFF) << 8)]
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


def disc_point(seed: int, k: int, l: int) -> tuple[float, float]:
    """Uniform point of the unit disc for the l-th selected constraint of trial k (R-24)."""
    for a in range(8):
        x = trial_words(seed, k, l, TAG_DISC, a)
        for h in (0, 2):
            e0 = oracle.u32_to_pm1(int(x[h]))
            e1 = oracle.u32_to_pm1(int(x[h + 1]))
            if e0 * e0 + e1 * e1 <= 1.0:
                return e0, e1
    return 0.0, 0.0


def bearing(y, K) -> np.ndarray:
    """Unit vector of the ray through pixel y: K = (fx, fy, cx, cy), Pi(v) = [v1/v3, v2/v3]."""
    m0 = (y[0] - K[2]) / K[0]
    m1 = (y[1] - K[3]) / K[1]
    nrm = np.sqrt(m0 * m0 + m1 * m1 + 1.0)
    return np.array([m0 / nrm, m1 / nrm, 1.0 / nrm])


def p3p_quartic(f: np.ndarray, X: np.ndarray):
    """Coefficients (ascending) of the quartic in v = d_3/d_1, and p, q with u = d_2/d_1 = p(v)/q(v).

    c_ij = f_i . f_j, a_ij = |X_i - X_j|^2.  The law of cosines in the three faces of the tetrahedron (camera
    centre, X_1, X_2, X_3):
        d_1^2 (1 + u^2 - 2 c_12 u)       = a_12        (1)
        d_1^2 (1 + v^2 - 2 c_13 v)       = a_13        (2)
        d_1^2 (u^2 + v^2 - 2 c_23 u v)   = a_23        (3)
    (1)/(2):  a_13 (1 + u^2 - 2 c_12 u) = a_12 s(v),   s(v) = 1 + v^2 - 2 c_13 v        (A)
    (3)/(2):  a_13 (u^2 + v^2 - 2 c_23 u v) = a_23 s(v)                                  (B)
    (A) - (B) is linear in u:  u q(v) = p(v),  p = (a_23 - a_12) s(v) + a_13 (1 - v^2),  q = 2 a_13 (c_12 - c_23 v).
    u = p/q in (A) times q^2:  G(v) = a_13 (q^2 + p^2 - 2 c_12 p q) - a_12 s q^2 = 0.
    """
    P = np.polynomial.polynomial
    c12, c13, c23 = float(f[0] @ f[1]), float(f[0] @ f[2]), float(f[1] @ f[2])
    a12 = float((X[0] - X[1]) @ (X[0] - X[1]))
    a13 = float((X[0] - X[2]) @ (X[0] - X[2]))
    a23 = float((X[1] - X[2]) @ (X[1] - X[2]))
    s = np.array([1.0, -2.0 * c13, 1.0])
    p = P.polyadd((a23 - a12) * s, a13 * np.array([1.0, 0.0, -1.0]))
    q = 2.0 * a13 * np.array([c12, -c23])
    q2 = P.polymul(q, q)
    G = P.polysub(a13 * P.polyadd(P.polyadd(q2, P.polymul(p, p)), -2.0 * c12 * P.polymul(p, q)),
                  a12 * P.polymul(s, q2))
    G = np.concatenate([G, np.zeros(5 - G.size)])
    return G, p, q, (c12, c13, c23), (a12, a13, a23)


def p3p(f: np.ndarray, X: np.ndarray):
    """All poses (R, t) with  d_l f_l = R X_l + t, d_l > 0  ->  (list of (d, R, t) in ascending d_1, ill_conditioned).

    `ill_conditioned` is True when the set of solutions is not stable under rounding (a nearly double root of the
    quartic, a vanishing leading coefficient or q(v), a nearly singular Jacobian of the distance equations): the
    parity test does not compare such trials.
    """
    P = np.polynomial.polynomial
    f = np.asarray(f, dtype=np.float64)
    X = np.asarray(X, dtype=np.float64)
    G, p, q, (c12, c13, c23), (a12, a13, a23) = p3p_quartic(f, X)
    ill = False
    gmax = np.abs(G).max()
    if not (gmax > 0.0) or abs(G[4]) < 1e-9 * gmax:
        return [], True
    roots = np.roots(G[::-1])
    dG = P.polyder(G)
    sols = []
    for r in roots:
        rel_im = abs(r.imag) / (1.0 + abs(r.real))
        if rel_im > 1e-7:
            if rel_im < 3e-5:
                ill = True                                   # a complex pair within rounding of the real axis
            continue
        v = float(r.real)
        for _ in range(20):                                  # Newton on G from numpy's eigenvalue
            g1 = P.polyval(v, dG)
            if g1 == 0.0:
                break
            v -= P.polyval(v, G) / g1
        scale = sum(abs(G[i]) * abs(v) ** i for i in range(5))
        if abs(P.polyval(v, dG)) * (1.0 + abs(v)) < 1e-10 * scale:
            ill = True                                       # nearly a double root
        if not v > 0.0:
            continue
        if any(abs(v - w[0]) <= 1e-9 * (1.0 + abs(v)) for w in sols):
            ill = True
            continue
        qv = P.polyval(v, q)
        if abs(qv) < 1e-9 * (abs(q[0]) + abs(q[1] * v)):
            ill = True
            continue
        u = P.polyval(v, p) / qv
        if not u > 0.0:
            if abs(u) < 1e-9:
                ill = True
            continue
        d1 = np.sqrt(a13 / (1.0 + v * v - 2.0 * c13 * v))
        d = np.array([d1, u * d1, v * d1])
        for _ in range(3):                                   # Newton on the three distance equations
            F = np.array([d[0] * d[0] + d[1] * d[1] - 2.0 * c12 * d[0] * d[1] - a12,
                          d[0] * d[0] + d[2] * d[2] - 2.0 * c13 * d[0] * d[2] - a13,
                          d[1] * d[1] + d[2] * d[2] - 2.0 * c23 * d[1] * d[2] - a23])
            J = 2.0 * np.array([[d[0] - c12 * d[1], d[1] - c12 * d[0], 0.0],
                                [d[0] - c13 * d[2], 0.0, d[2] - c13 * d[0]],
                                [0.0, d[1] - c23 * d[2], d[2] - c23 * d[1]]])
            if np.linalg.cond(J) > 1e8:
                ill = True
                break
            d = d - np.linalg.solve(J, F)
        if not np.all(d > 0.0):
            continue
        sols.append((v, d))
    out = []
    for v, d in sorted(sols, key=lambda w: w[1][0]):
        cand = arun(X, d[:, None] * f)
        if cand is None:
            continue
        out.append((d, cand[0], cand[1]))
    for a, b in zip(out, out[1:]):
        if b[0][0] - a[0][0] < 1e-9 * b[0][0]:
            ill = True                                       # the order of the candidates is not decided
    return out, ill


def p3p_trial(inst, seed: int, k: int):
    """The candidate poses of trial k of Ex.1 -> (list of (d, R, t), ill_conditioned, (indices, pixels))."""
    meas = np.asarray(inst.measurements, dtype=np.float64)
    betas = np.asarray(inst.betas, dtype=np.float64).reshape(-1)
    K = np.asarray(inst.intrinsics, dtype=np.float64).reshape(4)
    idx = list(triplet(seed, k, meas.shape[0]))
    ys = []
    for l, i in enumerate(idx):
        e0, e1 = disc_point(seed, k, l)
        if int(inst.residual_type) == REPROJ_2D3D_ELL:
            # uniform in the ellipse (y - z)^T Lambda (y - z) <= beta^2: with Lambda = L L^T the map
            # e -> z + beta L^-T e takes the unit disc onto it (a linear map keeps the uniform measure uniform)
            L = np.linalg.cholesky(meas[i, 5:9].reshape(2, 2))
            x = np.linalg.solve(L.T, np.array([e0, e1]))
            ys.append((meas[i, 0] + betas[i] * x[0], meas[i, 1] + betas[i] * x[1]))
        else:
            ys.append((meas[i, 0] + betas[i] * e0, meas[i, 1] + betas[i] * e1))
    X = meas[idx, 2:5]
    ac = X - X.mean(axis=0)
    if np.linalg.norm(np.cross(ac[0], ac[1])) < 1e-8:
        return [], False, (idx, ys)
    f = np.stack([bearing(y, K) for y in ys])
    sols, ill = p3p(f, X)
    return sols, ill, (idx, ys)


def init_sample(inst, num_trials: int, seed: int, trial_begin: int = 0):
    """-> poses (num_trials, 12) (zeros where rejected), ok (num_trials,) uint8, in trial order."""
    ty = int(inst.residual_type)
    meas = np.asarray(inst.measurements, dtype=np.float64)
    n = meas.shape[0]
    poses = np.zeros((num_trials, 12))
    ok = np.zeros(num_trials, dtype=np.uint8)
    for q in range(num_trials):
        k = trial_begin + q
        if ty in (REG_3D3D, REG_3D3D_ELL):               # the ellipsoid norm changes the PURSE test only
            if n < 3:
                raise ValueError("RANSAG needs at least 3 correspondences")
            idx = list(triplet(seed, k, n))
            cand = arun(meas[idx, 0:3], meas[idx, 3:6])
        elif ty in (POSE_REG, POSE_REG_SPLIT):
            cand = convex_pose(meas, convex_weights(seed, k, n))
        elif ty in (REPROJ_2D3D, REPROJ_2D3D_ELL):
            if n < 3:
                raise ValueError("RANSAG needs at least 3 correspondences")
            cand = None
            for _, Rc, tc in p3p_trial(inst, seed, k)[0]:        # ascending d_1: the first feasible one
                if oracle.in_purse(inst, Rc.reshape(9), tc):
                    cand = (Rc, tc)
                    break
        else:
            raise ValueError("Step I is not built for this residual type")
        if cand is None:
            continue
        R, t = cand
        if oracle.in_purse(inst, R.reshape(9), t):
            poses[q, :9] = R.reshape(9)
            poses[q, 9:] = t
            ok[q] = 1
    return poses, ok
