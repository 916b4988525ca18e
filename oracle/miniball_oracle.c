/*
 * miniball_oracle.c -- plain CPU oracle for Step III of CLOSURE:
 * the minimum enclosing ball of the boundary samples in R^3 (translations, eq. (12)
 * PAPER.md:131) and in R^4 (unit quaternions), and the geodesic radius.
 *
 * TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as closure_oracle.c).  Shares nothing
 * with the library's Gaertner-style solver in paper_2403_09990_b200/csrc/.
 *
 * The minimum enclosing ball is unique, so the oracle is its definition:
 *   ora_meb_brute  -- the definition written out: the smallest ball among those spanned
 *                     by every subset of <= d+1 points that contains all points
 *                     (tiny inputs only, O(n^(d+2)));
 *   ora_meb_welzl  -- Welzl's recursion (E. Welzl, "Smallest enclosing disks (balls and
 *                     ellipsoids)", 1991) with move-to-front, for the sample clouds.
 * tests/test_oracle_miniball.py pins the second to the first, and both to closed forms.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define MB_MAXD 8

typedef struct {
    int d;
    const double *pts;
    double c[MB_MAXD];
    double r2;
} mb_ball;

/* Smallest ball whose boundary passes through the k given points (k <= d+1), centre in
 * their affine hull: c = p0 + sum_j lam_j (p_j - p0), 2 (p_j-p0).(p_l-p0) lam = |p_j-p0|^2.
 * Returns 0 when the points are (numerically) affinely dependent. */
static int ball_through(int d, const double *pts, const int64_t *idx, int k, double *c, double *r2)
{
    if (k == 0) {
        for (int a = 0; a < d; ++a) c[a] = 0.0;
        *r2 = -1.0;
        return 1;
    }
    const double *p0 = pts + (size_t)idx[0] * d;
    int m = k - 1;
    double Q[MB_MAXD][MB_MAXD + 1], V[MB_MAXD][MB_MAXD];
    for (int j = 0; j < m; ++j)
        for (int a = 0; a < d; ++a)
            V[j][a] = pts[(size_t)idx[j + 1] * d + a] - p0[a];
    double scale = 0.0;
    for (int j = 0; j < m; ++j) {
        for (int l = 0; l < m; ++l) {
            double s = 0.0;
            for (int a = 0; a < d; ++a) s += V[j][a] * V[l][a];
            Q[j][l] = 2.0 * s;
        }
        Q[j][m] = 0.5 * Q[j][j];
        if (Q[j][j] > scale) scale = Q[j][j];
    }
    /* Gaussian elimination, partial pivoting */
    for (int col = 0; col < m; ++col) {
        int piv = col;
        for (int r = col + 1; r < m; ++r)
            if (fabs(Q[r][col]) > fabs(Q[piv][col])) piv = r;
        if (fabs(Q[piv][col]) <= 1e-14 * scale) return 0;
        if (piv != col)
            for (int e = 0; e <= m; ++e) { double tmp = Q[col][e]; Q[col][e] = Q[piv][e]; Q[piv][e] = tmp; }
        for (int r = col + 1; r < m; ++r) {
            double f = Q[r][col] / Q[col][col];
            for (int e = col; e <= m; ++e) Q[r][e] -= f * Q[col][e];
        }
    }
    double lam[MB_MAXD];
    for (int r = m - 1; r >= 0; --r) {
        double s = Q[r][m];
        for (int e = r + 1; e < m; ++e) s -= Q[r][e] * lam[e];
        lam[r] = s / Q[r][r];
    }
    double rr = 0.0;
    for (int a = 0; a < d; ++a) {
        double off = 0.0;
        for (int j = 0; j < m; ++j) off += lam[j] * V[j][a];
        c[a] = p0[a] + off;
        rr += off * off;
    }
    *r2 = rr;
    return 1;
}

static double dist2(int d, const double *a, const double *b)
{
    double s = 0.0;
    for (int e = 0; e < d; ++e) s += (a[e] - b[e]) * (a[e] - b[e]);
    return s;
}

/* ---- the definition, by enumeration ---- */
static void brute_rec(int d, const double *pts, int64_t n, int64_t start, int64_t *sub, int k, int kmax,
                      double *best_c, double *best_r2, int64_t *best_sub, int *best_k)
{
    if (k > 0) {
        double c[MB_MAXD], r2;
        if (ball_through(d, pts, sub, k, c, &r2)) {
            int all_in = 1;
            double tol = 1e-12 * (r2 > 1.0 ? r2 : 1.0);
            for (int64_t q = 0; q < n && all_in; ++q)
                if (dist2(d, pts + (size_t)q * d, c) > r2 + tol) all_in = 0;
            if (all_in && (*best_r2 < 0.0 || r2 < *best_r2)) {
                *best_r2 = r2;
                memcpy(best_c, c, sizeof(double) * d);
                memcpy(best_sub, sub, sizeof(int64_t) * k);
                *best_k = k;
            }
        }
    }
    if (k == kmax) return;
    for (int64_t q = start; q < n; ++q) {
        sub[k] = q;
        brute_rec(d, pts, n, q + 1, sub, k + 1, kmax, best_c, best_r2, best_sub, best_k);
    }
}

int ora_meb_brute(const double *pts, int64_t n, int d, double *center, double *radius,
                  int64_t *support, int *n_support)
{
    if (n <= 0 || d <= 0 || d > MB_MAXD) return -1;
    int64_t sub[MB_MAXD + 1];
    double best_r2 = -1.0;
    int best_k = 0;
    brute_rec(d, pts, n, 0, sub, 0, d + 1, center, &best_r2, support, &best_k);
    if (best_r2 < 0.0) return -1;
    *radius = sqrt(best_r2);
    *n_support = best_k;
    return 0;
}

/* ---- Welzl's recursion with move-to-front ---- */
typedef struct {
    int d;
    const double *pts;
    int64_t *order;        /* permutation of point indices, front = most recently violating */
    int64_t basis[MB_MAXD + 1];
    int nb;
    double c[MB_MAXD];
    double r2;
} welzl_state;

static void welzl(welzl_state *S, int64_t n_end)
{
    /* ball of the current basis */
    if (!ball_through(S->d, S->pts, S->basis, S->nb, S->c, &S->r2)) return;
    if (S->nb == S->d + 1) return;
    for (int64_t i = 0; i < n_end; ++i) {
        int64_t p = S->order[i];
        double e = dist2(S->d, S->pts + (size_t)p * S->d, S->c) - S->r2;
        double tol = 1e-14 * (S->r2 > 0.0 ? S->r2 : 0.0);
        if (S->r2 < 0.0 || e > tol) {
            /* p lies outside: it is on the boundary of the ball of the first i+1 points */
            double c_save[MB_MAXD], r2_save = S->r2;
            memcpy(c_save, S->c, sizeof(c_save));
            S->basis[S->nb++] = p;
            double c_try[MB_MAXD], r2_try;
            if (ball_through(S->d, S->pts, S->basis, S->nb, c_try, &r2_try)) {
                welzl(S, i);
                /* keep the basis found by the recursion: trim to points on the boundary happens
                 * in the final support extraction */
                memmove(S->order + 1, S->order, sizeof(int64_t) * (size_t)i);
                S->order[0] = p;
                /* the recursion leaves S->basis possibly longer than nb+1; reset nb to the
                 * level of this frame and recompute with p included */
            } else {
                /* affinely dependent push: ignore the point (Gaertner's safeguard) */
                memcpy(S->c, c_save, sizeof(c_save));
                S->r2 = r2_save;
            }
            S->nb--;
        }
    }
}

/* The recursion above returns with the ball in (c, r2) but pops the basis on the way
 * out; the support set is recovered as the points at distance r (1e-10 relative). */
int ora_meb_welzl(const double *pts, int64_t n, int d, uint64_t shuffle_seed, double *center,
                  double *radius, int64_t *support, int *n_support, int max_support)
{
    if (n <= 0 || d <= 0 || d > MB_MAXD) return -1;
    welzl_state S;
    S.d = d; S.pts = pts; S.nb = 0; S.r2 = -1.0;
    S.order = (int64_t *)malloc(sizeof(int64_t) * (size_t)n);
    if (!S.order) return -1;
    for (int64_t i = 0; i < n; ++i) S.order[i] = i;
    /* random permutation (xorshift64*), expected linear time */
    uint64_t st = shuffle_seed * 0x9E3779B97F4A7C15ull + 0x2545F4914F6CDD1Dull;
    for (int64_t i = n - 1; i > 0; --i) {
        st ^= st >> 12; st ^= st << 25; st ^= st >> 27;
        uint64_t r = (st * 0x2545F4914F6CDD1Dull) >> 11;
        int64_t j = (int64_t)(r % (uint64_t)(i + 1));
        int64_t tmp = S.order[i]; S.order[i] = S.order[j]; S.order[j] = tmp;
    }
    welzl(&S, n);
    memcpy(center, S.c, sizeof(double) * d);
    double r2 = S.r2 > 0.0 ? S.r2 : 0.0;
    *radius = sqrt(r2);
    int ns = 0;
    for (int64_t i = 0; i < n && ns < max_support; ++i) {
        double e = dist2(d, pts + (size_t)i * d, S.c);
        if (fabs(e - r2) <= 1e-10 * (r2 > 1e-300 ? r2 : 1.0)) support[ns++] = i;
    }
    *n_support = ns;
    free(S.order);
    return 0;
}

/* ---- rotation matrix <-> unit quaternion (w, x, y, z), Shepperd's branch selection ---- */
void ora_quat_from_rotation(const double R[9], double q[4])
{
    double tr = R[0] + R[4] + R[8];
    if (tr > 0.0) {
        double s = sqrt(tr + 1.0) * 2.0;
        q[0] = 0.25 * s; q[1] = (R[7] - R[5]) / s; q[2] = (R[2] - R[6]) / s; q[3] = (R[3] - R[1]) / s;
    } else if (R[0] > R[4] && R[0] > R[8]) {
        double s = sqrt(1.0 + R[0] - R[4] - R[8]) * 2.0;
        q[0] = (R[7] - R[5]) / s; q[1] = 0.25 * s; q[2] = (R[1] + R[3]) / s; q[3] = (R[2] + R[6]) / s;
    } else if (R[4] > R[8]) {
        double s = sqrt(1.0 + R[4] - R[0] - R[8]) * 2.0;
        q[0] = (R[2] - R[6]) / s; q[1] = (R[1] + R[3]) / s; q[2] = 0.25 * s; q[3] = (R[5] + R[7]) / s;
    } else {
        double s = sqrt(1.0 + R[8] - R[0] - R[4]) * 2.0;
        q[0] = (R[3] - R[1]) / s; q[1] = (R[2] + R[6]) / s; q[2] = (R[5] + R[7]) / s; q[3] = 0.25 * s;
    }
    double nq = sqrt(q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3]);
    for (int e = 0; e < 4; ++e) q[e] /= nq;
}

void ora_rotation_from_quat(const double q[4], double R[9])
{
    double w = q[0], x = q[1], y = q[2], z = q[3];
    R[0] = 1 - 2 * (y * y + z * z); R[1] = 2 * (x * y - z * w); R[2] = 2 * (x * z + y * w);
    R[3] = 2 * (x * y + z * w); R[4] = 1 - 2 * (x * x + z * z); R[5] = 2 * (y * z - x * w);
    R[6] = 2 * (x * z - y * w); R[7] = 2 * (y * z + x * w); R[8] = 1 - 2 * (x * x + y * y);
}

/* MEGB of a sample cloud (Alg. 1 l.6-7).
 *   translations: MEB in R^3.
 *   rotations: q(R), sign aligned to q(Rbar) (R-15); MEB (c4, r4) in R^4; centre
 *   C = R(c4/|c4|); geodesic radius D = 2 arccos((1 + h^2 - r4^2) / (2h)), h = |c4| (R-16).
 * out[0..8] = C, out[9..11] = c, out[12] = D (rad), out[13] = d. */
int ora_megb(const double *samples, int64_t count, const double *Rbar, double *out,
             int64_t *rot_support, int *n_rot_support, int64_t *trans_support, int *n_trans_support)
{
    if (count <= 0) return -1;
    double *tp = (double *)malloc(sizeof(double) * 3 * (size_t)count);
    double *qp = (double *)malloc(sizeof(double) * 4 * (size_t)count);
    if (!tp || !qp) { free(tp); free(qp); return -1; }
    double qbar[4];
    ora_quat_from_rotation(Rbar, qbar);
    for (int64_t i = 0; i < count; ++i) {
        memcpy(tp + 3 * i, samples + 12 * i + 9, 3 * sizeof(double));
        double q[4];
        ora_quat_from_rotation(samples + 12 * i, q);
        double dot = q[0] * qbar[0] + q[1] * qbar[1] + q[2] * qbar[2] + q[3] * qbar[3];
        double sg = dot < 0.0 ? -1.0 : 1.0;
        for (int e = 0; e < 4; ++e) qp[4 * i + e] = sg * q[e];
    }
    double c3[3], d3, c4[4], r4;
    int rc = ora_meb_welzl(tp, count, 3, 12345u, c3, &d3, trans_support, n_trans_support, 4);
    if (rc == 0) rc = ora_meb_welzl(qp, count, 4, 54321u, c4, &r4, rot_support, n_rot_support, 5);
    if (rc == 0) {
        double h = sqrt(c4[0] * c4[0] + c4[1] * c4[1] + c4[2] * c4[2] + c4[3] * c4[3]);
        double qc[4] = { c4[0] / h, c4[1] / h, c4[2] / h, c4[3] / h };
        ora_rotation_from_quat(qc, out);
        out[9] = c3[0]; out[10] = c3[1]; out[11] = c3[2];
        double cosang = (1.0 + h * h - r4 * r4) / (2.0 * h);
        if (cosang > 1.0) cosang = 1.0;
        if (cosang < -1.0) cosang = -1.0;
        out[12] = 2.0 * acos(cosang);
        out[13] = d3;
    }
    free(tp); free(qp);
    return rc;
}
