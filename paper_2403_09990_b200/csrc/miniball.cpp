// Host side of Step III: exact smallest enclosing ball of a point cloud in
// R^d, d <= 4, after B. Gaertner, "Fast and robust smallest enclosing balls", ESA 1999 (the
// paper's ref. [23]): an incrementally orthogonalised support basis (each push costs O(d^2)),
// Welzl's move-to-front recursion over a short list of support candidates, and an outer
// pivoting loop that repeatedly adds the point farthest from the current centre.
//
// Written from the algorithm's description; independent of oracle/miniball_oracle.c (which
// solves the support ball by Gaussian elimination and runs plain Welzl over all points).
#include <algorithm>
#include <cmath>
#include <cstring>
#include <list>

#include "closure_internal.h"

namespace closure {
namespace {

constexpr int kD = 4;

// Ball through a growing set of affinely independent points q_0 .. q_{m-1}.
// Level m keeps the centre c[m-1] and squared radius r2[m-1] of the smallest ball with all pushed
// points on its boundary; v[k] is q_k - q_0 made orthogonal to v[1..k-1]; z[k] = 2 |v[k]|^2.
// Pushing p moves the centre along v[m] by f = e / z, e = |p - c|^2 - r2, which keeps the old
// points equidistant and brings p to the same distance: r2' = r2 + e f / 2.
class Basis {
public:
    explicit Basis(int d) : d_(d), m_(0) {}
    int size() const { return m_; }
    void reset() { m_ = 0; }
    const double *center() const { return c_[m_ - 1]; }
    double sq_radius() const { return m_ ? r2_[m_ - 1] : -1.0; }
    long long point(int k) const { return idx_[k]; }

    double excess(const double *p) const
    {
        if (m_ == 0) return 1.0;
        double s = 0.0;
        for (int a = 0; a < d_; ++a) s += (p[a] - c_[m_ - 1][a]) * (p[a] - c_[m_ - 1][a]);
        return s - r2_[m_ - 1];
    }

    bool push(const double *p, long long index)
    {
        if (m_ == 0) {
            std::memcpy(q0_, p, sizeof(double) * d_);
            std::memcpy(c_[0], p, sizeof(double) * d_);
            r2_[0] = 0.0;
        } else {
            double *v = v_[m_];
            for (int a = 0; a < d_; ++a) v[a] = p[a] - q0_[a];
            for (int k = 1; k < m_; ++k) {                      // Gram-Schmidt against earlier directions
                double dot = 0.0;
                for (int a = 0; a < d_; ++a) dot += v_[k][a] * v[a];
                const double coef = 2.0 * dot / z_[k];
                for (int a = 0; a < d_; ++a) v[a] -= coef * v_[k][a];
            }
            double nv = 0.0;
            for (int a = 0; a < d_; ++a) nv += v[a] * v[a];
            z_[m_] = 2.0 * nv;
            if (z_[m_] < 1e-28 * std::max(r2_[m_ - 1], 1e-300) || !(z_[m_] > 0.0))
                return false;                                   // (numerically) affinely dependent
            double e = -r2_[m_ - 1];
            for (int a = 0; a < d_; ++a) e += (p[a] - c_[m_ - 1][a]) * (p[a] - c_[m_ - 1][a]);
            const double f = e / z_[m_];
            for (int a = 0; a < d_; ++a) c_[m_][a] = c_[m_ - 1][a] + f * v[a];
            r2_[m_] = r2_[m_ - 1] + 0.5 * e * f;
        }
        idx_[m_] = index;
        ++m_;
        return true;
    }
    void pop() { --m_; }

private:
    int d_, m_;
    double q0_[kD];
    double v_[kD + 1][kD];
    double z_[kD + 1];
    double c_[kD + 1][kD];
    double r2_[kD + 1];
    long long idx_[kD + 1];
};

// Host cloud: the points as they are; the pivot is a plain scan.
class HostCloud : public PointSource {
public:
    HostCloud(const double *p, long long n, int d) : pts_(p), n_(n), d_(d) {}
    bool farthest(const double *center, long long *index, double *sq_dist) override
    {
        long long far = -1;
        double far_d2 = -1.0;
        for (long long i = 0; i < n_; ++i) {
            const double *p = pts_ + (size_t)i * d_;
            double s = 0.0;
            for (int a = 0; a < d_; ++a) s += (p[a] - center[a]) * (p[a] - center[a]);
            if (s > far_d2) { far_d2 = s; far = i; }
        }
        *index = far;
        *sq_dist = far_d2;
        return true;
    }
    const double *point(long long i) override { return pts_ + (size_t)i * d_; }

private:
    const double *pts_;
    long long n_;
    int d_;
};

struct Solver {
    PointSource *src;
    int d;
    Basis basis;
    std::list<long long> cand;          // support candidates, most recently violating first
    double center[kD];
    double r2;
    long long support[kD + 1];
    int n_support;

    Solver(PointSource *p, int dim) : src(p), d(dim), basis(dim), r2(-1.0), n_support(0) {}

    void snapshot()
    {
        std::memcpy(center, basis.center(), sizeof(double) * d);
        r2 = basis.sq_radius();
        n_support = basis.size();
        for (int k = 0; k < n_support; ++k) support[k] = basis.point(k);
    }

    double excess(long long i) const
    {
        const double *p = src->point(i);
        double s = 0.0;
        for (int a = 0; a < d; ++a) s += (p[a] - center[a]) * (p[a] - center[a]);
        return s - r2;
    }

    // Welzl's recursion restricted to the candidate list: smallest ball containing the first
    // `end` candidates with the current basis on its boundary.
    void move_to_front(std::list<long long>::iterator end)
    {
        snapshot();
        if (basis.size() == d + 1) return;
        for (auto it = cand.begin(); it != end;) {
            auto cur = it++;
            if (excess(*cur) > 1e-15 * std::max(r2, 0.0)) {
                if (basis.push(src->point(*cur), *cur)) {
                    move_to_front(cur);
                    basis.pop();
                    cand.splice(cand.begin(), cand, cur);
                }
            }
        }
    }
};

}  // namespace

bool miniball_source(PointSource *src, long long n, int d, Ball *out)
{
    if (n <= 0 || d <= 0 || d > kD || !src) return false;
    Solver S(src, d);
    const double *p0 = src->point(0);
    if (!p0) return false;
    std::memcpy(S.center, p0, sizeof(double) * d);
    S.r2 = -1.0;                      // no ball yet: the first pivot always makes progress
    S.n_support = 1;
    S.support[0] = 0;
    for (int iter = 0; iter < 10000; ++iter) {
        // pivot: the point farthest from the current centre (the only pass over the whole cloud)
        long long far = -1;
        double far_d2 = -1.0;
        if (!src->farthest(S.center, &far, &far_d2) || far < 0) return false;
        if (far_d2 - S.r2 <= 1e-14 * far_d2) break;           // everything inside: optimal
        const double old_r2 = S.r2;
        const double *pf = src->point(far);
        if (!pf) return false;
        S.basis.reset();
        S.basis.push(pf, far);
        S.move_to_front(S.cand.end());
        S.basis.reset();
        S.cand.remove(far);
        S.cand.push_front(far);
        if (!(S.r2 > old_r2)) break;                           // no progress (rounding floor)
    }
    std::memset(out->center, 0, sizeof(out->center));
    std::memcpy(out->center, S.center, sizeof(double) * d);
    out->sq_radius = S.r2 > 0.0 ? S.r2 : 0.0;
    out->n_support = S.n_support;
    for (int k = 0; k < S.n_support; ++k) out->support[k] = S.support[k];
    std::sort(out->support, out->support + out->n_support);
    return true;
}

bool miniball(const double *pts, long long n, int d, Ball *out)
{
    if (!pts || n <= 0 || d <= 0 || d > kD) return false;
    HostCloud cloud(pts, n, d);
    return miniball_source(&cloud, n, d, out);
}

// Unit quaternion (w, x, y, z) of a rotation matrix: take the largest of the four squared
// components 4w^2 = 1 + tr, 4x^2 = 1 + R00 - R11 - R22, ... and fill the rest from the
// symmetric / antisymmetric off-diagonal parts.
void rotation_to_quat(const double R[9], double q[4])
{
    const double sq[4] = { 1.0 + R[0] + R[4] + R[8], 1.0 + R[0] - R[4] - R[8], 1.0 - R[0] + R[4] - R[8],
                           1.0 - R[0] - R[4] + R[8] };
    int big = 0;
    for (int k = 1; k < 4; ++k)
        if (sq[k] > sq[big]) big = k;
    const double g = 0.5 * std::sqrt(sq[big]);
    const double h = 0.25 / g;
    switch (big) {
    case 0: q[0] = g; q[1] = (R[7] - R[5]) * h; q[2] = (R[2] - R[6]) * h; q[3] = (R[3] - R[1]) * h; break;
    case 1: q[1] = g; q[0] = (R[7] - R[5]) * h; q[2] = (R[1] + R[3]) * h; q[3] = (R[2] + R[6]) * h; break;
    case 2: q[2] = g; q[0] = (R[2] - R[6]) * h; q[1] = (R[1] + R[3]) * h; q[3] = (R[5] + R[7]) * h; break;
    default: q[3] = g; q[0] = (R[3] - R[1]) * h; q[1] = (R[2] + R[6]) * h; q[2] = (R[5] + R[7]) * h; break;
    }
    const double nq = std::sqrt(q[0] * q[0] + q[1] * q[1] + q[2] * q[2] + q[3] * q[3]);
    for (int k = 0; k < 4; ++k) q[k] /= nq;
}

void quat_to_rotation(const double q[4], double R[9])
{
    const double w = q[0], x = q[1], y = q[2], z = q[3];
    const double xx = x * x, yy = y * y, zz = z * z, xy = x * y, xz = x * z, yz = y * z, wx = w * x, wy = w * y,
                 wz = w * z;
    R[0] = 1.0 - 2.0 * (yy + zz); R[1] = 2.0 * (xy - wz);       R[2] = 2.0 * (xz + wy);
    R[3] = 2.0 * (xy + wz);       R[4] = 1.0 - 2.0 * (xx + zz); R[5] = 2.0 * (yz - wx);
    R[6] = 2.0 * (xz - wy);       R[7] = 2.0 * (yz + wx);       R[8] = 1.0 - 2.0 * (xx + yy);
}

// proj_SO(3)(M) for det M > 0: orthogonal polar factor by Newton's iteration
// X <- (X + X^-T) / 2 (quadratically convergent), started from M scaled to unit Frobenius norm.
bool project_so3(const double M[9], double R[9])
{
    double X[9], nrm = 0.0;
    for (int e = 0; e < 9; ++e) nrm += M[e] * M[e];
    nrm = std::sqrt(nrm);
    if (!(nrm > 0.0) || !std::isfinite(nrm)) return false;
    for (int e = 0; e < 9; ++e) X[e] = M[e] * (std::sqrt(3.0) / nrm);
    for (int it = 0; it < 100; ++it) {
        const double c00 = X[4] * X[8] - X[5] * X[7], c01 = X[5] * X[6] - X[3] * X[8], c02 = X[3] * X[7] - X[4] * X[6];
        const double det = X[0] * c00 + X[1] * c01 + X[2] * c02;
        if (!(det > 1e-12)) return false;                       // reflection or singular sum
        // X^-T = cofactor matrix / det
        const double C[9] = { c00, c01, c02,
                              X[2] * X[7] - X[1] * X[8], X[0] * X[8] - X[2] * X[6], X[1] * X[6] - X[0] * X[7],
                              X[1] * X[5] - X[2] * X[4], X[2] * X[3] - X[0] * X[5], X[0] * X[4] - X[1] * X[3] };
        double change = 0.0;
        for (int e = 0; e < 9; ++e) {
            const double nx = 0.5 * (X[e] + C[e] / det);
            change = std::max(change, std::fabs(nx - X[e]));
            X[e] = nx;
        }
        if (change < 1e-16) break;
    }
    std::memcpy(R, X, sizeof(X));
    return true;
}

// PCA normalisation of the centre velocity (R-23): S = sqrtm(C) / sqrt(lambda_max),
// C the covariance of the initial translations, by cyclic Jacobi rotations on the symmetric 3x3.
void pca_velocity_scale(const double *poses, int n0, double S[9])
{
    for (int e = 0; e < 9; ++e) S[e] = (e % 4 == 0) ? 1.0 : 0.0;
    if (n0 < 2) return;
    double mean[3] = { 0, 0, 0 }, C[3][3] = { { 0 } };
    for (int s = 0; s < n0; ++s)
        for (int r = 0; r < 3; ++r) mean[r] += poses[(size_t)s * 12 + 9 + r];
    for (int r = 0; r < 3; ++r) mean[r] /= (double)n0;
    for (int s = 0; s < n0; ++s)
        for (int r = 0; r < 3; ++r)
            for (int c = 0; c < 3; ++c)
                C[r][c] += (poses[(size_t)s * 12 + 9 + r] - mean[r]) * (poses[(size_t)s * 12 + 9 + c] - mean[c]);
    for (int r = 0; r < 3; ++r)
        for (int c = 0; c < 3; ++c) C[r][c] /= (double)n0;
    double U[3][3] = { { 1, 0, 0 }, { 0, 1, 0 }, { 0, 0, 1 } };
    for (int sweep = 0; sweep < 50; ++sweep) {
        const double off = std::fabs(C[0][1]) + std::fabs(C[0][2]) + std::fabs(C[1][2]);
        if (!(off > 1e-300) || off <= 1e-17 * (std::fabs(C[0][0]) + std::fabs(C[1][1]) + std::fabs(C[2][2]))) break;
        for (int p = 0; p < 2; ++p)
            for (int q = p + 1; q < 3; ++q) {
                if (C[p][q] == 0.0) continue;
                const double theta = (C[q][q] - C[p][p]) / (2.0 * C[p][q]);
                const double tt = (theta >= 0.0 ? 1.0 : -1.0) / (std::fabs(theta) + std::sqrt(theta * theta + 1.0));
                const double c = 1.0 / std::sqrt(tt * tt + 1.0), sn = tt * c;
                for (int k = 0; k < 3; ++k) {                      // C <- C G
                    const double ckp = C[k][p], ckq = C[k][q];
                    C[k][p] = c * ckp - sn * ckq; C[k][q] = sn * ckp + c * ckq;
                }
                for (int k = 0; k < 3; ++k) {                      // C <- G^T C
                    const double cpk = C[p][k], cqk = C[q][k];
                    C[p][k] = c * cpk - sn * cqk; C[q][k] = sn * cpk + c * cqk;
                }
                for (int k = 0; k < 3; ++k) {                      // U <- U G
                    const double ukp = U[k][p], ukq = U[k][q];
                    U[k][p] = c * ukp - sn * ukq; U[k][q] = sn * ukp + c * ukq;
                }
            }
    }
    double lam[3] = { std::max(C[0][0], 0.0), std::max(C[1][1], 0.0), std::max(C[2][2], 0.0) };
    const double lmax = std::max(lam[0], std::max(lam[1], lam[2]));
    if (!(lmax > 0.0)) return;
    for (int r = 0; r < 3; ++r)
        for (int c = 0; c < 3; ++c) {
            double v = 0.0;
            for (int k = 0; k < 3; ++k) v += U[r][k] * std::sqrt(lam[k] / lmax) * U[c][k];
            S[3 * r + c] = v;
        }
}

}  // namespace closure
