// Step I of CLOSURE, "initialize starting poses", for
// Ex.1, Ex.2 and Ex.3: independent trials, one per thread.
//
//   Ex.1  RANSAG trial: three distinct random constraints, a random 2D point in each, the
//                        perspective-3-point problem for the three rays; up to four poses, tried in ascending
//                        order of the first depth, the first one that satisfies (PURSE2D3D) is kept;
//   Ex.2  RANSAG trial: three distinct random correspondences, Arun's least-squares rigid
//                        fit [6], kept iff the pose satisfies (PURSE3D3D);
//   Ex.3  a random convex combination of the pose hypotheses, kept iff it satisfies (PURSEreg).
//
// Readings R-21 / R-22: random words of trial k = Philox4x32-10 with counter
// (k_lo32, c, 0, tag | k_hi32 << 8), tag 2 = triplet, tag 3 = weights; i1 = x0 mod N, i2 = x1 mod (N-1),
// i3 = x2 mod (N-2), skipping indices already taken; degenerate triangles (normal < 1e-8) rejected;
// w_i = u_i / sum u, u_i = (x_i + 1/2) 2^-32; R = proj_SO(3)(sum w_i R_i), t = sum w_i t_i.
//
// Arun's rotation is V diag(1, 1, det(V U^T)) U^T for H = sum a'_k b'_k^T = U S V^T.  Three points make
// H rank 2, with null directions n_a (normal of the source triangle) and n_b (target): instead of an SVD
// the kernel completes H^T to M = H^T + lambda n_b n_a^T = V diag(s1, s2, +-lambda) U^T, picks the sign of
// lambda that makes det M > 0 -- exactly the determinant guard -- and takes the orthogonal polar factor of
// M by Newton's iteration X <- (X + X^-T) / 2.  The same iteration gives proj_SO(3) for Ex.3.
//
// Ex.1, reading R-24: y_l = z_l + beta_l e_l, e_l uniform in the unit disc by rejection from the
// square (Philox counter (k_lo32, l, a, 4 | k_hi32 << 8), attempts a = 0..7, two candidates per call).  P3P in
// the classical distance form: unit bearings f_l, depths d_l with |d_i f_i - d_j f_j|^2 = |Z_i - Z_j|^2; with
// d_2 = u d_1, d_3 = v d_1 the law of cosines in the three faces gives
//     a13 (1 + u^2 - 2 c12 u) = a12 s(v),   a13 (u^2 + v^2 - 2 c23 u v) = a23 s(v),   s(v) = 1 + v^2 - 2 c13 v,
// whose difference is linear in u:  u q(v) = p(v),  p = (a23 - a12) s + a13 (1 - v^2),  q = 2 a13 (c12 - c23 v),
// and u = p/q in the first one times q^2 is the quartic  G(v) = a13 (q^2 + p^2 - 2 c12 p q) - a12 s q^2.
// Its positive real roots are isolated without complex arithmetic: the roots of G'' (a quadratic) cut (0, B)
// into intervals on which G' is monotone, bisection there gives the critical points of G, which cut (0, B)
// into intervals on which G is monotone, bisection there gives the roots (B = Cauchy's bound).  Every root
// with u > 0 is polished by three Newton steps on the three distance equations; the pose is the rigid fit of
// Z_l -> d_l f_l (the same polar completion as Ex.2; the triangles are congruent, the fit is exact).
#include <cuda_runtime.h>
#include <math_constants.h>
#include <stdint.h>

#include "closure_internal.h"
#include "walker_common.cuh"

namespace closure {
namespace {

constexpr int kStep1Block = 128;

__device__ __forceinline__ double det3(const double (&X)[9])
{
    return X[0] * (X[4] * X[8] - X[5] * X[7]) + X[1] * (X[5] * X[6] - X[3] * X[8]) + X[2] * (X[3] * X[7] - X[4] * X[6]);
}

// Orthogonal polar factor of M (det M > 0): the rotation nearest to M in the Frobenius norm.
__device__ __forceinline__ bool polar_rotation(const double (&M)[9], double (&R)[9])
{
    double X[9], nrm = 0.0;
#pragma unroll
    for (int e = 0; e < 9; ++e) nrm = fma(M[e], M[e], nrm);
    nrm = sqrt(nrm);
    if (!(nrm > 0.0) || !(nrm < CUDART_INF)) return false;
    const double sc = 1.7320508075688772 / nrm;
#pragma unroll
    for (int e = 0; e < 9; ++e) X[e] = M[e] * sc;
    for (int it = 0; it < 100; ++it) {
        const double c00 = X[4] * X[8] - X[5] * X[7], c01 = X[5] * X[6] - X[3] * X[8], c02 = X[3] * X[7] - X[4] * X[6];
        const double det = X[0] * c00 + X[1] * c01 + X[2] * c02;
        if (!(det > 1e-300)) return false;
        const double C[9] = { c00, c01, c02,
                              X[2] * X[7] - X[1] * X[8], X[0] * X[8] - X[2] * X[6], X[1] * X[6] - X[0] * X[7],
                              X[1] * X[5] - X[2] * X[4], X[2] * X[3] - X[0] * X[5], X[0] * X[4] - X[1] * X[3] };
        const double inv = 1.0 / det;
        double change = 0.0;
#pragma unroll
        for (int e = 0; e < 9; ++e) {
            const double nx = 0.5 * (X[e] + C[e] * inv);
            change = fmax(change, fabs(nx - X[e]));
            X[e] = nx;
        }
        if (change < 4e-16) break;
    }
#pragma unroll
    for (int e = 0; e < 9; ++e) R[e] = X[e];
    return true;
}

// Arun's least-squares rigid fit of three points, b_k ~ R a_k + t (header).  false: degenerate triangle.
__device__ __forceinline__ bool arun3(const double (&p)[3][3], const double (&w)[3][3], double (&R)[9], double (&t)[3])
{
    double ab[3], bb[3], a[3][3], b[3][3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        ab[c] = ((p[0][c] + p[1][c]) + p[2][c]) / 3.0;
        bb[c] = ((w[0][c] + w[1][c]) + w[2][c]) / 3.0;
        a[0][c] = p[0][c] - ab[c]; a[1][c] = p[1][c] - ab[c]; a[2][c] = p[2][c] - ab[c];
        b[0][c] = w[0][c] - bb[c]; b[1][c] = w[1][c] - bb[c]; b[2][c] = w[2][c] - bb[c];
    }
    double na[3] = { a[0][1] * a[1][2] - a[0][2] * a[1][1], a[0][2] * a[1][0] - a[0][0] * a[1][2],
                     a[0][0] * a[1][1] - a[0][1] * a[1][0] };
    double nb[3] = { b[0][1] * b[1][2] - b[0][2] * b[1][1], b[0][2] * b[1][0] - b[0][0] * b[1][2],
                     b[0][0] * b[1][1] - b[0][1] * b[1][0] };
    const double la = sqrt(na[0] * na[0] + na[1] * na[1] + na[2] * na[2]);
    const double lb = sqrt(nb[0] * nb[0] + nb[1] * nb[1] + nb[2] * nb[2]);
    if (la < 1e-8 || lb < 1e-8 || !(la == la) || !(lb == lb)) return false;
    // M = H^T + lambda n_b n_a^T,  H^T[r][c] = sum_k b'_k[r] a'_k[c]
    double M[9], fro = 0.0;
#pragma unroll
    for (int r = 0; r < 3; ++r)
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            M[3 * r + c] = b[0][r] * a[0][c] + b[1][r] * a[1][c] + b[2][r] * a[2][c];
            fro = fma(M[3 * r + c], M[3 * r + c], fro);
        }
    const double lam = sqrt(fro) * 0.7071067811865476 / (la * lb);
    double Mp[9], Mm[9];
#pragma unroll
    for (int r = 0; r < 3; ++r)
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const double o = lam * nb[r] * na[c];
            Mp[3 * r + c] = M[3 * r + c] + o;
            Mm[3 * r + c] = M[3 * r + c] - o;
        }
    const bool have = det3(Mp) > 0.0 ? polar_rotation(Mp, R) : polar_rotation(Mm, R);
    if (have) {
#pragma unroll
        for (int r = 0; r < 3; ++r) t[r] = bb[r] - (R[3 * r] * ab[0] + R[3 * r + 1] * ab[1] + R[3 * r + 2] * ab[2]);
    }
    return have;
}

// ---------------------------------------------------------------------------------- Ex.1: P3P (header)
__device__ __forceinline__ double poly_eval(const double *g, int deg, double v)
{
    double r = g[deg];
    for (int i = deg - 1; i >= 0; --i) r = fma(r, v, g[i]);
    return r;
}

// The sign change of g in [lo, hi] (g(lo) = flo and g(hi) have opposite signs), to adjacent doubles.
__device__ __forceinline__ double bisect(const double *g, int deg, double lo, double hi, double flo)
{
    for (int it = 0; it < 1100; ++it) {
        const double mid = 0.5 * (lo + hi);
        if (!(mid > lo && mid < hi)) break;
        const double fm = poly_eval(g, deg, mid);
        if (fm == 0.0) return mid;
        if ((fm < 0.0) == (flo < 0.0)) lo = mid; else hi = mid;
    }
    return 0.5 * (lo + hi);
}

// Simple real roots of g in (lo, hi), ascending; br[0..nbr) are the roots of g' in (lo, hi), ascending,
// so that g is monotone between consecutive breakpoints.
__device__ __forceinline__ int roots_between(const double *g, int deg, const double *br, int nbr, double lo, double hi,
                                             double *out)
{
    int m = 0;
    double a = lo, fa = poly_eval(g, deg, a);
    for (int i = 0; i <= nbr; ++i) {
        const double b = i < nbr ? br[i] : hi;
        const double fb = poly_eval(g, deg, b);
        if (fa != 0.0 && fb != 0.0 && ((fa < 0.0) != (fb < 0.0))) out[m++] = bisect(g, deg, a, b, fa);
        a = b;
        fa = fb;
    }
    return m;
}

// Depth triples (d_1, d_2, d_3) of the P3P problem, sorted by d_1 -> count (<= 4).
__device__ __noinline__ int p3p_depths(const double (&f)[3][3], const double (&X)[3][3], double (&dsol)[4][3])
{
    const double c12 = f[0][0] * f[1][0] + f[0][1] * f[1][1] + f[0][2] * f[1][2];
    const double c13 = f[0][0] * f[2][0] + f[0][1] * f[2][1] + f[0][2] * f[2][2];
    const double c23 = f[1][0] * f[2][0] + f[1][1] * f[2][1] + f[1][2] * f[2][2];
    double a12 = 0.0, a13 = 0.0, a23 = 0.0;
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const double e12 = X[0][c] - X[1][c], e13 = X[0][c] - X[2][c], e23 = X[1][c] - X[2][c];
        a12 += e12 * e12; a13 += e13 * e13; a23 += e23 * e23;
    }
    const double s[3] = { 1.0, -2.0 * c13, 1.0 };
    const double w = a23 - a12;
    const double p[3] = { w + a13, w * s[1], w - a13 };
    const double q[2] = { 2.0 * a13 * c12, -2.0 * a13 * c23 };
    const double q2[3] = { q[0] * q[0], 2.0 * q[0] * q[1], q[1] * q[1] };
    const double p2[5] = { p[0] * p[0], 2.0 * p[0] * p[1], 2.0 * p[0] * p[2] + p[1] * p[1], 2.0 * p[1] * p[2], p[2] * p[2] };
    const double pq[4] = { p[0] * q[0], p[0] * q[1] + p[1] * q[0], p[1] * q[1] + p[2] * q[0], p[2] * q[1] };
    const double sq2[5] = { s[0] * q2[0], s[0] * q2[1] + s[1] * q2[0], s[0] * q2[2] + s[1] * q2[1] + s[2] * q2[0],
                            s[1] * q2[2] + s[2] * q2[1], s[2] * q2[2] };
    double G[5];
#pragma unroll
    for (int i = 0; i < 5; ++i) {
        const double qq = i < 3 ? q2[i] : 0.0, pp = i < 4 ? pq[i] : 0.0;
        G[i] = a13 * (qq + p2[i] - 2.0 * c12 * pp) - a12 * sq2[i];
    }
    double gmax = 0.0;
#pragma unroll
    for (int i = 0; i < 5; ++i) gmax = fmax(gmax, fabs(G[i]));
    if (!(gmax > 0.0) || !(gmax < CUDART_INF) || !(fabs(G[4]) >= 1e-9 * gmax)) return 0;
    const double B = 1.0 + gmax / fabs(G[4]);                           // Cauchy: every root has |v| < B
    const double G1[4] = { G[1], 2.0 * G[2], 3.0 * G[3], 4.0 * G[4] };
    const double G2[3] = { G1[1], 2.0 * G1[2], 3.0 * G1[3] };
    // roots of the quadratic G'' in (0, B)
    double r2[2];
    int n2 = 0;
    {
        const double disc = G2[1] * G2[1] - 4.0 * G2[2] * G2[0];
        if (disc > 0.0) {
            const double sd = sqrt(disc);
            const double z = -0.5 * (G2[1] + (G2[1] < 0.0 ? -sd : sd));  // no cancellation
            double x0 = z / G2[2], x1 = (z != 0.0) ? G2[0] / z : x0;
            if (x0 > x1) { const double tmp = x0; x0 = x1; x1 = tmp; }
            if (x0 > 0.0 && x0 < B) r2[n2++] = x0;
            if (x1 > 0.0 && x1 < B && x1 > x0) r2[n2++] = x1;
        }
    }
    double r1[3], r0[4];
    const int n1 = roots_between(G1, 3, r2, n2, 0.0, B, r1);
    const int n0 = roots_between(G, 4, r1, n1, 0.0, B, r0);
    int m = 0;
    for (int i = 0; i < n0; ++i) {
        const double v = r0[i];
        const double qv = fma(q[1], v, q[0]);
        if (fabs(qv) < 1e-9 * (fabs(q[0]) + fabs(q[1] * v))) continue;
        const double u = poly_eval(p, 2, v) / qv;
        if (!(u > 0.0)) continue;
        const double d1 = sqrt(a13 / (1.0 + v * v - 2.0 * c13 * v));
        double d[3] = { d1, u * d1, v * d1 };
        for (int it = 0; it < 3; ++it) {                                // Newton on the three distance equations
            const double F0 = d[0] * d[0] + d[1] * d[1] - 2.0 * c12 * d[0] * d[1] - a12;
            const double F1 = d[0] * d[0] + d[2] * d[2] - 2.0 * c13 * d[0] * d[2] - a13;
            const double F2 = d[1] * d[1] + d[2] * d[2] - 2.0 * c23 * d[1] * d[2] - a23;
            // J = 2 [[A, Bq, 0], [C, 0, Dq], [0, E, Fq]]
            const double A = d[0] - c12 * d[1], Bq = d[1] - c12 * d[0], C = d[0] - c13 * d[2], Dq = d[2] - c13 * d[0];
            const double E = d[1] - c23 * d[2], Fq = d[2] - c23 * d[1];
            const double det = -A * Dq * E - Bq * C * Fq;             // det of J / 2
            if (det == 0.0) break;
            const double h0 = 0.5 * F0, h1 = 0.5 * F1, h2 = 0.5 * F2;   // (J/2) x = F/2
            const double x0 = (h0 * (-Dq * E) - Bq * (h1 * Fq - Dq * h2)) / det;
            const double x1 = (A * (h1 * Fq - Dq * h2) - h0 * (C * Fq)) / det;
            const double x2 = (A * (-E * h1) - Bq * (C * h2) + h0 * (C * E)) / det;
            d[0] -= x0; d[1] -= x1; d[2] -= x2;
        }
        if (!(d[0] > 0.0) || !(d[1] > 0.0) || !(d[2] > 0.0)) continue;
        int at = m++;
        while (at > 0 && dsol[at - 1][0] > d[0]) {                      // insertion by d_1
            dsol[at][0] = dsol[at - 1][0]; dsol[at][1] = dsol[at - 1][1]; dsol[at][2] = dsol[at - 1][2];
            --at;
        }
        dsol[at][0] = d[0]; dsol[at][1] = d[1]; dsol[at][2] = d[2];
    }
    return m;
}

template <int RES>
__global__ void __launch_bounds__(kStep1Block) step1_kernel(const InstanceDesc *__restrict__ D, long long trial_begin,
                                                             long long num_trials, unsigned long long seed,
                                                             double *__restrict__ out_poses,
                                                             unsigned char *__restrict__ out_ok)
{
    using RS = Res<RES>;
    constexpr int ROW = RS::ROW;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    uint64_t *bar = reinterpret_cast<uint64_t *>(smem_raw);
    const double *rows = reinterpret_cast<const double *>(smem_raw + 16);
    const int n = D->n;
    stage_rows(smem_raw + 16, bar, D->rows, D->rows_bytes);
    const long long q = (long long)blockIdx.x * kStep1Block + threadIdx.x;
    if (q >= num_trials) return;
    const unsigned long long k = (unsigned long long)(trial_begin + q);
    const uint32_t k_lo = (uint32_t)k, k_hi8 = (uint32_t)(k >> 32) << 8;
    const uint32_t s0 = (uint32_t)seed, s1 = (uint32_t)(seed >> 32);
    const int *__restrict__ perm = D->perm;            // original constraint index -> row of the sorted table
    double K[4];
#pragma unroll
    for (int e = 0; e < 4; ++e) K[e] = D->K[e];

    double R[9], t[3];
    bool have = false;
    bool ok = false;
    if (RES == CLOSURE_REG_3D3D || RES == CLOSURE_REG_3D3D_ELL || RES == CLOSURE_REPROJ_2D3D || RES == CLOSURE_REPROJ_2D3D_ELL) {
        uint32_t x[4];
        philox4x32_10(k_lo, 0u, 0u, 2u | k_hi8, s0, s1, x);
        int i1 = (int)(x[0] % (uint32_t)n);
        int i2 = (int)(x[1] % (uint32_t)(n - 1));
        if (i2 >= i1) ++i2;
        int i3 = (int)(x[2] % (uint32_t)(n - 2));
        const int lo = min(i1, i2), hi = max(i1, i2);
        if (i3 >= lo) ++i3;
        if (i3 >= hi) ++i3;
        const double *r1 = rows + perm[i1] * ROW, *r2 = rows + perm[i2] * ROW, *r3 = rows + perm[i3] * ROW;
        if (RES == CLOSURE_REG_3D3D || RES == CLOSURE_REG_3D3D_ELL) {
            double a[3][3], b[3][3];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                a[0][c] = r1[c]; a[1][c] = r2[c]; a[2][c] = r3[c];
                b[0][c] = r1[3 + c]; b[1][c] = r2[3 + c]; b[2][c] = r3[3 + c];
            }
            have = arun3(a, b, R, t);
        } else {
            // rows are [z(2) Z(3) beta]: a 2D point in each of the three constraints, its unit bearing
            const double *rr[3] = { r1, r2, r3 };
            double f[3][3], X[3][3];
#pragma unroll
            for (int l = 0; l < 3; ++l) {
                double e0 = 0.0, e1 = 0.0;
                bool found = false;
                for (int a = 0; a < 8 && !found; ++a) {
                    philox4x32_10(k_lo, (uint32_t)l, (uint32_t)a, 4u | k_hi8, s0, s1, x);
#pragma unroll
                    for (int h = 0; h < 4; h += 2) {
                        const double c0 = pm1(x[h]), c1 = pm1(x[h + 1]);
                        if (!found && __dadd_rn(__dmul_rn(c0, c0), __dmul_rn(c1, c1)) <= 1.0) {
                            e0 = c0; e1 = c1; found = true;
                        }
                    }
                }
                if (RES == CLOSURE_REPROJ_2D3D_ELL) {
                    // uniform in the ellipse: e <- L^-T e with Lambda = L L^T (rows hold L00 L01 L11 of Lambda at 7..9)
                    const double l00 = sqrt(rr[l][7]), l10 = rr[l][8] / l00;
                    const double l11 = sqrt(rr[l][9] - l10 * l10);
                    e1 = e1 / l11;
                    e0 = (e0 - l10 * e1) / l00;
                }
                const double y0 = __dadd_rn(rr[l][0], __dmul_rn(rr[l][5], e0));
                const double y1 = __dadd_rn(rr[l][1], __dmul_rn(rr[l][5], e1));
                const double m0 = (y0 - K[2]) / K[0], m1 = (y1 - K[3]) / K[1];
                const double nrm = sqrt(__dadd_rn(__dadd_rn(__dmul_rn(m0, m0), __dmul_rn(m1, m1)), 1.0));
                f[l][0] = m0 / nrm; f[l][1] = m1 / nrm; f[l][2] = 1.0 / nrm;
                X[l][0] = rr[l][2]; X[l][1] = rr[l][3]; X[l][2] = rr[l][4];
            }
            // degenerate source triangle (normal of the centred triangle shorter than 1e-8): rejected
            double e1v[3], e2v[3];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const double mc = ((X[0][c] + X[1][c]) + X[2][c]) / 3.0;
                e1v[c] = X[0][c] - mc; e2v[c] = X[1][c] - mc;
            }
            const double nx = e1v[1] * e2v[2] - e1v[2] * e2v[1], ny = e1v[2] * e2v[0] - e1v[0] * e2v[2],
                         nz = e1v[0] * e2v[1] - e1v[1] * e2v[0];
            if (!(sqrt(nx * nx + ny * ny + nz * nz) < 1e-8)) {
                double dsol[4][3];
                const int m = p3p_depths(f, X, dsol);
                for (int c = 0; c < m && !ok; ++c) {                 // ascending d_1: the first feasible pose
                    double wv[3][3];
#pragma unroll
                    for (int l = 0; l < 3; ++l)
#pragma unroll
                        for (int e = 0; e < 3; ++e) wv[l][e] = dsol[c][l] * f[l][e];
                    if (arun3(X, wv, R, t)) {
                        unsigned long long pairs = 0;
                        ok = in_purse_direct<RES>(R, t, rows, n, K, pairs);
                    }
                }
                have = false;                                        // decided above
            }
        }
    } else {
        // sum of the uniforms first (left to right, original hypothesis order), then the weighted sums
        double ssum = 0.0;
        for (int c = 0; 4 * c < n; ++c) {
            uint32_t x[4];
            philox4x32_10(k_lo, (uint32_t)c, 0u, 3u | k_hi8, s0, s1, x);
#pragma unroll
            for (int l = 0; l < 4; ++l)
                if (4 * c + l < n) ssum += ((double)x[l] + 0.5) * 2.3283064365386963e-10;
        }
        double M[9] = { 0, 0, 0, 0, 0, 0, 0, 0, 0 };
        t[0] = t[1] = t[2] = 0.0;
        for (int c = 0; 4 * c < n; ++c) {
            uint32_t x[4];
            philox4x32_10(k_lo, (uint32_t)c, 0u, 3u | k_hi8, s0, s1, x);
#pragma unroll
            for (int l = 0; l < 4; ++l) {
                const int i = 4 * c + l;
                if (i < n) {
                    const double wgt = (((double)x[l] + 0.5) * 2.3283064365386963e-10) / ssum;
                    const double *row = rows + perm[i] * ROW;
#pragma unroll
                    for (int e = 0; e < 9; ++e) M[e] += wgt * row[e];
#pragma unroll
                    for (int e = 0; e < 3; ++e) t[e] += wgt * row[9 + e];
                }
            }
        }
        have = det3(M) > 0.0 && polar_rotation(M, R);
    }

    if (have) {
        unsigned long long pairs = 0;
        ok = in_purse_direct<RES>(R, t, rows, n, K, pairs);
    }
    double2 *dst = reinterpret_cast<double2 *>(out_poses + 12 * q);
    if (ok) {
        dst[0] = make_double2(R[0], R[1]); dst[1] = make_double2(R[2], R[3]); dst[2] = make_double2(R[4], R[5]);
        dst[3] = make_double2(R[6], R[7]); dst[4] = make_double2(R[8], t[0]); dst[5] = make_double2(t[1], t[2]);
    } else {
#pragma unroll
        for (int e = 0; e < 6; ++e) dst[e] = make_double2(0.0, 0.0);
    }
    out_ok[q] = ok ? 1 : 0;
}

template <int RES>
cudaError_t launch_t(const InstanceDesc *d_desc, int rows_bytes, long long trial_begin, long long num_trials,
                     unsigned long long seed, double *out_poses, unsigned char *out_ok, cudaStream_t stream)
{
    const size_t smem = 16 + (size_t)((rows_bytes + 15) & ~15);
    if (smem > 200 * 1024) return cudaErrorInvalidConfiguration;
    cudaError_t e = cudaFuncSetAttribute(step1_kernel<RES>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const long long blocks = (num_trials + kStep1Block - 1) / kStep1Block;
    if (blocks > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    step1_kernel<RES><<<(unsigned)blocks, kStep1Block, smem, stream>>>(d_desc, trial_begin, num_trials, seed, out_poses, out_ok);
    return cudaGetLastError();
}

}  // namespace

cudaError_t launch_step1(int residual_type, const InstanceDesc *d_desc, int rows_bytes, long long trial_begin,
                         long long num_trials, unsigned long long seed, double *out_poses, unsigned char *out_ok,
                         cudaStream_t stream)
{
    if (num_trials <= 0) return cudaSuccess;
    switch (residual_type) {
    case CLOSURE_REPROJ_2D3D: return launch_t<CLOSURE_REPROJ_2D3D>(d_desc, rows_bytes, trial_begin, num_trials, seed, out_poses, out_ok, stream);
    case CLOSURE_REPROJ_2D3D_ELL: return launch_t<CLOSURE_REPROJ_2D3D_ELL>(d_desc, rows_bytes, trial_begin, num_trials, seed, out_poses, out_ok, stream);
    case CLOSURE_REG_3D3D_ELL: return launch_t<CLOSURE_REG_3D3D_ELL>(d_desc, rows_bytes, trial_begin, num_trials, seed, out_poses, out_ok, stream);
    case CLOSURE_REG_3D3D: return launch_t<CLOSURE_REG_3D3D>(d_desc, rows_bytes, trial_begin, num_trials, seed, out_poses, out_ok, stream);
    case CLOSURE_POSE_REG: return launch_t<CLOSURE_POSE_REG>(d_desc, rows_bytes, trial_begin, num_trials, seed, out_poses, out_ok, stream);
    case CLOSURE_POSE_REG_SPLIT: return launch_t<CLOSURE_POSE_REG_SPLIT>(d_desc, rows_bytes, trial_begin, num_trials, seed, out_poses, out_ok, stream);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace closure
