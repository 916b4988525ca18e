// Device helpers shared by the walker kernels (Philox, small 3x3 math, residual traits, top-k
// list, TMA staging, walker initialisation).  Included inside `namespace closure { namespace {`.
#pragma once
#include <cuda_runtime.h>
#include <math_constants.h>
#include <stdint.h>

#include "closure_internal.h"

namespace closure {
namespace {

constexpr int kJT = 10;   // perturbations evaluated together from registers (ILP for the FP64 pipe)

// ---------------------------------------------------------------------------------- RNG
// Philox4x32-10 (Salmon et al., SC'11).  Counter (w_lo, s, j, tag | w_hi << 8), key = seed (R-5).
__device__ __forceinline__ void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                              uint32_t k0, uint32_t k1, uint32_t (&o)[4])
{
#pragma unroll
    for (int r = 0; r < 10; ++r) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        c0 = hi1 ^ c1 ^ k0;
        c1 = lo1;
        c2 = hi0 ^ c3 ^ k1;
        c3 = lo0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    o[0] = c0; o[1] = c1; o[2] = c2; o[3] = c3;
}

// uniform in (-1,1): (2x+1) 2^-32 - 1 = x 2^-31 + (2^-32 - 1); exact (33 significant bits).
__device__ __forceinline__ double pm1(uint32_t x)
{
    return fma((double)x, 4.656612873077392578125e-10, 2.3283064365386962890625e-10 - 1.0);
}

struct Rng {
    uint32_t w_lo, w_hi8, k0, k1;
    __device__ __forceinline__ void xi3(uint32_t s, uint32_t j, uint32_t tag, double &x, double &y, double &z) const
    {
        uint32_t o[4];
        philox4x32_10(w_lo, s, j, tag | w_hi8, k0, k1, o);
        x = pm1(o[0]); y = pm1(o[1]); z = pm1(o[2]);
    }
};

// max / min by compare-select: fmax()/fmin() on doubles compile to DSETP + FSEL + SEL + LOP3 + moves
// (IEEE NaN handling); no NaN reaches these call sites (inf - inf never occurs: see margin paths).
__device__ __forceinline__ double dmax(double a, double b) { return a > b ? a : b; }
__device__ __forceinline__ double dmin(double a, double b) { return a < b ? a : b; }

// ---------------------------------------------------------------------------------- small math
// Every multiply-add below is written as an explicit fma(): several kernels share these helpers and must
// round identically (the tests compare them bit for bit), which implicit contraction does not guarantee.
__device__ __forceinline__ void mat3_mul(const double (&A)[9], const double (&B)[9], double (&C)[9])
{
#pragma unroll
    for (int r = 0; r < 3; ++r)
#pragma unroll
        for (int c = 0; c < 3; ++c)
            C[3 * r + c] = fma(A[3 * r + 2], B[6 + c], fma(A[3 * r + 1], B[3 + c], A[3 * r] * B[c]));
}

// Rodrigues coefficients of Exp(phi): Exp = I + A [phi]x + B [phi]x^2 (series below 1e-4).
__device__ __forceinline__ void exp_coeffs(double th2, double &A, double &B)
{
    const double th = sqrt(th2);
    if (th < 1e-4) {
        A = 1.0 - th2 / 6.0;
        B = 0.5 - th2 / 24.0;
    } else {
        double s, c, sh, ch;
        sincos(th, &s, &c);
        sincos(0.5 * th, &sh, &ch);
        A = s / th;
        B = 2.0 * sh * sh / th2;
    }
}

// E = Exp(phi)
__device__ __forceinline__ void exp_so3(double p0, double p1, double p2, double (&E)[9])
{
    double A, B;
    exp_coeffs(fma(p2, p2, fma(p1, p1, p0 * p0)), A, B);
    const double K[9] = { 0.0, -p2, p1, p2, 0.0, -p0, -p1, p0, 0.0 };
    double K2[9];
    mat3_mul(K, K, K2);
#pragma unroll
    for (int e = 0; e < 9; ++e) E[e] = fma(B, K2[e], fma(A, K[e], (e % 4 == 0) ? 1.0 : 0.0));
}

// Rm = R + a (w x R) + b (w x (w x R)), cross products taken column by column:
// Exp(dT w) R with a = A dT, b = B dT^2.
__device__ __forceinline__ void rotate_left(const double (&R)[9], double w0, double w1, double w2,
                                            double a, double b, double (&Rm)[9])
{
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const double x = R[c], y = R[3 + c], z = R[6 + c];
        const double p0 = fma(w1, z, -(w2 * y)), p1 = fma(w2, x, -(w0 * z)), p2 = fma(w0, y, -(w1 * x));       // w x col
        const double q0 = fma(w1, p2, -(w2 * p1)), q1 = fma(w2, p0, -(w0 * p2)), q2 = fma(w0, p1, -(w1 * p0)); // w x (w x col)
        Rm[c] = fma(b, q0, fma(a, p0, x));
        Rm[3 + c] = fma(b, q1, fma(a, p1, y));
        Rm[6 + c] = fma(b, q2, fma(a, p2, z));
    }
}

// ---------------------------------------------------------------------------------- residuals
template <int RES> struct Res;
template <> struct Res<CLOSURE_REG_3D3D> { static constexpr int ROW = 8, BETA = 6; static constexpr bool AFFINE = true; };
template <> struct Res<CLOSURE_REPROJ_2D3D> { static constexpr int ROW = 8, BETA = 5; static constexpr bool AFFINE = false; };
template <> struct Res<CLOSURE_POSE_REG> { static constexpr int ROW = 16, BETA = 12; static constexpr bool AFFINE = true; };
template <> struct Res<CLOSURE_POSE_REG_SPLIT> { static constexpr int ROW = 16, BETA = 14; static constexpr bool AFFINE = true; };
// ellipse / ellipsoid norm (eq. (6)): rows [a b beta beta^2 L00 L01 L02 L11 L12 L22] and [z Z beta beta^2 L00 L01 L11]
template <> struct Res<CLOSURE_REG_3D3D_ELL> { static constexpr int ROW = 16, BETA = 6; static constexpr bool AFFINE = false; };
template <> struct Res<CLOSURE_REPROJ_2D3D_ELL> { static constexpr int ROW = 10, BETA = 5; static constexpr bool AFFINE = false; };

__device__ __forceinline__ double frob_sq(const double (&R)[9], const double *Ri)
{
    double s = 0.0;
#pragma unroll
    for (int e = 0; e < 9; ++e) {
        const double g = R[e] - Ri[e];
        s = fma(g, g, s);
    }
    return s;
}

// ROT-mode set-up of row i at rotation R and base translation t: the squared residual of the
// translation-dependent constraint at translation t + d is  c - 2 u.d + |d|^2.
template <int RES>
__device__ __forceinline__ void affine_setup(const double (&R)[9], const double (&t)[3], const double *row,
                                             double &u0, double &u1, double &u2, double &c)
{
    if (RES == CLOSURE_REG_3D3D) {
        const double a0 = row[0], a1 = row[1], a2 = row[2];
        u0 = row[3] - (fma(R[0], a0, fma(R[1], a1, R[2] * a2)) + t[0]);
        u1 = row[4] - (fma(R[3], a0, fma(R[4], a1, R[5] * a2)) + t[1]);
        u2 = row[5] - (fma(R[6], a0, fma(R[7], a1, R[8] * a2)) + t[2]);
        c = fma(u2, u2, fma(u1, u1, u0 * u0));
    } else {
        u0 = row[9] - t[0];
        u1 = row[10] - t[1];
        u2 = row[11] - t[2];
        c = fma(u2, u2, fma(u1, u1, u0 * u0));
        if (RES == CLOSURE_POSE_REG) c += frob_sq(R, row);
    }
}

// Reprojection residual (eq. (2)) with the rotation part shared by all perturbations of a
// pose: P = R Z_i once per constraint, then the squared residual at the camera-frame point P + s,
// s = t* + d_j; +inf behind the camera (R-10).  Used by the plain kernel and by the fp64 paths of the
// cooperative kernel, so both take bit-identical decisions.
__device__ __forceinline__ void reproj_point(const double (&R)[9], const double *row, double &P0, double &P1, double &P2)
{
    const double Z0 = row[2], Z1 = row[3], Z2 = row[4];
    P0 = fma(R[0], Z0, fma(R[1], Z1, R[2] * Z2));
    P1 = fma(R[3], Z0, fma(R[4], Z1, R[5] * Z2));
    P2 = fma(R[6], Z0, fma(R[7], Z1, R[8] * Z2));
}
__device__ __forceinline__ double reproj_sq(double P0, double P1, double P2, double s0, double s1, double s2,
                                            const double *row, const double (&K)[4])
{
    const double p0 = P0 + s0, p1 = P1 + s1, p2 = P2 + s2;
    if (!(p2 > 0.0)) return CUDART_INF;
    const double g0 = row[0] - fma(K[0], p0 / p2, K[2]);
    const double g1 = row[1] - fma(K[1], p1 / p2, K[3]);
    return fma(g1, g1, g0 * g0);
}

// Direct evaluation of the squared residual at pose (R, t) (generic path).
// part: POSE_REG_SPLIT only, 0 = rotation bound, 1 = translation bound.
template <int RES>
__device__ __forceinline__ double direct_sq(const double (&R)[9], const double (&t)[3], const double *row,
                                            const double (&K)[4], int part)
{
    if (RES == CLOSURE_REG_3D3D) {
        const double a0 = row[0], a1 = row[1], a2 = row[2];
        const double g0 = row[3] - (fma(R[0], a0, fma(R[1], a1, R[2] * a2)) + t[0]);
        const double g1 = row[4] - (fma(R[3], a0, fma(R[4], a1, R[5] * a2)) + t[1]);
        const double g2 = row[5] - (fma(R[6], a0, fma(R[7], a1, R[8] * a2)) + t[2]);
        return fma(g2, g2, fma(g1, g1, g0 * g0));
    } else if (RES == CLOSURE_REPROJ_2D3D) {
        double P0, P1, P2;
        reproj_point(R, row, P0, P1, P2);
        return reproj_sq(P0, P1, P2, t[0], t[1], t[2], row, K);      // cheirality (R-10) inside
    } else if (RES == CLOSURE_REG_3D3D_ELL) {                        // g^T Lambda g, g = b - (R a + t)
        const double a0 = row[0], a1 = row[1], a2 = row[2];
        const double g0 = row[3] - (fma(R[0], a0, fma(R[1], a1, R[2] * a2)) + t[0]);
        const double g1 = row[4] - (fma(R[3], a0, fma(R[4], a1, R[5] * a2)) + t[1]);
        const double g2 = row[5] - (fma(R[6], a0, fma(R[7], a1, R[8] * a2)) + t[2]);
        const double h0 = fma(row[8], g0, fma(row[9], g1, row[10] * g2));
        const double h1 = fma(row[9], g0, fma(row[11], g1, row[12] * g2));
        const double h2 = fma(row[10], g0, fma(row[12], g1, row[13] * g2));
        return fma(g2, h2, fma(g1, h1, g0 * h0));
    } else if (RES == CLOSURE_REPROJ_2D3D_ELL) {                     // g^T Lambda g, g = z - Pi(K (R Z + t))
        const double Z0 = row[2], Z1 = row[3], Z2 = row[4];
        const double p0 = fma(R[0], Z0, fma(R[1], Z1, R[2] * Z2)) + t[0];
        const double p1 = fma(R[3], Z0, fma(R[4], Z1, R[5] * Z2)) + t[1];
        const double p2 = fma(R[6], Z0, fma(R[7], Z1, R[8] * Z2)) + t[2];
        if (!(p2 > 0.0)) return CUDART_INF;                          // cheirality (R-10)
        const double g0 = row[0] - fma(K[0], p0 / p2, K[2]);
        const double g1 = row[1] - fma(K[1], p1 / p2, K[3]);
        const double h0 = fma(row[7], g0, row[8] * g1), h1 = fma(row[8], g0, row[9] * g1);
        return fma(g1, h1, g0 * h0);
    } else {
        double s = 0.0;
        if (RES == CLOSURE_POSE_REG || part == 0) s = frob_sq(R, row);
        if (RES == CLOSURE_POSE_REG || part == 1) {
#pragma unroll
            for (int r = 0; r < 3; ++r) {
                const double g = t[r] - row[9 + r];
                s = fma(g, g, s);
            }
        }
        return s;
    }
}

// eq. (14): min over constraints of beta - ||g|| at one pose (generic path).
template <int RES>
__device__ __forceinline__ double margin_direct(const double (&R)[9], const double (&t)[3], const double *rows,
                                                int n, const double (&K)[4])
{
    double d = CUDART_INF;
    for (int i = 0; i < n; ++i) {
        const double *row = rows + i * Res<RES>::ROW;
        if (RES == CLOSURE_POSE_REG_SPLIT) {
            d = fmin(d, row[12] - sqrt(direct_sq<RES>(R, t, row, K, 0)));
            d = fmin(d, row[14] - sqrt(direct_sq<RES>(R, t, row, K, 1)));
        } else {
            d = fmin(d, row[Res<RES>::BETA] - sqrt(direct_sq<RES>(R, t, row, K, 0)));
        }
    }
    return d;
}

template <int RES>
__device__ __forceinline__ bool in_purse_direct(const double (&R)[9], const double (&t)[3], const double *rows,
                                                int n, const double (&K)[4], unsigned long long &pairs)
{
    for (int i = 0; i < n; ++i) {
        const double *row = rows + i * Res<RES>::ROW;
        ++pairs;
        if (RES == CLOSURE_POSE_REG_SPLIT) {
            if (!(direct_sq<RES>(R, t, row, K, 0) <= row[13])) return false;
            if (!(direct_sq<RES>(R, t, row, K, 1) <= row[15])) return false;
        } else {
            if (!(direct_sq<RES>(R, t, row, K, 0) <= row[Res<RES>::BETA + 1])) return false;
        }
    }
    return true;
}

// ---------------------------------------------------------------------------------- top-k list
// Sorted by (d descending, j ascending) (R-8).  Capacity KCAP is static so the list stays in
// registers; only the first n_p_star entries are used by the ladder.
template <int KCAP>
struct TopK {
    double d[KCAP];
    int j[KCAP];
    __device__ __forceinline__ void clear()
    {
#pragma unroll
        for (int k = 0; k < KCAP; ++k) { d[k] = -CUDART_INF; j[k] = 0x7fffffff; }
    }
    static __device__ __forceinline__ bool before(double da, int ja, double db, int jb)
    {
        return da > db || (da == db && ja < jb);
    }
    __device__ __forceinline__ void insert(double dn, int jn)
    {
        if (!before(dn, jn, d[KCAP - 1], j[KCAP - 1])) return;
        bool placed = false;
#pragma unroll
        for (int k = KCAP - 1; k >= 1; --k) {
            if (!placed) {
                if (before(dn, jn, d[k - 1], j[k - 1])) {
                    d[k] = d[k - 1]; j[k] = j[k - 1];
                } else {
                    d[k] = dn; j[k] = jn; placed = true;
                }
            }
        }
        if (!placed) { d[0] = dn; j[0] = jn; }
    }
};

// ---------------------------------------------------------------------------------- TMA staging
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

// One elected thread issues a 1-D bulk copy global -> shared, completion on an mbarrier.
__device__ __forceinline__ void stage_rows(unsigned char *smem_dst, uint64_t *bar, const double *src, int bytes)
{
    if (threadIdx.x == 0) {
        const uint32_t b = smem_u32(bar);
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(b));
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(b), "r"(bytes) : "memory");
        asm volatile(
            "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                smem_u32(smem_dst)),
            "l"(src), "r"(bytes), "r"(b)
            : "memory");
    }
    __syncthreads();   // barrier initialised before anyone polls it
    const uint32_t b = smem_u32(bar);
    uint32_t done = 0;
    while (!done) {
        asm volatile(
            "{\n\t.reg .pred p;\n\t"
            "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], 0;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(done)
            : "r"(b)
            : "memory");
    }
}


// ---------------------------------------------------------------------------------- walker init
// a1 (Alg. 2 l.8-9 / A8 l.8-9): start pose S_0[w mod n0] and the velocity
// pointing away from the centre of S_0 plus a random unit vector.
template <int MODE>
__device__ __forceinline__ void init_walker(const InstanceDesc *__restrict__ D, const WalkLaunch &L, const Rng &rng,
                                            unsigned long long w, double (&R)[9], double (&t)[3], double (&vel)[3])
{
    {
        const double *init = D->S0 + 12 * (size_t)(w % (unsigned long long)D->n0);
#pragma unroll
        for (int e = 0; e < 9; ++e) R[e] = init[e];
#pragma unroll
        for (int e = 0; e < 3; ++e) t[e] = init[9 + e];
    }
    uint32_t o[4];
    philox4x32_10(rng.w_lo, 0u, 0u, 0u | rng.w_hi8, rng.k0, rng.k1, o);
    const double z = pm1(o[0]);
    const double phi = CUDART_PI * (pm1(o[1]) + 1.0);
    const double s = sqrt(fma(-z, z, 1.0));
    double sp, cp;
    sincos(phi, &sp, &cp);
    const double r0 = s * cp, r1 = s * sp, r2 = z;                    // random unit vector (R-4)
    if (MODE == CLOSURE_MODE_ROT) {
        double Rb[9], M[9];
#pragma unroll
        for (int e = 0; e < 9; ++e) Rb[e] = D->Rbar[e];
#pragma unroll
        for (int r = 0; r < 3; ++r)                                   // M = R_0 Rbar^T (R-2)
#pragma unroll
            for (int c = 0; c < 3; ++c)
                M[3 * r + c] = fma(R[3 * r + 2], Rb[3 * c + 2], fma(R[3 * r + 1], Rb[3 * c + 1], R[3 * r] * Rb[3 * c]));
        const double v0 = M[7] - M[5], v1 = M[2] - M[6], v2 = M[3] - M[1];
        const double nv = sqrt(fma(v2, v2, fma(v1, v1, v0 * v0)));
        const double theta = atan2(nv, (M[0] + M[4] + M[8]) - 1.0);
        double u0 = 0.0, u1 = 0.0, u2 = 0.0;
        if (nv > 0.0 && !(theta < 1e-12)) { u0 = v0 / nv; u1 = v1 / nv; u2 = v2 / nv; }   // R-3
        vel[0] = L.omega0 * (u0 + r0);
        vel[1] = L.omega0 * (u1 + r1);
        vel[2] = L.omega0 * (u2 + r2);
    } else {
        const double d0 = t[0] - D->tbar[0], d1 = t[1] - D->tbar[1], d2 = t[2] - D->tbar[2];
        const double nd = sqrt(fma(d2, d2, fma(d1, d1, d0 * d0)));
        const bool far = !(nd < 1e-12);
        const double w0 = L.v0 * ((far ? d0 / nd : 0.0) + r0);
        const double w1 = L.v0 * ((far ? d1 / nd : 0.0) + r1);
        const double w2 = L.v0 * ((far ? d2 / nd : 0.0) + r2);
        // PCA normalisation (R-23): identity unless CLOSURE_FLAG_PCA_VELOCITY was set
#pragma unroll
        for (int r = 0; r < 3; ++r)
            vel[r] = fma(D->vscale[3 * r + 2], w2, fma(D->vscale[3 * r + 1], w1, D->vscale[3 * r] * w0));
    }
}

// ladder dT_m = gamma^(m-1) by repeated multiplication (Alg. 2 l.20) and the coefficients of
// Exp(dT_m w) = I + a_m [w]x + b_m [w]x^2, (a_m, b_m) = (A dT_m, B dT_m^2); m-major so that the
// lanes of a warp hit distinct banks.
__device__ __forceinline__ void fill_ladder(const WalkLaunch &L, const double (&vel)[3], double2 *ladder)
{
    double dT = 1.0;
    for (int m = 0; m < L.n_t; ++m) {
        const double p0 = dT * vel[0], p1 = dT * vel[1], p2 = dT * vel[2];
        double A, B;
        exp_coeffs(fma(p2, p2, fma(p1, p1, p0 * p0)), A, B);
        ladder[m * kBlock + threadIdx.x] = make_double2(A * dT, B * dT * dT);
        dT = dT * L.gamma;
    }
}

}  // namespace
}  // namespace closure
