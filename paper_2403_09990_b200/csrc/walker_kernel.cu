// Walker kernel: Step II of CLOSURE (Alg. 2; Alg. A8 PAPER.md:1001-1066;
// tensorised prior art Alg. 3 / A9 PAPER.md:295-322, 1078-1099) for sm_100a.
//
// One walker per thread.  The pose (R*, t*) lives in registers for all N_I iterations; the
// instance's constraint table is staged ONCE per CTA into shared memory by a TMA bulk copy
// (cp.async.bulk + mbarrier) and is then read with warp-uniform (broadcast) loads; randomness
// is Philox4x32-10 keyed by (seed; walker, iteration, perturbation) (R-5), so the
// kernel stores no perturbation: the kept ones are re-generated from their index.
//
// What differs from the paper's CuPy formulation:
//  * ROT mode shares R* across the N_P perturbations and Exp(dT_m w)R* across the N_P* ladder
//    candidates, so per constraint the R-dependent part u_i = b_i - R a_i - t* is set up once
//    and each (perturbation, constraint) pair costs 3 FMA + 1 max:
//        ||u_i - d_j||^2 = (|u_i|^2 - 2 u_i.d_j) + |d_j|^2 .
//  * eq. (14)'s min_i(beta_i - ||g_i||) takes one sqrt per run of equal bounds (rows are sorted
//    by bound): min_i(beta - x_i) = beta - sqrt(max_i x_i^2), exact because sqrt and the
//    subtraction are monotone.
//  * The ladder is searched m = 1, 2, ... and stops at the first feasible rung (same result
//    as Alg. 3's dense evaluation followed by find_farthest); a rung's constraint loop stops as
//    soon as no candidate of any lane in the warp is still alive (warp-uniform exit).
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
__device__ __forceinline__ void mat3_mul(const double (&A)[9], const double (&B)[9], double (&C)[9])
{
#pragma unroll
    for (int r = 0; r < 3; ++r)
#pragma unroll
        for (int c = 0; c < 3; ++c)
            C[3 * r + c] = A[3 * r] * B[c] + A[3 * r + 1] * B[3 + c] + A[3 * r + 2] * B[6 + c];
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
    exp_coeffs(p0 * p0 + p1 * p1 + p2 * p2, A, B);
    const double K[9] = { 0.0, -p2, p1, p2, 0.0, -p0, -p1, p0, 0.0 };
    double K2[9];
    mat3_mul(K, K, K2);
#pragma unroll
    for (int e = 0; e < 9; ++e) E[e] = ((e % 4 == 0) ? 1.0 : 0.0) + A * K[e] + B * K2[e];
}

// Rm = R + a (w x R) + b (w x (w x R)), cross products taken column by column:
// Exp(dT w) R with a = A dT, b = B dT^2.
__device__ __forceinline__ void rotate_left(const double (&R)[9], double w0, double w1, double w2,
                                            double a, double b, double (&Rm)[9])
{
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const double x = R[c], y = R[3 + c], z = R[6 + c];
        const double p0 = w1 * z - w2 * y, p1 = w2 * x - w0 * z, p2 = w0 * y - w1 * x;       // w x col
        const double q0 = w1 * p2 - w2 * p1, q1 = w2 * p0 - w0 * p2, q2 = w0 * p1 - w1 * p0; // w x (w x col)
        Rm[c] = x + a * p0 + b * q0;
        Rm[3 + c] = y + a * p1 + b * q1;
        Rm[6 + c] = z + a * p2 + b * q2;
    }
}

// ---------------------------------------------------------------------------------- residuals
template <int RES> struct Res;
template <> struct Res<CLOSURE_REG_3D3D> { static constexpr int ROW = 8, BETA = 6; static constexpr bool AFFINE = true; };
template <> struct Res<CLOSURE_REPROJ_2D3D> { static constexpr int ROW = 8, BETA = 5; static constexpr bool AFFINE = false; };
template <> struct Res<CLOSURE_POSE_REG> { static constexpr int ROW = 16, BETA = 12; static constexpr bool AFFINE = true; };
template <> struct Res<CLOSURE_POSE_REG_SPLIT> { static constexpr int ROW = 16, BETA = 14; static constexpr bool AFFINE = true; };

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

// Direct evaluation of the squared residual at pose (R, t) (generic path).
// part: POSE_REG_SPLIT only, 0 = rotation bound, 1 = translation bound.
template <int RES>
__device__ __forceinline__ double direct_sq(const double (&R)[9], const double (&t)[3], const double *row,
                                            const double (&K)[4], int part)
{
    if (RES == CLOSURE_REG_3D3D) {
        const double a0 = row[0], a1 = row[1], a2 = row[2];
        const double g0 = row[3] - ((R[0] * a0 + R[1] * a1 + R[2] * a2) + t[0]);
        const double g1 = row[4] - ((R[3] * a0 + R[4] * a1 + R[5] * a2) + t[1]);
        const double g2 = row[5] - ((R[6] * a0 + R[7] * a1 + R[8] * a2) + t[2]);
        return g0 * g0 + g1 * g1 + g2 * g2;
    } else if (RES == CLOSURE_REPROJ_2D3D) {
        const double Z0 = row[2], Z1 = row[3], Z2 = row[4];
        const double p0 = (R[0] * Z0 + R[1] * Z1 + R[2] * Z2) + t[0];
        const double p1 = (R[3] * Z0 + R[4] * Z1 + R[5] * Z2) + t[1];
        const double p2 = (R[6] * Z0 + R[7] * Z1 + R[8] * Z2) + t[2];
        if (!(p2 > 0.0)) return CUDART_INF;                       // cheirality (R-10)
        const double g0 = row[0] - (K[0] * (p0 / p2) + K[2]);
        const double g1 = row[1] - (K[1] * (p1 / p2) + K[3]);
        return g0 * g0 + g1 * g1;
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

// ---------------------------------------------------------------------------------- the kernel
template <int RES, int MODE, int KCAP, bool STATS>
__global__ void __launch_bounds__(kBlock, 2) walker_kernel(const __grid_constant__ WalkLaunch L)
{
    using RS = Res<RES>;
    constexpr int ROW = RS::ROW;
    constexpr unsigned FULL = 0xffffffffu;

    extern __shared__ __align__(16) unsigned char smem_raw[];
    uint64_t *bar = reinterpret_cast<uint64_t *>(smem_raw);
    double *rows = reinterpret_cast<double *>(smem_raw + 16);

    const InstanceDesc *__restrict__ D = L.desc[blockIdx.y];
    const int n = D->n;
    const int rows_bytes = D->rows_bytes;
    stage_rows(smem_raw + 16, bar, D->rows, rows_bytes);
    // ladder table (ROT): per walker (a_m, b_m), m-major so that lanes hit distinct banks
    double2 *ladder = reinterpret_cast<double2 *>(smem_raw + 16 + ((rows_bytes + 15) & ~15));

    const long long local = (long long)blockIdx.x * kBlock + threadIdx.x;
    const bool valid = local < L.num_walkers;
    // threads past the end shadow the last walker (keeps every warp-collective full) and write nothing
    const unsigned long long w = (unsigned long long)(L.walker_begin + (valid ? local : L.num_walkers - 1));
    const unsigned long long seed = L.seed[blockIdx.y];
    Rng rng;
    rng.w_lo = (uint32_t)w;
    rng.w_hi8 = (uint32_t)(w >> 32) << 8;
    rng.k0 = (uint32_t)seed;
    rng.k1 = (uint32_t)(seed >> 32);

    double K[4];
#pragma unroll
    for (int e = 0; e < 4; ++e) K[e] = D->K[e];

    // ---- a1: walker init (Alg. 2 l.8-9 / A8 l.8-9)
    double R[9], t[3];
    {
        const double *init = D->S0 + 12 * (size_t)(w % (unsigned long long)D->n0);
#pragma unroll
        for (int e = 0; e < 9; ++e) R[e] = init[e];
#pragma unroll
        for (int e = 0; e < 3; ++e) t[e] = init[9 + e];
    }
    double vel[3];   // omega (ROT) or v (TRANS)
    {
        uint32_t o[4];
        philox4x32_10(rng.w_lo, 0u, 0u, 0u | rng.w_hi8, rng.k0, rng.k1, o);
        const double z = pm1(o[0]);
        const double phi = CUDART_PI * (pm1(o[1]) + 1.0);
        const double s = sqrt(1.0 - z * z);
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
                    M[3 * r + c] = R[3 * r] * Rb[3 * c] + R[3 * r + 1] * Rb[3 * c + 1] + R[3 * r + 2] * Rb[3 * c + 2];
            const double v0 = M[7] - M[5], v1 = M[2] - M[6], v2 = M[3] - M[1];
            const double nv = sqrt(v0 * v0 + v1 * v1 + v2 * v2);
            const double theta = atan2(nv, (M[0] + M[4] + M[8]) - 1.0);
            double u0 = 0.0, u1 = 0.0, u2 = 0.0;
            if (nv > 0.0 && !(theta < 1e-12)) { u0 = v0 / nv; u1 = v1 / nv; u2 = v2 / nv; }   // R-3
            vel[0] = L.omega0 * (u0 + r0);
            vel[1] = L.omega0 * (u1 + r1);
            vel[2] = L.omega0 * (u2 + r2);
        } else {
            const double d0 = t[0] - D->tbar[0], d1 = t[1] - D->tbar[1], d2 = t[2] - D->tbar[2];
            const double nd = sqrt(d0 * d0 + d1 * d1 + d2 * d2);
            const bool far = !(nd < 1e-12);
            vel[0] = L.v0 * ((far ? d0 / nd : 0.0) + r0);
            vel[1] = L.v0 * ((far ? d1 / nd : 0.0) + r1);
            vel[2] = L.v0 * ((far ? d2 / nd : 0.0) + r2);
        }
    }
    if (MODE == CLOSURE_MODE_ROT) {
        // ladder dT_m = gamma^(m-1) by repeated multiplication (Alg. 2 l.20); Exp(dT_m w) coefficients
        double dT = 1.0;
        for (int m = 0; m < L.n_t; ++m) {
            const double p0 = dT * vel[0], p1 = dT * vel[1], p2 = dT * vel[2];
            double A, B;
            exp_coeffs(p0 * p0 + p1 * p1 + p2 * p2, A, B);
            ladder[m * kBlock + threadIdx.x] = make_double2(A * dT, B * dT * dT);
            dT = dT * L.gamma;
        }
    }

    unsigned long long st_pp = 0, st_lp = 0, st_ps = 0, st_ls = 0, st_acc = 0;
    bool hit = false;
    const int n_p = L.n_p, n_ps = L.n_p_star, n_t = L.n_t;
    const unsigned kmask = n_ps >= 32 ? 0xffffffffu : ((1u << n_ps) - 1u);

    for (int s = 1; s <= L.num_steps; ++s) {
        TopK<KCAP> top;
        top.clear();

        // ================================================== a2-a4: perturb, eq. (14), top-k
        if (MODE == CLOSURE_MODE_ROT) {
            double rot_margin = CUDART_INF;     // POSE_REG_SPLIT: rotation bounds do not see d_j
            if (RES == CLOSURE_POSE_REG_SPLIT) {
                for (int i = 0; i < n; ++i) {
                    const double *row = rows + i * ROW;
                    rot_margin = dmin(rot_margin, row[12] - sqrt(frob_sq(R, row)));
                }
            }
            for (int j0 = 0; j0 < n_p; j0 += kJT) {
                double e0[kJT], e1[kJT], e2[kJT], dd[kJT], acc_mx[kJT], dmn[kJT];
#pragma unroll
                for (int jj = 0; jj < kJT; ++jj) {
                    double x, y, z;
                    rng.xi3((uint32_t)s, (uint32_t)(j0 + jj), 1u, x, y, z);
                    const double d0 = L.t_p * x, d1 = L.t_p * y, d2 = L.t_p * z;
                    e0[jj] = d0; e1[jj] = d1; e2[jj] = d2;
                    dd[jj] = fma(d2, d2, fma(d1, d1, d0 * d0));
                    acc_mx[jj] = -CUDART_INF;
                    dmn[jj] = rot_margin;
                }
                if (RS::AFFINE) {
#pragma unroll
                    for (int jj = 0; jj < kJT; ++jj) { e0[jj] *= -2.0; e1[jj] *= -2.0; e2[jj] *= -2.0; }
                    for (int i = 0; i < n; ++i) {
                        const double *row = rows + i * ROW;
                        double u0, u1, u2, c;
                        affine_setup<RES>(R, t, row, u0, u1, u2, c);
#pragma unroll
                        for (int jj = 0; jj < kJT; ++jj)
                            acc_mx[jj] = dmax(acc_mx[jj], fma(u0, e0[jj], fma(u1, e1[jj], fma(u2, e2[jj], c))));
                        const double beta = row[RS::BETA];
                        const bool run_ends = (i == n - 1) || (rows[(i + 1) * ROW + RS::BETA] != beta);
                        if (run_ends) {                          // warp-uniform
#pragma unroll
                            for (int jj = 0; jj < kJT; ++jj) {
                                dmn[jj] = dmin(dmn[jj], beta - sqrt(dmax(acc_mx[jj] + dd[jj], 0.0)));
                                acc_mx[jj] = -CUDART_INF;
                            }
                        }
                    }
                    if (STATS) { st_pp += (unsigned long long)n * kJT; st_ps += n; }
                } else {
                    // REPROJ: P_i = R Z_i + t* once per constraint, then one projection per perturbation
                    for (int i = 0; i < n; ++i) {
                        const double *row = rows + i * ROW;
                        const double Z0 = row[2], Z1 = row[3], Z2 = row[4];
                        const double P0 = R[0] * Z0 + R[1] * Z1 + R[2] * Z2;
                        const double P1 = R[3] * Z0 + R[4] * Z1 + R[5] * Z2;
                        const double P2 = R[6] * Z0 + R[7] * Z1 + R[8] * Z2;
                        const double beta = row[RS::BETA];
#pragma unroll
                        for (int jj = 0; jj < kJT; ++jj) {
                            const double p0 = P0 + (t[0] + e0[jj]), p1 = P1 + (t[1] + e1[jj]), p2 = P2 + (t[2] + e2[jj]);
                            double sq = CUDART_INF;
                            if (p2 > 0.0) {
                                const double g0 = row[0] - (K[0] * (p0 / p2) + K[2]);
                                const double g1 = row[1] - (K[1] * (p1 / p2) + K[3]);
                                sq = g0 * g0 + g1 * g1;
                            }
                            dmn[jj] = dmin(dmn[jj], beta - sqrt(sq));
                        }
                    }
                    if (STATS) { st_pp += (unsigned long long)n * kJT; st_ps += n; }
                }
#pragma unroll
                for (int jj = 0; jj < kJT; ++jj)
                    if (j0 + jj < n_p) top.insert(dmn[jj], j0 + jj);
            }
        } else {
            // TRANS (A8 l.12-15, A9): R_j = Exp(theta_p xi_j) R*, t_j = t*
            for (int j = 0; j < n_p; ++j) {
                double x, y, z, E[9], Rj[9];
                rng.xi3((uint32_t)s, (uint32_t)j, 1u, x, y, z);
                exp_so3(L.theta_p * x, L.theta_p * y, L.theta_p * z, E);
                mat3_mul(E, R, Rj);
                top.insert(margin_direct<RES>(Rj, t, rows, n, K), j);
            }
            if (STATS) { st_pp += (unsigned long long)n * n_p; st_ps += (unsigned long long)n * n_p; }
        }

        // ================================================== a5-a6: ladder, first feasible rung
        int m0 = 0, j_win = 0;
        if (MODE == CLOSURE_MODE_ROT) {
            // re-generate the kept perturbations from their indices
            double k0[KCAP], k1[KCAP], k2[KCAP], kdd[KCAP];
#pragma unroll
            for (int k = 0; k < KCAP; ++k) {
                double x, y, z;
                rng.xi3((uint32_t)s, (uint32_t)top.j[k], 1u, x, y, z);
                const double d0 = L.t_p * x, d1 = L.t_p * y, d2 = L.t_p * z;
                kdd[k] = -fma(d2, d2, fma(d1, d1, d0 * d0));
                if (RS::AFFINE) { k0[k] = -2.0 * d0; k1[k] = -2.0 * d1; k2[k] = -2.0 * d2; }
                else { k0[k] = d0; k1[k] = d1; k2[k] = d2; }
            }
            unsigned win = 0;
            for (int m = 0; m < n_t; ++m) {
                if (!__any_sync(FULL, m0 == 0)) break;
                const double2 ab = ladder[m * kBlock + threadIdx.x];
                double Rm[9];
                rotate_left(R, vel[0], vel[1], vel[2], ab.x, ab.y, Rm);
                unsigned alive = (m0 == 0) ? kmask : 0u;
                int i = 0;
                for (; i < n; ++i) {
                    const double *row = rows + i * ROW;
                    if (RS::AFFINE) {
                        double u0, u1, u2, c;
                        affine_setup<RES>(Rm, t, row, u0, u1, u2, c);
                        if (RES == CLOSURE_POSE_REG_SPLIT) {
                            if (!(frob_sq(Rm, row) <= row[13])) alive = 0u;
                        }
                        const double cb = c - row[RS::BETA + 1];
#pragma unroll
                        for (int k = 0; k < KCAP; ++k) {
                            const double v = fma(u0, k0[k], fma(u1, k1[k], fma(u2, k2[k], cb)));
                            if (!(v <= kdd[k])) alive &= ~(1u << k);
                        }
                    } else {
                        const double Z0 = row[2], Z1 = row[3], Z2 = row[4];
                        const double P0 = Rm[0] * Z0 + Rm[1] * Z1 + Rm[2] * Z2;
                        const double P1 = Rm[3] * Z0 + Rm[4] * Z1 + Rm[5] * Z2;
                        const double P2 = Rm[6] * Z0 + Rm[7] * Z1 + Rm[8] * Z2;
                        const double b2 = row[RS::BETA + 1];
#pragma unroll
                        for (int k = 0; k < KCAP; ++k) {
                            const double p0 = P0 + (t[0] + k0[k]), p1 = P1 + (t[1] + k1[k]), p2 = P2 + (t[2] + k2[k]);
                            bool ok = false;
                            if (p2 > 0.0) {
                                const double g0 = row[0] - (K[0] * (p0 / p2) + K[2]);
                                const double g1 = row[1] - (K[1] * (p1 / p2) + K[3]);
                                ok = (g0 * g0 + g1 * g1) <= b2;
                            }
                            if (!ok) alive &= ~(1u << k);
                        }
                    }
                    if (!__any_sync(FULL, alive != 0u)) { ++i; break; }
                }
                if (STATS) { st_lp += (unsigned long long)i * n_ps; st_ls += i; }
                if (alive) { m0 = m + 1; win = alive; }
            }
            if (m0) {
                const int kw = __ffs(win) - 1;                    // lowest rank among the feasible (R-8)
                int jw = 0;
#pragma unroll
                for (int k = 0; k < KCAP; ++k) if (k == kw) jw = top.j[k];
                j_win = jw;
                const double2 ab = ladder[(m0 - 1) * kBlock + threadIdx.x];
                double Rm[9];
                rotate_left(R, vel[0], vel[1], vel[2], ab.x, ab.y, Rm);
#pragma unroll
                for (int e = 0; e < 9; ++e) R[e] = Rm[e];
                double x, y, z;
                rng.xi3((uint32_t)s, (uint32_t)jw, 1u, x, y, z);
                t[0] = __dadd_rn(t[0], __dmul_rn(L.t_p, x));
                t[1] = __dadd_rn(t[1], __dmul_rn(L.t_p, y));
                t[2] = __dadd_rn(t[2], __dmul_rn(L.t_p, z));
            }
        } else {
            double dT = 1.0;
            for (int m = 0; m < n_t && m0 == 0; ++m) {
                double tm[3];
                tm[0] = __dadd_rn(t[0], __dmul_rn(dT, vel[0]));
                tm[1] = __dadd_rn(t[1], __dmul_rn(dT, vel[1]));
                tm[2] = __dadd_rn(t[2], __dmul_rn(dT, vel[2]));
#pragma unroll 1
                for (int k = 0; k < n_ps; ++k) {
                    int jk = 0;
#pragma unroll
                    for (int q = 0; q < KCAP; ++q) if (q == k) jk = top.j[q];
                    double x, y, z, E[9], Rj[9];
                    rng.xi3((uint32_t)s, (uint32_t)jk, 1u, x, y, z);
                    exp_so3(L.theta_p * x, L.theta_p * y, L.theta_p * z, E);
                    mat3_mul(E, R, Rj);
                    if (STATS) st_ls += n;
                    if (in_purse_direct<RES>(Rj, tm, rows, n, K, st_lp)) {
#pragma unroll
                        for (int e = 0; e < 9; ++e) R[e] = Rj[e];
                        t[0] = tm[0]; t[1] = tm[1]; t[2] = tm[2];
                        m0 = m + 1; j_win = jk;
                        break;
                    }
                }
                dT = dT * L.gamma;
            }
        }
        if (m0 != 1) hit = true;                                   // R-12 (R-11: nothing feasible -> unchanged)
        if (STATS && m0) ++st_acc;
        if (L.out_trace != nullptr && valid)
            L.out_trace[((size_t)blockIdx.y * L.num_walkers + local) * L.num_steps + (s - 1)] = m0 | (j_win << 8);
    }

    // ---- a7: emit
    if (valid) {
        const size_t o = (size_t)blockIdx.y * L.num_walkers + local;
        double2 *dst = reinterpret_cast<double2 *>(L.out_samples + 12 * o);
        dst[0] = make_double2(R[0], R[1]); dst[1] = make_double2(R[2], R[3]); dst[2] = make_double2(R[4], R[5]);
        dst[3] = make_double2(R[6], R[7]); dst[4] = make_double2(R[8], t[0]); dst[5] = make_double2(t[1], t[2]);
        L.out_flags[o] = hit ? 1 : 0;
    }
    if (STATS && L.stats != nullptr && valid) {
        atomicAdd(L.stats + 0, st_pp); atomicAdd(L.stats + 1, st_lp); atomicAdd(L.stats + 2, st_ps);
        atomicAdd(L.stats + 3, st_ls); atomicAdd(L.stats + 4, st_acc);
        atomicAdd(L.stats + 5, (unsigned long long)L.num_steps);
    }
}

template <int RES, int MODE, int KCAP>
cudaError_t launch_k(bool stats, const WalkLaunch &L, dim3 grid, size_t smem, cudaStream_t stream)
{
    cudaError_t e;
    if (stats) {
        e = cudaFuncSetAttribute(walker_kernel<RES, MODE, KCAP, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        walker_kernel<RES, MODE, KCAP, true><<<grid, kBlock, smem, stream>>>(L);
    } else {
        e = cudaFuncSetAttribute(walker_kernel<RES, MODE, KCAP, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        walker_kernel<RES, MODE, KCAP, false><<<grid, kBlock, smem, stream>>>(L);
    }
    return cudaGetLastError();
}

template <int RES, int MODE>
cudaError_t launch_rm(bool stats, const WalkLaunch &L, dim3 grid, size_t smem, cudaStream_t stream)
{
    if (L.n_p_star <= 2) return launch_k<RES, MODE, 2>(stats, L, grid, smem, stream);
    if (L.n_p_star <= 10) return launch_k<RES, MODE, 10>(stats, L, grid, smem, stream);
    return launch_k<RES, MODE, kMaxKStar>(stats, L, grid, smem, stream);
}

template <int RES>
cudaError_t launch_r(int mode, bool stats, const WalkLaunch &L, dim3 grid, size_t smem, cudaStream_t stream)
{
    if (mode == CLOSURE_MODE_ROT) return launch_rm<RES, CLOSURE_MODE_ROT>(stats, L, grid, smem, stream);
    return launch_rm<RES, CLOSURE_MODE_TRANS>(stats, L, grid, smem, stream);
}

}  // namespace

int row_doubles(int residual_type)
{
    switch (residual_type) {
    case CLOSURE_REG_3D3D: return Res<CLOSURE_REG_3D3D>::ROW;
    case CLOSURE_REPROJ_2D3D: return Res<CLOSURE_REPROJ_2D3D>::ROW;
    case CLOSURE_POSE_REG: return Res<CLOSURE_POSE_REG>::ROW;
    case CLOSURE_POSE_REG_SPLIT: return Res<CLOSURE_POSE_REG_SPLIT>::ROW;
    default: return 0;
    }
}

cudaError_t launch_walkers(int residual_type, int mode, bool stats, const WalkLaunch &L, int n_instances,
                           int max_rows_bytes, cudaStream_t stream, std::string *why)
{
    if (L.num_walkers <= 0 || n_instances <= 0) return cudaSuccess;
    const long long blocks = (L.num_walkers + kBlock - 1) / kBlock;
    if (blocks > 0x7fffffffLL) {
        if (why) *why = "too many walkers for one launch";
        return cudaErrorInvalidValue;
    }
    dim3 grid((unsigned)blocks, (unsigned)n_instances, 1);
    const size_t smem = 16 + (size_t)((max_rows_bytes + 15) & ~15) + (size_t)L.n_t * kBlock * sizeof(double2);
    if (smem > 200 * 1024) {
        if (why) *why = "instance too large for shared-memory staging";
        return cudaErrorInvalidValue;
    }
    switch (residual_type) {
    case CLOSURE_REG_3D3D: return launch_r<CLOSURE_REG_3D3D>(mode, stats, L, grid, smem, stream);
    case CLOSURE_REPROJ_2D3D: return launch_r<CLOSURE_REPROJ_2D3D>(mode, stats, L, grid, smem, stream);
    case CLOSURE_POSE_REG: return launch_r<CLOSURE_POSE_REG>(mode, stats, L, grid, smem, stream);
    case CLOSURE_POSE_REG_SPLIT: return launch_r<CLOSURE_POSE_REG_SPLIT>(mode, stats, L, grid, smem, stream);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace closure
