// Warp-cooperative walker kernel, DENSE variant (every perturbation against every constraint), for the rotation-
// boundary sampler (Alg. 2) on
// the residuals whose squared norm is quadratic in the translation perturbation (Ex.2 registration,
// Ex.3 pose regression, stacked or split).  One WARP owns one walker; the 32 lanes split the work
// that Alg. 3 tensorises per walker:
//
//   a2-a4  the N_P perturbations are dealt to the lanes (j = lane + 32 q); the per-constraint
//          set-up u_i = b_i - (R* a_i + t*) is computed ONCE per accepted move (lane i mod 32)
//          and broadcast through shared memory; a pair costs 3 FFMA + 1 FMNMX in fp32
//          (packed FFMA2 + FMNMX3 in SASS).  eq. (14)'s values d~_j carry a rigorous error bound
//          `unc`; the top-N_P* are extracted with warp reductions and the ranking is accepted only
//          if consecutive values (and the N_P*-th against the next) are more than 2 unc apart.
//          Otherwise the step falls back to the fp64 evaluation of the plain kernel.
//   a5-a6  every rung m = 1..N_T is screened first (lane = (rung, half of the candidates)) against the
//          rung's two tightest constraints and against a Lipschitz bound on what the rotation to R_m
//          can repair; rungs with a surviving candidate are then evaluated in full, lane =
//          (candidate, constraint chunk), in fp32 with a three-way outcome per candidate: violated
//          for sure / satisfied for sure / undecided -> fp64.
//
// launch_walkers_coop (walker_coop_kernel.cu) sends short tables with many perturbations here (N_P > 32 and at most 32
// pair-entries: BASELINE configs 1, 2 and 4): the branch and bound of walker_coop_kernel.cu saves arithmetic but its
// bookkeeping only pays on longer tables or few perturbations.
//
// Every accept/reject decision is therefore the decision the fp64 arithmetic of walker_kernel.cu
// takes (DESIGN.md 6.1b "Certified fp32 evaluation"); the pose itself is only ever updated in fp64.
// Unlike the one-walker-per-thread kernel all lanes of a warp follow the same walker: no divergence
// between walkers, the set-up is not repeated per register tile, 128 registers (16 warps per SM).
#include <cuda_runtime.h>
#include <math_constants.h>
#include <stdint.h>

#include "closure_internal.h"
#include "walker_common.cuh"
#include "walker_coop_common.cuh"

#ifndef CLOSURE_COOP_MIN_CTAS
#define CLOSURE_COOP_MIN_CTAS 4   // resident CTAs per SM the register allocation aims at (128 registers per thread)
#endif

#ifndef CLOSURE_ELL_MIN_CTAS
#define CLOSURE_ELL_MIN_CTAS 4    // ellipsoid pair loop: nine packed FMAs per pair want the registers
#endif

namespace closure {
namespace {

// Measured on B200: the pose-regression kernel, whose rows are twice as long, gains 3.7 % at 6 resident
// CTAs (80 registers); the registration kernel gains 1 % at 5 (96 registers) in the NQ = 5 instantiation (64 < N_P <= 160: C2) and stays at 4 for
// fewer perturbations, where the table of a C5-sized instance allows 4 CTAs anyway.
template <int RES, int NQ> constexpr int coop_min_ctas()
{
    if (CLOSURE_COOP_MIN_CTAS != 4) return CLOSURE_COOP_MIN_CTAS;
    if (RES == CLOSURE_POSE_REG || RES == CLOSURE_POSE_REG_SPLIT) return 6;
    if (RES == CLOSURE_REG_3D3D_ELL) return CLOSURE_ELL_MIN_CTAS;
    return NQ == 5 ? 5 : 4;
}

// fp32 image of one set-up row and the bound eps on |v32 - v64| for ANY perturbation with
// |d_c| <= t_p, where v = c - 2 u.d is evaluated as three chained FMAs:
//   inputs: (u, c) rounded to fp32 (relative 2^-24 each); e = -2 d from pm1f (absolute 6 * 2^-24 * 2 t_p);
//   three FFMA roundings (2^-24 of the partial sums, each <= |c| + 2 t_p |u|_1)
//   =>  |v32 - v64| <= 2^-24 (4 |c| + 10 * 2 t_p |u|_1).
// eps = 2^-19 (|c| + 2 t_p |u|_1 + 3 t_p^2) leaves a factor > 3 for the roundings of eps itself,
// of the threshold -|d|^2 in fp32 (<= 15 * 2^-24 * 3 t_p^2) and of the shifted constants c -+ eps.
__device__ __forceinline__ void screen_row(double u0, double u1, double u2, double c, float tp2, float tp2sq3,
                                           float &f0, float &f1, float &f2, float &fc, float &eps)
{
    f0 = (float)u0; f1 = (float)u1; f2 = (float)u2; fc = (float)c;
    const float mag = fabsf(fc) + tp2 * (fabsf(f0) + fabsf(f1) + fabsf(f2)) + tp2sq3;
    eps = mag * (kMu19 * 1.001f);
}

// ---------------------------------------------------------------------------------- ellipsoid norm (eq. (6), Lambda_i != I)
// CLOSURE_REG_3D3D_ELL: |g|_L^2 = g^T L g with g = u - d, u = b - (R a + t*):
//     (u - d)^T L (u - d) = c - 2 w.d + d^T L d,      w = L u,   c = u^T L u,
// i.e. the affine form of Ex.2 with (w, c) in place of (u, |u|^2) plus a quadratic form in the perturbation whose six
// coefficients are constants of the constraint.  With e = -2 d (what the lanes hold) the pair is
//     v = c + e0 (w0 + Q00 e0 + Q01 e1 + Q02 e2) + e1 (w1 + Q11 e1 + Q12 e2) + e2 (w2 + Q22 e2),
//     Q00 = L00/4, Q11 = L11/4, Q22 = L22/4, Q01 = L01/2, Q02 = L02/2, Q12 = L12/2              (9 FMA)
// Error of the fp32 evaluation against the plain kernel's fp64 g^T (L g), for |e_a| <= 2 t_p, with
// M = |c| + 2 t_p |w|_1 + (2 t_p)^2 sum|Q|:  nine FMA roundings (<= 9 2^-24 M), (w, c, Q) rounded to fp32 (<= 2^-24 M),
// e from pm1f (6 2^-24 2 t_p per component, times |dv/de_a| <= |w_a| + 2 (2 t_p) sum_b |Q_ab|: <= 24 2^-24 M):
// |v32 - v64| <= 34 2^-24 M.  eps = 2^-18 1.001 M (= 64 2^-24 M) leaves a factor 1.9 over that worst case.
constexpr float kMuEll = 3.814697265625e-06f;   // 2^-18 (measured: 2^-17 sends 7.8 % of the iterations to the fp64 fall-back, 2^-18 see DESIGN.md)
constexpr int kEll = CLOSURE_REG_3D3D_ELL;

__device__ __forceinline__ void ell_setup(const double (&R)[9], const double (&t)[3], const double *row, double &w0, double &w1,
                                          double &w2, double &c)
{
    const double a0 = row[0], a1 = row[1], a2 = row[2];
    const double u0 = row[3] - (fma(R[0], a0, fma(R[1], a1, R[2] * a2)) + t[0]);
    const double u1 = row[4] - (fma(R[3], a0, fma(R[4], a1, R[5] * a2)) + t[1]);
    const double u2 = row[5] - (fma(R[6], a0, fma(R[7], a1, R[8] * a2)) + t[2]);
    w0 = fma(row[8], u0, fma(row[9], u1, row[10] * u2));
    w1 = fma(row[9], u0, fma(row[11], u1, row[12] * u2));
    w2 = fma(row[10], u0, fma(row[12], u1, row[13] * u2));
    c = fma(u2, w2, fma(u1, w1, u0 * w0));
}

// |Lambda_i|_F (>= its largest eigenvalue): |x|_Lambda^2 <= |Lambda|_F |x|^2, for the Lipschitz bound of a rung
__device__ __forceinline__ double ell_lip_scale(const double *row)
{
    const double d = row[8] * row[8] + row[11] * row[11] + row[13] * row[13];
    const double o = row[9] * row[9] + row[10] * row[10] + row[12] * row[12];
    return sqrt(d + 2.0 * o) * 1.0000001;
}

// set-up of one constraint row at (R, t): (u, |u|^2 [+ |R - R_i|_F^2]) for the ball forms, (w, c) for the ellipsoid
template <int RES>
__device__ __forceinline__ void pair_setup(const double (&R)[9], const double (&t)[3], const double *row, double &u0, double &u1,
                                           double &u2, double &c)
{
    if (RES == kEll) ell_setup(R, t, row, u0, u1, u2, c);
    else affine_setup<RES>(R, t, row, u0, u1, u2, c);
}

// fp32 image and error bound of one row; qmag = (2 t_p)^2 sum|Q| of the constraint (ellipsoid only)
template <int RES>
__device__ __forceinline__ void screen_row_any(double u0, double u1, double u2, double c, float tp2, float tp2sq3, float qmag,
                                               float &f0, float &f1, float &f2, float &fc, float &eps)
{
    if (RES == kEll) {
        f0 = (float)u0; f1 = (float)u1; f2 = (float)u2; fc = (float)c;
        const float mag = fabsf(fc) + tp2 * (fabsf(f0) + fabsf(f1) + fabsf(f2)) + qmag;
        eps = mag * (kMuEll * 1.001f);
    } else {
        screen_row(u0, u1, u2, c, tp2, tp2sq3, f0, f1, f2, fc, eps);
    }
}

// q(e) of the constraint whose coefficients are (A, B) = (Q00 Q01 Q02 Q11) (Q12 Q22 . .), plus the linear part w.e + cw
__device__ __forceinline__ float ell_value(const float4 &r, const float4 &A, const float4 &B, const float4 &e)
{
    const float t0 = fmaf(A.z, e.z, fmaf(A.y, e.y, fmaf(A.x, e.x, r.x)));
    const float t1 = fmaf(B.x, e.z, fmaf(A.w, e.y, r.y));
    const float t2 = fmaf(B.y, e.z, r.z);
    return fmaf(t0, e.x, fmaf(t1, e.y, fmaf(t2, e.z, r.w)));
}

// The plain kernel's phase A for the NQ perturbations of this lane (same arithmetic as
// walker_kernel.cu): exact eq. (14) margins, one sqrt per run of equal bounds.  jv[q] < 0: empty.
template <int RES, int NJ>
__device__ __forceinline__ void exact_margins(const double (&R)[9], const double (&t)[3], const double *rows, int n,
                                              const Rng &rng, uint32_t s, double t_p, double rot_margin,
                                              const int (&jv)[NJ], double (&d)[NJ])
{
    using RS = Res<RES>;
    constexpr int ROW = RS::ROW;
    uint32_t x[NJ], y[NJ], z[NJ];
    philox_batch<NJ>(rng, s, jv, x, y, z);
    double e0[NJ], e1[NJ], e2[NJ], dd[NJ], acc_mx[NJ];
#pragma unroll
    for (int q = 0; q < NJ; ++q) {
        const double d0 = t_p * pm1(x[q]), d1 = t_p * pm1(y[q]), d2 = t_p * pm1(z[q]);
        dd[q] = fma(d2, d2, fma(d1, d1, d0 * d0));
        e0[q] = d0 * -2.0; e1[q] = d1 * -2.0; e2[q] = d2 * -2.0;
        acc_mx[q] = -CUDART_INF;
        d[q] = rot_margin;
    }
#pragma unroll 1
#pragma unroll 1
    for (int i = 0; i < n; ++i) {
        const double *row = rows + i * ROW;
        double u0, u1, u2, c;
        affine_setup<RES>(R, t, row, u0, u1, u2, c);
#pragma unroll
        for (int q = 0; q < NJ; ++q)
            acc_mx[q] = dmax(acc_mx[q], fma(u0, e0[q], fma(u1, e1[q], fma(u2, e2[q], c))));
        const double beta = row[RS::BETA];
        const bool run_ends = (i == n - 1) || (rows[(i + 1) * ROW + RS::BETA] != beta);
        if (run_ends) {                          // warp-uniform
#pragma unroll
            for (int q = 0; q < NJ; ++q) {
                d[q] = dmin(d[q], beta - sqrt(dmax(acc_mx[q] + dd[q], 0.0)));
                acc_mx[q] = -CUDART_INF;
            }
        }
    }
}

// eq. (14) of one perturbation in the plain kernel's arithmetic (functor for topk_fp64)
template <int RES>
struct ExactMargin {
    const double (&R)[9];
    const double (&t)[3];
    const double *rows;
    int n;
    const Rng &rng;
    uint32_t s;
    double t_p, rot_margin;
    __device__ __forceinline__ double operator()(int j) const
    {
        if (RES == kEll) {                            // the plain kernel's direct evaluation (walker_kernel.cu, non-affine branch)
            double x, y, z;
            rng.xi3(s, (uint32_t)j, 1u, x, y, z);
            const double tj[3] = { t[0] + t_p * x, t[1] + t_p * y, t[2] + t_p * z };
            const double K0[4] = { 0.0, 0.0, 0.0, 0.0 };
            double d = rot_margin;
#pragma unroll 1
            for (int i = 0; i < n; ++i) {
                const double *row = rows + i * Res<RES>::ROW;
                d = dmin(d, row[Res<RES>::BETA] - sqrt(direct_sq<RES>(R, tj, row, K0, 0)));
            }
            return d;
        }
        const int jv[1] = { j };
        double d[1];
        exact_margins<RES, 1>(R, t, rows, n, rng, s, t_p, rot_margin, jv, d);
        return d[0];
    }
};

// fp64 in_purse of ladder candidate (Rm, t* + d_j), constraints dealt to the lanes; the arithmetic
// of the plain kernel's ladder.  Warp-uniform result.
template <int RES>
__device__ __forceinline__ bool exact_candidate_feasible(const double (&Rm)[9], const double (&t)[3], const double *rows,
                                                         int n, const Rng &rng, uint32_t s, int j, double t_p, int lane)
{
    using RS = Res<RES>;
    constexpr int ROW = RS::ROW;
    double x, y, z;
    rng.xi3(s, (uint32_t)j, 1u, x, y, z);
    const double d0 = t_p * x, d1 = t_p * y, d2 = t_p * z;
    if (RES == kEll) {                                // the plain kernel's direct ladder test
        const double tk[3] = { t[0] + d0, t[1] + d1, t[2] + d2 };
        const double K0[4] = { 0.0, 0.0, 0.0, 0.0 };
        bool okl = true;
#pragma unroll 1
        for (int i = lane; i < n; i += 32) {
            const double *row = rows + i * ROW;
            if (!(direct_sq<RES>(Rm, tk, row, K0, 0) <= row[RS::BETA + 1])) okl = false;
        }
        return __all_sync(FULL, okl);
    }
    const double kdd = -fma(d2, d2, fma(d1, d1, d0 * d0));
    const double k0 = -2.0 * d0, k1 = -2.0 * d1, k2 = -2.0 * d2;
    bool ok = true;
#pragma unroll 1
    for (int i = lane; i < n; i += 32) {
        const double *row = rows + i * ROW;
        double u0, u1, u2, c;
        affine_setup<RES>(Rm, t, row, u0, u1, u2, c);
        if (RES == CLOSURE_POSE_REG_SPLIT) {
            if (!(frob_sq(Rm, row) <= row[13])) ok = false;
        }
        const double cb = c - row[RS::BETA + 1];
        const double v = fma(u0, k0, fma(u1, k1, fma(u2, k2, cb)));
        if (!(v <= kdd)) ok = false;
    }
    return __all_sync(FULL, ok);
}

// float4 words per constraint of the CTA-level fp32 table behind the set-up's search for screening rows:
// Ex.2 (a_i, beta_i^2); Ex.3 stacked (R_i row 0, beta_i^2) (R_i row 1, 0) (R_i row 2, 0); split form: none (old search)
template <int RES> __host__ __device__ constexpr int af_width()
{
    return RES == CLOSURE_REG_3D3D ? 1 : (RES == CLOSURE_POSE_REG ? 3 : (RES == CLOSURE_REG_3D3D_ELL ? 2 : 0));
}
// ellipsoid: the table holds the quadratic-form coefficients instead, by constraint (2 float4) and by pair-entry (3 float4)
template <int RES> __host__ __device__ constexpr int af_extra(int pairs) { return RES == CLOSURE_REG_3D3D_ELL ? pairs * 48 : 0; }

// ---------------------------------------------------------------------------------- screening rows of every rung
// Per rung the ladder screens its candidates against two constraint rows at R_m and against a Lipschitz bound.  ANY two
// constraints give valid rows (a violated row kills a candidate whichever row it is); the two TIGHTEST ones kill most.
// Round 1 found them by setting up all N rows of all N_T rungs in fp64 (N N_T set-ups per move: 59 % of the warp cycles at
// N_I = 5, where most iterations move).  Here the SEARCH runs in plain fp32 from what the set-up at R* already holds,
//     Ex.2:  u^m_i = u*_i - (R_m - R*) a_i,    key_i = |u^m_i|^2 - beta_i^2        (9 + 3 + 3 FMA)
//     Ex.3:  key_i = |u_i|^2 + |R_m - R_i|_F^2 - beta_i^2                            (9 SUB + 9 FMA)
// with no error analysis (a near-tie picks another, equally valid pair), and only the two chosen rows per rung get the
// rigorous fp64 set-up + screen_row() of before (2 N_T set-ups per move, rung m on lane m).  The Lipschitz bound of Ex.2,
// max_i |(R_m - R*) a_i|, comes out of the same fp32 pass with a slack that covers its rounding (|g32 - g| <= 5 2^-24
// |R_m - R*|_F |a_i| per component chain; 4e-6 |dR|_F max|a| is > 10x that); Ex.3's |R_m - R*|_F stays in fp64.
template <int RES>
__device__ __forceinline__ void fast_rung_rows(unsigned char *smem_raw, const CoopSmem &lay, unsigned char *wp, int lane, int n,
                                               int n_t, const double (&R)[9], const double (&t)[3], float tp2, float tp2sq3,
                                               float amax)
{
    using RS = Res<RES>;
    constexpr int ROW = RS::ROW;
    constexpr bool REG = RES == CLOSURE_REG_3D3D;
    const double *rows = reinterpret_cast<const double *>(smem_raw + 16);
    const int *pos = reinterpret_cast<const int *>(smem_raw + lay.pos);
    const float4 *af = reinterpret_cast<const float4 *>(smem_raw + lay.af);
    const float *rowsAf = reinterpret_cast<const float *>(wp + lay.rowsA);
    const float4 *rm32 = reinterpret_cast<const float4 *>(wp + lay.rm32);
    int2 *ridx = reinterpret_cast<int2 *>(wp + lay.ridx);
    float4 *qrow = reinterpret_cast<float4 *>(wp + lay.qrow);
    const double *RmS = reinterpret_cast<const double *>(wp + lay.RmS);
    float *qL = reinterpret_cast<float *>(wp + lay.qL);

    // fp32 data of one constraint: its set-up u* at R* and (Ex.2) a_i, beta_i^2 / (Ex.3) R_i, beta_i^2
    struct RowF { float us0, us1, us2; float4 r0, r1, r2; };
    auto load_row = [&](int i) -> RowF {
        RowF w;
        const int sp = pos[i] & 0x3fffffff;
        const float *S = rowsAf + (sp >> 1) * 8 + (sp & 1);
        w.us0 = S[0]; w.us1 = S[2]; w.us2 = S[4];
        if (REG) { w.r0 = af[i]; w.r1 = w.r0; w.r2 = w.r0; }
        else { w.r0 = af[3 * i]; w.r1 = af[3 * i + 1]; w.r2 = af[3 * i + 2]; }
        return w;
    };
    // key of that constraint at the rung whose fp32 rotation image is (m0, m1, m2); lipv = |(R_m - R*) a_i|^2 (Ex.2)
    auto key_of = [&](const RowF &w, const float4 &m0, const float4 &m1, const float4 &m2, float &lipv) -> float {
        if (REG) {
            const float4 a = w.r0;
            const float g0 = fmaf(m0.z, a.z, fmaf(m0.y, a.y, m0.x * a.x));
            const float g1 = fmaf(m1.z, a.z, fmaf(m1.y, a.y, m1.x * a.x));
            const float g2 = fmaf(m2.z, a.z, fmaf(m2.y, a.y, m2.x * a.x));
            lipv = fmaf(g2, g2, fmaf(g1, g1, g0 * g0));
            const float u0 = w.us0 - g0, u1 = w.us1 - g1, u2 = w.us2 - g2;
            return fmaf(u2, u2, fmaf(u1, u1, u0 * u0)) - a.w;
        } else {
            float f = fmaf(w.us2, w.us2, fmaf(w.us1, w.us1, w.us0 * w.us0)) - w.r0.w;
            float d;
            d = m0.x - w.r0.x; f = fmaf(d, d, f); d = m0.y - w.r0.y; f = fmaf(d, d, f); d = m0.z - w.r0.z; f = fmaf(d, d, f);
            d = m1.x - w.r1.x; f = fmaf(d, d, f); d = m1.y - w.r1.y; f = fmaf(d, d, f); d = m1.z - w.r1.z; f = fmaf(d, d, f);
            d = m2.x - w.r2.x; f = fmaf(d, d, f); d = m2.y - w.r2.y; f = fmaf(d, d, f); d = m2.z - w.r2.z; f = fmaf(d, d, f);
            lipv = 0.f;
            return f;
        }
    };

    if (n <= 16) {
        // lane = (rung parity, constraint): the lanes are not left idle by a loop over 8 - 16 constraints
        const int c = lane & 15;
        const bool has = c < n;
        const unsigned hm = 0xFFFFu << (lane & 16);
        const RowF w = load_row(has ? c : 0);
#pragma unroll 1
        for (int m = lane >> 4; m < n_t; m += 2) {
            const float4 m0 = rm32[3 * m], m1 = rm32[3 * m + 1], m2 = rm32[3 * m + 2];
            float lipv = 0.f;
            const float kv = key_of(w, m0, m1, m2, lipv);
            const uint32_t key = has ? ((fkey(kv) & ~15u) | (uint32_t)c) : (uint32_t)c;
            uint32_t k1, k2;
            float lm;
            group_top2_max(hm, 16, key, has ? lipv : 0.f, k1, k2, lm);
            if (key == k1) {
                ridx[m] = make_int2((int)(k1 & 15u), n > 1 ? (int)(k2 & 15u) : (int)(k1 & 15u));
                qL[m] = lm;
            }
        }
    } else {
        // lanes over the constraints; the first two rows of a lane stay in registers over the rungs (n <= 64 needs no more),
        // the two largest keys of a lane are kept as (key bits | constraint index) words: max / min, no branches
        const RowF wA = load_row(lane < n ? lane : 0), wB = load_row(lane + 32 < n ? lane + 32 : 0);
#pragma unroll 1
        for (int m = 0; m < n_t; ++m) {
            const float4 m0 = rm32[3 * m], m1 = rm32[3 * m + 1], m2 = rm32[3 * m + 2];
            uint32_t b1 = 0u, b2 = 0u;
            float lipl = 0.f;
            auto take = [&](float kv, float lipv, int i, bool on) {
                const uint32_t k = on ? ((fkey(kv) & ~0xFFFu) | (uint32_t)i) : 0u;      // n <= 4096: 12 index bits
                const uint32_t lo = min(k, b1);
                b1 = max(k, b1);
                b2 = max(b2, lo);
                lipl = fmaxf(lipl, on ? lipv : 0.f);
            };
            float lv;
            const float kA = key_of(wA, m0, m1, m2, lv);
            take(kA, lv, lane, lane < n);
            const float kB = key_of(wB, m0, m1, m2, lv);
            take(kB, lv, lane + 32, lane + 32 < n);
#pragma unroll 1
            for (int i = lane + 64; i < n; i += 32) {
                const RowF w = load_row(i);
                const float kv = key_of(w, m0, m1, m2, lv);
                take(kv, lv, i, true);
            }
            const uint32_t g1 = __reduce_max_sync(FULL, b1);
            const uint32_t g2 = __reduce_max_sync(FULL, b1 == g1 ? b2 : b1);    // (indices make the words distinct)
            const float lm = wmax_nonneg(lipl);
            if (lane == 0) { ridx[m] = make_int2((int)(g1 & 0xFFFu), (int)((n > 1 ? g2 : g1) & 0xFFFu)); qL[m] = lm; }
        }
    }
    __syncwarp();
    // the two chosen rows of rung m in fp64 with their error bounds, and the rung's Lipschitz bound: lane m
    for (int m = lane; m < n_t; m += 32) {
        double Rm[9];
#pragma unroll
        for (int e = 0; e < 9; ++e) Rm[e] = RmS[m * 9 + e];
        const int2 ii = ridx[m];
#pragma unroll
        for (int q = 0; q < 2; ++q) {
            const double *row = rows + (q ? ii.y : ii.x) * ROW;
            double u0, u1, u2, cc;
            affine_setup<RES>(Rm, t, row, u0, u1, u2, cc);
            float g0, g1, g2, fcb, eps;
            screen_row(u0, u1, u2, cc - row[RS::BETA + 1], tp2, tp2sq3, g0, g1, g2, fcb, eps);
            qrow[2 * m + q] = make_float4(g0, g1, g2, fcb - eps);
        }
        float lf;
        if (REG) {
            lf = sqrtf(qL[m]) * 1.000001f + 4.0e-6f * rm32[3 * m].w * amax;
        } else {
            double lip = 0.0;
#pragma unroll
            for (int e = 0; e < 9; ++e) { const double d = Rm[e] - R[e]; lip = fma(d, d, lip); }      // |R_m - R*|_F^2
            lf = (float)sqrt(lip);
        }
        qL[m] = lf * 1.001f + 1e-30f;
    }
}

// ---------------------------------------------------------------------------------- set-up after a move
// Everything that depends on the pose only (DESIGN.md 6.1b "state that only changes on an accepted
// move"): fp32 set-up rows at R* (rowsA), Exp(dT_m w) R* for every rung (RmS), per rung the two
// tightest rows (qrow) and the Lipschitz bound (qL).  fp64-heavy and rare, so it is kept out of line:
// its registers do not count against the per-iteration code.  Results epsA, rot_margin -> pose[16], pose[15].
template <int RES>
__device__ __noinline__ void coop_setup_on_move(unsigned char *smem_raw, int warp, int lane, int rows_bytes, int n,
                                                int n_t, int nq, int pairs, double t_p, float amax, bool stats)
{
    using RS = Res<RES>;
    constexpr int ROW = RS::ROW;
    constexpr bool FAST = RES == CLOSURE_REG_3D3D || RES == CLOSURE_POSE_REG;   // fp32 search for the screening rows (below)
    const CoopSmem lay = coop_layout(rows_bytes, n, n_t, nq, 1, pairs, kCoopWarps, af_width<RES>(), af_extra<RES>(pairs));
    const double *rows = reinterpret_cast<const double *>(smem_raw + 16);
    const int *pos = reinterpret_cast<const int *>(smem_raw + lay.pos);
    unsigned char *wp = smem_raw + lay.warp0 + (size_t)warp * lay.per_warp;
    float4 *rowsA = reinterpret_cast<float4 *>(wp + lay.rowsA);
    const double2 *ab = reinterpret_cast<const double2 *>(wp + lay.ab);
    float4 *qrow = reinterpret_cast<float4 *>(wp + lay.qrow);
    double *RmS = reinterpret_cast<double *>(wp + lay.RmS);
    float *qL = reinterpret_cast<float *>(wp + lay.qL);
    double *pose = reinterpret_cast<double *>(wp + lay.pose);
    unsigned long long *stc = reinterpret_cast<unsigned long long *>(wp + lay.stc);
    const float tpf = (float)t_p * 1.0000002f;          // >= t_p
    const float tp2 = 2.0f * tpf, tp2sq3 = 3.0f * tpf * tpf;
    const float4 *QL = reinterpret_cast<const float4 *>(smem_raw + lay.af);   // ellipsoid: (Q00 Q01 Q02 Q11) (Q12 Q22 qmag .) per constraint
    int2 *ridx = reinterpret_cast<int2 *>(wp + lay.ridx);                      // ellipsoid: constraints of each rung's screening rows
    double R[9], t[3], vel[3];
#pragma unroll
    for (int e = 0; e < 9; ++e) R[e] = pose[e];
#pragma unroll
    for (int e = 0; e < 3; ++e) { t[e] = pose[9 + e]; vel[e] = pose[12 + e]; }
    float eps_l = 0.f;
    double rm_l = CUDART_INF;
#pragma unroll 1
    for (int i = lane; i < n; i += 32) {
        const double *row = rows + i * ROW;
        double u0, u1, u2, c;
        pair_setup<RES>(R, t, row, u0, u1, u2, c);
        float f0, f1, f2, fc, eps;
        screen_row_any<RES>(u0, u1, u2, c, tp2, tp2sq3, RES == kEll ? QL[2 * i + 1].z : 0.f, f0, f1, f2, fc, eps);
        {
            const int pp = pos[i], p = pp & 0x3fffffff;
            float *A = reinterpret_cast<float *>(rowsA) + (p >> 1) * 8 + (p & 1);
            A[0] = f0; A[2] = f1; A[4] = f2; A[6] = fc;
            if (pp & 0x40000000) { A[1] = f0; A[3] = f1; A[5] = f2; A[7] = fc; }
        }
        eps_l = fmaxf(eps_l, eps);
        if (RES == CLOSURE_POSE_REG_SPLIT) rm_l = dmin(rm_l, row[12] - sqrt(frob_sq(R, row)));
    }
    const float epsA = wmax_nonneg(eps_l);
    double rot_margin = CUDART_INF;
    if (RES == CLOSURE_POSE_REG_SPLIT) rot_margin = wmin_f64(rm_l);
    for (int m = lane; m < n_t; m += 32) {       // Exp(dT_m w) R* for every rung
        const double2 c2 = ab[m];
        double Rm[9];
        rotate_left(R, vel[0], vel[1], vel[2], c2.x, c2.y, Rm);
#pragma unroll
        for (int e = 0; e < 9; ++e) RmS[m * 9 + e] = Rm[e];
        if (FAST) {                                  // fp32 image for the search: R_m - R* (Ex.2), R_m (Ex.3)
            float v[9], fro = 0.f;
#pragma unroll
            for (int e = 0; e < 9; ++e) {
                v[e] = (float)(RES == CLOSURE_REG_3D3D ? Rm[e] - R[e] : Rm[e]);
                fro = fmaf(v[e], v[e], fro);
            }
            float4 *rm32 = reinterpret_cast<float4 *>(wp + lay.rm32);
            rm32[3 * m] = make_float4(v[0], v[1], v[2], sqrtf(fro));
            rm32[3 * m + 1] = make_float4(v[3], v[4], v[5], 0.f);
            rm32[3 * m + 2] = make_float4(v[6], v[7], v[8], 0.f);
        }
    }
    __syncwarp();
    if (FAST) {
        fast_rung_rows<RES>(smem_raw, lay, wp, lane, n, n_t, R, t, tp2, tp2sq3, amax);
        if (stats) { stc[2] += n; stc[3] += 2ull * n_t; }
    } else {
    // the two tightest constraints of every rung (largest c - beta^2 at the unperturbed
    // translation): the rows the ladder screens each rung against while the pose stays here
    if (n <= 16) {
        // short tables (Ex.1 / Ex.3 sizes): lane = (rung, constraint), two rungs per pass, so that the lanes are not
        // left idle by a loop over 8 - 16 constraints; same rows, same bounds as the loop below
        const int c = lane & 15;
        const bool has = c < n;
        const double *row = rows + (has ? c : 0) * ROW;
        const unsigned hm = 0xFFFFu << (lane & 16);
#pragma unroll 1
        for (int m = lane >> 4; m < n_t; m += 2) {
            double Rm[9], dR[9], lip = 0.0;
#pragma unroll
            for (int e = 0; e < 9; ++e) { Rm[e] = RmS[m * 9 + e]; dR[e] = Rm[e] - R[e]; }
            double u0, u1, u2, cc;
            pair_setup<RES>(Rm, t, row, u0, u1, u2, cc);
            if (RES == CLOSURE_REG_3D3D || RES == kEll) {           // ||(R_m - R*) a_i||^2
                const double q0 = dR[0] * row[0] + dR[1] * row[1] + dR[2] * row[2];
                const double q1 = dR[3] * row[0] + dR[4] * row[1] + dR[5] * row[2];
                const double q2 = dR[6] * row[0] + dR[7] * row[1] + dR[8] * row[2];
                lip = q0 * q0 + q1 * q1 + q2 * q2;
                if (RES == kEll) lip *= ell_lip_scale(row);          // ... in the norm of Lambda_i: |x|_L^2 <= |Lambda|_F |x|^2
            } else {
#pragma unroll
                for (int e = 0; e < 9; ++e) lip = fma(dR[e], dR[e], lip);      // ||R_m - R*||_F^2
            }
            bool rdead = false;
            if (RES == CLOSURE_POSE_REG_SPLIT) rdead = has && !(frob_sq(Rm, row) <= row[13]);
            float g0, g1, g2, fcb, eps;
            screen_row_any<RES>(u0, u1, u2, cc - row[RS::BETA + 1], tp2, tp2sq3, RES == kEll ? QL[2 * (has ? c : 0) + 1].z : 0.f,
                                g0, g1, g2, fcb, eps);
            float4 r4 = make_float4(g0, g1, g2, has ? fcb - eps : -CUDART_INF_F);
            const uint32_t key = has ? ((fkey(r4.w) & ~15u) | (uint32_t)c) : (uint32_t)c;
            uint32_t m1, m2;
            float lf;
            group_top2_max(hm, 16, key, has ? (float)sqrt(lip) : 0.f, m1, m2, lf);
            const uint32_t key2 = (key == m1) ? 0u : key;
            const bool dead_any = (__ballot_sync(hm, rdead) & hm) != 0u;
            if (key == m1) {
                if (dead_any) r4.w = CUDART_INF_F;                     // rung dead for every candidate
                qrow[2 * m] = r4;
                qL[m] = lf * 1.001f + 1e-30f;
                if (n == 1) qrow[2 * m + 1] = r4;
                if (RES == kEll) { ridx[m].x = c; if (n == 1) ridx[m].y = c; }
            }
            if (key2 == m2 && n > 1) { qrow[2 * m + 1] = r4; if (RES == kEll) ridx[m].y = c; }
        }
    } else {
#pragma unroll 1
    for (int m = 0; m < n_t; ++m) {
        double Rm[9];
#pragma unroll
        for (int e = 0; e < 9; ++e) Rm[e] = RmS[m * 9 + e];
        float4 b1 = make_float4(0.f, 0.f, 0.f, -CUDART_INF_F), b2 = b1;
        int jb1 = 0, jb2 = 0;                        // their constraints (the ellipsoid's screening needs the quadratic part)
        bool rdead = false;
        double dR[9], lip = 0.0;                     // max_i | ||g_i(R_m, .)|| - ||g_i(R*, .)|| | <= sqrt(lip)
#pragma unroll
        for (int e = 0; e < 9; ++e) dR[e] = Rm[e] - R[e];
        if (RES != CLOSURE_REG_3D3D && RES != kEll) {
#pragma unroll
            for (int e = 0; e < 9; ++e) lip = fma(dR[e], dR[e], lip);      // ||R_m - R*||_F^2
        }
#pragma unroll 1
        for (int i = lane; i < n; i += 32) {
            const double *row = rows + i * ROW;
            double u0, u1, u2, c;
            pair_setup<RES>(Rm, t, row, u0, u1, u2, c);
            if (RES == CLOSURE_REG_3D3D || RES == kEll) {           // ||(R_m - R*) a_i||^2
                const double q0 = dR[0] * row[0] + dR[1] * row[1] + dR[2] * row[2];
                const double q1 = dR[3] * row[0] + dR[4] * row[1] + dR[5] * row[2];
                const double q2 = dR[6] * row[0] + dR[7] * row[1] + dR[8] * row[2];
                lip = dmax(lip, (q0 * q0 + q1 * q1 + q2 * q2) * (RES == kEll ? ell_lip_scale(row) : 1.0));
            }
            if (RES == CLOSURE_POSE_REG_SPLIT) {
                if (!(frob_sq(Rm, row) <= row[13])) rdead = true;
            }
            float g0, g1, g2, fcb, eps;
            screen_row_any<RES>(u0, u1, u2, c - row[RS::BETA + 1], tp2, tp2sq3, RES == kEll ? QL[2 * i + 1].z : 0.f, g0, g1, g2, fcb, eps);
            const float4 r4 = make_float4(g0, g1, g2, fcb - eps);
            if (r4.w > b1.w) { b2 = b1; jb2 = jb1; b1 = r4; jb1 = i; } else if (r4.w > b2.w) { b2 = r4; jb2 = i; }
        }
        const uint32_t k1 = fkey(b1.w);
        const uint32_t m1 = __reduce_max_sync(FULL, k1);
        const int src1 = __ffs(__ballot_sync(FULL, k1 == m1)) - 1;
        const uint32_t k2 = (lane == src1) ? fkey(b2.w) : k1;
        const uint32_t m2 = __reduce_max_sync(FULL, k2);
        const int src2 = __ffs(__ballot_sync(FULL, k2 == m2)) - 1;
        if (__any_sync(FULL, rdead)) b1.w = CUDART_INF_F;          // rung dead for every candidate
        if (lane == src1) qrow[2 * m] = b1;
        if (lane == src2) qrow[2 * m + 1] = (lane == src1) ? b2 : b1;
        if (RES == kEll) {
            const int i1 = __shfl_sync(FULL, jb1, src1);
            const int i2 = __shfl_sync(FULL, src2 == src1 ? jb2 : jb1, src2);
            if (lane == 0) ridx[m] = make_int2(i1, i2);
        }
        const float lf = wmax_nonneg((float)sqrt(lip));
        if (lane == 0) qL[m] = lf * 1.001f + 1e-30f;
    }
    }
    if (stats) { stc[2] += n; stc[3] += (unsigned long long)n * n_t; }
    }
    __syncwarp();
    if (lane == 0) {                                 // suffix maximum: qL[m] holds for every rung >= m
        float sm = 0.f;
        for (int m = n_t - 1; m >= 0; --m) { sm = fmaxf(sm, qL[m]); qL[m] = sm; }
    }
    __syncwarp();
    if (lane == 0) { pose[15] = rot_margin; pose[16] = (double)epsA; }
    __syncwarp();
}

// ---------------------------------------------------------------------------------- the kernel
template <int RES, int NQ>
__global__ void __launch_bounds__(kCoopThreads, coop_min_ctas<RES, NQ>()) walker_dense_kernel(const __grid_constant__ WalkLaunch L)
{
    using RS = Res<RES>;
    constexpr int ROW = RS::ROW;
    constexpr int NPK = NQ / 2;            // packed pairs of perturbations
    constexpr bool ODD = (NQ & 1) != 0;    // plus one scalar slot

    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ int n_runs_s;
    __shared__ float amax_s;
    const int warp = threadIdx.x >> 5;
    int lane = threadIdx.x & 31;
    const InstanceDesc *__restrict__ D = L.desc[blockIdx.y];
    const int n = D->n;
    const int rows_bytes = D->rows_bytes;
    int n_p = L.n_p, n_ps = L.n_p_star, n_t = L.n_t;
    // Values the iteration uses all the time are made opaque to the compiler: under register pressure it otherwise
    // re-derives them from special registers and the constant bank inside the loop instead of keeping them in a register.
#define CLOSURE_PIN_R(x) asm volatile("" : "+r"(x))
#define CLOSURE_PIN_F(x) asm volatile("" : "+f"(x))
    CLOSURE_PIN_R(lane); CLOSURE_PIN_R(n_p); CLOSURE_PIN_R(n_ps); CLOSURE_PIN_R(n_t);
    uint64_t *bar = reinterpret_cast<uint64_t *>(smem_raw);
    double *rows = reinterpret_cast<double *>(smem_raw + 16);
    stage_rows(smem_raw + 16, bar, D->rows, rows_bytes);                        // a0 (TMA bulk copy)
    const CoopSmem lay = coop_layout(rows_bytes, n, n_t, NQ, 1, L.pairs_cap, kCoopWarps, af_width<RES>(), af_extra<RES>(L.pairs_cap));
    int *run_end = reinterpret_cast<int *>(smem_raw + lay.run_end);
    float *run_bf = reinterpret_cast<float *>(smem_raw + lay.run_bf);
    int *run_pend = reinterpret_cast<int *>(smem_raw + lay.run_pend);   // end of run r in rowsA, in PAIRS of rows
    int *pos = reinterpret_cast<int *>(smem_raw + lay.pos);             // row of constraint i in rowsA (bit 30: write it twice)
    if (warp == 0) {                                   // runs of equal bounds (rows are sorted by bound)
        int cnt = 0;
        for (int base = 0; base < n; base += 32) {
            const int i = base + lane;
            bool end = false;
            double beta = 0.0;
            if (i < n) {
                beta = rows[i * ROW + RS::BETA];
                end = (i == n - 1) || (rows[(i + 1) * ROW + RS::BETA] != beta);
            }
            const unsigned m = __ballot_sync(FULL, end);
            if (end) {
                const int r = cnt + __popc(m & ((1u << lane) - 1u));
                run_end[r] = i;
                run_bf[r] = (float)beta;
            }
            cnt += __popc(m);
        }
        __syncwarp();
        if (lane == 0) {
            // rowsA holds the fp32 set-ups two constraints per entry; a run of odd length repeats its last
            // constraint (a maximum does not see duplicates), so no pair straddles two bounds
            n_runs_s = cnt;
            int p = 0, start = 0, longest = 0;
            for (int r = 0; r < cnt; ++r) {
                const int end = run_end[r];
                const int p_begin = p >> 1;
                for (int i = start; i <= end; ++i) pos[i] = p++;
                if (p & 1) { pos[end] |= 0x40000000; ++p; }
                run_pend[r] = p >> 1;
                longest = max(longest, (p >> 1) - p_begin);
                start = end + 1;
            }
        }
    }
    if (RES == CLOSURE_REG_3D3D || RES == CLOSURE_POSE_REG) {
        // fp32 image of the constraints for the set-up's search (fast_rung_rows), and max_i |a_i| for its Lipschitz slack
        float4 *af = reinterpret_cast<float4 *>(smem_raw + lay.af);
        float am = 0.f;
        for (int i = threadIdx.x; i < n; i += kCoopThreads) {
            const double *row = rows + i * ROW;
            const float b2 = (float)row[RS::BETA + 1];
            if (RES == CLOSURE_REG_3D3D) {
                af[i] = make_float4((float)row[0], (float)row[1], (float)row[2], b2);
                am = fmaxf(am, (float)sqrt(row[0] * row[0] + row[1] * row[1] + row[2] * row[2]) * 1.000001f);
            } else {
                af[3 * i] = make_float4((float)row[0], (float)row[1], (float)row[2], b2);
                af[3 * i + 1] = make_float4((float)row[3], (float)row[4], (float)row[5], 0.f);
                af[3 * i + 2] = make_float4((float)row[6], (float)row[7], (float)row[8], 0.f);
            }
        }
        if (RES == CLOSURE_REG_3D3D) {
            if (threadIdx.x == 0) amax_s = 0.f;
            __syncthreads();
            atomicMax(reinterpret_cast<unsigned int *>(&amax_s), __float_as_uint(wmax_nonneg(am)));   // non-negative floats order as uints
        }
    }
    __syncthreads();
    const int n_runs = n_runs_s;
    if (RES == kEll) {
        float4 *QLw = reinterpret_cast<float4 *>(smem_raw + lay.af);
        float *QAw = reinterpret_cast<float *>(QLw + 2 * n);
        const float tpq = (float)L.t_p * 1.0000002f;
        for (int i = threadIdx.x; i < n; i += kCoopThreads) {
            const double *row = rows + i * ROW;
            const float q00 = (float)(0.25 * row[8]), q01 = (float)(0.5 * row[9]), q02 = (float)(0.5 * row[10]);
            const float q11 = (float)(0.25 * row[11]), q12 = (float)(0.5 * row[12]), q22 = (float)(0.25 * row[13]);
            const float qsum = (fabsf(q00) + fabsf(q01) + fabsf(q02) + fabsf(q11) + fabsf(q12) + fabsf(q22)) * 1.000001f;
            QLw[2 * i] = make_float4(q00, q01, q02, q11);
            QLw[2 * i + 1] = make_float4(q12, q22, 4.0f * tpq * tpq * qsum, 0.f);     // qmag = (2 t_p)^2 sum|Q|
            const int pp = pos[i], p = pp & 0x3fffffff;
            float *A = QAw + (p >> 1) * 12 + (p & 1);           // (Q00a Q00b Q01a Q01b) (Q02a Q02b Q11a Q11b) (Q12a Q12b Q22a Q22b)
            A[0] = q00; A[2] = q01; A[4] = q02; A[6] = q11; A[8] = q12; A[10] = q22;
            if (pp & 0x40000000) { A[1] = q00; A[3] = q01; A[5] = q02; A[7] = q11; A[9] = q12; A[11] = q22; }
        }
        __syncthreads();
    }

    const long long local = (long long)blockIdx.x * kCoopWarps + warp;
    if (local >= L.num_walkers) return;                // no block-wide barrier below this line
    unsigned char *wp = smem_raw + lay.warp0 + (size_t)warp * lay.per_warp;
    float4 *rowsA = reinterpret_cast<float4 *>(wp + lay.rowsA);
    float4 *rowsL = reinterpret_cast<float4 *>(wp + lay.rowsL);
    float4 *pert = reinterpret_cast<float4 *>(wp + lay.pert);
    double2 *ab = reinterpret_cast<double2 *>(wp + lay.ab);
    float4 *qrow = reinterpret_cast<float4 *>(wp + lay.qrow);     // [rung][2]: the two tightest rows of each rung
    double *RmS = reinterpret_cast<double *>(wp + lay.RmS);
    double *dex = reinterpret_cast<double *>(wp + lay.dex);      // fp64 fallback: exact d_j, [q][lane]
    float *qL = reinterpret_cast<float *>(wp + lay.qL);           // [rung]: bound on the change of any residual norm
    float4 *cand4 = reinterpret_cast<float4 *>(wp + lay.cand4);   // the kept perturbations (-2 d_j, -|d_j|^2), by rank
    int *candj = reinterpret_cast<int *>(wp + lay.candj);
    float *candd = reinterpret_cast<float *>(wp + lay.candd);     // upper bounds of the candidates' eq. (14) values
    double *pose = reinterpret_cast<double *>(wp + lay.pose);     // R*(9) t*(3) omega(3): fp64, touched only on moves / fp64 paths
    // ellipsoid norm: quadratic-form coefficients of the constraints, by constraint (QL) and by pair-entry of rowsA (QA)
    const float4 *QL = reinterpret_cast<const float4 *>(smem_raw + lay.af);
    const float4 *QA = QL + 2 * n;
    const int2 *ridx = reinterpret_cast<const int2 *>(wp + lay.ridx);

    const unsigned long long w = (unsigned long long)(L.walker_begin + local);
    const unsigned long long seed = L.seed[blockIdx.y];
    Rng rng;
    rng.w_lo = (uint32_t)w;
    rng.w_hi8 = (uint32_t)(w >> 32) << 8;
    rng.k0 = (uint32_t)seed;
    rng.k1 = (uint32_t)(seed >> 32);

    // ---- a1: walker init, replicated on the lanes (Alg. 2 l.8-9)
    {
        double R[9], t[3], vel[3];
        init_walker<CLOSURE_MODE_ROT>(D, L, rng, w, R, t, vel);
        for (int m = lane; m < n_t; m += 32) {         // ladder dT_m = gamma^(m-1) by repeated multiplication
            double dT = 1.0;
            for (int q = 0; q < m; ++q) dT = dT * L.gamma;
            const double p0 = dT * vel[0], p1 = dT * vel[1], p2 = dT * vel[2];
            double A, B;
            exp_coeffs(fma(p2, p2, fma(p1, p1, p0 * p0)), A, B);
            ab[m] = make_double2(A * dT, B * dT * dT);
        }
        if (lane == 0) {
#pragma unroll
            for (int e = 0; e < 9; ++e) pose[e] = R[e];
#pragma unroll
            for (int e = 0; e < 3; ++e) { pose[9 + e] = t[e]; pose[12 + e] = vel[e]; }
        }
    }
    __syncwarp();

    const double t_p = L.t_p;
    const float tpf = (float)t_p * 1.0000002f;          // >= t_p
    float tp2 = 2.0f * tpf, tp2sq3 = 3.0f * tpf * tpf;
    float m2tp = -2.0f * (float)t_p;
    CLOSURE_PIN_F(tp2); CLOSURE_PIN_F(tp2sq3); CLOSURE_PIN_F(m2tp);
    const int KP = n_ps;                                // ladder candidates
    const int NCH = 32 / KP;                            // constraint chunks of the full evaluation
    const int ek = lane % KP, ech = lane / KP;
    const bool e_act = ech < NCH;

    // executed-work counters (closure_get_stats): in shared memory, touched by lane 0 and only when asked for
    unsigned long long *stc = reinterpret_cast<unsigned long long *>(wp + lay.stc);
    const bool stats = (L.stats != nullptr) && lane == 0;
    if (stats) {
        for (int k = 0; k < kNumStats; ++k) stc[k] = 0ull;
    }
    const long long clk_begin = stats ? clock64() : 0ll;
    bool hit = false;
    bool moved = true;
    float epsA = 0.f;
    double rot_margin = CUDART_INF;
    // cached across iterations while the pose does not move
    int full_m = -1;                                    // rung whose rows sit in rowsL
    float epsL = 0.f;
    bool rdeadL = false;

    for (int s = 1; s <= L.num_steps; ++s) {
        // ================================================== set-up at the current pose (only after a move)
        if (moved) {
            const long long c0 = stats ? clock64() : 0ll;
            coop_setup_on_move<RES>(smem_raw, warp, lane, rows_bytes, n, n_t, NQ, L.pairs_cap, t_p, amax_s, stats);
            if (stats) stc[10] += (unsigned long long)(clock64() - c0);
            epsA = (float)pose[16];
            rot_margin = pose[15];
            full_m = -1;
        }

        // ================================================== a2: perturbations of this lane
        unsigned long long p0[NPK > 0 ? NPK : 1], p1[NPK > 0 ? NPK : 1], p2[NPK > 0 ? NPK : 1];
        float o0 = 0.f, o1 = 0.f, o2 = 0.f;                  // the odd slot NQ-1
        float dd[NQ];
        {
            int jv[NQ];
            uint32_t x[NQ], y[NQ], z[NQ];
#pragma unroll
            for (int q = 0; q < NQ; ++q) jv[q] = lane + 32 * q;
            philox_batch<NQ>(rng, (uint32_t)s, jv, x, y, z);
            float e0[NQ], e1[NQ], e2[NQ];
            // packed slots are produced by packed instructions so that they live in aligned register pairs
            // (same roundings as the scalar pm1f() * m2tp)
            const unsigned long long C1 = pk2(4.656612873077392578125e-10f, 4.656612873077392578125e-10f);
            const unsigned long long C2 = pk2(2.3283064365386962890625e-10f - 1.0f, 2.3283064365386962890625e-10f - 1.0f);
            const unsigned long long M2 = pk2(m2tp, m2tp);
#pragma unroll
            for (int k = 0; k < NPK; ++k) {
                p0[k] = mul2(M2, fma2(pk2((float)x[2 * k], (float)x[2 * k + 1]), C1, C2));
                p1[k] = mul2(M2, fma2(pk2((float)y[2 * k], (float)y[2 * k + 1]), C1, C2));
                p2[k] = mul2(M2, fma2(pk2((float)z[2 * k], (float)z[2 * k + 1]), C1, C2));
                upk2(p0[k], e0[2 * k], e0[2 * k + 1]);
                upk2(p1[k], e1[2 * k], e1[2 * k + 1]);
                upk2(p2[k], e2[2 * k], e2[2 * k + 1]);
            }
            if (ODD) { e0[NQ - 1] = m2tp * pm1f(x[NQ - 1]); e1[NQ - 1] = m2tp * pm1f(y[NQ - 1]); e2[NQ - 1] = m2tp * pm1f(z[NQ - 1]); }
#pragma unroll
            for (int q = 0; q < NQ; ++q) {
                // (ellipsoid: the pair carries its own quadratic form d^T Lambda_i d, nothing is added per run and thresholds are 0)
                dd[q] = RES == kEll ? 0.f : 0.25f * fmaf(e2[q], e2[q], fmaf(e1[q], e1[q], e0[q] * e0[q]));
                pert[32 * q + lane] = make_float4(e0[q], e1[q], e2[q], -dd[q]);
            }
            if (ODD) { o0 = e0[NQ - 1]; o1 = e1[NQ - 1]; o2 = e2[NQ - 1]; }
        }

        // ================================================== a3: eq. (14) in fp32 with error bound
        float dt[NQ];
        float unc_l = 0.f;
        {
#pragma unroll
            for (int q = 0; q < NQ; ++q) dt[q] = CUDART_INF_F;
            const float E0 = epsA + tp2sq3 * kMu19;          // bound on |a32 - a64| up to its own rounding
            int pp = 0;
            for (int r = 0; r < n_runs; ++r) {
                const int pend = run_pend[r];
                const float bf = run_bf[r];
                float mx[NQ];
#pragma unroll
                for (int q = 0; q < NQ; ++q) mx[q] = -CUDART_INF_F;
#pragma unroll(NQ <= 2 ? 4 : 1)   // measured: unrolling the NQ = 5 body further costs 2-4 % (C2, C4)
                for (; pp < pend; ++pp) {
                    // two constraints a, b per entry: X = (f0a f0b f1a f1b), Y = (f2a f2b fca fcb)
                    const float4 X = rowsA[2 * pp], Y = rowsA[2 * pp + 1];
                    if (RES == kEll) {
                        // (w, c) as above plus the quadratic form: U = (Q00a Q00b Q01a Q01b) V = (Q02a Q02b Q11a Q11b) W = (Q12a Q12b Q22a Q22b)
                        const float4 U = QA[3 * pp], V = QA[3 * pp + 1], W = QA[3 * pp + 2];
#pragma unroll
                        for (int k = 0; k < NPK; ++k) {
                            const unsigned long long ta0 = fma2(pk2(V.x, V.x), p2[k], fma2(pk2(U.z, U.z), p1[k], fma2(pk2(U.x, U.x), p0[k], pk2(X.x, X.x))));
                            const unsigned long long ta1 = fma2(pk2(W.x, W.x), p2[k], fma2(pk2(V.z, V.z), p1[k], pk2(X.z, X.z)));
                            const unsigned long long ta2 = fma2(pk2(W.z, W.z), p2[k], pk2(Y.x, Y.x));
                            const unsigned long long va = fma2(ta0, p0[k], fma2(ta1, p1[k], fma2(ta2, p2[k], pk2(Y.z, Y.z))));
                            const unsigned long long tb0 = fma2(pk2(V.y, V.y), p2[k], fma2(pk2(U.w, U.w), p1[k], fma2(pk2(U.y, U.y), p0[k], pk2(X.y, X.y))));
                            const unsigned long long tb1 = fma2(pk2(W.y, W.y), p2[k], fma2(pk2(V.w, V.w), p1[k], pk2(X.w, X.w)));
                            const unsigned long long tb2 = fma2(pk2(W.w, W.w), p2[k], pk2(Y.y, Y.y));
                            const unsigned long long vb = fma2(tb0, p0[k], fma2(tb1, p1[k], fma2(tb2, p2[k], pk2(Y.w, Y.w))));
                            float la, ha, lb, hb;
                            upk2(va, la, ha);
                            upk2(vb, lb, hb);
                            mx[2 * k] = fmaxf(mx[2 * k], fmaxf(la, lb));
                            mx[2 * k + 1] = fmaxf(mx[2 * k + 1], fmaxf(ha, hb));
                        }
                        if (ODD) {                      // the odd slot takes both constraints in one packed chain
                            const unsigned long long E0o = pk2(o0, o0), E1o = pk2(o1, o1), E2o = pk2(o2, o2);
                            const unsigned long long t0 = fma2(pk2(V.x, V.y), E2o, fma2(pk2(U.z, U.w), E1o, fma2(pk2(U.x, U.y), E0o, pk2(X.x, X.y))));
                            const unsigned long long t1 = fma2(pk2(W.x, W.y), E2o, fma2(pk2(V.z, V.w), E1o, pk2(X.z, X.w)));
                            const unsigned long long t2 = fma2(pk2(W.z, W.w), E2o, pk2(Y.x, Y.y));
                            const unsigned long long vo = fma2(t0, E0o, fma2(t1, E1o, fma2(t2, E2o, pk2(Y.z, Y.w))));
                            float lo, hi;
                            upk2(vo, lo, hi);
                            mx[NQ - 1] = fmaxf(mx[NQ - 1], fmaxf(lo, hi));
                        }
                        continue;
                    }
#pragma unroll
                    for (int k = 0; k < NPK; ++k) {
                        const unsigned long long va =
                            fma2(pk2(X.x, X.x), p0[k], fma2(pk2(X.z, X.z), p1[k], fma2(pk2(Y.x, Y.x), p2[k], pk2(Y.z, Y.z))));
                        const unsigned long long vb =
                            fma2(pk2(X.y, X.y), p0[k], fma2(pk2(X.w, X.w), p1[k], fma2(pk2(Y.y, Y.y), p2[k], pk2(Y.w, Y.w))));
                        float la, ha, lb, hb;
                        upk2(va, la, ha);
                        upk2(vb, lb, hb);
                        mx[2 * k] = fmaxf(mx[2 * k], fmaxf(la, lb));
                        mx[2 * k + 1] = fmaxf(mx[2 * k + 1], fmaxf(ha, hb));
                    }
                    if (ODD) {                          // the odd slot takes both constraints in one packed chain
                        const unsigned long long vo = fma2(pk2(X.x, X.y), pk2(o0, o0),
                                                           fma2(pk2(X.z, X.w), pk2(o1, o1),
                                                                fma2(pk2(Y.x, Y.y), pk2(o2, o2), pk2(Y.z, Y.w))));
                        float lo, hi;
                        upk2(vo, lo, hi);
                        mx[NQ - 1] = fmaxf(mx[NQ - 1], fmaxf(lo, hi));
                    }
                }
#pragma unroll
                for (int q = 0; q < NQ; ++q) {
                    // a ~ max_i |u_i - d|^2 within E0 + 2^-22 a;  sq ~ sqrt(a) within 2^-21 relative
                    const float a = fmaxf(mx[q] + dd[q], 1e-30f);
                    const float rr = rsqrt_normal(a);
                    const float sq = a * rr;
                    const float du = 1.01f * fmaf(E0, rr, (bf + sq) * kMu19);
                    unc_l = fmaxf(unc_l, du);
                    dt[q] = fminf(dt[q], bf - sq);
                }
            }
            if (stats) stc[6] += (unsigned long long)n * n_p;
        }

        // ================================================== a4: top-N_P* with certified ranking
        const float rmf = (float)rot_margin;                // +inf unless POSE_REG_SPLIT
        float dv[NQ];
#pragma unroll
        for (int q = 0; q < NQ; ++q) dv[q] = (lane + 32 * q < n_p) ? fminf(dt[q], rmf) : -CUDART_INF_F;
        float unc = wmax_nonneg(unc_l), myval;
        if (RES == CLOSURE_POSE_REG_SPLIT) unc += 1.2e-7f * fabsf(rmf);
        // (exact_only & 4: debug, every step takes the fp64 fall-back; & 16: on all N_P perturbations)
        if (!topk_certified<NQ>(dv, n_ps, unc, (L.exact_only & 4) != 0, (L.exact_only & 32) != 0, lane, candj, candd, myval)) {
            double R[9], t[3];
#pragma unroll
            for (int e = 0; e < 9; ++e) R[e] = pose[e];
#pragma unroll
            for (int e = 0; e < 3; ++e) t[e] = pose[9 + e];
            const ExactMargin<RES> exact{ R, t, rows, n, rng, (uint32_t)s, t_p, rot_margin };
            const int cnt = topk_fp64<NQ>(dv, n_p, n_ps, unc, myval, (L.exact_only & 16) != 0, lane, dex, candj, candd, exact);
            if (stats) { stc[8] += 1; stc[0] += (unsigned long long)n * cnt; }
        }
        __syncwarp();                                       // pert[], candj[] visible to all lanes
        if (lane < n_ps) cand4[lane] = pert[candj[lane]];
        __syncwarp();

        // ================================================== a5-a6: ladder, first feasible rung
        int m0 = 0;
        unsigned win = 0u;
        bool lip_stop = false;
        const int khalf = (KP + 1) >> 1;
        for (int mb = 0; mb < n_t && m0 == 0 && !lip_stop; mb += 16) {
            // ---- screening of 16 rungs, lane = (rung, half of the candidates): a candidate is dead for sure
            // at rung m if one of the two tightest rows is violated beyond its error bound, or if its margin
            // at R* is more negative than the rotation to R_m (or any smaller one: qL is a suffix maximum)
            // can repair
            const int mq = mb + (lane & 15), hq = lane >> 4;
            const bool q_act = mq < n_t;
            unsigned alive = 0u;
            float Lm = CUDART_INF_F;
            if (q_act) {
                const float4 r0 = qrow[2 * mq], r1 = qrow[2 * mq + 1];
                Lm = qL[mq];
                const int k1 = min(KP, (hq + 1) * khalf);
                if (RES == kEll) {
                    const int2 ii = ridx[mq];
                    const float4 A0 = QL[2 * ii.x], B0 = QL[2 * ii.x + 1], A1 = QL[2 * ii.y], B1 = QL[2 * ii.y + 1];
                    for (int k = hq * khalf; k < k1; ++k) {
                        const float4 c4 = cand4[k];
                        const float v0 = ell_value(r0, A0, B0, c4), v1 = ell_value(r1, A1, B1, c4);
                        if (!(v0 > c4.w) && !(v1 > c4.w) && !(candd[k] + Lm < 0.f)) alive |= 1u << k;
                    }
                } else {
                for (int k = hq * khalf; k < k1; ++k) {
                    const float4 c4 = cand4[k];
                    const float v0 = fmaf(r0.x, c4.x, fmaf(r0.y, c4.y, fmaf(r0.z, c4.z, r0.w)));
                    const float v1 = fmaf(r1.x, c4.x, fmaf(r1.y, c4.y, fmaf(r1.z, c4.z, r1.w)));
                    if (!(v0 > c4.w) && !(v1 > c4.w) && !(candd[k] + Lm < 0.f)) alive |= 1u << k;
                }
                }
            }
            alive |= __shfl_xor_sync(FULL, alive, 16);
            if (L.exact_only & 2) alive = q_act ? ((KP >= 32) ? FULL : ((1u << KP) - 1u)) : 0u;   // debug: nothing is screened out
            if (mb + 16 < n_t && !(L.exact_only & 2)) {
                // no candidate can be repaired at the last rung of this block => none at any later rung
                float cdm = candd[0];
                for (int k = 1; k < KP; ++k) cdm = fmaxf(cdm, candd[k]);
                if (cdm + qL[mb + 15] < 0.f) lip_stop = true;
            }
            unsigned qmask = __ballot_sync(FULL, lane < 16 && alive != 0u);
            if (stats) stc[7] += (unsigned long long)(min(n_t, mb + 16) - mb) * 2 * KP;

            // ---- full evaluation of the surviving rungs, in order
            while (qmask != 0u && m0 == 0) {
                const int l0 = __ffs(qmask) - 1;
                qmask &= qmask - 1u;
                const int m1 = mb + l0;
                const unsigned cand_alive = __shfl_sync(FULL, alive, l0);
                double Rm[9], t[3];
#pragma unroll
                for (int e = 0; e < 9; ++e) Rm[e] = RmS[m1 * 9 + e];
#pragma unroll
                for (int e = 0; e < 3; ++e) t[e] = pose[9 + e];
                if (full_m != m1) {
                    __syncwarp();                            // earlier readers of rowsL are done
                    float eps_l = 0.f;
                    bool rdead = false;
#pragma unroll 1
                    for (int i = lane; i < n; i += 32) {
                        const double *row = rows + i * ROW;
                        double u0, u1, u2, c;
                        pair_setup<RES>(Rm, t, row, u0, u1, u2, c);
                        if (RES == CLOSURE_POSE_REG_SPLIT) {
                            if (!(frob_sq(Rm, row) <= row[13])) rdead = true;     // exact: no perturbation involved
                        }
                        float g0, g1, g2, fcb, eps;
                        screen_row_any<RES>(u0, u1, u2, c - row[RS::BETA + 1], tp2, tp2sq3, RES == kEll ? QL[2 * i + 1].z : 0.f,
                                            g0, g1, g2, fcb, eps);
                        rowsL[i] = make_float4(g0, g1, g2, fcb - eps);
                        eps_l = fmaxf(eps_l, eps);
                    }
                    epsL = wmax_nonneg(eps_l);
                    rdeadL = __any_sync(FULL, rdead);
                    full_m = m1;
                    if (stats) stc[3] += n;
                    __syncwarp();
                }
                if (stats) { stc[9] += 1; stc[7] += (unsigned long long)n * KP; }
                unsigned feas = 0u;
                if (!rdeadL) {
                    float M = -CUDART_INF_F;
                    float4 c4 = make_float4(0.f, 0.f, 0.f, 0.f);
                    if (e_act) {
                        c4 = cand4[ek];
                        for (int i = ech; i < n; i += NCH) {
                            const float4 f = rowsL[i];
                            if (RES == kEll) M = fmaxf(M, ell_value(f, QL[2 * i], QL[2 * i + 1], c4));
                            else M = fmaxf(M, fmaf(f.x, c4.x, fmaf(f.y, c4.y, fmaf(f.z, c4.z, f.w))));
                        }
                    }
                    M = chunk_max_to_first(M, KP, NCH);      // valid on the lanes with ech == 0 (`mine` below)
                    // M = max_i (v32_i - eps_i):  M > th  => some constraint violated for sure;
                    // M + 2 eps_max <= th => every constraint satisfied for sure.
                    const bool dead = M > c4.w;
                    const bool sure = (epsL < CUDART_INF_F) && (M <= c4.w - 2.0f * epsL);
                    const bool mine = e_act && ech == 0;
                    unsigned alive2 = __ballot_sync(FULL, mine && !dead) & cand_alive;
                    unsigned undecided = __ballot_sync(FULL, mine && !dead && !sure) & cand_alive;
                    if (L.exact_only & 2) { alive2 = cand_alive; undecided = cand_alive; }
                    if (L.exact_only & 32) { alive2 &= ~undecided; undecided = 0u; }   // fp32 mode: undecided counts as VIOLATED, so every emitted sample stays inside S (Prop. 4)
                    while (undecided != 0u) {                // rare: fp64 decides
                        const int k = __ffs(undecided) - 1;
                        undecided &= undecided - 1u;
                        if (!exact_candidate_feasible<RES>(Rm, t, rows, n, rng, (uint32_t)s, candj[k], t_p, lane))
                            alive2 &= ~(1u << k);
                        if (stats) stc[1] += n;
                    }
                    feas = alive2;
                }
                if (feas != 0u) { m0 = m1 + 1; win = feas; }
            }
        }

        int j_win = 0;
        if (m0) {
            const int kw = __ffs(win) - 1;                    // lowest rank among the feasible (R-8)
            j_win = candj[kw];
            double x, y, z;
            rng.xi3((uint32_t)s, (uint32_t)j_win, 1u, x, y, z);
            const double t0 = __dadd_rn(pose[9], __dmul_rn(t_p, x));
            const double t1 = __dadd_rn(pose[10], __dmul_rn(t_p, y));
            const double t2 = __dadd_rn(pose[11], __dmul_rn(t_p, z));
            const double re = (lane < 9) ? RmS[(m0 - 1) * 9 + lane] : 0.0;
            __syncwarp();
            if (lane < 9) pose[lane] = re;
            if (lane == 9) { pose[9] = t0; pose[10] = t1; pose[11] = t2; }
            if (stats) stc[4] += 1;
        }
        moved = (m0 != 0);
        if (m0 != 1) hit = true;                              // R-12 (R-11: nothing feasible -> unchanged)
        if (L.out_trace != nullptr && lane == 0)
            L.out_trace[((size_t)blockIdx.y * L.num_walkers + local) * L.num_steps + (s - 1)] = m0 | (j_win << 8);
        __syncwarp();                                         // RmS / pert / candj readers done before the next step writes
    }

    // ---- a7: emit
    if (lane == 0) {
        const size_t o = (size_t)blockIdx.y * L.num_walkers + local;
        double2 *dst = reinterpret_cast<double2 *>(L.out_samples + 12 * o);
#pragma unroll
        for (int e = 0; e < 6; ++e) dst[e] = make_double2(pose[2 * e], pose[2 * e + 1]);
        L.out_flags[o] = hit ? 1 : 0;
        if (stats) {
            stc[5] = (unsigned long long)L.num_steps;
            stc[11] = (unsigned long long)(clock64() - clk_begin);
            for (int k = 0; k < kNumStats; ++k) atomicAdd(L.stats + k, stc[k]);
        }
    }
}

// ---------------------------------------------------------------------------------- the kernel, two warps per walker
// For launches that leave the GPU mostly empty (up to kPipeMaxWalkers walkers in all: BASELINE config 1, the paper's own 200
// walks per instance) the time is one warp's latency per iteration, not throughput.  Here a walker owns a PAIR of warps, one
// iteration apart: the odd warp (producer) draws the perturbations of iteration s + 1, evaluates eq. (14) and selects the
// N_P* candidates (a2-a4: what needs the pose only) while the even warp (consumer) walks the ladder of iteration s and updates
// the pose (a5-a6).  The candidates are handed over through two buffers in shared memory; the warps meet at one named barrier
// per iteration.  The producer's work is speculative: it assumes that iteration s does not move the walker, which holds for a
// walker that has reached the boundary (95 % of the iterations at config 1).  When the consumer does accept a move it redoes
// the set-up, the producer recomputes iteration s + 1 at the new pose (two more barriers), and nothing of the discarded pass
// is used -- so every decision is the one-warp kernel's, bit for bit (tests/test_gpu_parity.py).  Same code as above otherwise.
constexpr int kPipeBytes = 32 * 16 + 32 * 4 + 32 * 4 + 16;    // second candidate buffer + the moved flags, per walker
constexpr long long kPipeMaxWalkers = 148 * 8;                // two CTAs of four walker pairs per SM: everything resident at once

#ifndef CLOSURE_PIPE_WALKERS
#define CLOSURE_PIPE_WALKERS 4     // walkers (pairs of warps) per CTA
#endif
constexpr int kPipeWalkers = CLOSURE_PIPE_WALKERS;
constexpr int kPipeThreads = 64 * kPipeWalkers;

template <int RES, int NQ>
__global__ void __launch_bounds__(kPipeThreads, 512 / kPipeThreads) walker_dense_pipe_kernel(const __grid_constant__ WalkLaunch L)
{
    using RS = Res<RES>;
    constexpr int ROW = RS::ROW;
    constexpr int NPK = NQ / 2;            // packed pairs of perturbations
    constexpr bool ODD = (NQ & 1) != 0;    // plus one scalar slot

    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ int n_runs_s;
    __shared__ float amax_s;
    const int warp_raw = threadIdx.x >> 5;
    // warps w and w + kPipeWalkers serve walker slot w: with four slots the two warps of a walker share a scheduler (warp id mod 4)
    // and every scheduler holds one producer and one consumer (measured: pairs on adjacent warp ids put all producers, the longer
    // stage, on two of the four schedulers)
    const int warp = warp_raw % kPipeWalkers;           // walker slot of the CTA
    const bool producer = warp_raw >= kPipeWalkers;
    int lane = threadIdx.x & 31;
    const InstanceDesc *__restrict__ D = L.desc[blockIdx.y];
    const int n = D->n;
    const int rows_bytes = D->rows_bytes;
    int n_p = L.n_p, n_ps = L.n_p_star, n_t = L.n_t;
    // Values the iteration uses all the time are made opaque to the compiler: under register pressure it otherwise
    // re-derives them from special registers and the constant bank inside the loop instead of keeping them in a register.
#define CLOSURE_PIN_R(x) asm volatile("" : "+r"(x))
#define CLOSURE_PIN_F(x) asm volatile("" : "+f"(x))
    CLOSURE_PIN_R(lane); CLOSURE_PIN_R(n_p); CLOSURE_PIN_R(n_ps); CLOSURE_PIN_R(n_t);
    uint64_t *bar = reinterpret_cast<uint64_t *>(smem_raw);
    double *rows = reinterpret_cast<double *>(smem_raw + 16);
    stage_rows(smem_raw + 16, bar, D->rows, rows_bytes);                        // a0 (TMA bulk copy)
    const CoopSmem lay = coop_layout(rows_bytes, n, n_t, NQ, 1, L.pairs_cap, kCoopWarps, af_width<RES>(), af_extra<RES>(L.pairs_cap));
    int *run_end = reinterpret_cast<int *>(smem_raw + lay.run_end);
    float *run_bf = reinterpret_cast<float *>(smem_raw + lay.run_bf);
    int *run_pend = reinterpret_cast<int *>(smem_raw + lay.run_pend);   // end of run r in rowsA, in PAIRS of rows
    int *pos = reinterpret_cast<int *>(smem_raw + lay.pos);             // row of constraint i in rowsA (bit 30: write it twice)
    if (warp_raw == 0) {                               // runs of equal bounds (rows are sorted by bound)
        int cnt = 0;
        for (int base = 0; base < n; base += 32) {
            const int i = base + lane;
            bool end = false;
            double beta = 0.0;
            if (i < n) {
                beta = rows[i * ROW + RS::BETA];
                end = (i == n - 1) || (rows[(i + 1) * ROW + RS::BETA] != beta);
            }
            const unsigned m = __ballot_sync(FULL, end);
            if (end) {
                const int r = cnt + __popc(m & ((1u << lane) - 1u));
                run_end[r] = i;
                run_bf[r] = (float)beta;
            }
            cnt += __popc(m);
        }
        __syncwarp();
        if (lane == 0) {
            // rowsA holds the fp32 set-ups two constraints per entry; a run of odd length repeats its last
            // constraint (a maximum does not see duplicates), so no pair straddles two bounds
            n_runs_s = cnt;
            int p = 0, start = 0, longest = 0;
            for (int r = 0; r < cnt; ++r) {
                const int end = run_end[r];
                const int p_begin = p >> 1;
                for (int i = start; i <= end; ++i) pos[i] = p++;
                if (p & 1) { pos[end] |= 0x40000000; ++p; }
                run_pend[r] = p >> 1;
                longest = max(longest, (p >> 1) - p_begin);
                start = end + 1;
            }
        }
    }
    if (RES == CLOSURE_REG_3D3D || RES == CLOSURE_POSE_REG) {
        // fp32 image of the constraints for the set-up's search (fast_rung_rows), and max_i |a_i| for its Lipschitz slack
        float4 *af = reinterpret_cast<float4 *>(smem_raw + lay.af);
        float am = 0.f;
        for (int i = threadIdx.x; i < n; i += kPipeThreads) {
            const double *row = rows + i * ROW;
            const float b2 = (float)row[RS::BETA + 1];
            if (RES == CLOSURE_REG_3D3D) {
                af[i] = make_float4((float)row[0], (float)row[1], (float)row[2], b2);
                am = fmaxf(am, (float)sqrt(row[0] * row[0] + row[1] * row[1] + row[2] * row[2]) * 1.000001f);
            } else {
                af[3 * i] = make_float4((float)row[0], (float)row[1], (float)row[2], b2);
                af[3 * i + 1] = make_float4((float)row[3], (float)row[4], (float)row[5], 0.f);
                af[3 * i + 2] = make_float4((float)row[6], (float)row[7], (float)row[8], 0.f);
            }
        }
        if (RES == CLOSURE_REG_3D3D) {
            if (threadIdx.x == 0) amax_s = 0.f;
            __syncthreads();
            atomicMax(reinterpret_cast<unsigned int *>(&amax_s), __float_as_uint(wmax_nonneg(am)));   // non-negative floats order as uints
        }
    }
    __syncthreads();
    const int n_runs = n_runs_s;
    if (RES == kEll) {
        float4 *QLw = reinterpret_cast<float4 *>(smem_raw + lay.af);
        float *QAw = reinterpret_cast<float *>(QLw + 2 * n);
        const float tpq = (float)L.t_p * 1.0000002f;
        for (int i = threadIdx.x; i < n; i += kPipeThreads) {
            const double *row = rows + i * ROW;
            const float q00 = (float)(0.25 * row[8]), q01 = (float)(0.5 * row[9]), q02 = (float)(0.5 * row[10]);
            const float q11 = (float)(0.25 * row[11]), q12 = (float)(0.5 * row[12]), q22 = (float)(0.25 * row[13]);
            const float qsum = (fabsf(q00) + fabsf(q01) + fabsf(q02) + fabsf(q11) + fabsf(q12) + fabsf(q22)) * 1.000001f;
            QLw[2 * i] = make_float4(q00, q01, q02, q11);
            QLw[2 * i + 1] = make_float4(q12, q22, 4.0f * tpq * tpq * qsum, 0.f);     // qmag = (2 t_p)^2 sum|Q|
            const int pp = pos[i], p = pp & 0x3fffffff;
            float *A = QAw + (p >> 1) * 12 + (p & 1);           // (Q00a Q00b Q01a Q01b) (Q02a Q02b Q11a Q11b) (Q12a Q12b Q22a Q22b)
            A[0] = q00; A[2] = q01; A[4] = q02; A[6] = q11; A[8] = q12; A[10] = q22;
            if (pp & 0x40000000) { A[1] = q00; A[3] = q01; A[5] = q02; A[7] = q11; A[9] = q12; A[11] = q22; }
        }
        __syncthreads();
    }

    const long long local = (long long)blockIdx.x * kPipeWalkers + warp;
    if (local >= L.num_walkers) return;                // no block-wide barrier below this line
    unsigned char *wp = smem_raw + lay.warp0 + (size_t)warp * lay.per_warp;
    float4 *rowsA = reinterpret_cast<float4 *>(wp + lay.rowsA);
    float4 *rowsL = reinterpret_cast<float4 *>(wp + lay.rowsL);
    float4 *pert = reinterpret_cast<float4 *>(wp + lay.pert);
    double2 *ab = reinterpret_cast<double2 *>(wp + lay.ab);
    float4 *qrow = reinterpret_cast<float4 *>(wp + lay.qrow);     // [rung][2]: the two tightest rows of each rung
    double *RmS = reinterpret_cast<double *>(wp + lay.RmS);
    double *dex = reinterpret_cast<double *>(wp + lay.dex);      // fp64 fallback: exact d_j, [q][lane]
    float *qL = reinterpret_cast<float *>(wp + lay.qL);           // [rung]: bound on the change of any residual norm
    // the kept perturbations (-2 d_j, -|d_j|^2) by rank, their indices and upper bounds of their eq. (14) values: two
    // buffers, iteration s uses buffer s & 1
    unsigned char *pp = smem_raw + lay.total + (size_t)warp * kPipeBytes;     // behind the one-warp kernel's layout
    float4 *cand4_0 = reinterpret_cast<float4 *>(wp + lay.cand4), *cand4_1 = reinterpret_cast<float4 *>(pp);
    int *candj_0 = reinterpret_cast<int *>(wp + lay.candj), *candj_1 = reinterpret_cast<int *>(pp + 512);
    float *candd_0 = reinterpret_cast<float *>(wp + lay.candd), *candd_1 = reinterpret_cast<float *>(pp + 640);
    volatile int *moved_flag = reinterpret_cast<volatile int *>(pp + 768);
    const int bar_id = warp + 1;                                  // named barrier of this walker's pair of warps
    auto pair_sync = [&]() { asm volatile("bar.sync %0, 64;" ::"r"(bar_id) : "memory"); };
    double *pose = reinterpret_cast<double *>(wp + lay.pose);     // R*(9) t*(3) omega(3): fp64, touched only on moves / fp64 paths
    // ellipsoid norm: quadratic-form coefficients of the constraints, by constraint (QL) and by pair-entry of rowsA (QA)
    const float4 *QL = reinterpret_cast<const float4 *>(smem_raw + lay.af);
    const float4 *QA = QL + 2 * n;
    const int2 *ridx = reinterpret_cast<const int2 *>(wp + lay.ridx);

    const unsigned long long w = (unsigned long long)(L.walker_begin + local);
    const unsigned long long seed = L.seed[blockIdx.y];
    Rng rng;
    rng.w_lo = (uint32_t)w;
    rng.w_hi8 = (uint32_t)(w >> 32) << 8;
    rng.k0 = (uint32_t)seed;
    rng.k1 = (uint32_t)(seed >> 32);

    // ---- a1: walker init, replicated on the lanes (Alg. 2 l.8-9): the consumer
    if (!producer) {
        double R[9], t[3], vel[3];
        init_walker<CLOSURE_MODE_ROT>(D, L, rng, w, R, t, vel);
        for (int m = lane; m < n_t; m += 32) {         // ladder dT_m = gamma^(m-1) by repeated multiplication
            double dT = 1.0;
            for (int q = 0; q < m; ++q) dT = dT * L.gamma;
            const double p0 = dT * vel[0], p1 = dT * vel[1], p2 = dT * vel[2];
            double A, B;
            exp_coeffs(fma(p2, p2, fma(p1, p1, p0 * p0)), A, B);
            ab[m] = make_double2(A * dT, B * dT * dT);
        }
        if (lane == 0) {
#pragma unroll
            for (int e = 0; e < 9; ++e) pose[e] = R[e];
#pragma unroll
            for (int e = 0; e < 3; ++e) { pose[9 + e] = t[e]; pose[12 + e] = vel[e]; }
        }
    }
    __syncwarp();

    const double t_p = L.t_p;
    const float tpf = (float)t_p * 1.0000002f;          // >= t_p
    float tp2 = 2.0f * tpf, tp2sq3 = 3.0f * tpf * tpf;
    float m2tp = -2.0f * (float)t_p;
    CLOSURE_PIN_F(tp2); CLOSURE_PIN_F(tp2sq3); CLOSURE_PIN_F(m2tp);
    const int KP = n_ps;                                // ladder candidates
    const int NCH = 32 / KP;                            // constraint chunks of the full evaluation
    const int ek = lane % KP, ech = lane / KP;
    const bool e_act = ech < NCH;

    // executed-work counters (closure_get_stats): in shared memory, touched by lane 0 and only when asked for
    unsigned long long *stc = reinterpret_cast<unsigned long long *>(wp + lay.stc);
    const bool stats = false;                           // (launches that count executed work take the one-warp kernel)
    if (stats) {
        for (int k = 0; k < kNumStats; ++k) stc[k] = 0ull;
    }
    const long long clk_begin = stats ? clock64() : 0ll;
    bool hit = false;
    bool moved = true;
    float epsA = 0.f;
    double rot_margin = CUDART_INF;
    // cached across iterations while the pose does not move
    int full_m = -1;                                    // rung whose rows sit in rowsL
    float epsL = 0.f;
    bool rdeadL = false;

    pair_sync();                                        // the walker's pose, velocity and ladder are in shared memory
    if (producer) {
        // ============================================================ producer: a2-a4 of iteration s into buffer s & 1
        int s = 1;
        bool redo = false;
        pair_sync();                                    // the first set-up is done
        while (s <= L.num_steps) {
            epsA = (float)pose[16];
            rot_margin = pose[15];
            float4 *c4b = (s & 1) ? cand4_1 : cand4_0;
            int *cj = (s & 1) ? candj_1 : candj_0;
            float *cd = (s & 1) ? candd_1 : candd_0;
            // ================================================== a2: perturbations of this lane
            unsigned long long p0[NPK > 0 ? NPK : 1], p1[NPK > 0 ? NPK : 1], p2[NPK > 0 ? NPK : 1];
            float o0 = 0.f, o1 = 0.f, o2 = 0.f;                  // the odd slot NQ-1
            float dd[NQ];
            {
                int jv[NQ];
                uint32_t x[NQ], y[NQ], z[NQ];
    #pragma unroll
                for (int q = 0; q < NQ; ++q) jv[q] = lane + 32 * q;
                philox_batch<NQ>(rng, (uint32_t)s, jv, x, y, z);
                float e0[NQ], e1[NQ], e2[NQ];
                // packed slots are produced by packed instructions so that they live in aligned register pairs
                // (same roundings as the scalar pm1f() * m2tp)
                const unsigned long long C1 = pk2(4.656612873077392578125e-10f, 4.656612873077392578125e-10f);
                const unsigned long long C2 = pk2(2.3283064365386962890625e-10f - 1.0f, 2.3283064365386962890625e-10f - 1.0f);
                const unsigned long long M2 = pk2(m2tp, m2tp);
    #pragma unroll
                for (int k = 0; k < NPK; ++k) {
                    p0[k] = mul2(M2, fma2(pk2((float)x[2 * k], (float)x[2 * k + 1]), C1, C2));
                    p1[k] = mul2(M2, fma2(pk2((float)y[2 * k], (float)y[2 * k + 1]), C1, C2));
                    p2[k] = mul2(M2, fma2(pk2((float)z[2 * k], (float)z[2 * k + 1]), C1, C2));
                    upk2(p0[k], e0[2 * k], e0[2 * k + 1]);
                    upk2(p1[k], e1[2 * k], e1[2 * k + 1]);
                    upk2(p2[k], e2[2 * k], e2[2 * k + 1]);
                }
                if (ODD) { e0[NQ - 1] = m2tp * pm1f(x[NQ - 1]); e1[NQ - 1] = m2tp * pm1f(y[NQ - 1]); e2[NQ - 1] = m2tp * pm1f(z[NQ - 1]); }
    #pragma unroll
                for (int q = 0; q < NQ; ++q) {
                    // (ellipsoid: the pair carries its own quadratic form d^T Lambda_i d, nothing is added per run and thresholds are 0)
                    dd[q] = RES == kEll ? 0.f : 0.25f * fmaf(e2[q], e2[q], fmaf(e1[q], e1[q], e0[q] * e0[q]));
                    pert[32 * q + lane] = make_float4(e0[q], e1[q], e2[q], -dd[q]);
                }
                if (ODD) { o0 = e0[NQ - 1]; o1 = e1[NQ - 1]; o2 = e2[NQ - 1]; }
            }

            // ================================================== a3: eq. (14) in fp32 with error bound
            float dt[NQ];
            float unc_l = 0.f;
            {
    #pragma unroll
                for (int q = 0; q < NQ; ++q) dt[q] = CUDART_INF_F;
                const float E0 = epsA + tp2sq3 * kMu19;          // bound on |a32 - a64| up to its own rounding
                int pp = 0;
                for (int r = 0; r < n_runs; ++r) {
                    const int pend = run_pend[r];
                    const float bf = run_bf[r];
                    float mx[NQ];
    #pragma unroll
                    for (int q = 0; q < NQ; ++q) mx[q] = -CUDART_INF_F;
    #pragma unroll(NQ <= 2 ? 4 : 1)   // measured: unrolling the NQ = 5 body further costs 2-4 % (C2, C4)
                    for (; pp < pend; ++pp) {
                        // two constraints a, b per entry: X = (f0a f0b f1a f1b), Y = (f2a f2b fca fcb)
                        const float4 X = rowsA[2 * pp], Y = rowsA[2 * pp + 1];
                        if (RES == kEll) {
                            // (w, c) as above plus the quadratic form: U = (Q00a Q00b Q01a Q01b) V = (Q02a Q02b Q11a Q11b) W = (Q12a Q12b Q22a Q22b)
                            const float4 U = QA[3 * pp], V = QA[3 * pp + 1], W = QA[3 * pp + 2];
    #pragma unroll
                            for (int k = 0; k < NPK; ++k) {
                                const unsigned long long ta0 = fma2(pk2(V.x, V.x), p2[k], fma2(pk2(U.z, U.z), p1[k], fma2(pk2(U.x, U.x), p0[k], pk2(X.x, X.x))));
                                const unsigned long long ta1 = fma2(pk2(W.x, W.x), p2[k], fma2(pk2(V.z, V.z), p1[k], pk2(X.z, X.z)));
                                const unsigned long long ta2 = fma2(pk2(W.z, W.z), p2[k], pk2(Y.x, Y.x));
                                const unsigned long long va = fma2(ta0, p0[k], fma2(ta1, p1[k], fma2(ta2, p2[k], pk2(Y.z, Y.z))));
                                const unsigned long long tb0 = fma2(pk2(V.y, V.y), p2[k], fma2(pk2(U.w, U.w), p1[k], fma2(pk2(U.y, U.y), p0[k], pk2(X.y, X.y))));
                                const unsigned long long tb1 = fma2(pk2(W.y, W.y), p2[k], fma2(pk2(V.w, V.w), p1[k], pk2(X.w, X.w)));
                                const unsigned long long tb2 = fma2(pk2(W.w, W.w), p2[k], pk2(Y.y, Y.y));
                                const unsigned long long vb = fma2(tb0, p0[k], fma2(tb1, p1[k], fma2(tb2, p2[k], pk2(Y.w, Y.w))));
                                float la, ha, lb, hb;
                                upk2(va, la, ha);
                                upk2(vb, lb, hb);
                                mx[2 * k] = fmaxf(mx[2 * k], fmaxf(la, lb));
                                mx[2 * k + 1] = fmaxf(mx[2 * k + 1], fmaxf(ha, hb));
                            }
                            if (ODD) {                      // the odd slot takes both constraints in one packed chain
                                const unsigned long long E0o = pk2(o0, o0), E1o = pk2(o1, o1), E2o = pk2(o2, o2);
                                const unsigned long long t0 = fma2(pk2(V.x, V.y), E2o, fma2(pk2(U.z, U.w), E1o, fma2(pk2(U.x, U.y), E0o, pk2(X.x, X.y))));
                                const unsigned long long t1 = fma2(pk2(W.x, W.y), E2o, fma2(pk2(V.z, V.w), E1o, pk2(X.z, X.w)));
                                const unsigned long long t2 = fma2(pk2(W.z, W.w), E2o, pk2(Y.x, Y.y));
                                const unsigned long long vo = fma2(t0, E0o, fma2(t1, E1o, fma2(t2, E2o, pk2(Y.z, Y.w))));
                                float lo, hi;
                                upk2(vo, lo, hi);
                                mx[NQ - 1] = fmaxf(mx[NQ - 1], fmaxf(lo, hi));
                            }
                            continue;
                        }
    #pragma unroll
                        for (int k = 0; k < NPK; ++k) {
                            const unsigned long long va =
                                fma2(pk2(X.x, X.x), p0[k], fma2(pk2(X.z, X.z), p1[k], fma2(pk2(Y.x, Y.x), p2[k], pk2(Y.z, Y.z))));
                            const unsigned long long vb =
                                fma2(pk2(X.y, X.y), p0[k], fma2(pk2(X.w, X.w), p1[k], fma2(pk2(Y.y, Y.y), p2[k], pk2(Y.w, Y.w))));
                            float la, ha, lb, hb;
                            upk2(va, la, ha);
                            upk2(vb, lb, hb);
                            mx[2 * k] = fmaxf(mx[2 * k], fmaxf(la, lb));
                            mx[2 * k + 1] = fmaxf(mx[2 * k + 1], fmaxf(ha, hb));
                        }
                        if (ODD) {                          // the odd slot takes both constraints in one packed chain
                            const unsigned long long vo = fma2(pk2(X.x, X.y), pk2(o0, o0),
                                                               fma2(pk2(X.z, X.w), pk2(o1, o1),
                                                                    fma2(pk2(Y.x, Y.y), pk2(o2, o2), pk2(Y.z, Y.w))));
                            float lo, hi;
                            upk2(vo, lo, hi);
                            mx[NQ - 1] = fmaxf(mx[NQ - 1], fmaxf(lo, hi));
                        }
                    }
    #pragma unroll
                    for (int q = 0; q < NQ; ++q) {
                        // a ~ max_i |u_i - d|^2 within E0 + 2^-22 a;  sq ~ sqrt(a) within 2^-21 relative
                        const float a = fmaxf(mx[q] + dd[q], 1e-30f);
                        const float rr = rsqrt_normal(a);
                        const float sq = a * rr;
                        const float du = 1.01f * fmaf(E0, rr, (bf + sq) * kMu19);
                        unc_l = fmaxf(unc_l, du);
                        dt[q] = fminf(dt[q], bf - sq);
                    }
                }
                if (stats) stc[6] += (unsigned long long)n * n_p;
            }

            // ================================================== a4: top-N_P* with certified ranking
            const float rmf = (float)rot_margin;                // +inf unless POSE_REG_SPLIT
            float dv[NQ];
    #pragma unroll
            for (int q = 0; q < NQ; ++q) dv[q] = (lane + 32 * q < n_p) ? fminf(dt[q], rmf) : -CUDART_INF_F;
            float unc = wmax_nonneg(unc_l), myval;
            if (RES == CLOSURE_POSE_REG_SPLIT) unc += 1.2e-7f * fabsf(rmf);
            // (exact_only & 4: debug, every step takes the fp64 fall-back; & 16: on all N_P perturbations)
            if (!topk_certified<NQ>(dv, n_ps, unc, (L.exact_only & 4) != 0, (L.exact_only & 32) != 0, lane, cj, cd, myval)) {
                double R[9], t[3];
    #pragma unroll
                for (int e = 0; e < 9; ++e) R[e] = pose[e];
    #pragma unroll
                for (int e = 0; e < 3; ++e) t[e] = pose[9 + e];
                const ExactMargin<RES> exact{ R, t, rows, n, rng, (uint32_t)s, t_p, rot_margin };
                const int cnt = topk_fp64<NQ>(dv, n_p, n_ps, unc, myval, (L.exact_only & 16) != 0, lane, dex, cj, cd, exact);
                if (stats) { stc[8] += 1; stc[0] += (unsigned long long)n * cnt; }
            }
            __syncwarp();                                       // pert[], cj[] visible to all lanes
            if (lane < n_ps) c4b[lane] = pert[cj[lane]];
            __syncwarp();
            pair_sync();                                // candidates of iteration s are ready; the consumer has decided s - 1
            if (s > 1 && !redo && moved_flag[(s - 1) & 1] != 0) {
                pair_sync();                            // iteration s - 1 moved the walker: wait for the set-up, then redo s
                redo = true;
                continue;
            }
            redo = false;
            ++s;
        }
        return;
    }
    // ================================================================ consumer: set-ups, a5-a6 of iteration s, pose update
    {
        const long long c0 = stats ? clock64() : 0ll;
        coop_setup_on_move<RES>(smem_raw, warp, lane, rows_bytes, n, n_t, NQ, L.pairs_cap, t_p, amax_s, stats);
        if (stats) stc[10] += (unsigned long long)(clock64() - c0);
        epsA = (float)pose[16];
        rot_margin = pose[15];
        full_m = -1;
    }
    pair_sync();
    for (int s = 1; s <= L.num_steps; ++s) {
        pair_sync();                                    // candidates of iteration s are ready
        if (s > 1 && moved) {
            const long long c0 = stats ? clock64() : 0ll;
            coop_setup_on_move<RES>(smem_raw, warp, lane, rows_bytes, n, n_t, NQ, L.pairs_cap, t_p, amax_s, stats);
            if (stats) stc[10] += (unsigned long long)(clock64() - c0);
            epsA = (float)pose[16];
            rot_margin = pose[15];
            full_m = -1;
            pair_sync();                                // set-up done: the producer recomputes iteration s
            pair_sync();                                // ... and is done
        }
        const float4 *c4b = (s & 1) ? cand4_1 : cand4_0;
        const int *cj = (s & 1) ? candj_1 : candj_0;
        const float *cd = (s & 1) ? candd_1 : candd_0;
        // ================================================== a5-a6: ladder, first feasible rung
        int m0 = 0;
        unsigned win = 0u;
        bool lip_stop = false;
        const int khalf = (KP + 1) >> 1;
        for (int mb = 0; mb < n_t && m0 == 0 && !lip_stop; mb += 16) {
            // ---- screening of 16 rungs, lane = (rung, half of the candidates): a candidate is dead for sure
            // at rung m if one of the two tightest rows is violated beyond its error bound, or if its margin
            // at R* is more negative than the rotation to R_m (or any smaller one: qL is a suffix maximum)
            // can repair
            const int mq = mb + (lane & 15), hq = lane >> 4;
            const bool q_act = mq < n_t;
            unsigned alive = 0u;
            float Lm = CUDART_INF_F;
            if (q_act) {
                const float4 r0 = qrow[2 * mq], r1 = qrow[2 * mq + 1];
                Lm = qL[mq];
                const int k1 = min(KP, (hq + 1) * khalf);
                if (RES == kEll) {
                    const int2 ii = ridx[mq];
                    const float4 A0 = QL[2 * ii.x], B0 = QL[2 * ii.x + 1], A1 = QL[2 * ii.y], B1 = QL[2 * ii.y + 1];
                    for (int k = hq * khalf; k < k1; ++k) {
                        const float4 c4 = c4b[k];
                        const float v0 = ell_value(r0, A0, B0, c4), v1 = ell_value(r1, A1, B1, c4);
                        if (!(v0 > c4.w) && !(v1 > c4.w) && !(cd[k] + Lm < 0.f)) alive |= 1u << k;
                    }
                } else {
                for (int k = hq * khalf; k < k1; ++k) {
                    const float4 c4 = c4b[k];
                    const float v0 = fmaf(r0.x, c4.x, fmaf(r0.y, c4.y, fmaf(r0.z, c4.z, r0.w)));
                    const float v1 = fmaf(r1.x, c4.x, fmaf(r1.y, c4.y, fmaf(r1.z, c4.z, r1.w)));
                    if (!(v0 > c4.w) && !(v1 > c4.w) && !(cd[k] + Lm < 0.f)) alive |= 1u << k;
                }
                }
            }
            alive |= __shfl_xor_sync(FULL, alive, 16);
            if (L.exact_only & 2) alive = q_act ? ((KP >= 32) ? FULL : ((1u << KP) - 1u)) : 0u;   // debug: nothing is screened out
            if (mb + 16 < n_t && !(L.exact_only & 2)) {
                // no candidate can be repaired at the last rung of this block => none at any later rung
                float cdm = cd[0];
                for (int k = 1; k < KP; ++k) cdm = fmaxf(cdm, cd[k]);
                if (cdm + qL[mb + 15] < 0.f) lip_stop = true;
            }
            unsigned qmask = __ballot_sync(FULL, lane < 16 && alive != 0u);
            if (stats) stc[7] += (unsigned long long)(min(n_t, mb + 16) - mb) * 2 * KP;

            // ---- full evaluation of the surviving rungs, in order
            while (qmask != 0u && m0 == 0) {
                const int l0 = __ffs(qmask) - 1;
                qmask &= qmask - 1u;
                const int m1 = mb + l0;
                const unsigned cand_alive = __shfl_sync(FULL, alive, l0);
                double Rm[9], t[3];
#pragma unroll
                for (int e = 0; e < 9; ++e) Rm[e] = RmS[m1 * 9 + e];
#pragma unroll
                for (int e = 0; e < 3; ++e) t[e] = pose[9 + e];
                if (full_m != m1) {
                    __syncwarp();                            // earlier readers of rowsL are done
                    float eps_l = 0.f;
                    bool rdead = false;
#pragma unroll 1
                    for (int i = lane; i < n; i += 32) {
                        const double *row = rows + i * ROW;
                        double u0, u1, u2, c;
                        pair_setup<RES>(Rm, t, row, u0, u1, u2, c);
                        if (RES == CLOSURE_POSE_REG_SPLIT) {
                            if (!(frob_sq(Rm, row) <= row[13])) rdead = true;     // exact: no perturbation involved
                        }
                        float g0, g1, g2, fcb, eps;
                        screen_row_any<RES>(u0, u1, u2, c - row[RS::BETA + 1], tp2, tp2sq3, RES == kEll ? QL[2 * i + 1].z : 0.f,
                                            g0, g1, g2, fcb, eps);
                        rowsL[i] = make_float4(g0, g1, g2, fcb - eps);
                        eps_l = fmaxf(eps_l, eps);
                    }
                    epsL = wmax_nonneg(eps_l);
                    rdeadL = __any_sync(FULL, rdead);
                    full_m = m1;
                    if (stats) stc[3] += n;
                    __syncwarp();
                }
                if (stats) { stc[9] += 1; stc[7] += (unsigned long long)n * KP; }
                unsigned feas = 0u;
                if (!rdeadL) {
                    float M = -CUDART_INF_F;
                    float4 c4 = make_float4(0.f, 0.f, 0.f, 0.f);
                    if (e_act) {
                        c4 = c4b[ek];
                        for (int i = ech; i < n; i += NCH) {
                            const float4 f = rowsL[i];
                            if (RES == kEll) M = fmaxf(M, ell_value(f, QL[2 * i], QL[2 * i + 1], c4));
                            else M = fmaxf(M, fmaf(f.x, c4.x, fmaf(f.y, c4.y, fmaf(f.z, c4.z, f.w))));
                        }
                    }
                    M = chunk_max_to_first(M, KP, NCH);      // valid on the lanes with ech == 0 (`mine` below)
                    // M = max_i (v32_i - eps_i):  M > th  => some constraint violated for sure;
                    // M + 2 eps_max <= th => every constraint satisfied for sure.
                    const bool dead = M > c4.w;
                    const bool sure = (epsL < CUDART_INF_F) && (M <= c4.w - 2.0f * epsL);
                    const bool mine = e_act && ech == 0;
                    unsigned alive2 = __ballot_sync(FULL, mine && !dead) & cand_alive;
                    unsigned undecided = __ballot_sync(FULL, mine && !dead && !sure) & cand_alive;
                    if (L.exact_only & 2) { alive2 = cand_alive; undecided = cand_alive; }
                    if (L.exact_only & 32) { alive2 &= ~undecided; undecided = 0u; }   // fp32 mode: undecided counts as VIOLATED, so every emitted sample stays inside S (Prop. 4)
                    while (undecided != 0u) {                // rare: fp64 decides
                        const int k = __ffs(undecided) - 1;
                        undecided &= undecided - 1u;
                        if (!exact_candidate_feasible<RES>(Rm, t, rows, n, rng, (uint32_t)s, cj[k], t_p, lane))
                            alive2 &= ~(1u << k);
                        if (stats) stc[1] += n;
                    }
                    feas = alive2;
                }
                if (feas != 0u) { m0 = m1 + 1; win = feas; }
            }
        }

        int j_win = 0;
        if (m0) {
            const int kw = __ffs(win) - 1;                    // lowest rank among the feasible (R-8)
            j_win = cj[kw];
            double x, y, z;
            rng.xi3((uint32_t)s, (uint32_t)j_win, 1u, x, y, z);
            const double t0 = __dadd_rn(pose[9], __dmul_rn(t_p, x));
            const double t1 = __dadd_rn(pose[10], __dmul_rn(t_p, y));
            const double t2 = __dadd_rn(pose[11], __dmul_rn(t_p, z));
            const double re = (lane < 9) ? RmS[(m0 - 1) * 9 + lane] : 0.0;
            __syncwarp();
            if (lane < 9) pose[lane] = re;
            if (lane == 9) { pose[9] = t0; pose[10] = t1; pose[11] = t2; }
            if (stats) stc[4] += 1;
        }
        moved = (m0 != 0);
        if (m0 != 1) hit = true;                              // R-12 (R-11: nothing feasible -> unchanged)
        if (L.out_trace != nullptr && lane == 0)
            L.out_trace[((size_t)blockIdx.y * L.num_walkers + local) * L.num_steps + (s - 1)] = m0 | (j_win << 8);
        __syncwarp();                                         // RmS readers done before the next step writes
        if (lane == 0) moved_flag[s & 1] = moved ? 1 : 0;
    }

    // ---- a7: emit
    if (lane == 0) {
        const size_t o = (size_t)blockIdx.y * L.num_walkers + local;
        double2 *dst = reinterpret_cast<double2 *>(L.out_samples + 12 * o);
#pragma unroll
        for (int e = 0; e < 6; ++e) dst[e] = make_double2(pose[2 * e], pose[2 * e + 1]);
        L.out_flags[o] = hit ? 1 : 0;
        if (stats) {
            stc[5] = (unsigned long long)L.num_steps;
            stc[11] = (unsigned long long)(clock64() - clk_begin);
            for (int k = 0; k < kNumStats; ++k) atomicAdd(L.stats + k, stc[k]);
        }
    }
}


template <int RES, int NQ>
cudaError_t launch_pipe_q(const WalkLaunch &L, int n_instances, int max_rows_bytes, int max_n, cudaStream_t stream)
{
    const CoopSmem lay = coop_layout(max_rows_bytes, max_n, L.n_t, NQ, 1, L.pairs_cap, kCoopWarps, af_width<RES>(), af_extra<RES>(L.pairs_cap));
    const size_t smem = lay.total + (size_t)kCoopWarps * kPipeBytes;        // (laid out for kCoopWarps >= kPipeWalkers walkers)
    if (smem > 100 * 1024) return cudaErrorInvalidConfiguration;               // two CTAs per SM
    cudaError_t e = cudaFuncSetAttribute(walker_dense_pipe_kernel<RES, NQ>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    const long long blocks = (L.num_walkers + kPipeWalkers - 1) / kPipeWalkers;
    dim3 grid((unsigned)blocks, (unsigned)n_instances, 1);
    walker_dense_pipe_kernel<RES, NQ><<<grid, kPipeThreads, smem, stream>>>(L);
    return cudaGetLastError();
}

template <int RES, int NQ>
cudaError_t launch_q(const WalkLaunch &L, int n_instances, int max_rows_bytes, int max_n, cudaStream_t stream)
{
    const CoopSmem lay = coop_layout(max_rows_bytes, max_n, L.n_t, NQ, 1, L.pairs_cap, kCoopWarps, af_width<RES>(), af_extra<RES>(L.pairs_cap));
    if (lay.total > 200 * 1024) return cudaErrorInvalidConfiguration;
    cudaError_t e = cudaFuncSetAttribute(walker_dense_kernel<RES, NQ>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)lay.total);
    if (e != cudaSuccess) return e;
    const long long blocks = (L.num_walkers + kCoopWarps - 1) / kCoopWarps;
    if (blocks > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    dim3 grid((unsigned)blocks, (unsigned)n_instances, 1);
    walker_dense_kernel<RES, NQ><<<grid, kCoopThreads, lay.total, stream>>>(L);
    return cudaGetLastError();
}

template <int RES>
cudaError_t launch_r(const WalkLaunch &L, int n_instances, int max_rows_bytes, int max_n, cudaStream_t stream)
{
    // launches that leave the GPU mostly empty: two warps per walker, one iteration apart (walker_dense_pipe_kernel)
    if (L.stats == nullptr && !(L.exact_only & 64) && L.num_walkers * (long long)n_instances <= kPipeMaxWalkers) {
        cudaError_t e = cudaErrorInvalidConfiguration;
        if (L.n_p <= 64) e = launch_pipe_q<RES, 2>(L, n_instances, max_rows_bytes, max_n, stream);
        else if (L.n_p <= 160) e = launch_pipe_q<RES, 5>(L, n_instances, max_rows_bytes, max_n, stream);
        else e = launch_pipe_q<RES, 8>(L, n_instances, max_rows_bytes, max_n, stream);
        if (e != cudaErrorInvalidConfiguration) return e;
    }
    if (L.n_p <= 64) return launch_q<RES, 2>(L, n_instances, max_rows_bytes, max_n, stream);
    if (L.n_p <= 160) return launch_q<RES, 5>(L, n_instances, max_rows_bytes, max_n, stream);
    return launch_q<RES, 8>(L, n_instances, max_rows_bytes, max_n, stream);
}

}  // namespace

cudaError_t launch_walkers_coop_dense(int residual_type, const WalkLaunch &L, int n_instances, int max_rows_bytes,
                                      cudaStream_t stream)
{
    const int max_n = max_rows_bytes / (row_doubles(residual_type) * 8);
    switch (residual_type) {
    case CLOSURE_REG_3D3D: return launch_r<CLOSURE_REG_3D3D>(L, n_instances, max_rows_bytes, max_n, stream);
    case CLOSURE_POSE_REG: return launch_r<CLOSURE_POSE_REG>(L, n_instances, max_rows_bytes, max_n, stream);
    case CLOSURE_POSE_REG_SPLIT: return launch_r<CLOSURE_POSE_REG_SPLIT>(L, n_instances, max_rows_bytes, max_n, stream);
    case CLOSURE_REG_3D3D_ELL: return launch_r<CLOSURE_REG_3D3D_ELL>(L, n_instances, max_rows_bytes, max_n, stream);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace closure
