// Warp-cooperative walker kernel for the rotation-boundary sampler (Alg. 2) on the
// 2D reprojection residual z_i - Pi(K(R Z_i + t)) (eq. (2)).  Same organisation as
// walker_coop_kernel.cu (one warp per walker, set-ups once per accepted move, fp32 evaluation with
// rigorous error bounds, fp64 only where a decision is not certain); what differs is the pair:
//
//   with p = R Z_i + t* + d and zeta = z_i - (cx, cy), for p_3 > 0
//       ||z_i - Pi(K p)||  =  || (zeta_1 p_3 - fx p_1, zeta_2 p_3 - fy p_2) || / p_3  =:  ||q|| / p_3 ,
//   and q, p_3 are AFFINE in the translation perturbation d:
//       q_1 = A_1 + zeta_1 d_3 - fx d_1,   q_2 = A_2 + zeta_2 d_3 - fy d_2,   p_3 = P_3 + d_3 ,
//   (A, P_3) depending on the pose only.  eq. (14) needs ||q||^2 / p_3^2 (one MUFU.RCP per pair, one
//   rsqrt per run of equal bounds); in_purse is the cone test ||q||^2 - (beta p_3)^2 <= 0, no division.
//
// Error bounds (u = 2^-24; |d32 - d64| <= 6 u t_p per component, see walker_coop_kernel.cu):
//   E_q1 = u (3 |A_1| + 9 t_p (|zeta_1| + fx)),  E_q2 alike,  E_p = u (2 |P_3| + 7 t_p),
//   p_lo = P_3 - t_p > 0 (else nothing is certified),  rho_hi = (|A_1| + |A_2| + t_p (...)) / p_lo,
//   |rho32 - rho64| <= (E_q1 + E_q2) / p_lo + rho_hi (E_p / p_lo + 2^-19)      (unc uses twice that)
//   cone value g:  E_g = 2 (q1_hi E_q1 + q2_hi E_q2 + w_hi E_w) + 4 u (q1_hi^2 + q2_hi^2 + w_hi^2), x 1.5.
// The fp64 reference of every decision is the plain kernel's arithmetic (reproj_point / reproj_sq in
// walker_common.cuh); its own rounding (~1e-13 px) is far inside these bounds.
// The ellipse norm of eq. (6) (CLOSURE_REPROJ_2D3D_ELL) is the <NQ, true> instantiation: see RJ below.
#include <cuda_runtime.h>
#include <math_constants.h>
#include <stdint.h>

#include "closure_internal.h"
#include "walker_common.cuh"
#include "walker_coop_common.cuh"

#ifndef CLOSURE_COOP_MIN_CTAS
#define CLOSURE_COOP_MIN_CTAS 4   // resident CTAs per SM the register allocation aims at (128 registers per thread)
#endif

namespace closure {
namespace {

// One walker (warp) per CTA: the staged table is 8-10 rows, so nothing is gained by sharing it, and a CTA's slot is
// free again as soon as its walker ends instead of when the slowest of four does (measured at C3: 474 -> 496 M
// walker-steps/s; the affine kernels, with tables of 50-200 rows, do not gain and keep kCoopWarps = 4).
constexpr int kReprojWarps = 1;
constexpr int kReprojThreads = 32 * kReprojWarps;
// resident warps per SM the register allocation aims at: 20 (96 registers) measured best at C3 (16: 496, 20: 510, 24: 464 M)
constexpr int kReprojMinCtas = (CLOSURE_COOP_MIN_CTAS == 4 ? 5 : CLOSURE_COOP_MIN_CTAS) * (kCoopWarps / kReprojWarps);

// ELL = the ellipse norm of eq. (6) (CLOSURE_REPROJ_2D3D_ELL, rows [z Z beta beta^2 L00 L01 L11]): with the Cholesky factor
// Lambda = L L^T,  g^T Lambda g = |L^T q|^2 / p_3^2, and q' = L^T q is again affine in the perturbation,
//     q'_0 = A'_0 + a d_0 + b d_1 + c d_2,   q'_1 = A'_1 + d' d_1 + e d_2,
//     A'_0 = l00 A_0 + l10 A_1, A'_1 = l11 A_1,  a = -l00 fx, b = -l10 fy, c = l00 zeta_0 + l10 zeta_1, d' = -l11 fy, e = l11 zeta_1
// (the ball form is l00 = l11 = 1, l10 = 0: a = -fx, b = 0, c = zeta_0, d' = -fy, e = zeta_1).  Rows carry a third float4 with
// (a, b, d'); one more FMA in q'_0, so E_q0 = u (4 |A'_0| + 10 t_p (|a| + |b| + |c|)); everything else is the ball form's bound.
template <bool ELL> struct RJ {
    static constexpr int RES = ELL ? CLOSURE_REPROJ_2D3D_ELL : CLOSURE_REPROJ_2D3D;
    static constexpr int ROW = Res<RES>::ROW;
    static constexpr int BETA = Res<RES>::BETA;
    static constexpr int F4 = ELL ? 3 : 2;          // float4 words per fp32 row
};
constexpr double kU = 5.9604644775390625e-08;   // 2^-24

// 1 / x for the error and Lipschitz bounds (x > 0): MUFU.RCP and one Newton step in fp64 instead of the ~20 instructions of a
// correctly rounded fp64 division; relative error < 1e-13, far inside the 1.0001 - 1.001 slack every bound carries.  An x that
// fp32 cannot hold gives 0 or inf from MUFU.RCP: callers get +inf ("nothing certified"), never a bound that is too small.
__device__ __forceinline__ double bound_rcp(double x)
{
    const double r = (double)__frcp_rn((float)x);
    if (!(r > 0.0) || !(r < CUDART_INF)) return CUDART_INF;
    return r * fma(-x, r, 2.0);
}

// fp32 row of one constraint at the camera-frame point P (= R Z_i + t*): (A_1, A_2, P_3 or beta P_3, zeta_1),
// (zeta_2, beta, -E_g, rho bound) and the error constants above.
struct ReprojRow {
    float4 a, b, c;   // c = (a, b, d', .) of the whitened form (ELL only)
    float unc;      // bound on |rho32 - rho64| for eq. (14) (phase A rows)
    float g0;       // cone value at d = 0 minus E_g (ladder rows: tightness key)
};

template <bool LADDER, bool ELL>
__device__ __forceinline__ ReprojRow reproj_row(double P0, double P1, double P2, const double *row, const double (&K)[4],
                                                double t_p)
{
    constexpr int BETA = RJ<ELL>::BETA;
    const double zz0 = row[0] - K[2], zz1 = row[1] - K[3], beta = row[BETA];
    const double B0 = zz0 * P2 - K[0] * P0, B1 = zz1 * P2 - K[1] * P1;
    double l00 = 1.0, l10 = 0.0, l11 = 1.0;
    if (ELL) {                                                  // Cholesky of [[L00 L01] [L01 L11]] (positive definite: closure_create)
        l00 = sqrt(row[7]);
        l10 = row[8] / l00;
        l11 = sqrt(row[9] - l10 * l10);
    }
    const double A0 = ELL ? l00 * B0 + l10 * B1 : B0, A1 = ELL ? l11 * B1 : B1;
    const double ca = -l00 * K[0], cb = -l10 * K[1], cd = -l11 * K[1];          // a, b, d'
    const double z0 = ELL ? l00 * zz0 + l10 * zz1 : zz0, z1 = ELL ? l11 * zz1 : zz1;   // c, e
    const double s0 = fabs(ca) + fabs(cb) + fabs(z0), s1 = fabs(cd) + fabs(z1);
    const double Eq0 = kU * ((ELL ? 4.0 : 3.0) * fabs(A0) + (ELL ? 10.0 : 9.0) * t_p * s0);
    const double Eq1 = kU * (3.0 * fabs(A1) + 9.0 * t_p * s1);
    const double Ep = kU * (2.0 * fabs(P2) + 7.0 * t_p);       // phase A only: p_3 = P_3 + d_3
    const double plo = P2 - 1.001 * t_p;
    const double q0hi = fabs(A0) + t_p * s0, q1hi = fabs(A1) + t_p * s1;
    ReprojRow r;
    r.c = make_float4((float)ca, (float)cb, (float)cd, 0.f);
    if (!LADDER) {
        r.a = make_float4((float)A0, (float)A1, (float)P2, (float)z0);
        r.b = make_float4((float)z1, (float)beta, 0.f, 0.f);
        r.g0 = 0.f;
        if (plo > 0.0) {
            const double inv = bound_rcp(plo);
            const double rho_hi = (q0hi + q1hi) * inv;
            const double Erho = (Eq0 + Eq1) * inv + rho_hi * (Ep * inv + 1.9073486328125e-06);
            r.unc = (float)(2.0 * Erho + 4.76837158203125e-07 * beta + 1e-12 * (rho_hi + beta)) * 1.0001f;
        } else {
            r.unc = CUDART_INF_F;
        }
    } else {
        const double Bp = beta * P2;
        const double whi = fabs(Bp) + beta * t_p;
        const double Ew = kU * (2.0 * fabs(Bp) + 8.0 * beta * t_p);
        const double ss = q0hi * q0hi + q1hi * q1hi + whi * whi;
        double Eg = 1.5 * (2.0 * (q0hi * Eq0 + q1hi * Eq1 + whi * Ew) + 4.0 * kU * ss) + 1e-12 * ss;
        float Egf = (float)Eg * 1.0001f;
        if (!(plo > 0.0)) Egf = CUDART_INF_F;           // cheirality not certain: never certified, fp64 decides
        r.a = make_float4((float)A0, (float)A1, (float)Bp, (float)z0);
        r.b = make_float4((float)z1, (float)beta, -Egf, 0.f);
        r.unc = Egf;
        r.g0 = (float)(A0 * A0 + A1 * A1 - Bp * Bp) - Egf;
    }
    return r;
}

// Lipschitz bound of one constraint between R* (camera-frame point P + t) and R_m (Q + t), valid for |d_c| <= t_p:
//   |d/dtau fx p_1/p_3| <= fx (|dP_1| + |p_1/p_3| |dP_3|) / p_3 along p(tau) = p + tau dP
__device__ __forceinline__ double reproj_lip(double P0, double P1, double P2, double Q0, double Q1, double Q2, const double (&t)[3],
                                             const double (&K)[4], double t_p)
{
    const double plo = dmin(P2, Q2) + t[2] - 1.001 * t_p;
    if (!(plo > 0.0)) return CUDART_INF;
    const double inv = bound_rcp(plo);
    if (!(inv < CUDART_INF)) return CUDART_INF;
    const double x_hi = dmax(fabs(P0 + t[0]), fabs(Q0 + t[0])) + t_p;
    const double y_hi = dmax(fabs(P1 + t[1]), fabs(Q1 + t[1])) + t_p;
    const double d0 = fabs(Q0 - P0), d1 = fabs(Q1 - P1), d2i = fabs(Q2 - P2) * inv;
    return (K[0] * fma(x_hi, d2i, d0) + K[1] * fma(y_hi, d2i, d1)) * inv;
}

// eq. (14) of perturbation j in the plain kernel's arithmetic (functor for topk_fp64)
template <bool ELL> struct ExactMarginReproj {
    const double (&R)[9];
    const double (&t)[3];
    const double (&K)[4];
    const double *rows;
    int n;
    const Rng &rng;
    uint32_t s;
    double t_p;
    __device__ __forceinline__ double operator()(int j) const
    {
        double x, y, z;
        rng.xi3(s, (uint32_t)j, 1u, x, y, z);
        const double e0 = t_p * x, e1 = t_p * y, e2 = t_p * z;
        double d = CUDART_INF;
        const double tj[3] = { t[0] + e0, t[1] + e1, t[2] + e2 };
#pragma unroll 1
        for (int i = 0; i < n; ++i) {
            const double *row = rows + i * RJ<ELL>::ROW;
            double sq;
            if (ELL) {
                sq = direct_sq<RJ<ELL>::RES>(R, tj, row, K, 0);
            } else {
                double P0, P1, P2;
                reproj_point(R, row, P0, P1, P2);
                sq = reproj_sq(P0, P1, P2, tj[0], tj[1], tj[2], row, K);
            }
            d = dmin(d, row[RJ<ELL>::BETA] - sqrt(sq));
        }
        return d;
    }
};

// fp64 in_purse of ladder candidate (Rm, t* + d_j), constraints dealt to the lanes (plain kernel's arithmetic)
template <bool ELL>
__device__ __forceinline__ bool exact_candidate_feasible_reproj(const double (&Rm)[9], const double (&t)[3],
                                                                const double (&K)[4], const double *rows, int n,
                                                                const Rng &rng, uint32_t s, int j, double t_p, int lane)
{
    double x, y, z;
    rng.xi3(s, (uint32_t)j, 1u, x, y, z);
    const double k0 = t_p * x, k1 = t_p * y, k2 = t_p * z;
    bool ok = true;
    const double tk[3] = { t[0] + k0, t[1] + k1, t[2] + k2 };
#pragma unroll 1
    for (int i = lane; i < n; i += 32) {
        const double *row = rows + i * RJ<ELL>::ROW;
        double sq;
        if (ELL) {
            sq = direct_sq<RJ<ELL>::RES>(Rm, tk, row, K, 0);
        } else {
            double P0, P1, P2;
            reproj_point(Rm, row, P0, P1, P2);
            sq = reproj_sq(P0, P1, P2, tk[0], tk[1], tk[2], row, K);
        }
        if (!(sq <= row[RJ<ELL>::BETA + 1])) ok = false;
    }
    return __all_sync(FULL, ok);
}

// cone value of one (ladder row, candidate) pair minus its error bound
__device__ __forceinline__ float cone_lo(const float4 &ra, const float4 &rb, const float4 &c, float nfx, float nfy)
{
    const float q0 = fmaf(ra.w, c.z, fmaf(nfx, c.x, ra.x));
    const float q1 = fmaf(rb.x, c.z, fmaf(nfy, c.y, ra.y));
    const float w = fmaf(rb.y, c.z, ra.z);
    return fmaf(q0, q0, fmaf(q1, q1, fmaf(-w, w, rb.z)));
}
// the same on the whitened rows of the ellipse norm: rc = (a, b, d', .)
__device__ __forceinline__ float cone_lo_ell(const float4 &ra, const float4 &rb, const float4 &rc, const float4 &c)
{
    const float q0 = fmaf(ra.w, c.z, fmaf(rc.y, c.y, fmaf(rc.x, c.x, ra.x)));
    const float q1 = fmaf(rb.x, c.z, fmaf(rc.z, c.y, ra.y));
    const float w = fmaf(rb.y, c.z, ra.z);
    return fmaf(q0, q0, fmaf(q1, q1, fmaf(-w, w, rb.z)));
}
template <bool ELL>
__device__ __forceinline__ float cone_row(const float4 *r, const float4 &c, float nfx, float nfy)
{
    if (ELL) return cone_lo_ell(r[0], r[1], r[2], c);
    return cone_lo(r[0], r[1], c, nfx, nfy);
}

// ---------------------------------------------------------------------------------- the kernel
template <int NQ, bool ELL>
__global__ void __launch_bounds__(kReprojThreads, kReprojMinCtas) walker_coop_reproj_kernel(const __grid_constant__ WalkLaunch L)
{
    constexpr int ROW = RJ<ELL>::ROW, BETA = RJ<ELL>::BETA, F4 = RJ<ELL>::F4;
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ int n_runs_s;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const InstanceDesc *__restrict__ D = L.desc[blockIdx.y];
    const int n = D->n;
    const int rows_bytes = D->rows_bytes;
    const int n_p = L.n_p, n_ps = L.n_p_star, n_t = L.n_t;
    uint64_t *bar = reinterpret_cast<uint64_t *>(smem_raw);
    double *rows = reinterpret_cast<double *>(smem_raw + 16);
    stage_rows(smem_raw + 16, bar, D->rows, rows_bytes);                        // a0 (TMA bulk copy)
    const CoopSmem lay = coop_layout(rows_bytes, n, n_t, NQ, F4, (n * F4 + 1) / 2, kReprojWarps);
    int *run_end = reinterpret_cast<int *>(smem_raw + lay.run_end);
    float *run_bf = reinterpret_cast<float *>(smem_raw + lay.run_bf);
    if (warp == 0) {                                   // runs of equal bounds (rows are sorted by bound)
        int cnt = 0;
        for (int base = 0; base < n; base += 32) {
            const int i = base + lane;
            bool end = false;
            double beta = 0.0;
            if (i < n) {
                beta = rows[i * ROW + BETA];
                end = (i == n - 1) || (rows[(i + 1) * ROW + BETA] != beta);
            }
            const unsigned m = __ballot_sync(FULL, end);
            if (end) {
                const int r = cnt + __popc(m & ((1u << lane) - 1u));
                run_end[r] = i;
                run_bf[r] = (float)beta;
            }
            cnt += __popc(m);
        }
        if (lane == 0) n_runs_s = cnt;
    }
    __syncthreads();
    const int n_runs = n_runs_s;

    const long long local = (long long)blockIdx.x * kReprojWarps + warp;
    if (local >= L.num_walkers) return;                // no block-wide barrier below this line
    unsigned char *wp = smem_raw + lay.warp0 + (size_t)warp * lay.per_warp;
    float4 *rowsA = reinterpret_cast<float4 *>(wp + lay.rowsA);   // [n][F4]
    float4 *rowsL = reinterpret_cast<float4 *>(wp + lay.rowsL);   // [n][F4]
    float4 *pert = reinterpret_cast<float4 *>(wp + lay.pert);     // (d_j, 0)
    double2 *ab = reinterpret_cast<double2 *>(wp + lay.ab);
    float4 *qrow = reinterpret_cast<float4 *>(wp + lay.qrow);     // [rung][2 rows][F4]
    double *RmS = reinterpret_cast<double *>(wp + lay.RmS);
    double *dex = reinterpret_cast<double *>(wp + lay.dex);
    float *qL = reinterpret_cast<float *>(wp + lay.qL);
    float4 *cand4 = reinterpret_cast<float4 *>(wp + lay.cand4);
    int *candj = reinterpret_cast<int *>(wp + lay.candj);
    float *candd = reinterpret_cast<float *>(wp + lay.candd);
    double *pose = reinterpret_cast<double *>(wp + lay.pose);

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
    const float tpfl = (float)t_p;
    const float nfx = -(float)D->K[0], nfy = -(float)D->K[1];
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
    float uncA = CUDART_INF_F;
    int full_m = -1;                                    // rung whose rows sit in rowsL
    float epsL = 0.f;

    for (int s = 1; s <= L.num_steps; ++s) {
        // ================================================== set-up at the current pose (only after a move)
        if (moved) {
            const long long clk0 = stats ? clock64() : 0ll;
            double R[9], t[3], vel[3], K[4];
#pragma unroll
            for (int e = 0; e < 9; ++e) R[e] = pose[e];
#pragma unroll
            for (int e = 0; e < 3; ++e) { t[e] = pose[9 + e]; vel[e] = pose[12 + e]; }
#pragma unroll
            for (int e = 0; e < 4; ++e) K[e] = D->K[e];
            float unc_l = 0.f;
#pragma unroll 1
            for (int i = lane; i < n; i += 32) {
                const double *row = rows + i * ROW;
                double P0, P1, P2;
                reproj_point(R, row, P0, P1, P2);
                const ReprojRow r = reproj_row<false, ELL>(P0 + t[0], P1 + t[1], P2 + t[2], row, K, t_p);
                rowsA[F4 * i] = r.a;
                rowsA[F4 * i + 1] = r.b;
                if (ELL) rowsA[F4 * i + 2] = r.c;
                unc_l = fmaxf(unc_l, r.unc);
            }
            uncA = wmax_nonneg(unc_l);
            for (int m = lane; m < n_t; m += 32) {       // Exp(dT_m w) R* for every rung
                const double2 c2 = ab[m];
                double Rm[9];
                rotate_left(R, vel[0], vel[1], vel[2], c2.x, c2.y, Rm);
#pragma unroll
                for (int e = 0; e < 9; ++e) RmS[m * 9 + e] = Rm[e];
            }
            full_m = -1;
            __syncwarp();
            // per rung: the two tightest cone rows at d = 0 and the Lipschitz bound L_m on the change of
            // any reprojection residual norm between R* and R_m, valid for every |d_c| <= t_p:
            //   |d/dtau fx p_1/p_3| <= fx (|dP_1| + |p_1/p_3| |dP_3|) / p_3 along p(tau) = p + tau dP
            if (n <= 16) {
                // short tables (Ex.1 has ~8-10 keypoints): lane = (rung, constraint), 32 / G rungs per pass with G = 8 or
                // 16 lanes per rung, so that the lanes are not left idle by a loop over 8 constraints; same rows and bounds
                const int G = n <= 8 ? 8 : 16;
                const int c = lane & (G - 1);
                const bool has = c < n;
                const double *row = rows + (has ? c : 0) * ROW;
                const unsigned hm = ((G == 8) ? 0xFFu : 0xFFFFu) << (lane & ~(G - 1));
                double P0, P1, P2;
                reproj_point(R, row, P0, P1, P2);
                // ellipse norm: | ||g_m||_L - ||g_*||_L | <= ||L^T||_2 ||g_m - g_*||_2 <= sqrt(tr Lambda) (|dg_0| + |dg_1|)
                const double lam_scale = ELL ? sqrt(row[ELL ? 7 : 0] + row[ELL ? 9 : 0]) * 1.0000001 : 1.0;
#pragma unroll 1
                for (int m = lane / G; m < n_t; m += 32 / G) {
                    double Rm[9];
#pragma unroll
                    for (int e = 0; e < 9; ++e) Rm[e] = RmS[m * 9 + e];
                    double Q0, Q1, Q2;
                    reproj_point(Rm, row, Q0, Q1, Q2);
                    ReprojRow r = reproj_row<true, ELL>(Q0 + t[0], Q1 + t[1], Q2 + t[2], row, K, t_p);
                    double lip = reproj_lip(P0, P1, P2, Q0, Q1, Q2, t, K, t_p);
                    if (ELL) lip *= lam_scale;
                    if (!has) { r.g0 = -CUDART_INF_F; r.b.z = -CUDART_INF_F; }      // a row that never kills
                    const uint32_t key = has ? ((fkey(r.g0) & ~15u) | (uint32_t)c) : (uint32_t)c;
                    uint32_t m1, m2;
                    float lf;
                    group_top2_max(hm, G, key, has ? (float)lip : 0.f, m1, m2, lf);
                    const uint32_t key2 = (key == m1) ? 0u : key;
                    if (key == m1) {
                        qrow[2 * F4 * m] = r.a; qrow[2 * F4 * m + 1] = r.b;
                        if (ELL) qrow[2 * F4 * m + 2] = r.c;
                        qL[m] = lf * 1.001f + 1e-30f;
                        if (n == 1) {
                            qrow[2 * F4 * m + F4] = r.a; qrow[2 * F4 * m + F4 + 1] = r.b;
                            if (ELL) qrow[2 * F4 * m + F4 + 2] = r.c;
                        }
                    }
                    if (key2 == m2 && n > 1) {
                        qrow[2 * F4 * m + F4] = r.a; qrow[2 * F4 * m + F4 + 1] = r.b;
                        if (ELL) qrow[2 * F4 * m + F4 + 2] = r.c;
                    }
                }
            } else {
#pragma unroll 1
            for (int m = 0; m < n_t; ++m) {
                double Rm[9];
#pragma unroll
                for (int e = 0; e < 9; ++e) Rm[e] = RmS[m * 9 + e];
                ReprojRow b1, b2;
                b1.g0 = b2.g0 = -CUDART_INF_F;
                b1.a = b1.b = b1.c = b2.a = b2.b = b2.c = make_float4(0.f, 0.f, 0.f, 0.f);
                b1.b.z = b2.b.z = -CUDART_INF_F;            // a row that never kills
                double lip = 0.0;
#pragma unroll 1
                for (int i = lane; i < n; i += 32) {
                    const double *row = rows + i * ROW;
                    double P0, P1, P2, Q0, Q1, Q2;
                    reproj_point(R, row, P0, P1, P2);
                    reproj_point(Rm, row, Q0, Q1, Q2);
                    const ReprojRow r = reproj_row<true, ELL>(Q0 + t[0], Q1 + t[1], Q2 + t[2], row, K, t_p);
                    if (r.g0 > b1.g0) { b2 = b1; b1 = r; } else if (r.g0 > b2.g0) b2 = r;
                    lip = dmax(lip, reproj_lip(P0, P1, P2, Q0, Q1, Q2, t, K, t_p) *
                                        (ELL ? sqrt(row[ELL ? 7 : 0] + row[ELL ? 9 : 0]) * 1.0000001 : 1.0));
                }
                const uint32_t k1 = fkey(b1.g0);
                const uint32_t m1 = __reduce_max_sync(FULL, k1);
                const int src1 = __ffs(__ballot_sync(FULL, k1 == m1)) - 1;
                const uint32_t k2 = (lane == src1) ? fkey(b2.g0) : k1;
                const uint32_t m2 = __reduce_max_sync(FULL, k2);
                const int src2 = __ffs(__ballot_sync(FULL, k2 == m2)) - 1;
                if (lane == src1) {
                    qrow[2 * F4 * m] = b1.a; qrow[2 * F4 * m + 1] = b1.b;
                    if (ELL) qrow[2 * F4 * m + 2] = b1.c;
                }
                if (lane == src2) {
                    qrow[2 * F4 * m + F4] = (lane == src1) ? b2.a : b1.a;
                    qrow[2 * F4 * m + F4 + 1] = (lane == src1) ? b2.b : b1.b;
                    if (ELL) qrow[2 * F4 * m + F4 + 2] = (lane == src1) ? b2.c : b1.c;
                }
                const float lf = wmax_nonneg((float)lip);
                if (lane == 0) qL[m] = lf * 1.001f + 1e-30f;
            }
            }
            if (stats) { stc[2] += n; stc[3] += (unsigned long long)n * n_t; }
            __syncwarp();
            if (lane == 0) {                                 // suffix maximum: qL[m] holds for every rung >= m
                float sm = 0.f;
                for (int m = n_t - 1; m >= 0; --m) { sm = fmaxf(sm, qL[m]); qL[m] = sm; }
            }
            __syncwarp();
            if (stats) stc[10] += (unsigned long long)(clock64() - clk0);
        }

        // ================================================== a2: perturbations of this lane (d_j = t_p xi_j)
        float d0[NQ], d1[NQ], d2[NQ];
        {
            int jv[NQ];
            uint32_t x[NQ], y[NQ], z[NQ];
#pragma unroll
            for (int q = 0; q < NQ; ++q) jv[q] = lane + 32 * q;
            philox_batch<NQ>(rng, (uint32_t)s, jv, x, y, z);
#pragma unroll
            for (int q = 0; q < NQ; ++q) {
                d0[q] = tpfl * pm1f(x[q]); d1[q] = tpfl * pm1f(y[q]); d2[q] = tpfl * pm1f(z[q]);
                pert[32 * q + lane] = make_float4(d0[q], d1[q], d2[q], 0.f);
            }
        }

        // ================================================== a3: eq. (14) in fp32: max_i ||q||^2 / p_3^2 per run
        float dv[NQ];
        {
#pragma unroll
            for (int q = 0; q < NQ; ++q) dv[q] = CUDART_INF_F;
            int i = 0;
            for (int r = 0; r < n_runs; ++r) {
                const int end = run_end[r];
                const float bf = run_bf[r];
                float mx[NQ];
#pragma unroll
                for (int q = 0; q < NQ; ++q) mx[q] = 0.f;
#pragma unroll 1                         // measured: +2 % at C3 against the default unrolling
                for (; i <= end; ++i) {
                    const float4 ra = rowsA[F4 * i], rb = rowsA[F4 * i + 1];
                    float4 rc = make_float4(nfx, 0.f, nfy, 0.f);
                    if (ELL) rc = rowsA[F4 * i + 2];
#pragma unroll
                    for (int q = 0; q < NQ; ++q) {
                        const float q0 = ELL ? fmaf(ra.w, d2[q], fmaf(rc.y, d1[q], fmaf(rc.x, d0[q], ra.x)))
                                             : fmaf(ra.w, d2[q], fmaf(nfx, d0[q], ra.x));
                        const float q1 = fmaf(rb.x, d2[q], fmaf(ELL ? rc.z : nfy, d1[q], ra.y));
                        float wr;
                        asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(wr) : "f"(ra.z + d2[q]));
                        mx[q] = fmaxf(mx[q], fmaf(q0, q0, q1 * q1) * (wr * wr));
                    }
                }
#pragma unroll
                for (int q = 0; q < NQ; ++q) {
                    const float a = fmaxf(mx[q], 1e-30f);
                    dv[q] = fminf(dv[q], bf - a * rsqrt_normal(a));
                }
            }
#pragma unroll
            for (int q = 0; q < NQ; ++q)
                if (lane + 32 * q >= n_p) dv[q] = -CUDART_INF_F;
            if (stats) stc[6] += (unsigned long long)n * n_p;
        }

        // ================================================== a4: top-N_P* with certified ranking
        float myval;
        if (!topk_certified<NQ>(dv, n_ps, uncA, (L.exact_only & 4) != 0, (L.exact_only & 32) != 0, lane, candj, candd, myval)) {
            double R[9], t[3], K[4];
#pragma unroll
            for (int e = 0; e < 9; ++e) R[e] = pose[e];
#pragma unroll
            for (int e = 0; e < 3; ++e) t[e] = pose[9 + e];
#pragma unroll
            for (int e = 0; e < 4; ++e) K[e] = D->K[e];
            const ExactMarginReproj<ELL> exact{ R, t, K, rows, n, rng, (uint32_t)s, t_p };
            const int cnt = topk_fp64<NQ>(dv, n_p, n_ps, uncA, myval, (L.exact_only & 16) != 0, lane, dex, candj, candd, exact);
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
            // ---- screening of 16 rungs, lane = (rung, half of the candidates) (see walker_coop_kernel.cu)
            const int mq = mb + (lane & 15), hq = lane >> 4;
            const bool q_act = mq < n_t;
            unsigned alive = 0u;
            if (q_act) {
                float4 r0[F4], r1[F4];
#pragma unroll
                for (int e = 0; e < F4; ++e) { r0[e] = qrow[2 * F4 * mq + e]; r1[e] = qrow[2 * F4 * mq + F4 + e]; }
                const float Lm = qL[mq];
                const int k1 = min(KP, (hq + 1) * khalf);
                for (int k = hq * khalf; k < k1; ++k) {
                    const float4 c4 = cand4[k];
                    const float v0 = cone_row<ELL>(r0, c4, nfx, nfy);
                    const float v1 = cone_row<ELL>(r1, c4, nfx, nfy);
                    if (!(v0 > 0.f) && !(v1 > 0.f) && !(candd[k] + Lm < 0.f)) alive |= 1u << k;
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
                double Rm[9], t[3], K[4];
#pragma unroll
                for (int e = 0; e < 9; ++e) Rm[e] = RmS[m1 * 9 + e];
#pragma unroll
                for (int e = 0; e < 3; ++e) t[e] = pose[9 + e];
#pragma unroll
                for (int e = 0; e < 4; ++e) K[e] = D->K[e];
                if (full_m != m1) {
                    __syncwarp();                            // earlier readers of rowsL are done
                    float eps_l = 0.f;
#pragma unroll 1
                    for (int i = lane; i < n; i += 32) {
                        const double *row = rows + i * ROW;
                        double Q0, Q1, Q2;
                        reproj_point(Rm, row, Q0, Q1, Q2);
                        const ReprojRow r = reproj_row<true, ELL>(Q0 + t[0], Q1 + t[1], Q2 + t[2], row, K, t_p);
                        rowsL[F4 * i] = r.a;
                        rowsL[F4 * i + 1] = r.b;
                        if (ELL) rowsL[F4 * i + 2] = r.c;
                        eps_l = fmaxf(eps_l, r.unc);
                    }
                    epsL = wmax_nonneg(eps_l);
                    full_m = m1;
                    if (stats) stc[3] += n;
                    __syncwarp();
                }
                if (stats) { stc[9] += 1; stc[7] += (unsigned long long)n * KP; }
                float M = -CUDART_INF_F;
                if (e_act) {
                    const float4 c4 = cand4[ek];
                    for (int i = ech; i < n; i += NCH) M = fmaxf(M, cone_row<ELL>(rowsL + F4 * i, c4, nfx, nfy));
                }
                M = chunk_max_to_first(M, KP, NCH);          // valid on the lanes with ech == 0 (`mine` below)
                // M = max_i (g32_i - E_g,i):  M > 0 => some constraint violated for sure;
                // M + 2 max_i E_g,i <= 0 => every constraint satisfied (and in front of the camera) for sure.
                const bool dead = M > 0.f;
                const bool sure = (epsL < CUDART_INF_F) && (M <= -2.0f * epsL);   // (an infinite bound certifies nothing)
                const bool mine = e_act && ech == 0;
                unsigned alive2 = __ballot_sync(FULL, mine && !dead) & cand_alive;
                unsigned undecided = __ballot_sync(FULL, mine && !dead && !sure) & cand_alive;
                if (L.exact_only & 2) { alive2 = cand_alive; undecided = cand_alive; }
                if (L.exact_only & 32) { alive2 &= ~undecided; undecided = 0u; }   // fp32 mode: undecided counts as VIOLATED, so every emitted sample stays inside S (Prop. 4)
                while (undecided != 0u) {                    // rare: fp64 decides
                    const int k = __ffs(undecided) - 1;
                    undecided &= undecided - 1u;
                    if (!exact_candidate_feasible_reproj<ELL>(Rm, t, K, rows, n, rng, (uint32_t)s, candj[k], t_p, lane))
                        alive2 &= ~(1u << k);
                    if (stats) stc[1] += n;
                }
                if (alive2 != 0u) { m0 = m1 + 1; win = alive2; }
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

template <int NQ, bool ELL>
cudaError_t launch_q(const WalkLaunch &L, int n_instances, int max_rows_bytes, int max_n, cudaStream_t stream)
{
    constexpr int F4 = RJ<ELL>::F4;
    const CoopSmem lay = coop_layout(max_rows_bytes, max_n, L.n_t, NQ, F4, (max_n * F4 + 1) / 2, kReprojWarps);
    if (lay.total > 200 * 1024) return cudaErrorInvalidConfiguration;
    cudaError_t e = cudaFuncSetAttribute(walker_coop_reproj_kernel<NQ, ELL>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)lay.total);
    if (e != cudaSuccess) return e;
    const long long blocks = (L.num_walkers + kReprojWarps - 1) / kReprojWarps;
    if (blocks > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    dim3 grid((unsigned)blocks, (unsigned)n_instances, 1);
    walker_coop_reproj_kernel<NQ, ELL><<<grid, kReprojThreads, lay.total, stream>>>(L);
    return cudaGetLastError();
}

template <bool ELL>
cudaError_t launch_e(const WalkLaunch &L, int n_instances, int max_rows_bytes, cudaStream_t stream)
{
    const int max_n = max_rows_bytes / (RJ<ELL>::ROW * 8);
    if (L.n_p <= 32) return launch_q<1, ELL>(L, n_instances, max_rows_bytes, max_n, stream);
    if (L.n_p <= 64) return launch_q<2, ELL>(L, n_instances, max_rows_bytes, max_n, stream);
    if (L.n_p <= 160) return launch_q<5, ELL>(L, n_instances, max_rows_bytes, max_n, stream);
    return launch_q<8, ELL>(L, n_instances, max_rows_bytes, max_n, stream);
}

}  // namespace

cudaError_t launch_walkers_coop_reproj(int residual_type, const WalkLaunch &L, int n_instances, int max_rows_bytes,
                                       cudaStream_t stream)
{
    if (residual_type == CLOSURE_REPROJ_2D3D_ELL) return launch_e<true>(L, n_instances, max_rows_bytes, stream);
    return launch_e<false>(L, n_instances, max_rows_bytes, stream);
}

}  // namespace closure
