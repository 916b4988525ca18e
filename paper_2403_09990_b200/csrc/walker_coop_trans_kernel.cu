// Warp-cooperative walker kernel for the TRANSLATION-boundary sampler (Alg. A8 PAPER.md:1001-1066,
// tensorised as Alg. A9), all four residuals.  One warp owns one walker:
//
//   a2-a3  the N_P perturbed rotations R_j = Exp(theta_p xi_j) R* are dealt to the lanes
//          (j = lane + 32 q); each lane evaluates eq. (14) of its poses (R_j, t*) in fp64;
//   a4     the N_P* best by (d descending, j ascending) are extracted with warp reductions on
//          order-preserving 64-bit keys;
//   a5-a6  the N_P* x N_T ladder candidates (R_{j_k}, t* + dT_m v) are dealt to the lanes in the
//          order (m, k) Alg. A8 visits them, 32 at a time, each lane running in_purse on its
//          candidate with an exit at the first violated constraint; the first feasible one wins.
//
// Every fp64 residual is evaluated by the same functions as in the one-walker-per-thread kernel
// (margin_direct / in_purse_direct in walker_common.cuh), so the two kernels agree bit for bit.
//
// Reprojection residual (Ex.1, the one example the paper runs this sampler on): eq. (14) of the N_P
// poses is evaluated in fp32 with a certificate, as in walker_coop_reproj_kernel.cu.  With
// P_i = R* Z_i, b_i = P_i + t* and A = (zeta_1 b_3 - fx b_1, zeta_2 b_3 - fy b_2) set up in fp64 once per move,
// a pair is g = D_j P_i, q = A + (zeta_1 g_3 - fx g_1, zeta_2 g_3 - fy g_2), p_3 = b_3 + g_3, rho = ||q|| / p_3,
// where D_j = Exp(theta_p xi_j) - I comes from the series of sin(th)/th and (1 - cos th)/th^2
// (|theta_p xi| <= 0.7): only the small rotation part is computed in fp32.  Error bounds, u = 2^-24,
// th_max = sqrt(3) theta_p, |g| <= th_max |P_i|:
//   |D32 - D64| <= e_D = 2 u (13.5 th_max + 13 th_max^2) per entry (phi from pm1f: 6 u theta_p; series 5 u),
//   E_g = (e_D + 4 u th_max) |P_i|_1 + 3 u |g|_hi,   E_q1 = (|zeta_1| + fx)(E_g + 4 u |g|_hi) + 3 u |A_1|,
//   E_p = E_g + 2 u (|b_3| + |g|_hi),   p_lo = b_3 - |g|_hi - E_p > 0 (else nothing is certified),
//   rho_hi = (|A_1| + |A_2| + (|zeta_1| + fx + |zeta_2| + fy) |g|_hi) / p_lo,
//   |rho32 - rho64| <= (E_q1 + E_q2) / p_lo + rho_hi (E_p / p_lo + 2^-19)          (unc = twice that).
// The ranking is accepted only if consecutive values differ by more than 2 unc; otherwise the candidates
// that can still be in the top N_P* are re-evaluated in fp64 (topk_fp64).
// The ladder candidate (k, m) has the cone value g(s) = (q_1 + s c_1)^2 + (q_2 + s c_2)^2 - (w + s c_w)^2 at s = dT_m,
// q, w = beta p_3 of candidate k as above, c = (zeta_1 v_3 - fx v_1, zeta_2 v_3 - fy v_2), c_w = beta v_3:
//   |g32 - g| <= 2 W (E_q + E_w) + 8 u W^2 + 4097 E_q^2 + E_w^2 + (2^-12 + 4 u) |g|,   W = beta p3_hi + |c_w|,
// (2 Q E_q <= 2^-12 |g| + 2^12 E_q^2 + 2 W E_q with Q^2 = g + W^2), so with tau = 1.5 x the absolute part
// g32 > tau means violated, g32 < -tau with beta p_3 > E_w satisfied,
// and anything else goes to the fp64 in_purse of the plain kernel.
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

constexpr double kU = 5.9604644775390625e-08;   // 2^-24

struct TransSmem {
    size_t run_end, run_bf, warp0, per_warp, pose, dex, Rc, candj, candd, stc, rowsA, crow, betaf, Dc, krow, sT, total;
};

// Walkers (warps) per CTA: one for the reprojection residual (tables of 8-10 rows: a CTA's slot is free as soon as its
// walker ends; measured at C3 in TRANS mode 236 -> 248 M walker-steps/s), kCoopWarps for the residuals with long tables.
template <int RES> constexpr int kTransWarps = (RES == CLOSURE_REPROJ_2D3D) ? 1 : kCoopWarps;

constexpr int kKrowMax = 512;                  // (candidate, constraint) rows of the certified ladder

// krows: (candidate, constraint) rows of the certified ladder that the launch can need (0: none) -- sized by N_P* x N, not by
// kKrowMax, so that 16 one-warp CTAs of a short reprojection table fit an SM (at kKrowMax rows shared memory allowed 14)
__host__ __device__ inline TransSmem trans_layout(int rows_bytes, int nq, int n_fast, int krows, int warps)
{
    TransSmem s;
    size_t o = 16 + (size_t)((rows_bytes + 15) & ~15);
    s.run_end = o; o += (size_t)((n_fast * 4 + 15) & ~15);     // runs of equal bounds (reprojection only)
    s.run_bf = o;  o += (size_t)((n_fast * 4 + 15) & ~15);
    s.warp0 = o;
    size_t w = 0;
    s.pose = w;  w += 16 * 8;                    // R*(9) t*(3) v(3)
    s.dex = w;   w += (size_t)nq * 32 * 8;       // eq. (14) values, [q][lane]
    s.Rc = w;    w += 32 * 9 * 8;                // rotations of the kept perturbations, by rank
    s.candj = w; w += 32 * 4;
    s.candd = w; w += 32 * 4;
    s.stc = w;   w += 16 * 8;
    s.rowsA = w; w += (size_t)n_fast * 32;       // reprojection only: fp32 rows (R* Z_i, zeta) of the certified eq. (14)
    s.crow = w;  w += (size_t)n_fast * 16;       // per constraint: shift of the cone row per unit step along v, -tau
    s.betaf = w; w += (size_t)((n_fast * 4 + 15) & ~15);
    s.Dc = w;    w += (n_fast ? 32 * 12 * 4 : 0);               // D = Exp - I of the kept perturbations (fp32)
    s.krow = w;  w += (n_fast ? (size_t)krows * 16 : 0);        // cone rows of (candidate, constraint) at step 0
    s.sT = w;    w += (n_fast ? 64 * 4 : 0);                    // ladder steps dT_m in fp32
    s.per_warp = w;
    s.total = o + (size_t)warps * w;
    return s;
}

// eq. (14) at (Exp(theta_p xi_j) R*, t*): the plain kernel's phase A of TRANS mode (functor for topk_fp64)
template <int RES>
struct ExactMarginTrans {
    const double (&R)[9];
    const double (&t)[3];
    const double (&K)[4];
    const double *rows;
    int n;
    const Rng &rng;
    uint32_t s;
    double theta_p;
    __device__ __forceinline__ double operator()(int j) const
    {
        double x, y, z, E[9], Rj[9];
        rng.xi3(s, (uint32_t)j, 1u, x, y, z);
        exp_so3(theta_p * x, theta_p * y, theta_p * z, E);
        mat3_mul(E, R, Rj);
        return margin_direct<RES>(Rj, t, rows, n, K);
    }
};

template <int RES, int NQ>
__global__ void __launch_bounds__(32 * kTransWarps<RES>, CLOSURE_COOP_MIN_CTAS * (kCoopWarps / kTransWarps<RES>)) walker_coop_trans_kernel(const __grid_constant__ WalkLaunch L)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const InstanceDesc *__restrict__ D = L.desc[blockIdx.y];
    const int n = D->n;
    const int rows_bytes = D->rows_bytes;
    const int n_p = L.n_p, n_ps = L.n_p_star, n_t = L.n_t;
    uint64_t *bar = reinterpret_cast<uint64_t *>(smem_raw);
    const double *rows = reinterpret_cast<const double *>(smem_raw + 16);
    stage_rows(smem_raw + 16, bar, D->rows, rows_bytes);                        // a0 (TMA bulk copy)
    const TransSmem lay = trans_layout(rows_bytes, NQ, RES == CLOSURE_REPROJ_2D3D ? n : 0,
                                       n_ps * n <= kKrowMax ? n_ps * n : 0, kTransWarps<RES>);   // as fast_ladder below
    __shared__ int n_runs_s;
    int *run_end = reinterpret_cast<int *>(smem_raw + lay.run_end);
    float *run_bf = reinterpret_cast<float *>(smem_raw + lay.run_bf);
    if (RES == CLOSURE_REPROJ_2D3D) {                  // runs of equal bounds (rows are sorted by bound)
        if (warp == 0) {
            int cnt = 0;
            for (int base = 0; base < n; base += 32) {
                const int i = base + lane;
                bool end = false;
                double beta = 0.0;
                if (i < n) {
                    beta = rows[i * Res<RES>::ROW + Res<RES>::BETA];
                    end = (i == n - 1) || (rows[(i + 1) * Res<RES>::ROW + Res<RES>::BETA] != beta);
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
    }
    const int n_runs = (RES == CLOSURE_REPROJ_2D3D) ? n_runs_s : 0;

    const long long local = (long long)blockIdx.x * kTransWarps<RES> + warp;
    if (local >= L.num_walkers) return;                // no block-wide barrier below this line
    unsigned char *wp = smem_raw + lay.warp0 + (size_t)warp * lay.per_warp;
    double *dex = reinterpret_cast<double *>(wp + lay.dex);
    double *Rc = reinterpret_cast<double *>(wp + lay.Rc);
    int *candj = reinterpret_cast<int *>(wp + lay.candj);
    float *candd = reinterpret_cast<float *>(wp + lay.candd);
    unsigned long long *stc = reinterpret_cast<unsigned long long *>(wp + lay.stc);

    const unsigned long long w = (unsigned long long)(L.walker_begin + local);
    const unsigned long long seed = L.seed[blockIdx.y];
    Rng rng;
    rng.w_lo = (uint32_t)w;
    rng.w_hi8 = (uint32_t)(w >> 32) << 8;
    rng.k0 = (uint32_t)seed;
    rng.k1 = (uint32_t)(seed >> 32);

    double K[4];
#pragma unroll
    for (int e = 0; e < 4; ++e) K[e] = D->K[e];

    // ---- a1: walker init (Alg. A8 l.8-9), replicated on the lanes
    double R[9], t[3], vel[3];
    init_walker<CLOSURE_MODE_TRANS>(D, L, rng, w, R, t, vel);
    const bool stats = (L.stats != nullptr) && lane == 0;
    if (stats) {
        for (int k = 0; k < kNumStats; ++k) stc[k] = 0ull;
    }
    bool hit = false;
    // Reprojection residual: eq. (14) of the N_P poses in certified fp32 (see the header); needs the series of
    // Exp to hold (|theta_p xi| <= 0.7).  exact_only & 4 keeps the fp64 ranking (tests).
    constexpr bool FAST = (RES == CLOSURE_REPROJ_2D3D);
    const bool fast = FAST && (1.7320508075688772 * L.theta_p <= 0.7);
    float4 *rowsA = reinterpret_cast<float4 *>(wp + lay.rowsA);
    const float thpf = (float)L.theta_p;
    const float nfx = -(float)K[0], nfy = -(float)K[1];
    float4 *crow = reinterpret_cast<float4 *>(wp + lay.crow);
    float *betaf = reinterpret_cast<float *>(wp + lay.betaf);
    float *Dc = reinterpret_cast<float *>(wp + lay.Dc);
    float4 *krow = reinterpret_cast<float4 *>(wp + lay.krow);
    float *sT = reinterpret_cast<float *>(wp + lay.sT);
    // the ladder is certified too when its (candidate, constraint) rows fit; exact_only & 2: every candidate to fp64
    const bool fast_ladder = fast && (n_ps * n <= kKrowMax);
    if (fast) {
        for (int m = lane; m < n_t; m += 32) {
            double dT = 1.0;
            for (int q = 0; q < m; ++q) dT = dT * L.gamma;
            sT[m] = (float)dT;
        }
    }
    float uncA = CUDART_INF_F, tauMax = CUDART_INF_F, ewMax = CUDART_INF_F;
    int i_tight = 0;
    bool moved = true;
    const int KP = n_ps;
    const int items = KP * n_t;                          // ladder candidates, in Alg. A8's order (m, k)
    const FastDiv divKP(KP), divN(n);                     // items <= 20 x 64, KP n <= 20 x 4096: inside FastDiv's range

    for (int s = 1; s <= L.num_steps; ++s) {
        // ================================================== a2-a4: perturb, eq. (14), top-N_P*
        bool ranked = false;
        if (fast) {
            if (moved) {
                // pose-only part of the pairs: P_i = R* Z_i and the bound unc on |rho32 - rho64| (header)
                // With D_j = E_j - I (entries O(theta)):  p = (P_i + t*) + D_j P_i,
                //   q_1 = A_1 + zeta_1 (D P)_3 - fx (D P)_1,   A_1 = zeta_1 (P + t)_3 - fx (P + t)_1  (fp64, then rounded),
                // so that only the small rotation part is computed in fp32.
                const double th = 1.7320508075688772 * L.theta_p;
                const double eD = 2.0 * kU * (13.5 * th + 13.0 * th * th);          // |D32 - D64| per entry
                float unc_l = 0.f, tau_l = 0.f, ew_l = 0.f;
                uint32_t tight_l = 0u;                                              // (key of the cone value at the pose | constraint)
                for (int i = lane; i < n; i += 32) {
                    const double *row = rows + i * Res<RES>::ROW;
                    double P0, P1, P2;
                    reproj_point(R, row, P0, P1, P2);
                    const double zs0 = row[0] - K[2], zs1 = row[1] - K[3], beta = row[Res<RES>::BETA];
                    const double z0 = fabs(zs0), z1 = fabs(zs1);
                    const double b0 = P0 + t[0], b1 = P1 + t[1], b2 = P2 + t[2];
                    const double A0 = zs0 * b2 - K[0] * b0, A1 = zs1 * b2 - K[1] * b1;
                    tight_l = max(tight_l, (fkey((float)(A0 * A0 + A1 * A1 - (beta * b2) * (beta * b2))) & ~0xFFFu) | (uint32_t)i);
                    const double Pn = sqrt(P0 * P0 + P1 * P1 + P2 * P2), P1n = fabs(P0) + fabs(P1) + fabs(P2);
                    const double dhi = th * Pn * 1.01;                              // |D P| <= 2 sin(th/2) |P| <= th |P|
                    const double Ed = (eD + 4.0 * kU * th) * P1n + 3.0 * kU * dhi + 1e-13;   // error of each (D P)_r
                    const double Ep2 = Ed + 2.0 * kU * (fabs(b2) + dhi);           // p_3 = b_3 + (D P)_3
                    const double plo = b2 - dhi - Ep2;
                    const double Eq0 = (z0 + K[0]) * Ed + 3.0 * kU * fabs(A0) + 4.0 * kU * (z0 + K[0]) * dhi;
                    const double Eq1 = (z1 + K[1]) * Ed + 3.0 * kU * fabs(A1) + 4.0 * kU * (z1 + K[1]) * dhi;
                    float unc_i = CUDART_INF_F;
                    if (plo > 0.0) {
                        const double rho_hi = (fabs(A0) + fabs(A1) + (z0 + K[0] + z1 + K[1]) * dhi) / plo;
                        const double Erho = (Eq0 + Eq1) / plo + rho_hi * (Ep2 / plo + 1.9073486328125e-06);
                        unc_i = (float)(2.0 * Erho + 4.76837158203125e-07 * beta + 1e-12 * (rho_hi + beta)) * 1.0001f;
                    }
                    unc_l = fmaxf(unc_l, unc_i);
                    rowsA[2 * i] = make_float4((float)P0, (float)P1, (float)P2, (float)zs0);
                    rowsA[2 * i + 1] = make_float4((float)zs1, (float)A0, (float)A1, (float)b2);
                    // ladder: cone value g(s) = (q_1 + s c_1)^2 + (q_2 + s c_2)^2 - (w + s c_w)^2, s = dT_m in [0, 1],
                    // with c = (zeta_1 v_3 - fx v_1, zeta_2 v_3 - fy v_2), w = beta p_3, c_w = beta v_3.  |g32 - g| <=
                    // a + b |g| with the a below (header), so g32 > tau => violated, g32 < -tau => satisfied.
                    const double c0 = zs0 * vel[2] - K[0] * vel[0], c1 = zs1 * vel[2] - K[1] * vel[1], cw = beta * vel[2];
                    const double q0khi = fabs(A0) + (z0 + K[0]) * dhi, q1khi = fabs(A1) + (z1 + K[1]) * dhi;
                    const double p2hi = fabs(b2) + dhi;
                    const double EqL = (Eq0 + 3.0 * kU * fabs(c0) + kU * q0khi) + (Eq1 + 3.0 * kU * fabs(c1) + kU * q1khi);
                    const double EwL = beta * Ep2 + 3.0 * kU * beta * p2hi + 3.0 * kU * fabs(cw);
                    const double Whi = beta * p2hi + fabs(cw);
                    const double a = 2.0 * Whi * (EqL + EwL) + 8.0 * kU * Whi * Whi + 4097.0 * EqL * EqL + EwL * EwL;
                    float tau = (float)(1.5 * a + 1e-12 * Whi * Whi) * 1.0001f;
                    ew_l = fmaxf(ew_l, (float)EwL * 1.0001f);
                    crow[i] = make_float4((float)c0, (float)c1, (float)cw, -tau);
                    betaf[i] = (float)beta;
                    tau_l = fmaxf(tau_l, tau);
                }
                tauMax = wmax_nonneg(tau_l);
                ewMax = wmax_nonneg(ew_l);
                i_tight = min((int)(__reduce_max_sync(FULL, tight_l) & 0xFFFu), n - 1);     // where the ladder's constraint loop starts
                uncA = wmax_nonneg(unc_l);
                __syncwarp();
            }
            float dv[NQ];
            {
                int jv[NQ];
                uint32_t x[NQ], y[NQ], z[NQ];
#pragma unroll
                for (int q = 0; q < NQ; ++q) jv[q] = lane + 32 * q;
                philox_batch<NQ>(rng, (uint32_t)s, jv, x, y, z);
                float E[NQ][9], mx[NQ];
#pragma unroll
                for (int q = 0; q < NQ; ++q) {
                    // Exp(phi) = I + A [phi]x + B [phi]x^2 with the series of A = sin(th)/th, B = (1 - cos th)/th^2
                    const float f0 = thpf * pm1f(x[q]), f1 = thpf * pm1f(y[q]), f2 = thpf * pm1f(z[q]);
                    const float s0 = f0 * f0, s1 = f1 * f1, s2 = f2 * f2;
                    const float th2 = s0 + s1 + s2;
                    const float A = fmaf(th2, fmaf(th2, fmaf(th2, fmaf(th2, 2.7557319e-06f, -1.9841270e-04f), 8.3333333e-03f), -1.6666667e-01f), 1.0f);
                    const float B = fmaf(th2, fmaf(th2, fmaf(th2, fmaf(th2, 2.7557319e-07f, -2.4801587e-05f), 1.3888889e-03f), -4.1666667e-02f), 0.5f);
                    const float a0 = A * f0, a1 = A * f1, a2 = A * f2;
                    // D = E - I
                    E[q][0] = -B * (s1 + s2);        E[q][1] = fmaf(B, f0 * f1, -a2); E[q][2] = fmaf(B, f0 * f2, a1);
                    E[q][3] = fmaf(B, f0 * f1, a2);  E[q][4] = -B * (s0 + s2);        E[q][5] = fmaf(B, f1 * f2, -a0);
                    E[q][6] = fmaf(B, f0 * f2, -a1); E[q][7] = fmaf(B, f1 * f2, a0);  E[q][8] = -B * (s0 + s1);
                    dv[q] = CUDART_INF_F;
                }
                // perturbations 2k, 2k+1 share packed instructions (fma.rn.f32x2: the same roundings as the scalar chain below,
                // which the odd slot NQ-1 keeps): 18 packed + 2 MUFU.RCP + 2 max per two pairs instead of 40 scalar instructions
                constexpr int NPK = NQ / 2;
                unsigned long long EP[NPK > 0 ? NPK : 1][9];
#pragma unroll
                for (int k = 0; k < NPK; ++k)
#pragma unroll
                    for (int e = 0; e < 9; ++e) EP[k][e] = pk2(E[2 * k][e], E[2 * k + 1][e]);
                const unsigned long long NFX = pk2(nfx, nfx), NFY = pk2(nfy, nfy), ONE = pk2(1.0f, 1.0f);
                int i = 0;
                for (int r = 0; r < n_runs; ++r) {
                    const int end = run_end[r];
                    const float bf = run_bf[r];
#pragma unroll
                    for (int q = 0; q < NQ; ++q) mx[q] = 0.f;
                    for (; i <= end; ++i) {
                        const float4 ra = rowsA[2 * i], rb = rowsA[2 * i + 1];
#pragma unroll
                        for (int k = 0; k < NPK; ++k) {
                            const unsigned long long X = pk2(ra.x, ra.x), Y = pk2(ra.y, ra.y), Z = pk2(ra.z, ra.z);
                            const unsigned long long g0 = fma2(EP[k][0], X, fma2(EP[k][1], Y, mul2(EP[k][2], Z)));   // D P
                            const unsigned long long g1 = fma2(EP[k][3], X, fma2(EP[k][4], Y, mul2(EP[k][5], Z)));
                            const unsigned long long g2 = fma2(EP[k][6], X, fma2(EP[k][7], Y, mul2(EP[k][8], Z)));
                            const unsigned long long q0 = fma2(pk2(ra.w, ra.w), g2, fma2(NFX, g0, pk2(rb.y, rb.y)));
                            const unsigned long long q1 = fma2(pk2(rb.x, rb.x), g2, fma2(NFY, g1, pk2(rb.z, rb.z)));
                            const unsigned long long p2 = fma2(g2, ONE, pk2(rb.w, rb.w));                            // rb.w + g2
                            float pl, ph, wl, wh;
                            upk2(p2, pl, ph);
                            asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(wl) : "f"(pl));
                            asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(wh) : "f"(ph));
                            const unsigned long long wr = pk2(wl, wh);
                            const unsigned long long val = mul2(fma2(q0, q0, mul2(q1, q1)), mul2(wr, wr));
                            float vl, vh;
                            upk2(val, vl, vh);
                            mx[2 * k] = fmaxf(mx[2 * k], vl);
                            mx[2 * k + 1] = fmaxf(mx[2 * k + 1], vh);
                        }
#pragma unroll
                        for (int q = 2 * NPK; q < NQ; ++q) {
                            const float g0 = fmaf(E[q][0], ra.x, fmaf(E[q][1], ra.y, E[q][2] * ra.z));   // D P
                            const float g1 = fmaf(E[q][3], ra.x, fmaf(E[q][4], ra.y, E[q][5] * ra.z));
                            const float g2 = fmaf(E[q][6], ra.x, fmaf(E[q][7], ra.y, E[q][8] * ra.z));
                            const float q0 = fmaf(ra.w, g2, fmaf(nfx, g0, rb.y));
                            const float q1 = fmaf(rb.x, g2, fmaf(nfy, g1, rb.z));
                            const float p2 = rb.w + g2;
                            float wr;
                            asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(wr) : "f"(p2));
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
            float myval;
            ranked = topk_certified<NQ>(dv, n_ps, uncA, (L.exact_only & 4) != 0, false, lane, candj, candd, myval);
            if (!ranked) {
                const ExactMarginTrans<RES> exact{ R, t, K, rows, n, rng, (uint32_t)s, L.theta_p };
                const int cnt = topk_fp64<NQ>(dv, n_p, n_ps, uncA, myval, (L.exact_only & 16) != 0, lane, dex, candj, candd, exact);
                if (stats) { stc[8] += 1; stc[0] += (unsigned long long)n * cnt; stc[2] += (unsigned long long)n * cnt; }
                ranked = true;
            }
        }
        if (!ranked) {
            const ExactMarginTrans<RES> exact{ R, t, K, rows, n, rng, (uint32_t)s, L.theta_p };
            float dummy[NQ];
#pragma unroll
            for (int q = 0; q < NQ; ++q) dummy[q] = 0.f;
            topk_fp64<NQ>(dummy, n_p, n_ps, 0.f, 0.f, true, lane, dex, candj, candd, exact);
            if (stats) { stc[0] += (unsigned long long)n * n_p; stc[2] += (unsigned long long)n * n_p; }
        }
        __syncwarp();
        int win = -1;
        double Rw[9];                                        // rotation of the winning candidate
        if (fast_ladder) {
            // ================================================== a5-a6, certified fp32 ladder (reprojection)
            if (lane < KP) {                                 // D = Exp(theta_p xi) - I of the kept perturbations, as in a2
                uint32_t o[4];
                philox4x32_10(rng.w_lo, (uint32_t)s, (uint32_t)candj[lane], 1u | rng.w_hi8, rng.k0, rng.k1, o);
                const float f0 = thpf * pm1f(o[0]), f1 = thpf * pm1f(o[1]), f2 = thpf * pm1f(o[2]);
                const float s0 = f0 * f0, s1 = f1 * f1, s2 = f2 * f2;
                const float th2 = s0 + s1 + s2;
                const float A = fmaf(th2, fmaf(th2, fmaf(th2, fmaf(th2, 2.7557319e-06f, -1.9841270e-04f), 8.3333333e-03f), -1.6666667e-01f), 1.0f);
                const float B = fmaf(th2, fmaf(th2, fmaf(th2, fmaf(th2, 2.7557319e-07f, -2.4801587e-05f), 1.3888889e-03f), -4.1666667e-02f), 0.5f);
                const float a0 = A * f0, a1 = A * f1, a2 = A * f2;
                float *d = Dc + 12 * lane;
                d[0] = -B * (s1 + s2);        d[1] = fmaf(B, f0 * f1, -a2); d[2] = fmaf(B, f0 * f2, a1);
                d[3] = fmaf(B, f0 * f1, a2);  d[4] = -B * (s0 + s2);        d[5] = fmaf(B, f1 * f2, -a0);
                d[6] = fmaf(B, f0 * f2, -a1); d[7] = fmaf(B, f1 * f2, a0);  d[8] = -B * (s0 + s1);
            }
            __syncwarp();
            for (int pi = lane; pi < KP * n; pi += 32) {    // cone rows of (candidate k, constraint i) at step 0
                const int k = divN.div(pi), i = pi - k * n;
                const float4 ra = rowsA[2 * i], rb = rowsA[2 * i + 1];
                const float *d = Dc + 12 * k;
                const float g0 = fmaf(d[0], ra.x, fmaf(d[1], ra.y, d[2] * ra.z));
                const float g1 = fmaf(d[3], ra.x, fmaf(d[4], ra.y, d[5] * ra.z));
                const float g2 = fmaf(d[6], ra.x, fmaf(d[7], ra.y, d[8] * ra.z));
                krow[i * KP + k] = make_float4(fmaf(ra.w, g2, fmaf(nfx, g0, rb.y)), fmaf(rb.x, g2, fmaf(nfy, g1, rb.z)),
                                       betaf[i] * (rb.w + g2), 0.f);
            }
            __syncwarp();
            for (int base = 0; base < items && win < 0; base += 32) {
                const int it = base + lane;
                bool dead = true, sure = false;
                int done = 0;
                {
                    // All lanes run the constraint loop (idle ones on item 0) so that the warp can leave it together: it starts
                    // at the constraint that is tightest at the current pose (i_tight, chosen at the set-up) and ends as soon as
                    // every candidate of the round is violated for sure -- a maximum only grows, so the rest cannot change that.
                    const bool act = it < items;
                    const int itc = act ? it : 0;
                    const int m = divKP.div(itc), k = itc - m * KP;
                    const float sm = sT[m];
                    float M = -CUDART_INF_F, Wmin = CUDART_INF_F;
                    int i = i_tight;
                    while (done < n) {
                        const float4 kr = krow[i * KP + k], cr = crow[i];          // [i][k]: lanes of a round differ in k
                        const float q0 = fmaf(sm, cr.x, kr.x), q1 = fmaf(sm, cr.y, kr.y), w = fmaf(sm, cr.z, kr.z);
                        M = fmaxf(M, fmaf(q0, q0, fmaf(q1, q1, fmaf(-w, w, cr.w))));
                        Wmin = fminf(Wmin, w);
                        ++done;
                        if (++i == n) i = 0;
                        if (__all_sync(FULL, !act || M > 0.f)) break;
                    }
                    // g32 - tau > 0: violated for sure (behind the camera counts as violated either way, R-10);
                    // satisfied for sure needs every g32 + tau <= 0 and beta p_3 > 0 beyond its error
                    if (act) {
                        dead = M > 0.f;
                        sure = (tauMax < CUDART_INF_F) && (M <= -2.0f * tauMax) && (Wmin > ewMax);
                        if (L.exact_only & 2) { dead = false; sure = false; }
                    }
                }
                if (stats) stc[7] += (unsigned long long)done * min(32, items - base);
                unsigned alive = __ballot_sync(FULL, !dead);
                const unsigned sures = __ballot_sync(FULL, sure);
                while (alive != 0u && win < 0) {             // in Alg. A8's order; undecided ones go to fp64
                    const int l = __ffs(alive) - 1;
                    alive &= alive - 1u;
                    const int itl = base + l;
                    const int m = divKP.div(itl), k = itl - m * KP;
                    double x, y, z, E[9];
                    rng.xi3((uint32_t)s, (uint32_t)candj[k], 1u, x, y, z);
                    exp_so3(L.theta_p * x, L.theta_p * y, L.theta_p * z, E);
                    mat3_mul(E, R, Rw);
                    bool ok = (sures >> l) & 1u;
                    if (!ok) {
                        double dT = 1.0;
                        for (int q = 0; q < m; ++q) dT = dT * L.gamma;
                        double tm[3];
                        tm[0] = __dadd_rn(t[0], __dmul_rn(dT, vel[0]));
                        tm[1] = __dadd_rn(t[1], __dmul_rn(dT, vel[1]));
                        tm[2] = __dadd_rn(t[2], __dmul_rn(dT, vel[2]));
                        unsigned long long pairs = 0;
                        ok = in_purse_direct<RES>(Rw, tm, rows, n, K, pairs);
                        if (stats) { stc[1] += pairs; stc[3] += pairs; stc[9] += 1; }
                    }
                    if (ok) win = itl;
                }
            }
        } else {
        if (lane < KP) {                                 // rotations of the kept perturbations
            double x, y, z, E[9], Rj[9];
            rng.xi3((uint32_t)s, (uint32_t)candj[lane], 1u, x, y, z);
            exp_so3(L.theta_p * x, L.theta_p * y, L.theta_p * z, E);
            mat3_mul(E, R, Rj);
#pragma unroll
            for (int e = 0; e < 9; ++e) Rc[lane * 9 + e] = Rj[e];
        }
        __syncwarp();

        // ================================================== a5-a6: ladder, first feasible candidate in (m, k) order
        for (int base = 0; base < items && win < 0; base += 32) {
            const int it = base + lane;
            bool ok = false;
            if (it < items) {
                const int m = divKP.div(it), k = it - m * KP;
                double dT = 1.0;
                for (int q = 0; q < m; ++q) dT = dT * L.gamma;          // dT_m = gamma^(m-1) by repeated multiplication
                double tm[3], Rj[9];
                tm[0] = __dadd_rn(t[0], __dmul_rn(dT, vel[0]));
                tm[1] = __dadd_rn(t[1], __dmul_rn(dT, vel[1]));
                tm[2] = __dadd_rn(t[2], __dmul_rn(dT, vel[2]));
#pragma unroll
                for (int e = 0; e < 9; ++e) Rj[e] = Rc[k * 9 + e];
                unsigned long long pairs = 0;
                ok = in_purse_direct<RES>(Rj, tm, rows, n, K, pairs);
                if (L.stats != nullptr) {
                    atomicAdd(&stc[1], pairs);
                    atomicAdd(&stc[3], pairs);
                }
            }
            const unsigned fm = __ballot_sync(FULL, ok);
            if (fm != 0u) win = base + __ffs(fm) - 1;
        }
        if (win >= 0) {
            const int k = win % KP;
#pragma unroll
            for (int e = 0; e < 9; ++e) Rw[e] = Rc[k * 9 + e];
        }
        }

        int m0 = 0, j_win = 0;
        if (win >= 0) {
            const int m = win / KP, k = win - m * KP;
            m0 = m + 1;
            j_win = candj[k];
            double dT = 1.0;
            for (int q = 0; q < m; ++q) dT = dT * L.gamma;
            t[0] = __dadd_rn(t[0], __dmul_rn(dT, vel[0]));
            t[1] = __dadd_rn(t[1], __dmul_rn(dT, vel[1]));
            t[2] = __dadd_rn(t[2], __dmul_rn(dT, vel[2]));
#pragma unroll
            for (int e = 0; e < 9; ++e) R[e] = Rw[e];
            if (stats) stc[4] += 1;
        }
        moved = (m0 != 0);
        if (m0 != 1) hit = true;                              // R-12 (R-11: nothing feasible -> unchanged)
        if (L.out_trace != nullptr && lane == 0)
            L.out_trace[((size_t)blockIdx.y * L.num_walkers + local) * L.num_steps + (s - 1)] = m0 | (j_win << 8);
        __syncwarp();                                         // Rc / candj readers done before the next step writes
    }

    // ---- a7: emit
    if (lane == 0) {
        const size_t o = (size_t)blockIdx.y * L.num_walkers + local;
        double2 *dst = reinterpret_cast<double2 *>(L.out_samples + 12 * o);
        dst[0] = make_double2(R[0], R[1]); dst[1] = make_double2(R[2], R[3]); dst[2] = make_double2(R[4], R[5]);
        dst[3] = make_double2(R[6], R[7]); dst[4] = make_double2(R[8], t[0]); dst[5] = make_double2(t[1], t[2]);
        L.out_flags[o] = hit ? 1 : 0;
        if (stats) {
            stc[5] = (unsigned long long)L.num_steps;
            for (int k = 0; k < kNumStats; ++k) atomicAdd(L.stats + k, stc[k]);
        }
    }
}

template <int RES, int NQ>
cudaError_t launch_q(const WalkLaunch &L, int n_instances, int max_rows_bytes, cudaStream_t stream)
{
    // the largest table of the batch bounds every instance's layout (an instance with fewer constraints needs at most as much)
    const int n_max = max_rows_bytes / (Res<RES>::ROW * 8);
    const long long kr = (long long)L.n_p_star * n_max;
    const TransSmem lay = trans_layout(max_rows_bytes, NQ, RES == CLOSURE_REPROJ_2D3D ? n_max : 0,
                                       (int)(kr < kKrowMax ? kr : kKrowMax), kTransWarps<RES>);
    if (lay.total > 200 * 1024) return cudaErrorInvalidConfiguration;
    cudaError_t e = cudaFuncSetAttribute(walker_coop_trans_kernel<RES, NQ>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)lay.total);
    if (e != cudaSuccess) return e;
    const long long blocks = (L.num_walkers + kTransWarps<RES> - 1) / kTransWarps<RES>;
    if (blocks > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    dim3 grid((unsigned)blocks, (unsigned)n_instances, 1);
    walker_coop_trans_kernel<RES, NQ><<<grid, 32 * kTransWarps<RES>, lay.total, stream>>>(L);
    return cudaGetLastError();
}

template <int RES>
cudaError_t launch_r(const WalkLaunch &L, int n_instances, int max_rows_bytes, cudaStream_t stream)
{
    if (L.n_p <= 32) return launch_q<RES, 1>(L, n_instances, max_rows_bytes, stream);
    if (L.n_p <= 64) return launch_q<RES, 2>(L, n_instances, max_rows_bytes, stream);
    if (L.n_p <= 160) return launch_q<RES, 5>(L, n_instances, max_rows_bytes, stream);
    return launch_q<RES, 8>(L, n_instances, max_rows_bytes, stream);
}

}  // namespace

cudaError_t launch_walkers_coop_trans(int residual_type, const WalkLaunch &L, int n_instances, int max_rows_bytes,
                                      cudaStream_t stream)
{
    switch (residual_type) {
    case CLOSURE_REG_3D3D: return launch_r<CLOSURE_REG_3D3D>(L, n_instances, max_rows_bytes, stream);
    case CLOSURE_REPROJ_2D3D: return launch_r<CLOSURE_REPROJ_2D3D>(L, n_instances, max_rows_bytes, stream);
    case CLOSURE_POSE_REG: return launch_r<CLOSURE_POSE_REG>(L, n_instances, max_rows_bytes, stream);
    case CLOSURE_POSE_REG_SPLIT: return launch_r<CLOSURE_POSE_REG_SPLIT>(L, n_instances, max_rows_bytes, stream);
    case CLOSURE_REG_3D3D_ELL: return launch_r<CLOSURE_REG_3D3D_ELL>(L, n_instances, max_rows_bytes, stream);
    case CLOSURE_REPROJ_2D3D_ELL: return launch_r<CLOSURE_REPROJ_2D3D_ELL>(L, n_instances, max_rows_bytes, stream);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace closure
