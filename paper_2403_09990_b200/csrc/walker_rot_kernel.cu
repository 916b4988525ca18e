// Fast walker kernel for the rotation-boundary sampler (Alg. 2) on the residuals
// whose squared norm is quadratic in the translation perturbation (Ex.2 registration, Ex.3 pose
// regression, stacked or split).  Same results as the plain fp64 kernel in walker_kernel.cu, bit
// for bit (tests/test_gpu_parity.py::test_screened_kernel_is_bit_identical_to_exact_kernel); what
// changes is WHERE the arithmetic runs:
//
//   * every (perturbation, constraint) and (ladder candidate, constraint) pair is first evaluated
//     in fp32 (3 FFMA + 1 FMNMX on the FP32/ALU pipes, 4x the FP64 pipe's rate) with a rigorous
//     error bound (DESIGN.md 6.1 "Screening");
//   * phase A (eq. (14) + top-N_P*): the fp32 values d~_j with uncertainty +-D select a short
//     candidate list (N_P* + 6 entries) that provably contains the exact top-N_P*; only those are
//     re-evaluated in fp64 and ranked by (d desc, j asc).  If the list cannot be proven complete
//     (near-ties, e.g. t_p = 0) the warp falls back to the exact evaluation of all N_P;
//   * phase B (ladder): a rung's candidates are tested leniently in fp32 (certainly-violated
//     candidates die); rungs on which some lane still has a survivor are re-run in fp64, so every
//     accept/reject decision is taken on fp64 values exactly as in the plain kernel.
#include <cuda_runtime.h>
#include <math_constants.h>
#include <stdint.h>

#include "closure_internal.h"
#include "walker_common.cuh"

namespace closure {
namespace {

constexpr int kJS = 20;   // fp32 screening tile (perturbations per register tile)
constexpr int kJE = 8;    // fp64 exact tile
constexpr float kMu20 = 9.5367431640625e-07f;   // 2^-20

// Philox4x32-10 for NJ counters that differ only in word 2 (= perturbation index), advanced round
// by round in a rolled loop: small code, NJ independent dependency chains.
template <int NJ>
__device__ __forceinline__ void philox_batch(const Rng &rng, uint32_t s, const int (&j)[NJ], uint32_t (&x)[NJ],
                                             uint32_t (&y)[NJ], uint32_t (&z)[NJ])
{
    uint32_t c0[NJ], c1[NJ], c2[NJ], c3[NJ];
#pragma unroll
    for (int q = 0; q < NJ; ++q) { c0[q] = rng.w_lo; c1[q] = s; c2[q] = (uint32_t)j[q]; c3[q] = 1u | rng.w_hi8; }
    uint32_t k0 = rng.k0, k1 = rng.k1;
#pragma unroll 1
    for (int r = 0; r < 10; ++r) {
#pragma unroll
        for (int q = 0; q < NJ; ++q) {
            const uint32_t hi0 = __umulhi(0xD2511F53u, c0[q]), lo0 = 0xD2511F53u * c0[q];
            const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2[q]), lo1 = 0xCD9E8D57u * c2[q];
            c0[q] = hi1 ^ c1[q] ^ k0;
            c1[q] = lo1;
            c2[q] = hi0 ^ c3[q] ^ k1;
            c3[q] = lo0;
        }
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
#pragma unroll
    for (int q = 0; q < NJ; ++q) { x[q] = c0[q]; y[q] = c1[q]; z[q] = c2[q]; }
}

// fp32 image of pm1(): |pm1f(x) - pm1(x)| <= 2^-22.
__device__ __forceinline__ float pm1f(uint32_t x)
{
    return fmaf((float)x, 4.656612873077392578125e-10f, 2.3283064365386962890625e-10f - 1.0f);
}

// Per-thread lists live in shared memory, slot-major ([slot][thread]: conflict-free, no
// synchronisation needed since a thread only touches its own column).  Keeping them out of the
// register file lets insertion be ONE rolled routine (the unrolled register version was ~60 % of the
// kernel's code and thrashed the instruction cache).

// Candidate list of phase A: the CAND largest screening values (descending) with their indices.
struct CandList {
    float *d;   // [CAND][kBlock]
    int *j;
    int cap;
    __device__ __forceinline__ float &D(int k) const { return d[k * kBlock]; }
    __device__ __forceinline__ int &J(int k) const { return j[k * kBlock]; }
    __device__ __forceinline__ void clear() const
    {
        for (int k = 0; k < cap; ++k) { D(k) = -CUDART_INF_F; J(k) = -1; }
    }
    __device__ __forceinline__ void insert(float dn, int jn) const
    {
        if (!(dn > D(cap - 1))) return;
        int k = cap - 1;
        while (k > 0 && dn > D(k - 1)) { D(k) = D(k - 1); J(k) = J(k - 1); --k; }
        D(k) = dn; J(k) = jn;
    }
};

// Top-N_P* list of the exact pass, ordered by (d descending, j ascending) (R-8).
struct TopList {
    double *d;  // [KCAP][kBlock]
    int *j;
    int cap;
    __device__ __forceinline__ double &D(int k) const { return d[k * kBlock]; }
    __device__ __forceinline__ int &J(int k) const { return j[k * kBlock]; }
    static __device__ __forceinline__ bool before(double da, int ja, double db, int jb)
    {
        return da > db || (da == db && ja < jb);
    }
    __device__ __forceinline__ void clear() const
    {
        for (int k = 0; k < cap; ++k) { D(k) = -CUDART_INF; J(k) = 0x7fffffff; }
    }
    __device__ __forceinline__ void insert(double dn, int jn) const
    {
        if (!before(dn, jn, D(cap - 1), J(cap - 1))) return;
        int k = cap - 1;
        while (k > 0 && before(dn, jn, D(k - 1), J(k - 1))) { D(k) = D(k - 1); J(k) = J(k - 1); --k; }
        D(k) = dn; J(k) = jn;
    }
};

// Exact (fp64) eq. (14) margins of NJ perturbations given by index: the arithmetic of the plain
// kernel's phase A, unchanged.  jv[q] < 0 marks an empty slot (its result is unused).
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

// fp32 set-up of one row for the screening passes: (u, c) rounded to fp32 and the bound eps on
// |v32 - v64| for ANY perturbation with |d_c| <= t_p, where v = c - 2 u.d:
// inputs carry relative error 2^-24 (u, c) and absolute error 6 * 2^-24 * 2 t_p (-2d, from pm1f),
// the three FFMA add 3 roundings  =>  |v32 - v64| <= 10 * 2^-24 * (|c| + 2 t_p |u|_1 + 3 t_p^2);
// eps uses 16 * 2^-24 = 2^-20 and a further 0.1 % for its own rounding.
__device__ __forceinline__ void screen_row(double u0, double u1, double u2, double c, float tp2, float tp2sq3,
                                           float &f0, float &f1, float &f2, float &fc, float &eps)
{
    f0 = (float)u0; f1 = (float)u1; f2 = (float)u2; fc = (float)c;
    const float mag = fabsf(fc) + tp2 * (fabsf(f0) + fabsf(f1) + fabsf(f2)) + tp2sq3;
    eps = mag * (kMu20 * 1.001f);
}

template <int RES, int KCAP, bool STATS>
__global__ void __launch_bounds__(kBlock, 2) walker_rot_kernel(const __grid_constant__ WalkLaunch L)
{
    using RS = Res<RES>;
    constexpr int ROW = RS::ROW;
    constexpr unsigned FULL = 0xffffffffu;
    constexpr int CAND = ((KCAP + 6 + kJE - 1) / kJE) * kJE;   // candidate list, a whole number of exact tiles

    extern __shared__ __align__(16) unsigned char smem_raw[];
    uint64_t *bar = reinterpret_cast<uint64_t *>(smem_raw);
    double *rows = reinterpret_cast<double *>(smem_raw + 16);
    const InstanceDesc *__restrict__ D = L.desc[blockIdx.y];
    const int n = D->n;
    const int rows_bytes = D->rows_bytes;
    stage_rows(smem_raw + 16, bar, D->rows, rows_bytes);
    unsigned char *sp = smem_raw + 16 + ((rows_bytes + 15) & ~15);
    double2 *ladder = reinterpret_cast<double2 *>(sp);
    sp += (size_t)L.n_t * kBlock * sizeof(double2);
    TopList top;
    top.cap = KCAP;
    top.d = reinterpret_cast<double *>(sp) + threadIdx.x;  sp += (size_t)KCAP * kBlock * sizeof(double);
    top.j = reinterpret_cast<int *>(sp) + threadIdx.x;     sp += (size_t)KCAP * kBlock * sizeof(int);
    CandList cl;
    cl.cap = CAND;
    cl.d = reinterpret_cast<float *>(sp) + threadIdx.x;    sp += (size_t)CAND * kBlock * sizeof(float);
    cl.j = reinterpret_cast<int *>(sp) + threadIdx.x;      sp += (size_t)CAND * kBlock * sizeof(int);
    double *scr_d = reinterpret_cast<double *>(sp) + threadIdx.x;    // [kJE][kBlock] exact tile results
    sp += (size_t)kJE * kBlock * sizeof(double);
    float *scr_f = reinterpret_cast<float *>(sp) + threadIdx.x;      // [kJS][kBlock] screening tile results
    // (separate regions: a thread's float column and another thread's double column would overlap)

    const long long local = (long long)blockIdx.x * kBlock + threadIdx.x;
    const bool valid = local < L.num_walkers;
    const unsigned long long w = (unsigned long long)(L.walker_begin + (valid ? local : L.num_walkers - 1));
    const unsigned long long seed = L.seed[blockIdx.y];
    Rng rng;
    rng.w_lo = (uint32_t)w;
    rng.w_hi8 = (uint32_t)(w >> 32) << 8;
    rng.k0 = (uint32_t)seed;
    rng.k1 = (uint32_t)(seed >> 32);

    double R[9], t[3], vel[3];
    init_walker<CLOSURE_MODE_ROT>(D, L, rng, w, R, t, vel);
    fill_ladder(L, vel, ladder);

    unsigned long long st_pp = 0, st_lp = 0, st_ps = 0, st_ls = 0, st_acc = 0, st_pp32 = 0, st_lp32 = 0, st_fb = 0,
                       st_vr = 0;
    bool hit = false;
    const int n_p = L.n_p, n_ps = L.n_p_star, n_t = L.n_t;
    const unsigned kmask = (1u << n_ps) - 1u;            // n_ps <= 20
    const double t_p = L.t_p;
    const float tpf = (float)t_p * 1.0000002f;          // >= t_p
    const float tp2 = 2.0f * tpf, tp2sq3 = 3.0f * tpf * tpf;
    const float m2tp = -2.0f * (float)t_p;

    for (int s = 1; s <= L.num_steps; ++s) {
        top.clear();

        double rot_margin = CUDART_INF;                 // POSE_REG_SPLIT: rotation bounds do not see d_j
        if (RES == CLOSURE_POSE_REG_SPLIT) {
            for (int i = 0; i < n; ++i) {
                const double *row = rows + i * ROW;
                rot_margin = dmin(rot_margin, row[12] - sqrt(frob_sq(R, row)));
            }
        }

        // ================================================== a2-a4, screening pass (fp32)
        bool complete = false;                          // candidate list proven to hold the exact top-KCAP
        cl.clear();
        if (n_p > CAND) {
            float unc = 0.0f;                           // uncertainty of d~ (max over this iteration)
            for (int j0 = 0; j0 < n_p; j0 += kJS) {
                int jv[kJS];
                uint32_t x[kJS], y[kJS], z[kJS];
#pragma unroll
                for (int q = 0; q < kJS; ++q) jv[q] = j0 + q;
                philox_batch<kJS>(rng, (uint32_t)s, jv, x, y, z);
                float e0[kJS], e1[kJS], e2[kJS], mx[kJS], dt[kJS];
#pragma unroll
                for (int q = 0; q < kJS; ++q) {
                    e0[q] = m2tp * pm1f(x[q]); e1[q] = m2tp * pm1f(y[q]); e2[q] = m2tp * pm1f(z[q]);
                    mx[q] = -CUDART_INF_F;
                    dt[q] = CUDART_INF_F;
                }
                float eps_run = 0.0f;
                for (int i = 0; i < n; ++i) {
                    const double *row = rows + i * ROW;
                    double u0, u1, u2, c;
                    affine_setup<RES>(R, t, row, u0, u1, u2, c);
                    float f0, f1, f2, fc, eps;
                    screen_row(u0, u1, u2, c, tp2, tp2sq3, f0, f1, f2, fc, eps);
                    eps_run = fmaxf(eps_run, eps);
#pragma unroll
                    for (int q = 0; q < kJS; ++q)
                        mx[q] = fmaxf(mx[q], fmaf(f0, e0[q], fmaf(f1, e1[q], fmaf(f2, e2[q], fc))));
                    const double beta = row[RS::BETA];
                    const bool run_ends = (i == n - 1) || (rows[(i + 1) * ROW + RS::BETA] != beta);
                    if (run_ends) {                     // warp-uniform
                        const float bf = (float)beta;
#pragma unroll
                        for (int q = 0; q < kJS; ++q) {
                            // a ~ max_i |u_i - d|^2, within eps_run + 2^-22 |a|
                            const float ddq = 0.25f * fmaf(e2[q], e2[q], fmaf(e1[q], e1[q], e0[q] * e0[q]));
                            const float a = fmaxf(mx[q] + ddq, 1e-30f);
                            const float r = rsqrtf(a);
                            const float sq = a * r;                       // sqrt(a) within 2^-21 relative
                            // |sqrt(A*) - sq| <= (eps_run + 2^-22 a) r + 2^-21 sq ; beta, subtraction: 2^-22 (beta + sq)
                            const float du = 1.01f * fmaf(eps_run, r, (bf + sq) * 1.9073486328125e-06f);
                            unc = fmaxf(unc, du);
                            dt[q] = fminf(dt[q], bf - sq);
                            mx[q] = -CUDART_INF_F;
                        }
                        eps_run = 0.0f;
                    }
                }
                if (STATS) { st_pp32 += (unsigned long long)n * kJS; st_ps += n; }
#pragma unroll
                for (int q = 0; q < kJS; ++q) scr_f[q * kBlock] = fminf(dt[q], (float)rot_margin);
                const int q_end = min(kJS, n_p - j0);
                for (int q = 0; q < q_end; ++q) cl.insert(scr_f[q * kBlock], j0 + q);     // one rolled copy
            }
            // exact d_j lies in [d~_j - unc', d~_j + unc'] for every j (unc' also covers the rounding of
            // rot_margin); the exact top-KCAP are inside the list if its last entry is separated from
            // the KCAP-th by more than 2 unc'.
            const float uncp = unc + 1.2e-7f * fabsf((float)rot_margin == CUDART_INF_F ? 0.0f : (float)rot_margin);
            complete = cl.D(CAND - 1) < cl.D(KCAP - 1) - 2.0f * uncp;
        }
        if (L.exact_only & 4) complete = false;          // debug: no screening of phase A
        complete = __all_sync(FULL, complete);

        // ================================================== a2-a4, exact pass (fp64)
        // One rolled loop: tiles of kJE indices taken from the candidate list, or 0..N_P-1 when the list
        // could not be proven complete.
        {
            const int total = complete ? CAND : n_p;
            for (int c0 = 0; c0 < total; c0 += kJE) {
                int jv[kJE];
                double d[kJE];
#pragma unroll
                for (int q = 0; q < kJE; ++q) jv[q] = complete ? cl.J(c0 + q) : (c0 + q < n_p ? c0 + q : -1);
                exact_margins<RES, kJE>(R, t, rows, n, rng, (uint32_t)s, t_p, rot_margin, jv, d);
#pragma unroll
                for (int q = 0; q < kJE; ++q) scr_d[q * kBlock] = d[q];
                for (int q = 0; q < kJE; ++q) {                                        // one rolled copy
                    const int jq = complete ? cl.J(c0 + q) : (c0 + q < n_p ? c0 + q : -1);
                    if (jq >= 0) top.insert(scr_d[q * kBlock], jq);
                }
                if (STATS) { st_pp += (unsigned long long)n * kJE; st_ps += n; }
            }
            if (STATS && !complete) ++st_fb;
        }

        // ================================================== a5-a6: ladder, first feasible rung
        int m0 = 0, j_win = 0;
        unsigned win = 0;
        float kf0[KCAP], kf1[KCAP], kf2[KCAP], kth[KCAP];    // fp32 image of the kept perturbations
        {
            int jv[KCAP];
            uint32_t x[KCAP], y[KCAP], z[KCAP];
#pragma unroll
            for (int k = 0; k < KCAP; ++k) jv[k] = top.J(k);
            philox_batch<KCAP>(rng, (uint32_t)s, jv, x, y, z);
#pragma unroll
            for (int k = 0; k < KCAP; ++k) {
                const double d0 = t_p * pm1(x[k]), d1 = t_p * pm1(y[k]), d2 = t_p * pm1(z[k]);
                kf0[k] = (float)(-2.0 * d0); kf1[k] = (float)(-2.0 * d1); kf2[k] = (float)(-2.0 * d2);
                kth[k] = (float)(-fma(d2, d2, fma(d1, d1, d0 * d0)));
            }
        }
        for (int m = 0; m < n_t; ++m) {
            if (!__any_sync(FULL, m0 == 0)) break;
            const double2 ab = ladder[m * kBlock + threadIdx.x];
            double Rm[9];
            rotate_left(R, vel[0], vel[1], vel[2], ab.x, ab.y, Rm);
            const bool act = (m0 == 0);
            // ---- lenient fp32 pass: a candidate survives unless it is violated beyond the error bound
            float M[KCAP];
#pragma unroll
            for (int k = 0; k < KCAP; ++k) M[k] = -CUDART_INF_F;
            bool rot_dead = false;
            unsigned alive = act ? kmask : 0u;
            int i = 0;
            for (; i < n; ++i) {
                const double *row = rows + i * ROW;
                double u0, u1, u2, c;
                affine_setup<RES>(Rm, t, row, u0, u1, u2, c);
                if (RES == CLOSURE_POSE_REG_SPLIT) {
                    if (!(frob_sq(Rm, row) <= row[13])) rot_dead = true;      // exact: no perturbation involved
                }
                float f0, f1, f2, fcb, eps;
                screen_row(u0, u1, u2, c - row[RS::BETA + 1], tp2, tp2sq3, f0, f1, f2, fcb, eps);
                const float cbl = fcb - eps;
#pragma unroll
                for (int k = 0; k < KCAP; ++k)
                    M[k] = fmaxf(M[k], fmaf(f0, kf0[k], fmaf(f1, kf1[k], fmaf(f2, kf2[k], cbl))));
                if (i < 3 || (i & 3) == 3 || i == n - 1) {                   // warp-uniform
                    unsigned a2 = 0u;
#pragma unroll
                    for (int k = 0; k < KCAP; ++k)
                        if (!(M[k] > kth[k])) a2 |= 1u << k;
                    if (L.exact_only & 2) a2 = kmask;             // debug: lenient pass kills nothing
                    alive = (act && !rot_dead) ? (a2 & kmask) : 0u;
                    if (!__any_sync(FULL, alive != 0u)) { ++i; break; }
                }
            }
            if (STATS) { st_lp32 += (unsigned long long)i * n_ps; st_ls += i; }
            // ---- exact fp64 pass over the rung if any lane has a survivor (same arithmetic as the plain kernel)
            if (__any_sync(FULL, alive != 0u)) {
                double k0[KCAP], k1[KCAP], k2[KCAP], kdd[KCAP];
                {
                    int jv[KCAP];
                    uint32_t x[KCAP], y[KCAP], z[KCAP];
#pragma unroll
                    for (int k = 0; k < KCAP; ++k) jv[k] = top.J(k);
                    philox_batch<KCAP>(rng, (uint32_t)s, jv, x, y, z);
#pragma unroll
                    for (int k = 0; k < KCAP; ++k) {
                        const double d0 = t_p * pm1(x[k]), d1 = t_p * pm1(y[k]), d2 = t_p * pm1(z[k]);
                        kdd[k] = -fma(d2, d2, fma(d1, d1, d0 * d0));
                        k0[k] = -2.0 * d0; k1[k] = -2.0 * d1; k2[k] = -2.0 * d2;
                    }
                }
                int i2 = 0;
                for (; i2 < n; ++i2) {
                    const double *row = rows + i2 * ROW;
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
                    if (!__any_sync(FULL, alive != 0u)) { ++i2; break; }
                }
                if (STATS) { st_lp += (unsigned long long)i2 * n_ps; st_ls += i2; ++st_vr; }
            }
            if (alive) { m0 = m + 1; win = alive; }
        }
        if (m0) {
            const int kw = __ffs(win) - 1;                    // lowest rank among the feasible (R-8)
            const int jw = top.J(kw);
            j_win = jw;
            const double2 ab = ladder[(m0 - 1) * kBlock + threadIdx.x];
            double Rm[9];
            rotate_left(R, vel[0], vel[1], vel[2], ab.x, ab.y, Rm);
#pragma unroll
            for (int e = 0; e < 9; ++e) R[e] = Rm[e];
            double x, y, z;
            rng.xi3((uint32_t)s, (uint32_t)jw, 1u, x, y, z);
            t[0] = __dadd_rn(t[0], __dmul_rn(t_p, x));
            t[1] = __dadd_rn(t[1], __dmul_rn(t_p, y));
            t[2] = __dadd_rn(t[2], __dmul_rn(t_p, z));
        }
        if (m0 != 1) hit = true;                              // R-12 (R-11: nothing feasible -> unchanged)
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
        atomicAdd(L.stats + 6, st_pp32); atomicAdd(L.stats + 7, st_lp32);
        atomicAdd(L.stats + 8, st_fb); atomicAdd(L.stats + 9, st_vr);
    }
}

template <int RES, int KCAP>
cudaError_t launch_k(bool stats, const WalkLaunch &L, dim3 grid, int max_rows_bytes, cudaStream_t stream)
{
    constexpr int CAND = ((KCAP + 6 + kJE - 1) / kJE) * kJE;
    constexpr size_t scratch = kJS * sizeof(float) + kJE * sizeof(double);
    const size_t smem = 16 + (size_t)((max_rows_bytes + 15) & ~15) +
                        (size_t)kBlock * ((size_t)L.n_t * sizeof(double2) + KCAP * 12 + CAND * 8 + scratch);
    if (smem > 220 * 1024) return cudaErrorInvalidValue;
    cudaError_t e;
    if (stats) {
        e = cudaFuncSetAttribute(walker_rot_kernel<RES, KCAP, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        walker_rot_kernel<RES, KCAP, true><<<grid, kBlock, smem, stream>>>(L);
    } else {
        e = cudaFuncSetAttribute(walker_rot_kernel<RES, KCAP, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        walker_rot_kernel<RES, KCAP, false><<<grid, kBlock, smem, stream>>>(L);
    }
    return cudaGetLastError();
}

template <int RES>
cudaError_t launch_r(bool stats, const WalkLaunch &L, dim3 grid, int max_rows_bytes, cudaStream_t stream)
{
    if (L.n_p_star <= 2) return launch_k<RES, 2>(stats, L, grid, max_rows_bytes, stream);
    if (L.n_p_star <= 10) return launch_k<RES, 10>(stats, L, grid, max_rows_bytes, stream);
    return launch_k<RES, kMaxKStar>(stats, L, grid, max_rows_bytes, stream);
}

}  // namespace

bool rot_fast_path_available(int residual_type, int mode)
{
    return mode == CLOSURE_MODE_ROT && residual_type != CLOSURE_REPROJ_2D3D;
}

cudaError_t launch_walkers_rot_fast(int residual_type, bool stats, const WalkLaunch &L, dim3 grid,
                                    int max_rows_bytes, cudaStream_t stream)
{
    switch (residual_type) {
    case CLOSURE_REG_3D3D: return launch_r<CLOSURE_REG_3D3D>(stats, L, grid, max_rows_bytes, stream);
    case CLOSURE_POSE_REG: return launch_r<CLOSURE_POSE_REG>(stats, L, grid, max_rows_bytes, stream);
    case CLOSURE_POSE_REG_SPLIT: return launch_r<CLOSURE_POSE_REG_SPLIT>(stats, L, grid, max_rows_bytes, stream);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace closure
