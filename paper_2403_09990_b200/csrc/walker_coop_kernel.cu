// Warp-cooperative walker kernel for the rotation-boundary sampler (Alg. 2) on
// the residuals whose squared norm is quadratic in the translation perturbation (Ex.2 registration,
// Ex.3 pose regression, stacked or split).  One WARP owns one walker; the 32 lanes split the work
// that Alg. 3 tensorises per walker.  Per iteration:
//
//   a2     the N_P perturbations are dealt to the lanes (j = lane + 32 q), Philox4x32-10 per perturbation.
//   a3/a4  eq. (14) and the top-N_P* by exact branch and bound:
//            phase 1  every perturbation against the few constraints that are tightest at the current pose
//                     (a max over a subset is a lower bound of the max over all: an UPPER bound ub_j of d_j);
//            select   a threshold U with N_P*+2 <= #{ub_j >= U} <= 32 is found by probing counts (warp sums);
//                     no perturbation below U can be among the N_P* best once N_P* exact values above U exist;
//            phase 2  only the survivors are evaluated against all N constraints, lane = (survivor, chunk of
//                     the table); they are ranked by counting, and the ranking is CERTIFIED iff consecutive
//                     values (and the N_P*-th against both the next one and U) are more than 2 unc apart,
//                     unc being a rigorous bound on |fp32 - fp64|.  Otherwise the step falls back to the fp64
//                     evaluation of the plain kernel.
//          A pair costs 3 FFMA + 1 FMNMX in fp32 (packed FFMA2 + FMNMX3 in SASS); the per-constraint set-up
//          u_i = b_i - (R* a_i + t*) is computed ONCE per accepted move and kept in shared memory.
//   a5-a6  rungs are screened first, lane = (rung, candidate), against two tight constraint rows per rung
//          and against a Lipschitz bound on what the rotation to R_m can repair; rungs with a surviving
//          candidate are then evaluated in full, lane = (candidate, constraint chunk), in fp32 with a
//          three-way outcome per candidate: violated for sure / satisfied for sure / undecided -> fp64.
//
// Every accept/reject decision is therefore the decision the fp64 arithmetic of walker_kernel.cu
// takes (DESIGN.md 6.1b "Certified fp32 evaluation"); the pose itself is only ever updated in fp64.
#include <cuda_runtime.h>
#include <math_constants.h>
#include <stdint.h>

#include "closure_internal.h"
#include "walker_common.cuh"
#include "walker_coop_common.cuh"

#ifndef CLOSURE_COOP_MIN_CTAS
#define CLOSURE_COOP_MIN_CTAS 4   // resident CTAs per SM the register allocation aims at (128 registers per thread)
#endif

#ifndef CLOSURE_NEED_EXTRA
#define CLOSURE_NEED_EXTRA 3   // the threshold keeps at least N_P* + this many perturbations
#define CLOSURE_RT_EXTRA 3     // the next threshold is the value ranked N_P* + this + (N_P* >> CLOSURE_RT_SHIFT)
#define CLOSURE_RT_SHIFT 2
#endif

namespace closure {
namespace {

// Resident CTAs per SM the register allocation aims at.  Only NQ = 1 (N_P <= 32) is built from this file; the table of a
// C5-sized instance allows four CTAs of four warps anyway.
template <int RES, int NQ> constexpr int coop_min_ctas()
{
    return CLOSURE_COOP_MIN_CTAS;      // 128 registers: measured at 3 / 4 / 5 on config 5 (672 / 777 / 587 M walker-steps/s)
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

// ---------------------------------------------------------------------------------- shared-memory layout
constexpr int kTight = 8;     // constraints of the phase-1 table (the tightest of eight strided groups at the current pose)
constexpr int kCset = 16;     // constraints the rung-screening rows are picked from (kTight + the tightest at a middle rung)

struct AffSmem {
    size_t run_end, run_bf, run_pend, pos, warp0, per_warp;
    size_t rowsA, rowsL, pert, ab, qrow, RmS, dex, qL, total;
};

// Per-warp block: the small fixed-size arrays first, at compile-time offsets from the warp's base (the per-iteration
// code addresses them without keeping pointers in registers), then the arrays sized by NQ, then those sized by the
// instance (rowsA first: its offset is still a constant).
constexpr size_t kOffCand4 = 0;                       // 32 x float4: the kept perturbations (-2 d_j, -|d_j|^2), by rank
constexpr size_t kOffCandj = kOffCand4 + 32 * 16;     // 32 x int
constexpr size_t kOffCandd = kOffCandj + 32 * 4;      // 32 x float: upper bounds of the candidates' eq. (14) values
constexpr size_t kOffVals = kOffCandd + 32 * 4;       // 32 x float: the N_P* + 1 largest eq. (14) values, by rank
constexpr size_t kOffSjv = kOffVals + 32 * 4;         // 32 x (int, float): survivors of the threshold (index, phase-1 value)
constexpr size_t kOffRowsT = kOffSjv + 32 * 8;        // kTight x 32 B
constexpr size_t kOffRunTp = kOffRowsT + (size_t)kTight * 32;
constexpr size_t kOffRunTb = kOffRunTp + (size_t)kTight * 4;
constexpr size_t kOffCset = kOffRunTb + (size_t)kTight * 4;
constexpr size_t kOffPose = kOffCset + (size_t)kCset * 4;   // 20 doubles: R*(9) t*(3) omega(3) + set-up results
constexpr size_t kOffStc = kOffPose + 20 * 8;               // 16 counters
constexpr size_t kOffPert = kOffStc + 16 * 8;               // NQ x 32 x float4
__host__ __device__ constexpr size_t aff_off_dex(int nq) { return kOffPert + (size_t)nq * 32 * 16; }    // NQ x 32 doubles
__host__ __device__ constexpr size_t aff_off_rowsA(int nq) { return aff_off_dex(nq) + (size_t)nq * 32 * 8; }
static_assert(kOffPose % 16 == 0 && kOffPert % 16 == 0 && kOffRowsT % 16 == 0, "alignment of the per-warp block");

// pairs = 32-byte entries of rowsA (pair-entries, runs padded to even length)
__host__ __device__ inline AffSmem aff_layout(int rows_bytes, int n, int n_t, int nq, int pairs, int warps = kCoopWarps)
{
    AffSmem s;
    size_t o = 16 + (size_t)((rows_bytes + 15) & ~15);
    s.run_end = o; o += (size_t)((n * 4 + 15) & ~15);
    s.run_bf = o;  o += (size_t)((n * 4 + 15) & ~15);
    s.run_pend = o; o += (size_t)((n * 4 + 15) & ~15);
    s.pos = o;     o += (size_t)((n * 4 + 15) & ~15);
    s.warp0 = o;
    s.pert = kOffPert;
    s.dex = aff_off_dex(nq);
    size_t w = aff_off_rowsA(nq);
    s.rowsA = w; w += (size_t)pairs * 32;          // pair-transposed, runs padded to even length
    s.rowsL = w; w += (size_t)n * 16;
    s.qrow = w;  w += (size_t)n_t * 32;
    s.RmS = w;   w += (size_t)((n_t * 72 + 15) & ~15);
    s.ab = w;    w += (size_t)n_t * 16;
    s.qL = w;    w += (size_t)((n_t * 4 + 15) & ~15);
    s.per_warp = w;
    s.total = o + (size_t)warps * w;
    return s;
}

// ---------------------------------------------------------------------------------- set-up after a move
// Everything that depends on the pose only (DESIGN.md 6.1c "state that only changes on an accepted move"):
//   rowsA   fp32 set-up rows at R* for all N constraints (fp64 set-up, then rounded: the cancellation in
//           b - (R a + t) is taken in fp64);
//   rowsT   the phase-1 table: the tightest constraint of each of eight strided groups of rows, as pair-entries
//           grouped by runs of equal bound (any choice of rows is valid: a subset gives an upper bound);
//   RmS     Exp(dT_m w) R* for every rung;
//   qrow    per rung the two tightest rows among kCset candidate constraints (the kTight above and the tightest
//           of each group at a middle rung) -- screening rows; any choice is valid, a violated row kills.
// fp64-heavy and rare, so it is kept out of line.  Results epsA, rot_margin, the number of runs of rowsT
// -> pose[16], pose[15], pose[17].  full_p1: the table is short, phase 1 runs on all of it and rowsT is not built.
template <int RES>
__device__ __noinline__ void aff_setup_on_move(unsigned char *smem_raw, int warp, int lane, int rows_bytes, int n,
                                               int n_t, int nq, int pairs, double t_p, bool full_p1, bool stats)
{
    using RS = Res<RES>;
    constexpr int ROW = RS::ROW;
    const AffSmem lay = aff_layout(rows_bytes, n, n_t, nq, pairs);
    const double *rows = reinterpret_cast<const double *>(smem_raw + 16);
    const int *pos = reinterpret_cast<const int *>(smem_raw + lay.pos);
    unsigned char *wp = smem_raw + lay.warp0 + (size_t)warp * lay.per_warp;
    float *rowsA = reinterpret_cast<float *>(wp + lay.rowsA);
    float *rowsT = reinterpret_cast<float *>(wp + kOffRowsT);
    int *runT_pend = reinterpret_cast<int *>(wp + kOffRunTp);
    float *runT_bf = reinterpret_cast<float *>(wp + kOffRunTb);
    int *cset = reinterpret_cast<int *>(wp + kOffCset);
    const double2 *ab = reinterpret_cast<const double2 *>(wp + lay.ab);
    float4 *qrow = reinterpret_cast<float4 *>(wp + lay.qrow);
    double *RmS = reinterpret_cast<double *>(wp + lay.RmS);
    double *pose = reinterpret_cast<double *>(wp + kOffPose);
    unsigned long long *stc = reinterpret_cast<unsigned long long *>(wp + kOffStc);
    const float tpf = (float)t_p * 1.0000002f;          // >= t_p
    const float tp2 = 2.0f * tpf, tp2sq3 = 3.0f * tpf * tpf;
    double R[9], t[3], vel[3];
#pragma unroll
    for (int e = 0; e < 9; ++e) R[e] = pose[e];
#pragma unroll
    for (int e = 0; e < 3; ++e) { t[e] = pose[9 + e]; vel[e] = pose[12 + e]; }

    // Exp(dT_m w) R* for every rung
    for (int m = lane; m < n_t; m += 32) {
        const double2 c2 = ab[m];
        double Rm[9];
        rotate_left(R, vel[0], vel[1], vel[2], c2.x, c2.y, Rm);
#pragma unroll
        for (int e = 0; e < 9; ++e) RmS[m * 9 + e] = Rm[e];
    }
    __syncwarp();
    const int m_mid = min(n_t - 1, 4);                  // middle rung whose tight rows join the screening candidates
    double Rq[9];
#pragma unroll
    for (int e = 0; e < 9; ++e) Rq[e] = RmS[m_mid * 9 + e];

    const float velf0 = (float)vel[0], velf1 = (float)vel[1], velf2 = (float)vel[2];
    float eps_l = 0.f;
    double rm_l = CUDART_INF;
    uint32_t best1 = 0u, best2 = 0u;                    // (20 key bits | row index): tightest row of this lane at R*, at R_mid
#pragma unroll 1
    for (int i = lane; i < n; i += 32) {
        const double *row = rows + i * ROW;
        double u0, u1, u2, c;
        affine_setup<RES>(R, t, row, u0, u1, u2, c);
        float f0, f1, f2, fc, eps;
        screen_row(u0, u1, u2, c, tp2, tp2sq3, f0, f1, f2, fc, eps);
        {
            const int pp = pos[i], p = pp & 0x3fffffff;
            float *A = rowsA + (p >> 1) * 8 + (p & 1);
            A[0] = f0; A[2] = f1; A[4] = f2; A[6] = fc;
            if (pp & 0x40000000) { A[1] = f0; A[3] = f1; A[5] = f2; A[7] = fc; }
        }
        eps_l = fmaxf(eps_l, eps);
        const float bfi = (float)row[RS::BETA];
        float tk1 = sqrtf(fmaxf(fc, 0.f)) - bfi;         // larger = tighter (heuristic key only)
        if (RES == CLOSURE_POSE_REG_SPLIT) {
            const double rmi = row[12] - sqrt(frob_sq(R, row));
            rm_l = dmin(rm_l, rmi);
            tk1 = fmaxf(tk1, -(float)rmi);
        }
        float tk2;
        if (RES == CLOSURE_REG_3D3D) {
            // lever arm of R* a_i about the rotation axis, relative to the bound: a rotation by any angle moves this
            // constraint's centre by 2 sin(angle / 2) times it, so these rows are the first to be violated at the large rungs
            const float r0 = (float)(row[3] - t[0] - u0), r1 = (float)(row[4] - t[1] - u1), r2 = (float)(row[5] - t[2] - u2);
            const float x0 = velf1 * r2 - velf2 * r1, x1 = velf2 * r0 - velf0 * r2, x2 = velf0 * r1 - velf1 * r0;
            tk2 = sqrtf(fmaf(x2, x2, fmaf(x1, x1, x0 * x0))) / bfi;
        } else {
            double v0, v1, v2, cq;
            affine_setup<RES>(Rq, t, row, v0, v1, v2, cq);
            tk2 = sqrtf(fmaxf((float)cq, 0.f)) - bfi;
            if (RES == CLOSURE_POSE_REG_SPLIT) tk2 = fmaxf(tk2, sqrtf((float)frob_sq(Rq, row)) - (float)row[12]);
        }
        best1 = max(best1, (fkey(tk1) & 0xFFFFF000u) | (uint32_t)i);
        best2 = max(best2, (fkey(tk2) & 0xFFFFF000u) | (uint32_t)i);
    }
    const float epsA = wmax_nonneg(eps_l);
    double rot_margin = CUDART_INF;
    if (RES == CLOSURE_POSE_REG_SPLIT) rot_margin = wmin_f64(rm_l);
    // the tightest row of each group of four lanes (rows i with (i mod 32) / 4 = g)
    best1 = max(best1, __shfl_xor_sync(FULL, best1, 1)); best1 = max(best1, __shfl_xor_sync(FULL, best1, 2));
    best2 = max(best2, __shfl_xor_sync(FULL, best2, 1)); best2 = max(best2, __shfl_xor_sync(FULL, best2, 2));
    const int g8 = lane & 7;
    const int idx1 = (int)(__shfl_sync(FULL, best1, g8 * 4) & 0xFFFu);
    const int idx2 = (int)(__shfl_sync(FULL, best2, g8 * 4) & 0xFFFu);
    if (lane < 8) cset[kTight + lane] = idx2;
    // sort the eight tight rows by index (= by bound: rows are sorted by bound), lane r < 8 takes the r-th
    int rank = 0;
#pragma unroll
    for (int r = 0; r < 8; ++r) {
        const int o = __shfl_sync(FULL, idx1, r);
        rank += (o < idx1 || (o == idx1 && r < g8)) ? 1 : 0;
    }
    if (lane < 8) cset[rank] = idx1;
    __syncwarp();                                        // rowsA and cset[] are complete
    int nT_runs = 0;
    if (!full_p1) {
        const int myi = cset[g8];
        const double myb = rows[myi * ROW + RS::BETA];
        int p = 0, myp = 0;
        bool mydup = false;
        double prev = __shfl_sync(FULL, myb, 0);
#pragma unroll
        for (int r = 0; r < 8; ++r) {
            const double br = __shfl_sync(FULL, myb, r);
            if (r > 0 && br != prev) {                   // close the run: odd length repeats its last row
                if (p & 1) { if (lane == r - 1) mydup = true; ++p; }
                if (lane == 0) { runT_pend[nT_runs] = p >> 1; runT_bf[nT_runs] = (float)prev; }
                ++nT_runs;
                prev = br;
            }
            if (lane == r) myp = p;
            ++p;
        }
        if (p & 1) { if (lane == 7) mydup = true; ++p; }
        if (lane == 0) { runT_pend[nT_runs] = p >> 1; runT_bf[nT_runs] = (float)prev; }
        ++nT_runs;
        if (lane < 8) {
            const int sp = pos[myi] & 0x3fffffff;
            const float *S = rowsA + (sp >> 1) * 8 + (sp & 1);
            float *T = rowsT + (myp >> 1) * 8 + (myp & 1);
            const float a0 = S[0], a1 = S[2], a2 = S[4], a3 = S[6];
            T[0] = a0; T[2] = a1; T[4] = a2; T[6] = a3;
            if (mydup) { T[1] = a0; T[3] = a1; T[5] = a2; T[7] = a3; }
        }
    }
    // screening rows of every rung: lane = (rung, candidate constraint), two rungs per pass
    {
        const int c = lane & 15;
        const int ci = cset[c];
        const double *row = rows + ci * ROW;
        const unsigned hm = 0xFFFFu << (lane & 16);
#pragma unroll 1
        for (int m = lane >> 4; m < n_t; m += 2) {
            double Rm[9];
#pragma unroll
            for (int e = 0; e < 9; ++e) Rm[e] = RmS[m * 9 + e];
            double u0, u1, u2, cc;
            affine_setup<RES>(Rm, t, row, u0, u1, u2, cc);
            bool rdead = false;
            if (RES == CLOSURE_POSE_REG_SPLIT) rdead = !(frob_sq(Rm, row) <= row[13]);   // exact: a violated constraint kills the rung
            float g0, g1, g2, fcb, eps;
            screen_row(u0, u1, u2, cc - row[RS::BETA + 1], tp2, tp2sq3, g0, g1, g2, fcb, eps);
            float4 r4 = make_float4(g0, g1, g2, fcb - eps);
            const uint32_t key = (fkey(r4.w) & ~15u) | (uint32_t)c;
            uint32_t m1, m2;
            float unused;
            group_top2_max(hm, 16, key, 0.f, m1, m2, unused);
            const uint32_t key2 = (key == m1) ? 0u : key;
            if (RES == CLOSURE_POSE_REG_SPLIT) {
                if ((__ballot_sync(hm, rdead) & hm) != 0u) r4.w = CUDART_INF_F;       // rung dead for every candidate
            }
            if (key == m1) qrow[2 * m] = r4;
            if (key2 == m2) qrow[2 * m + 1] = r4;        // key2 = 0 for the winner only (keys of the others carry c != its c or are larger)
        }
    }
    if (stats) { stc[2] += 2 * n; stc[3] += (unsigned long long)kCset * n_t; }
    if (lane == 0) { pose[15] = rot_margin; pose[16] = (double)epsA; pose[17] = (double)nT_runs; }
    __syncwarp();
}

// ---------------------------------------------------------------------------------- eq. (14), perturbation-major
// NQ perturbations per lane in registers (packed pairs + an odd slot) against a table of pair-entries
// (two constraints per 32-byte entry) organised in runs of equal bound: per perturbation the maximum over the
// run's constraints of c - 2 u.d, one rsqrt per run.  dt[q] = min over runs of beta - sqrt(max + |d|^2);
// unc_l accumulates the bound on |dt - fp64|.
template <int NQ>
__device__ __forceinline__ void eq14_table(const float4 *tab, int n_runs, const int *rpend, const float *rbf,
                                           const unsigned long long (&p0)[NQ / 2 > 0 ? NQ / 2 : 1],
                                           const unsigned long long (&p1)[NQ / 2 > 0 ? NQ / 2 : 1],
                                           const unsigned long long (&p2)[NQ / 2 > 0 ? NQ / 2 : 1], float o0, float o1,
                                           float o2, const float (&dd)[NQ], float E0, float (&dt)[NQ], float &unc_l)
{
    constexpr int NPK = NQ / 2;
    constexpr bool ODD = (NQ & 1) != 0;
#pragma unroll
    for (int q = 0; q < NQ; ++q) dt[q] = CUDART_INF_F;
    int pp = 0;
    for (int r = 0; r < n_runs; ++r) {
        const int pend = rpend[r];
        const float bf = rbf[r];
        float mx[NQ];
#pragma unroll
        for (int q = 0; q < NQ; ++q) mx[q] = -CUDART_INF_F;
#pragma unroll(NQ <= 2 ? 4 : 1)   // measured: unrolling the NQ = 5 body further costs 2-4 % (C2, C4)
        for (; pp < pend; ++pp) {
            // two constraints a, b per entry: X = (f0a f0b f1a f1b), Y = (f2a f2b fca fcb)
            const float4 X = tab[2 * pp], Y = tab[2 * pp + 1];
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
}

// ---------------------------------------------------------------------------------- the kernel
template <int RES, int NQ>
__global__ void __launch_bounds__(kCoopThreads, coop_min_ctas<RES, NQ>()) walker_coop_kernel(const __grid_constant__ WalkLaunch L)
{
    using RS = Res<RES>;
    constexpr int ROW = RS::ROW;
    constexpr int NPK = NQ / 2;            // packed pairs of perturbations
    constexpr int NPK1 = NPK > 0 ? NPK : 1;
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
    // re-derives them from special registers, the constant bank and shared memory inside the loop (measured: ~10 % of
    // the executed instructions) instead of keeping them in a register.
#define CLOSURE_PIN_R(x) asm volatile("" : "+r"(x))
#define CLOSURE_PIN_F(x) asm volatile("" : "+f"(x))
    CLOSURE_PIN_R(lane); CLOSURE_PIN_R(n_p); CLOSURE_PIN_R(n_ps); CLOSURE_PIN_R(n_t);
    uint64_t *bar = reinterpret_cast<uint64_t *>(smem_raw);
    double *rows = reinterpret_cast<double *>(smem_raw + 16);
    stage_rows(smem_raw + 16, bar, D->rows, rows_bytes);                        // a0 (TMA bulk copy)
    const AffSmem lay = aff_layout(rows_bytes, n, n_t, NQ, L.pairs_cap);
    int *run_end = reinterpret_cast<int *>(smem_raw + lay.run_end);
    float *run_bf = reinterpret_cast<float *>(smem_raw + lay.run_bf);
    int *run_pend = reinterpret_cast<int *>(smem_raw + lay.run_pend);   // end of run r in rowsA, in PAIRS of rows
    int *pos = reinterpret_cast<int *>(smem_raw + lay.pos);             // row of constraint i in rowsA (bit 30: write it twice)
    if (warp == 0) {                                   // runs of equal bounds (rows are sorted by bound)
        int cnt = 0;
        float am = 0.f;
        for (int base = 0; base < n; base += 32) {
            const int i = base + lane;
            bool end = false;
            double beta = 0.0;
            if (i < n) {
                beta = rows[i * ROW + RS::BETA];
                end = (i == n - 1) || (rows[(i + 1) * ROW + RS::BETA] != beta);
                if (RES == CLOSURE_REG_3D3D) {
                    const double a0 = rows[i * ROW], a1 = rows[i * ROW + 1], a2 = rows[i * ROW + 2];
                    am = fmaxf(am, (float)sqrt(a0 * a0 + a1 * a1 + a2 * a2) * 1.000001f);
                }
            }
            const unsigned m = __ballot_sync(FULL, end);
            if (end) {
                const int r = cnt + __popc(m & ((1u << lane) - 1u));
                run_end[r] = i;
                run_bf[r] = (float)beta;
            }
            cnt += __popc(m);
        }
        // Lipschitz constant of the residual norms in the rotation: ||(R' - R) a_i|| <= angle * max_i ||a_i|| (Ex.2);
        // ||R' - R||_F <= sqrt(2) angle (Ex.3)
        am = (RES == CLOSURE_REG_3D3D) ? wmax_nonneg(am) : 1.4142137f;
        __syncwarp();
        if (lane == 0) {
            // rowsA holds the fp32 set-ups two constraints per entry; a run of odd length repeats its last
            // constraint (a maximum does not see duplicates), so no pair straddles two bounds
            n_runs_s = cnt;
            amax_s = am;
            int p = 0, start = 0;
            for (int r = 0; r < cnt; ++r) {
                const int end = run_end[r];
                for (int i = start; i <= end; ++i) pos[i] = p++;
                if (p & 1) { pos[end] |= 0x40000000; ++p; }
                run_pend[r] = p >> 1;
                start = end + 1;
            }
        }
    }
    __syncthreads();
    const int n_runs = n_runs_s;

    const long long local = (long long)blockIdx.x * (blockDim.x >> 5) + warp;   // 1, 2 or 4 walkers per CTA (launch_q)
    if (local >= L.num_walkers) return;                // no block-wide barrier below this line
    unsigned char *wp = smem_raw + lay.warp0 + (size_t)warp * lay.per_warp;
    float4 *rowsA = reinterpret_cast<float4 *>(wp + lay.rowsA);
    float4 *rowsL = reinterpret_cast<float4 *>(wp + lay.rowsL);
    float4 *pert = reinterpret_cast<float4 *>(wp + kOffPert);
    double2 *ab = reinterpret_cast<double2 *>(wp + lay.ab);
    float4 *qrow = reinterpret_cast<float4 *>(wp + lay.qrow);     // [rung][2]: two tight rows of each rung
    double *RmS = reinterpret_cast<double *>(wp + lay.RmS);
    double *dex = reinterpret_cast<double *>(wp + aff_off_dex(NQ));      // fp64 fallback: exact d_j, [q][lane]
    float *qL = reinterpret_cast<float *>(wp + lay.qL);           // [rung]: bound on the change of any residual norm, non-increasing
    float4 *cand4 = reinterpret_cast<float4 *>(wp + kOffCand4);   // the kept perturbations (-2 d_j, -|d_j|^2), by rank
    int *candj = reinterpret_cast<int *>(wp + kOffCandj);
    float *candd = reinterpret_cast<float *>(wp + kOffCandd);     // upper bounds of the candidates' eq. (14) values
    int2 *sjv = reinterpret_cast<int2 *>(wp + kOffSjv);           // survivors of the threshold: (perturbation index, phase-1 value)
    const float4 *rowsT = reinterpret_cast<const float4 *>(wp + kOffRowsT);
    const int *runT_pend = reinterpret_cast<const int *>(wp + kOffRunTp);
    const float *runT_bf = reinterpret_cast<const float *>(wp + kOffRunTb);
    double *pose = reinterpret_cast<double *>(wp + kOffPose);     // R*(9) t*(3) omega(3): fp64, touched only on moves / fp64 paths

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
        const double wn = sqrt(fma(vel[2], vel[2], fma(vel[1], vel[1], vel[0] * vel[0])));
        for (int m = lane; m < n_t; m += 32) {         // ladder dT_m = gamma^(m-1) by repeated multiplication
            double dT = 1.0;
            for (int q = 0; q < m; ++q) dT = dT * L.gamma;
            const double p0 = dT * vel[0], p1 = dT * vel[1], p2 = dT * vel[2];
            double A, B;
            exp_coeffs(fma(p2, p2, fma(p1, p1, p0 * p0)), A, B);
            ab[m] = make_double2(A * dT, B * dT * dT);
            // rotation angle of rung m times the Lipschitz constant (gamma <= 1: non-increasing in m)
            qL[m] = (float)(dT * wn) * amax_s * 1.001f + 1e-30f;
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
    const unsigned kp_all = (KP >= 32) ? FULL : ((1u << KP) - 1u);
    unsigned sortdir = 0u;                              // bit t: this lane keeps the larger key at stage t of the bitonic network
    {
        int stage = 0;
        for (int k = 2; k <= 32; k <<= 1)
            for (int j = k >> 1; j > 0; j >>= 1) {
                if (((lane & j) == 0) == ((lane & k) == 0)) sortdir |= 1u << stage;
                ++stage;
            }
    }
    const unsigned inv_kp = (65536u + (unsigned)KP - 1u) / (unsigned)KP;   // t / KP = (t * inv_kp) >> 16 for t < 3,000

    // selection constants: at most s_max survivors (a power of two), at least need_lo
    int s_max = 8;
    while (s_max < 2 * n_ps + 4 && s_max < 32) s_max <<= 1;
    const int need_lo = min(n_p, n_ps + CLOSURE_NEED_EXTRA);
    const int r_target = n_ps + CLOSURE_RT_EXTRA + (n_ps >> CLOSURE_RT_SHIFT);        // rank whose value seeds the next iteration's threshold
    const float step0 = 0.0625f * run_bf[n_runs - 1];
    float U_state = 0.f;

    // executed-work counters (closure_get_stats): in shared memory, touched by lane 0 and only when asked for
    unsigned long long *stc = reinterpret_cast<unsigned long long *>(wp + kOffStc);
    const bool stats = (L.stats != nullptr) && lane == 0;
    if (stats) {
        for (int k = 0; k < kNumStats; ++k) stc[k] = 0ull;
    }
    const long long clk_begin = stats ? clock64() : 0ll;
    bool hit = false;
    bool moved = true;
    float epsA = 0.f;
    double rot_margin = CUDART_INF;
    int nT_runs = 0;
    int pairs_total = run_pend[n_runs - 1];
    CLOSURE_PIN_R(pairs_total);
    const bool full_p1 = pairs_total <= kTight;          // short tables: phase 1 evaluates every constraint, no phase 2
    // N_P <= 32 and one run of equal bounds (BASELINE config 5): best-first branch and bound, one perturbation at a time
    // against the whole table, which the lanes keep in registers while the walker stays (up to four pair-entries each)
    const bool best_first = NQ == 1 && n_runs == 1 && pairs_total <= 128;
    const int pe_rt = (pairs_total + 31) >> 5;
    unsigned long long CA0[4], CA1[4], CA2[4], CA3[4];   // (f0a f0b) (f1a f1b) (f2a f2b) (fca fcb) of entries lane + 32 k
    float *vals = reinterpret_cast<float *>(wp + kOffVals);       // best_first: the N_P* + 1 largest eq. (14) values, by rank
    // cached across iterations while the pose does not move
    int full_m = -1;                                    // rung whose rows sit in rowsL
    float epsL = 0.f;
    bool rdeadL = false;

    for (int s = 1; s <= L.num_steps; ++s) {
        // ================================================== set-up at the current pose (only after a move)
        if (moved) {
            const long long c0 = stats ? clock64() : 0ll;
            aff_setup_on_move<RES>(smem_raw, warp, lane, rows_bytes, n, n_t, NQ, L.pairs_cap, t_p, full_p1, stats);
            if (stats) stc[10] += (unsigned long long)(clock64() - c0);
            epsA = (float)pose[16];
            rot_margin = pose[15];
            nT_runs = (int)pose[17];
            full_m = -1;
            if (NQ == 1 && best_first && !full_p1) {
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const int e = lane + 32 * k;
                    if (e < pairs_total) {
                        const float4 X = rowsA[2 * e], Y = rowsA[2 * e + 1];
                        CA0[k] = pk2(X.x, X.y); CA1[k] = pk2(X.z, X.w); CA2[k] = pk2(Y.x, Y.y); CA3[k] = pk2(Y.z, Y.w);
                    } else {
                        CA0[k] = CA1[k] = CA2[k] = pk2(0.f, 0.f);
                        CA3[k] = pk2(-CUDART_INF_F, -CUDART_INF_F);
                    }
                }
            }
        }

        // ================================================== a2: perturbations of this lane
        unsigned long long p0[NPK1], p1[NPK1], p2[NPK1];
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
                dd[q] = 0.25f * fmaf(e2[q], e2[q], fmaf(e1[q], e1[q], e0[q] * e0[q]));
                pert[32 * q + lane] = make_float4(e0[q], e1[q], e2[q], -dd[q]);
            }
            if (ODD) { o0 = e0[NQ - 1]; o1 = e1[NQ - 1]; o2 = e2[NQ - 1]; }
        }

        // ================================================== a3 / a4: eq. (14) and the top-N_P* by branch and bound
        const float rmf = (float)rot_margin;                // +inf unless POSE_REG_SPLIT
        const float E0 = epsA + tp2sq3 * kMu19;             // bound on |a32 - a64| up to its own rounding
        float unc_l = 0.f;
        float ub[NQ];                                       // phase 1: upper bounds of d_j (the values themselves if full_p1)
        const bool use_p1 = full_p1 || n_p > s_max || best_first;   // few perturbations: all of them are "survivors"
        if (use_p1) {
            eq14_table<NQ>(full_p1 ? rowsA : rowsT, full_p1 ? n_runs : nT_runs, full_p1 ? run_pend : runT_pend,
                           full_p1 ? run_bf : runT_bf, p0, p1, p2, o0, o1, o2, dd, E0, ub, unc_l);
#pragma unroll
            for (int q = 0; q < NQ; ++q) ub[q] = (lane + 32 * q < n_p) ? fminf(ub[q], rmf) : -CUDART_INF_F;
            if (stats) stc[6] += (unsigned long long)(full_p1 ? n : kTight) * n_p;
        } else {
#pragma unroll
            for (int q = 0; q < NQ; ++q) ub[q] = (lane + 32 * q < n_p) ? CUDART_INF_F : -CUDART_INF_F;
        }

        // ---- threshold U with need <= #{ub_j >= U} <= s_max (a NaN counts as a survivor and fails the certificate),
        // found by probing counts; if too few of the survivors turn out to lie above U (their phase-1 values are only
        // upper bounds) the threshold is lowered and the selection repeated (at most twice) before fp64 takes over
        float U = -CUDART_INF_F;
        int cnt = n_p;
        bool found = true;
        float lo = -CUDART_INF_F, hi = CUDART_INF_F, step = step0;
        int need = need_lo;
        if (n_p > s_max) U = U_state;
        bool certified = false;
        float myval = -CUDART_INF_F;
        float unc = 0.f;
        if (NQ == 1 && best_first) {
            // ---- best-first branch and bound (lane j = perturbation j): the perturbation with the largest upper bound is
            // evaluated against the whole table (lane = pair-entries, one warp maximum) until N_P* exact values lie more
            // than 2 unc above every remaining upper bound; no other perturbation can then be among the N_P* best
            const float ub0 = ub[0];
            const bool valid = lane < n_p;
            uint32_t pool = (valid && !full_p1) ? ((fkey(ub0) & ~31u) | (uint32_t)(31 - lane)) : 0u;   // not yet evaluated
            if (valid && !full_p1 && (ub0 != ub0)) pool = 0xffffffe0u | (uint32_t)(31 - lane);             // a NaN is evaluated first
            float dexv = (valid && full_p1) ? ub0 : -CUDART_INF_F;     // exact eq. (14) value of this lane's perturbation
            bool evald = valid && full_p1;
            float uncw = wmax_nonneg(unc_l);
            const float bf0 = run_bf[0];
            float Umax = -CUDART_INF_F;
            int rank = 0;                                             // of this lane's value among the evaluated ones
            uint32_t g = __reduce_max_sync(FULL, pool);
#pragma unroll 1
            while (g != 0u) {
                const int jsel = 31 - (int)(g & 31u);
                if (lane == jsel) pool = 0u;
                const uint32_t gnext = __reduce_max_sync(FULL, pool);    // issued early: its latency hides behind the evaluation
                const float4 pj = pert[jsel];
                const unsigned long long E0p = pk2(pj.x, pj.x), E1p = pk2(pj.y, pj.y), E2p = pk2(pj.z, pj.z);
                float m = -CUDART_INF_F;
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    if (k < pe_rt) {
                        const unsigned long long vo = fma2(CA0[k], E0p, fma2(CA1[k], E1p, fma2(CA2[k], E2p, CA3[k])));
                        float l2, h2;
                        upk2(vo, l2, h2);
                        m = fmaxf(m, fmaxf(l2, h2));
                    }
                }
                const float mv = fkey_inv(__reduce_max_sync(FULL, fkey(m)));   // one warp maximum and one square root
                const float a = fmaxf(mv - pj.w, 1e-30f);              // pj.w = -|d|^2
                const float rr = rsqrt_normal(a);
                const float sq = a * rr;
                uncw = fmaxf(uncw, 1.01f * fmaf(E0, rr, (bf0 + sq) * kMu19));
                const float dnew = fminf(bf0 - sq, rmf);                // the same on every lane
                // ranks are kept up to date: values below the new one move down, the new one goes below those not smaller
                const unsigned ge = __ballot_sync(FULL, evald && !(dexv < dnew));
                if (evald && dexv < dnew) ++rank;
                if (lane == jsel) { dexv = dnew; evald = true; rank = __popc(ge); }
                if (stats) { stc[6] += (unsigned long long)n; stc[13] += 1; }
                g = gnext;
                Umax = (g != 0u) ? fkey_inv(g | 31u) : -CUDART_INF_F;  // >= every remaining upper bound
                const float needl = fmaf(2.0f, uncw, 4.0f * kMu19 * (fabsf(dexv) + fabsf(Umax)));
                const int above = __popc(__ballot_sync(FULL, evald && (dexv - Umax > needl)));
                if (above >= n_ps) break;
            }
            unc = uncw;
            if (RES == CLOSURE_POSE_REG_SPLIT) unc += 1.2e-7f * fabsf(rmf);
            // ---- the N_P* + 1 best go to vals[] / candj[] by rank (short tables: everything was evaluated by phase 1 and
            // is ranked by counting here)
            const unsigned evm = __ballot_sync(FULL, evald);
            const bool nan_any = __any_sync(FULL, evald && (dexv != dexv));
            if (full_p1) {
                rank = 0;
                for (unsigned rem = evm; rem != 0u; rem &= rem - 1u) {
                    const int e = __ffs(rem) - 1;
                    const float xe = __shfl_sync(FULL, dexv, e);
                    rank += (xe > dexv || (xe == dexv && e < lane)) ? 1 : 0;
                }
            }
            if (evald && rank <= n_ps) {
                vals[rank] = dexv;
                if (rank < n_ps) candj[rank] = lane;
            }
            __syncwarp();
            const int nev = __popc(evm);
            myval = (lane <= n_ps && lane < nev) ? vals[lane] : -CUDART_INF_F;
            const float prev = __shfl_up_sync(FULL, myval, 1);
            const bool trust = (L.exact_only & 32) != 0;
            bool ok = true;
            if (lane < n_ps) ok = (myval > -CUDART_INF_F) && (myval < CUDART_INF_F);
            if (lane >= 1 && lane <= n_ps) {
                const bool none_left = (lane == n_ps) && (myval == -CUDART_INF_F);
                const float needg = fmaf(2.0f, unc, 4.0f * kMu19 * (fabsf(prev) + fabsf(myval)));
                ok = ok && (none_left || (prev - myval > needg));
            }
            if (trust) ok = true;                       // fp32 mode: the fp32 ranking is taken as it is
            if (lane == n_ps - 1 && Umax > -CUDART_INF_F) {
                const float needu = fmaf(2.0f, unc, 4.0f * kMu19 * (fabsf(Umax) + fabsf(myval)));
                ok = ok && (trust ? (myval >= Umax) : (myval - Umax > needu));
            }
            if (nan_any || (L.exact_only & 4)) ok = false;
            certified = __all_sync(FULL, ok);
            if (certified && lane < n_ps) candd[lane] = myval + fmaf(1.01f, unc, 4.0f * kMu19 * fabsf(myval));    // >= the fp64 value d_j
        } else if (full_p1) {
            // ---- short tables: phase 1 gave the exact eq. (14) value of every perturbation; the N_P* + 1 largest are
            // extracted by rounds of warp maxima over the lanes' locally sorted keys and certified by their gaps
            unc = wmax_nonneg(unc_l);
            if (RES == CLOSURE_POSE_REG_SPLIT) unc += 1.2e-7f * fabsf(rmf);
            certified = topk_certified<NQ>(ub, n_ps, unc, (L.exact_only & 4) != 0, (L.exact_only & 32) != 0, lane, candj, candd, myval);
        } else {
#pragma unroll 1
        for (int attempt = 0; attempt < 3; ++attempt) {
        if (n_p > s_max) {
            found = false;
#pragma unroll 1
            for (int it = 0; it < 24; ++it) {
                int c = 0;
#pragma unroll
                for (int q = 0; q < NQ; ++q) c += (!(ub[q] < U)) ? 1 : 0;
                cnt = (int)__reduce_add_sync(FULL, (unsigned)c);
                if (stats) stc[12] += 1;
                if (cnt < need) hi = U;
                else if (cnt > s_max) lo = U;
                else { found = true; break; }
                if (lo == -CUDART_INF_F) { U = U - step; step = step + step; }
                else if (hi == CUDART_INF_F) { U = U + step; step = step + step; }
                else {
                    const float mid = 0.5f * (lo + hi);
                    if (!(mid > lo && mid < hi)) break;      // ties: no threshold separates them
                    U = mid;
                }
                if (!(fabsf(U) < 3.0e38f)) break;
            }
        }
        bool ufail = false;
        if (found) {
            // ---- compaction of the survivors: (j, phase-1 value) by slot
            {
                int base = 0;
                const unsigned lt = (1u << lane) - 1u;
#pragma unroll
                for (int q = 0; q < NQ; ++q) {
                    const bool in = (lane + 32 * q < n_p) && !(ub[q] < U);
                    const unsigned b = __ballot_sync(FULL, in);
                    if (in) sjv[base + __popc(b & lt)] = make_int2(lane + 32 * q, __float_as_int(ub[q]));
                    base += __popc(b);
                }
            }
            __syncwarp();                                   // sjv[], pert[] visible to all lanes
            if (stats) stc[13] += (unsigned long long)cnt;
            // ---- phase 2: the survivors against all constraints, lane = (survivor slot, chunk of the table)
            const int lgS = 32 - __clz(max(cnt, 1) - 1);    // S = 2^lgS >= cnt survivors' slots, C = 32 / S chunks of the table
            const int S = 1 << lgS;
            const int slot = lane & (S - 1);
            const bool act = slot < cnt;
            const int2 mine = sjv[act ? slot : 0];
            float val;
            if (full_p1) {
                val = __int_as_float(mine.y);
            } else {
                const int lgC = 5 - lgS, chunk = lane >> lgS;
                const float4 pj = pert[mine.x];
                const unsigned long long E0p = pk2(pj.x, pj.x), E1p = pk2(pj.y, pj.y), E2p = pk2(pj.z, pj.z);
                float v = CUDART_INF_F;
                int pp = 0;
                for (int r = 0; r < n_runs; ++r) {
                    const int pend = run_pend[r];
                    const float bf = run_bf[r];
                    float mx = -CUDART_INF_F;
                    // the same trip count on every lane (a lane past the end of the run re-reads its last entry: a maximum
                    // does not see duplicates), so that the warp stays converged
                    const int trips = (pend - pp + (1 << lgC) - 1) >> lgC;
                    const float4 *e = rowsA + 2 * (pp + chunk);
                    const float4 *elast = rowsA + 2 * (pend - 1);
#pragma unroll 2
                    for (int it = 1; it < trips; ++it) {               // all trips but the last are inside the run on every lane
                        const float4 X = e[0], Y = e[1];
                        const unsigned long long vo =
                            fma2(pk2(X.x, X.y), E0p, fma2(pk2(X.z, X.w), E1p, fma2(pk2(Y.x, Y.y), E2p, pk2(Y.z, Y.w))));
                        float l2, h2;
                        upk2(vo, l2, h2);
                        mx = fmaxf(mx, fmaxf(l2, h2));
                        e += 2 << lgC;
                    }
                    {
                        const float4 *ec = e < elast ? e : elast;
                        const float4 X = ec[0], Y = ec[1];
                        const unsigned long long vo =
                            fma2(pk2(X.x, X.y), E0p, fma2(pk2(X.z, X.w), E1p, fma2(pk2(Y.x, Y.y), E2p, pk2(Y.z, Y.w))));
                        float l2, h2;
                        upk2(vo, l2, h2);
                        mx = fmaxf(mx, fmaxf(l2, h2));
                    }
                    pp = pend;
                    for (int off = S; off < 32; off <<= 1) mx = fmaxf(mx, __shfl_xor_sync(FULL, mx, off));
                    const float a = fmaxf(mx - pj.w, 1e-30f);          // pj.w = -|d|^2
                    const float rr = rsqrt_normal(a);
                    const float sq = a * rr;
                    const float du = 1.01f * fmaf(E0, rr, (bf + sq) * kMu19);
                    if (act) unc_l = fmaxf(unc_l, du);
                    v = fminf(v, bf - sq);
                }
                val = fminf(v, rmf);
                if (stats) stc[6] += (unsigned long long)n * cnt;
            }
            unc = wmax_nonneg(unc_l);
            if (RES == CLOSURE_POSE_REG_SPLIT) unc += 1.2e-7f * fabsf(rmf);
            // ---- ranking: a sorting network on order-preserving keys whose 5 low bits carry the slot (values move down by
            // < 2^-18 relative: covered by the certificate); lanes 0 .. cnt-1 hold one survivor each
            const bool nan_any = __any_sync(FULL, act && (val != val));
            uint32_t key = (lane < cnt) ? ((fkey(val) & ~31u) | (uint32_t)(31 - lane)) : 0u;
            // bitonic sorting network over the 32 lanes, descending: lane r ends with the r-th largest key
            {
                int stage = 0;
#pragma unroll
                for (int k = 2; k <= 32; k <<= 1) {
#pragma unroll
                    for (int j = k >> 1; j > 0; j >>= 1) {
                        const uint32_t o = __shfl_xor_sync(FULL, key, j);
                        key = ((sortdir >> stage) & 1u) ? max(key, o) : min(key, o);
                        ++stage;
                    }
                }
            }
            const bool have = lane < cnt;                   // this lane holds the survivor ranked `lane`
            myval = have ? fkey_inv(key & ~31u) : -CUDART_INF_F;    // the value the key stands for (<= the survivor's value)
            const int myj = sjv[have ? 31 - (int)(key & 31u) : 0].x;
            if (lane < n_ps) candj[lane] = myj;
            // the next iteration's threshold: the value ranked r_target (the distribution is stationary while the walker stays)
            {
                const float ut = __shfl_sync(FULL, myval, min(cnt - 1, r_target));
                U_state = (fabsf(ut) < 3.0e38f) ? ut : U;
            }
            // ---- certificate: consecutive values more than 2 unc apart, and the N_P*-th more than 2 unc above both the
            // next one and the threshold (every perturbation that was not evaluated has d_j <= ub_j < U + unc)
            if (lane > n_ps) myval = -CUDART_INF_F;
            const float prev = __shfl_up_sync(FULL, myval, 1);
            const bool trust = (L.exact_only & 32) != 0;
            bool ok = true;
            if (lane < n_ps) ok = (myval > -CUDART_INF_F) && (myval < CUDART_INF_F);
            if (lane >= 1 && lane <= n_ps) {
                const bool none_left = (lane == n_ps) && (myval == -CUDART_INF_F);
                const float needg = fmaf(2.0f, unc, 4.0f * kMu19 * (fabsf(prev) + fabsf(myval)));
                ok = ok && (none_left || (prev - myval > needg));
            }
            if (trust) ok = true;                       // fp32 mode: the fp32 ranking is taken as it is
            bool oku = true;
            if (lane == n_ps - 1 && U > -CUDART_INF_F) {
                const float needu = fmaf(2.0f, unc, 4.0f * kMu19 * (fabsf(U) + fabsf(myval)));
                oku = trust ? (myval >= U) : (myval - U > needu);
            }
            if (nan_any || (L.exact_only & 4)) ok = false;
            const bool gaps_ok = __all_sync(FULL, ok);
            ufail = !__all_sync(FULL, oku);
            certified = gaps_ok && !ufail;
            if (certified && lane < n_ps) candd[lane] = myval + fmaf(1.01f, unc, 4.0f * kMu19 * fabsf(myval));    // >= the fp64 value d_j
            if (certified || !gaps_ok || cnt >= s_max) break;
            // only the threshold failed: lower it so that at least two more perturbations survive
            if (stats) stc[14] += 1;
            need = min(cnt + 2, s_max);
            hi = U;
            if (lo == -CUDART_INF_F) { U = U - step; step = step + step; } else U = 0.5f * (lo + hi);
            __syncwarp();                                   // sjv[], vals[] are rewritten by the next attempt
        } else {
            unc = wmax_nonneg(unc_l);
            if (stats) stc[15] += 1;
            break;
        }
        }
        }
        if (!certified) {
            // fp64 fall-back (near-ties, a threshold too close to the N_P*-th value, no separating threshold)
            double R[9], t[3];
#pragma unroll
            for (int e = 0; e < 9; ++e) R[e] = pose[e];
#pragma unroll
            for (int e = 0; e < 3; ++e) t[e] = pose[9 + e];
            const ExactMargin<RES> exact{ R, t, rows, n, rng, (uint32_t)s, t_p, rot_margin };
            const bool all = !found || (L.exact_only & 16) != 0;
            const int cntf = topk_fp64<NQ>(ub, n_p, n_ps, unc, myval, all, lane, dex, candj, candd, exact);
            if (stats) { stc[8] += 1; stc[0] += (unsigned long long)n * cntf; }
        }
        __syncwarp();                                       // pert[], candj[], candd[] visible to all lanes
        if (lane < n_ps) cand4[lane] = pert[candj[lane]];
        const float mycd = (lane < n_ps) ? candd[lane] : -CUDART_INF_F;
        const float cdm = fkey_inv(__reduce_max_sync(FULL, fkey(mycd)));    // the best any candidate can be at R*
        __syncwarp();

        // ================================================== a5-a6: ladder, first feasible rung
        int m0 = 0;
        unsigned win = 0u;
        for (int mb = 0; mb < n_t && m0 == 0; mb += 32) {
            // ---- rungs that the rotation can still repair: cdm + qL[m] >= 0 (qL is non-increasing in m: a prefix)
            const int mq = mb + lane;
            const bool lip_ok = (mq < n_t) && !(cdm + qL[min(mq, n_t - 1)] < 0.f);
            unsigned livemask = __ballot_sync(FULL, lip_ok);
            if (L.exact_only & 2) livemask = __ballot_sync(FULL, mq < n_t);       // debug: nothing is screened out
            const int nlive = __popc(livemask);             // a prefix of the block
            if (nlive == 0) break;
            // ---- screening, lane = (rung, candidate): a candidate is dead for sure at rung m if one of the rung's two
            // tight rows is violated beyond its error bound, or if its margin at R* is more negative than the
            // rotation to R_m can repair
            unsigned rmask = 0u;
            const int tasks = nlive * KP;
#pragma unroll 1
            for (int tq = lane; tq < tasks; tq += 32) {
                const int ml = (int)(((unsigned)tq * inv_kp) >> 16);
                const int k = tq - ml * KP;
                const int m = mb + ml;
                const float4 r0 = qrow[2 * m], r1 = qrow[2 * m + 1];
                const float4 c4 = cand4[k];
                const float v0 = fmaf(r0.x, c4.x, fmaf(r0.y, c4.y, fmaf(r0.z, c4.z, r0.w)));
                const float v1 = fmaf(r1.x, c4.x, fmaf(r1.y, c4.y, fmaf(r1.z, c4.z, r1.w)));
                if (!(v0 > c4.w) && !(v1 > c4.w) && !(candd[k] + qL[m] < 0.f)) rmask |= 1u << ml;
            }
            unsigned qmask = __reduce_or_sync(FULL, rmask);
            if (L.exact_only & 2) qmask = livemask;
            if (stats) stc[7] += (unsigned long long)tasks * 2;

            // ---- full evaluation of the surviving rungs, in order
            while (qmask != 0u && m0 == 0) {
                const int l0 = __ffs(qmask) - 1;
                qmask &= qmask - 1u;
                const int m1 = mb + l0;
                double Rm[9], t[3];
#pragma unroll
                for (int e = 0; e < 9; ++e) Rm[e] = RmS[m1 * 9 + e];
#pragma unroll
                for (int e = 0; e < 3; ++e) t[e] = pose[9 + e];
                if (full_m != m1) {
                    __syncwarp();                            // earlier readers of rowsL are done
                    float eps_l = 0.f;
                    bool rdead = false;
                    float w1 = -CUDART_INF_F, w2 = -CUDART_INF_F;    // this lane's two tightest rows of the rung
                    int i1 = 0, i2 = 0;
#pragma unroll 1
                    for (int i = lane; i < n; i += 32) {
                        const double *row = rows + i * ROW;
                        double u0, u1, u2, c;
                        affine_setup<RES>(Rm, t, row, u0, u1, u2, c);
                        if (RES == CLOSURE_POSE_REG_SPLIT) {
                            if (!(frob_sq(Rm, row) <= row[13])) rdead = true;     // exact: no perturbation involved
                        }
                        float g0, g1, g2, fcb, eps;
                        screen_row(u0, u1, u2, c - row[RS::BETA + 1], tp2, tp2sq3, g0, g1, g2, fcb, eps);
                        const float wv = fcb - eps;
                        rowsL[i] = make_float4(g0, g1, g2, wv);
                        eps_l = fmaxf(eps_l, eps);
                        if (wv > w1) { w2 = w1; i2 = i1; w1 = wv; i1 = i; } else if (wv > w2) { w2 = wv; i2 = i; }
                    }
                    epsL = wmax_nonneg(eps_l);
                    rdeadL = __any_sync(FULL, rdead);
                    full_m = m1;
                    if (stats) stc[3] += n;
                    __syncwarp();
                    // the rung's screening rows become its two tightest rows among ALL constraints (they stay until the
                    // next move): the candidate rows of the set-up let this rung through, these will not do so as easily
                    {
                        const uint32_t k1 = fkey(w1);
                        const uint32_t g1m = __reduce_max_sync(FULL, k1);
                        const int src1 = __ffs(__ballot_sync(FULL, k1 == g1m)) - 1;
                        const uint32_t k2 = (lane == src1) ? fkey(w2) : k1;
                        const uint32_t g2m = __reduce_max_sync(FULL, k2);
                        const int src2 = __ffs(__ballot_sync(FULL, k2 == g2m)) - 1;
                        if (lane == src1) {
                            float4 r4 = rowsL[i1];
                            if (rdeadL) r4.w = CUDART_INF_F;
                            qrow[2 * m1] = r4;
                        }
                        if (lane == src2) qrow[2 * m1 + 1] = rowsL[(lane == src1) ? i2 : i1];
                        __syncwarp();
                    }
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
                            M = fmaxf(M, fmaf(f.x, c4.x, fmaf(f.y, c4.y, fmaf(f.z, c4.z, f.w))));
                        }
                    }
                    M = chunk_max_to_first(M, KP, NCH);      // valid on the lanes with ech == 0 (`mine` below)
                    // M = max_i (v32_i - eps_i):  M > th  => some constraint violated for sure;
                    // M + 2 eps_max <= th => every constraint satisfied for sure.
                    const bool dead = M > c4.w;
                    const bool sure = (epsL < CUDART_INF_F) && (M <= c4.w - 2.0f * epsL);
                    const bool mine = e_act && ech == 0;
                    unsigned alive2 = __ballot_sync(FULL, mine && !dead) & kp_all;
                    unsigned undecided = __ballot_sync(FULL, mine && !dead && !sure) & kp_all;
                    if (L.exact_only & 2) { alive2 = kp_all; undecided = kp_all; }
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
            if (nlive < 32) break;                          // the live rungs are a prefix: none beyond this block
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

template <int RES, int NQ>
cudaError_t launch_q(const WalkLaunch &L, int n_instances, int max_rows_bytes, int max_n, cudaStream_t stream)
{
    // Walkers (warps) per CTA: four share one staged table; fewer only when four tables' worth of per-warp state does not fit.
    int wpc = kCoopWarps;                                // measured at 1 / 2 / 4: four is best at every size, also with few walkers or iterations
    AffSmem lay = aff_layout(max_rows_bytes, max_n, L.n_t, NQ, L.pairs_cap, wpc);
    while (lay.total > 200 * 1024 && wpc > 1) { wpc >>= 1; lay = aff_layout(max_rows_bytes, max_n, L.n_t, NQ, L.pairs_cap, wpc); }
    if (lay.total > 200 * 1024) return cudaErrorInvalidConfiguration;
    cudaError_t e = cudaFuncSetAttribute(walker_coop_kernel<RES, NQ>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)lay.total);
    if (e != cudaSuccess) return e;
    const long long blocks = (L.num_walkers + wpc - 1) / wpc;
    if (blocks > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    dim3 grid((unsigned)blocks, (unsigned)n_instances, 1);
    walker_coop_kernel<RES, NQ><<<grid, 32 * wpc, lay.total, stream>>>(L);
    return cudaGetLastError();
}

template <int RES>
cudaError_t launch_r(const WalkLaunch &L, int n_instances, int max_rows_bytes, int max_n, cudaStream_t stream)
{
    // the kernel is written for NQ perturbations per lane; only NQ = 1 (N_P <= 32) is built: launch_walkers_coop sends
    // larger N_P to the dense kernel
    if (L.n_p <= 32) return launch_q<RES, 1>(L, n_instances, max_rows_bytes, max_n, stream);
    return cudaErrorInvalidConfiguration;
}

}  // namespace

bool coop_path_available(int residual_type, int mode, int n_p, int max_n)
{
    return mode == CLOSURE_MODE_ROT && n_p <= 256 && max_n <= 4096;
}

cudaError_t launch_walkers_coop(int residual_type, const WalkLaunch &L, int n_instances, int max_rows_bytes,
                                cudaStream_t stream)
{
    const int max_n = max_rows_bytes / (row_doubles(residual_type) * 8);
    switch (residual_type) {
    case CLOSURE_REPROJ_2D3D:
    case CLOSURE_REPROJ_2D3D_ELL: return launch_walkers_coop_reproj(residual_type, L, n_instances, max_rows_bytes, stream);
    // the ellipsoid norm of Ex.2 (eq. (6), Lambda_i != I): the dense kernel with the quadratic form in the pair, any N_P
    case CLOSURE_REG_3D3D_ELL: return launch_walkers_coop_dense(residual_type, L, n_instances, max_rows_bytes, stream);
    default: break;
    }
    // More than 32 perturbations per iteration (BASELINE configs 1, 2, 4): the dense kernel, several perturbations per
    // lane against every constraint.  At most 32 (config 5): branch and bound (this file), one perturbation per lane.
    // Both take the fp64 decisions bit for bit.  (Measured with N_P = 150 on tables of 30 - 200 constraints: the
    // batched branch and bound of this file saves 2/3 of the pairs but loses 1.4 - 4x to its bookkeeping and to the
    // fp64 fall-backs that loose phase-1 bounds cause; with N_P <= 32 the best-first form wins.)
    if (L.n_p > 32) return launch_walkers_coop_dense(residual_type, L, n_instances, max_rows_bytes, stream);
    switch (residual_type) {
    case CLOSURE_REG_3D3D: return launch_r<CLOSURE_REG_3D3D>(L, n_instances, max_rows_bytes, max_n, stream);
    case CLOSURE_POSE_REG: return launch_r<CLOSURE_POSE_REG>(L, n_instances, max_rows_bytes, max_n, stream);
    case CLOSURE_POSE_REG_SPLIT: return launch_r<CLOSURE_POSE_REG_SPLIT>(L, n_instances, max_rows_bytes, max_n, stream);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace closure
