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
#include "walker_common.cuh"

namespace closure {
namespace {

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
    double R[9], t[3], vel[3];   // vel = omega (ROT) or v (TRANS)
    init_walker<MODE>(D, L, rng, w, R, t, vel);
    if (MODE == CLOSURE_MODE_ROT) fill_ladder(L, vel, ladder);

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
                } else if (RES != CLOSURE_REPROJ_2D3D) {
                    // ellipse / ellipsoid norms (eq. (6)): the residual at the perturbed translation, directly
                    for (int i = 0; i < n; ++i) {
                        const double *row = rows + i * ROW;
                        const double beta = row[RS::BETA];
#pragma unroll
                        for (int jj = 0; jj < kJT; ++jj) {
                            const double tj[3] = { t[0] + e0[jj], t[1] + e1[jj], t[2] + e2[jj] };
                            dmn[jj] = dmin(dmn[jj], beta - sqrt(direct_sq<RES>(R, tj, row, K, 0)));
                        }
                    }
                    if (STATS) { st_pp += (unsigned long long)n * kJT; st_ps += n; }
                } else {
                    // REPROJ: P_i = R Z_i + t* once per constraint, then one projection per perturbation
                    for (int i = 0; i < n; ++i) {
                        const double *row = rows + i * ROW;
                        double P0, P1, P2;
                        reproj_point(R, row, P0, P1, P2);
                        const double beta = row[RS::BETA];
#pragma unroll
                        for (int jj = 0; jj < kJT; ++jj) {
                            const double sq = reproj_sq(P0, P1, P2, t[0] + e0[jj], t[1] + e1[jj], t[2] + e2[jj], row, K);
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
                    } else if (RES != CLOSURE_REPROJ_2D3D) {
                        const double b2 = row[RS::BETA + 1];
#pragma unroll
                        for (int k = 0; k < KCAP; ++k) {
                            const double tk[3] = { t[0] + k0[k], t[1] + k1[k], t[2] + k2[k] };
                            if (!(direct_sq<RES>(Rm, tk, row, K, 0) <= b2)) alive &= ~(1u << k);
                        }
                    } else {
                        double P0, P1, P2;
                        reproj_point(Rm, row, P0, P1, P2);
                        const double b2 = row[RS::BETA + 1];
#pragma unroll
                        for (int k = 0; k < KCAP; ++k) {
                            const double sq = reproj_sq(P0, P1, P2, t[0] + k0[k], t[1] + k1[k], t[2] + k2[k], row, K);
                            if (!(sq <= b2)) alive &= ~(1u << k);
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
    case CLOSURE_REG_3D3D_ELL: return Res<CLOSURE_REG_3D3D_ELL>::ROW;
    case CLOSURE_REPROJ_2D3D_ELL: return Res<CLOSURE_REPROJ_2D3D_ELL>::ROW;
    default: return 0;
    }
}

size_t plain_kernel_smem_bytes(int rows_bytes, int n_t)
{
    return 16 + (size_t)((rows_bytes + 15) & ~15) + (size_t)n_t * kBlock * sizeof(double2);
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
    const size_t smem = plain_kernel_smem_bytes(max_rows_bytes, L.n_t);
    if ((L.exact_only & 32) && !coop_path_available(residual_type, mode, L.n_p, max_rows_bytes / (row_doubles(residual_type) * 8))) {
        if (why) *why = "fp32 mode needs the cooperative kernel";
        return cudaErrorInvalidValue;
    }
    // the cooperative kernels report cudaErrorInvalidConfiguration when their per-warp shared memory does not
    // fit (very large N x N_T): the one-walker-per-thread kernel below then takes the launch
    if ((!(L.exact_only & 1) || (L.exact_only & 32)) &&
        coop_path_available(residual_type, mode, L.n_p, max_rows_bytes / (row_doubles(residual_type) * 8))) {
        const cudaError_t e = launch_walkers_coop(residual_type, L, n_instances, max_rows_bytes, stream);
        if (e != cudaErrorInvalidConfiguration) return e;
        if (L.exact_only & 32) {
            if (why) *why = "instance too large for the fp32-mode kernel";
            return cudaErrorInvalidValue;
        }
    }
    if (!(L.exact_only & 1) && mode == CLOSURE_MODE_TRANS && L.n_p <= 256) {
        const cudaError_t e = launch_walkers_coop_trans(residual_type, L, n_instances, max_rows_bytes, stream);
        if (e != cudaErrorInvalidConfiguration) return e;
    }
    // the one-walker-per-thread kernel: rows + a per-thread ladder table (closure_create / closure_set_params reject
    // instances it cannot stage, so this does not fire for a handle that was created successfully)
    if (smem > kMaxStageBytes) {
        if (why) *why = "instance too large for shared-memory staging";
        return cudaErrorInvalidValue;
    }
    switch (residual_type) {
    case CLOSURE_REG_3D3D: return launch_r<CLOSURE_REG_3D3D>(mode, stats, L, grid, smem, stream);
    case CLOSURE_REPROJ_2D3D: return launch_r<CLOSURE_REPROJ_2D3D>(mode, stats, L, grid, smem, stream);
    case CLOSURE_POSE_REG: return launch_r<CLOSURE_POSE_REG>(mode, stats, L, grid, smem, stream);
    case CLOSURE_POSE_REG_SPLIT: return launch_r<CLOSURE_POSE_REG_SPLIT>(mode, stats, L, grid, smem, stream);
    case CLOSURE_REG_3D3D_ELL: return launch_r<CLOSURE_REG_3D3D_ELL>(mode, stats, L, grid, smem, stream);
    case CLOSURE_REPROJ_2D3D_ELL: return launch_r<CLOSURE_REPROJ_2D3D_ELL>(mode, stats, L, grid, smem, stream);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace closure
