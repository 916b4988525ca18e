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
// Every residual is evaluated by the same fp64 functions as in the one-walker-per-thread kernel
// (margin_direct / in_purse_direct in walker_common.cuh), so the two kernels agree bit for bit;
// unlike the rotation sampler nothing is shared between the perturbations of a pose (each has its
// own rotation), so there is no cheap fp32 image to certify and this kernel stays in fp64.
#include <cuda_runtime.h>
#include <math_constants.h>
#include <stdint.h>

#include "closure_internal.h"
#include "walker_common.cuh"
#include "walker_coop_common.cuh"

namespace closure {
namespace {

struct TransSmem {
    size_t warp0, per_warp, pose, dex, Rc, candj, candd, stc, total;
};

__host__ __device__ inline TransSmem trans_layout(int rows_bytes, int nq)
{
    TransSmem s;
    const size_t o = 16 + (size_t)((rows_bytes + 15) & ~15);
    s.warp0 = o;
    size_t w = 0;
    s.pose = w;  w += 16 * 8;                    // R*(9) t*(3) v(3)
    s.dex = w;   w += (size_t)nq * 32 * 8;       // eq. (14) values, [q][lane]
    s.Rc = w;    w += 32 * 9 * 8;                // rotations of the kept perturbations, by rank
    s.candj = w; w += 32 * 4;
    s.candd = w; w += 32 * 4;
    s.stc = w;   w += 16 * 8;
    s.per_warp = w;
    s.total = o + (size_t)kCoopWarps * w;
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
__global__ void __launch_bounds__(kCoopThreads, 4) walker_coop_trans_kernel(const __grid_constant__ WalkLaunch L)
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

    const long long local = (long long)blockIdx.x * kCoopWarps + warp;
    if (local >= L.num_walkers) return;                // no block-wide barrier below this line
    const TransSmem lay = trans_layout(rows_bytes, NQ);
    unsigned char *wp = smem_raw + lay.warp0 + (size_t)warp * lay.per_warp;
    double *pose = reinterpret_cast<double *>(wp + lay.pose);
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
        for (int k = 0; k < 10; ++k) stc[k] = 0ull;
    }
    bool hit = false;
    const int KP = n_ps;
    const int items = KP * n_t;                          // ladder candidates, in Alg. A8's order (m, k)

    for (int s = 1; s <= L.num_steps; ++s) {
        // ================================================== a2-a4: perturb, eq. (14), top-N_P* (fp64)
        {
            const ExactMarginTrans<RES> exact{ R, t, K, rows, n, rng, (uint32_t)s, L.theta_p };
            float dummy[NQ];
#pragma unroll
            for (int q = 0; q < NQ; ++q) dummy[q] = 0.f;
            topk_fp64<NQ>(dummy, n_p, n_ps, 0.f, 0.f, true, lane, dex, candj, candd, exact);
            if (stats) { stc[0] += (unsigned long long)n * n_p; stc[2] += (unsigned long long)n * n_p; }
        }
        __syncwarp();
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
        int win = -1;
        for (int base = 0; base < items && win < 0; base += 32) {
            const int it = base + lane;
            bool ok = false;
            if (it < items) {
                const int m = it / KP, k = it - m * KP;
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
            for (int e = 0; e < 9; ++e) R[e] = Rc[k * 9 + e];
            if (stats) stc[4] += 1;
        }
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
            for (int k = 0; k < 10; ++k) atomicAdd(L.stats + k, stc[k]);
        }
    }
}

template <int RES, int NQ>
cudaError_t launch_q(const WalkLaunch &L, int n_instances, int max_rows_bytes, cudaStream_t stream)
{
    const TransSmem lay = trans_layout(max_rows_bytes, NQ);
    if (lay.total > 200 * 1024) return cudaErrorInvalidConfiguration;
    cudaError_t e = cudaFuncSetAttribute(walker_coop_trans_kernel<RES, NQ>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                         (int)lay.total);
    if (e != cudaSuccess) return e;
    const long long blocks = (L.num_walkers + kCoopWarps - 1) / kCoopWarps;
    if (blocks > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
    dim3 grid((unsigned)blocks, (unsigned)n_instances, 1);
    walker_coop_trans_kernel<RES, NQ><<<grid, kCoopThreads, lay.total, stream>>>(L);
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
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace closure
