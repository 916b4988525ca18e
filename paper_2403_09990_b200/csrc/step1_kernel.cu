// Step I of CLOSURE, "initialize starting poses", for
// Ex.2 and Ex.3: independent trials, one per thread.
//
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
    if (RES == CLOSURE_REG_3D3D) {
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
        double ab[3], bb[3], a[3][3], b[3][3];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            ab[c] = ((r1[c] + r2[c]) + r3[c]) / 3.0;
            bb[c] = ((r1[3 + c] + r2[3 + c]) + r3[3 + c]) / 3.0;
            a[0][c] = r1[c] - ab[c]; a[1][c] = r2[c] - ab[c]; a[2][c] = r3[c] - ab[c];
            b[0][c] = r1[3 + c] - bb[c]; b[1][c] = r2[3 + c] - bb[c]; b[2][c] = r3[3 + c] - bb[c];
        }
        double na[3] = { a[0][1] * a[1][2] - a[0][2] * a[1][1], a[0][2] * a[1][0] - a[0][0] * a[1][2],
                         a[0][0] * a[1][1] - a[0][1] * a[1][0] };
        double nb[3] = { b[0][1] * b[1][2] - b[0][2] * b[1][1], b[0][2] * b[1][0] - b[0][0] * b[1][2],
                         b[0][0] * b[1][1] - b[0][1] * b[1][0] };
        const double la = sqrt(na[0] * na[0] + na[1] * na[1] + na[2] * na[2]);
        const double lb = sqrt(nb[0] * nb[0] + nb[1] * nb[1] + nb[2] * nb[2]);
        if (!(la < 1e-8) && !(lb < 1e-8)) {
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
            have = det3(Mp) > 0.0 ? polar_rotation(Mp, R) : polar_rotation(Mm, R);
            if (have) {
#pragma unroll
                for (int r = 0; r < 3; ++r) t[r] = bb[r] - (R[3 * r] * ab[0] + R[3 * r + 1] * ab[1] + R[3 * r + 2] * ab[2]);
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

    bool ok = false;
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
    case CLOSURE_REG_3D3D: return launch_t<CLOSURE_REG_3D3D>(d_desc, rows_bytes, trial_begin, num_trials, seed, out_poses, out_ok, stream);
    case CLOSURE_POSE_REG: return launch_t<CLOSURE_POSE_REG>(d_desc, rows_bytes, trial_begin, num_trials, seed, out_poses, out_ok, stream);
    case CLOSURE_POSE_REG_SPLIT: return launch_t<CLOSURE_POSE_REG_SPLIT>(d_desc, rows_bytes, trial_begin, num_trials, seed, out_poses, out_ok, stream);
    default: return cudaErrorInvalidValue;
    }
}

}  // namespace closure
