// Internal declarations shared by the translation units of libclosure_b200.
// Not part of the C ABI (include/closure.h is).  Nothing here is seen by oracle/.
#pragma once

#include <cuda_runtime.h>

#include <string>
#include <vector>

#include "../../include/closure.h"

namespace closure {

// Device-side description of one PURSE instance.  `rows` is the packed constraint table the
// walker kernel stages into shared memory with one bulk copy (TMA, cp.async.bulk):
//   REG_3D3D        row = [a0 a1 a2 b0 b1 b2 beta beta^2]                      (8 doubles)
//   REPROJ_2D3D     row = [zx zy Z0 Z1 Z2 beta beta^2 0]                       (8 doubles)
//   POSE_REG        row = [R_i(9) t_i(3) beta beta^2 0 0]                      (16 doubles)
//   POSE_REG_SPLIT  row = [R_i(9) t_i(3) betaR betaR^2 betaT betaT^2]          (16 doubles)
// Rows are sorted by the translation-side bound (beta / betaT) so that equal bounds are
// adjacent: eq. (14)'s min_i(beta_i - ||g_i||) then needs one square root per run of equal
// bounds instead of one per constraint (min/AND over constraints are order-free).
struct InstanceDesc {
    const double *rows;     // device
    int n;                  // rows (= N hypotheses / correspondences)
    int rows_bytes;         // n * ROW * 8, a multiple of 16
    const double *S0;       // device, n0 x 12
    int n0;
    int pad_;
    const int *perm;        // device, n: row of the caller's constraint i in the sorted table (Step I draws by i)
    double Rbar[9];
    double tbar[3];
    double K[4];            // fx fy cx cy
    double vscale[9];       // TRANS: v <- vscale v (PCA normalisation of the centre velocity, R-23); identity if off
};

constexpr int kMaxBatch = 96;
constexpr int kBlock = 128;       // walkers per CTA (one per thread)
constexpr int kMaxNT = 64;
constexpr int kMaxKStar = 20;
constexpr int kNumStats = 16;

struct WalkLaunch {
    const InstanceDesc *desc[kMaxBatch];      // device pointers, one per instance (gridDim.y)
    unsigned long long seed[kMaxBatch];
    long long walker_begin;
    long long num_walkers;                    // per instance
    int num_steps;
    int n_p, n_p_star, n_t;
    double omega0, v0, gamma, t_p, theta_p;
    double *out_samples;
    unsigned char *out_flags;
    int *out_trace;                           // nullable
    unsigned long long *stats;                // nullable, kNumStats counters
    int pairs_cap;                            // affine cooperative kernel: 32-byte entries of rowsA (max over the batch)
    int exact_only;                           // bit 0: plain fp64 kernel everywhere; bits 1, 2, 4: debug switches of walker_coop_kernel
};

int row_doubles(int residual_type);
// shared memory of the one-walker-per-thread kernel (the kernel of last resort: every instance must fit it)
constexpr size_t kMaxStageBytes = 200 * 1024;
size_t plain_kernel_smem_bytes(int rows_bytes, int n_t);

// walker_kernel.cu
cudaError_t launch_walkers(int residual_type, int mode, bool stats, const WalkLaunch &L, int n_instances,
                           int max_rows_bytes, cudaStream_t stream, std::string *why);

// walker_coop_kernel.cu: warp-cooperative, fp32-certified kernel for ROT mode on REG / POSE_REG / POSE_REG_SPLIT
bool coop_path_available(int residual_type, int mode, int n_p, int max_n);
cudaError_t launch_walkers_coop(int residual_type, const WalkLaunch &L, int n_instances, int max_rows_bytes,
                                cudaStream_t stream);

// walker_dense_kernel.cu: the dense variant of the above (every perturbation against every constraint), N_P > 32 on short tables
cudaError_t launch_walkers_coop_dense(int residual_type, const WalkLaunch &L, int n_instances, int max_rows_bytes,
                                      cudaStream_t stream);

// walker_coop_reproj_kernel.cu: the same organisation for the reprojection residual (ROT mode)
cudaError_t launch_walkers_coop_reproj(int residual_type, const WalkLaunch &L, int n_instances, int max_rows_bytes,
                                       cudaStream_t stream);

// walker_coop_trans_kernel.cu: warp-cooperative fp64 kernel for TRANS mode (Alg. A8), all residuals
cudaError_t launch_walkers_coop_trans(int residual_type, const WalkLaunch &L, int n_instances, int max_rows_bytes,
                                      cudaStream_t stream);

// compact_kernel.cu: t <- t - R c on n poses (back from the pivot-relative translation, closure_set_pivot)
cudaError_t launch_pivot_back(double *poses, long long n, const double *pivot, cudaStream_t stream);

// step1_kernel.cu: Step I trials (RANSAG with Arun's method for Ex.2, convex combinations for Ex.3)
cudaError_t launch_step1(int residual_type, const InstanceDesc *d_desc, int rows_bytes, long long trial_begin,
                         long long num_trials, unsigned long long seed, double *out_poses, unsigned char *out_ok,
                         cudaStream_t stream);

// compact_kernel.cu
size_t compact_scratch_bytes(long long n);
cudaError_t launch_compact(const double *samples, const unsigned char *flags, long long n, double *out,
                           long long *out_count, void *scratch, cudaStream_t stream);
// the same kernel on the file-scope static scratch of compact_kernel.cu (closure_compact_static: allocates nothing)
cudaError_t launch_compact_static(const double *samples, const unsigned char *flags, long long n, double *out,
                                  long long *out_count, cudaStream_t stream);

// alu_peak.cu
cudaError_t measure_alu_peak(int precision, double *flops_per_s, double *seconds, cudaStream_t stream);

// miniball.cpp (host)
struct Ball {
    double center[4];
    double sq_radius;
    long long support[5];
    int n_support;
};
// Gaertner-style exact smallest enclosing ball of n points in R^d (d <= 4), points row-major.
bool miniball(const double *pts, long long n, int d, Ball *out);
// The same solver over an abstract cloud: the pivot step ("the point farthest from the centre") is the
// only pass over all points; everything else touches single points by index.
struct PointSource {
    virtual ~PointSource() {}
    virtual bool farthest(const double *center, long long *index, double *sq_dist) = 0;   // lowest index among ties
    virtual const double *point(long long i) = 0;                                           // valid until the next call
};
bool miniball_source(PointSource *src, long long n, int d, Ball *out);

// megb_kernels.cu: Step III with the cloud kept on the device.  Quaternion
// embedding + sign alignment in one pass, then the miniball pivot as a max-reduction per iteration.
struct DeviceMegb;
DeviceMegb *device_megb_create(cudaError_t *err);
cudaError_t device_megb_prepare(DeviceMegb *m, const double *d_samples, long long count, const double qbar[4],
                                cudaStream_t stream);
PointSource *device_megb_quats(DeviceMegb *m);     // cloud of aligned unit quaternions in R^4
PointSource *device_megb_trans(DeviceMegb *m);     // cloud of translations in R^3
cudaError_t device_megb_status(DeviceMegb *m);
void device_megb_accounting(DeviceMegb *m, double *d2h_bytes, double *max_pivot_seconds, int *pivots);
void device_megb_destroy(DeviceMegb *m);
void rotation_to_quat(const double R[9], double q[4]);
void quat_to_rotation(const double q[4], double R[9]);
bool project_so3(const double M[9], double R[9]);   // nearest rotation to M (polar factor)
// sqrtm(Cov(t_j)) / sqrt(lambda_max) of the translations of n0 poses (n0 x 12); identity if there is no spread
void pca_velocity_scale(const double *poses, int n0, double S[9]);

}  // namespace closure
