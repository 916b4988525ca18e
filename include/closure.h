/*
 * closure.h -- C ABI of libclosure_b200: the data-parallel hot path of CLOSURE
 * (arXiv 2403.09990) on NVIDIA B200 (sm_100a).
 *
 * "PAPER.md:<n>" cites /root/reference/PAPER.md line n; "R-n" cites the numbered readings
 * of silent / garbled passages in DESIGN.md.
 *
 * The path: boundary walks (Step II: Alg. 2, Alg. 3 PAPER.md:295-322,
 * Alg. A8/A9 PAPER.md:1001-1099) -> stream compaction of boundary samples -> minimum
 * enclosing geodesic ball (Step III).  Step I (initial poses S_0,
 * PAPER.md:201, 217-219) is off the path and enters as data through closure_set_init.
 *
 * Conventions
 *   - Plain C99, no exceptions cross the boundary.  Every call returns an int status:
 *     CLOSURE_OK (0) or a negative CLOSURE_E* code; closure_last_error(h) gives the text of
 *     the last failure on that handle (owned by the handle; valid until the next call on it).
 *   - "host" pointers are ordinary CPU memory, "DEVICE" pointers are CUDA device memory of the
 *     current device.  The caller owns every buffer it passes; inputs of closure_create /
 *     closure_set_init are copied; outputs are written into caller-allocated buffers.
 *   - `cuda_stream` is a cudaStream_t passed as void* (NULL = default stream).  Calls marked
 *     ASYNC only enqueue work on it and do not synchronise with the host.
 *   - There is no CPU fallback and no other backend: without a usable CUDA device every
 *     compute call returns CLOSURE_ECUDA.
 *   - A pose is 12 doubles: R row-major (9) then t (3).  One sample record = 96 bytes.
 */
#ifndef CLOSURE_B200_H
#define CLOSURE_B200_H

#ifdef __cplusplus
extern "C" {
#endif

#define CLOSURE_ABI_VERSION 2

/* status codes */
#define CLOSURE_OK 0
#define CLOSURE_EINVAL (-1)   /* bad enum / size / NULL / non-finite input / beta <= 0 / n_p_star > n_p */
#define CLOSURE_EINIT (-2)    /* an initial pose is not inside the PURSE (PAPER.md:217-219 admit only such) */
#define CLOSURE_ENOINIT (-3)  /* closure_sample before closure_set_init */
#define CLOSURE_ECUDA (-4)    /* CUDA runtime failure (message in closure_last_error) */
#define CLOSURE_ENOMEM (-5)
#define CLOSURE_EUNSUPPORTED (-6) /* combination not built (e.g. n_p_star > 32) */
#define CLOSURE_ETOOLARGE (-7)    /* closure_compact_static: n exceeds CLOSURE_COMPACT_STATIC_MAX */

/* residual g(x, y_i) -- eqs. (2)-(4).  Measurement row layouts (doubles):
 *   CLOSURE_REPROJ_2D3D     [z(2) Z(3)]          g = z - Pi(K (R Z + t)), pixels; depth<=0 violates (R-10)
 *   CLOSURE_REG_3D3D        [a(3) b(3)]          g = b - (R a + t)
 *   CLOSURE_POSE_REG        [R_i(9 row-major) t_i(3)]   g = [vec(R)-vec(R_i); t-t_i], ONE bound per hypothesis
 *   CLOSURE_POSE_REG_SPLIT  same rows; TWO bounds per hypothesis, betas[2i] on ||vec(R)-vec(R_i)||,
 *                           betas[2i+1] on ||t-t_i||  (PURSEreg; R-13)
 *   CLOSURE_REPROJ_2D3D_ELL [z(2) Z(3) Lambda(4: 2x2 row-major)]    the same g, bounded in the ellipse norm
 *   CLOSURE_REG_3D3D_ELL    [a(3) b(3) Lambda(9: 3x3 row-major)]    ||g||_Lambda = sqrt(g^T Lambda_i g) <= beta_i
 * Lambda_i = I for the first four (R-14).  The _ELL types carry the positive definite Lambda_i of eq. (6)
 * (the ellipses / ellipsoids of PAPER.md:179-191): symmetric, positive definite
 * (CLOSURE_EINVAL otherwise).  Rotation sampler: CLOSURE_REG_3D3D_ELL runs on the warp-cooperative certified-fp32 kernel
 * (the pair carries the quadratic form d^T Lambda_i d; same decisions as the fp64 kernel, bit for bit), and so does
 * CLOSURE_REPROJ_2D3D_ELL (rows whitened by the Cholesky factor of Lambda_i at every set-up); translation sampler: the
 * warp-cooperative fp64 kernel.  There is no fp32 mode (precision = 32) for them: CLOSURE_EUNSUPPORTED.
 * Step I: as for the ball forms; the 2D point of Ex.1 is then uniform in the ellipse (R-24). */
enum { CLOSURE_REPROJ_2D3D = 1, CLOSURE_REG_3D3D = 2, CLOSURE_POSE_REG = 3, CLOSURE_POSE_REG_SPLIT = 4,
       CLOSURE_REG_3D3D_ELL = 5, CLOSURE_REPROJ_2D3D_ELL = 6 };

/* which boundary is sampled: CLOSURE_MODE_ROT = Alg. 2 (fixed angular velocity, translation
 * perturbations); CLOSURE_MODE_TRANS = Alg. A8 (fixed centre velocity, rotation perturbations). */
enum { CLOSURE_MODE_ROT = 0, CLOSURE_MODE_TRANS = 1 };

/* The paper's simulation-parameter tuple P (values PAPER.md:374, 440, 464). */
typedef struct {
    int mode;        /* CLOSURE_MODE_* */
    int n_p;         /* N_P   perturbations per iteration, >= 1 */
    int n_p_star;    /* N_P*  kept perturbations, 1..min(n_p, 32) */
    int n_t;         /* N_T   ladder length, 1..64; Delta T_m = gamma^(m-1) */
    double omega0;   /* base angular velocity magnitude (ROT) */
    double v0;       /* base centre velocity magnitude (TRANS) */
    double gamma;    /* time-step decay, in (0, 1] */
    double t_p;      /* translation perturbation scale: uniform on [-t_p, t_p]^3 (R-6) */
    double theta_p;  /* rotation perturbation scale (the paper's R_p): rotation vector uniform on
                        [-theta_p, theta_p]^3 (R-6) */
    int precision;   /* 64: every decision is the fp64 decision (the parity path).  32: rotation sampler only --
                        the fp32 ranking is taken as it is and a ladder candidate whose fp32 bound straddles the
                        threshold counts as violated (no fp64 fall-back; every emitted pose is still inside S);
                        poses stay fp64.  Differs from 64 only where an fp32 error bound straddles a
                        threshold; bench.py --precision 32 reports the measured difference. */
    int flags;       /* bit 0 (CLOSURE_FLAG_EXACT_ONLY): run the plain fp64 one-walker-per-thread kernel even where
                        the warp-cooperative fp32-certified kernel exists (same results bit for bit; for
                        verification and timing).  Bits 1, 2, 4 force the cooperative kernel's fp64 fall-back
                        paths (tests only): 2 = every ladder candidate is decided in fp64, 4 = every top-N_P*
                        ranking is redone in fp64, 16 = ... on all N_P perturbations. */
} closure_params;
#define CLOSURE_FLAG_EXACT_ONLY 1
#define CLOSURE_FLAG_PCA_VELOCITY 64 /* translation sampler: rescale the centre velocity by the relative spread of S_0's
                                        translations along their principal axes, v <- sqrtm(Cov) / sqrt(lambda_max) v
                                        (PAPER.md:324, 1074-1076); read by closure_set_init */
#define CLOSURE_FLAG_HOST_MEGB 8    /* closure_megb: copy the cloud to the host and run the miniball there, whatever its size */
#define CLOSURE_FLAG_ONE_WARP 128   /* rotation sampler, launches of at most 1,184 walkers: keep one warp per walker instead of the
                                        pair of warps one iteration apart (same results bit for bit; for verification and timing) */

typedef struct closure_s closure_t;   /* opaque; owns device copies of the instance and of S_0 */

/* Fill *p with the defaults this build uses for `residual_type` (paper values where units carry
 * over).  Returns CLOSURE_EINVAL on a bad type / NULL. */
int closure_default_params(int residual_type, closure_params *p);

/* Describe a PURSE  S = { (R,t) : ||g(x, y_i)|| <= beta_i } and upload it.
 *   measurements  host, n rows in the layout of `residual_type`
 *   betas         host, n bounds (2n for CLOSURE_POSE_REG_SPLIT), each finite and > 0
 *   intrinsics    host, {fx, fy, cx, cy}; required for CLOSURE_REPROJ_2D3D(_ELL), ignored (may be NULL) else
 *   p             walk parameters (copied)
 *   out           receives the handle; destroy with closure_destroy
 * Synchronous (small H2D copy).  Errors: CLOSURE_EINVAL, CLOSURE_ECUDA, CLOSURE_ENOMEM; CLOSURE_EUNSUPPORTED if the
 * constraint table (64 B per row, 128 B for pose regression) plus the ladder (2 KB per rung) exceeds the 200 KB a
 * CTA can stage (n <= 4096 otherwise: e.g. n <= 2,700 registration rows at n_t = 15).
 * Thread / stream safety: a handle carries per-handle device scratch (compaction tile states, statistics, closure_run's
 * buffers).  Use one handle from one host thread and ONE stream at a time; different handles are independent. */
int closure_create(int residual_type, const double *measurements, int n, const double *betas,
                   const double *intrinsics, const closure_params *p, closure_t **out);

/* Replace the walk parameters of an existing handle (same validation as closure_create). */
int closure_set_params(closure_t *h, const closure_params *p);

/* Body pivot of update_rotation (Alg. 2 l.20, which the paper never defines; R-1).
 * With pivot c (host, 3 doubles, in the frame of the source points a_i / Z_i) a rotation step keeps the image of
 * the body point c fixed:  R' = Exp(dT w) R,  t' = t + (R - R') c  -- the "object movement" reading of
 * PAPER.md:328, 336.  The default c = 0 is rotation about the origin of the source frame (t untouched).
 * Rotation sampler (CLOSURE_MODE_ROT) and residuals with source points (REG_3D3D, REPROJ_2D3D) only:
 * CLOSURE_EUNSUPPORTED otherwise for a non-zero pivot.  Invalidates S_0: call closure_set_init (or
 * closure_init_from_trials) again.  Inputs and outputs of every call stay in the caller's (R, t). */
int closure_set_pivot(closure_t *h, const double *pivot);

/* Give the initial pose set S_0 (output of Step I).  poses: host, n0 x 12.  Computes
 * R_bar = proj_SO(3)(sum R_j) and t_bar = mean t_j on the host (Alg. 2 l.3-4),
 * checks every pose against the PURSE (CLOSURE_EINIT if one is outside) and uploads.
 * mean_out (host, 12 doubles, may be NULL) receives [R_bar, t_bar]. */
int closure_set_init(closure_t *h, const double *poses, int n0, double *mean_out);

/* Step I: independent trials on the device.
 *   CLOSURE_REG_3D3D               RANSAG trial: 3 distinct random correspondences, Arun's least-squares rigid
 *                                  fit, kept iff the pose satisfies the PURSE
 *   CLOSURE_POSE_REG / _SPLIT      a random convex combination of the hypotheses (rotation = proj_SO(3) of the
 *                                  weighted sum), kept iff it satisfies the PURSE
 *   CLOSURE_REPROJ_2D3D            RANSAG trial: 3 distinct random constraints, a random 2D point inside each
 *                                  (uniform in the disc of radius beta_i around z_i), the perspective-3-point
 *                                  problem for the three rays; its (up to four) poses are tried in ascending
 *                                  order of the first depth and the first one that satisfies the PURSE is kept
 *                                  (R-24)
 * CLOSURE_EINVAL if a RANSAG residual has fewer than 3 constraints.
 * Trial k = trial_begin + q draws from Philox4x32-10 keyed by (seed; k) (R-21, R-22, R-24), so any trial can
 * be replayed alone.  ASYNC.
 *   out_poses  DEVICE, num_trials x 12 doubles: the candidate (R row-major, t), zeros where rejected
 *   out_ok     DEVICE, num_trials bytes: 1 iff the candidate is inside the PURSE
 * closure_compact(out_poses, out_ok) yields S_0 in trial order. */
int closure_init_sample(closure_t *h, long long trial_begin, long long num_trials, unsigned long long seed,
                        double *out_poses, unsigned char *out_ok, void *cuda_stream);

/* Step I end to end: num_trials trials (closure_init_sample from trial 0), compaction, and closure_set_init with
 * the first max_poses accepted poses.  Synchronises the stream.  *n0_out (may be NULL) = |S_0|.
 * CLOSURE_EINIT if no trial produced a pose inside the PURSE. */
int closure_init_from_trials(closure_t *h, long long num_trials, unsigned long long seed, int max_poses, int *n0_out,
                             void *cuda_stream);

/* Step II.  ASYNC.  Runs walkers w = walker_begin .. walker_begin + num_walkers - 1, each for
 * exactly num_steps iterations of Alg. 2 (ROT) / Alg. A8 (TRANS) from S_0[w mod n0]
 * (the paper's repeat(S_0, N_W)), with Philox4x32-10 randomness keyed by
 * (seed; w, iteration, perturbation) (R-5) so that any walker can be replayed alone.
 *   out_samples      DEVICE, num_walkers x 12 doubles: final (R*, t*)      (Alg. 2 l.30)
 *   out_on_boundary  DEVICE, num_walkers bytes: 1 iff some iteration could not take the full
 *                    step (m_0 > 1 or nothing feasible) (R-12)
 *   out_trace        DEVICE or NULL, num_walkers x num_steps int32: per iteration
 *                    m_0 | (j_{k_0} << 8), 0 when nothing was feasible (parity protocol)
 * closure_sample(h, W, S, seed, samples, flags, stream) of the north star is the
 * walker_begin = 0, out_trace = NULL case.  One launch takes at most 2^31 - 1 walkers (one CTA per walker in the
 * reprojection kernels; 258 GB of samples): more than that returns CLOSURE_ECUDA, split the range instead. */
int closure_sample_range(closure_t *h, long long walker_begin, long long num_walkers, int num_steps,
                         unsigned long long seed, double *out_samples, unsigned char *out_on_boundary,
                         int *out_trace, void *cuda_stream);
int closure_sample(closure_t *h, long long num_walkers, int num_steps, unsigned long long seed,
                   double *out_samples, unsigned char *out_on_boundary, void *cuda_stream);

/* Step II for a batch of independent instances in ONE launch (BASELINE config 5).  All handles
 * must share residual type, walk parameters and precision; N and S_0 may differ.  Instance b runs
 * walkers 0 .. walkers_per_instance-1 with seeds[b]; outputs are instance-major:
 * out_samples[(b * walkers_per_instance + w) * 12], out_on_boundary[b * walkers_per_instance + w].
 * handles / seeds: host arrays of n_instances.  ASYNC. */
int closure_sample_batch(closure_t *const *handles, int n_instances, long long walkers_per_instance,
                         int num_steps, const unsigned long long *seeds, double *out_samples,
                         unsigned char *out_on_boundary, void *cuda_stream);

/* Stable stream compaction of the samples whose flag is non-zero, in walker order.  ASYNC.
 *   samples, flags   DEVICE, n x 12 doubles / n bytes
 *   out_compacted    DEVICE, room for n x 12 doubles
 *   out_count        DEVICE, one long long: number of kept samples */
int closure_compact(closure_t *h, const double *samples, const unsigned char *flags, long long n,
                    double *out_compacted, long long *out_count, void *cuda_stream);

/* closure_compact without any allocation, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid it).  Same kernel, same result bit for bit; its scratch (8 bytes per tile of
 * 2,048 records) is a static device array inside the library, sized for at most CLOSURE_COMPACT_STATIC_MAX records
 * (32 KB + 8 B, held by every GPU that loads the library until exit).  Needs no handle.  ASYNC; calls no cudaMalloc,
 * cudaFree or allocating library routine (the first call on a device resolves the array's device address, once).
 *   samples, flags, out_compacted, out_count   DEVICE, as for closure_compact; sample buffers 16-byte aligned
 * Errors: CLOSURE_ETOOLARGE if n > CLOSURE_COMPACT_STATIC_MAX (nothing is launched; use closure_compact),
 * CLOSURE_EINVAL (negative n, NULL or misaligned buffers), CLOSURE_ECUDA.
 * ALL calls on one device share the one array: it is cleared at the start of every call on the caller's stream, and
 * two calls that can overlap on the GPU (different streams, or concurrent host threads) RACE -- serialise them. */
#define CLOSURE_COMPACT_STATIC_MAX 8388608
int closure_compact_static(const double *samples, const unsigned char *flags, long long n, double *out_compacted,
                           long long *out_count, void *cuda_stream);

/* Step III result.  Geodesic distance on SO(3): arccos((tr(C^T R) - 1) / 2). */
typedef struct {
    double R[9];              /* centre rotation C^ (row-major) */
    double t[3];              /* centre translation c^ */
    double rot_radius;        /* D^ in radians */
    double trans_radius;      /* d^ */
    long long rot_support[5]; /* indices (into the given samples) of the rotation ball's support set */
    long long trans_support[4];
    int n_rot_support, n_trans_support;
    double host_seconds;      /* wall time of Step III inside closure_megb, device passes and copies included
                                 (reported separately) */
    double d2h_bytes;         /* bytes closure_megb copied device -> host: the whole cloud (count x 96) on the host path;
                                 16 per pivot + 8 d per fetched support candidate on the device path */
    double max_pivot_seconds; /* device path: the slowest single pivot (launch + 16-byte copy + synchronise); 0 on the host path */
    int pivots;               /* device path: farthest-point launches of both balls; 0 on the host path */
    int pad_;
    double prepare_seconds;   /* device path: the embedding pass, including the (re)allocation of the per-device buffers when the
                                 cloud is larger than any seen before in this process (cudaMalloc: tens of ms, once per size) */
} closure_megb_result;

/* Step III (Alg. 1 l.6-7): minimum enclosing ball of {t} in R^3 and of the
 * sign-aligned unit quaternions {q(R)} in R^4 (R-15, R-16) by Gaertner's miniball.
 *   samples  DEVICE, count x 12 (e.g. closure_compact's output)
 * Synchronises `cuda_stream`.  The support basis is solved on the host; for count >= 4096 the cloud stays on
 * the device (one embedding pass, one max-reduction launch per miniball pivot, 16 bytes back per pivot),
 * smaller clouds -- or every cloud with CLOSURE_FLAG_HOST_MEGB -- are copied to the host.  Same result either way.
 * Errors: CLOSURE_EINVAL (count <= 0), CLOSURE_ENOINIT (R_bar needed for the sign), CLOSURE_ECUDA. */
int closure_megb(closure_t *h, const double *samples, long long count, closure_megb_result *out,
                 void *cuda_stream);

/* Whole path from host buffers: walk, compact, MEGB; samples never leave the device except the
 * compacted cloud for the miniball.  out_count (host, may be NULL) receives the number of
 * boundary samples.  Synchronous. */
int closure_run(closure_t *h, long long num_walkers, int num_steps, unsigned long long seed,
                closure_megb_result *out, long long *out_count, void *cuda_stream);

/* Counters of the last closure_sample* launch on this handle when statistics were enabled with
 * closure_enable_stats(h, 1): executed constraint evaluations per phase (for the roofline's
 * executed-flop count).  closure_get_stats synchronises the stream of that launch. */
typedef struct {
    unsigned long long perturb_pairs;   /* (perturbation, constraint) pairs evaluated in fp64, step a3 */
    unsigned long long ladder_pairs;    /* (candidate, constraint) pairs evaluated in fp64, step a5 */
    unsigned long long perturb_setups;  /* per-constraint set-ups (R-dependent part), a3 */
    unsigned long long ladder_setups;   /* per-(rung, constraint) set-ups, a5 */
    unsigned long long accepted_steps;  /* iterations that moved the walker */
    unsigned long long walker_steps;    /* walkers x iterations */
    unsigned long long perturb_pairs_f32; /* pairs evaluated in certified fp32, a3 */
    unsigned long long ladder_pairs_f32;  /* pairs evaluated in certified fp32 (rung screening + full rungs), a5 */
    unsigned long long fallback_steps;  /* iterations whose fp32 ranking was not certified (fp64 re-ranking) */
    unsigned long long verified_rungs;  /* ladder rungs evaluated in full (ROT) / candidates sent to fp64 (TRANS) */
    unsigned long long setup_cycles;    /* SM cycles the walkers' warps spent in the set-up that follows an accepted move
                                           (cooperative rotation-sampler kernels; 0 elsewhere) */
    unsigned long long total_cycles;    /* SM cycles of the walkers' warps from init to emit (same kernels) */
    unsigned long long threshold_probes;   /* branch and bound of eq. (14) (affine cooperative kernel): counts taken to find the threshold */
    unsigned long long survivors;          /* perturbations evaluated against all constraints (phase 2), summed over iterations */
    unsigned long long reserved_;
    unsigned long long threshold_failures; /* iterations in which no threshold separated the values (ties): fp64 on all N_P */
} closure_stats;
int closure_enable_stats(closure_t *h, int on);
int closure_get_stats(closure_t *h, closure_stats *out);

/* Measured CUDA-core peak of this device: a register-resident FMA chain, fp64 (precision = 64)
 * or fp32 (32).  Returns FLOP/s (FMA = 2) in *flops_per_s and the kernel time in *seconds.
 * precision = 4 measures the integer side instead: Philox4x32-10 calls per second (in *flops_per_s).
 * Synchronous.  Used as the roofline denominators for the walker kernel. */
int closure_alu_peak(int precision, double *flops_per_s, double *seconds, void *cuda_stream);

/* The host solver of Step III on its own: exact smallest enclosing ball of n points in R^d
 * (1 <= d <= 4), points row-major in HOST memory.  center (d doubles), radius, support (up to d+1
 * indices, ascending) and n_support are written.  Pure host code: needs no device. */
int closure_miniball_host(const double *points, long long n, int d, double *center, double *radius,
                          long long *support, int *n_support);

const char *closure_last_error(const closure_t *h);
const char *closure_strerror(int status);
int closure_abi_version(void);
void closure_destroy(closure_t *h);

#ifdef __cplusplus
}
#endif
#endif /* CLOSURE_B200_H */
