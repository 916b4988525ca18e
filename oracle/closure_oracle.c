/*
 * closure_oracle.c -- plain CPU oracle for the CLOSURE boundary walk (arXiv 2403.09990).
 *
 * TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may build, load or call this file.
 * It shares no code, header, table or constant generator with the CUDA path under
 * paper_2403_09990_b200/csrc/, and neither includes the other.
 *
 * What it is: the walk of PAPER.md Alg. 2 (rotation-boundary sampler)
 * and Alg. A8 (translation-boundary sampler) transcribed step by step
 * in the paper's order and notation, in fp64, one pose evaluation at a time, with no
 * blocking, fusion, algebraic reuse or early exit beyond what the listings state.  Where
 * the paper is silent or garbled the reading is the one listed in DESIGN.md ("Readings",
 * R-1 ... R-20, same numbering as SURVEY.md section 8(c) S-n); each is marked below.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): Philox known-answer vectors; Exp-map
 * identities; Frobenius/geodesic identity for Example 3; generating pose inside the PURSE;
 * rotation-frozen walk against the closed-form ray exit from an intersection of balls
 * (PAPER.md:168); N=1 sphere case; feasibility of every emitted sample; replay;
 * permutation invariance; brute-force grid extent (Prop. 4).
 * Parity with the AUTHORS' implementation is unpinned (no code, data or printed worked
 * example exists; the perturbation distribution, R-6, is this build's reading).
 *
 * Build: gcc -O2 -std=c99 -fopenmp -shared -fPIC (see oracle/__init__.py).  No -ffast-math,
 * no FMA contraction (-ffp-contract=off): every product and sum below rounds once.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define ORA_REPROJ_2D3D 1
#define ORA_REG_3D3D 2
#define ORA_POSE_REG 3
#define ORA_POSE_REG_SPLIT 4
#define ORA_REG_3D3D_ELL 5      /* eq. (6) with a general Lambda_i: ellipsoids */
#define ORA_REPROJ_2D3D_ELL 6   /* eq. (6) with a general Lambda_i: ellipses */
#define ORA_MODE_ROT 0
#define ORA_MODE_TRANS 1

static const double ORA_PI = 3.14159265358979323846;

/* ------------------------------------------------------------------ Philox4x32-10 */
/* Salmon, Moraes, Dror, Shaw, "Parallel random numbers: as easy as 1, 2, 3" (SC'11):
 * 10 rounds; multipliers 0xD2511F53 / 0xCD9E8D57; Weyl key increments 0x9E3779B9 /
 * 0xBB67AE85.  north_star fixes this generator; R-5 fixes the counter layout. */
void ora_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
        uint64_t p1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
        uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
        uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
        uint32_t n0 = hi1 ^ c1 ^ k0;
        uint32_t n1 = lo1;
        uint32_t n2 = hi0 ^ c3 ^ k1;
        uint32_t n3 = lo0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* R-5: X(w, s, j, tag) = Philox(counter = (w_lo32, s, j, tag | w_hi32 << 8), key = seed). */
static void walk_random(uint64_t seed, uint64_t w, uint32_t s, uint32_t j, uint32_t tag, uint32_t out[4])
{
    uint32_t ctr[4], key[2];
    ctr[0] = (uint32_t)(w & 0xFFFFFFFFu);
    ctr[1] = s;
    ctr[2] = j;
    ctr[3] = tag | ((uint32_t)(w >> 32) << 8);
    key[0] = (uint32_t)(seed & 0xFFFFFFFFu);
    key[1] = (uint32_t)(seed >> 32);
    ora_philox4x32_10(ctr, key, out);
}

/* R-5: uniform in (-1, 1): xi = (2x + 1) 2^-32 - 1, exact in fp64. */
double ora_u32_to_pm1(uint32_t x)
{
    return (2.0 * (double)x + 1.0) * (1.0 / 4294967296.0) - 1.0;
}

/* ------------------------------------------------------------------ small 3x3 helpers */
static void mat3_mul(const double A[9], const double B[9], double C[9])
{
    for (int r = 0; r < 3; ++r)
        for (int c = 0; c < 3; ++c)
            C[3 * r + c] = A[3 * r + 0] * B[0 + c] + A[3 * r + 1] * B[3 + c] + A[3 * r + 2] * B[6 + c];
}

static void mat3_mul_bt(const double A[9], const double B[9], double C[9]) /* C = A B^T */
{
    for (int r = 0; r < 3; ++r)
        for (int c = 0; c < 3; ++c)
            C[3 * r + c] = A[3 * r + 0] * B[3 * c + 0] + A[3 * r + 1] * B[3 * c + 1] + A[3 * r + 2] * B[3 * c + 2];
}

static void mat3_vec(const double A[9], const double x[3], double y[3])
{
    for (int r = 0; r < 3; ++r)
        y[r] = A[3 * r + 0] * x[0] + A[3 * r + 1] * x[1] + A[3 * r + 2] * x[2];
}

/* Exp(phi) = I + A [phi]x + B [phi]x^2, A = sin(th)/th, B = 2 sin^2(th/2)/th^2 (Rodrigues);
 * th < 1e-4: A = 1 - th^2/6, B = 1/2 - th^2/24.  (SURVEY.md 8(c).) */
void ora_exp_so3(const double phi[3], double R[9])
{
    double th2 = phi[0] * phi[0] + phi[1] * phi[1] + phi[2] * phi[2];
    double th = sqrt(th2);
    double A, B;
    if (th < 1e-4) {
        A = 1.0 - th2 / 6.0;
        B = 0.5 - th2 / 24.0;
    } else {
        double sh = sin(0.5 * th);
        A = sin(th) / th;
        B = 2.0 * sh * sh / th2;
    }
    double K[9] = { 0.0, -phi[2], phi[1], phi[2], 0.0, -phi[0], -phi[1], phi[0], 0.0 };
    double K2[9];
    mat3_mul(K, K, K2);
    for (int e = 0; e < 9; ++e)
        R[e] = ((e % 4 == 0) ? 1.0 : 0.0) + A * K[e] + B * K2[e];
}

/* ------------------------------------------------------------------ residuals, PURSE */
int ora_num_constraints(int type, int n)
{
    return type == ORA_POSE_REG_SPLIT ? 2 * n : n;
}

static int row_len(int type)
{
    switch (type) {
    case ORA_REPROJ_2D3D: return 5;      /* [z(2) Z(3)] */
    case ORA_REG_3D3D: return 6;         /* [a(3) b(3)] */
    case ORA_REG_3D3D_ELL: return 15;    /* [a(3) b(3) Lambda(9 row-major)] */
    case ORA_REPROJ_2D3D_ELL: return 9;  /* [z(2) Z(3) Lambda(4 row-major)] */
    default: return 12;                  /* [R_i(9 row-major) t_i(3)] */
    }
}

/* Squared norm of the residual of constraint c at pose (R, t), summed left to right.
 *   Ex.1 eq.(2), Pi(v) = [v1/v3, v2/v3] PAPER.md:50, pixels through K (BASELINE
 *        config 3); depth <= 0 counts as violated with norm +inf (R-10).
 *   Ex.2 eq.(3) PAPER.md:33.
 *   Ex.3 eq.(4) PAPER.md:39 (stacked, one bound) or PURSEreg PAPER.md:173 (split: constraint
 *        2i bounds ||vec(R)-vec(R_i)||, constraint 2i+1 bounds ||t-t_i||) (R-13).
 * Lambda_i = I (R-14), except the _ELL types: ||g||_Lambda^2 = g^T Lambda_i g, eq. (6) PAPER.md:58,
 * written out as the double sum over the entries of Lambda_i. */
double ora_residual_sq(int type, int c, const double *meas, const double *K, const double R[9], const double t[3])
{
    double sq = 0.0;
    if (type == ORA_REG_3D3D) {
        const double *a = meas + 6 * c, *b = a + 3;
        double Ra[3];
        mat3_vec(R, a, Ra);
        for (int r = 0; r < 3; ++r) {
            double g = b[r] - (Ra[r] + t[r]);
            sq = sq + g * g;
        }
    } else if (type == ORA_REG_3D3D_ELL) {
        const double *a = meas + 15 * c, *b = a + 3, *Lam = a + 6;
        double Ra[3], g[3];
        mat3_vec(R, a, Ra);
        for (int r = 0; r < 3; ++r) g[r] = b[r] - (Ra[r] + t[r]);
        for (int r = 0; r < 3; ++r)
            for (int q = 0; q < 3; ++q) sq = sq + g[r] * Lam[3 * r + q] * g[q];
    } else if (type == ORA_REPROJ_2D3D_ELL) {
        const double *z = meas + 9 * c, *Z = z + 2, *Lam = z + 5;
        double p[3], g[2];
        mat3_vec(R, Z, p);
        for (int r = 0; r < 3; ++r) p[r] = p[r] + t[r];
        if (!(p[2] > 0.0)) return INFINITY;
        g[0] = z[0] - (K[0] * (p[0] / p[2]) + K[2]);
        g[1] = z[1] - (K[1] * (p[1] / p[2]) + K[3]);
        for (int r = 0; r < 2; ++r)
            for (int q = 0; q < 2; ++q) sq = sq + g[r] * Lam[2 * r + q] * g[q];
    } else if (type == ORA_REPROJ_2D3D) {
        const double *z = meas + 5 * c, *Z = z + 2;
        double p[3];
        mat3_vec(R, Z, p);
        for (int r = 0; r < 3; ++r) p[r] = p[r] + t[r];
        if (!(p[2] > 0.0)) return INFINITY;
        double u = K[0] * (p[0] / p[2]) + K[2];
        double v = K[1] * (p[1] / p[2]) + K[3];
        double g0 = z[0] - u, g1 = z[1] - v;
        sq = g0 * g0 + g1 * g1;
    } else if (type == ORA_POSE_REG) {
        const double *Ri = meas + 12 * c, *ti = Ri + 9;
        for (int e = 0; e < 9; ++e) {
            double g = R[e] - Ri[e];
            sq = sq + g * g;
        }
        for (int r = 0; r < 3; ++r) {
            double g = t[r] - ti[r];
            sq = sq + g * g;
        }
    } else { /* ORA_POSE_REG_SPLIT */
        const double *Ri = meas + 12 * (c / 2), *ti = Ri + 9;
        if (c % 2 == 0) {
            for (int e = 0; e < 9; ++e) {
                double g = R[e] - Ri[e];
                sq = sq + g * g;
            }
        } else {
            for (int r = 0; r < 3; ++r) {
                double g = t[r] - ti[r];
                sq = sq + g * g;
            }
        }
    }
    return sq;
}

/* in_purse: every constraint holds, tested on squared norms, beta^2 = beta*beta (R-9).
 * PURSE definition PAPER.md:63. */
int ora_in_purse(int type, int n, const double *meas, const double *beta, const double *K,
                 const double R[9], const double t[3])
{
    int nc = ora_num_constraints(type, n);
    for (int c = 0; c < nc; ++c) {
        double sq = ora_residual_sq(type, c, meas, K, R, t);
        if (!(sq <= beta[c] * beta[c])) return 0;
    }
    return 1;
}

/* Heuristic distance to the boundary, eq.(14): min_i (beta_i - ||g_i||). */
double ora_margin(int type, int n, const double *meas, const double *beta, const double *K,
                  const double R[9], const double t[3])
{
    int nc = ora_num_constraints(type, n);
    double d = INFINITY;
    for (int c = 0; c < nc; ++c) {
        double m = beta[c] - sqrt(ora_residual_sq(type, c, meas, K, R, t));
        if (m < d) d = m;
    }
    return d;
}

/* ------------------------------------------------------------------ the walk */
typedef struct {
    int mode;                 /* ORA_MODE_ROT: Alg. 2; ORA_MODE_TRANS: Alg. A8 */
    int n_p, n_p_star, n_t;   /* N_P, N_P*, N_T */
    double omega0, v0, gamma, t_p, theta_p;
    double vel_scale[9];      /* PCA normalisation of the centre velocity (R-23); I if off */
    double pivot[3];          /* body pivot c of update_rotation (R-1 alternative); 0: rotation about the origin */
} ora_params;

/* random unit vector from two uniforms (R-4): z = xi0, phi = pi (xi1 + 1). */
static void unit_vector(uint32_t x0, uint32_t x1, double u[3])
{
    double z = ora_u32_to_pm1(x0);
    double phi = ORA_PI * (ora_u32_to_pm1(x1) + 1.0);
    double s = sqrt(1.0 - z * z);
    u[0] = s * cos(phi);
    u[1] = s * sin(phi);
    u[2] = z;
}

/* axis-angle (u, theta) of a rotation matrix: v = vee(M - M^T) = 2 sin(theta) u,
 * tr(M) - 1 = 2 cos(theta); theta = atan2(|v|, tr - 1). */
static double axis_angle(const double M[9], double u[3])
{
    double v[3] = { M[7] - M[5], M[2] - M[6], M[3] - M[1] };
    double nv = sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
    double tr = M[0] + M[4] + M[8];
    double theta = atan2(nv, tr - 1.0);
    if (nv > 0.0) {
        u[0] = v[0] / nv; u[1] = v[1] / nv; u[2] = v[2] / nv;
    } else {
        u[0] = u[1] = u[2] = 0.0;
    }
    return theta;
}

typedef struct { double d; int j; } ranked;

/* order: d descending, then j ascending (R-8) */
static int ranked_before(const ranked *a, const ranked *b)
{
    if (a->d > b->d) return 1;
    if (a->d < b->d) return 0;
    return a->j < b->j;
}

/* One walker, all N_I iterations.  trace/slack may be NULL.
 *   trace[s-1] = m_0 | (j_{k_0} << 8), m_0 = 0 when no (k, m) was feasible.
 *   slack[s-1] = how close the closest decision of iteration s was to flipping:
 *                min over the examined ladder candidates of |margin(candidate)| and over
 *                consecutive ranks 1..N_P*+1 of the gap in d.  (Parity protocol.) */
static void walk_one(int type, int n, const double *meas, const double *beta, const double *K,
                     const ora_params *P, const double *S0, int n0, const double Rbar[9],
                     const double tbar[3], uint64_t w, int n_steps, uint64_t seed,
                     double *sample, unsigned char *on_boundary, int32_t *trace, double *slack,
                     double *Rj, double *tj, ranked *rk)
{
    const double *init = S0 + 12 * (size_t)(w % (uint64_t)n0);   /* repeat(S_0, N_W) */
    double R[9], t[3];
    memcpy(R, init, 9 * sizeof(double));
    memcpy(t, init + 9, 3 * sizeof(double));

    /* Alg. 2 l.8 / Alg. A8 l.8 + PAPER.md:293, 324: velocity pointing away from the centre */
    uint32_t x[4];
    double rnd[3], omega[3] = { 0, 0, 0 }, v[3] = { 0, 0, 0 };
    walk_random(seed, w, 0u, 0u, 0u, x);
    unit_vector(x[0], x[1], rnd);
    if (P->mode == ORA_MODE_ROT) {
        double Rrel[9], u[3];
        mat3_mul_bt(R, Rbar, Rrel);                    /* R_0 Rbar^T (R-2) */
        double theta = axis_angle(Rrel, u);
        if (theta < 1e-12) u[0] = u[1] = u[2] = 0.0;   /* R-3 */
        for (int r = 0; r < 3; ++r) omega[r] = P->omega0 * (u[r] + rnd[r]);
    } else {
        double dvec[3] = { t[0] - tbar[0], t[1] - tbar[1], t[2] - tbar[2] };
        double nd = sqrt(dvec[0] * dvec[0] + dvec[1] * dvec[1] + dvec[2] * dvec[2]);
        double v_raw[3];
        for (int r = 0; r < 3; ++r) {
            double dir = nd < 1e-12 ? 0.0 : dvec[r] / nd;   /* R-3 */
            v_raw[r] = P->v0 * (dir + rnd[r]);
        }
        /* "additional normalization to the translation velocity according to the PCA analysis of S_0"
         * (App. E): v <- S v, S = sqrtm(Cov(S_t0)) / sqrt(lambda_max) (R-23) */
        for (int r = 0; r < 3; ++r)
            v[r] = P->vel_scale[3 * r] * v_raw[0] + P->vel_scale[3 * r + 1] * v_raw[1] + P->vel_scale[3 * r + 2] * v_raw[2];
    }

    int hit = 0;
    for (int s = 1; s <= n_steps; ++s) {                    /* Alg. 2 l.11 */
        /* l.12-15: N_P perturbations and their distance to the boundary */
        for (int j = 0; j < P->n_p; ++j) {
            walk_random(seed, w, (uint32_t)s, (uint32_t)j, 1u, x);
            double xi[3] = { ora_u32_to_pm1(x[0]), ora_u32_to_pm1(x[1]), ora_u32_to_pm1(x[2]) };
            double *Rp = Rj + 9 * j, *tp = tj + 3 * j;
            if (P->mode == ORA_MODE_ROT) {                  /* t_j = t* + perturbation(t_p) (R-6) */
                memcpy(Rp, R, 9 * sizeof(double));
                for (int r = 0; r < 3; ++r) tp[r] = t[r] + P->t_p * xi[r];
            } else {                                        /* R_j = R_p R*, A8 l.13-14, A9 (R-6, R-7) */
                double phi[3] = { P->theta_p * xi[0], P->theta_p * xi[1], P->theta_p * xi[2] };
                double E[9];
                ora_exp_so3(phi, E);
                mat3_mul(E, R, Rp);
                memcpy(tp, t, 3 * sizeof(double));
            }
            rk[j].d = ora_margin(type, n, meas, beta, K, Rp, tp);   /* eq. (14) */
            rk[j].j = j;
        }
        /* l.17: top_k_indices -- plain selection of the N_P* best by (d desc, j asc) (R-8) */
        int kk = P->n_p_star;
        for (int k = 0; k < kk + 1 && k < P->n_p; ++k) {     /* one extra rank for the slack */
            int best = k;
            for (int q = k + 1; q < P->n_p; ++q)
                if (ranked_before(&rk[q], &rk[best])) best = q;
            ranked tmp = rk[k]; rk[k] = rk[best]; rk[best] = tmp;
        }
        double sl = INFINITY;
        if (slack) {
            for (int k = 0; k < kk && k + 1 < P->n_p; ++k) {
                double gap = rk[k].d - rk[k + 1].d;
                if (gap < sl) sl = gap;              /* NaN-free: inf - inf only if both -inf */
                if (isnan(gap)) sl = 0.0;
            }
        }
        /* l.18-29: ladder Delta T = gamma^(m-1); first feasible (m ascending, k ascending) wins */
        int m0 = 0, j0 = 0;
        double dT = 1.0;
        for (int m = 1; m <= P->n_t && m0 == 0; ++m) {
            for (int k = 0; k < kk; ++k) {
                const double *Rp = Rj + 9 * rk[k].j, *tp = tj + 3 * rk[k].j;
                double Rc[9], tc[3];
                if (P->mode == ORA_MODE_ROT) {              /* update_rotation: Exp(dT w) R (R-1) */
                    double phi[3] = { dT * omega[0], dT * omega[1], dT * omega[2] };
                    double E[9];
                    ora_exp_so3(phi, E);
                    mat3_mul(E, Rp, Rc);
                    memcpy(tc, tp, 3 * sizeof(double));
                    if (P->pivot[0] != 0.0 || P->pivot[1] != 0.0 || P->pivot[2] != 0.0) {
                        /* rotate about the body point c ("object movement"): the image
                         * R c + t of c stays where it is, t' = t + (R - R') c  (R-1, alternative reading) */
                        for (int r = 0; r < 3; ++r) {
                            double before = Rp[3 * r] * P->pivot[0] + Rp[3 * r + 1] * P->pivot[1] + Rp[3 * r + 2] * P->pivot[2];
                            double after = Rc[3 * r] * P->pivot[0] + Rc[3 * r + 1] * P->pivot[1] + Rc[3 * r + 2] * P->pivot[2];
                            tc[r] = tp[r] + (before - after);
                        }
                    }
                } else {                                    /* update_translation: t + dT v (R-7) */
                    memcpy(Rc, Rp, 9 * sizeof(double));
                    for (int r = 0; r < 3; ++r) tc[r] = tp[r] + dT * v[r];
                }
                int ok = ora_in_purse(type, n, meas, beta, K, Rc, tc);
                if (slack) {
                    double mg = fabs(ora_margin(type, n, meas, beta, K, Rc, tc));
                    if (mg < sl) sl = mg;
                }
                if (ok) {                                   /* l.25-28 */
                    memcpy(R, Rc, sizeof(Rc));
                    memcpy(t, tc, sizeof(tc));
                    m0 = m; j0 = rk[k].j;
                    break;
                }
            }
            dT = dT * P->gamma;                             /* l.20 */
        }
        /* R-11: nothing feasible -> pose unchanged.  R-12: sticky boundary flag. */
        if (m0 != 1) hit = 1;
        if (trace) trace[s - 1] = (int32_t)(m0 | (j0 << 8));
        if (slack) slack[s - 1] = sl;
    }
    memcpy(sample, R, 9 * sizeof(double));                  /* l.30 */
    memcpy(sample + 9, t, 3 * sizeof(double));
    *on_boundary = (unsigned char)hit;
}

/* Walk the listed walkers.  Returns 0, or -1 on bad arguments / allocation failure.
 * n_threads > 1 splits WALKERS over OpenMP threads (walkers are independent);
 * the per-walker computation is unchanged. */
int ora_walk(int type, int n, const double *meas, const double *beta, const double *K,
             const ora_params *P, const double *S0, int n0, const double *Rbar, const double *tbar,
             const int64_t *walker_ids, int64_t n_walkers, int n_steps, uint64_t seed,
             double *out_samples, unsigned char *out_on_boundary, int32_t *out_trace,
             double *out_slack, int n_threads)
{
    if (n <= 0 || n0 <= 0 || P->n_p <= 0 || P->n_p_star <= 0 || P->n_p_star > P->n_p || P->n_t <= 0)
        return -1;
    int fail = 0;
    (void)row_len;
#pragma omp parallel num_threads(n_threads > 0 ? n_threads : 1)
    {
        double *Rj = (double *)malloc(sizeof(double) * 9 * (size_t)P->n_p);
        double *tj = (double *)malloc(sizeof(double) * 3 * (size_t)P->n_p);
        ranked *rk = (ranked *)malloc(sizeof(ranked) * (size_t)P->n_p);
        if (!Rj || !tj || !rk) {
#pragma omp atomic write
            fail = 1;
        } else {
#pragma omp for schedule(dynamic, 1)
            for (int64_t q = 0; q < n_walkers; ++q) {
                walk_one(type, n, meas, beta, K, P, S0, n0, Rbar, tbar, (uint64_t)walker_ids[q],
                         n_steps, seed, out_samples + 12 * q, out_on_boundary + q,
                         out_trace ? out_trace + (size_t)q * n_steps : NULL,
                         out_slack ? out_slack + (size_t)q * n_steps : NULL, Rj, tj, rk);
            }
        }
        free(Rj); free(tj); free(rk);
    }
    return fail ? -1 : 0;
}

/* Stable compaction: keep flagged samples in walker order (north_star (2)). */
int64_t ora_compact(const double *samples, const unsigned char *flags, int64_t n, double *out)
{
    int64_t cnt = 0;
    for (int64_t q = 0; q < n; ++q)
        if (flags[q]) {
            memcpy(out + 12 * cnt, samples + 12 * q, 12 * sizeof(double));
            ++cnt;
        }
    return cnt;
}
