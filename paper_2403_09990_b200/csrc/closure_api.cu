// C ABI of libclosure_b200 (include/closure.h): argument validation, instance packing and
// upload, launches of the walker / compaction kernels on the caller's stream, and the host
// side of closure_megb.  No CPU fallback exists: every compute entry point needs a CUDA device.
#include <cuda_runtime.h>

#include <algorithm>
#include <chrono>
#include <cmath>
#include <cstring>
#include <mutex>
#include <new>
#include <numeric>
#include <string>
#include <vector>

#include "closure_internal.h"

using namespace closure;

struct closure_s {
    int type = 0;
    int n = 0;
    closure_params P{};
    std::vector<double> meas;        // as given (validation of S_0 on the host)
    std::vector<double> betas;
    double K[4] = { 0, 0, 0, 0 };
    InstanceDesc h_desc{};
    std::vector<int> order;          // sorted row k holds the caller's constraint order[k]
    double pivot[3] = { 0, 0, 0 };   // body pivot of update_rotation (closure_set_pivot, R-1); zero: rotation about the origin
    bool has_pivot = false;
    int n_pairs = 0;                 // pair-entries of the cooperative kernel's fp32 table: sum over runs of equal bound of ceil(len / 2)
    double *d_rows = nullptr;
    int *d_perm = nullptr;
    InstanceDesc *d_desc = nullptr;
    double *d_S0 = nullptr;
    bool has_init = false;
    void *d_scratch = nullptr;
    size_t scratch_bytes = 0;
    unsigned long long *d_stats = nullptr;
    bool stats_on = false;
    cudaStream_t last_stream = nullptr;
    // buffers of closure_run
    double *d_samples = nullptr, *d_compact = nullptr;
    unsigned char *d_flags = nullptr;
    long long *d_count = nullptr;
    long long run_capacity = 0;
    std::string err;
};

namespace {

constexpr long long kDeviceMegbMin = 4096;
constexpr int kMaxDevices = 64;
std::mutex g_megb_mutex;
DeviceMegb *g_megb[kMaxDevices] = { nullptr };   // device-side Step III state, one per device, kept for the process   // below this the D2H of the cloud is cheaper than the pivot launches

int fail(closure_t *h, int code, const std::string &msg)
{
    if (h) h->err = msg;
    return code;
}

int cuda_fail(closure_t *h, cudaError_t e, const char *what)
{
    return fail(h, CLOSURE_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

bool all_finite(const double *p, size_t n)
{
    for (size_t i = 0; i < n; ++i)
        if (!std::isfinite(p[i])) return false;
    return true;
}

int meas_cols(int type)
{
    switch (type) {
    case CLOSURE_REPROJ_2D3D: return 5;
    case CLOSURE_REG_3D3D: return 6;
    case CLOSURE_REG_3D3D_ELL: return 15;
    case CLOSURE_REPROJ_2D3D_ELL: return 9;
    case CLOSURE_POSE_REG:
    case CLOSURE_POSE_REG_SPLIT: return 12;
    default: return 0;
    }
}

int check_params(const closure_params *p, std::string *why)
{
    if (!p) { *why = "params is NULL"; return CLOSURE_EINVAL; }
    if (p->mode != CLOSURE_MODE_ROT && p->mode != CLOSURE_MODE_TRANS) { *why = "bad mode"; return CLOSURE_EINVAL; }
    if (p->n_p < 1 || p->n_p_star < 1 || p->n_p_star > p->n_p) { *why = "need 1 <= n_p_star <= n_p"; return CLOSURE_EINVAL; }
    if (p->n_t < 1 || p->n_t > kMaxNT) { *why = "need 1 <= n_t <= 64"; return CLOSURE_EINVAL; }
    if (p->n_p >= (1 << 23)) { *why = "n_p too large"; return CLOSURE_EINVAL; }
    const double v[6] = { p->omega0, p->v0, p->gamma, p->t_p, p->theta_p, 0.0 };
    if (!all_finite(v, 5)) { *why = "non-finite parameter"; return CLOSURE_EINVAL; }
    if (!(p->gamma > 0.0 && p->gamma <= 1.0)) { *why = "need 0 < gamma <= 1"; return CLOSURE_EINVAL; }
    if (p->omega0 < 0.0 || p->v0 < 0.0 || p->t_p < 0.0 || p->theta_p < 0.0) { *why = "negative scale"; return CLOSURE_EINVAL; }
    if (p->precision != 64 && p->precision != 32) { *why = "precision must be 64 or 32"; return CLOSURE_EINVAL; }
    if (p->n_p_star > kMaxKStar) { *why = "n_p_star > 20 is not built"; return CLOSURE_EUNSUPPORTED; }
    if (p->precision == 32 && (p->mode != CLOSURE_MODE_ROT || p->n_p > 256)) {
        *why = "fp32 mode exists for the rotation sampler with n_p <= 256 only"; return CLOSURE_EUNSUPPORTED;
    }
    return CLOSURE_OK;
}

// PURSE membership on the host, used only to validate S_0 (squared form, R-9).
bool host_in_purse(const closure_t *h, const double *pose)
{
    const double *R = pose, *t = pose + 9;
    for (int i = 0; i < h->n; ++i) {
        const double *m = h->meas.data() + (size_t)i * meas_cols(h->type);
        if (h->type == CLOSURE_REG_3D3D || h->type == CLOSURE_REG_3D3D_ELL) {
            double g[3], sq = 0.0;
            for (int r = 0; r < 3; ++r)
                g[r] = m[3 + r] - ((R[3 * r] * m[0] + R[3 * r + 1] * m[1] + R[3 * r + 2] * m[2]) + t[r]);
            if (h->type == CLOSURE_REG_3D3D) {
                for (int r = 0; r < 3; ++r) sq += g[r] * g[r];
            } else {                                       // g^T Lambda g (eq. (6))
                for (int r = 0; r < 3; ++r)
                    for (int c = 0; c < 3; ++c) sq += g[r] * m[6 + 3 * r + c] * g[c];
            }
            if (!(sq <= h->betas[i] * h->betas[i])) return false;
        } else if (h->type == CLOSURE_REPROJ_2D3D || h->type == CLOSURE_REPROJ_2D3D_ELL) {
            double p[3];
            for (int r = 0; r < 3; ++r) p[r] = (R[3 * r] * m[2] + R[3 * r + 1] * m[3] + R[3 * r + 2] * m[4]) + t[r];
            if (!(p[2] > 0.0)) return false;
            const double g0 = m[0] - (h->K[0] * (p[0] / p[2]) + h->K[2]);
            const double g1 = m[1] - (h->K[1] * (p[1] / p[2]) + h->K[3]);
            const double sq = h->type == CLOSURE_REPROJ_2D3D
                                  ? g0 * g0 + g1 * g1
                                  : g0 * (m[5] * g0 + m[6] * g1) + g1 * (m[7] * g0 + m[8] * g1);
            if (!(sq <= h->betas[i] * h->betas[i])) return false;
        } else {
            double sr = 0.0, st = 0.0;
            for (int e = 0; e < 9; ++e) sr += (R[e] - m[e]) * (R[e] - m[e]);
            for (int r = 0; r < 3; ++r) st += (t[r] - m[9 + r]) * (t[r] - m[9 + r]);
            if (h->type == CLOSURE_POSE_REG) {
                if (!(sr + st <= h->betas[i] * h->betas[i])) return false;
            } else {
                if (!(sr <= h->betas[2 * i] * h->betas[2 * i])) return false;
                if (!(st <= h->betas[2 * i + 1] * h->betas[2 * i + 1])) return false;
            }
        }
    }
    return true;
}

// closure_run's device buffers.  A destroyed handle parks them in a one-slot cache per device instead of
// freeing them (cudaFree of tens of MB costs up to ~100 ms now and then), so a create / run / destroy loop
// allocates once.
struct RunBuffers {
    double *samples = nullptr, *compact = nullptr;
    unsigned char *flags = nullptr;
    long long *count = nullptr;
    long long capacity = 0;
};
RunBuffers g_run_cache[kMaxDevices];

void cuda_free_run(RunBuffers &b)
{
    cudaFree(b.samples); cudaFree(b.compact); cudaFree(b.flags); cudaFree(b.count);
    b = RunBuffers();
}

void free_run_buffers(closure_t *h)
{
    RunBuffers mine;
    mine.samples = h->d_samples; mine.compact = h->d_compact; mine.flags = h->d_flags; mine.count = h->d_count;
    mine.capacity = h->run_capacity;
    h->d_samples = h->d_compact = nullptr; h->d_flags = nullptr; h->d_count = nullptr;
    h->run_capacity = 0;
    if (mine.capacity == 0) return;
    int dev = -1;
    std::lock_guard<std::mutex> lock(g_megb_mutex);
    if (cudaGetDevice(&dev) == cudaSuccess && dev >= 0 && dev < kMaxDevices && g_run_cache[dev].capacity < mine.capacity)
        std::swap(g_run_cache[dev], mine);
    if (mine.capacity) cuda_free_run(mine);
}

bool take_cached_run_buffers(closure_t *h, long long need)
{
    int dev = -1;
    std::lock_guard<std::mutex> lock(g_megb_mutex);
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= kMaxDevices || g_run_cache[dev].capacity < need) return false;
    RunBuffers &c = g_run_cache[dev];
    h->d_samples = c.samples; h->d_compact = c.compact; h->d_flags = c.flags; h->d_count = c.count;
    h->run_capacity = c.capacity;
    c = RunBuffers();
    return true;
}

int ensure_scratch(closure_t *h, long long n)
{
    const size_t need = compact_scratch_bytes(n);
    if (need <= h->scratch_bytes) return CLOSURE_OK;
    cudaFree(h->d_scratch);
    h->d_scratch = nullptr;
    h->scratch_bytes = 0;
    cudaError_t e = cudaMalloc(&h->d_scratch, need);
    if (e != cudaSuccess) return cuda_fail(h, e, "cudaMalloc(scratch)");
    h->scratch_bytes = need;
    return CLOSURE_OK;
}

// Device rows, sorted by the translation-side bound: [measurement, beta, beta^2, ...].  With a body pivot c
// (closure_set_pivot) the source points are stored as a - c (Z - c): the kernels then walk (R, tau = t + R c),
// for which "rotate about c" is the plain left multiplication (R-1).
void pack_rows(const closure_t *h, std::vector<double> &rows)
{
    const int type = h->type, n = h->n, row = row_doubles(type), cols = meas_cols(type);
    rows.assign((size_t)n * row, 0.0);
    const double *betas = h->betas.data();
    for (int k = 0; k < n; ++k) {
        const int i = h->order[k];
        const double *m = h->meas.data() + (size_t)i * cols;
        double *r = rows.data() + (size_t)k * row;
        if (type == CLOSURE_REG_3D3D) {
            std::memcpy(r, m, 6 * sizeof(double));
            for (int c = 0; c < 3; ++c) r[c] = m[c] - h->pivot[c];
            r[6] = betas[i]; r[7] = betas[i] * betas[i];
        } else if (type == CLOSURE_REPROJ_2D3D) {
            std::memcpy(r, m, 5 * sizeof(double));
            for (int c = 0; c < 3; ++c) r[2 + c] = m[2 + c] - h->pivot[c];
            r[5] = betas[i]; r[6] = betas[i] * betas[i];
        } else if (type == CLOSURE_REG_3D3D_ELL) {         // [a - c, b, beta, beta^2, L00 L01 L02 L11 L12 L22]
            std::memcpy(r, m, 6 * sizeof(double));
            for (int c = 0; c < 3; ++c) r[c] = m[c] - h->pivot[c];
            r[6] = betas[i]; r[7] = betas[i] * betas[i];
            r[8] = m[6]; r[9] = m[7]; r[10] = m[8]; r[11] = m[10]; r[12] = m[11]; r[13] = m[14];
        } else if (type == CLOSURE_REPROJ_2D3D_ELL) {      // [z, Z - c, beta, beta^2, L00 L01 L11]
            std::memcpy(r, m, 5 * sizeof(double));
            for (int c = 0; c < 3; ++c) r[2 + c] = m[2 + c] - h->pivot[c];
            r[5] = betas[i]; r[6] = betas[i] * betas[i];
            r[7] = m[5]; r[8] = m[6]; r[9] = m[8];
        } else if (type == CLOSURE_POSE_REG) {
            std::memcpy(r, m, 12 * sizeof(double));
            r[12] = betas[i]; r[13] = betas[i] * betas[i];
        } else {
            std::memcpy(r, m, 12 * sizeof(double));
            r[12] = betas[2 * i]; r[13] = betas[2 * i] * betas[2 * i];
            r[14] = betas[2 * i + 1]; r[15] = betas[2 * i + 1] * betas[2 * i + 1];
        }
    }
}

void fill_launch(const closure_t *h, WalkLaunch &L)
{
    std::memset(&L, 0, sizeof(L));
    L.n_p = h->P.n_p; L.n_p_star = h->P.n_p_star; L.n_t = h->P.n_t;
    L.omega0 = h->P.omega0; L.v0 = h->P.v0; L.gamma = h->P.gamma; L.t_p = h->P.t_p; L.theta_p = h->P.theta_p;
    L.pairs_cap = h->n_pairs;
    L.exact_only = (h->P.flags & 31) | (h->P.precision == 32 ? 32 : 0) | (h->P.flags & CLOSURE_FLAG_ONE_WARP ? 64 : 0);           // bit 0 documented; bits 1-2: debug switches of the screened kernel
}

bool same_params(const closure_params &a, const closure_params &b)
{
    return a.mode == b.mode && a.n_p == b.n_p && a.n_p_star == b.n_p_star && a.n_t == b.n_t && a.omega0 == b.omega0 &&
           a.v0 == b.v0 && a.gamma == b.gamma && a.t_p == b.t_p && a.theta_p == b.theta_p && a.precision == b.precision && a.flags == b.flags;
}

}  // namespace

extern "C" {

int closure_abi_version(void) { return CLOSURE_ABI_VERSION; }

const char *closure_strerror(int status)
{
    switch (status) {
    case CLOSURE_OK: return "ok";
    case CLOSURE_EINVAL: return "invalid argument";
    case CLOSURE_EINIT: return "initial pose outside the PURSE";
    case CLOSURE_ENOINIT: return "closure_set_init has not been called";
    case CLOSURE_ECUDA: return "CUDA failure";
    case CLOSURE_ENOMEM: return "out of memory";
    case CLOSURE_EUNSUPPORTED: return "combination not built";
    case CLOSURE_ETOOLARGE: return "n exceeds CLOSURE_COMPACT_STATIC_MAX (8,388,608 records), the size of the static scratch of closure_compact_static: use closure_compact";
    default: return "unknown status";
    }
}

const char *closure_last_error(const closure_t *h) { return h ? h->err.c_str() : "null handle"; }

int closure_default_params(int residual_type, closure_params *p)
{
    if (!p || meas_cols(residual_type) == 0) return CLOSURE_EINVAL;
    std::memset(p, 0, sizeof(*p));
    p->mode = CLOSURE_MODE_ROT;
    p->n_p = 150; p->n_p_star = 10; p->n_t = 15;
    p->gamma = 0.5;
    p->precision = 64;
    if (residual_type == CLOSURE_REPROJ_2D3D || residual_type == CLOSURE_REPROJ_2D3D_ELL) {   // PAPER.md:374 (t_p rescaled to metres at ~1 m depth)
        p->omega0 = 1.0; p->v0 = 2.0; p->theta_p = 0.2; p->t_p = 0.01;
    } else {
        p->omega0 = 0.5; p->v0 = 0.0; p->theta_p = 0.0; p->t_p = 0.1;
        if (residual_type != CLOSURE_REG_3D3D && residual_type != CLOSURE_REG_3D3D_ELL) p->n_t = 10;
    }
    return CLOSURE_OK;
}

int closure_set_params(closure_t *h, const closure_params *p)
{
    if (!h) return CLOSURE_EINVAL;
    std::string why;
    const int rc = check_params(p, &why);
    if (rc != CLOSURE_OK) return fail(h, rc, why);
    if (h->has_pivot && p->mode != CLOSURE_MODE_ROT)
        return fail(h, CLOSURE_EUNSUPPORTED, "a body pivot is set: Alg. A8 has no update_rotation (clear it with closure_set_pivot first)");
    if (plain_kernel_smem_bytes(h->h_desc.rows_bytes, p->n_t) > kMaxStageBytes)
        return fail(h, CLOSURE_EUNSUPPORTED, "constraint table and ladder do not fit shared memory for this n and n_t");
    if (p->precision == 32 && (h->type == CLOSURE_REG_3D3D_ELL || h->type == CLOSURE_REPROJ_2D3D_ELL))
        return fail(h, CLOSURE_EUNSUPPORTED, "fp32 mode does not exist for the ellipse / ellipsoid norms");
    h->P = *p;
    return CLOSURE_OK;
}

int closure_create(int residual_type, const double *measurements, int n, const double *betas,
                   const double *intrinsics, const closure_params *p, closure_t **out)
{
    if (!out) return CLOSURE_EINVAL;
    *out = nullptr;
    const int cols = meas_cols(residual_type);
    if (cols == 0 || !measurements || !betas || n <= 0 || n > 4096) return CLOSURE_EINVAL;
    std::string why;
    int rc = check_params(p, &why);
    if (rc != CLOSURE_OK) return rc;
    if (p->precision == 32 && (residual_type == CLOSURE_REG_3D3D_ELL || residual_type == CLOSURE_REPROJ_2D3D_ELL)) return CLOSURE_EUNSUPPORTED;
    // every instance must be stageable by the kernel of last resort (rows + per-thread ladder table)
    if (plain_kernel_smem_bytes(n * row_doubles(residual_type) * 8, p->n_t) > kMaxStageBytes) return CLOSURE_EUNSUPPORTED;
    const int nb = residual_type == CLOSURE_POSE_REG_SPLIT ? 2 * n : n;
    if (!all_finite(measurements, (size_t)n * cols) || !all_finite(betas, nb)) return CLOSURE_EINVAL;
    for (int i = 0; i < nb; ++i)
        if (!(betas[i] > 0.0)) return CLOSURE_EINVAL;
    if (residual_type == CLOSURE_REPROJ_2D3D || residual_type == CLOSURE_REPROJ_2D3D_ELL) {
        if (!intrinsics || !all_finite(intrinsics, 4) || !(intrinsics[0] > 0.0) || !(intrinsics[1] > 0.0))
            return CLOSURE_EINVAL;
    }
    if (residual_type == CLOSURE_REG_3D3D_ELL || residual_type == CLOSURE_REPROJ_2D3D_ELL) {
        // Lambda_i symmetric positive definite (eq. (6)): leading principal minors > 0
        for (int i = 0; i < n; ++i) {
            const double *m = measurements + (size_t)i * cols;
            if (residual_type == CLOSURE_REPROJ_2D3D_ELL) {
                const double *A = m + 5;
                if (A[1] != A[2] || !(A[0] > 0.0) || !(A[0] * A[3] - A[1] * A[2] > 0.0)) return CLOSURE_EINVAL;
            } else {
                const double *A = m + 6;
                if (A[1] != A[3] || A[2] != A[6] || A[5] != A[7]) return CLOSURE_EINVAL;
                const double d2 = A[0] * A[4] - A[1] * A[3];
                const double d3 = A[0] * (A[4] * A[8] - A[5] * A[7]) - A[1] * (A[3] * A[8] - A[5] * A[6]) +
                                  A[2] * (A[3] * A[7] - A[4] * A[6]);
                if (!(A[0] > 0.0) || !(d2 > 0.0) || !(d3 > 0.0)) return CLOSURE_EINVAL;
            }
        }
    }
    closure_t *h = new (std::nothrow) closure_s;
    if (!h) return CLOSURE_ENOMEM;
    h->type = residual_type;
    h->n = n;
    h->P = *p;
    h->meas.assign(measurements, measurements + (size_t)n * cols);
    h->betas.assign(betas, betas + nb);
    if (residual_type == CLOSURE_REPROJ_2D3D || residual_type == CLOSURE_REPROJ_2D3D_ELL) std::memcpy(h->K, intrinsics, sizeof(h->K));

    // pack rows, sorted by the translation-side bound (stable)
    auto key = [&](int i) { return residual_type == CLOSURE_POSE_REG_SPLIT ? betas[2 * i + 1] : betas[i]; };
    std::vector<int> order(n);
    std::iota(order.begin(), order.end(), 0);
    std::stable_sort(order.begin(), order.end(), [&](int a, int b) { return key(a) < key(b); });
    h->order = order;
    std::vector<double> rows;
    pack_rows(h, rows);
    for (int k = 0, len = 0; k < n; ++k) {                 // runs of equal bound in sorted order
        ++len;
        if (k == n - 1 || key(order[k + 1]) != key(order[k])) { h->n_pairs += (len + 1) / 2; len = 0; }
    }
    const size_t bytes = rows.size() * sizeof(double);     // row is 8 or 16 doubles: multiple of 16 B
    std::vector<int> perm(n);
    for (int k = 0; k < n; ++k) perm[order[k]] = k;
    cudaError_t e = cudaMalloc(&h->d_rows, bytes);
    if (e == cudaSuccess) e = cudaMemcpy(h->d_rows, rows.data(), bytes, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMalloc(&h->d_perm, sizeof(int) * (size_t)n);
    if (e == cudaSuccess) e = cudaMemcpy(h->d_perm, perm.data(), sizeof(int) * (size_t)n, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMalloc(&h->d_desc, sizeof(InstanceDesc));
    if (e == cudaSuccess) e = cudaMalloc(&h->d_stats, kNumStats * sizeof(unsigned long long));
    if (e != cudaSuccess) {
        // no handle is returned: the failure text can only be seen through the status code
        cudaFree(h->d_rows); cudaFree(h->d_perm); cudaFree(h->d_desc); cudaFree(h->d_stats);
        delete h;
        return CLOSURE_ECUDA;
    }
    h->h_desc.rows = h->d_rows;
    h->h_desc.perm = h->d_perm;
    h->h_desc.n = n;
    h->h_desc.rows_bytes = (int)bytes;
    std::memcpy(h->h_desc.K, h->K, sizeof(h->K));
    // the descriptor is complete for Step I now; closure_set_init adds S_0, R_bar, t_bar
    e = cudaMemcpy(h->d_desc, &h->h_desc, sizeof(InstanceDesc), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) {
        cudaFree(h->d_rows); cudaFree(h->d_perm); cudaFree(h->d_desc); cudaFree(h->d_stats);
        delete h;
        return CLOSURE_ECUDA;
    }
    *out = h;
    return CLOSURE_OK;
}

int closure_set_pivot(closure_t *h, const double *pivot)
{
    if (!h) return CLOSURE_EINVAL;
    if (!pivot || !all_finite(pivot, 3)) return fail(h, CLOSURE_EINVAL, "pivot is NULL or not finite");
    const bool nonzero = pivot[0] != 0.0 || pivot[1] != 0.0 || pivot[2] != 0.0;
    if (nonzero && (h->type == CLOSURE_POSE_REG || h->type == CLOSURE_POSE_REG_SPLIT))
        return fail(h, CLOSURE_EUNSUPPORTED, "a body pivot needs source points (Ex.1 / Ex.2)");
    if (nonzero && h->P.mode != CLOSURE_MODE_ROT)
        return fail(h, CLOSURE_EUNSUPPORTED, "Alg. A8 has no update_rotation: a body pivot applies to the rotation sampler only");
    std::memcpy(h->pivot, pivot, sizeof(h->pivot));
    h->has_pivot = nonzero;
    h->has_init = false;                                 // S_0 is stored relative to the pivot: give it again
    std::vector<double> rows;
    pack_rows(h, rows);
    cudaError_t e = cudaMemcpy(h->d_rows, rows.data(), rows.size() * sizeof(double), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return cuda_fail(h, e, "upload of constraint rows");
    return CLOSURE_OK;
}

int closure_set_init(closure_t *h, const double *poses, int n0, double *mean_out)
{
    if (!h) return CLOSURE_EINVAL;
    if (!poses || n0 <= 0) return fail(h, CLOSURE_EINVAL, "poses is NULL or n0 <= 0");
    if (!all_finite(poses, (size_t)n0 * 12)) return fail(h, CLOSURE_EINVAL, "non-finite initial pose");
    for (int s = 0; s < n0; ++s)
        if (!host_in_purse(h, poses + (size_t)s * 12))
            return fail(h, CLOSURE_EINIT, "initial pose " + std::to_string(s) + " violates a constraint");
    // Alg. 2 l.3-4: R_bar = proj_SO(3)(sum R_j), t_bar = mean t_j
    double M[9] = { 0 }, tb[3] = { 0 };
    for (int s = 0; s < n0; ++s) {
        for (int e = 0; e < 9; ++e) M[e] += poses[(size_t)s * 12 + e];
        for (int r = 0; r < 3; ++r) tb[r] += poses[(size_t)s * 12 + 9 + r];
    }
    for (int r = 0; r < 3; ++r) tb[r] /= (double)n0;
    double Rb[9];
    if (!project_so3(M, Rb)) return fail(h, CLOSURE_EINVAL, "sum of initial rotations has no projection onto SO(3)");
    cudaFree(h->d_S0);
    h->d_S0 = nullptr;
    h->has_init = false;
    cudaError_t e = cudaMalloc(&h->d_S0, (size_t)n0 * 12 * sizeof(double));
    if (e == cudaSuccess) {
        if (h->has_pivot) {                              // the kernels walk (R, tau = t + R c)
            std::vector<double> tau(poses, poses + (size_t)n0 * 12);
            for (int s = 0; s < n0; ++s) {
                double *q = tau.data() + (size_t)s * 12;
                for (int r = 0; r < 3; ++r)
                    q[9 + r] = q[9 + r] + (q[3 * r] * h->pivot[0] + q[3 * r + 1] * h->pivot[1] + q[3 * r + 2] * h->pivot[2]);
            }
            e = cudaMemcpy(h->d_S0, tau.data(), (size_t)n0 * 12 * sizeof(double), cudaMemcpyHostToDevice);
        } else {
            e = cudaMemcpy(h->d_S0, poses, (size_t)n0 * 12 * sizeof(double), cudaMemcpyHostToDevice);
        }
    }
    if (e != cudaSuccess) return cuda_fail(h, e, "upload of S_0");
    h->h_desc.S0 = h->d_S0;
    h->h_desc.n0 = n0;
    std::memcpy(h->h_desc.Rbar, Rb, sizeof(Rb));
    std::memcpy(h->h_desc.tbar, tb, sizeof(tb));
    if (h->P.flags & CLOSURE_FLAG_PCA_VELOCITY) {
        pca_velocity_scale(poses, n0, h->h_desc.vscale);
    } else {
        for (int e = 0; e < 9; ++e) h->h_desc.vscale[e] = (e % 4 == 0) ? 1.0 : 0.0;
    }
    e = cudaMemcpy(h->d_desc, &h->h_desc, sizeof(InstanceDesc), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return cuda_fail(h, e, "upload of instance descriptor");
    h->has_init = true;
    if (mean_out) {
        std::memcpy(mean_out, Rb, sizeof(Rb));
        std::memcpy(mean_out + 9, tb, sizeof(tb));
    }
    return CLOSURE_OK;
}

int closure_init_sample(closure_t *h, long long trial_begin, long long num_trials, unsigned long long seed,
                        double *out_poses, unsigned char *out_ok, void *cuda_stream)
{
    if (!h) return CLOSURE_EINVAL;
    if (trial_begin < 0 || num_trials < 0) return fail(h, CLOSURE_EINVAL, "negative size");
    if ((h->type == CLOSURE_REG_3D3D || h->type == CLOSURE_REG_3D3D_ELL || h->type == CLOSURE_REPROJ_2D3D ||
         h->type == CLOSURE_REPROJ_2D3D_ELL) && h->n < 3) return fail(h, CLOSURE_EINVAL, "RANSAG needs at least 3 correspondences");
    if (num_trials == 0) return CLOSURE_OK;
    if (!out_poses || !out_ok) return fail(h, CLOSURE_EINVAL, "output buffer is NULL");
    if (reinterpret_cast<uintptr_t>(out_poses) & 15u) return fail(h, CLOSURE_EINVAL, "pose buffer must be 16-byte aligned");
    cudaError_t e = launch_step1(h->type, h->d_desc, h->h_desc.rows_bytes, trial_begin, num_trials, seed, out_poses,
                                 out_ok, static_cast<cudaStream_t>(cuda_stream));
    if (e == cudaSuccess && h->has_pivot) e = launch_pivot_back(out_poses, num_trials, h->pivot, static_cast<cudaStream_t>(cuda_stream));
    if (e != cudaSuccess) return cuda_fail(h, e, "Step I kernel launch");
    return CLOSURE_OK;
}

int closure_init_from_trials(closure_t *h, long long num_trials, unsigned long long seed, int max_poses, int *n0_out,
                             void *cuda_stream)
{
    if (!h) return CLOSURE_EINVAL;
    if (num_trials <= 0 || max_poses <= 0) return fail(h, CLOSURE_EINVAL, "need num_trials > 0 and max_poses > 0");
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    double *d_poses = nullptr, *d_kept = nullptr;
    unsigned char *d_ok = nullptr;
    long long *d_cnt = nullptr;
    cudaError_t e = cudaMalloc(&d_poses, (size_t)num_trials * 96);
    if (e == cudaSuccess) e = cudaMalloc(&d_kept, (size_t)num_trials * 96);
    if (e == cudaSuccess) e = cudaMalloc(&d_ok, (size_t)num_trials);
    if (e == cudaSuccess) e = cudaMalloc(&d_cnt, sizeof(long long));
    int rc = e == cudaSuccess ? CLOSURE_OK : cuda_fail(h, e, "cudaMalloc(Step I buffers)");
    if (rc == CLOSURE_OK) rc = closure_init_sample(h, 0, num_trials, seed, d_poses, d_ok, cuda_stream);
    if (rc == CLOSURE_OK) rc = closure_compact(h, d_poses, d_ok, num_trials, d_kept, d_cnt, cuda_stream);   // trial order kept
    long long cnt = 0;
    std::vector<double> host;
    if (rc == CLOSURE_OK) {
        e = cudaMemcpyAsync(&cnt, d_cnt, sizeof(cnt), cudaMemcpyDeviceToHost, stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(stream);
        if (e == cudaSuccess && cnt > 0) {
            const long long take = std::min<long long>(cnt, max_poses);
            host.resize((size_t)take * 12);
            e = cudaMemcpy(host.data(), d_kept, host.size() * sizeof(double), cudaMemcpyDeviceToHost);
        }
        if (e != cudaSuccess) rc = cuda_fail(h, e, "Step I trials");
    }
    cudaFree(d_poses); cudaFree(d_kept); cudaFree(d_ok); cudaFree(d_cnt);
    if (rc != CLOSURE_OK) return rc;
    if (n0_out) *n0_out = (int)(host.size() / 12);
    if (host.empty()) return fail(h, CLOSURE_EINIT, "no Step I trial produced a pose inside the PURSE");
    return closure_set_init(h, host.data(), (int)(host.size() / 12), nullptr);
}

int closure_sample_range(closure_t *h, long long walker_begin, long long num_walkers, int num_steps,
                         unsigned long long seed, double *out_samples, unsigned char *out_on_boundary,
                         int *out_trace, void *cuda_stream)
{
    if (!h) return CLOSURE_EINVAL;
    if (!h->has_init) return fail(h, CLOSURE_ENOINIT, "closure_set_init has not been called");
    if (walker_begin < 0 || num_walkers < 0 || num_steps < 0) return fail(h, CLOSURE_EINVAL, "negative size");
    if (num_walkers == 0) return CLOSURE_OK;
    if (!out_samples || !out_on_boundary) return fail(h, CLOSURE_EINVAL, "output buffer is NULL");
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    WalkLaunch L;
    fill_launch(h, L);
    L.desc[0] = h->d_desc;
    L.seed[0] = seed;
    L.walker_begin = walker_begin;
    L.num_walkers = num_walkers;
    L.num_steps = num_steps;
    L.out_samples = out_samples;
    L.out_flags = out_on_boundary;
    L.out_trace = out_trace;
    if (h->stats_on) {
        cudaError_t e = cudaMemsetAsync(h->d_stats, 0, kNumStats * sizeof(unsigned long long), stream);
        if (e != cudaSuccess) return cuda_fail(h, e, "cudaMemsetAsync(stats)");
        L.stats = h->d_stats;
    }
    std::string why;
    cudaError_t e = launch_walkers(h->type, h->P.mode, h->stats_on, L, 1, h->h_desc.rows_bytes, stream, &why);
    if (e == cudaSuccess && h->has_pivot) e = launch_pivot_back(out_samples, num_walkers, h->pivot, stream);   // t = tau - R c
    h->last_stream = stream;
    if (e != cudaSuccess) return cuda_fail(h, e, why.empty() ? "walker kernel launch" : why.c_str());
    return CLOSURE_OK;
}

int closure_sample(closure_t *h, long long num_walkers, int num_steps, unsigned long long seed,
                   double *out_samples, unsigned char *out_on_boundary, void *cuda_stream)
{
    return closure_sample_range(h, 0, num_walkers, num_steps, seed, out_samples, out_on_boundary, nullptr,
                                cuda_stream);
}

int closure_sample_batch(closure_t *const *handles, int n_instances, long long walkers_per_instance,
                         int num_steps, const unsigned long long *seeds, double *out_samples,
                         unsigned char *out_on_boundary, void *cuda_stream)
{
    if (!handles || n_instances <= 0 || !handles[0]) return CLOSURE_EINVAL;
    closure_t *h0 = handles[0];
    if (!seeds || walkers_per_instance < 0 || num_steps < 0) return fail(h0, CLOSURE_EINVAL, "bad batch arguments");
    for (int b = 0; b < n_instances; ++b) {
        if (!handles[b]) return fail(h0, CLOSURE_EINVAL, "NULL handle in batch");
        if (!handles[b]->has_init) return fail(h0, CLOSURE_ENOINIT, "batch member without S_0");
        if (handles[b]->type != h0->type || !same_params(handles[b]->P, h0->P))
            return fail(h0, CLOSURE_EINVAL, "batch members must share residual type and parameters");
    }
    if (walkers_per_instance == 0) return CLOSURE_OK;
    if (!out_samples || !out_on_boundary) return fail(h0, CLOSURE_EINVAL, "output buffer is NULL");
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    if (h0->stats_on) {
        cudaError_t e = cudaMemsetAsync(h0->d_stats, 0, kNumStats * sizeof(unsigned long long), stream);
        if (e != cudaSuccess) return cuda_fail(h0, e, "cudaMemsetAsync(stats)");
    }
    for (int b0 = 0; b0 < n_instances; b0 += kMaxBatch) {
        const int nb = std::min(kMaxBatch, n_instances - b0);
        WalkLaunch L;
        fill_launch(h0, L);
        int max_bytes = 0;
        for (int b = 0; b < nb; ++b) {
            L.desc[b] = handles[b0 + b]->d_desc;
            L.seed[b] = seeds[b0 + b];
            max_bytes = std::max(max_bytes, handles[b0 + b]->h_desc.rows_bytes);
            L.pairs_cap = std::max(L.pairs_cap, handles[b0 + b]->n_pairs);
        }
        L.walker_begin = 0;
        L.num_walkers = walkers_per_instance;
        L.num_steps = num_steps;
        L.out_samples = out_samples + (size_t)b0 * walkers_per_instance * 12;
        L.out_flags = out_on_boundary + (size_t)b0 * walkers_per_instance;
        L.out_trace = nullptr;
        L.stats = h0->stats_on ? h0->d_stats : nullptr;
        std::string why;
        cudaError_t e = launch_walkers(h0->type, h0->P.mode, h0->stats_on, L, nb, max_bytes, stream, &why);
        for (int b = 0; b < nb && e == cudaSuccess; ++b)
            if (handles[b0 + b]->has_pivot)
                e = launch_pivot_back(L.out_samples + (size_t)b * walkers_per_instance * 12, walkers_per_instance,
                                      handles[b0 + b]->pivot, stream);
        if (e != cudaSuccess) return cuda_fail(h0, e, why.empty() ? "walker kernel launch" : why.c_str());
    }
    h0->last_stream = stream;
    return CLOSURE_OK;
}

int closure_compact(closure_t *h, const double *samples, const unsigned char *flags, long long n,
                    double *out_compacted, long long *out_count, void *cuda_stream)
{
    if (!h) return CLOSURE_EINVAL;
    if (n < 0 || !out_count || (n > 0 && (!samples || !flags || !out_compacted)))
        return fail(h, CLOSURE_EINVAL, "bad compaction arguments");
    if ((reinterpret_cast<uintptr_t>(samples) | reinterpret_cast<uintptr_t>(out_compacted)) & 15u)
        return fail(h, CLOSURE_EINVAL, "sample buffers must be 16-byte aligned");
    int rc = ensure_scratch(h, std::max<long long>(n, 1));
    if (rc != CLOSURE_OK) return rc;
    cudaError_t e = launch_compact(samples, flags, n, out_compacted, out_count, h->d_scratch,
                                   static_cast<cudaStream_t>(cuda_stream));
    if (e != cudaSuccess) return cuda_fail(h, e, "compaction kernel launch");
    return CLOSURE_OK;
}

int closure_compact_static(const double *samples, const unsigned char *flags, long long n, double *out_compacted,
                           long long *out_count, void *cuda_stream)
{
    if (n < 0 || !out_count || (n > 0 && (!samples || !flags || !out_compacted))) return CLOSURE_EINVAL;
    if (n > CLOSURE_COMPACT_STATIC_MAX) return CLOSURE_ETOOLARGE;
    if ((reinterpret_cast<uintptr_t>(samples) | reinterpret_cast<uintptr_t>(out_compacted)) & 15u) return CLOSURE_EINVAL;
    const cudaError_t e = launch_compact_static(samples, flags, n, out_compacted, out_count, static_cast<cudaStream_t>(cuda_stream));
    return e == cudaSuccess ? CLOSURE_OK : CLOSURE_ECUDA;
}

int closure_megb(closure_t *h, const double *samples, long long count, closure_megb_result *out,
                 void *cuda_stream)
{
    if (!h) return CLOSURE_EINVAL;
    if (!out || !samples || count <= 0) return fail(h, CLOSURE_EINVAL, "closure_megb needs count > 0 samples");
    if (!h->has_init) return fail(h, CLOSURE_ENOINIT, "R_bar (closure_set_init) is needed to align quaternion signs");
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    double qbar[4];
    rotation_to_quat(h->h_desc.Rbar, qbar);
    Ball bt, bq;
    double d2h_bytes = 0.0, max_pivot_s = 0.0, prepare_s = 0.0;
    int pivots = 0;
    const auto t0 = std::chrono::steady_clock::now();
    if (count >= kDeviceMegbMin && !(h->P.flags & CLOSURE_FLAG_HOST_MEGB)) {
        // the cloud stays on the device: one embedding pass, then one max-reduction per miniball pivot
        // (its buffers are shared by all handles of the process on this device and grow on demand)
        std::lock_guard<std::mutex> lock(g_megb_mutex);
        int dev = 0;
        cudaError_t e = cudaGetDevice(&dev);
        if (e == cudaSuccess && (dev < 0 || dev >= kMaxDevices)) e = cudaErrorInvalidDevice;
        if (e == cudaSuccess && !g_megb[dev]) g_megb[dev] = device_megb_create(&e);
        if (e == cudaSuccess) e = device_megb_prepare(g_megb[dev], samples, count, qbar, stream);
        if (e != cudaSuccess) return cuda_fail(h, e, "device MEGB set-up");
        prepare_s = std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
        DeviceMegb *dm = g_megb[dev];
        const bool ok = miniball_source(device_megb_trans(dm), count, 3, &bt) &&
                        miniball_source(device_megb_quats(dm), count, 4, &bq);
        if (device_megb_status(dm) != cudaSuccess) return cuda_fail(h, device_megb_status(dm), "device MEGB pivot");
        if (!ok) return fail(h, CLOSURE_EINVAL, "miniball failed");
        device_megb_accounting(dm, &d2h_bytes, &max_pivot_s, &pivots);
    } else {
        std::vector<double> host;
        try {
            host.resize((size_t)count * 12);
        } catch (const std::bad_alloc &) {
            return fail(h, CLOSURE_ENOMEM, "host buffer for samples");
        }
        cudaError_t e = cudaMemcpyAsync(host.data(), samples, host.size() * sizeof(double), cudaMemcpyDeviceToHost, stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(stream);
        if (e != cudaSuccess) return cuda_fail(h, e, "copy of samples to the host");
        d2h_bytes = (double)(host.size() * sizeof(double));
        std::vector<double> tp((size_t)count * 3), qp((size_t)count * 4);
        for (long long i = 0; i < count; ++i) {
            const double *s = host.data() + (size_t)i * 12;
            std::memcpy(tp.data() + (size_t)i * 3, s + 9, 3 * sizeof(double));
            double q[4];
            rotation_to_quat(s, q);
            const double dot = q[0] * qbar[0] + q[1] * qbar[1] + q[2] * qbar[2] + q[3] * qbar[3];
            const double sg = dot < 0.0 ? -1.0 : 1.0;                   // R-15
            for (int k = 0; k < 4; ++k) qp[(size_t)i * 4 + k] = sg * q[k];
        }
        if (!miniball(tp.data(), count, 3, &bt) || !miniball(qp.data(), count, 4, &bq))
            return fail(h, CLOSURE_EINVAL, "miniball failed");
    }
    std::memset(out, 0, sizeof(*out));
    const double hn = std::sqrt(bq.center[0] * bq.center[0] + bq.center[1] * bq.center[1] +
                                bq.center[2] * bq.center[2] + bq.center[3] * bq.center[3]);
    if (!(hn > 0.0)) return fail(h, CLOSURE_EINVAL, "rotation samples span the whole quaternion sphere");
    const double qc[4] = { bq.center[0] / hn, bq.center[1] / hn, bq.center[2] / hn, bq.center[3] / hn };
    quat_to_rotation(qc, out->R);
    std::memcpy(out->t, bt.center, 3 * sizeof(double));
    double ca = (1.0 + hn * hn - bq.sq_radius) / (2.0 * hn);       // R-16
    ca = std::min(1.0, std::max(-1.0, ca));
    out->rot_radius = 2.0 * std::acos(ca);
    out->trans_radius = std::sqrt(bt.sq_radius);
    out->n_rot_support = bq.n_support;
    out->n_trans_support = bt.n_support;
    for (int k = 0; k < bq.n_support; ++k) out->rot_support[k] = bq.support[k];
    for (int k = 0; k < bt.n_support; ++k) out->trans_support[k] = bt.support[k];
    out->host_seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
    out->d2h_bytes = d2h_bytes;
    out->max_pivot_seconds = max_pivot_s;
    out->pivots = pivots;
    out->prepare_seconds = prepare_s;
    return CLOSURE_OK;
}

int closure_run(closure_t *h, long long num_walkers, int num_steps, unsigned long long seed,
                closure_megb_result *out, long long *out_count, void *cuda_stream)
{
    if (!h) return CLOSURE_EINVAL;
    if (!out || num_walkers <= 0) return fail(h, CLOSURE_EINVAL, "closure_run needs walkers and a result");
    cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
    if (num_walkers > h->run_capacity) {
        free_run_buffers(h);
        if (!take_cached_run_buffers(h, num_walkers)) {
            cudaError_t e = cudaMalloc(&h->d_samples, (size_t)num_walkers * 96);
            if (e == cudaSuccess) e = cudaMalloc(&h->d_compact, (size_t)num_walkers * 96);
            if (e == cudaSuccess) e = cudaMalloc(&h->d_flags, (size_t)num_walkers);
            if (e == cudaSuccess) e = cudaMalloc(&h->d_count, sizeof(long long));
            h->run_capacity = num_walkers;
            if (e != cudaSuccess) {
                RunBuffers b;
                b.samples = h->d_samples; b.compact = h->d_compact; b.flags = h->d_flags; b.count = h->d_count;
                cuda_free_run(b);
                h->d_samples = h->d_compact = nullptr; h->d_flags = nullptr; h->d_count = nullptr;
                h->run_capacity = 0;
                return cuda_fail(h, e, "cudaMalloc(run buffers)");
            }
        }
    }
    int rc = closure_sample(h, num_walkers, num_steps, seed, h->d_samples, h->d_flags, cuda_stream);
    if (rc != CLOSURE_OK) return rc;
    rc = closure_compact(h, h->d_samples, h->d_flags, num_walkers, h->d_compact, h->d_count, cuda_stream);
    if (rc != CLOSURE_OK) return rc;
    long long count = 0;
    cudaError_t e = cudaMemcpyAsync(&count, h->d_count, sizeof(count), cudaMemcpyDeviceToHost, stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(stream);
    if (e != cudaSuccess) return cuda_fail(h, e, "walk / compaction");
    if (out_count) *out_count = count;
    if (count == 0) {
        // no walker was stopped by the boundary: every final pose is still a valid subset of S (Prop. 4)
        return closure_megb(h, h->d_samples, num_walkers, out, cuda_stream);
    }
    return closure_megb(h, h->d_compact, count, out, cuda_stream);
}

int closure_enable_stats(closure_t *h, int on)
{
    if (!h) return CLOSURE_EINVAL;
    h->stats_on = on != 0;
    return CLOSURE_OK;
}

int closure_get_stats(closure_t *h, closure_stats *out)
{
    if (!h || !out) return CLOSURE_EINVAL;
    unsigned long long v[kNumStats];
    cudaError_t e = cudaStreamSynchronize(h->last_stream);
    if (e == cudaSuccess) e = cudaMemcpy(v, h->d_stats, sizeof(v), cudaMemcpyDeviceToHost);
    if (e != cudaSuccess) return cuda_fail(h, e, "read of statistics");
    out->perturb_pairs = v[0]; out->ladder_pairs = v[1]; out->perturb_setups = v[2];
    out->ladder_setups = v[3]; out->accepted_steps = v[4]; out->walker_steps = v[5];
    out->perturb_pairs_f32 = v[6]; out->ladder_pairs_f32 = v[7]; out->fallback_steps = v[8];
    out->verified_rungs = v[9]; out->setup_cycles = v[10]; out->total_cycles = v[11];
    out->threshold_probes = v[12]; out->survivors = v[13]; out->reserved_ = v[14]; out->threshold_failures = v[15];
    return CLOSURE_OK;
}

int closure_alu_peak(int precision, double *flops_per_s, double *seconds, void *cuda_stream)
{
    if (!flops_per_s || !seconds || (precision != 64 && precision != 32 && precision != 4)) return CLOSURE_EINVAL;
    cudaError_t e = measure_alu_peak(precision, flops_per_s, seconds, static_cast<cudaStream_t>(cuda_stream));
    return e == cudaSuccess ? CLOSURE_OK : CLOSURE_ECUDA;
}

int closure_miniball_host(const double *points, long long n, int d, double *center, double *radius,
                          long long *support, int *n_support)
{
    if (!points || !center || !radius || !support || !n_support || n <= 0 || d < 1 || d > 4) return CLOSURE_EINVAL;
    Ball b;
    if (!miniball(points, n, d, &b)) return CLOSURE_EINVAL;
    for (int a = 0; a < d; ++a) center[a] = b.center[a];
    *radius = std::sqrt(b.sq_radius);
    *n_support = b.n_support;
    for (int k = 0; k < b.n_support; ++k) support[k] = b.support[k];
    return CLOSURE_OK;
}

void closure_destroy(closure_t *h)
{
    if (!h) return;
    cudaFree(h->d_rows); cudaFree(h->d_perm); cudaFree(h->d_desc); cudaFree(h->d_S0); cudaFree(h->d_scratch);
    cudaFree(h->d_stats);
    free_run_buffers(h);
    delete h;
}

}  // extern "C"
