// Step III with the sample cloud kept on the device.
//
// Gaertner's miniball touches the whole cloud only in its pivot step, "find the point farthest from
// the current centre": an HBM-bound max-reduction.  closure_megb therefore leaves the compacted
// samples where the walker kernel wrote them:
//   megb_embed_kernel     one pass: unit quaternion of every rotation, sign aligned to q(R_bar)
//                         (R-15), and the translation, as two dense fp64 arrays (32 + 24 B per sample);
//   megb_farthest_kernel  per pivot: squared distance of every point to the centre, block maxima,
//                         the last block reduces them -> (index, distance), 16 bytes back to the host.
// The host keeps the <= 5-point support basis (miniball.cpp) and fetches single points by index.
// Squared distances use the same unfused left-to-right arithmetic as the host scan, and ties go to
// the lowest index, so both paths pivot on the same points.
#include <cuda_runtime.h>
#include <math_constants.h>

#include <algorithm>
#include <array>
#include <chrono>
#include <unordered_map>
#include <vector>

#include "closure_internal.h"

namespace closure {
namespace {

constexpr int kFarThreads = 256;

__device__ __forceinline__ void rotation_to_quat_dev(const double *R, double (&q)[4])
{
    const double sq[4] = { 1.0 + R[0] + R[4] + R[8], 1.0 + R[0] - R[4] - R[8], 1.0 - R[0] + R[4] - R[8],
                           1.0 - R[0] - R[4] + R[8] };
    int big = 0;
#pragma unroll
    for (int k = 1; k < 4; ++k)
        if (sq[k] > sq[big]) big = k;
    const double sb = big == 0 ? sq[0] : (big == 1 ? sq[1] : (big == 2 ? sq[2] : sq[3]));
    const double g = 0.5 * sqrt(sb);
    const double h = 0.25 / g;
    switch (big) {
    case 0: q[0] = g; q[1] = (R[7] - R[5]) * h; q[2] = (R[2] - R[6]) * h; q[3] = (R[3] - R[1]) * h; break;
    case 1: q[1] = g; q[0] = (R[7] - R[5]) * h; q[2] = (R[1] + R[3]) * h; q[3] = (R[2] + R[6]) * h; break;
    case 2: q[2] = g; q[0] = (R[2] - R[6]) * h; q[1] = (R[1] + R[3]) * h; q[3] = (R[5] + R[7]) * h; break;
    default: q[3] = g; q[0] = (R[3] - R[1]) * h; q[1] = (R[2] + R[6]) * h; q[2] = (R[5] + R[7]) * h; break;
    }
    const double nq = sqrt(__dadd_rn(__dadd_rn(__dadd_rn(__dmul_rn(q[0], q[0]), __dmul_rn(q[1], q[1])),
                                               __dmul_rn(q[2], q[2])), __dmul_rn(q[3], q[3])));
#pragma unroll
    for (int k = 0; k < 4; ++k) q[k] /= nq;
}

__global__ void __launch_bounds__(256) megb_embed_kernel(const double *__restrict__ samples, long long n, double qb0,
                                                         double qb1, double qb2, double qb3, double *__restrict__ Q,
                                                         double *__restrict__ T)
{
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const double2 *s2 = reinterpret_cast<const double2 *>(samples + 12 * i);
        double s[12];
#pragma unroll
        for (int e = 0; e < 6; ++e) { const double2 v = s2[e]; s[2 * e] = v.x; s[2 * e + 1] = v.y; }
        double q[4];
        rotation_to_quat_dev(s, q);
        const double dot = __dadd_rn(__dadd_rn(__dadd_rn(__dmul_rn(q[0], qb0), __dmul_rn(q[1], qb1)), __dmul_rn(q[2], qb2)),
                                     __dmul_rn(q[3], qb3));
        const double sg = dot < 0.0 ? -1.0 : 1.0;                   // R-15
        reinterpret_cast<double2 *>(Q + 4 * i)[0] = make_double2(sg * q[0], sg * q[1]);
        reinterpret_cast<double2 *>(Q + 4 * i)[1] = make_double2(sg * q[2], sg * q[3]);
        T[3 * i] = s[9]; T[3 * i + 1] = s[10]; T[3 * i + 2] = s[11];
    }
}

struct FarResult {
    double d2;
    long long idx;
};

__device__ __forceinline__ void far_merge(double &d2, long long &idx, double od2, long long oidx)
{
    if (od2 > d2 || (od2 == d2 && oidx < idx)) { d2 = od2; idx = oidx; }
}

// Point of P (n x D) farthest from c; ties to the lowest index.  partial: one FarResult per block;
// ticket: zero before the launch, zero again after it.
template <int D>
__global__ void __launch_bounds__(kFarThreads) megb_farthest_kernel(const double *__restrict__ P, long long n, double c0,
                                                                     double c1, double c2, double c3, FarResult *partial,
                                                                     unsigned int *ticket, FarResult *out)
{
    __shared__ double sd[kFarThreads / 32];
    __shared__ long long si[kFarThreads / 32];
    __shared__ bool last;
    double best = -1.0;
    long long bi = 0x7fffffffffffffffLL;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const double *p = P + D * i;
        const double e0 = p[0] - c0, e1 = p[1] - c1, e2 = p[2] - c2;
        double s = __dadd_rn(__dadd_rn(__dmul_rn(e0, e0), __dmul_rn(e1, e1)), __dmul_rn(e2, e2));
        if (D == 4) { const double e3 = p[3] - c3; s = __dadd_rn(s, __dmul_rn(e3, e3)); }
        if (s > best) { best = s; bi = i; }              // i ascends within a thread: first maximum kept
    }
    auto block_reduce = [&]() {
#pragma unroll
        for (int o = 16; o >= 1; o >>= 1)
            far_merge(best, bi, __shfl_xor_sync(0xffffffffu, best, o), __shfl_xor_sync(0xffffffffu, bi, o));
        if ((threadIdx.x & 31) == 0) { sd[threadIdx.x >> 5] = best; si[threadIdx.x >> 5] = bi; }
        __syncthreads();
        if (threadIdx.x < 32) {
            best = threadIdx.x < kFarThreads / 32 ? sd[threadIdx.x] : -1.0;
            bi = threadIdx.x < kFarThreads / 32 ? si[threadIdx.x] : 0x7fffffffffffffffLL;
#pragma unroll
            for (int o = 16; o >= 1; o >>= 1)
                far_merge(best, bi, __shfl_xor_sync(0xffffffffu, best, o), __shfl_xor_sync(0xffffffffu, bi, o));
        }
    };
    block_reduce();
    if (threadIdx.x == 0) {
        partial[blockIdx.x].d2 = best;
        partial[blockIdx.x].idx = bi;
        __threadfence();
        last = atomicAdd(ticket, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!last) return;
    __threadfence();
    best = -1.0;
    bi = 0x7fffffffffffffffLL;
    for (int b = threadIdx.x; b < (int)gridDim.x; b += blockDim.x) far_merge(best, bi, partial[b].d2, partial[b].idx);
    __syncthreads();
    block_reduce();
    if (threadIdx.x == 0) {
        out->d2 = best;
        out->idx = bi;
        *ticket = 0u;
    }
}

}  // namespace

struct DeviceMegb {
    cudaStream_t stream = nullptr;
    long long n = 0;
    double *Q = nullptr, *T = nullptr;
    FarResult *partial = nullptr, *out = nullptr;
    unsigned int *ticket = nullptr;
    FarResult *h_out = nullptr;          // pinned
    double *h_pt = nullptr;              // pinned, 4 doubles
    int blocks = 0, sms = 148;
    long long capacity = 0;
    cudaError_t err = cudaSuccess;
    // accounting of one closure_megb call (closure_megb_result.d2h_bytes / pivots / max_pivot_seconds)
    double d2h_bytes = 0.0, max_pivot_s = 0.0;
    int pivots = 0;

    class Cloud : public PointSource {
    public:
        Cloud(DeviceMegb *m, int d) : m_(m), d_(d) {}
        bool farthest(const double *c, long long *index, double *sq_dist) override
        {
            if (m_->err != cudaSuccess) return false;
            const auto t0 = std::chrono::steady_clock::now();
            const double c3 = d_ == 4 ? c[3] : 0.0;
            if (d_ == 4)
                megb_farthest_kernel<4><<<m_->blocks, kFarThreads, 0, m_->stream>>>(m_->Q, m_->n, c[0], c[1], c[2], c3,
                                                                                     m_->partial, m_->ticket, m_->out);
            else
                megb_farthest_kernel<3><<<m_->blocks, kFarThreads, 0, m_->stream>>>(m_->T, m_->n, c[0], c[1], c[2], c3,
                                                                                     m_->partial, m_->ticket, m_->out);
            cudaError_t e = cudaGetLastError();
            if (e == cudaSuccess) e = cudaMemcpyAsync(m_->h_out, m_->out, sizeof(FarResult), cudaMemcpyDeviceToHost, m_->stream);
            if (e == cudaSuccess) e = cudaStreamSynchronize(m_->stream);
            if (e != cudaSuccess) { m_->err = e; return false; }
            m_->d2h_bytes += (double)sizeof(FarResult);
            m_->pivots += 1;
            m_->max_pivot_s = std::max(m_->max_pivot_s, std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count());
            *index = m_->h_out->idx;
            *sq_dist = m_->h_out->d2;
            return true;
        }
        const double *point(long long i) override
        {
            auto it = cache_.find(i);
            if (it != cache_.end()) return it->second.data();
            if (m_->err != cudaSuccess || i < 0 || i >= m_->n) return nullptr;
            const double *src = d_ == 4 ? m_->Q + 4 * i : m_->T + 3 * i;
            cudaError_t e = cudaMemcpyAsync(m_->h_pt, src, sizeof(double) * d_, cudaMemcpyDeviceToHost, m_->stream);
            if (e == cudaSuccess) e = cudaStreamSynchronize(m_->stream);
            if (e != cudaSuccess) { m_->err = e; return nullptr; }
            m_->d2h_bytes += (double)(sizeof(double) * d_);
            std::array<double, 4> v = { 0, 0, 0, 0 };
            for (int a = 0; a < d_; ++a) v[a] = m_->h_pt[a];
            return cache_.emplace(i, v).first->second.data();
        }

        void clear() { cache_.clear(); }

    private:
        DeviceMegb *m_;
        int d_;
        std::unordered_map<long long, std::array<double, 4>> cache_;
    };
    Cloud quats{ this, 4 };
    Cloud trans{ this, 3 };
};

// Buffers live in the handle and grow on demand (no allocation on the closure_megb path once warm).
DeviceMegb *device_megb_create(cudaError_t *err)
{
    DeviceMegb *m = new DeviceMegb;
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&m->sms, cudaDevAttrMultiProcessorCount, dev);
    cudaError_t e = cudaMalloc(&m->partial, sizeof(FarResult) * (size_t)m->sms * 8);
    if (e == cudaSuccess) e = cudaMalloc(&m->out, sizeof(FarResult));
    if (e == cudaSuccess) e = cudaMalloc(&m->ticket, sizeof(unsigned int));
    if (e == cudaSuccess) e = cudaMemset(m->ticket, 0, sizeof(unsigned int));
    if (e == cudaSuccess) e = cudaMallocHost(&m->h_out, sizeof(FarResult));
    if (e == cudaSuccess) e = cudaMallocHost(&m->h_pt, sizeof(double) * 4);
    m->err = e;
    if (err) *err = e;
    return m;
}

cudaError_t device_megb_prepare(DeviceMegb *m, const double *d_samples, long long count, const double qbar[4],
                                cudaStream_t stream)
{
    m->stream = stream;
    m->n = count;
    m->quats.clear();
    m->trans.clear();
    m->d2h_bytes = 0.0; m->max_pivot_s = 0.0; m->pivots = 0;
    cudaError_t e = (m->partial && m->out && m->ticket && m->h_out && m->h_pt) ? cudaSuccess : cudaErrorMemoryAllocation;
    if (e == cudaSuccess) e = cudaMemsetAsync(m->ticket, 0, sizeof(unsigned int), stream);
    if (e == cudaSuccess && count > m->capacity) {
        cudaFree(m->Q); cudaFree(m->T);
        m->Q = m->T = nullptr;
        m->capacity = 0;
        e = cudaMalloc(&m->Q, sizeof(double) * 4 * (size_t)count);
        if (e == cudaSuccess) e = cudaMalloc(&m->T, sizeof(double) * 3 * (size_t)count);
        if (e == cudaSuccess) m->capacity = count;
    }
    const long long want = (count + kFarThreads - 1) / kFarThreads;
    const long long cap = (long long)m->sms * 8;          // grid: a multiple of the SM count when the cloud is large
    m->blocks = (int)(want < cap ? (want > 0 ? want : 1) : cap);
    if (e == cudaSuccess) {
        megb_embed_kernel<<<m->blocks, 256, 0, stream>>>(d_samples, count, qbar[0], qbar[1], qbar[2], qbar[3], m->Q, m->T);
        e = cudaGetLastError();
    }
    m->err = e;
    return e;
}

PointSource *device_megb_quats(DeviceMegb *m) { return &m->quats; }
PointSource *device_megb_trans(DeviceMegb *m) { return &m->trans; }
cudaError_t device_megb_status(DeviceMegb *m) { return m->err; }
void device_megb_accounting(DeviceMegb *m, double *d2h_bytes, double *max_pivot_seconds, int *pivots)
{
    *d2h_bytes = m->d2h_bytes; *max_pivot_seconds = m->max_pivot_s; *pivots = m->pivots;
}

void device_megb_destroy(DeviceMegb *m)
{
    if (!m) return;
    cudaFree(m->Q); cudaFree(m->T); cudaFree(m->partial); cudaFree(m->out); cudaFree(m->ticket);
    cudaFreeHost(m->h_out); cudaFreeHost(m->h_pt);
    delete m;
}

}  // namespace closure
