// Helpers shared by the warp-cooperative walker kernels (walker_coop_kernel.cu for the residuals that
// are quadratic in the translation perturbation, walker_coop_reproj_kernel.cu for the reprojection
// residual): order-preserving keys, warp reductions, packed fp32 pairs, batched Philox, and step a4 --
// the top-N_P* selection on fp32 values with a certificate, and its fp64 fall-back.
#pragma once
#include <cuda_runtime.h>
#include <math_constants.h>
#include <stdint.h>

#include "closure_internal.h"
#include "walker_common.cuh"

namespace closure {
namespace {

constexpr int kCoopWarps = 4;                 // walkers per CTA
constexpr int kCoopThreads = 32 * kCoopWarps;
constexpr unsigned FULL = 0xffffffffu;
constexpr float kMu19 = 1.9073486328125e-06f;   // 2^-19

struct CoopSmem {
    size_t run_end, run_bf, run_pend, pos, af, warp0, per_warp, rowsA, rowsL, pert, ab, qrow, RmS, dex, qL, cand4, candj, candd, pose, stc, rm32, ridx, total;
};

// Shared-memory layout; f4 = float4 words per fp32 constraint row (1: affine residuals, 2: reprojection);
// pairs = 32-byte entries of rowsA (affine: pair-entries, runs padded to even length; otherwise n)
// af_f4 > 0 (dense kernel, Ex.2: 1, Ex.3: 3): a CTA-level fp32 image of the constraints (af_f4 float4 per row) and per warp the
// fp32 rung rotations (rm32) and the indices of each rung's screening rows (ridx), for the fp32 search of the set-up
__host__ __device__ inline CoopSmem coop_layout(int rows_bytes, int n, int n_t, int nq, int f4, int pairs, int warps = kCoopWarps,
                                                int af_f4 = 0, int af_extra_bytes = 0)
{
    CoopSmem s;
    size_t o = 16 + (size_t)((rows_bytes + 15) & ~15);
    s.run_end = o; o += (size_t)((n * 4 + 15) & ~15);
    s.run_bf = o;  o += (size_t)((n * 4 + 15) & ~15);
    s.run_pend = o; o += (size_t)((n * 4 + 15) & ~15);
    s.pos = o;     o += (size_t)((n * 4 + 15) & ~15);
    s.af = o;      o += (size_t)n * 16 * af_f4 + (size_t)((af_extra_bytes + 15) & ~15);
    s.warp0 = o;
    size_t w = 0;
    s.rowsA = w; w += (size_t)pairs * 32;          // affine: pair-transposed, runs padded to even length
    s.rowsL = w; w += (size_t)n * 16 * f4;
    s.pert = w;  w += (size_t)nq * 32 * 16;
    s.ab = w;    w += (size_t)n_t * 16;
    s.qrow = w;  w += (size_t)n_t * 32 * f4;
    s.RmS = w;   w += (size_t)((n_t * 72 + 15) & ~15);
    s.dex = w;   w += (size_t)nq * 32 * 8;
    s.qL = w;    w += (size_t)((n_t * 4 + 15) & ~15);
    s.cand4 = w; w += 32 * 16;
    s.candj = w; w += 32 * 4;
    s.candd = w; w += 32 * 4;
    s.pose = w;  w += 18 * 8;
    s.stc = w;   w += 16 * 8;
    s.rm32 = w;  w += af_f4 > 0 ? (size_t)n_t * 48 : 0;
    s.ridx = w;  w += af_f4 > 0 ? (size_t)((n_t * 8 + 15) & ~15) : 0;
    s.per_warp = w;
    s.total = o + (size_t)warps * w;
    return s;
}

// ---------------------------------------------------------------------------------- small helpers
// order-preserving maps to unsigned keys
__device__ __forceinline__ uint32_t fkey(float x)
{
    const uint32_t b = __float_as_uint(x);
    return b ^ ((uint32_t)((int32_t)b >> 31) | 0x80000000u);
}
// MUFU.RSQ alone: rsqrtf() adds a rescaling path for subnormal arguments; callers pass a >= 1e-30 (normal), for
// which both return the same bits
__device__ __forceinline__ float rsqrt_normal(float a)
{
    float r;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(a));
    return r;
}
__device__ __forceinline__ float fkey_inv(uint32_t k)
{
    return __uint_as_float((k & 0x80000000u) ? (k ^ 0x80000000u) : ~k);
}
__device__ __forceinline__ unsigned long long dkey(double x)
{
    const unsigned long long b = (unsigned long long)__double_as_longlong(x);
    return b ^ ((unsigned long long)((long long)b >> 63) | 0x8000000000000000ull);
}
__device__ __forceinline__ float wmax_nonneg(float v)      // v >= 0 (or NaN, which wins: callers then fall back)
{
    return __uint_as_float(__reduce_max_sync(FULL, __float_as_uint(v)));
}
__device__ __forceinline__ double wmin_f64(double v)
{
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) v = dmin(v, __shfl_xor_sync(FULL, v, o));
    return v;
}

// The two largest of the (distinct) keys and the maximum of a non-negative float over the aligned group of G = 8 or 16 lanes
// this lane belongs to (gm = the group's lanes), by XOR butterflies.  REDUX with a different member mask per group is
// serialised group by group (measured: ~30 instructions per reduction in the set-up of the short tables).
__device__ __forceinline__ void group_top2_max(unsigned gm, int G, uint32_t key, float f, uint32_t &k1, uint32_t &k2, float &fm)
{
    uint32_t b1 = key, b2 = 0u, fb = __float_as_uint(f);
#pragma unroll
    for (int o = 1; o < 16; o <<= 1) {
        if (o < G) {
            const uint32_t p1 = __shfl_xor_sync(gm, b1, o), p2 = __shfl_xor_sync(gm, b2, o), pf = __shfl_xor_sync(gm, fb, o);
            const uint32_t lo = min(b1, p1);
            b1 = max(b1, p1);
            b2 = max(max(b2, p2), lo);
            fb = max(fb, pf);
        }
    }
    k1 = b1; k2 = b2; fm = __uint_as_float(fb);
}

// Maximum over the lanes ek + c KP, c < NCH (the constraint chunks of one ladder candidate in the full evaluation of a rung),
// delivered to the lane with c = 0: a tree of SHFL.DOWN on order-preserving keys (NaN stays the largest, as under REDUX.MAX).
// Lanes beyond NCH KP pass -inf.  A REDUX with one member mask per candidate is serialised mask by mask.
__device__ __forceinline__ float chunk_max_to_first(float M, int KP, int NCH)
{
    uint32_t k = fkey(M);
    for (int off = 1; off < NCH; off <<= 1) k = max(k, __shfl_down_sync(FULL, k, off * KP));
    return fkey_inv(k);
}

// x / d by one IMAD.HI (a division by a run-time integer is ~20 instructions): magic = ceil(2^32 / d); exact while x d < 2^32
// (floor(x magic / 2^32) = floor(x / d + x e / 2^32) with 0 <= e < 1, and frac(x / d) <= 1 - 1/d).  d = 1 wraps magic to 0.
struct FastDiv {
    uint32_t magic;
    int d;
    __device__ __forceinline__ explicit FastDiv(int dd) : magic(0xFFFFFFFFu / (uint32_t)dd + 1u), d(dd) {}
    __device__ __forceinline__ int div(int x) const { return d == 1 ? x : (int)__umulhi((uint32_t)x, magic); }
};

// packed fp32 pairs (FFMA2 on sm_100a)
__device__ __forceinline__ unsigned long long pk2(float lo, float hi)
{
    unsigned long long r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void upk2(unsigned long long v, float &lo, float &hi)
{
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ unsigned long long fma2(unsigned long long a, unsigned long long b, unsigned long long c)
{
    unsigned long long r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}

__device__ __forceinline__ unsigned long long mul2(unsigned long long a, unsigned long long b)
{
    unsigned long long r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}

// Philox4x32-10 for NJ counters that differ only in word 2 (= perturbation index): NJ independent
// dependency chains, rounds unrolled (a rolled loop costs two register moves per chain and round).
template <int NJ>
__device__ __forceinline__ void philox_batch(const Rng &rng, uint32_t s, const int (&j)[NJ], uint32_t (&x)[NJ],
                                             uint32_t (&y)[NJ], uint32_t (&z)[NJ])
{
    uint32_t c0[NJ], c1[NJ], c2[NJ], c3[NJ];
#pragma unroll
    for (int q = 0; q < NJ; ++q) { c0[q] = rng.w_lo; c1[q] = s; c2[q] = (uint32_t)j[q]; c3[q] = 1u | rng.w_hi8; }
    uint32_t k0 = rng.k0, k1 = rng.k1;
#pragma unroll
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


// ---------------------------------------------------------------------------------- a4: top-N_P*
// fp32 part.  v[q] = d~ of perturbation j = lane + 32 q (-inf for an empty slot), each within `unc`
// of the fp64 value d_j.  The N_P* + 1 largest are extracted by rounds of REDUX.MAX over the lanes'
// locally sorted keys (the 3 low key bits carry q: values move by < 2^-20 relative, covered below).
// The ranking is certified iff consecutive extracted values differ by more than 2 unc: then the exact
// ranking is the same, strictly, so no tie-break is involved.  On success lane r < N_P* writes
// candj[r] (index) and candd[r] (an upper bound of the fp64 value).  myval: lane r holds the r-th value.
template <int NQ>
__device__ __forceinline__ bool topk_certified(const float (&v)[NQ], int n_ps, float unc, bool force_fail, bool trust, int lane,
                                               int *candj, float *candd, float &myval)
{
    uint32_t key[NQ];
#pragma unroll
    for (int q = 0; q < NQ; ++q) key[q] = (fkey(v[q]) & ~7u) | (uint32_t)q;
    // local sort, descending (odd-even transposition network)
#pragma unroll
    for (int pass = 0; pass < NQ; ++pass)
#pragma unroll
        for (int a = (pass & 1); a + 1 < NQ; a += 2) {
            const uint32_t hi = max(key[a], key[a + 1]), lo = min(key[a], key[a + 1]);
            key[a] = hi; key[a + 1] = lo;
        }
    uint32_t myg = fkey(-CUDART_INF_F);
    unsigned mywho = 1u;
    for (int r = 0; r <= n_ps; ++r) {               // extract the N_P* + 1 largest
        // every lane whose head equals the maximum pops it: the next reduction waits for one compare only.
        // Two lanes popping together (equal keys) is a tie: detected below, never certified, and the values
        // reported from then on are not larger than the true ones, which keeps the fall-back's threshold valid.
        const uint32_t g = __reduce_max_sync(FULL, key[0]);
        const bool pop = key[0] == g;
        const unsigned who = __ballot_sync(FULL, pop);
        if (lane == r) { myg = g; mywho = who; }
        if (pop) {
#pragma unroll
            for (int q = 0; q + 1 < NQ; ++q) key[q] = key[q + 1];
            key[NQ - 1] = 0u;
        }
    }
    // an empty slot carries the key of -inf with its slot index in the low bits: decode it as -inf, not as the NaN those bits spell
    myval = ((myg & ~7u) == (fkey(-CUDART_INF_F) & ~7u)) ? -CUDART_INF_F : fkey_inv(myg);
    const int myj = (__ffs(mywho) - 1) + 32 * (int)(myg & 7u);
    const bool tie = (lane <= n_ps) && ((mywho & (mywho - 1u)) != 0u) && (myval > -CUDART_INF_F);   // empty slots all look alike
    const float prev = __shfl_up_sync(FULL, myval, 1);
    bool ok = true;
    if (lane < n_ps) ok = (myval > -CUDART_INF_F) && (myval < CUDART_INF_F);
    if (lane >= 1 && lane <= n_ps) {
        const bool none_left = (lane == n_ps) && (myval == -CUDART_INF_F);
        const float need = fmaf(2.0f, unc, kMu19 * (fabsf(prev) + fabsf(myval)));
        ok = ok && (none_left || (prev - myval > need));
    }
    if (tie) ok = false;
    if (trust) ok = true;                       // fp32 mode: the fp32 ranking is taken as it is
    if (force_fail) ok = false;
    const bool certified = __all_sync(FULL, ok);
    if (certified && lane < n_ps) {
        candj[lane] = myj;
        candd[lane] = myval + fmaf(1.01f, unc, kMu19 * fabsf(myval));    // >= the fp64 value d_j
    }
    return certified;
}

// fp64 fall-back (near-ties): exact(j) is the plain kernel's eq. (14) value of perturbation j; the
// N_P* best by (d descending, j ascending) (R-8) go to candj[].  Only perturbations with
// d~_j >= T = (N_P*-th largest d~) - 2 unc can be among the exact top-N_P* (any other has N_P*
// exact values strictly above it); if they fit one per lane only those are evaluated, otherwise
// (or with all = true) every perturbation is.  Returns the number of fp64 evaluations per lane-slot.
template <int NQ, class Exact>
__device__ __forceinline__ int topk_fp64(const float (&v)[NQ], int n_p, int n_ps, float unc, float myval, bool all,
                                         int lane, double *dex, int *candj, float *candd, Exact exact)
{
    const float Tn = __shfl_sync(FULL, myval, n_ps - 1);
    const float T = Tn - fmaf(2.02f, unc, 2.0f * kMu19 * fabsf(Tn));
    int cnt = 33;
    int *fbj = reinterpret_cast<int *>(dex);
    if ((T > -CUDART_INF_F) && (T < CUDART_INF_F) && !all) {
        cnt = 0;
#pragma unroll
        for (int q = 0; q < NQ; ++q) {
            const bool in = (lane + 32 * q < n_p) && (v[q] >= T);
            const unsigned b = __ballot_sync(FULL, in);
            if (in && cnt <= 32) {
                const int pos = cnt + __popc(b & ((1u << lane) - 1u));
                if (pos < 32) fbj[pos] = lane + 32 * q;
            }
            cnt += __popc(b);
        }
        __syncwarp();
    }
    if (cnt <= 32) {
        const int j = lane < cnt ? fbj[lane] : -1;
        const double d = exact(j);
        unsigned long long key = (lane < cnt) ? dkey(d) : 0ull;
#pragma unroll 1
        for (int r = 0; r < n_ps; ++r) {
            const uint32_t ghi = __reduce_max_sync(FULL, (uint32_t)(key >> 32));
            const uint32_t glo = __reduce_max_sync(FULL, ((uint32_t)(key >> 32) == ghi) ? (uint32_t)key : 0u);
            const unsigned long long g = ((unsigned long long)ghi << 32) | glo;
            const int jm = (key == g && key != 0ull) ? j : 0x7fffffff;
            const int jwin = __reduce_min_sync(FULL, jm);
            if (jm == jwin) key = 0ull;
            if (lane == 0) { candj[r] = jwin; candd[r] = CUDART_INF_F; }
        }
        return cnt;
    }
    // every perturbation in fp64; written for few registers: one at a time, values in shared memory
    __syncwarp();
#pragma unroll 1
    for (int q = 0; q < NQ; ++q) {
        const int j = lane + 32 * q;
        const double d = exact(j);
        dex[32 * q + lane] = (j < n_p) ? d : -CUDART_INF;
    }
    unsigned taken = 0u;                             // slots of this lane already extracted
#pragma unroll 1
    for (int r = 0; r < n_ps; ++r) {
        unsigned long long best = 0ull;
        int bq = 0;
#pragma unroll 1
        for (int q = 0; q < NQ; ++q) {
            const unsigned long long kq = ((taken >> q) & 1u) || (lane + 32 * q >= n_p) ? 0ull : dkey(dex[32 * q + lane]);
            if (kq > best) { best = kq; bq = q; }
        }
        const uint32_t ghi = __reduce_max_sync(FULL, (uint32_t)(best >> 32));
        const uint32_t glo = __reduce_max_sync(FULL, ((uint32_t)(best >> 32) == ghi) ? (uint32_t)best : 0u);
        const unsigned long long g = ((unsigned long long)ghi << 32) | glo;
        const int jm = (best == g && best != 0ull) ? lane + 32 * bq : 0x7fffffff;
        const int jwin = __reduce_min_sync(FULL, jm);
        if (jm == jwin) taken |= 1u << bq;
        if (lane == 0) { candj[r] = jwin; candd[r] = CUDART_INF_F; }
    }
    return n_p;
}

}  // namespace
}  // namespace closure
