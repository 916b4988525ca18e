// Compaction kernel (north_star (2)): stable stream compaction of the
// 96-byte sample records whose on_boundary flag is set, in walker order.
//
// HBM-bound: algorithmic traffic = 1 B (flag) + 96 B read + 96 B written per kept walker.
// One pass ("decoupled look-back" chained scan): a CTA takes a tile of kTile records by ticket,
// counts its flags with byte-wise popcounts, publishes its aggregate, sums its predecessors'
// published aggregates / inclusive prefixes, then copies its kept records with 16-byte vector
// loads and stores.  Kept records of a tile are contiguous in the output and consecutive threads
// move consecutive 16-byte chunks, so both sides are coalesced without staging the payload.
#include <cuda_runtime.h>
#include <stdint.h>

#include <mutex>

#include "closure_internal.h"

namespace closure {
namespace {

constexpr int kCThreads = 256;
constexpr int kPerThread = 8;                       // flags per thread = one 8-byte load
constexpr int kTile = kCThreads * kPerThread;       // 2048 records = 192 KiB of payload per CTA
constexpr int kChunksPerRec = 6;                    // 96 B = 6 x 16 B

constexpr unsigned long long kStatusShift = 62;
constexpr unsigned long long kAggregate = 1ull << kStatusShift;
constexpr unsigned long long kPrefix = 2ull << kStatusShift;
constexpr unsigned long long kValueMask = (1ull << kStatusShift) - 1;

__device__ __forceinline__ unsigned long long ld_state(const unsigned long long *p)
{
    return *reinterpret_cast<const volatile unsigned long long *>(p);
}
__device__ __forceinline__ void st_state(unsigned long long *p, unsigned long long v)
{
    *reinterpret_cast<volatile unsigned long long *>(p) = v;
}

// scratch layout: [0] ticket counter, [1 .. 1+tiles) tile states; zeroed before each launch.
__global__ void __launch_bounds__(kCThreads) compact_kernel(const uint4 *__restrict__ samples,
                                                           const unsigned char *__restrict__ flags, long long n,
                                                           uint4 *__restrict__ out, long long *__restrict__ out_count,
                                                           unsigned long long *scratch, int num_tiles)
{
    __shared__ short offs[kTile];
    __shared__ int warp_tot[kCThreads / 32];
    __shared__ int s_tile;
    __shared__ long long s_excl;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    if (tid == 0) s_tile = (int)atomicAdd(scratch, 1ull);     // ticket: predecessors are already running
    __syncthreads();
    const int tile = s_tile;
    unsigned long long *state = scratch + 1;
    const long long base = (long long)tile * kTile;

    // ---- flags -> per-thread count
    const long long f0 = base + (long long)tid * kPerThread;
    unsigned long long bits = 0;                    // byte k = flag k (0/1 after normalisation)
    if (f0 + kPerThread <= n && ((reinterpret_cast<uintptr_t>(flags + f0) & 7u) == 0)) {
        bits = *reinterpret_cast<const unsigned long long *>(flags + f0);
    } else {
        for (int k = 0; k < kPerThread; ++k)
            if (f0 + k < n) bits |= (unsigned long long)flags[f0 + k] << (8 * k);
    }
    // normalise every non-zero byte to 0x01
    unsigned long long nz = bits | (bits >> 4);
    nz |= nz >> 2;
    nz |= nz >> 1;
    nz &= 0x0101010101010101ull;
    const int cnt = __popcll(nz);

    // ---- block exclusive scan of cnt
    int incl = cnt;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        const int v = __shfl_up_sync(0xffffffffu, incl, d);
        if (lane >= d) incl += v;
    }
    if (lane == 31) warp_tot[warp] = incl;
    __syncthreads();
    int warp_base = 0, tile_total = 0;
#pragma unroll
    for (int q = 0; q < kCThreads / 32; ++q) {
        const int v = warp_tot[q];
        if (q < warp) warp_base += v;
        tile_total += v;
    }
    int run = warp_base + incl - cnt;               // exclusive offset of this thread's first record
#pragma unroll
    for (int k = 0; k < kPerThread; ++k) {
        const bool keep = (nz >> (8 * k)) & 1ull;
        offs[tid * kPerThread + k] = keep ? (short)run : (short)-1;
        run += keep ? 1 : 0;
    }

    // ---- decoupled look-back (warp 0)
    if (warp == 0) {
        long long excl = 0;
        if (tile == 0) {
            if (lane == 0) st_state(state, kPrefix | (unsigned long long)tile_total);
        } else {
            if (lane == 0) st_state(state + tile, kAggregate | (unsigned long long)tile_total);
            int look = tile - 1;
            while (true) {
                const int idx = look - lane;
                unsigned long long v = kPrefix;      // virtual predecessors before tile 0: prefix 0
                if (idx >= 0) {
                    do { v = ld_state(state + idx); } while ((v >> kStatusShift) == 0ull);
                }
                const unsigned pm = __ballot_sync(0xffffffffu, (v >> kStatusShift) == 2ull);
                const int first = pm ? (__ffs(pm) - 1) : 32;
                long long val = (lane <= first) ? (long long)(v & kValueMask) : 0ll;
#pragma unroll
                for (int d = 16; d >= 1; d >>= 1) val += __shfl_xor_sync(0xffffffffu, val, d);
                excl += val;
                if (pm) break;
                look -= 32;
            }
            if (lane == 0) st_state(state + tile, kPrefix | (unsigned long long)(excl + tile_total));
        }
        if (lane == 0) {
            s_excl = excl;
            if (tile == num_tiles - 1) *out_count = excl + tile_total;
        }
    }
    __syncthreads();
    const long long excl = s_excl;

    // ---- copy kept records, 16 bytes per thread per iteration
    const long long rec_left = n - base;
    const int recs = rec_left < kTile ? (int)rec_left : kTile;
    const int chunks = recs * kChunksPerRec;
    const uint4 *src = samples + base * kChunksPerRec;
    uint4 *dst = out + excl * kChunksPerRec;
    if (tile_total == recs) {
        // every record of the tile is kept (the usual case: a walker that has run for a while has been stopped by the
        // boundary): a straight copy, eight independent 16-byte loads in flight per thread, no offset look-ups
        int c = tid;
        for (; c + 7 * kCThreads < chunks; c += 8 * kCThreads) {
            uint4 v[8];
#pragma unroll
            for (int k = 0; k < 8; ++k) v[k] = __ldcs(src + c + k * kCThreads);
#pragma unroll
            for (int k = 0; k < 8; ++k) __stcs(dst + c + k * kCThreads, v[k]);
        }
        for (; c < chunks; c += kCThreads) __stcs(dst + c, __ldcs(src + c));
        return;
    }
#pragma unroll 4
    for (int c = tid; c < chunks; c += kCThreads) {
        const int rec = c / kChunksPerRec;
        const int part = c - rec * kChunksPerRec;
        const int o = offs[rec];
        if (o >= 0) dst[o * kChunksPerRec + part] = __ldcs(src + c);
    }
}

}  // namespace

size_t compact_scratch_bytes(long long n)
{
    const long long tiles = (n + kTile - 1) / kTile;
    return (size_t)(tiles + 1) * sizeof(unsigned long long);
}

// t <- t - R c on n poses [R row-major (9), t (3)]: the walk with a body pivot c (closure_set_pivot, R-1)
// runs on (R, tau = t + R c); this turns its output back into the caller's translation.  One pose per thread.
__global__ void pivot_back_kernel(double *__restrict__ poses, long long n, double c0, double c1, double c2)
{
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double *q = poses + 12 * i;
#pragma unroll
    for (int r = 0; r < 3; ++r)
        q[9 + r] = q[9 + r] - (q[3 * r] * c0 + q[3 * r + 1] * c1 + q[3 * r + 2] * c2);
}

cudaError_t launch_pivot_back(double *poses, long long n, const double *pivot, cudaStream_t stream)
{
    if (n <= 0) return cudaSuccess;
    const long long blocks = (n + 255) / 256;
    if (blocks > 0x7fffffffLL) return cudaErrorInvalidValue;
    pivot_back_kernel<<<(unsigned)blocks, 256, 0, stream>>>(poses, n, pivot[0], pivot[1], pivot[2]);
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------- no-allocation variant
// closure_compact_static (include/closure.h): the same kernel, with its scratch (ticket counter + one look-back state
// per tile of 2,048 records) in a file-scope device array instead of a cudaMalloc'ed per-handle buffer, for callers that
// cannot allocate (CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).  Every GPU that loads
// the library holds these 32 KB + 8 B until exit.  All calls on a device share the array: it keeps the last call's
// contents (cleared at the start of every call, on the caller's stream), and two calls that overlap on the GPU race.
namespace {

constexpr long long kStaticMaxTiles = CLOSURE_COMPACT_STATIC_MAX / kTile;       // 8,388,608 records = 4,096 tiles
static_assert(kStaticMaxTiles * kTile == CLOSURE_COMPACT_STATIC_MAX, "the static maximum is a whole number of tiles");
static __device__ __align__(256) unsigned long long g_compact_static_scratch[kStaticMaxTiles + 1];

// In HOST code the array's name is a host-side stand-in, not a device address: the address the kernel needs comes from
// cudaGetSymbolAddress, resolved once per device with that device current and cached here.
constexpr int kStaticMaxDevices = 64;
std::mutex g_static_mutex;
unsigned long long *g_static_ptr[kStaticMaxDevices] = { nullptr };

cudaError_t static_scratch_of_current_device(unsigned long long **ptr)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kStaticMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (g_static_ptr[dev] == nullptr) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_compact_static_scratch);
        if (e != cudaSuccess) return e;
        g_static_ptr[dev] = static_cast<unsigned long long *>(p);
    }
    *ptr = g_static_ptr[dev];
    return cudaSuccess;
}

}  // namespace

cudaError_t launch_compact_static(const double *samples, const unsigned char *flags, long long n, double *out,
                                  long long *out_count, cudaStream_t stream)
{
    if (n <= 0) return cudaMemsetAsync(out_count, 0, sizeof(long long), stream);
    if (n > CLOSURE_COMPACT_STATIC_MAX) return cudaErrorInvalidValue;             // (the C entry point reports it first)
    const long long tiles = (n + kTile - 1) / kTile;
    unsigned long long *scratch = nullptr;
    cudaError_t e = static_scratch_of_current_device(&scratch);
    if (e != cudaSuccess) return e;
    // the ticket and the tile states of this call must start at zero: the array still holds the previous call's
    e = cudaMemsetAsync(scratch, 0, (size_t)(tiles + 1) * sizeof(unsigned long long), stream);
    if (e != cudaSuccess) return e;
    compact_kernel<<<(unsigned)tiles, kCThreads, 0, stream>>>(reinterpret_cast<const uint4 *>(samples), flags, n,
                                                             reinterpret_cast<uint4 *>(out), out_count, scratch, (int)tiles);
    return cudaGetLastError();
}

cudaError_t launch_compact(const double *samples, const unsigned char *flags, long long n, double *out,
                           long long *out_count, void *scratch, cudaStream_t stream)
{
    if (n <= 0) return cudaMemsetAsync(out_count, 0, sizeof(long long), stream);
    const long long tiles = (n + kTile - 1) / kTile;
    if (tiles > 0x7fffffffLL) return cudaErrorInvalidValue;
    cudaError_t e = cudaMemsetAsync(scratch, 0, compact_scratch_bytes(n), stream);
    if (e != cudaSuccess) return e;
    compact_kernel<<<(unsigned)tiles, kCThreads, 0, stream>>>(reinterpret_cast<const uint4 *>(samples), flags, n,
                                                             reinterpret_cast<uint4 *>(out), out_count,
                                                             reinterpret_cast<unsigned long long *>(scratch),
                                                             (int)tiles);
    return cudaGetLastError();
}

}  // namespace closure
