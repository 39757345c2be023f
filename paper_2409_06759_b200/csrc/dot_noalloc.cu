// dot_noalloc.cu -- tcb_dot_noalloc: the inner product D = alpha * sum_i conj?(X[i]) * Y[i] for callers that cannot allocate
// (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).
//
// tcb_dot keeps its per-block partial sums in a stream-ordered allocation made for the call (cudaMallocAsync /
// cudaFreeAsync).  This variant keeps them in ONE file-scope device array, g_scratch below:
//   * 256 bytes of header (an arrival counter) + kNoAllocMaxBlocks = 8192 partial sums of 16 bytes = 131 328 bytes, held by
//     every GPU that loads the library, from the load until the process exits;
//   * a block reduces one TILE of consecutive elements; the tile is the smallest power of two >= 2048 elements for which
//     ceil(n / tile) <= 8192, at most 65 536 (256 threads x 256 elements), so the largest n is
//         kNoAllocMaxElems = 8192 x 65536 = 536 870 912 elements (8.6 GB per operand);
//     a larger n is refused by the entry point (TCB_EUNSUPPORTED), never truncated;
//   * the grid depends on n alone (not on the SM count), partial sums are added in block order by whichever block arrives
//     last: the result is bit-reproducible from call to call and from GPU model to GPU model.  It differs from tcb_dot's
//     (whose grid is 4 blocks per SM with a grid-stride loop) by summation order only.
//   * ONE launch (tcb_dot: two) and one 4-byte cudaMemsetAsync; no cudaMalloc, cudaMallocAsync, cudaFree or any library
//     routine that allocates.
//
// The array is shared by every call on the device and keeps the last call's contents.  What must start at zero -- the
// arrival counter -- is cleared on the call's stream in front of the launch (and left at zero by the last block); the
// partial sums need no clearing: blocks 0 .. nblocks-1 overwrite theirs before the last block reads exactly those.
// Two tcb_dot_noalloc calls that overlap on the GPU (different streams / lanes / contexts of one device, or two host
// threads) RACE on the array: issue them on one stream, or order them with events.
//
// g_scratch in HOST code is a host-side stand-in for the symbol, not a device address; the address a kernel can use comes
// from cudaGetSymbolAddress, asked once per device with that device current (dot_noalloc_scratch below).
#include "kernels.h"

#include <algorithm>
#include <mutex>

namespace tcb {

namespace {

constexpr int kHeaderBytes = 256;                       // arrival counter; keeps the partial sums 256-byte aligned
constexpr int kMinTileLog2 = 11, kMaxTileLog2 = 16;     // 2048 ... 65536 elements per block
constexpr size_t kScratchBytes = kHeaderBytes + (size_t)kNoAllocMaxBlocks * sizeof(double2);

static __device__ __align__(256) unsigned char g_scratch[kScratchBytes];

static_assert(kNoAllocMaxElems == (int64_t)kNoAllocMaxBlocks << kMaxTileLog2, "kernels.h states the limit");

template <bool CONJ>
__global__ void __launch_bounds__(256)
dot_noalloc_kernel(const double2 *__restrict__ X, const double2 *__restrict__ Y, long long n, int tile_log2,
                   unsigned char *scratch, double2 *D, double ar, double ai)
{
    unsigned int *counter = reinterpret_cast<unsigned int *>(scratch);
    double2 *partial = reinterpret_cast<double2 *>(scratch + kHeaderBytes);
    const long long t0 = (long long)blockIdx.x << tile_log2;
    const long long t1 = min(n, t0 + (1LL << tile_log2));
    double sr = 0.0, si = 0.0;
    for (long long i = t0 + threadIdx.x; i < t1; i += 256) {
        const double2 x = X[i], y = Y[i];
        const double xi = CONJ ? -x.y : x.y;
        // products rounded separately (no FMA contraction), as in tcb_dot: <x|x> has an exactly zero imaginary part
        sr = __dadd_rn(sr, __dsub_rn(__dmul_rn(x.x, y.x), __dmul_rn(xi, y.y)));
        si = __dadd_rn(si, __dadd_rn(__dmul_rn(x.x, y.y), __dmul_rn(xi, y.x)));
    }
    __shared__ double wr[8], wi[8];
    __shared__ bool last;
#pragma unroll
    for (int d = 16; d >= 1; d >>= 1) {                 // fixed tree
        sr = __dadd_rn(sr, __shfl_down_sync(0xffffffffu, sr, d));
        si = __dadd_rn(si, __shfl_down_sync(0xffffffffu, si, d));
    }
    if ((threadIdx.x & 31) == 0) { wr[threadIdx.x >> 5] = sr; wi[threadIdx.x >> 5] = si; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 8; ++w) { sr = __dadd_rn(sr, wr[w]); si = __dadd_rn(si, wi[w]); }
        partial[blockIdx.x] = make_double2(sr, si);
        __threadfence();                                // the partial sum is visible before the arrival is
        last = atomicAdd(counter, 1u) == gridDim.x - 1;
    }
    __syncthreads();
    if (!last) return;
    // ---- the block that arrived last adds the partial sums in block order (the same order whichever block it is)
    __threadfence();
    const volatile double2 *vp = partial;
    sr = 0.0; si = 0.0;
    for (unsigned b = threadIdx.x; b < gridDim.x; b += 256) {
        sr = __dadd_rn(sr, vp[b].x);
        si = __dadd_rn(si, vp[b].y);
    }
#pragma unroll
    for (int d = 16; d >= 1; d >>= 1) {
        sr = __dadd_rn(sr, __shfl_down_sync(0xffffffffu, sr, d));
        si = __dadd_rn(si, __shfl_down_sync(0xffffffffu, si, d));
    }
    __syncthreads();                                    // wr / wi are reused
    if ((threadIdx.x & 31) == 0) { wr[threadIdx.x >> 5] = sr; wi[threadIdx.x >> 5] = si; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 8; ++w) { sr = __dadd_rn(sr, wr[w]); si = __dadd_rn(si, wi[w]); }
        *D = make_double2(ar * sr - ai * si, ar * si + ai * sr);
        *counter = 0;                                   // the next call on this stream finds it cleared (it clears it anyway)
    }
}

// The device address of g_scratch on the CURRENT device: cudaGetSymbolAddress once per device, cached.
constexpr int kMaxDev = 64;
std::mutex g_mu;
unsigned char *g_addr[kMaxDev];

cudaError_t dot_noalloc_scratch(unsigned char **out)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDev) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_mu);
    if (!g_addr[dev]) {
        void *p = nullptr;
        e = cudaGetSymbolAddress(&p, g_scratch);        // set-up, with device `dev` current: no allocation, a lookup
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_addr[dev] = static_cast<unsigned char *>(p);
    }
    *out = g_addr[dev];
    return cudaSuccess;
}

}  // namespace

static int dot_noalloc_tile_log2(int64_t n)
{
    int t = kMinTileLog2;
    while (t < kMaxTileLog2 && ((n + (1LL << t) - 1) >> t) > kNoAllocMaxBlocks) ++t;
    return t;
}

cudaError_t launch_dot_noalloc(void *D, const void *X, const void *Y, int64_t n, bool conj_x, double re, double im,
                               cudaStream_t s, int64_t *launches)
{
    if (n < 0 || n > kNoAllocMaxElems) return cudaErrorInvalidValue;      // the entry point has refused it already
    unsigned char *scratch = nullptr;
    cudaError_t e = dot_noalloc_scratch(&scratch);
    if (e != cudaSuccess) return e;
    const int tl = dot_noalloc_tile_log2(n);
    const int nblocks = (int)std::max<int64_t>(1, (n + (1LL << tl) - 1) >> tl);
    e = cudaMemsetAsync(scratch, 0, sizeof(unsigned int), s);             // the arrival counter starts at zero
    if (e != cudaSuccess) return e;
    if (conj_x)
        dot_noalloc_kernel<true><<<nblocks, 256, 0, s>>>((const double2 *)X, (const double2 *)Y, n, tl, scratch, (double2 *)D, re, im);
    else
        dot_noalloc_kernel<false><<<nblocks, 256, 0, s>>>((const double2 *)X, (const double2 *)Y, n, tl, scratch, (double2 *)D, re, im);
    e = cudaGetLastError();
    if (e == cudaSuccess && launches) ++*launches;
    return e;
}

}  // namespace tcb
