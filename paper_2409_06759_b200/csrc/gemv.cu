// gemv.cu -- S2 regime "GEMV": contractions in which one operand is contracted away completely (N = 1), e.g.
//   Fae(a,e) += ovvv(m,a,f,e) * T1(f,m)      R1(a,i) += T2(a,e,i,m) * Fme(m,e)        (CCSD: still binary)
// As a GEMM these waste 63 of 64 tile columns and, worse, first permute the big operand into matrix form (1.6 GB for
// ovvv at v = 150).  But a tensor's element offset is a SUM over its indices, so any operand is a matrix with a row table
// and a column table:  A[m,k] = L[offAm[m] + offAk[k]].  This kernel reads the big operand once, in place, in its own
// memory order:
//   D[offD[m]] (+)= alpha * sum_k L[offAm[m] + offAk[k]] * R[offBk[k]]
// m-fast (L's unit-stride index is free): one thread per m, consecutive threads read consecutive addresses, the R values
//   and column offsets of a k-tile are staged in shared memory;
// k-fast (L's unit-stride index is contracted): one warp per m, lanes along k, shuffle reduction in a fixed tree.
// K can be cut into `ksplit` chunks (few rows, long K): partial sums are written per chunk and added in chunk order by
// gemv_reduce_kernel -- deterministic, no atomics.  HBM-bound: algorithmic bytes = 16 (M K + K + M (2 if += else 1)).
#include "kernels.h"

#include <algorithm>

namespace tcb {

namespace {

constexpr int GT = 256;        // threads per CTA
constexpr int KT = 256;        // k-tile staged in shared memory (m-fast)

struct GemvParams {
    long long M, K, kchunk;
    const double2 *A, *B;
    double2 *D, *partial;        // partial: [ksplit][M] when ksplit > 1
    const long long *offAm, *offAk, *offBk, *offD;
    double ar, ai;
    int accumulate, ksplit;
};

__device__ __forceinline__ void cmac(double2 &acc, const double2 a, const double2 b)
{
    acc.x = fma(a.x, b.x, fma(-a.y, b.y, acc.x));
    acc.y = fma(a.x, b.y, fma(a.y, b.x, acc.y));
}

__device__ __forceinline__ void finish(const GemvParams &p, long long m, double2 acc, long long chunk)
{
    if (p.ksplit > 1) {
        p.partial[chunk * p.M + m] = acc;
        return;
    }
    double2 v = make_double2(p.ar * acc.x - p.ai * acc.y, p.ar * acc.y + p.ai * acc.x);
    double2 *dst = p.D + p.offD[m];
    if (p.accumulate) { const double2 d = *dst; v.x += d.x; v.y += d.y; }
    *dst = v;
}

__global__ void __launch_bounds__(GT) gemv_mfast_kernel(const __grid_constant__ GemvParams p)
{
    __shared__ double2 s_b[KT];
    __shared__ long long s_o[KT];
    const long long m = (long long)blockIdx.x * GT + threadIdx.x;
    const long long k0 = (long long)blockIdx.y * p.kchunk, k1 = min(p.K, k0 + p.kchunk);
    const double2 *row = p.A + (m < p.M ? p.offAm[m] : 0);
    double2 acc = make_double2(0.0, 0.0);
    for (long long kb = k0; kb < k1; kb += KT) {
        const int nk = (int)min((long long)KT, k1 - kb);
        __syncthreads();
        if (threadIdx.x < nk) {
            s_b[threadIdx.x] = p.B[p.offBk[kb + threadIdx.x]];
            s_o[threadIdx.x] = p.offAk[kb + threadIdx.x];
        }
        __syncthreads();
        if (m < p.M) {
            int k = 0;
            for (; k + 4 <= nk; k += 4) {              // four independent loads in flight per thread
                const double2 a0 = row[s_o[k]], a1 = row[s_o[k + 1]], a2 = row[s_o[k + 2]], a3 = row[s_o[k + 3]];
                cmac(acc, a0, s_b[k]); cmac(acc, a1, s_b[k + 1]); cmac(acc, a2, s_b[k + 2]); cmac(acc, a3, s_b[k + 3]);
            }
            for (; k < nk; ++k) cmac(acc, row[s_o[k]], s_b[k]);
        }
    }
    if (m < p.M) finish(p, m, acc, blockIdx.y);
}

__global__ void __launch_bounds__(GT) gemv_kfast_kernel(const __grid_constant__ GemvParams p)
{
    // one warp per (row, k-chunk) pair, rows fastest: with few rows (M = 1: a full contraction into a rank-0 tensor) all
    // eight warps of a CTA still have work (one warp per CTA ran E() = V(i,j,a,b) T(a,b,i,j) at 0.8 TB/s)
    const int lane = threadIdx.x & 31;
    const long long pair = (long long)blockIdx.x * (GT / 32) + (threadIdx.x >> 5);
    const long long chunk = pair / p.M, m = pair - chunk * p.M;
    if (chunk >= p.ksplit) return;
    const long long k0 = chunk * p.kchunk, k1 = min(p.K, k0 + p.kchunk);
    const double2 *row = p.A + p.offAm[m];
    double2 acc[2] = {make_double2(0.0, 0.0), make_double2(0.0, 0.0)};
    long long k = k0 + lane;
    for (; k + 32 < k1; k += 64) {                      // two independent chains per lane
        const double2 a0 = row[p.offAk[k]], a1 = row[p.offAk[k + 32]];
        cmac(acc[0], a0, p.B[p.offBk[k]]);
        cmac(acc[1], a1, p.B[p.offBk[k + 32]]);
    }
    if (k < k1) cmac(acc[0], row[p.offAk[k]], p.B[p.offBk[k]]);
    double2 s = make_double2(acc[0].x + acc[1].x, acc[0].y + acc[1].y);
#pragma unroll
    for (int d = 16; d >= 1; d >>= 1) {                 // fixed tree: bit-reproducible
        s.x += __shfl_down_sync(0xffffffffu, s.x, d);
        s.y += __shfl_down_sync(0xffffffffu, s.y, d);
    }
    if (lane == 0) finish(p, m, s, chunk);
}

// chunk partials -> D: one warp per row, lanes stride over the chunks in order, then a fixed shuffle tree (deterministic)
__global__ void __launch_bounds__(GT) gemv_reduce_kernel(const __grid_constant__ GemvParams p)
{
    const int lane = threadIdx.x & 31;
    const long long m = (long long)blockIdx.x * (GT / 32) + (threadIdx.x >> 5);
    if (m >= p.M) return;
    double2 acc = make_double2(0.0, 0.0);
    for (int s = lane; s < p.ksplit; s += 32) {
        const double2 v = p.partial[(long long)s * p.M + m];
        acc.x += v.x; acc.y += v.y;
    }
#pragma unroll
    for (int d = 16; d >= 1; d >>= 1) {
        acc.x += __shfl_down_sync(0xffffffffu, acc.x, d);
        acc.y += __shfl_down_sync(0xffffffffu, acc.y, d);
    }
    if (lane != 0) return;
    double2 v = make_double2(p.ar * acc.x - p.ai * acc.y, p.ar * acc.y + p.ai * acc.x);
    double2 *dst = p.D + p.offD[m];
    if (p.accumulate) { const double2 d = *dst; v.x += d.x; v.y += d.y; }
    *dst = v;
}

// ---- regime "outer product" (K = 1: no index is contracted), e.g. tt(a,b,i,j) = T1(a,i) * T1(b,j) of CCSD -----------------
//   D[offM[m] + offN[n]] (+)= alpha * A[rowA[m]] * B[rowB[n]]
// A pure store (or read-modify-write) stream: through the DMMA GEMM it ran with K padded to 4 and 64 x 64 tiles at 0.53 of
// the HBM bound.  Here a CTA owns 256 rows x 32 columns; lanes run along m (D's unit-stride index leads the row order), the
// row's A value lives in a register, the 32 B values and column offsets in shared memory.
struct OuterParams {
    long long M, N;
    const double2 *A, *B;
    double2 *D;
    const long long *rowA, *rowB, *offM, *offN;
    double ar, ai;
    int accumulate;
};
constexpr int kOuterCols = 32;

__global__ void __launch_bounds__(GT) outer_kernel(const __grid_constant__ OuterParams p)
{
    __shared__ double2 s_b[kOuterCols];
    __shared__ long long s_on[kOuterCols];
    const long long mtiles = (p.M + GT - 1) / GT, ntiles = (p.N + kOuterCols - 1) / kOuterCols;
    for (long long tile = blockIdx.x; tile < mtiles * ntiles; tile += gridDim.x) {
        const long long tn = tile / mtiles, tm = tile - tn * mtiles;
        const long long n0 = tn * kOuterCols;
        const int nn = (int)min((long long)kOuterCols, p.N - n0);
        __syncthreads();
        if (threadIdx.x < nn) {
            const double2 b = p.B[p.rowB[n0 + threadIdx.x]];
            // alpha * b once per column: the element then costs one complex product
            s_b[threadIdx.x] = make_double2(p.ar * b.x - p.ai * b.y, p.ar * b.y + p.ai * b.x);
            s_on[threadIdx.x] = p.offN[n0 + threadIdx.x];
        }
        __syncthreads();
        const long long m = tm * GT + threadIdx.x;
        if (m >= p.M) continue;
        const double2 a = p.A[p.rowA[m]];
        double2 *drow = p.D + p.offM[m];
        if (p.accumulate) {
#pragma unroll 4
            for (int j = 0; j < nn; ++j) {
                const double2 b = s_b[j];
                double2 *dst = drow + s_on[j];
                const double2 d = *dst;
                *dst = make_double2(fma(a.x, b.x, fma(-a.y, b.y, d.x)), fma(a.x, b.y, fma(a.y, b.x, d.y)));
            }
        } else {
#pragma unroll 4
            for (int j = 0; j < nn; ++j) {
                const double2 b = s_b[j];
                drow[s_on[j]] = make_double2(fma(a.x, b.x, -a.y * b.y), fma(a.x, b.y, a.y * b.x));
            }
        }
    }
}

}  // namespace

cudaError_t launch_outer(const OuterDesc &g, cudaStream_t stream, int64_t *launches)
{
    OuterParams p;
    p.M = g.M; p.N = g.N;
    p.A = (const double2 *)g.A; p.B = (const double2 *)g.B; p.D = (double2 *)g.D;
    p.rowA = (const long long *)g.rowA; p.rowB = (const long long *)g.rowB;
    p.offM = (const long long *)g.offM; p.offN = (const long long *)g.offN;
    p.ar = g.alpha_re; p.ai = g.alpha_im;
    p.accumulate = g.accumulate ? 1 : 0;
    const long long tiles = ((g.M + GT - 1) / GT) * ((g.N + kOuterCols - 1) / kOuterCols);
    const int blocks = (int)std::max<long long>(1, std::min<long long>(tiles, 8LL * sm_count()));
    outer_kernel<<<blocks, GT, 0, stream>>>(p);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess && launches) ++*launches;
    return e;
}

int gemv_ksplit(int64_t M, int64_t K, bool kfast)
{
    const int64_t sms = sm_count();
    if (kfast) {                                  // a warp per (row, chunk): 32 warps per SM wanted, chunks of >= 512
        const int64_t want = 32 * sms;
        const int64_t s = std::min<int64_t>((want + M - 1) / M, K / 512);
        return (int)std::max<int64_t>(1, std::min<int64_t>(s, want));
    }
    const int64_t ctas_m = (M + GT - 1) / GT;
    int64_t s = (4 * sms + ctas_m - 1) / ctas_m;
    s = std::min<int64_t>(s, K / 256);
    return (int)std::max<int64_t>(1, std::min<int64_t>(s, 64));
}

cudaError_t launch_gemv(const GemvDesc &g, cudaStream_t stream, int64_t *launches)
{
    GemvParams p;
    p.M = g.M; p.K = g.K;
    p.A = (const double2 *)g.A; p.B = (const double2 *)g.B; p.D = (double2 *)g.D;
    p.partial = (double2 *)g.partial;
    p.offAm = (const long long *)g.offAm; p.offAk = (const long long *)g.offAk;
    p.offBk = (const long long *)g.offBk; p.offD = (const long long *)g.offD;
    p.ar = g.alpha_re; p.ai = g.alpha_im;
    p.accumulate = g.accumulate ? 1 : 0;
    p.ksplit = gemv_ksplit(g.M, g.K, g.kfast);
    if (p.ksplit > 1 && !p.partial) return cudaErrorInvalidValue;
    p.kchunk = (g.K + p.ksplit - 1) / p.ksplit;
    p.kchunk = (p.kchunk + 63) / 64 * 64;
    p.ksplit = (int)((g.K + p.kchunk - 1) / p.kchunk);
    if (g.kfast) {
        const long long pairs = (long long)g.M * p.ksplit;
        gemv_kfast_kernel<<<(unsigned)((pairs + GT / 32 - 1) / (GT / 32)), GT, 0, stream>>>(p);
    } else {
        dim3 grid((unsigned)((g.M + GT - 1) / GT), (unsigned)p.ksplit);
        gemv_mfast_kernel<<<grid, GT, 0, stream>>>(p);
    }
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    if (launches) ++*launches;
    if (p.ksplit > 1) {
        gemv_reduce_kernel<<<(unsigned)((g.M + GT / 32 - 1) / (GT / 32)), GT, 0, stream>>>(p);
        e = cudaGetLastError();
        if (e == cudaSuccess && launches) ++*launches;
    }
    return e;
}

}  // namespace tcb
