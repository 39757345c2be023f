// elementwise.cu -- S7: fill, scale, axpy on dense complex128 tensors (north_star "tensor add/scale";
// the scalar factor of PAPER.md:230).  Memory-bound, one 16-byte access per element, grid-stride.
#include "kernels.h"

#include <algorithm>

namespace tcb {

namespace {

__global__ void __launch_bounds__(256) fill_kernel(double2 *D, long long n, double re, double im)
{
    const double2 v = make_double2(re, im);
    for (long long i = blockIdx.x * 256LL + threadIdx.x; i < n; i += gridDim.x * 256LL) D[i] = v;
}

__global__ void __launch_bounds__(256) scale_kernel(double2 *D, long long n, double ar, double ai)
{
    for (long long i = blockIdx.x * 256LL + threadIdx.x; i < n; i += gridDim.x * 256LL) {
        const double2 d = D[i];
        D[i] = make_double2(__dsub_rn(__dmul_rn(ar, d.x), __dmul_rn(ai, d.y)),
                            __dadd_rn(__dmul_rn(ar, d.y), __dmul_rn(ai, d.x)));
    }
}

template <bool ACC>
__global__ void __launch_bounds__(256)
axpy_kernel(double2 *D, const double2 *__restrict__ L, long long n, double ar, double ai)
{
    for (long long i = blockIdx.x * 256LL + threadIdx.x; i < n; i += gridDim.x * 256LL) {
        const double2 x = L[i];
        double2 y = make_double2(__dsub_rn(__dmul_rn(ar, x.x), __dmul_rn(ai, x.y)),
                                 __dadd_rn(__dmul_rn(ar, x.y), __dmul_rn(ai, x.x)));
        if (ACC) {
            const double2 d = D[i];
            y.x = __dadd_rn(d.x, y.x);
            y.y = __dadd_rn(d.y, y.y);
        }
        D[i] = y;
    }
}

int grid_for(long long n)
{
    long long b = (n + 255) / 256;
    if (b > sm_count() * 16LL) b = sm_count() * 16LL;
    return b < 1 ? 1 : (int)b;
}

}  // namespace

cudaError_t launch_fill(void *D, int64_t n, double re, double im, cudaStream_t s, int64_t *launches)
{
    fill_kernel<<<grid_for(n), 256, 0, s>>>((double2 *)D, n, re, im);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess && launches) ++*launches;
    return e;
}

cudaError_t launch_scale(void *D, int64_t n, double re, double im, cudaStream_t s, int64_t *launches)
{
    scale_kernel<<<grid_for(n), 256, 0, s>>>((double2 *)D, n, re, im);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess && launches) ++*launches;
    return e;
}

cudaError_t launch_axpy(void *D, const void *L, int64_t n, double re, double im, bool accumulate, cudaStream_t s,
                        int64_t *launches)
{
    if (accumulate)
        axpy_kernel<true><<<grid_for(n), 256, 0, s>>>((double2 *)D, (const double2 *)L, n, re, im);
    else
        axpy_kernel<false><<<grid_for(n), 256, 0, s>>>((double2 *)D, (const double2 *)L, n, re, im);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess && launches) ++*launches;
    return e;
}

// D = alpha * sum_i (conj?) X[i] * Y[i] -- the inner product a DIIS extrapolation needs.  Two deterministic stages:
// every block sums its grid-stride share in a fixed order (thread-sequential, then a fixed shuffle / shared-memory
// tree), then one block sums the per-block partials in index order.
template <bool CONJ>
__global__ void __launch_bounds__(256)
dot_partial_kernel(const double2 *__restrict__ X, const double2 *__restrict__ Y, long long n, double2 *partial)
{
    double sr = 0.0, si = 0.0;
    for (long long i = blockIdx.x * 256LL + threadIdx.x; i < n; i += gridDim.x * 256LL) {
        const double2 x = X[i], y = Y[i];
        const double xi = CONJ ? -x.y : x.y;
        // products rounded separately (no FMA contraction): <x|x> then has an exactly zero imaginary part
        sr = __dadd_rn(sr, __dsub_rn(__dmul_rn(x.x, y.x), __dmul_rn(xi, y.y)));
        si = __dadd_rn(si, __dadd_rn(__dmul_rn(x.x, y.y), __dmul_rn(xi, y.x)));
    }
#pragma unroll
    for (int d = 16; d >= 1; d >>= 1) {
        sr += __shfl_down_sync(0xffffffffu, sr, d);
        si += __shfl_down_sync(0xffffffffu, si, d);
    }
    __shared__ double wr[8], wi[8];
    if ((threadIdx.x & 31) == 0) { wr[threadIdx.x >> 5] = sr; wi[threadIdx.x >> 5] = si; }
    __syncthreads();
    if (threadIdx.x == 0) {
        for (int w = 1; w < 8; ++w) { sr += wr[w]; si += wi[w]; }
        partial[blockIdx.x] = make_double2(sr, si);
    }
}

__global__ void __launch_bounds__(32) dot_final_kernel(const double2 *partial, int nblocks, double2 *D, double ar, double ai)
{
    if (threadIdx.x != 0) return;
    double sr = 0.0, si = 0.0;
    for (int b = 0; b < nblocks; ++b) { sr += partial[b].x; si += partial[b].y; }
    *D = make_double2(ar * sr - ai * si, ar * si + ai * sr);
}

cudaError_t launch_dot(void *D, const void *X, const void *Y, int64_t n, bool conj_x, double re, double im, void *partial,
                       int nblocks, cudaStream_t s, int64_t *launches)
{
    if (conj_x) dot_partial_kernel<true><<<nblocks, 256, 0, s>>>((const double2 *)X, (const double2 *)Y, n, (double2 *)partial);
    else dot_partial_kernel<false><<<nblocks, 256, 0, s>>>((const double2 *)X, (const double2 *)Y, n, (double2 *)partial);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    dot_final_kernel<<<1, 32, 0, s>>>((const double2 *)partial, nblocks, (double2 *)D, re, im);
    e = cudaGetLastError();
    if (e == cudaSuccess && launches) *launches += 2;
    return e;
}

// T[idx] += alpha * R[idx] / (sum_k eps_k[idx_k])  -- the Jacobi step of a CC solver (orbital-energy denominators)
// A CTA takes a slab (the leading `ninner` dims, >= 2048 elements when the tensor has them) at a time: the outer
// indices and their energies are decoded once per slab, an element costs ninner - 1 32-bit divisions (the first
// version decoded every element with six 64-bit divisions: 4.9 ms on a 6 GB rank-6 tensor, 3.7 TB/s).
struct DenomParams {
    int rank, ninner;
    long long e[kMaxRank];
    int eps_at[kMaxRank];            // start of dim k's energies in `eps`, -1: the index does not enter the denominator
    const double *eps;
    double2 *T;
    const double2 *R;
    long long nslabs;
    unsigned slab;                   // elements per slab
    double ar, ai;
};

template <bool ACC>
__global__ void __launch_bounds__(256) denominator_update_kernel(const __grid_constant__ DenomParams p)
{
    for (long long sl = blockIdx.x; sl < p.nslabs; sl += gridDim.x) {
        // energies of the outer indices, added in index order AFTER the inner ones (so the sum keeps index order)
        double outer[kMaxRank];
        unsigned long long rem = (unsigned long long)sl;
#pragma unroll
        for (int k = 0; k < kMaxRank; ++k) {
            outer[k] = 0.0;
            if (k >= p.ninner && k < p.rank) {
                const unsigned long long q = rem / (unsigned long long)p.e[k];
                const long long ik = (long long)(rem - q * (unsigned long long)p.e[k]);
                rem = q;
                if (p.eps_at[k] >= 0) outer[k] = p.eps[p.eps_at[k] + ik];
            }
        }
        const long long base = sl * (long long)p.slab;
        // four elements per thread and round: all eight loads are issued before the first division
        for (unsigned j0 = threadIdx.x; j0 < p.slab; j0 += 4 * 256) {
            double2 x[4], t[4];
            double d[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const unsigned j = j0 + u * 256;
                if (j < p.slab) {
                    x[u] = p.R[base + j];
                    t[u] = ACC ? p.T[base + j] : make_double2(0.0, 0.0);
                }
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                unsigned r = j0 + u * 256;
                d[u] = 0.0;
#pragma unroll
                for (int k = 0; k < kMaxRank; ++k)
                    if (k < p.rank) {
                        if (k < p.ninner) {
                            const unsigned ek = (unsigned)p.e[k];
                            const unsigned q = k + 1 < p.ninner ? r / ek : 0u;
                            const unsigned ik = min(r - q * ek, ek - 1);      // (a lane past the slab reads a valid slot)
                            r = q;
                            if (p.eps_at[k] >= 0) d[u] = __dadd_rn(d[u], p.eps[p.eps_at[k] + ik]);
                        } else if (p.eps_at[k] >= 0) {
                            d[u] = __dadd_rn(d[u], outer[k]);
                        }
                    }
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const unsigned j = j0 + u * 256;
                if (j < p.slab) {
                    const double qr = __ddiv_rn(x[u].x, d[u]), qi = __ddiv_rn(x[u].y, d[u]);
                    const double ur = __dsub_rn(__dmul_rn(p.ar, qr), __dmul_rn(p.ai, qi));
                    const double ui = __dadd_rn(__dmul_rn(p.ar, qi), __dmul_rn(p.ai, qr));
                    t[u].x = ACC ? __dadd_rn(t[u].x, ur) : ur;
                    t[u].y = ACC ? __dadd_rn(t[u].y, ui) : ui;
                    p.T[base + j] = t[u];
                }
            }
        }
    }
}

cudaError_t launch_denominator_update(void *T, const void *R, int rank, const int64_t *extent, const double *eps_dev,
                                      const int *eps_at, double re, double im, bool accumulate, cudaStream_t s,
                                      int64_t *launches)
{
    DenomParams p;
    p.rank = rank;
    long long n = 1, slab = 1;
    p.ninner = 0;
    for (int k = 0; k < kMaxRank; ++k) {
        p.e[k] = k < rank ? extent[k] : 1;
        p.eps_at[k] = k < rank ? eps_at[k] : -1;
        n *= p.e[k];
        // the inner block is a contiguous PREFIX of the dims: it stops growing at the first dim that does not fit
        if (k < rank && p.ninner == k && (slab < 2048 || k == 0) && slab * p.e[k] <= (1LL << 30)) {
            slab *= p.e[k];
            p.ninner = k + 1;
        }
    }
    if (p.ninner == 0) {                                    // a leading extent above 2^30 (rank 0 never gets here)
        if (n > (1LL << 31)) return cudaErrorInvalidValue;
        p.ninner = rank; slab = n;
    }
    p.slab = (unsigned)slab;
    p.nslabs = n / slab;
    p.eps = eps_dev;
    p.T = (double2 *)T;
    p.R = (const double2 *)R;
    p.ar = re; p.ai = im;
    const int blocks = (int)std::max<long long>(1, std::min<long long>(p.nslabs, sm_count() * 8LL));
    if (accumulate) denominator_update_kernel<true><<<blocks, 256, 0, s>>>(p);
    else denominator_update_kernel<false><<<blocks, 256, 0, s>>>(p);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess && launches) ++*launches;
    return e;
}

}  // namespace tcb
