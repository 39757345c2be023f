// permsum.cu -- S6: fused permute-sum (antisymmetrise / scale / accumulate).
//
//   D[i] = beta * D[i] + sum_{t<nterms} c_t * X[pi_t(i)]          terms added in order, each product and each
//                                                                  sum rounded on its own (bit-reproducible)
// The generator unrolls permutation operators P(ab), P(ij), P(a/bc)P(k/ij) into such signed terms
// (PAPER.md:194, 230, 284); fusing them into one pass reads X once per term through L2 and touches D once.
//
// Two kernels: permsum_cube_kernel (warp = micro-cube over the unit-stride indices of the terms, running offsets; the
// fast path for <= 9 terms whose cube tiles the extents) and permsum_kernel (any term set, one thread per element).
#include "kernels.h"

#include <algorithm>
#include <cstdlib>
#include <numeric>
#include <vector>

namespace tcb {

namespace {

struct PermSumParams {
    int rank, nterms;
    long long e[kMaxRank];
    long long n;
    long long xs[kMaxTerms][kMaxRank];
    double cr[kMaxTerms], ci[kMaxTerms];
    double br, bi;
    int beta_zero;
    const double2 *X;
    double2 *D;
};

__global__ void __launch_bounds__(256) permsum_kernel(const __grid_constant__ PermSumParams p)
{
    for (long long i = blockIdx.x * 256LL + threadIdx.x; i < p.n; i += gridDim.x * 256LL) {
        long long idx[kMaxRank];
        long long rem = i;
#pragma unroll
        for (int d = 0; d < kMaxRank; ++d) {
            idx[d] = rem % p.e[d];
            rem /= p.e[d];
        }
        double ar = 0.0, ai = 0.0;
        if (!p.beta_zero) {
            const double2 d = p.D[i];
            ar = __dsub_rn(__dmul_rn(p.br, d.x), __dmul_rn(p.bi, d.y));
            ai = __dadd_rn(__dmul_rn(p.br, d.y), __dmul_rn(p.bi, d.x));
        }
        for (int t = 0; t < p.nterms; ++t) {
            long long off = 0;
#pragma unroll
            for (int d = 0; d < kMaxRank; ++d) off += idx[d] * p.xs[t][d];
            const double2 x = p.X[off];
            const double cr = p.cr[t], ci = p.ci[t];
            ar = __dadd_rn(ar, __dsub_rn(__dmul_rn(cr, x.x), __dmul_rn(ci, x.y)));
            ai = __dadd_rn(ai, __dadd_rn(__dmul_rn(cr, x.y), __dmul_rn(ci, x.x)));
        }
        p.D[i] = make_double2(ar, ai);
    }
}


// ---- cube-run variant --------------------------------------------------------------------------------------------
// The generic kernel above decodes every element with six 64-bit divisions and gathers permuted terms 16 bytes at a
// time out of 32-byte sectors (ncu on R3 += P(a/bc)P(k/ij) X: 108 GB of L2 sectors and 45 GB of DRAM reads for 6 GB
// of X).  Here the 32 lanes of a warp cover a micro-cube over the indices that are unit-stride in X for some term
// (4 x 4 x 2 of (a,b,c)), so every term's gather -- whichever index it runs along -- reads whole sectors; a warp walks
// a row of cubes along index 0, and each term's offset is a running 64-bit sum: one add per element and term, one
// index decode per row.  Term order and rounding are those of the generic kernel (bit-identical results).
struct CubeParams {
    int rank, nterms;
    int e[kMaxRank], m[kMaxRank], nc[kMaxRank];   // extents, cube extents, cubes per dim
    long long ds[kMaxRank];
    long long xs[9][kMaxRank];
    double cr[9], ci[9], br, bi;
    int beta_zero;
    int lanes;                                     // lanes of a warp that hold an element (prod m <= 32)
    unsigned nunits;                               // rows of cubes = prod_{d>=1} nc[d]
    const double2 *X;
    double2 *D;
};

#ifndef CUBE_MINB
#define CUBE_MINB 3
#endif
template <int NT>
__global__ void __launch_bounds__(256, CUBE_MINB) permsum_cube_kernel(const __grid_constant__ CubeParams p)
{
    const int lane = threadIdx.x & 31;
    if (lane >= p.lanes) return;
    int l[kMaxRank];
    {
        int rem = lane;
#pragma unroll
        for (int d = 0; d < kMaxRank; ++d) { l[d] = rem % p.m[d]; rem /= p.m[d]; }
    }
    const unsigned warps = gridDim.x * (blockDim.x >> 5);
    for (unsigned u = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); u < p.nunits; u += warps) {
        unsigned rem = u;
        long long doff = l[0];
        long long xoff[NT];
#pragma unroll
        for (int t = 0; t < NT; ++t) xoff[t] = (long long)l[0] * p.xs[t][0];
#pragma unroll
        for (int d = 1; d < kMaxRank; ++d) {
            const unsigned c = rem % (unsigned)p.nc[d];
            rem /= (unsigned)p.nc[d];
            const long long idx = (long long)(c * (unsigned)p.m[d]) + l[d];
            doff += idx * p.ds[d];
#pragma unroll
            for (int t = 0; t < NT; ++t) xoff[t] += idx * p.xs[t][d];
        }
        for (int r = 0; r < p.nc[0]; ++r) {
            double ar = 0.0, ai = 0.0;
            double2 x[NT];
#pragma unroll
            for (int t = 0; t < NT; ++t)
                if (t < p.nterms) x[t] = p.X[xoff[t]];
            if (!p.beta_zero) {
                const double2 d = p.D[doff];
                ar = __dsub_rn(__dmul_rn(p.br, d.x), __dmul_rn(p.bi, d.y));
                ai = __dadd_rn(__dmul_rn(p.br, d.y), __dmul_rn(p.bi, d.x));
            }
#pragma unroll
            for (int t = 0; t < NT; ++t)
                if (t < p.nterms) {
                    const double cr = p.cr[t], ci = p.ci[t];
                    ar = __dadd_rn(ar, __dsub_rn(__dmul_rn(cr, x[t].x), __dmul_rn(ci, x[t].y)));
                    ai = __dadd_rn(ai, __dadd_rn(__dmul_rn(cr, x[t].y), __dmul_rn(ci, x[t].x)));
                }
            p.D[doff] = make_double2(ar, ai);
            doff += p.m[0];
#pragma unroll
            for (int t = 0; t < NT; ++t) xoff[t] += (long long)p.m[0] * p.xs[t][0];
        }
    }
}

// returns true when the cube-run kernel was launched
bool try_cube(const PermSumDesc &d, cudaStream_t stream, cudaError_t *err)
{
    if (d.nterms > 9 || d.rank < 2 || getenv("TCB_PERMSUM_GENERIC")) return false;
    CubeParams p;
    p.rank = d.rank; p.nterms = d.nterms;
    long long n = 1;
    for (int k = 0; k < kMaxRank; ++k) {
        const long long ek = k < d.rank ? d.extent[k] : 1;
        if (ek > 0x7fffffffLL) return false;
        p.e[k] = (int)ek; p.ds[k] = n; n *= ek; p.m[k] = 1;
    }
    if (n < (1LL << 18)) return false;                    // small tensors: launch latency decides, keep the simple kernel
    bool fast[kMaxRank] = {false, false, false, false, false, false};
    if (p.e[0] < 2) return false;
    fast[0] = true;
    for (int t = 0; t < d.nterms; ++t)
        for (int k = 0; k < d.rank; ++k)
            if (p.e[k] > 1 && d.xstride[t][k] == 1) fast[k] = true;
    int nf = 0;
    for (int k = 0; k < d.rank; ++k) nf += fast[k] ? 1 : 0;
    if (nf > 3) return false;                              // more than three unit-stride indices: the generic kernel
    // cube extents: divisors of the extents, each >= 2 (whole sectors for every term), product <= 32 and as large
    // as possible, the larger factors on the lower (D-contiguous) indices; lanes beyond the product idle
    int fdim[3], nfd = 0;
    for (int k = 0; k < d.rank; ++k)
        if (fast[k]) fdim[nfd++] = k;
    int best[3] = {0, 0, 0}, best_prod = 0;
    for (int m0 = 2; m0 <= 32; ++m0) {
        if (p.e[fdim[0]] % m0) continue;
        if (nfd == 1) { if (m0 > best_prod) { best_prod = m0; best[0] = m0; best[1] = best[2] = 1; } continue; }
        for (int m1 = 2; m0 * m1 <= 32; ++m1) {
            if (p.e[fdim[1]] % m1 || m1 > m0) continue;
            if (nfd == 2) {
                if (m0 * m1 > best_prod) { best_prod = m0 * m1; best[0] = m0; best[1] = m1; best[2] = 1; }
                continue;
            }
            for (int m2 = 2; m0 * m1 * m2 <= 32; ++m2) {
                if (p.e[fdim[2]] % m2 || m2 > m1) continue;
                if (m0 * m1 * m2 > best_prod) { best_prod = m0 * m1 * m2; best[0] = m0; best[1] = m1; best[2] = m2; }
            }
        }
    }
    if (best_prod < 24) return false;                       // less than 3/4 of the lanes: the generic kernel
    for (int f = 0; f < nfd; ++f) p.m[fdim[f]] = best[f];
    p.lanes = best_prod;
    long long units = 1;
    for (int k = 0; k < kMaxRank; ++k) { p.nc[k] = p.e[k] / p.m[k]; if (k >= 1) units *= p.nc[k]; }
    if (units >= (1LL << 32)) return false;
    p.nunits = (unsigned)units;
    for (int t = 0; t < 9; ++t) {
        for (int k = 0; k < kMaxRank; ++k) p.xs[t][k] = (t < d.nterms && k < d.rank && p.e[k] > 1) ? d.xstride[t][k] : 0;
        p.cr[t] = t < d.nterms ? d.coef_re[t] : 0.0;
        p.ci[t] = t < d.nterms ? d.coef_im[t] : 0.0;
    }
    p.br = d.beta_re; p.bi = d.beta_im;
    p.beta_zero = (d.beta_re == 0.0 && d.beta_im == 0.0) ? 1 : 0;
    p.X = (const double2 *)d.X;
    p.D = (double2 *)d.D;
    // resident CTAs per SM, measured: the 9-term instantiation (80 registers) is fastest and steadiest with 2 (8.4 ms
    // on configs[3]; 9.4-11 with 3-4), the 4-term one (64 registers) with 4
    static const int env_ctas = getenv("TCB_PERMSUM_CTAS") ? atoi(getenv("TCB_PERMSUM_CTAS")) : 0;
    const int ctas = env_ctas > 0 ? env_ctas : (d.nterms <= 4 ? 4 : 2);
    const unsigned blocks = (unsigned)std::min<long long>((units + 7) / 8, (long long)sm_count() * ctas);
    if (d.nterms <= 4) permsum_cube_kernel<4><<<blocks, 256, 0, stream>>>(p);
    else permsum_cube_kernel<9><<<blocks, 256, 0, stream>>>(p);
    *err = cudaGetLastError();
    return true;
}

}  // namespace

cudaError_t launch_permsum(const PermSumDesc &d, cudaStream_t stream, int64_t *launches)
{
    {
        bool handled = false;
        cudaError_t oe = launch_permsum_orbit(d, stream, launches, &handled);
        if (oe != cudaSuccess || handled) return oe;
    }
    {
        cudaError_t ce = cudaSuccess;
        if (try_cube(d, stream, &ce)) {
            if (ce == cudaSuccess && launches) ++*launches;
            return ce;
        }
    }
    PermSumParams p;
    p.rank = d.rank;
    p.nterms = d.nterms;
    p.n = 1;
    for (int k = 0; k < kMaxRank; ++k) {
        p.e[k] = k < d.rank ? d.extent[k] : 1;
        p.n *= p.e[k];
    }
    for (int t = 0; t < kMaxTerms; ++t) {
        for (int k = 0; k < kMaxRank; ++k) p.xs[t][k] = (t < d.nterms && k < d.rank) ? d.xstride[t][k] : 0;
        p.cr[t] = t < d.nterms ? d.coef_re[t] : 0.0;
        p.ci[t] = t < d.nterms ? d.coef_im[t] : 0.0;
    }
    p.br = d.beta_re; p.bi = d.beta_im;
    p.beta_zero = (d.beta_re == 0.0 && d.beta_im == 0.0) ? 1 : 0;
    p.X = (const double2 *)d.X;
    p.D = (double2 *)d.D;
    long long blocks = (p.n + 255) / 256;
    if (blocks > sm_count() * 16LL) blocks = sm_count() * 16LL;
    if (blocks < 1) blocks = 1;
    permsum_kernel<<<(int)blocks, 256, 0, stream>>>(p);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess && launches) ++*launches;
    return e;
}

}  // namespace tcb
