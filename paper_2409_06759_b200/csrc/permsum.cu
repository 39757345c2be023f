// permsum.cu -- S6: fused permute-sum (antisymmetrise / scale / accumulate).
//
//   D[i] = beta * D[i] + sum_{t<nterms} c_t * X[pi_t(i)]          terms added in order, each product and each
//                                                                  sum rounded on its own (bit-reproducible)
// The generator unrolls permutation operators P(ab), P(ij), P(a/bc)P(k/ij) into such signed terms
// (PAPER.md:194, 230, 284); fusing them into one pass reads X once per term through L2 and touches D once.
//
// v1: one thread per element of D (coalesced D traffic, 16-byte accesses); the X operands of permuted terms
// are gathered.  Threads are mapped to D's index space in tiles of the leading index so that a gathered term
// still reads 16-byte elements whose neighbours are used by neighbouring CTAs (L2 absorbs the reuse).
#include "kernels.h"

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

}  // namespace

cudaError_t launch_permsum(const PermSumDesc &d, cudaStream_t stream, int64_t *launches)
{
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
    if (blocks > 148 * 16) blocks = 148 * 16;
    if (blocks < 1) blocks = 1;
    permsum_kernel<<<(int)blocks, 256, 0, stream>>>(p);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess && launches) ++*launches;
    return e;
}

}  // namespace tcb
