// sympack.cu -- index-permutation-symmetric (antisymmetric) packed storage: tcb_pack / tcb_unpack.
//
// The paper names index-permutation symmetry as the feature its production code does not exploit yet (PAPER.md:202, 264,
// 440, 452).  Reading taken (reading 16, oracle/sym.py): a group a<b (a<b<c) of labels in which a tensor is
// antisymmetric is stored as ONE packed index over the strictly increasing tuples, first label fastest:
//     p(a<b) = b(b-1)/2 + a,        p(a<b<c) = c(c-1)(c-2)/6 + b(b-1)/2 + a.
// A packed tensor is an ordinary tensor handle whose packed index has extent n(n-1)/2 (n(n-1)(n-2)/6), so contractions over
// whole groups are plain tcb_contract calls on the packed indices: the pp ladder R(ab,ij) += V(ab,cd) T(cd,ij) runs at 1/8
// of the dense flops and with no factor 1/2.
//
//   pack   : Dp[.., p, ..] = L[.., a, .., b, ..]            pure data movement, bit-exact; one offset table per packed index
//   unpack : D[.., a, .., b, ..] (+)= alpha * sign * Lp[.., p(sorted), ..],  sign = parity of the sort, 0 on equal labels
//
// Both are HBM-bound streaming kernels over rows along the unit-stride index (pack: a CTA per row of the packed tensor;
// unpack: a warp per row of the dense tensor, 32 consecutive rows per warp); the row's multi-index is decoded once per row,
// per element only the group that holds the unit-stride index is evaluated.
#include "kernels.h"

#include <algorithm>

namespace tcb {

namespace {

struct PackParams {
    int rank;                          // of the packed tensor
    long long e[kMaxRank];             // packed extents
    const long long *tab[kMaxRank];    // device: offset into the dense tensor contributed by packed index value i of dim d
    long long nrows;                   // prod e[1..]
    const double2 *in;
    double2 *out;
};

__global__ void __launch_bounds__(256) pack_kernel(const __grid_constant__ PackParams p)
{
    const long long e0 = p.e[0];
    const long long *t0 = p.tab[0];
    for (long long row = blockIdx.x; row < p.nrows; row += gridDim.x) {
        long long r = row, off = 0;
#pragma unroll
        for (int d = 1; d < kMaxRank; ++d) {
            if (d >= p.rank) break;
            const long long i = r % p.e[d];
            r /= p.e[d];
            off += __ldg(p.tab[d] + i);
        }
        const double2 *src = p.in + off;
        double2 *dst = p.out + row * e0;
        for (long long i = threadIdx.x; i < e0; i += blockDim.x) dst[i] = src[__ldg(t0 + i)];
    }
}

struct UnpackParams {
    int rank;                          // dense rank
    long long e[kMaxRank];             // dense extents
    int ngroups;
    int glen[kMaxRank];                // labels per group (1..3)
    int gpos[kMaxRank][3];             // dense positions of the group's labels
    long long pstride[kMaxRank];       // stride of the group's packed index in Lp
    int g0, g0slot;                    // the group that holds dense position 0, and where in it
    long long nrows;
    double ar, ai;
    int accumulate;
    const double2 *in;
    double2 *out;
};

// packed position of a strictly increasing tuple
__device__ __forceinline__ long long tuple_pos(int len, long long a, long long b, long long c)
{
    if (len == 1) return a;
    if (len == 2) return b * (b - 1) / 2 + a;
    return c * (c - 1) * (c - 2) / 6 + b * (b - 1) / 2 + a;
}
// sorts (x, y, z) ascending (len of them valid); returns the sign of the sorting permutation, 0 if two coincide
__device__ __forceinline__ int sort_sign(int len, long long &x, long long &y, long long &z)
{
    int s = 1;
    if (len == 1) return 1;
    if (len == 2) {
        if (x == y) return 0;
        if (x > y) { const long long t = x; x = y; y = t; s = -1; }
        return s;
    }
    if (x == y || y == z || x == z) return 0;
    if (x > y) { const long long t = x; x = y; y = t; s = -s; }
    if (y > z) { const long long t = y; y = z; z = t; s = -s; }
    if (x > y) { const long long t = x; x = y; y = t; s = -s; }
    return s;
}

// idx[pos] with idx kept in registers (a dynamically indexed array would live in local memory)
__device__ __forceinline__ long long pick(const long long (&idx)[kMaxRank], int pos)
{
    long long r = idx[0];
#pragma unroll
    for (int d = 1; d < kMaxRank; ++d) r = pos == d ? idx[d] : r;
    return r;
}

constexpr int kRowChunk = 32;   // consecutive rows per warp: one 64-bit decode, then an odometer

// One WARP per row (a row = the dense tensor's unit-stride index, e0 elements), kRowChunk consecutive rows per warp.  The
// groups that do not hold the unit-stride index give one packed offset and one sign per row; per element only the group
// holding index 0 is sorted.  (The first version gave a 256-thread CTA one row at a time: 24 ms for a 6 GB tensor with
// e0 = 60, 0.5 TB/s.)
__global__ void __launch_bounds__(256) unpack_kernel(const __grid_constant__ UnpackParams p)
{
    const long long e0 = p.e[0];
    const int lane = threadIdx.x & 31;
    const long long gwarp = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    const long long nwarps = (long long)gridDim.x * (blockDim.x >> 5);
    const long long nchunks = (p.nrows + kRowChunk - 1) / kRowChunk;
    const int len0 = p.glen[p.g0];
    const long long ps0 = p.pstride[p.g0];
    for (long long chunk = gwarp; chunk < nchunks; chunk += nwarps) {
        const long long row0 = chunk * kRowChunk;
        const long long rend = row0 + kRowChunk < p.nrows ? row0 + kRowChunk : p.nrows;
        long long idx[kMaxRank];
        {
            long long r = row0;
            idx[0] = 0;
#pragma unroll
            for (int d = 1; d < kMaxRank; ++d) {
                idx[d] = 0;
                if (d < p.rank) { idx[d] = r % p.e[d]; r /= p.e[d]; }
            }
        }
        for (long long row = row0; row < rend; ++row) {
            long long off = 0;
            int sign = 1;
            for (int g = 0; g < p.ngroups; ++g) {
                if (g == p.g0) continue;
                const int gl = p.glen[g];
                long long x = pick(idx, p.gpos[g][0]), y = gl > 1 ? pick(idx, p.gpos[g][1]) : 0,
                          z = gl > 2 ? pick(idx, p.gpos[g][2]) : 0;
                sign *= sort_sign(gl, x, y, z);
                off += tuple_pos(gl, x, y, z) * p.pstride[g];
            }
            // the other members of the unit-stride index's group
            long long m1 = 0, m2 = 0;
            {
                int q = 0;
                for (int s = 0; s < len0; ++s) {
                    if (s == p.g0slot) continue;
                    const long long val = pick(idx, p.gpos[p.g0][s]);
                    if (q == 0) m1 = val; else m2 = val;
                    ++q;
                }
            }
            double2 *dst = p.out + row * e0;
            if (sign == 0) {
                if (!p.accumulate)
                    for (long long i = lane; i < e0; i += 32) dst[i] = make_double2(0.0, 0.0);
            } else {
                const double2 *src = p.in + off;
                for (long long i = lane; i < e0; i += 32) {
                    // the tuple in the group's own label order: i sits in slot g0slot
                    long long x, y = 0, z = 0;
                    if (len0 == 1) { x = i; }
                    else if (len0 == 2) { x = p.g0slot == 0 ? i : m1; y = p.g0slot == 0 ? m1 : i; }
                    else {
                        x = p.g0slot == 0 ? i : m1;
                        y = p.g0slot == 1 ? i : (p.g0slot == 0 ? m1 : m2);
                        z = p.g0slot == 2 ? i : m2;
                    }
                    const int sg = sign * sort_sign(len0, x, y, z);
                    double2 v = make_double2(0.0, 0.0);
                    if (sg != 0) {
                        const double2 w = src[tuple_pos(len0, x, y, z) * ps0];
                        // alpha * (sign * w): the sign is an exact negation; products and sums rounded one by one
                        const double wr = sg > 0 ? w.x : -w.x, wi = sg > 0 ? w.y : -w.y;
                        v.x = __dsub_rn(__dmul_rn(p.ar, wr), __dmul_rn(p.ai, wi));
                        v.y = __dadd_rn(__dmul_rn(p.ar, wi), __dmul_rn(p.ai, wr));
                    }
                    if (p.accumulate) {
                        const double2 d = dst[i];
                        v.x = __dadd_rn(d.x, v.x);
                        v.y = __dadd_rn(d.y, v.y);
                    }
                    dst[i] = v;
                }
            }
            // odometer over dims 1..rank-1
#pragma unroll
            for (int d = 1; d < kMaxRank; ++d) {
                if (d < p.rank) {
                    if (++idx[d] < p.e[d]) break;
                    idx[d] = 0;
                }
            }
        }
    }
}

// ---- symmap: D and L both packed (tcb_unpack onto a packed D, tcb_antisym_pack) ------------------------------------------------
struct SymMapParams {
    int nd, nl, nterms, accumulate;
    long long dext[kMaxRank];
    int dlen[kMaxRank];
    const SymTuple *dtab[kMaxRank];
    int llen[kMaxRank];
    int lsrc_dim[kMaxRank][3], lsrc_slot[kMaxRank][3];
    long long lstride[kMaxRank];
    unsigned char perm[kMaxSymTerms][kMaxRank][3];
    signed char sign[kMaxSymTerms];
    long long total;
    int touch0[kMaxRank];                   // L group g holds a label of D's index 0
    long long nrows;                        // total / dext[0]
    int tdim[kMaxRank];                     // rows are visited in an order of their own: position k (>= 1) runs D's index tdim[k]
    long long tdiv[kMaxRank];               // row / tdiv[k] % dext[tdim[k]] = that index
    long long dstride[kMaxRank];            // element stride of D's index d
    double ar, ai;
    const double2 *in;
    double2 *out;
};

__device__ __forceinline__ long long tuple_word(const SymMapParams &p, int d, long long i)
{
    if (p.dlen[d] == 1) return i;
    const SymTuple t = p.dtab[d][i];
    return (long long)t.v[0] | ((long long)t.v[1] << 16) | ((long long)t.v[2] << 32);
}

constexpr int kTileU = 8;                   // elements of D's index 0 per thread and tile

__device__ __forceinline__ int sort_sign32(int len, unsigned &x, unsigned &y, unsigned &z)
{
    int s = 1;
    if (len == 1) return 1;
    if (len == 2) {
        if (x == y) return 0;
        if (x > y) { const unsigned t = x; x = y; y = t; s = -1; }
        return s;
    }
    if (x == y || y == z || x == z) return 0;
    if (x > y) { const unsigned t = x; x = y; y = t; s = -s; }
    if (y > z) { const unsigned t = y; y = z; z = t; s = -s; }
    if (x > y) { const unsigned t = x; x = y; y = t; s = -s; }
    return s;
}
// packed position of a strictly increasing tuple; group labels are below 65536 (one label alone: any 32-bit value)
__device__ __forceinline__ long long tuple_pos32(int len, unsigned a, unsigned b, unsigned c)
{
    if (len == 1) return a;
    const unsigned pb = (b * (b - 1)) >> 1;
    if (len == 2) return (long long)pb + a;
    return (long long)((unsigned long long)((c * (c - 1)) >> 1) * (c - 2) / 3) + pb + a;
}

// The tiled kernel behind tcb_unpack onto a packed D (one identity term) and tcb_antisym_pack (the shuffles).  A tile =
// 256 * kTileU consecutive values of D's index 0 at fixed other indices ("row").  Per tile, through shared memory: the
// tuples of the row's indices (one 64-bit division each, by one thread each), the value every L label fed by them takes
// under every term, and per term the packed offset and sign of the L groups fed by the row alone.  Per element and term only
// the groups holding a label of D's index 0 are sorted, in 32-bit arithmetic.  (One thread per element with everything
// recomputed: 358 instructions per element, 21 ms for a 15 GB view; the first tiled version with a per-thread row decode:
// 12.8 ms.)
__global__ void __launch_bounds__(256) symtile_kernel(const __grid_constant__ SymMapParams p)
{
    __shared__ long long s_tup[kMaxRank];
    __shared__ long long s_idx[kMaxRank];
    __shared__ unsigned s_val[kMaxSymTerms][kMaxRank][3];
    __shared__ long long s_off[kMaxSymTerms];
    __shared__ int s_sgn[kMaxSymTerms];
    const long long e0 = p.dext[0];
    const long long tile_elems = 256 * kTileU;
    const long long tiles_per_row = (e0 + tile_elems - 1) / tile_elems;
    const long long ntiles = p.nrows * tiles_per_row;
    const int tid = threadIdx.x;
    const int len0 = p.dlen[0];
    for (long long tile = blockIdx.x; tile < ntiles; tile += gridDim.x) {
        const long long row = tile / tiles_per_row, chunk = tile - row * tiles_per_row;
        __syncthreads();
        if (tid >= 1 && tid < p.nd) {
            const int d = p.tdim[tid];
            const long long i = (row / p.tdiv[tid]) % p.dext[d];
            s_idx[d] = i;
            s_tup[d] = tuple_word(p, d, i);
        }
        __syncthreads();
        for (int q = tid; q < p.nterms * kMaxRank * 3; q += 256) {
            const int t = q / (kMaxRank * 3), g = (q / 3) % kMaxRank, sl = q % 3;
            unsigned val = 0;
            if (g < p.nl && sl < p.llen[g]) {
                const int d = p.lsrc_dim[g][sl];
                if (d != 0) {
                    const long long w = s_tup[d];
                    val = p.dlen[d] == 1 ? (unsigned)w : (unsigned)(w >> (16 * p.perm[t][d][p.lsrc_slot[g][sl]])) & 0xffffu;
                }
            }
            s_val[t][g][sl] = val;
        }
        __syncthreads();
        if (tid < p.nterms) {
            long long off = 0;
            int sg = p.sign[tid];
            for (int g = 0; g < p.nl; ++g) {
                if (p.touch0[g]) continue;
                unsigned x = s_val[tid][g][0], y = s_val[tid][g][1], z = s_val[tid][g][2];
                sg *= sort_sign32(p.llen[g], x, y, z);
                off += tuple_pos32(p.llen[g], x, y, z) * p.lstride[g];
            }
            s_off[tid] = off;
            s_sgn[tid] = sg;
        }
        __syncthreads();
        long long rowoff = 0;
#pragma unroll
        for (int d = 1; d < kMaxRank; ++d)
            if (d < p.nd) rowoff += s_idx[d] * p.dstride[d];
        double2 *dst = p.out + rowoff;
        for (int u = 0; u < kTileU; ++u) {
            const long long i0 = chunk * tile_elems + u * 256 + tid;
            if (i0 >= e0) break;
            long long w0 = i0;
            if (len0 > 1) {
                const SymTuple t0 = p.dtab[0][i0];
                w0 = (long long)t0.v[0] | ((long long)t0.v[1] << 16) | ((long long)t0.v[2] << 32);
            }
            double sr = 0.0, si = 0.0;
            for (int t = 0; t < p.nterms; ++t) {
                int sg = s_sgn[t];
                if (sg == 0) continue;
                long long off = s_off[t];
                for (int g = 0; g < p.nl; ++g) {
                    if (!p.touch0[g]) continue;
                    unsigned val[3] = {0, 0, 0};
#pragma unroll
                    for (int sl = 0; sl < 3; ++sl) {
                        if (sl < p.llen[g]) {
                            if (p.lsrc_dim[g][sl] == 0)
                                val[sl] = len0 == 1 ? (unsigned)w0 : (unsigned)(w0 >> (16 * p.perm[t][0][p.lsrc_slot[g][sl]])) & 0xffffu;
                            else
                                val[sl] = s_val[t][g][sl];
                        }
                    }
                    sg *= sort_sign32(p.llen[g], val[0], val[1], val[2]);
                    off += tuple_pos32(p.llen[g], val[0], val[1], val[2]) * p.lstride[g];
                }
                if (sg != 0) {
                    const double2 w = p.in[off];
                    sr = __dadd_rn(sr, sg > 0 ? w.x : -w.x);
                    si = __dadd_rn(si, sg > 0 ? w.y : -w.y);
                }
            }
            double2 v;
            v.x = __dsub_rn(__dmul_rn(p.ar, sr), __dmul_rn(p.ai, si));
            v.y = __dadd_rn(__dmul_rn(p.ar, si), __dmul_rn(p.ai, sr));
            if (p.accumulate) {
                const double2 d = dst[i0];
                v.x = __dadd_rn(d.x, v.x);
                v.y = __dadd_rn(d.y, v.y);
            }
            dst[i0] = v;
        }
    }
}

// Fallback (a short index 0 of D, where a tile would be mostly empty): one thread per element of D.  The tuple of every D index sits in one
// 64-bit register (16 bits per component; a single-label index keeps its full value), so nothing is indexed dynamically.
__global__ void __launch_bounds__(256) symmap_kernel(const __grid_constant__ SymMapParams p)
{
    const long long step = (long long)gridDim.x * blockDim.x;
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < p.total; e += step) {
        long long tup[kMaxRank];
        {
            long long r = e;
#pragma unroll
            for (int d = 0; d < kMaxRank; ++d) {
                tup[d] = 0;
                if (d < p.nd) {
                    const long long i = r % p.dext[d];
                    r /= p.dext[d];
                    if (p.dlen[d] == 1) tup[d] = i;
                    else {
                        const SymTuple t = p.dtab[d][i];
                        tup[d] = (long long)t.v[0] | ((long long)t.v[1] << 16) | ((long long)t.v[2] << 32);
                    }
                }
            }
        }
        double sr = 0.0, si = 0.0;
        for (int t = 0; t < p.nterms; ++t) {
            long long off = 0;
            int sg = p.sign[t];
            for (int g = 0; g < p.nl; ++g) {
                long long val[3] = {0, 0, 0};
#pragma unroll
                for (int s = 0; s < 3; ++s) {
                    if (s < p.llen[g]) {
                        const int d = p.lsrc_dim[g][s];
                        const long long w = pick(tup, d);
                        val[s] = p.dlen[d] == 1 ? w : (w >> (16 * p.perm[t][d][p.lsrc_slot[g][s]])) & 0xffff;
                    }
                }
                sg *= sort_sign(p.llen[g], val[0], val[1], val[2]);
                off += tuple_pos(p.llen[g], val[0], val[1], val[2]) * p.lstride[g];
            }
            if (sg != 0) {
                const double2 w = p.in[off];
                sr = __dadd_rn(sr, sg > 0 ? w.x : -w.x);
                si = __dadd_rn(si, sg > 0 ? w.y : -w.y);
            }
        }
        double2 v;
        v.x = __dsub_rn(__dmul_rn(p.ar, sr), __dmul_rn(p.ai, si));
        v.y = __dadd_rn(__dmul_rn(p.ar, si), __dmul_rn(p.ai, sr));
        if (p.accumulate) {
            const double2 d = p.out[e];
            v.x = __dadd_rn(d.x, v.x);
            v.y = __dadd_rn(d.y, v.y);
        }
        p.out[e] = v;
    }
}

}  // namespace

cudaError_t launch_pack(const PackDesc &d, cudaStream_t stream, int64_t *launches)
{
    PackParams p;
    p.rank = d.rank;
    p.nrows = 1;
    for (int k = 0; k < kMaxRank; ++k) {
        p.e[k] = k < d.rank ? d.extent[k] : 1;
        p.tab[k] = k < d.rank ? (const long long *)d.tab[k] : nullptr;
        if (k >= 1) p.nrows *= p.e[k];
    }
    p.in = (const double2 *)d.in;
    p.out = (double2 *)d.out;
    const int blocks = (int)std::max<long long>(1, std::min<long long>(p.nrows, 16LL * sm_count()));
    pack_kernel<<<blocks, 256, 0, stream>>>(p);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess && launches) ++*launches;
    return e;
}

cudaError_t launch_unpack(const UnpackDesc &d, cudaStream_t stream, int64_t *launches)
{
    UnpackParams p;
    p.rank = d.rank;
    p.nrows = 1;
    for (int k = 0; k < kMaxRank; ++k) {
        p.e[k] = k < d.rank ? d.extent[k] : 1;
        if (k >= 1) p.nrows *= p.e[k];
    }
    p.ngroups = d.ngroups;
    p.g0 = -1; p.g0slot = 0;
    for (int g = 0; g < kMaxRank; ++g) {
        p.glen[g] = g < d.ngroups ? d.glen[g] : 1;
        p.pstride[g] = g < d.ngroups ? d.pstride[g] : 0;
        for (int s = 0; s < 3; ++s) {
            p.gpos[g][s] = (g < d.ngroups && s < d.glen[g]) ? d.gpos[g][s] : 0;
            if (g < d.ngroups && s < d.glen[g] && d.gpos[g][s] == 0) { p.g0 = g; p.g0slot = s; }
        }
    }
    if (p.g0 < 0) return cudaErrorInvalidValue;
    p.ar = d.alpha_re; p.ai = d.alpha_im;
    p.accumulate = d.accumulate ? 1 : 0;
    p.in = (const double2 *)d.in;
    p.out = (double2 *)d.out;
    const long long chunks = (p.nrows + kRowChunk - 1) / kRowChunk;
    const int blocks = (int)std::max<long long>(1, std::min<long long>((chunks + 7) / 8, 8LL * sm_count()));
    unpack_kernel<<<blocks, 256, 0, stream>>>(p);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess && launches) ++*launches;
    return e;
}

cudaError_t launch_symmap(const SymMapDesc &d, cudaStream_t stream, int64_t *launches)
{
    SymMapParams p;
    p.nd = d.nd; p.nl = d.nl; p.nterms = d.nterms; p.accumulate = d.accumulate ? 1 : 0;
    p.total = 1;
    for (int k = 0; k < kMaxRank; ++k) {
        p.dext[k] = k < d.nd ? d.dext[k] : 1;
        p.dlen[k] = k < d.nd ? d.dlen[k] : 1;
        p.dtab[k] = k < d.nd ? d.dtab[k] : nullptr;
        p.llen[k] = k < d.nl ? d.llen[k] : 1;
        p.lstride[k] = k < d.nl ? d.lstride[k] : 0;
        for (int s = 0; s < 3; ++s) {
            p.lsrc_dim[k][s] = (k < d.nl && s < d.llen[k]) ? d.lsrc_dim[k][s] : 0;
            p.lsrc_slot[k][s] = (k < d.nl && s < d.llen[k]) ? d.lsrc_slot[k][s] : 0;
        }
        p.total *= p.dext[k];
    }
    if (d.nterms < 1 || d.nterms > kMaxSymTerms) return cudaErrorInvalidValue;
    for (int t = 0; t < kMaxSymTerms; ++t) {
        p.sign[t] = t < d.nterms ? d.sign[t] : 0;
        for (int k = 0; k < kMaxRank; ++k)
            for (int s = 0; s < 3; ++s) p.perm[t][k][s] = t < d.nterms ? d.perm[t][k][s] : (unsigned char)s;
    }
    p.ar = d.alpha_re; p.ai = d.alpha_im;
    p.in = (const double2 *)d.in;
    p.out = (double2 *)d.out;
    for (int g = 0; g < kMaxRank; ++g) {
        p.touch0[g] = 0;
        for (int s2 = 0; s2 < 3; ++s2)
            if (g < d.nl && s2 < d.llen[g] && d.lsrc_dim[g][s2] == 0) p.touch0[g] = 1;
    }
    p.nrows = p.total / p.dext[0];
    bool fits32 = true;
    {   // Row order: the index of D that feeds the L labels of SMALLEST stride runs fastest, so that consecutive tiles read the
        // same stretch of L (view Tr(b<c,j<k,e,m) of T3p at o=16, v=100: e before (j<k) keeps one 2.6 MB column of T3p in L2
        // instead of cycling through 120 of them: DRAM reads 38.7 GB -> see profiles/r2_sympack_ncu.md).
        long long key[kMaxRank], st = 1;
        for (int k = 0; k < kMaxRank; ++k) {
            p.dstride[k] = st;
            st *= p.dext[k];
            fits32 = fits32 && p.dext[k] < (1LL << 31);
            key[k] = 0;
            for (int g = 0; g < d.nl; ++g)
                for (int s2 = 0; s2 < d.llen[g]; ++s2)
                    if (d.lsrc_dim[g][s2] == k) key[k] = std::max<long long>(key[k], d.lstride[g]);
        }
        int order[kMaxRank];
        for (int k = 0; k < kMaxRank; ++k) order[k] = k;
        if (d.nd > 2) std::stable_sort(order + 1, order + d.nd, [&](int x, int y) { return key[x] < key[y]; });
        long long div = 1;
        for (int k = 0; k < kMaxRank; ++k) {
            p.tdim[k] = order[k];
            p.tdiv[k] = div;
            if (k >= 1 && k < d.nd) div *= p.dext[order[k]];
        }
    }
    if (p.dext[0] >= 128 && fits32) {
        const long long tiles = p.nrows * ((p.dext[0] + 256 * kTileU - 1) / (256 * kTileU));
        const int vb = (int)std::max<long long>(1, std::min<long long>(tiles, 16LL * sm_count()));
        symtile_kernel<<<vb, 256, 0, stream>>>(p);
        cudaError_t ve = cudaGetLastError();
        if (ve == cudaSuccess && launches) ++*launches;
        return ve;
    }
    const int blocks = (int)std::max<long long>(1, std::min<long long>((p.total + 255) / 256, 16LL * sm_count()));
    symmap_kernel<<<blocks, 256, 0, stream>>>(p);
    cudaError_t e = cudaGetLastError();
    if (e == cudaSuccess && launches) ++*launches;
    return e;
}

}  // namespace tcb
