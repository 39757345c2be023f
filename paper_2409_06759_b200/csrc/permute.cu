// permute.cu -- S3: tensor transposition ("reshape"), the memory-bound pass of TTGT, and the
// permuted add  D (+)= alpha * perm(L)  built on the same data movement.
//
//   out[sum_d idx_d * ostride[d]] (op)= in[sum_d idx_d * istride[d]]
//
// One element is one complex128 = one 16-byte vector access (LDG.128 / STG.128), so "vectorised" is per
// element.  The kernel is a generalised tiled transpose: a tile is a hyper-rectangle of the index space whose
// extents are chosen on the host so that (a) the leading INPUT dims inside the tile span >= 32 contiguous
// elements (512-byte read runs) and (b) the leading OUTPUT dims inside the tile span >= 32 contiguous elements
// of the output (512-byte write runs).  When an extent is small (occupied indices, 6..40) the tile simply
// spans the next index too (compound runs).  Threads read the tile in input order (coalesced), park it in
// shared memory, and write it in output order (coalesced); the shared-memory stride of the output-fastest dim
// is padded to an odd number of 16-byte slots so that the gather side is bank-conflict free.
// Each thread keeps its tile-local offsets in registers (they are identical for every tile) and the CTA
// loops over tiles (persistent grid), so the per-element index arithmetic is one add; boundary tiles mask with
// packed per-dim indices.  All global offsets are 64-bit (V of config 3 is 25.6 GB).
#include "kernels.h"

#include <algorithm>

namespace tcb {

namespace {

constexpr int PT = 256;            // threads per CTA
constexpr int kMaxVol = 4096;      // elements per tile (64 KB)

struct PermParams {
    int t[kMaxRank];               // tile extents
    int ntile[kMaxRank];
    int q[kMaxRank];               // dims in output order (q[0] = output unit stride)
    int ss[kMaxRank];              // shared-memory strides (elements)
    int sh[kMaxRank];              // bit position of dim d inside a packed tile-local index
    int mk[kMaxRank];              // (1 << bits(d)) - 1
    long long e[kMaxRank], is[kMaxRank], os[kMaxRank];
    int vol;
    long long ntiles;
    const double2 *in;
    double2 *out;
    double ar, ai;
};

// OffT: type of the tile-local offsets (int when every t[d]*stride[d] sum fits 31 bits, else long long)
template <int J, int OP, typename OffT>
__global__ void __launch_bounds__(PT) permute_kernel(const PermParams p)
{
    extern __shared__ double2 tile_smem[];
    const int tid = threadIdx.x;

    OffT inoff[J], outoff[J];
    unsigned inidx[J], outidx[J], sp[J];       // sp = smem slot for the load side | store side << 16
#pragma unroll
    for (int j = 0; j < J; ++j) {
        const int e = tid + PT * j;
        long long io = 0, oo = 0;
        unsigned ii = 0, oi = 0;
        int si = 0, so = 0;
        int rem = e;
#pragma unroll
        for (int d = 0; d < kMaxRank; ++d) {
            const int i = rem % p.t[d];
            rem /= p.t[d];
            io += (long long)i * p.is[d];
            si += i * p.ss[d];
            ii |= (unsigned)i << p.sh[d];
        }
        rem = e;
#pragma unroll
        for (int x = 0; x < kMaxRank; ++x) {
            const int d = p.q[x];
            const int i = rem % p.t[d];
            rem /= p.t[d];
            oo += (long long)i * p.os[d];
            so += i * p.ss[d];
            oi |= (unsigned)i << p.sh[d];
        }
        inoff[j] = (OffT)io; outoff[j] = (OffT)oo; inidx[j] = ii; outidx[j] = oi;
        sp[j] = (unsigned)si | ((unsigned)so << 16);
    }

    for (long long tile = blockIdx.x; tile < p.ntiles; tile += gridDim.x) {
        long long base_in = 0, base_out = 0;
        int lim[kMaxRank];               // last valid tile-local index per dim
        bool interior = true;
        {
            long long rem = tile;
#pragma unroll
            for (int d = 0; d < kMaxRank; ++d) {
                const long long tc = rem % p.ntile[d];
                rem /= p.ntile[d];
                const long long o = tc * p.t[d];
                base_in += o * p.is[d];
                base_out += o * p.os[d];
                const long long l = min((long long)p.t[d], p.e[d] - o);
                interior = interior && (l == p.t[d]);
                lim[d] = (int)l - 1;
            }
        }
        auto inside = [&](unsigned idx) {
            bool ok = true;
#pragma unroll
            for (int d = 0; d < kMaxRank; ++d) ok = ok && ((int)((idx >> p.sh[d]) & p.mk[d]) <= lim[d]);
            return ok;
        };
        const double2 *src = p.in + base_in;
        double2 *dst = p.out + base_out;

        double2 v[J];
#pragma unroll
        for (int j = 0; j < J; ++j) {
            const bool ok = (tid + PT * j < p.vol) && (interior || inside(inidx[j]));
            v[j] = ok ? src[inoff[j]] : make_double2(0.0, 0.0);
        }
#pragma unroll
        for (int j = 0; j < J; ++j)
            if (tid + PT * j < p.vol) tile_smem[sp[j] & 0xffffu] = v[j];
        __syncthreads();
        bool okv[J];
#pragma unroll
        for (int j = 0; j < J; ++j) {
            okv[j] = (tid + PT * j < p.vol) && (interior || inside(outidx[j]));
            if (OP == kPermAccumulate) v[j] = okv[j] ? dst[outoff[j]] : make_double2(0.0, 0.0);
        }
#pragma unroll
        for (int j = 0; j < J; ++j) {
            if (!okv[j]) continue;
            const double2 x = tile_smem[sp[j] >> 16];
            double2 y;
            if (OP == kPermCopy) {
                y = x;
            } else {
                y.x = __dsub_rn(__dmul_rn(p.ar, x.x), __dmul_rn(p.ai, x.y));
                y.y = __dadd_rn(__dmul_rn(p.ar, x.y), __dmul_rn(p.ai, x.x));
                if (OP == kPermAccumulate) {
                    y.x = __dadd_rn(v[j].x, y.x);
                    y.y = __dadd_rn(v[j].y, y.y);
                }
            }
            dst[outoff[j]] = y;
        }
        __syncthreads();
    }
}

template <int J, typename OffT>
cudaError_t launch_j(const PermParams &p, PermuteOp op, int blocks, size_t smem, cudaStream_t stream)
{
    auto set = [&](auto kern) {
        cudaError_t e = cudaSuccess;
        if (smem > 48 * 1024) e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
        kern<<<blocks, PT, smem, stream>>>(p);
        return cudaGetLastError();
    };
    switch (op) {
    case kPermCopy: return set(permute_kernel<J, kPermCopy, OffT>);
    case kPermScale: return set(permute_kernel<J, kPermScale, OffT>);
    default: return set(permute_kernel<J, kPermAccumulate, OffT>);
    }
}

int env_int(const char *name, int dflt)
{
    const char *s = getenv(name);
    return s ? atoi(s) : dflt;
}

}  // namespace

cudaError_t launch_permute(const PermuteDesc &pd, cudaStream_t stream, int64_t *launches)
{
    PermParams p;
    const int r = pd.rank;
    for (int d = 0; d < kMaxRank; ++d) {
        p.t[d] = 1; p.ntile[d] = 1; p.q[d] = d; p.ss[d] = 0; p.sh[d] = 0; p.mk[d] = 0;
        p.e[d] = d < r ? pd.extent[d] : 1;
        p.is[d] = d < r ? pd.istride[d] : 0;
        p.os[d] = d < r ? pd.ostride[d] : 0;
    }
    // dims in output order
    int q[kMaxRank];
    for (int d = 0; d < kMaxRank; ++d) q[d] = d;
    std::stable_sort(q, q + r, [&](int a, int b) { return pd.ostride[a] < pd.ostride[b]; });
    for (int d = 0; d < kMaxRank; ++d) p.q[d] = q[d];

    const int TI = env_int("TCB_PERM_TI", 32), TO = env_int("TCB_PERM_TO", 32);
    const int VOL = env_int("TCB_PERM_VOL", 1024);
    long long prod = 1;
    for (int d = 0; d < r && prod < TI; ++d) {
        const long long need = (TI + prod - 1) / prod;
        p.t[d] = (int)std::max<long long>(p.t[d], std::min<long long>(p.e[d], need));
        prod *= p.t[d];
    }
    prod = 1;
    for (int x = 0; x < r && prod < TO; ++x) {
        const int d = q[x];
        const long long need = (TO + prod - 1) / prod;
        p.t[d] = (int)std::max<long long>(p.t[d], std::min<long long>(p.e[d], need));
        prod *= p.t[d];
    }
    auto volume = [&] { long long v = 1; for (int d = 0; d < r; ++d) v *= p.t[d]; return v; };
    // grow (input-leading dims first: longer runs on both sides when dim 0 leads both) up to the volume target
    for (int d = 0; d < r && volume() < VOL; ++d) {
        while (p.t[d] < p.e[d] && p.t[d] < 1024 && volume() < VOL) {
            const long long room = VOL / (volume() / p.t[d]);
            int nt = (int)std::min<long long>(std::min<long long>(p.e[d], 1024), std::max<long long>(p.t[d] + 1, room));
            if (volume() / p.t[d] * nt > kMaxVol) break;
            p.t[d] = nt;
        }
    }
    // even out the tiles of each dim (e = 60, t = 32 -> 2 tiles of 30)
    for (int d = 0; d < r; ++d) {
        const long long n = (p.e[d] + p.t[d] - 1) / p.t[d];
        p.t[d] = (int)((p.e[d] + n - 1) / n);
        p.ntile[d] = (int)n;
    }
    if (volume() > kMaxVol) return cudaErrorInvalidValue;
    p.vol = (int)volume();
    p.ntiles = 1;
    for (int d = 0; d < r; ++d) p.ntiles *= p.ntile[d];
    // shared-memory strides in input order; the output-fastest dim gets an odd stride
    int s = 1;
    for (int d = 0; d < r; ++d) {
        if (d == q[0] && d != 0 && (s % 2 == 0)) s += 1;
        p.ss[d] = s;
        s *= p.t[d];
    }
    const size_t smem = (size_t)s * sizeof(double2);
    p.in = (const double2 *)pd.in;
    p.out = (double2 *)pd.out;
    p.ar = pd.alpha_re; p.ai = pd.alpha_im;

    const int J = (p.vol + PT - 1) / PT;
    const int ctas_per_sm = std::max(1, std::min(8, (int)(200 * 1024 / std::max<size_t>(smem, 8 * 1024))));
    int blocks = (int)std::min<long long>(p.ntiles, 148LL * env_int("TCB_PERM_CTAS", ctas_per_sm));
    // packed tile-local index: bits(d) = ceil(log2 t[d]); sum <= log2(vol) + rank <= 18
    int bit = 0;
    long long max_in = 0, max_out = 0;
    for (int d = 0; d < kMaxRank; ++d) {
        int b = 0;
        while ((1 << b) < p.t[d]) ++b;
        p.sh[d] = bit;
        p.mk[d] = (1 << b) - 1;
        bit += b;
        max_in += (long long)(p.t[d] - 1) * p.is[d];
        max_out += (long long)(p.t[d] - 1) * p.os[d];
    }
    if (bit > 31 || s >= 65536) return cudaErrorInvalidValue;
    const bool small = max_in < (1LL << 31) && max_out < (1LL << 31);
    cudaError_t e;
    if (small) {
        if (J <= 2) e = launch_j<2, int>(p, pd.op, blocks, smem, stream);
        else if (J <= 4) e = launch_j<4, int>(p, pd.op, blocks, smem, stream);
        else if (J <= 8) e = launch_j<8, int>(p, pd.op, blocks, smem, stream);
        else e = launch_j<16, int>(p, pd.op, blocks, smem, stream);
    } else {
        if (J <= 2) e = launch_j<2, long long>(p, pd.op, blocks, smem, stream);
        else if (J <= 4) e = launch_j<4, long long>(p, pd.op, blocks, smem, stream);
        else if (J <= 8) e = launch_j<8, long long>(p, pd.op, blocks, smem, stream);
        else e = launch_j<16, long long>(p, pd.op, blocks, smem, stream);
    }
    if (e == cudaSuccess && launches) ++*launches;
    return e;
}

}  // namespace tcb
