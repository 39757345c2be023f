// permute.cu -- S3: tensor transposition ("reshape"), the memory-bound pass of TTGT, and the
// permuted add  D (+)= alpha * perm(L)  built on the same data movement.
//
//   out[sum_d idx_d * ostride[d]] (op)= in[sum_d idx_d * istride[d]]
//
// One element is one complex128 = 16 bytes.  A tile is a hyper-rectangle of the index space whose extents are
// chosen on the host so that (a) the leading INPUT dims inside the tile span >= 32 contiguous elements and (b) the
// leading OUTPUT dims inside the tile span >= 32 contiguous elements of the output (512-byte runs on both sides;
// when an extent is small -- occupied indices, 6..40 -- the tile spans the next index too).
//
// B200 design (measured, profiles/r1b_permute.md): a load->sync->store tile loop cannot keep enough bytes in
// flight for HBM3e, so the LOAD side is asynchronous bulk copies (cp.async.bulk.shared::cluster.global, SASS
// UBLKCP): every contiguous input run of a tile ("row" = the tile's extent along the input unit-stride dim) is
// one bulk copy straight into shared memory, completion counted on an mbarrier; tiles rotate through a ring of
// 2 stages (TCB_PERM_STAGES: up to 4), so each CTA has one tile (~33 KB) in flight while it drains one.  Rows are copied to
// a padded pitch (the stride of the output-fastest dim is odd in 16-byte units), which makes the STORE side --
// threads gather the tile in output order with LDS.128 and write coalesced STG.128 -- bank-conflict free.
// A bulk copy costs its issuing warp ~32 cycles, so the rows of a tile are dealt round-robin to all 8 warps.
// Tile-local offsets are tile-invariant and live in registers; tile coordinates advance by a mixed-radix add
// (no division in the loop); boundary tiles mask with packed per-dim indices.  All global offsets are 64-bit
// (V of config 3 is 25.6 GB).
#include "kernels.h"
#include "ptx.cuh"

#include <algorithm>
#include <cstdlib>

namespace tcb {

namespace {

using namespace ptx;

constexpr int PT = 256;            // threads per CTA
constexpr int NW = PT / 32;
constexpr int kMaxVol = 4096;      // elements per tile (64 KB)
constexpr int kRowRegs = 2;        // rows per thread whose offsets are kept in registers
constexpr int kIdxBits = 18;       // packed tile-local index: sum_d ceil(log2 t[d]) <= 18; slot < 2^14
constexpr int kChunk = 8;          // elements a thread holds in registers at a time

struct PermParams {
    int t[kMaxRank];               // tile extents
    int ntile[kMaxRank];
    int step[kMaxRank];            // mixed-radix digits of gridDim.x (tile-coordinate increment)
    int q[kMaxRank];               // dims in output order (q[0] = output unit stride)
    int ss[kMaxRank];              // shared-memory strides (elements)
    int sh[kMaxRank];              // bit position of dim d inside a packed tile-local index
    int mk[kMaxRank];              // (1 << bits(d)) - 1
    long long e[kMaxRank], is[kMaxRank], os[kMaxRank];
    int vol, rows, stages, tile_bytes;
    long long ntiles;
    const double2 *in;
    double2 *out;
    double ar, ai;
};

__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void *src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}

// tile coordinates of one cursor (the load cursor runs `stages` tiles ahead of the store cursor)
struct Cursor {
    int c[kMaxRank];
    __device__ __forceinline__ void init(const PermParams &p, unsigned tile)   // tile < gridDim.x
    {
#pragma unroll
        for (int d = 0; d < kMaxRank; ++d) {
            c[d] = (int)(tile % (unsigned)p.ntile[d]);
            tile /= (unsigned)p.ntile[d];
        }
    }
    __device__ __forceinline__ void advance(const PermParams &p)
    {
        int carry = 0;
#pragma unroll
        for (int d = 0; d < kMaxRank; ++d) {
            int x = c[d] + p.step[d] + carry;
            carry = x >= p.ntile[d];
            c[d] = carry ? x - p.ntile[d] : x;
        }
    }
    // base offsets of the tile and the last valid tile-local index per dim
    __device__ __forceinline__ bool locate(const PermParams &p, const long long *stride, long long *base, int *lim) const
    {
        long long b = 0;
        bool interior = true;
#pragma unroll
        for (int d = 0; d < kMaxRank; ++d) {
            const long long o = (long long)c[d] * p.t[d];
            b += o * stride[d];
            const long long l = min((long long)p.t[d], p.e[d] - o);
            interior = interior && (l == p.t[d]);
            lim[d] = (int)l - 1;
        }
        *base = b;
        return interior;
    }
};

// OffT: type of the tile-local offsets (int when every t[d]*stride[d] sum fits 31 bits, else long long)
template <int J, int OP, typename OffT>
__global__ void __launch_bounds__(PT, (J > 8 ? 1 : 2)) permute_kernel(const __grid_constant__ PermParams p)
{
    extern __shared__ __align__(128) uint8_t perm_smem[];
    const uint32_t sbase = smem_u32(perm_smem);
    const uint32_t bars = sbase + (uint32_t)p.stages * p.tile_bytes;   // full[s] at +8s, empty[s] at +8(stages+s)
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int stages = p.stages;

    if (tid == 0) {
        for (int s = 0; s < stages; ++s) {
            mbar_init(bars + 8 * s, NW);
            mbar_init(bars + 8 * (stages + s), NW);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }

    // ---- store side: this thread's J elements of a tile, enumerated in OUTPUT order ------------------------
    // pack[j] = packed tile-local index (low kIdxBits bits) | shared-memory slot << kIdxBits
    OffT outoff[J];
    unsigned pack[J];
#pragma unroll
    for (int j = 0; j < J; ++j) {
        long long oo = 0;
        unsigned oi = 0;
        int so = 0;
        int rem = tid + PT * j;
#pragma unroll
        for (int x = 0; x < kMaxRank; ++x) {
            const int d = p.q[x];
            if (p.t[d] == 1) continue;
            const int i = rem % p.t[d];
            rem /= p.t[d];
            oo += (long long)i * p.os[d];
            so += i * p.ss[d];
            oi |= (unsigned)i << p.sh[d];
        }
        outoff[j] = (OffT)oo; pack[j] = oi | ((unsigned)so << kIdxBits);
    }
    // ---- load side: rows (runs along the input unit-stride dim) dealt round-robin to the warps ---------------
    // row r of a tile -> thread with lane * NW + warp == r mod PT
    auto decode_row = [&](int r, long long *goff, int *soff, unsigned *ridx) {
        long long g = 0;
        int s = 0;
        unsigned ii = 0;
#pragma unroll
        for (int d = 1; d < kMaxRank; ++d) {
            if (p.t[d] == 1) continue;
            const int i = r % p.t[d];
            r /= p.t[d];
            g += (long long)i * p.is[d];
            s += i * p.ss[d];
            ii |= (unsigned)i << p.sh[d];
        }
        *goff = g; *soff = s * 16; *ridx = ii;
    };
    const int row0 = lane * NW + warp;
    OffT rgoff[kRowRegs];
    int rsoff[kRowRegs];
    unsigned ridx[kRowRegs];
#pragma unroll
    for (int k = 0; k < kRowRegs; ++k) {
        long long g;
        decode_row(row0 + k * PT, &g, &rsoff[k], &ridx[k]);
        rgoff[k] = (OffT)g;
    }
    const int warp_rows = p.rows > warp ? (p.rows - 1 - warp) / NW + 1 : 0;
    const unsigned row_bytes = (unsigned)p.t[0] * 16u;
    __syncthreads();

    auto inside = [&](unsigned idx, const int *lim) {
        bool ok = true;
#pragma unroll
        for (int d = 0; d < kMaxRank; ++d) ok = ok && ((int)((idx >> p.sh[d]) & p.mk[d]) <= lim[d]);
        return ok;
    };

    const long long my_n = p.ntiles > blockIdx.x ? (p.ntiles - 1 - blockIdx.x) / gridDim.x + 1 : 0;
    Cursor lc, sc;
    lc.init(p, blockIdx.x);
    sc = lc;

    // issue every row of the load cursor's tile into stage s, then advance the cursor
    auto issue = [&](int s) {
        long long base_in;
        int lim[kMaxRank];
        const bool interior = lc.locate(p, p.is, &base_in, lim);
        lc.advance(p);
        const uint32_t dst = sbase + (uint32_t)s * p.tile_bytes, full = bars + 8 * s;
        const double2 *src = p.in + base_in;
        if (interior) {
            if (lane == 0) mbar_expect_tx(full, (unsigned)warp_rows * row_bytes);
            __syncwarp();
#pragma unroll
            for (int k = 0; k < kRowRegs; ++k)
                if (row0 + k * PT < p.rows) bulk_g2s(dst + rsoff[k], src + rgoff[k], row_bytes, full);
            for (int r = row0 + kRowRegs * PT; r < p.rows; r += PT) {
                long long g; int so; unsigned ri;
                decode_row(r, &g, &so, &ri);
                bulk_g2s(dst + so, src + g, row_bytes, full);
            }
        } else {
            const unsigned rb = (unsigned)(lim[0] + 1) * 16u;
            unsigned bytes = 0;
            for (int r = row0; r < p.rows; r += PT) {
                long long g; int so; unsigned ri;
                decode_row(r, &g, &so, &ri);
                if (inside(ri, lim)) bytes += rb;
            }
            bytes = __reduce_add_sync(0xffffffffu, bytes);
            if (lane == 0) mbar_expect_tx(full, bytes);
            __syncwarp();
            for (int r = row0; r < p.rows; r += PT) {
                long long g; int so; unsigned ri;
                decode_row(r, &g, &so, &ri);
                if (inside(ri, lim)) bulk_g2s(dst + so, src + g, rb, full);
            }
        }
    };

    const int npro = (int)min((long long)stages, my_n);
    for (int s = 0; s < npro; ++s) issue(s);

    int s = 0;
    uint32_t ph = 0;
    for (long long k = 0; k < my_n; ++k) {
        long long base_out;
        int lim[kMaxRank];
        const bool interior = sc.locate(p, p.os, &base_out, lim);
        sc.advance(p);
        double2 *dst = p.out + base_out;
        const uint32_t stile = sbase + (uint32_t)s * p.tile_bytes;

        mbar_wait(bars + 8 * s, ph);
#pragma unroll
        for (int j0 = 0; j0 < J; j0 += kChunk) {
            constexpr int C = J < kChunk ? J : kChunk;
            bool okv[C];
            double2 v[C], d[C];
#pragma unroll
            for (int c = 0; c < C; ++c) {
                const int j = j0 + c;
                okv[c] = (tid + PT * j < p.vol) && (interior || inside(pack[j] & ((1u << kIdxBits) - 1), lim));
                if (OP == kPermAccumulate && okv[c]) d[c] = dst[outoff[j]];
            }
#pragma unroll
            for (int c = 0; c < C; ++c)
                if (okv[c]) v[c] = lds128(stile + (pack[j0 + c] >> kIdxBits) * 16u);
            if (j0 + kChunk >= J) {          // last chunk: the stage is drained once these loads have landed
                __syncwarp();
                if (lane == 0) mbar_arrive(bars + 8 * (stages + s));
            }
#pragma unroll
            for (int c = 0; c < C; ++c) {
                if (!okv[c]) continue;
                const double2 x = v[c];
                double2 y;
                if (OP == kPermCopy) {
                    y = x;
                } else {
                    y.x = __dsub_rn(__dmul_rn(p.ar, x.x), __dmul_rn(p.ai, x.y));
                    y.y = __dadd_rn(__dmul_rn(p.ar, x.y), __dmul_rn(p.ai, x.x));
                    if (OP == kPermAccumulate) {
                        y.x = __dadd_rn(d[c].x, y.x);
                        y.y = __dadd_rn(d[c].y, y.y);
                    }
                }
                dst[outoff[j0 + c]] = y;
            }
        }
        if (k + stages < my_n) {
            mbar_wait(bars + 8 * (stages + s), ph);      // every warp has drained stage s
            issue(s);
        }
        if (++s == stages) { s = 0; ph ^= 1; }
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

cudaError_t launch_permute(const PermuteDesc &pd, cudaStream_t stream, int64_t *launches, bool dry_run)
{
    PermParams p;
    const int r = pd.rank;
    for (int d = 0; d < kMaxRank; ++d) {
        p.t[d] = 1; p.ntile[d] = 1; p.q[d] = d; p.ss[d] = 0; p.sh[d] = 0; p.mk[d] = 0; p.step[d] = 0;
        p.e[d] = d < r ? pd.extent[d] : 1;
        p.is[d] = d < r ? pd.istride[d] : 0;
        p.os[d] = d < r ? pd.ostride[d] : 0;
    }
    // dims in output order
    int q[kMaxRank];
    for (int d = 0; d < kMaxRank; ++d) q[d] = d;
    std::stable_sort(q, q + r, [&](int a, int b) { return pd.ostride[a] < pd.ostride[b]; });
    for (int d = 0; d < kMaxRank; ++d) p.q[d] = q[d];

    // Large tensors (>= 256 MB) whose output-fastest dim is long (>= 256 elements: 2-D-like transpositions such as
    // (a,b,i,j) -> (i,j,a,b)) take longer output runs and bigger tiles: >= 48 contiguous elements on the store side, ~3200
    // elements (50 KB) per tile.  Measured (profiles/r2_transpose_sweep.md): that transposition of (200,200,40,40) 5.07 ->
    // 6.0 TB/s, median of its 24 orders 5.41 -> 5.51 TB/s.  Applied to every large tensor it costs the shapes with short
    // leading extents (60^3 x 12^3: median 5.99 -> 5.68 TB/s), and the 64-76 MB shapes lose 10 % (too few tiles for 296 CTAs).
    long long total = 1;
    for (int d = 0; d < r; ++d) total *= pd.extent[d];
    const bool big = total >= (1LL << 24) && p.e[q[0]] >= env_int("TCB_PERM_BIGMIN", 256);
    const int TI = env_int("TCB_PERM_TI", 32), TO = env_int("TCB_PERM_TO", big ? 48 : 32);
    const int VOL = std::min(env_int("TCB_PERM_VOL", big ? 3200 : 2048), kMaxVol);
    // tile extent for a dim of extent e, between lo and hi: least padding first (ragged last tiles waste a CTA
    // slot), then 128-byte-aligned cuts (multiples of 8 elements: no cache line shared by two tiles), then
    // 32-byte-aligned cuts (even: no half-written sector), then the larger tile
    auto pick_tile = [](long long e, long long lo, long long hi) {
        hi = std::min(hi, e);
        lo = std::max<long long>(1, std::min(lo, hi));
        long long best = lo, best_score = -1;
        for (long long t = lo; t <= hi; ++t) {
            const long long padded = (e + t - 1) / t * t;
            const long long align = (t == e || t % 8 == 0) ? 0 : (t % 2 == 0 ? 1 : 2);
            const long long score = (padded * 4 + align) * 8192 + (8191 - t);
            if (best_score < 0 || score < best_score) { best = t; best_score = score; }
        }
        return best;
    };
    // minimal extents: >= ti contiguous elements on the input side, >= to on the output side.  A short leading
    // dim (<= twice the need: occupied indices) is taken whole rather than cut into two short runs; otherwise
    // the cut is picked in [need, 1.6 need] (two such sides still fit the volume target).  `plain` is the
    // fallback that always fits kMaxVol: each side spans < 2 * 32 elements.
    auto volume = [&] { long long v = 1; for (int d = 0; d < r; ++d) v *= p.t[d]; return v; };
    auto minimal = [&](int ti, int to, bool plain) {
        for (int d = 0; d < kMaxRank; ++d) p.t[d] = 1;
        for (int side = 0; side < 2; ++side) {
            const int target = side == 0 ? ti : to;
            long long prod = 1;
            for (int x = 0; x < r && prod < target; ++x) {
                const int d = side == 0 ? x : q[x];
                const long long need = (target + prod - 1) / prod;
                long long want = std::min<long long>(p.e[d], need);
                if (!plain && p.e[d] > need)
                    want = p.e[d] <= 2 * need ? p.e[d] : pick_tile(p.e[d], need, x == 0 ? (8 * need + 4) / 5 : 2 * need - 1);
                p.t[d] = (int)std::max<long long>(p.t[d], want);
                prod *= p.t[d];
            }
        }
    };
    minimal(TI, TO, false);
    if (volume() > kMaxVol) minimal(std::min(TI, 32), std::min(TO, 32), true);
    // grow (input-leading dims first: longer runs on both sides when dim 0 leads both) up to the volume target,
    // never beyond it
    for (int d = 0; d < r && volume() < VOL; ++d) {
        const long long others = volume() / p.t[d];
        const long long room = std::min<long long>(VOL / others, p.e[d]);
        if (room > p.t[d]) p.t[d] = (int)pick_tile(p.e[d], p.t[d], room);
        if (p.t[d] < p.e[d]) break;          // a partial dim ends the contiguous run: further dims add rows, not run length
    }
    for (int d = 0; d < r; ++d) p.ntile[d] = (int)((p.e[d] + p.t[d] - 1) / p.t[d]);
    if (volume() > kMaxVol) return cudaErrorNotSupported;
    p.vol = (int)volume();
    p.rows = p.vol / p.t[0];
    p.ntiles = 1;
    for (int d = 0; d < r; ++d) p.ntiles *= p.ntile[d];
    // shared-memory strides in input order; the output-fastest dim gets an odd stride
    int s = 1;
    for (int d = 0; d < r; ++d) {
        if (d == q[0] && d != 0 && (s % 2 == 0)) s += 1;
        p.ss[d] = s;
        s *= p.t[d];
    }
    p.tile_bytes = (int)(((size_t)s * sizeof(double2) + 127) / 128 * 128);
    // ring depth and CTAs per SM: ~200 KB of shared memory per SM, 2..4 stages per CTA
    int ctas_per_sm = std::max(1, std::min(4, env_int("TCB_PERM_CTAS", 2)));
    if (p.vol > 8 * PT) ctas_per_sm = 1;      // the J = 16 instantiation is compiled for one CTA per SM (registers)
    while (ctas_per_sm > 1 && 2 * p.tile_bytes > 200 * 1024 / ctas_per_sm - 128) --ctas_per_sm;
    const int budget = 200 * 1024 / ctas_per_sm - 128;
    // measured (r1c sweep): 2 stages beat 3-4 on every shape from 324 MB up (medians 4.9 -> 5.3, 5.2 -> 5.55, 5.6 -> 6.0 TB/s):
    // one tile in flight per CTA is enough with two CTAs per SM, and the shared memory not taken stays L1
    p.stages = std::max(2, std::min(env_int("TCB_PERM_STAGES", 2), budget / p.tile_bytes));
    const size_t smem = (size_t)p.stages * p.tile_bytes + 128;
    if (smem > 227 * 1024) return cudaErrorNotSupported;
    p.in = (const double2 *)pd.in;
    p.out = (double2 *)pd.out;
    p.ar = pd.alpha_re; p.ai = pd.alpha_im;

    const int J = (p.vol + PT - 1) / PT;
    const int blocks = (int)std::min<long long>(p.ntiles, (long long)sm_count() * ctas_per_sm);
    {   // mixed-radix digits of the grid size
        long long g = blocks;
        for (int d = 0; d < kMaxRank; ++d) { p.step[d] = (int)(g % p.ntile[d]); g /= p.ntile[d]; }
    }
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
    if (bit > kIdxBits || s >= (1 << (32 - kIdxBits))) return cudaErrorNotSupported;
    if (dry_run) return cudaSuccess;          // every check that can refuse the shape has passed; nothing is launched
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
