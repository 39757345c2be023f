// zgemm.cu -- S4 + S5: complex FP64 GEMM on the FP64 tensor cores with the permute-and-accumulate epilogue.
//
//   C[m,n] = sum_k A[m,k] B[k,n]     ("Use GEMM to execute the contraction")
//   D[offM[m] + offN[n]] (+)= alpha * C[m,n]   ("Transpose result array to obtain C", PAPER.md:91 -- done
//                                               here as a scatter through offset tables, no extra pass)
//
// B200 facts this design rests on (measured, profiles/r1b_fp64_peak.md): tcgen05 has no FP64 kind, the
// native FP64 tensor op is SASS DMMA.8x8x4 (mma.sync.m8n8k4.f64): one per 16 cycles per SM sub-partition =
// 128 flop/clk/SM = 37.0 TFLOP/s; its latency (~26 cycles) needs >= 2 independent accumulators per
// sub-partition.  The pipe is slow relative to shared memory (one 32x32 complex warp tile needs 8 LDS.128
// per 64 DMMA = 1024 cycles), so the kernel is built around keeping DMMA issuing, not around operand
// bandwidth:
//   * CTA tile 64x64 complex, 4 warps, warp tile 32x32 complex = 32 independent DMMA accumulator pairs
//     (128 accumulator registers per lane); 2 CTAs per SM (2 x 128 threads x 255 regs = the register file),
//     so one CTA's epilogue (global stores) overlaps the other CTA's main loop on the same tensor pipe.
//   * operands staged by TMA (cp.async.bulk.tensor.2d, SASS UTMALDG) into a 4-stage mbarrier ring,
//     BK = 8 complex = one 128-byte swizzle row; OOB (M, N, K tails) is zero-filled by the tensor map.
//   * shared layout = 1 KB atoms of 8x8 complex under SWIZZLE_128B.  The DMMA fragment row r (= lane>>2)
//     is mapped to row (r>>1) + 4*(r&1) of the atom: with that map every quarter-warp of an LDS.128 hits 8
//     distinct 16-byte bank groups for both operand layouts (K-major: chunk = k ^ row; M-major: chunk =
//     row ^ k), i.e. fragment loads are bank-conflict free without padding.
//   * complex product = 4 real DMMAs: Cr += Ar*Br; Cr += (-Ai)*Bi; Ci += Ar*Bi; Ci += Ai*Br  (the sign flip
//     is an exact XOR on the high word).
//   * persistent grid (2 CTAs per SM) with a stream-K schedule: whole tiles one CTA each while they fill the grid, the
//     remainder wave -- or everything, for skinny M x N with long K -- cut along K into chunks whose raw accumulator
//     fragments go to a workspace; zgemm_fixup_kernel (32 CTAs per cut tile) sums a tile's chunks in k order
//     (deterministic, no atomics on data) and applies the same scatter.  Tiles and chunks are claimed from two counters
//     (dynamic deal).  Summing inside the main kernel -- the CTA that delivers a tile's last chunk does it -- was built
//     and measured in round 2: one launch fewer, but 10 registers more in the main loop and a serial tail: 1600^3
//     0.965 -> 1.067 ms, configs[0] 33 -> 50 us (profiles/r2_gemm_ab.md); not kept.
//   * the producer (thread 0) walks the CTA's segment list 4 k-tiles ahead of the consumers and ACROSS tile
//     boundaries; segments reach the other warps through a small shared-memory queue.
//   * no tensor work on padding: the 8-wide blocks of M and N are dealt to the tiles in pairs, a warp multiplies only
//     the blocks it has (mma_ktile<MC, NC, KS>), the last k-tile of a K with <= 4 entries left does one k-step.
//   * epilogue: '+=' is two red.global.add.f64 per element (the add happens in L2, the SM never waits for D; every
//     element is touched by one thread, so the sum stays deterministic); no FP64 multiplies for alpha = 1 (the plain
//     FP64 pipe shares its datapath with DMMA).
//   * permutation-free operand loads (BSMTC / GETT): an operand that is not matrix-shaped
//     in memory is NOT copied into a workspace first.  A tensor's element offset is a sum over its indices, so any
//     operand is a matrix with a row table and a column table, A[m,k] = L[rowA[m] + colA[k]]; all 128 threads fetch
//     their share of the k-tile with 16-byte cp.async (LDGSTS, zero-fill for the tails) straight into the same swizzled
//     atoms the TMA path fills, completion counted on the same mbarrier (cp.async.mbarrier.arrive.noinc), so the
//     consumer side does not know the difference.  Lanes run along whichever of m / k is contiguous in memory.
// Measured history and the ncu evidence for each of these: DESIGN.md 6.2, profiles/r1b_zgemm_ncu_full.md.
#include "kernels.h"
#include "ptx.cuh"

#include <algorithm>
#include <cstdlib>
#include <cstring>
#include <mutex>

namespace tcb {

namespace {

using namespace ptx;

constexpr int BM = kGemmBM, BN = kGemmBN, BK = kGemmBK;
constexpr int STAGES = 4;
constexpr int A_BYTES = BM * BK * 16;   // 8 KB
constexpr int B_BYTES = BN * BK * 16;   // 8 KB
constexpr int STAGE_BYTES = A_BYTES + B_BYTES;
constexpr int kGatherAhead = 2;         // k-tiles a gathered operand is fetched ahead (its refill never waits for the
                                        // stage the CTA is still draining: no CTA-wide lock step per k-tile)
constexpr int kStages3M = 4;            // ring depth of the 3M kernel (24 KB stages)
constexpr int kQueue = 16;              // segment queue entries (producer is <= stages + 1 segments ahead)
constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + 1024 /*alignment slack*/ + 128 /*barriers*/ + 512 /*segment queue*/;
constexpr int SMEM_BYTES_3M = kStages3M * 24 * 1024 + 1024 + 128 + 512;   // 16-deep stages: 2 x 6 blocks x 2 KB
constexpr int NTHREADS = 128;

struct GemmParams {
    long long M, N, K;
    int mblocks, nblocks;          // ceil(M / 8), ceil(N / 8): the 8-row / 8-column DMMA blocks
    int mpair_base, mpair_extra;   // block pairs per M tile: base, and one more for the first `extra` tiles
    int npair_base, npair_extra;
    int mt, nt, gn;                // tile grid, column-group width of the tile order
    int ktiles, klast_steps;       // ceil(K / BK); k-steps of 4 in the last k-tile (1 or 2)
    long long dp_tiles;            // tiles [0, dp_tiles) are computed whole, tile c + w * grid by CTA c
    long long sk_tiles;            // tiles [dp_tiles, dp_tiles + sk_tiles): their (tile, k-tile) iterations are cut
    long long sk_chunks;           //   into sk_chunks chunks of sk_q iterations; chunk ch belongs to CTA ch % grid
    int sk_q, sk_slots;            // a chunk touches <= sk_slots tiles; partial slot = ch * sk_slots + ordinal
    double2 *D;
    const long long *offM;
    const long long *offN;
    double alpha_re, alpha_im;
    int accumulate, use_red;
    double2 *partial;              // [slot][32][128] raw accumulator fragments
    unsigned long long *counters;  // [3] whole tiles claimed, stream-K chunks claimed, CTAs done; zero at launch; null: static deal
    // gathered operands (mode kGather): X[row, k] = base[rowtab[row] + ktab[k]]
    const double2 *gA, *gB;
    const long long *gAm, *gAk, *gBn, *gBk;
    int a_mfast, b_mfast;          // lanes run along the rows (the operand's unit-stride index is free) or along k
};
enum { kTmaK = 0, kTmaM = 1, kGather = 2 };   // how an operand reaches shared memory


__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap *tm, int c0, int c1, uint32_t bar)
{
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
        ::"r"(dst), "l"(tm), "r"(c0), "r"(c1), "r"(bar)
        : "memory");
}
// 16-byte asynchronous copy global -> shared (LDGSTS), src_bytes = 0 writes zeros (tails)
__device__ __forceinline__ void cp_async16(uint32_t dst, const void *src, int src_bytes)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(src_bytes) : "memory");
}
// the mbarrier receives one arrival when all cp.async issued so far by this thread have landed
__device__ __forceinline__ void cp_async_arrive(uint32_t bar)
{
    asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(bar) : "memory");
}
// rows [row0, row0 + rows_in_tile) x k-tile k0 of a gathered operand into a stage, K-major atoms: element (m, k) of the
// tile at (m >> 3) * 1024 + (m & 7) * 128 + ((k ^ (m & 7)) * 16) -- the layout a SWIZZLE_128B K-major TMA box produces
__device__ __forceinline__ void gather_ktile(uint32_t sX, const double2 *base, const long long *rowtab, long long row0,
                                             int rows_in_tile, long long rows_total, const long long *ktab, long long k0,
                                             long long K, bool mfast, int tid)
{
    if (mfast) {
        const int m = tid & 63;
        if (m >= rows_in_tile) return;
        const bool rok = row0 + m < rows_total;
        const long long ro = rok ? __ldg(rowtab + row0 + m) : 0;
        const uint32_t drow = sX + (m >> 3) * 1024 + (m & 7) * 128;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int kk = (tid >> 6) + 2 * j;
            const bool ok = rok && k0 + kk < K;
            const long long ko = ok ? __ldg(ktab + k0 + kk) : 0;
            cp_async16(drow + ((kk ^ (m & 7)) * 16), base + ro + ko, ok ? 16 : 0);
        }
    } else {
        const int kk = tid & 7;
        const bool kok = k0 + kk < K;
        const long long ko = kok ? __ldg(ktab + k0 + kk) : 0;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int m = (tid >> 3) + 16 * j;
            if (m >= rows_in_tile) continue;
            const bool ok = kok && row0 + m < rows_total;
            const long long ro = ok ? __ldg(rowtab + row0 + m) : 0;
            cp_async16(sX + (m >> 3) * 1024 + (m & 7) * 128 + ((kk ^ (m & 7)) * 16), base + ro + ko, ok ? 16 : 0);
        }
    }
}
__device__ __forceinline__ void dmma(double &c0, double &c1, double a, double b)
{
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
        : "+d"(c0), "+d"(c1)
        : "d"(a), "d"(b));
}
__device__ __forceinline__ double neg_exact(double x)
{
    return __hiloint2double(__double2hiint(x) ^ 0x80000000, __double2loint(x));
}

// ---- work decomposition ("stream-K": data-parallel full waves, the remainder cut along K) ------------------
// A segment is a run of k-tiles [kb, ke) of one output tile.  slot < 0: the segment is the whole tile and the
// CTA writes D itself; otherwise its raw accumulators go to partial slot `slot` and the fix-up kernel sums the
// tile's slots in k order (fixed order: bit-reproducible, no atomics).
struct Segment {
    long long tile, slot;
    int kb, ke;
};
// With work counters the deal is dynamic: a CTA claims its next whole tile, and then its next stream-K chunk, by
// atomicAdd.  Tiles then cost what they
// cost (ragged tiles are cheaper, SMs differ in speed) and the chip still finishes together; the chunks are small
// (about three per CTA).  Which CTA computes what changes from run to run, the arithmetic does not: a tile's chunks
// are fixed k-ranges and are summed in k order.
struct SegmentIter {
    long long w, wn, ch;
    int sub, phase;
    bool ahead;                      // claim whole tiles one ahead of use (only when there are plenty)
    unsigned long long *cnt;
    __device__ __forceinline__ long long claim(int which, long long fallback)
    {
        return cnt ? (long long)atomicAdd(cnt + which, 1ULL) : fallback;
    }
    __device__ __forceinline__ void init(const GemmParams &p)
    {
        cnt = p.counters;
        // with many tiles per CTA the claim for the next tile is issued a whole tile early, and its latency never
        // shows; with few, a tile held in reserve by a busy CTA is a tile an idle CTA cannot take
        ahead = cnt && p.dp_tiles >= 8LL * gridDim.x;
        w = claim(0, blockIdx.x);
        wn = ahead ? claim(0, 0) : -1;
        ch = -1; sub = 0; phase = 0;
    }
    __device__ __forceinline__ bool next(const GemmParams &p, Segment *s)
    {
        if (phase == 0) {
            if (w < p.dp_tiles) {
                s->tile = w; s->slot = -1; s->kb = 0; s->ke = p.ktiles;
                if (ahead) { w = wn; wn = claim(0, 0); }
                else w = claim(0, w + gridDim.x);
                return true;
            }
            phase = 1;
            ch = claim(1, blockIdx.x);
        }
        const long long total = p.sk_tiles * p.ktiles;
        while (ch < p.sk_chunks) {
            const long long it0 = ch * p.sk_q, it1 = min(total, it0 + p.sk_q);
            const long long first = it0 / p.ktiles, last = (it1 - 1) / p.ktiles;
            const long long tl = first + sub;
            if (tl <= last) {
                const long long base = tl * p.ktiles;
                s->kb = (int)max(0LL, it0 - base);
                s->ke = (int)min((long long)p.ktiles, it1 - base);
                s->tile = p.dp_tiles + tl;
                s->slot = (s->kb == 0 && s->ke == p.ktiles) ? -1 : ch * p.sk_slots + sub;
                ++sub;
                return true;
            }
            ch = claim(1, ch + gridDim.x);
            sub = 0;
        }
        return false;
    }
};

// Tile order: groups of `gn` tile-columns, n fastest inside a group (concurrent CTAs form a near-square block of
// the output, so A row panels and B column panels are shared through L2).  The 8-wide DMMA blocks of M and N are
// dealt to the tiles evenly and IN PAIRS (N = 400 = 50 blocks -> 7 tiles of 8,8,8,8,6,6,6 blocks instead of six
// full tiles and a sliver), so that the two warp rows / columns of a CTA get the same number of blocks and the
// four sub-partitions' DMMA pipes carry the same load.
struct TileGeom {
    int m0, n0;          // element origin
    int mb, nb;          // blocks in this tile (<= 8 each)
};
__device__ __forceinline__ TileGeom tile_geom(const GemmParams &p, unsigned tile)
{
    const unsigned group_sz = (unsigned)p.gn * (unsigned)p.mt;
    const unsigned g = tile / group_sz, rem = tile - g * group_sz;
    const int n0t = (int)g * p.gn;
    const unsigned gw = (unsigned)min(p.gn, p.nt - n0t);
    const int tm = (int)(rem / gw), tn = n0t + (int)(rem - (rem / gw) * gw);
    // tile t of a dim owns pairs [t * base + min(t, extra), ...) -- base/extra precomputed on the host
    const int mp0 = tm * p.mpair_base + min(tm, p.mpair_extra), mp1 = mp0 + p.mpair_base + (tm < p.mpair_extra ? 1 : 0);
    const int np0 = tn * p.npair_base + min(tn, p.npair_extra), np1 = np0 + p.npair_base + (tn < p.npair_extra ? 1 : 0);
    TileGeom t;
    t.m0 = mp0 * 16; t.n0 = np0 * 16;
    t.mb = min(2 * mp1, p.mblocks) - 2 * mp0;
    t.nb = min(2 * np1, p.nblocks) - 2 * np0;
    return t;
}
// The two warp rows (columns) of a CTA split a tile's blocks ceil/floor (equal unless the last tile is odd).
struct WarpGeom {
    int moff, mcnt, noff, ncnt;      // in blocks, relative to the tile origin
};
__device__ __forceinline__ WarpGeom warp_geom(const TileGeom &t, int warp_m, int warp_n)
{
    WarpGeom w;
    const int mh = (t.mb + 1) / 2, nh = (t.nb + 1) / 2;      // blocks of warp row / column 0
    w.moff = warp_m ? mh : 0; w.mcnt = warp_m ? t.mb - mh : mh;
    w.noff = warp_n ? nh : 0; w.ncnt = warp_n ? t.nb - nh : nh;
    return w;
}

// permute-and-accumulate epilogue of one warp fragment: D[offM[m] + offN[n]] (+)= alpha * C[m, n]
__device__ __forceinline__ void store_fragment(const GemmParams &p, const double (&cr)[4][4][2],
                                               const double (&ci)[4][4][2], const TileGeom &t, const WarpGeom &w,
                                               int rowmap, int c)
{
    const long long mw = (long long)t.m0 + w.moff * 8 + rowmap;
    const long long nw = (long long)t.n0 + w.noff * 8 + c;
    long long om[4], on[4][2];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const long long m = mw + i * 8;
        om[i] = (i < w.mcnt && m < p.M) ? p.offM[m] : -1;
    }
#pragma unroll
    for (int j = 0; j < 4; ++j)
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const long long n = nw + j * 8 + h * 4;
            on[j][h] = (j < w.ncnt && n < p.N) ? p.offN[n] : -1;
        }
    // The plain FP64 pipe shares its datapath with DMMA: every DMUL/DFMA here queues behind the other resident
    // CTA's tensor work (ncu: 10 % of all stall samples of the K = 60 T3 contraction sat on the alpha multiply).
    // So the scaling does the least arithmetic alpha allows: none for alpha = 1, one FMA per component for real
    // alpha (fused with the accumulate), the full complex product only for complex alpha.
    const double ar = p.alpha_re, ai = p.alpha_im;
    const int mode = (ai != 0.0) ? 2 : (ar != 1.0 ? 1 : 0);
    if (p.accumulate && p.use_red) {
        // D += v as two red.global.add.f64 per element: the add happens in L2, the SM never waits for D.  Every element
        // of D is touched by exactly one thread of one CTA, so the sum is still deterministic.
#pragma unroll
        for (int j = 0; j < 4; ++j)
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                if (on[j][h] < 0) continue;
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    if (om[i] < 0) continue;
                    const double xr = cr[i][j][h], xi = ci[i][j][h];
                    double vx, vy;
                    if (mode == 0) { vx = xr; vy = xi; }
                    else if (mode == 1) { vx = ar * xr; vy = ar * xi; }
                    else { vx = fma(ar, xr, -ai * xi); vy = fma(ar, xi, ai * xr); }
                    double *dst = reinterpret_cast<double *>(p.D + om[i] + on[j][h]);
                    asm volatile("red.global.add.f64 [%0], %1;" ::"l"(dst), "d"(vx) : "memory");
                    asm volatile("red.global.add.f64 [%0], %1;" ::"l"(dst + 1), "d"(vy) : "memory");
                }
            }
        return;
    }
    if (p.accumulate) {            // A/B fallback (TCB_GEMM_RED=0): plain read-modify-write, one element in flight
#pragma unroll
        for (int j = 0; j < 4; ++j)
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                if (on[j][h] < 0) continue;
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    if (om[i] < 0) continue;
                    const double xr = cr[i][j][h], xi = ci[i][j][h];
                    double2 *dst = p.D + om[i] + on[j][h];
                    const double2 d = *dst;
                    double2 v;
                    if (mode == 0) v = make_double2(d.x + xr, d.y + xi);
                    else if (mode == 1) v = make_double2(fma(ar, xr, d.x), fma(ar, xi, d.y));
                    else v = make_double2(fma(ar, xr, fma(-ai, xi, d.x)), fma(ar, xi, fma(ai, xr, d.y)));
                    *dst = v;
                }
            }
        return;
    }
#pragma unroll
    for (int j = 0; j < 4; ++j)
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            if (on[j][h] < 0) continue;
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                if (om[i] < 0) continue;
                const double xr = cr[i][j][h], xi = ci[i][j][h];
                double2 v;
                if (mode == 0) v = make_double2(xr, xi);
                else if (mode == 1) v = make_double2(ar * xr, ar * xi);
                else v = make_double2(fma(ar, xr, -ai * xi), fma(ar, xi, ai * xr));
                p.D[om[i] + on[j][h]] = v;
            }
        }
}

// one k-tile (two k-steps of 4) of a warp tile of MC x NC blocks: complex product = 4 real DMMAs per block pair
// (KS = 1: the last k-tile of a K with <= 4 valid entries in it).  Straight-line code: a run-time test on the
// k-step would end the basic block and keep the second step's LDS from being hoisted over the first step's DMMAs.
template <int MC, int NC, int KS>
__device__ __forceinline__ void mma_ktile(double (&cr)[4][4][2], double (&ci)[4][4][2], uint32_t sA, uint32_t sB,
                                          const uint32_t (&offA)[4], const uint32_t (&offB)[4])
{
#pragma unroll
    for (int ks = 0; ks < KS; ++ks) {
        {
            double2 a[MC], b[NC];
#pragma unroll
            for (int i = 0; i < MC; ++i) a[i] = lds128(sA + i * 1024 + offA[ks]);
#pragma unroll
            for (int j = 0; j < NC; ++j) b[j] = lds128(sB + j * 1024 + offB[ks]);
#pragma unroll
            for (int i = 0; i < MC; ++i) {
                const double nai = neg_exact(a[i].y);
#pragma unroll
                for (int j = 0; j < NC; ++j) {
                    dmma(cr[i][j][0], cr[i][j][1], a[i].x, b[j].x);
                    dmma(ci[i][j][0], ci[i][j][1], a[i].x, b[j].y);
                    dmma(cr[i][j][0], cr[i][j][1], nai, b[j].y);
                    dmma(ci[i][j][0], ci[i][j][1], a[i].y, b[j].x);
                }
            }
        }
    }
}

// The same k-tile with THREE real products per complex product (the "3M" scheme of xGEMM3M):
//     P1 = Ar Br,  P2 = Ai Bi,  P3 = (Ar + Ai)(Br + Bi);      Re C = P1 - P2,  Im C = P3 - P1 - P2
// 3 DMMAs per block pair and k-step instead of 4, three accumulator sets instead of two -- which is why a warp holds at most
// 3 x 3 blocks here (108 accumulator registers; 4 x 4 would need 192 of the 255).  The operand sums cost MC + NC DADDs per
// k-step on the pipe DMMA runs on (6 against 27 DMMAs of 16 issue slots each).
template <int MC, int NC, int KS, int BLKA, int BLKB>
__device__ __forceinline__ void mma_ktile3(double (&p1)[3][3][2], double (&p2)[3][3][2], double (&p3)[3][3][2], uint32_t sA,
                                           uint32_t sB, const uint32_t (&offA)[4], const uint32_t (&offB)[4])
{
#pragma unroll
    for (int ks = 0; ks < KS; ++ks) {
        double2 a[MC], b[NC];
        double as[MC], bs[NC];
#pragma unroll
        for (int i = 0; i < MC; ++i) a[i] = lds128(sA + i * BLKA + offA[ks]);
#pragma unroll
        for (int j = 0; j < NC; ++j) b[j] = lds128(sB + j * BLKB + offB[ks]);
#pragma unroll
        for (int i = 0; i < MC; ++i) as[i] = __dadd_rn(a[i].x, a[i].y);
#pragma unroll
        for (int j = 0; j < NC; ++j) bs[j] = __dadd_rn(b[j].x, b[j].y);
#pragma unroll
        for (int i = 0; i < MC; ++i)
#pragma unroll
            for (int j = 0; j < NC; ++j) {
                dmma(p1[i][j][0], p1[i][j][1], a[i].x, b[j].x);
                dmma(p2[i][j][0], p2[i][j][1], a[i].y, b[j].y);
                dmma(p3[i][j][0], p3[i][j][1], as[i], bs[j]);
            }
    }
}
// the last k-tile of a K that does not fill it: 1 ... 3 k-steps, once per tile -- a plain loop
template <int MC, int NC, int BLKA, int BLKB>
__device__ __forceinline__ void mma_ktile3_tail(double (&p1)[3][3][2], double (&p2)[3][3][2], double (&p3)[3][3][2],
                                                uint32_t sA, uint32_t sB, const uint32_t (&offA)[4],
                                                const uint32_t (&offB)[4], int nks)
{
    uint32_t oa[4] = {offA[0], offA[1], offA[2], offA[3]}, ob[4] = {offB[0], offB[1], offB[2], offB[3]};
#pragma unroll 1
    for (int ks = 0; ks < nks; ++ks) {
        const uint32_t one_a[4] = {oa[0], 0, 0, 0}, one_b[4] = {ob[0], 0, 0, 0};
        mma_ktile3<MC, NC, 1, BLKA, BLKB>(p1, p2, p3, sA, sB, one_a, one_b);
        oa[0] = oa[1]; oa[1] = oa[2]; oa[2] = oa[3];
        ob[0] = ob[1]; ob[1] = ob[2]; ob[2] = ob[3];
    }
}

template <int AMODE, int BMODE, bool M3>
__global__ void __launch_bounds__(NTHREADS, 2)
zgemm_dmma_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB,
                  const __grid_constant__ GemmParams p)
{
    constexpr bool kAnyTma = AMODE != kGather || BMODE != kGather;
    constexpr bool kAnyGather = AMODE == kGather || BMODE == kGather;
    constexpr int TB = M3 ? 6 : 8;                       // 8 x 8 blocks per tile dimension at most (3M: 48 x 48 tiles)
    // ring: 4 stages of 16 KB; 3M: 4 stages of 24 KB (with 8-deep stages, 8 stages of 12 KB measured the same as 4: 491.7
    // against 493 ms on configs[2], and the same 1.1 TB of DRAM reads -- see profiles/r2_gemm_3m.md)
    constexpr int NST = M3 ? kStages3M : STAGES;
    // k-values per stage: 8; 3M: 16 (two 128-byte swizzle rows).  A 3M k-step is 27 DMMAs per warp instead of 64, so with 8-deep
    // stages the per-stage cost (barrier wait and arrive, refill, queue) weighed twice as much: DMMA pipe 84 % busy on
    // configs[2] against 95 % for 4M.  An M-major atom becomes one 16 x 8 box of 2 KB: half the TMA requests per flop.
    constexpr int KB = M3 ? 16 : 8, KH = KB / 8;
    constexpr int kAOff = TB * 1024 * KH, kStageBytes = 2 * kAOff;
    constexpr int kBlkA = AMODE == kTmaM ? 1024 * KH : 1024, kBlkB = BMODE == kTmaM ? 1024 * KH : 1024;   // 8-row block stride
    // An M-major operand takes one TMA per 8 x 8 atom (6 per operand and k-tile).  With 3M a k-tile is 27 DMMAs per k-step
    // instead of 64, and thread 0 issuing 12 UTMALDG per k-tile held its warp back (4500^3 M-major: 38 against 41 TFLOP/s
    // K-major).  So lane 0 of EVERY warp issues the atoms j = warp, warp + 4 of the k-tile, following thread 0's cursor
    // through the published segment list; thread 0 alone posts the byte count (a stage's barrier completes when its one
    // arrival is in and the bytes of all four issuers have landed, in whichever order).
    constexpr bool kSplitIssue = M3 && (AMODE == kTmaM || BMODE == kTmaM);
    constexpr int kIssuers = kSplitIssue ? NTHREADS / 32 : 1;
    constexpr uint32_t kTmaBytes = (AMODE != kGather ? TB * 1024 * (M3 ? 2 : 1) : 0) + (BMODE != kGather ? TB * 1024 * (M3 ? 2 : 1) : 0);
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t bar_base = smem_base + NST * kStageBytes;   // full[s] at +8s, empty[s] at +8(NST+s)

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int warp_m = warp & 1, warp_n = warp >> 1;

    if (tid == 0) {
        for (int s = 0; s < NST; ++s) {
            // full: thread 0's expect_tx arrival for the TMA part + one cp.async arrival per thread for the gathered part
            mbar_init(bar_base + 8 * s, (kAnyTma ? 1 : 0) + (kAnyGather ? NTHREADS : 0));
            mbar_init(bar_base + 8 * (NST + s), NTHREADS / 32);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        if (AMODE != kGather) asm volatile("prefetch.tensormap [%0];" ::"l"(&tmA) : "memory");
        if (BMODE != kGather) asm volatile("prefetch.tensormap [%0];" ::"l"(&tmB) : "memory");
        *reinterpret_cast<volatile int *>(smem_raw + (bar_base - smem_u32(smem_raw)) + 128 + kQueue * sizeof(Segment)) = 0;
    }
    __syncthreads();

    // ---- producer (thread 0): walks the same segment list, NST k-tiles ahead of the consumers, ACROSS tile
    // boundaries -- the next tile's operands are already in flight while this tile's epilogue stores drain
    SegmentIter pit;
    Segment pseg;
    int pk = 0, pm0 = 0, pn0 = 0;
    bool pvalid = false;
    int pstage = 0;
    uint32_t pphase = 0;                // parity of the ring round the producer is filling
    // segment queue: the producer decides (or claims) what this CTA computes and publishes every segment here
    // before its first operand load; the consumers pop them in order.  kQueue > NST + 1 entries suffice.
    Segment *q_seg = reinterpret_cast<Segment *>(smem_raw + (bar_base - smem_u32(smem_raw)) + 128);
    volatile int *q_pub = reinterpret_cast<volatile int *>(q_seg + kQueue);
    int npub = 0;
    auto producer_advance = [&]() {
        pvalid = pit.next(p, &pseg);
        Segment out = pseg;
        if (!pvalid) out.tile = -1;                 // terminator
        q_seg[npub % kQueue] = out;
        __threadfence_block();
        *q_pub = ++npub;
        if (pvalid) {
            const TileGeom t = tile_geom(p, (unsigned)pseg.tile);
            pm0 = t.m0; pn0 = t.n0; pk = pseg.kb;
        }
    };
    auto issue = [&]() {              // loads k-tile pk of the producer's segment into stage pstage (TMA operands)
        if (kAnyTma) {
            const uint32_t bar = bar_base + 8 * pstage;
            const uint32_t sA = smem_base + pstage * kStageBytes, sB = sA + kAOff;
            const int k0 = pk * KB;
            mbar_expect_tx(bar, kTmaBytes);
            if (AMODE == kTmaK) {
#pragma unroll
                for (int h = 0; h < KH; ++h) tma_load_2d(sA + h * TB * 1024, &tmA, 2 * (k0 + 8 * h), pm0, bar);
            } else if (AMODE == kTmaM) {
#pragma unroll
                for (int j = 0; j < TB; j += kIssuers) tma_load_2d(sA + j * kBlkA, &tmA, 2 * (pm0 + 8 * j), k0, bar);
            }
            if (BMODE == kTmaK) {
#pragma unroll
                for (int h = 0; h < KH; ++h) tma_load_2d(sB + h * TB * 1024, &tmB, 2 * (k0 + 8 * h), pn0, bar);
            } else if (BMODE == kTmaM) {
#pragma unroll
                for (int j = 0; j < TB; j += kIssuers) tma_load_2d(sB + j * kBlkB, &tmB, 2 * (pn0 + 8 * j), k0, bar);
            }
        }
        if (++pstage == NST) { pstage = 0; pphase ^= 1; }
        if (++pk == pseg.ke) producer_advance();
    };
    // ---- gathered operands: EVERY thread walks the published segment list with its own cursor, in step with thread 0's,
    // and fetches its share (4 x 16 bytes per operand and k-tile) of the same k-tile into the same stage
    int gq = 0, gk = 0, gke = 0, gstage = 0, gm0 = 0, gn0 = 0, gmr = 0, gnr = 0;
    uint32_t gphase = 0;
    bool gvalid = false;
    auto gather_enter = [&]() {       // moves the cursor into published segment gq
        while (*q_pub <= gq) { }
        __threadfence_block();
        const Segment sg = q_seg[gq % kQueue];
        gvalid = sg.tile >= 0;
        if (gvalid) {
            const TileGeom t = tile_geom(p, (unsigned)sg.tile);
            gm0 = t.m0; gn0 = t.n0; gmr = t.mb * 8; gnr = t.nb * 8;
            gk = sg.kb; gke = sg.ke;
        }
    };
    auto gather_issue = [&]() {
        const uint32_t sA = smem_base + gstage * kStageBytes, sB = sA + kAOff;
        const long long k0 = (long long)gk * KB;
#pragma unroll
        for (int h = 0; h < KH; ++h) {
            if (AMODE == kGather)
                gather_ktile(sA + h * TB * 1024, p.gA, p.gAm, gm0, gmr, p.M, p.gAk, k0 + 8 * h, p.K, p.a_mfast != 0, tid);
            if (BMODE == kGather)
                gather_ktile(sB + h * TB * 1024, p.gB, p.gBn, gn0, gnr, p.N, p.gBk, k0 + 8 * h, p.K, p.b_mfast != 0, tid);
        }
        cp_async_arrive(bar_base + 8 * gstage);
        if (++gstage == NST) { gstage = 0; gphase ^= 1; }
        if (++gk == gke) { ++gq; gather_enter(); }
    };
    int tq = 0, tk = 0, tke = 0, tstage = 0, tm0 = 0, tn0 = 0;
    uint32_t tphase = 0;
    bool tvalid = false;
    auto follow_enter = [&]() {
        while (*q_pub <= tq) { }
        __threadfence_block();
        const Segment sg = q_seg[tq % kQueue];
        tvalid = sg.tile >= 0;
        if (tvalid) {
            const TileGeom t = tile_geom(p, (unsigned)sg.tile);
            tm0 = t.m0; tn0 = t.n0; tk = sg.kb; tke = sg.ke;
        }
    };
    auto follow_issue = [&]() {       // this warp's atoms of k-tile tk, into the stage thread 0 fills with the same k-tile
        const uint32_t bar = bar_base + 8 * tstage;
        const uint32_t sA = smem_base + tstage * kStageBytes, sB = sA + kAOff;
        const int k0 = tk * KB;
        if (AMODE == kTmaM) {
#pragma unroll
            for (int j = 0; j < TB; ++j)
                if (j % kIssuers == warp) tma_load_2d(sA + j * kBlkA, &tmA, 2 * (tm0 + 8 * j), k0, bar);
        }
        if (BMODE == kTmaM) {
#pragma unroll
            for (int j = 0; j < TB; ++j)
                if (j % kIssuers == warp) tma_load_2d(sB + j * kBlkB, &tmB, 2 * (tn0 + 8 * j), k0, bar);
        }
        if (++tstage == NST) { tstage = 0; tphase ^= 1; }
        if (++tk == tke) { ++tq; follow_enter(); }
    };
    if (tid == 0) {
        pit.init(p);
        producer_advance();
        for (int s = 0; s < NST && pvalid; ++s) issue();
    }
    if (kSplitIssue && lane == 0 && warp != 0) {
        follow_enter();
        for (int s = 0; s < NST && tvalid; ++s) follow_issue();
    }
    if (kAnyGather) {
        gather_enter();
        for (int s = 0; s < kGatherAhead && gvalid; ++s) gather_issue();
    }

    // per-lane fragment offsets inside a 1 KB atom, for the two k-steps of a stage
    const int r = lane >> 2, c = lane & 3;
    const int rowmap = (r >> 1) + 4 * (r & 1);
    uint32_t offA[4], offB[4];
#pragma unroll
    for (int ks = 0; ks < 4; ++ks) {
        const int k = ks * 4 + c, kk = k & 7, h = k >> 3;       // 4M: ks < 2, h = 0
        offA[ks] = AMODE != kTmaM ? (h * TB * 1024 + rowmap * 128 + ((kk ^ rowmap) * 16)) : (k * 128 + ((rowmap ^ kk) * 16));
        offB[ks] = BMODE != kTmaM ? (h * TB * 1024 + rowmap * 128 + ((kk ^ rowmap) * 16)) : (k * 128 + ((rowmap ^ kk) * 16));
    }

    Segment seg;
    int npop = 0;
    int stage = 0;
    uint32_t phase = 0;
    long long done = 0;                 // k-tiles consumed by this CTA so far
    for (;;) {
        while (*q_pub <= npop) { }
        __threadfence_block();
        seg = q_seg[npop % kQueue];
        ++npop;
        if (seg.tile < 0) break;
        const TileGeom tg = tile_geom(p, (unsigned)seg.tile);
        const WarpGeom wg = warp_geom(tg, warp_m, warp_n);

        const bool shape44 = wg.mcnt == 4 && wg.ncnt == 4, shape43 = wg.mcnt == 4 && wg.ncnt == 3;
        const bool shape34 = wg.mcnt == 3 && wg.ncnt == 4, shape33 = wg.mcnt == 3 && wg.ncnt == 3;
        const bool shape32 = wg.mcnt == 3 && wg.ncnt == 2, shape23 = wg.mcnt == 2 && wg.ncnt == 3;
        double cr[4][4][2], ci[4][4][2];
        double p1[3][3][2], p2[3][3][2], p3[3][3][2];      // 3M only (dead otherwise)
        if (!M3) {
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    cr[i][j][0] = cr[i][j][1] = 0.0;
                    ci[i][j][0] = ci[i][j][1] = 0.0;
                }
        } else {
#pragma unroll
            for (int i = 0; i < 3; ++i)
#pragma unroll
                for (int j = 0; j < 3; ++j)
#pragma unroll
                    for (int h = 0; h < 2; ++h) p1[i][j][h] = p2[i][j][h] = p3[i][j][h] = 0.0;
        }

        for (int kt = seg.kb; kt < seg.ke; ++kt, ++done) {
            if (tid == 0 && done >= 1 && pvalid) {
                // refill the stage consumed in the previous iteration (the other warps had a whole k-tile to
                // release it).  A non-blocking variant (mbarrier.test_wait, refill whatever is free) measured 7 %
                // slower: the wait keeps the four warps of a CTA in step, which the shared DMMA pipe prefers.
                mbar_wait(bar_base + 8 * (NST + pstage), pphase ^ 1);
                issue();
            }
            if (kSplitIssue && lane == 0 && warp != 0 && done >= 1 && tvalid) {
                mbar_wait(bar_base + 8 * (NST + tstage), tphase ^ 1);
                follow_issue();
            }
            if (kAnyGather && gvalid) {
                // the gathered part of k-tile done + kGatherAhead goes into the stage that was consumed NST - kGatherAhead
                // iterations ago: every thread checks that all four warps have left it (they have, unless one lags two
                // k-tiles; a fresh barrier passes the parity test at once)
                mbar_wait(bar_base + 8 * (NST + gstage), gphase ^ 1);
                gather_issue();
            }
            mbar_wait(bar_base + 8 * stage, phase);
            const uint32_t sA = smem_base + stage * kStageBytes + wg.moff * kBlkA;
            const uint32_t sB = smem_base + stage * kStageBytes + kAOff + wg.noff * kBlkB;
            const int nks = (kt == p.ktiles - 1) ? p.klast_steps : 2 * KH;
            // The common warp shapes are tested directly, per segment flags: the jump table's indirect branch (BRX)
            // per k-tile cost 3 % of the pipe on full tiles (90.7 -> 93.4 % at 6400 x 512 x 6400).
            if (!M3) {
            if (nks == 2 && shape44) mma_ktile<4, 4, 2>(cr, ci, sA, sB, offA, offB);
            else if (nks == 2 && shape43) mma_ktile<4, 3, 2>(cr, ci, sA, sB, offA, offB);
            else if (nks == 2 && shape34) mma_ktile<3, 4, 2>(cr, ci, sA, sB, offA, offB);
            else if (nks == 2 && shape33) mma_ktile<3, 3, 2>(cr, ci, sA, sB, offA, offB);
            else
            switch (wg.mcnt * 5 + wg.ncnt) {      // only the blocks that exist are multiplied (no tensor work on padding)
#define TCB_CASE(MC, NC) case MC * 5 + NC:                                              \
    if (nks == 2) mma_ktile<MC, NC, 2>(cr, ci, sA, sB, offA, offB);                        \
    else mma_ktile<MC, NC, 1>(cr, ci, sA, sB, offA, offB);                                 \
    break;
                TCB_CASE(4, 4) TCB_CASE(4, 3) TCB_CASE(4, 2) TCB_CASE(4, 1)
                TCB_CASE(3, 4) TCB_CASE(3, 3) TCB_CASE(3, 2) TCB_CASE(3, 1)
                TCB_CASE(2, 4) TCB_CASE(2, 3) TCB_CASE(2, 2) TCB_CASE(2, 1)
                TCB_CASE(1, 4) TCB_CASE(1, 3) TCB_CASE(1, 2) TCB_CASE(1, 1)
#undef TCB_CASE
                default: break;                   // a warp without blocks only keeps the barriers moving
            }
            } else {
            if (nks == 4 && shape33) mma_ktile3<3, 3, 4, kBlkA, kBlkB>(p1, p2, p3, sA, sB, offA, offB);
            else if (nks == 4 && shape32) mma_ktile3<3, 2, 4, kBlkA, kBlkB>(p1, p2, p3, sA, sB, offA, offB);
            else if (nks == 4 && shape23) mma_ktile3<2, 3, 4, kBlkA, kBlkB>(p1, p2, p3, sA, sB, offA, offB);
            else
            switch (wg.mcnt * 5 + wg.ncnt) {
#define TCB_CASE(MC, NC) case MC * 5 + NC:                                              \
    if (nks == 4) mma_ktile3<MC, NC, 4, kBlkA, kBlkB>(p1, p2, p3, sA, sB, offA, offB);     \
    else mma_ktile3_tail<MC, NC, kBlkA, kBlkB>(p1, p2, p3, sA, sB, offA, offB, nks);       \
    break;
                TCB_CASE(3, 3) TCB_CASE(3, 2) TCB_CASE(3, 1)
                TCB_CASE(2, 3) TCB_CASE(2, 2) TCB_CASE(2, 1)
                TCB_CASE(1, 3) TCB_CASE(1, 2) TCB_CASE(1, 1)
#undef TCB_CASE
                default: break;
            }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(bar_base + 8 * (NST + stage));
            if (++stage == NST) { stage = 0; phase ^= 1; }
        }

        if (M3) {                               // Re C = P1 - P2, Im C = P3 - P1 - P2
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j)
#pragma unroll
                    for (int h = 0; h < 2; ++h) {
                        if (i < 3 && j < 3) {
                            cr[i][j][h] = __dsub_rn(p1[i][j][h], p2[i][j][h]);
                            ci[i][j][h] = __dsub_rn(p3[i][j][h], __dadd_rn(p1[i][j][h], p2[i][j][h]));
                        } else {
                            cr[i][j][h] = 0.0;
                            ci[i][j][h] = 0.0;
                        }
                    }
        }
        // ---- epilogue: lane holds C[m = block i, row rowmap][n = block j, column c (+4)] of its warp's blocks -----
        if (seg.slot < 0) {
            store_fragment(p, cr, ci, tg, wg, rowmap, c);
        } else {
            double2 *P = p.partial + seg.slot * (32LL * NTHREADS) + tid;
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j)
#pragma unroll
                    for (int h = 0; h < 2; ++h)
                        if (i < wg.mcnt && j < wg.ncnt)
                            P[((i * 4 + j) * 2 + h) * NTHREADS] = make_double2(cr[i][j][h], ci[i][j][h]);
        }
    }
    // counters[2] counts the CTAs that are done claiming; the last one leaves all three at zero for the next launch
    // (no memset node between contractions)
    if (tid == 0 && p.counters) {
        __threadfence();
        if (atomicAdd(p.counters + 2, 1ULL) == gridDim.x - 1) {
            p.counters[0] = 0; p.counters[1] = 0; p.counters[2] = 0;
            __threadfence();
        }
    }
}

// fix-up of the tiles that were cut along K into MANY chunks (skinny M x N, long K: one tile, a chunk per CTA): sums the
// tile's partial fragments in k order (deterministic) and applies the same permute-and-accumulate epilogue.
// grid = (stream-K tiles, 32): CTA y owns fragment entry (i, j, h) = (y >> 3, (y >> 1) & 3, y & 1) of every warp, one element
// per thread, same thread <-> element map as the main kernel; eight chunk loads in flight, additions in chunk order.
__global__ void __launch_bounds__(NTHREADS) zgemm_fixup_kernel(const __grid_constant__ GemmParams p)
{
    const long long tl = blockIdx.x;
    const long long base = tl * p.ktiles;
    const long long ch_lo = base / p.sk_q, ch_hi = (base + p.ktiles - 1) / p.sk_q;
    if (ch_lo == ch_hi) return;                       // computed whole by one CTA, already in D
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int i = blockIdx.y >> 3, j = (blockIdx.y >> 1) & 3, h = blockIdx.y & 1;
    const TileGeom tg = tile_geom(p, (unsigned)(p.dp_tiles + tl));
    const WarpGeom wg = warp_geom(tg, warp & 1, warp >> 1);
    if (i >= wg.mcnt || j >= wg.ncnt) return;
    const int r = lane >> 2, c = lane & 3;
    const int rowmap = (r >> 1) + 4 * (r & 1);
    const long long m = (long long)tg.m0 + wg.moff * 8 + rowmap + i * 8;
    const long long n = (long long)tg.n0 + wg.noff * 8 + c + j * 8 + h * 4;
    if (m >= p.M || n >= p.N) return;
    const long long entry = (long long)((i * 4 + j) * 2 + h) * NTHREADS + tid;
    double sr = 0.0, si = 0.0;
    for (long long ch0 = ch_lo; ch0 <= ch_hi; ch0 += 8) {
        double2 v[8];
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const long long ch = ch0 + u;
            if (ch <= ch_hi) {
                const long long first = (ch * p.sk_q) / p.ktiles;
                v[u] = __ldcg(p.partial + (ch * p.sk_slots + (tl - first)) * (32LL * NTHREADS) + entry);
            }
        }
#pragma unroll
        for (int u = 0; u < 8; ++u)
            if (ch0 + u <= ch_hi) { sr += v[u].x; si += v[u].y; }
    }
    // the same arithmetic as store_fragment (alpha = 1: none; real alpha: one product per component; complex: fma pairs)
    const double ar = p.alpha_re, ai = p.alpha_im;
    double vx, vy;
    if (ai != 0.0) { vx = fma(ar, sr, -ai * si); vy = fma(ar, si, ai * sr); }
    else if (ar != 1.0) { vx = ar * sr; vy = ar * si; }
    else { vx = sr; vy = si; }
    double2 *dst = p.D + p.offM[m] + p.offN[n];
    if (p.accumulate) {
        const double2 d = *dst;
        vx += d.x;
        vy += d.y;
    }
    *dst = make_double2(vx, vy);
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *,
                                  CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                  CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode_fn()
{
    static EncodeTiledFn fn = nullptr;
    static std::once_flag once;
    std::call_once(once, [] {
        void *ptr = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ptr, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)ptr;
    });
    return fn;
}

// one operand: K-major -> dims {2K doubles, rows}, box {16, 64};  M-major -> dims {2*rows doubles, K}, box {16, 8}
cudaError_t encode_operand(CUtensorMap *tm, const void *ptr, int64_t rows, int64_t K, int64_t ld, bool kmajor,
                           int box_rows, int box_k)
{
    EncodeTiledFn fn = get_encode_fn();
    if (!fn) return cudaErrorNotSupported;
    cuuint64_t dims[2], strides[1];
    cuuint32_t box[2], estr[2] = {1, 1};
    if (kmajor) {
        dims[0] = (cuuint64_t)(2 * K);
        dims[1] = (cuuint64_t)rows;
        box[0] = 16;
        box[1] = (cuuint32_t)box_rows;
    } else {
        dims[0] = (cuuint64_t)(2 * rows);
        dims[1] = (cuuint64_t)K;
        box[0] = 16;
        box[1] = (cuuint32_t)box_k;
    }
    strides[0] = (cuuint64_t)ld * 16;
    CUresult r = fn(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<void *>(ptr), dims, strides, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                    getenv("TCB_GEMM_PROMO") ? (CUtensorMapL2promotion)atoi(getenv("TCB_GEMM_PROMO")) : CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}


template <int AM, int BM_, bool M3>
cudaError_t launch_variant(const GemmTensorMaps &maps, const GemmParams &p, int grid, cudaStream_t stream)
{
    auto kern = zgemm_dmma_kernel<AM, BM_, M3>;
    constexpr int smem = M3 ? SMEM_BYTES_3M : SMEM_BYTES;
    if (first_use_on_device((const void *)kern)) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
        if (e != cudaSuccess) return e;
    }
    kern<<<grid, NTHREADS, smem, stream>>>(maps.a, maps.b, p);
    return cudaGetLastError();
}

template <int AM, bool M3>
cudaError_t launch_b(int bmode, const GemmTensorMaps &maps, const GemmParams &p, int grid, cudaStream_t stream)
{
    switch (bmode) {
    case kTmaK: return launch_variant<AM, kTmaK, M3>(maps, p, grid, stream);
    case kTmaM: return launch_variant<AM, kTmaM, M3>(maps, p, grid, stream);
    default: return launch_variant<AM, kGather, M3>(maps, p, grid, stream);
    }
}
template <bool M3>
cudaError_t launch_a(int amode, int bmode, const GemmTensorMaps &maps, const GemmParams &p, int grid, cudaStream_t stream)
{
    switch (amode) {
    case kTmaK: return launch_b<kTmaK, M3>(bmode, maps, p, grid, stream);
    case kTmaM: return launch_b<kTmaM, M3>(bmode, maps, p, grid, stream);
    default: return launch_b<kGather, M3>(bmode, maps, p, grid, stream);
    }
}


}  // namespace

GemmSchedule gemm_schedule(int64_t M, int64_t N, int64_t K, int splitk, bool m3)
{
    GemmSchedule s;
    const int64_t mblocks = (M + 7) / 8, nblocks = (N + 7) / 8;
    const int tb = m3 ? 6 : 8;                            // blocks per tile dimension (3M: 48 x 48 tiles)
    s.mt = (int)((mblocks + tb - 1) / tb);
    s.nt = (int)((nblocks + tb - 1) / tb);
    const int kb = m3 ? 16 : BK;                          // k-values per stage
    s.ktiles = (int)((K + kb - 1) / kb);
    const int64_t tiles = (int64_t)s.mt * s.nt, KT = s.ktiles;
    const int64_t slots = 2LL * sm_count();              // resident CTAs: the persistent grid is 2 per SM
    s.dp_tiles = tiles; s.sk_tiles = 0; s.sk_chunks = 0; s.sk_q = 1; s.sk_slots = 1; s.splits = 1;
    if (splitk > 1) {                                    // forced: every tile cut into ~splitk pieces
        s.dp_tiles = 0; s.sk_tiles = tiles;
        s.sk_q = (int)std::max<int64_t>(1, (KT + splitk - 1) / splitk);
        s.splits = (int)((KT + s.sk_q - 1) / s.sk_q);
    } else if (splitk == 0) {                            // auto: full waves whole, the remainder cut along K
        const int64_t rem = tiles % slots;
        // worth it when the remainder wave would leave most of the chip idle for a whole K sweep; a chunk
        // shorter than 8 k-tiles costs more in fix-up traffic than it saves
        if (rem > 0 && rem * KT / slots + (m3 ? 4 : 8) < KT * 9 / 10) {      // the fix-up costs about 8 k-tiles (4 of the 16-deep ones)
            s.dp_tiles = tiles - rem; s.sk_tiles = rem;
            // three to six chunks per CTA, claimed dynamically: they even out what whole tiles left uneven and what
            // ragged tiles make uneven among the chunks themselves (a 6 x 6-block tile costs half an 8 x 8 one).
            // With very few tiles (skinny M x N) one chunk per CTA: a tile's chunks are summed one after the other
            // by the fix-up, the fewer the better.
            // measured: 6 per CTA behind whole tiles (pp ladder 33.1 -> 33.7 TFLOP/s: the tail is half a chunk), 3 when
            // everything is chunks (more only lengthens the fix-up's sums)
            // A handful of tiles (2 ... 15, small M x N with a long K): four chunks per CTA of >= 24 k-tiles.  The tiles of
            // such a grid are ragged (M = 150 -> 64 + 48 + 38 rows) and a k-tile of a 6 x 6-block tile costs 9/16 of an
            // 8 x 8 one; with one equal chunk per CTA the CTAs on the small tiles idle while the full tiles finish
            // (150 x 150 x 135000 took as long as 192 x 192 x 135000: 1.13 ms; dynamic claims of smaller chunks: 0.90 ms).
            // A single tile has nothing to balance: one chunk per CTA.
            // Only where the tiles really differ (largest / mean warp work >= 1.25): with equal tiles (128 x 128, 192 x 192)
            // more chunks only lengthen the fix-up (0.53 -> 0.60 ms).
            auto warp_rows = [](int64_t blocks, int tiles_dim, int64_t *sum, int64_t *mx) {
                const int64_t pairs = (blocks + 1) / 2, base = pairs / tiles_dim, extra = pairs % tiles_dim;
                int64_t at = 0;
                *sum = 0; *mx = 0;
                for (int t = 0; t < tiles_dim; ++t) {
                    const int64_t np = base + (t < extra ? 1 : 0);
                    const int64_t b = std::min<int64_t>(2 * (at + np), blocks) - 2 * at;
                    at += np;
                    *sum += (b + 1) / 2;
                    *mx = std::max<int64_t>(*mx, (b + 1) / 2);
                }
            };
            int64_t sm_, mm_, sn_, mn_;
            warp_rows(mblocks, s.mt, &sm_, &mm_);
            warp_rows(nblocks, s.nt, &sn_, &mn_);
            const bool ragged = 4 * mm_ * mn_ * tiles >= 5 * sm_ * sn_;          // max >= 1.25 x mean
            const bool few = tiles > 1 && tiles < 16 && ragged;
            const int64_t per_cta = tiles >= slots ? 6 : tiles >= 16 ? 3 : few ? 4 : 1;
            // shortest chunk: 8 k-tiles; 5 of the 3M kernel's 16-deep ones (configs[0], 576 x 64 x 576 = 24 tiles of 36 k-tiles:
            // 5 chunks per tile 19.9 us per call in a graph, 6 chunks 16.7 us, 9 chunks 17.5 us, 18 chunks 20.2 us)
            const int64_t min_q = few ? 24 : m3 ? 5 : 8;
            const int64_t chunks = std::max<int64_t>(1, std::min<int64_t>(per_cta * slots, rem * KT / min_q));
            s.sk_q = (int)((rem * KT + chunks - 1) / chunks);
            if (s.dp_tiles == 0) s.splits = (int)((KT + s.sk_q - 1) / s.sk_q);
        }
    }
    s.partial_bytes = 0;
    if (s.sk_tiles > 0) {
        s.sk_chunks = (s.sk_tiles * KT + s.sk_q - 1) / s.sk_q;
        s.sk_slots = (int)((s.sk_q + KT - 2) / KT + 1);
        s.partial_bytes = (size_t)s.sk_chunks * s.sk_slots * 32 * NTHREADS * sizeof(double2);
    }
    const int64_t units = std::max<int64_t>(std::min<int64_t>(s.dp_tiles, slots), std::min<int64_t>(s.sk_chunks, slots));
    s.grid = (int)std::max<int64_t>(1, units);
    return s;
}

cudaError_t encode_gemm_maps(const GemmDesc &g, GemmTensorMaps *maps)
{
    // a strided dimension of extent 1 still needs a legal stride: ld >= 1 always holds here; a gathered operand has no map
    std::memset(maps, 0, sizeof *maps);
    const int box_rows = g.m3 ? 48 : BM;
    if (!g.gatherAm) {
        cudaError_t e = encode_operand(&maps->a, g.A, g.M, g.K, g.lda, g.a_kmajor, box_rows, g.m3 ? 16 : 8);
        if (e != cudaSuccess) return e;
    }
    if (!g.gatherBn) return encode_operand(&maps->b, g.B, g.N, g.K, g.ldb, g.b_kmajor, box_rows, g.m3 ? 16 : 8);
    return cudaSuccess;
}

cudaError_t launch_zgemm_with_maps(const GemmDesc &g, const GemmTensorMaps &maps, cudaStream_t stream,
                                   int64_t *launches)
{
    const GemmSchedule sc = gemm_schedule(g.M, g.N, g.K, g.splitk, g.m3);
    GemmParams p;
    p.M = g.M; p.N = g.N; p.K = g.K;
    p.mblocks = (int)((g.M + 7) / 8);
    p.nblocks = (int)((g.N + 7) / 8);
    p.mt = sc.mt; p.nt = sc.nt;
    if ((int64_t)sc.mt * sc.nt >= (1LL << 31)) return cudaErrorInvalidValue;      // 32-bit tile index
    const int mpairs = (p.mblocks + 1) / 2, npairs = (p.nblocks + 1) / 2;
    p.mpair_base = mpairs / sc.mt; p.mpair_extra = mpairs % sc.mt;
    p.npair_base = npairs / sc.nt; p.npair_extra = npairs % sc.nt;
    // width of a tile-column group: every tile column while there are at most 32 (a wave of 296 CTAs then shares each A row
    // panel among all of them), else 16.  configs[2] (25 tile columns), DRAM read per launch by ncu: 215 GB at 4, 145 GB at 8
    // and 16, 120 GB at 25 -- same 578 ms (profiles/r2_zgemm_configs2_ncu.md)
    p.gn = p.nt <= 32 ? p.nt : 16;
    if (getenv("TCB_GEMM_GN")) p.gn = std::max(1, std::min(p.nt, atoi(getenv("TCB_GEMM_GN"))));
    p.ktiles = sc.ktiles;
    p.klast_steps = (int)((g.K - (int64_t)(sc.ktiles - 1) * (g.m3 ? 16 : BK) + 3) / 4);
    p.dp_tiles = sc.dp_tiles; p.sk_tiles = sc.sk_tiles; p.sk_chunks = sc.sk_chunks;
    p.sk_q = sc.sk_q; p.sk_slots = sc.sk_slots;
    p.D = (double2 *)g.D;
    p.offM = (const long long *)g.offM;
    p.offN = (const long long *)g.offN;
    p.alpha_re = g.alpha_re; p.alpha_im = g.alpha_im;
    p.accumulate = g.accumulate ? 1 : 0;
    // measured: K = 30 into an 8 GB D 7.8 -> 6.5 ms, K = 64 plain GEMM 25.4 -> 27.7 TFLOP/s; TCB_GEMM_RED=0 keeps the
    // software-pipelined read-modify-write for A/B tests
    p.use_red = getenv("TCB_GEMM_RED") ? atoi(getenv("TCB_GEMM_RED")) : 1;
    p.partial = (double2 *)g.partial;
    p.counters = (unsigned long long *)g.counters;      // zero on entry; the last CTA to leave zeroes them again
    if (sc.partial_bytes && !p.partial) return cudaErrorInvalidValue;
    p.gA = (const double2 *)g.A; p.gB = (const double2 *)g.B;
    p.gAm = (const long long *)g.gatherAm; p.gAk = (const long long *)g.gatherAk;
    p.gBn = (const long long *)g.gatherBn; p.gBk = (const long long *)g.gatherBk;
    p.a_mfast = g.a_mfast ? 1 : 0; p.b_mfast = g.b_mfast ? 1 : 0;
    const int amode = g.gatherAm ? kGather : (g.a_kmajor ? kTmaK : kTmaM);
    const int bmode = g.gatherBn ? kGather : (g.b_kmajor ? kTmaK : kTmaM);
    cudaError_t e = g.m3 ? launch_a<true>(amode, bmode, maps, p, sc.grid, stream)
                         : launch_a<false>(amode, bmode, maps, p, sc.grid, stream);
    if (e != cudaSuccess) return e;
    if (launches) ++*launches;
    if (sc.sk_tiles > 0) {
        zgemm_fixup_kernel<<<dim3((unsigned)sc.sk_tiles, 32), NTHREADS, 0, stream>>>(p);
        e = cudaGetLastError();
        if (e != cudaSuccess) return e;
        if (launches) ++*launches;
    }
    return cudaSuccess;
}

cudaError_t launch_zgemm(const GemmDesc &g, cudaStream_t stream, int64_t *launches)
{
    GemmTensorMaps maps;
    cudaError_t e = encode_gemm_maps(g, &maps);
    if (e != cudaSuccess) return e;
    return launch_zgemm_with_maps(g, maps, stream, launches);
}

}  // namespace tcb
