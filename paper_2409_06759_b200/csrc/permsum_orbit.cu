// permsum_orbit.cu -- S6 fast path for antisymmetrisers over THREE leading indices of equal extent:
//   D = beta D + sum_t c_t X[pi_t(.)],  every pi_t permuting the leading indices {0,1,2} among themselves and the
//   remaining ("outer") indices among themselves -- the unrolled P(a/bc), P(a/bc)P(k/ij) of a CCSDT residual
//   (PAPER.md:194, 230, 284).
//
// Why (profiles/r1b_permsum.md): the gather kernels read every term straight from L2; with 9 terms that is 9 x 16
// bytes per element through l1tex, 10-16 cache lines per warp gather (tag stage 75 % busy), X fetched 4.9x from DRAM.
// Here the leading indices are cut into 6 x 6 x 6 cubes.  A permutation of the leading indices maps cubes to cubes, the
// cubes reachable from one another form an orbit of <= 6.  One work item = one orbit at one value of the outer indices:
//   * a producer warp loads the orbit's cubes of X, once per distinct outer permutation (k/ij: 3), with ONE tiled TMA
//     load per cube (cp.async.bulk.tensor.4d over the map {a, b, c, outer slab}, box 6 x 6 x 6 x 1, SASS UTMALDG) into
//     a 3-stage mbarrier ring -- L2 -> SM traffic 3 x X instead of 9 x X, no per-row copy instructions;
//   * a D warp loads the orbit's cubes of D two items ahead (tiled TMA loads into a ring of D buffers) and writes the
//     finished cubes back with tiled TMA stores (cp.async.bulk.tensor.4d.global.shared::cta, per-thread bulk groups);
//     ragged extents need no masks: TMA zero-fills loads and clips stores;
//   * 14 consumer warps compute in place in the D buffer from shared memory: a quarter-warp is a 2 x 2 x 2 micro-cube,
//     whose eight 16-byte accesses fall in eight different bank groups under EVERY permutation of (a,b,c) because the
//     cube strides 1, 6, 36 are 1, 6, 4 mod 8 (no padding, which TMA boxes could not have);
//   * items are ordered so that the (<= 6) outer slabs that are permutations of one another are processed together
//     by one CTA for one orbit: each cube of X comes from DRAM once.
// Terms are added in the caller's order with separately rounded products and sums: bit-identical to the generic
// kernel and to the oracle.
#include "kernels.h"
#include "ptx.cuh"

#include <algorithm>
#include <cstdlib>
#include <map>
#include <mutex>
#include <numeric>
#include <vector>

namespace tcb {

namespace {

using namespace ptx;

constexpr int T6 = 6;                       // cube edge
constexpr int kCube = T6 * T6 * T6;         // 216 elements, 3456 bytes = 27 x 128
constexpr int kCubeBytes = kCube * 16;
constexpr int kConsumerWarps = 14;          // 162 micro-cubes per orbit = 3 rounds of 14 warps x 4 quarter-warps
constexpr int kThreads = (kConsumerWarps + 2) * 32;   // + the X producer warp and the D load/store warp
constexpr int kRounds = 3;
constexpr int kMaxOmega = 6;                // cubes per orbit
constexpr int kMaxTau = 6;                  // distinct outer permutations
constexpr int kMaxStages = 8;
constexpr int kOrbTerms = 9;

struct alignas(4) OrbitEntry {              // one orbit of cube coordinates
    unsigned char n, pad;                            // cubes in the orbit
    unsigned char coord[kMaxOmega][3];               // block coordinates
    unsigned char src[kMaxOmega][kOrbTerms];         // cube of X that term t reads for cube w of D
};
static_assert(sizeof(OrbitEntry) == 76, "OrbitEntry is copied word by word");

struct OrbitParams {
    int nterms, ntau, nO, stages, dbufs, eI, beta_zero;
    int eO[3];                               // outer extents (dims 3..)
    long long slab_elems;                    // eI^3
    long long xsO[kMaxTau][3];               // stride in X of D's outer index k under outer class u
    int sstr[kOrbTerms][3];                  // shared-memory stride of D's leading index k under term t (1, 6 or 36)
    unsigned char tau[kOrbTerms];            // outer class of term t
    double cr[kOrbTerms], ci[kOrbTerms], br, bi;
    unsigned norbits, ngroups;
    const OrbitEntry *orbits;
    const unsigned *slab_order;              // slabs, group by group
    const unsigned *group_start;             // [ngroups + 1] into slab_order
    double2 *D;
};

__device__ __forceinline__ void tma_load_4d(uint32_t dst, const CUtensorMap *tm, int c0, int c1, int c2, int c3,
                                            uint32_t bar)
{
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
        ::"r"(dst), "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(bar)
        : "memory");
}

__device__ __forceinline__ void tma_store_4d(const CUtensorMap *tm, int c0, int c1, int c2, int c3, uint32_t src)
{
    asm volatile("cp.async.bulk.tensor.4d.global.shared::cta.bulk_group [%0, {%1, %2, %3, %4}], [%5];" ::"l"(tm),
                 "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(src)
                 : "memory");
}

struct alignas(16) StageMeta {               // written by the X producer warp before it arms the stage's barrier
    int slot[kMaxOmega][12];                 // element offset (in the stage) of the cube term t reads for cube w
    int n;
    unsigned ob[sizeof(OrbitEntry) / 4];     // producer scratch: the item's orbit entry
};

// Items: for group g of outer slabs (slabs that are permutations of one another), for orbit o: the group's slabs.
// CTA b takes the (g, o) pairs b, b + grid, ...; the two producer warps and the consumers walk the same sequence.
struct ItemCursor {
    unsigned long long pair, npairs;
    unsigned s, s_end, orbit;
    __device__ __forceinline__ void init(const OrbitParams &p)
    {
        npairs = (unsigned long long)p.ngroups * p.norbits;
        pair = blockIdx.x;
        load(p);
    }
    __device__ __forceinline__ void load(const OrbitParams &p)
    {
        if (pair < npairs) {
            const unsigned g = (unsigned)(pair / p.norbits);
            orbit = (unsigned)(pair - (unsigned long long)g * p.norbits);
            s = p.group_start[g];
            s_end = p.group_start[g + 1];
        }
    }
    __device__ __forceinline__ bool valid() const { return pair < npairs; }
    __device__ __forceinline__ void advance(const OrbitParams &p)
    {
        if (++s == s_end) {
            pair += gridDim.x;
            load(p);
        }
    }
};

// barrier indices
constexpr int kMaxDBufs = 6;
constexpr int kXFull = 0, kXEmpty = kMaxStages, kDFull = 2 * kMaxStages, kDReady = 2 * kMaxStages + kMaxDBufs;
constexpr int kNumBars = 2 * kMaxStages + 2 * kMaxDBufs;

__global__ void __launch_bounds__(kThreads, 1)
permsum_orbit_kernel(const __grid_constant__ CUtensorMap tmX, const __grid_constant__ CUtensorMap tmD,
                     const __grid_constant__ OrbitParams p)
{
    extern __shared__ __align__(128) uint8_t orb_smem[];
    __shared__ __align__(8) unsigned long long s_bar[kNumBars];
    __shared__ StageMeta s_meta[kMaxStages];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const uint32_t bar0 = smem_u32(s_bar);
    const uint32_t stage_bytes = (uint32_t)(kMaxOmega * p.ntau * kCubeBytes);
    const uint32_t dbuf_bytes = kMaxOmega * kCubeBytes;
    // shared memory: [2 D buffers of 6 cubes][stages x (6 * ntau cubes of X)]
    const uint32_t dbuf0 = smem_u32(orb_smem);
    const uint32_t data0 = dbuf0 + p.dbufs * dbuf_bytes;
    if (tid == 0) {
        for (int s = 0; s < p.stages; ++s) {
            mbar_init(bar0 + 8 * (kXFull + s), 1);                  // the producer's arrive + the bytes
            mbar_init(bar0 + 8 * (kXEmpty + s), kConsumerWarps);    // one arrive per consumer warp
        }
        for (int b = 0; b < p.dbufs; ++b) {
            mbar_init(bar0 + 8 * (kDFull + b), 1);                  // D cubes loaded (or, beta = 0, buffer free)
            mbar_init(bar0 + 8 * (kDReady + b), kConsumerWarps);    // results written: the buffer may be stored
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmX) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmD) : "memory");
    }
    __syncthreads();
    ItemCursor cur;
    cur.init(p);
    if (warp == kConsumerWarps) {
        // ================= X producer warp =================
        unsigned it = 0;
        for (; cur.valid(); cur.advance(p), ++it) {
            const int st = (int)(it % (unsigned)p.stages);
            const uint32_t par = (it / (unsigned)p.stages) & 1u;
            StageMeta &m = s_meta[st];
            // the item's orbit entry (word by word) and slab: fetched before the wait, so their latency hides behind it
            unsigned ob_word = 0;
            if (lane < (int)(sizeof(OrbitEntry) / 4))
                ob_word = __ldg(reinterpret_cast<const unsigned *>(p.orbits + cur.orbit) + lane);
            unsigned slab = __ldg(p.slab_order + cur.s);
            mbar_wait(bar0 + 8 * (kXEmpty + st), par ^ 1u);          // consumers are done with the stage
            if (lane < (int)(sizeof(OrbitEntry) / 4)) m.ob[lane] = ob_word;
            long long xoffO[kMaxTau];
#pragma unroll
            for (int u = 0; u < kMaxTau; ++u) xoffO[u] = 0;
#pragma unroll
            for (int k = 0; k < 3; ++k)
                if (k < p.nO) {
                    const long long v = slab % (unsigned)p.eO[k];
                    slab /= (unsigned)p.eO[k];
#pragma unroll
                    for (int u = 0; u < kMaxTau; ++u)
                        if (u < p.ntau) xoffO[u] += v * p.xsO[u][k];
                }
            __syncwarp();
            const OrbitEntry &ob = *reinterpret_cast<const OrbitEntry *>(m.ob);
            const int n = ob.n;
            for (int idx = lane; idx < kMaxOmega * kOrbTerms; idx += 32) {
                const int w = idx / kOrbTerms, t = idx - w * kOrbTerms;
                if (w < n && t < p.nterms) m.slot[w][t] = (ob.src[w][t] * p.ntau + p.tau[t]) * kCube;
            }
            if (lane == 0) m.n = n;
            __syncwarp();
            const uint32_t full = bar0 + 8 * (kXFull + st);
            if (lane == 0) mbar_expect_tx(full, (uint32_t)(n * p.ntau * kCubeBytes));
            __syncwarp();
            for (int idx = lane; idx < n * p.ntau; idx += 32) {
                const int g = idx / p.ntau, u = idx - g * p.ntau;
                long long xo = xoffO[0];
#pragma unroll
                for (int uu = 1; uu < kMaxTau; ++uu)
                    if (uu == u) xo = xoffO[uu];
                tma_load_4d(data0 + st * stage_bytes + (uint32_t)idx * kCubeBytes, &tmX, ob.coord[g][0] * (2 * T6),
                            ob.coord[g][1] * T6, ob.coord[g][2] * T6, (int)(xo / p.slab_elems), full);
            }
        }
        return;
    }
    if (warp == kConsumerWarps + 1) {
        // ================= D warp: loads the orbit's cubes of D two items ahead, stores the finished ones ==============
        // lane w < n owns cube w of the item: one tiled TMA load, one tiled TMA store (bulk groups are per thread)
        ItemCursor ld = cur;                                          // runs two items ahead of `cur`
        auto cube_coords = [&](const ItemCursor &c, int *n, int *c0, int *c1, int *c2, int *c3) {
            const OrbitEntry *ob = p.orbits + c.orbit;
            *n = __ldg(&ob->n);
            const int w = lane < kMaxOmega ? lane : 0;
            *c0 = __ldg(&ob->coord[w][0]) * (2 * T6);
            *c1 = __ldg(&ob->coord[w][1]) * T6;
            *c2 = __ldg(&ob->coord[w][2]) * T6;
            *c3 = (int)__ldg(p.slab_order + c.s);
        };
        auto load_item = [&](int b, int n, int c0, int c1, int c2, int c3) {
            const uint32_t full = bar0 + 8 * (kDFull + b);
            if (p.beta_zero) {                                       // nothing to read: just hand the buffer over
                if (lane == 0) mbar_arrive(full);
                return;
            }
            if (lane == 0) mbar_expect_tx(full, (uint32_t)(n * kCubeBytes));
            __syncwarp();
            if (lane < n) tma_load_4d(dbuf0 + b * dbuf_bytes + lane * kCubeBytes, &tmD, c0, c1, c2, c3, full);
        };
        for (int b = 0; b < p.dbufs; ++b)
            if (ld.valid()) {
                int n, c0, c1, c2, c3;
                cube_coords(ld, &n, &c0, &c1, &c2, &c3);
                load_item(b, n, c0, c1, c2, c3);
                ld.advance(p);
            }
        unsigned it = 0;
        for (; cur.valid(); cur.advance(p), ++it) {
            const int b = (int)(it % (unsigned)p.dbufs);
            int sn, s0, s1, s2, s3, ln = 0, l0 = 0, l1 = 0, l2 = 0, l3 = 0;
            cube_coords(cur, &sn, &s0, &s1, &s2, &s3);               // fetched before the wait
            const bool more = ld.valid();
            if (more) cube_coords(ld, &ln, &l0, &l1, &l2, &l3);
            mbar_wait(bar0 + 8 * (kDReady + b), (it / (unsigned)p.dbufs) & 1u);     // every consumer warp has written its results
            if (lane < sn) {
                tma_store_4d(&tmD, s0, s1, s2, s3, dbuf0 + b * dbuf_bytes + lane * kCubeBytes);
                asm volatile("cp.async.bulk.commit_group;" ::: "memory");
                asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");   // shared memory read: buffer reusable
            }
            __syncwarp();
            if (more) {
                load_item(b, ln, l0, l1, l2, l3);
                ld.advance(p);
            }
        }
        asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
        return;
    }
    // ================= consumer warps =================
    // A quarter-warp is a 2 x 2 x 2 micro-cube (conflict-free LDS.128 / STS.128 under every permutation of the three
    // indices); a cube has 27 of them, an orbit <= 162 = 3 rounds of 14 warps x 4.  Element <-> thread is the same for
    // every item.
    const int qw = lane >> 3, bits = lane & 7;
    int ew[kRounds], soff[kRounds][kOrbTerms], dl[kRounds];
#pragma unroll
    for (int j = 0; j < kRounds; ++j) {
        const int q = warp * 4 + qw + kConsumerWarps * 4 * j;
        ew[j] = q / 27;
        const int mc = q - ew[j] * 27, m2 = mc / 9, m1 = (mc - m2 * 9) / 3, m0 = mc - m2 * 9 - m1 * 3;
        const int l0 = 2 * m0 + (bits & 1), l1 = 2 * m1 + ((bits >> 1) & 1), l2 = 2 * m2 + (bits >> 2);
        dl[j] = ew[j] * kCube + l0 + T6 * l1 + T6 * T6 * l2;
#pragma unroll
        for (int t = 0; t < kOrbTerms; ++t) soff[j][t] = l0 * p.sstr[t][0] + l1 * p.sstr[t][1] + l2 * p.sstr[t][2];
    }
    unsigned it = 0;
    for (; cur.valid(); cur.advance(p), ++it) {
        const int st = (int)(it % (unsigned)p.stages);
        const uint32_t par = (it / (unsigned)p.stages) & 1u;
        const int b = (int)(it % (unsigned)p.dbufs);
        const StageMeta &m = s_meta[st];
        mbar_wait(bar0 + 8 * (kXFull + st), par);
        mbar_wait(bar0 + 8 * (kDFull + b), (it / (unsigned)p.dbufs) & 1u);
        const int n = m.n;
        const double2 *cubes = reinterpret_cast<const double2 *>(orb_smem + (size_t)p.dbufs * dbuf_bytes + (size_t)st * stage_bytes);
        double2 *dcube = reinterpret_cast<double2 *>(orb_smem + (size_t)b * dbuf_bytes);
#pragma unroll
        for (int j = 0; j < kRounds; ++j) {
            if (ew[j] >= n) continue;
            double ar = 0.0, ai = 0.0;
            if (!p.beta_zero) {
                const double2 dv = dcube[dl[j]];
                ar = __dsub_rn(__dmul_rn(p.br, dv.x), __dmul_rn(p.bi, dv.y));
                ai = __dadd_rn(__dmul_rn(p.br, dv.y), __dmul_rn(p.bi, dv.x));
            }
            int sl[12];
            {
                const int4 *sv = reinterpret_cast<const int4 *>(m.slot[ew[j]]);
#pragma unroll
                for (int q = 0; q < 3; ++q) {
                    const int4 v = sv[q];
                    sl[4 * q] = v.x; sl[4 * q + 1] = v.y; sl[4 * q + 2] = v.z; sl[4 * q + 3] = v.w;
                }
            }
#pragma unroll
            for (int t0 = 0; t0 < kOrbTerms; t0 += 3) {           // three conflict-free LDS.128 in flight, then their arithmetic
                double2 x[3];
#pragma unroll
                for (int u = 0; u < 3; ++u)
                    if (t0 + u < p.nterms) x[u] = cubes[sl[t0 + u] + soff[j][t0 + u]];
#pragma unroll
                for (int u = 0; u < 3; ++u)
                    if (t0 + u < p.nterms) {
                        const double cr = p.cr[t0 + u], ci = p.ci[t0 + u];
                        ar = __dadd_rn(ar, __dsub_rn(__dmul_rn(cr, x[u].x), __dmul_rn(ci, x[u].y)));
                        ai = __dadd_rn(ai, __dadd_rn(__dmul_rn(cr, x[u].y), __dmul_rn(ci, x[u].x)));
                    }
            }
            dcube[dl[j]] = make_double2(ar, ai);
        }
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // results visible to the TMA store
        __syncwarp();
        if (lane == 0) {
            mbar_arrive(bar0 + 8 * (kDReady + b));                    // this warp's results are in the D buffer
            mbar_arrive(bar0 + 8 * (kXEmpty + st));                   // this warp no longer reads the stage
        }
    }
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *,
                                  CUtensorMapInterleave, CUtensorMapSwizzle, CUtensorMapL2promotion,
                                  CUtensorMapFloatOOBfill);
EncodeTiledFn orbit_encode_fn()
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

// Everything about a call that does not depend on pointers and coefficients: built once per (shape, term set).
struct OrbitPlan {
    bool eligible = false;
    OrbitParams p;
    size_t smem = 0;
    long long nslabs = 1;
    int grid = 0;
};

std::vector<long long> plan_key(const PermSumDesc &d)
{
    std::vector<long long> k;
    int dev = 0;
    cudaGetDevice(&dev);
    k.push_back(dev);
    k.push_back(getenv("TCB_PERMSUM_ORBIT") ? 1 : 0);
    k.push_back(d.rank);
    k.push_back(d.nterms);
    for (int s = 0; s < d.rank; ++s) k.push_back(d.extent[s]);
    for (int t = 0; t < d.nterms; ++t)
        for (int s = 0; s < d.rank; ++s) k.push_back(d.xstride[t][s]);
    return k;
}

// Fills plan (tables on the device, allocated once and kept).  plan.eligible stays false when the term set is not of
// the "leading three equal-extent indices permuted among themselves" kind.
cudaError_t build_plan(const PermSumDesc &d, OrbitPlan &plan)
{
    const int r = d.rank;
    // measured on (60,60,60,12,12,12): 9 terms 4.3 ms here against 8.5 ms for the cube kernel; 3 terms 3.7 against 3.6 (both
    // near what HBM gives for 96-byte rows) -> the gather kernel keeps the short sums unless the caller forces this one
    const bool always = getenv("TCB_PERMSUM_ORBIT") != nullptr;
    if (r < 3 || d.nterms < (always ? 2 : 4) || d.nterms > kOrbTerms) return cudaSuccess;
    long long n = 1, ds[kMaxRank];
    for (int k = 0; k < r; ++k) {
        if (d.extent[k] < 2) return cudaSuccess;             // extent-1 indices: X strides are ambiguous
        ds[k] = n;
        n *= d.extent[k];
    }
    if (n < (1LL << 16)) return cudaSuccess;                 // small tensors: launch latency decides, keep the simple kernels
    // position in X of D's index s under term t (X strides are distinct: all extents >= 2)
    std::vector<std::vector<int>> pos(d.nterms, std::vector<int>(r));
    for (int t = 0; t < d.nterms; ++t)
        for (int s = 0; s < r; ++s) {
            int m = 0;
            for (int s2 = 0; s2 < r; ++s2) m += d.xstride[t][s2] < d.xstride[t][s] ? 1 : 0;
            pos[t][s] = m;
            if (d.extent[m] != d.extent[s] || d.xstride[t][s] != ds[m]) return cudaSuccess;   // X has D's shape
            if ((s < 3) != (m < 3)) return cudaSuccess;      // leading indices stay among the leading three
        }
    if (d.extent[0] != d.extent[1] || d.extent[0] != d.extent[2]) return cudaSuccess;
    {   // all three leading indices must really move (else the cube kernel is already coalesced and cheaper)
        bool moved[3] = {false, false, false};
        for (int t = 0; t < d.nterms; ++t)
            for (int s = 0; s < 3; ++s) moved[s] = moved[s] || pos[t][s] != s;
        if (!(moved[0] && moved[1] && moved[2])) return cudaSuccess;
    }
    OrbitParams &p = plan.p;
    p.nterms = d.nterms;
    p.eI = (int)d.extent[0];
    if (p.eI < T6 || d.extent[0] > 255 * T6) return cudaSuccess;
    const int nb = (p.eI + T6 - 1) / T6;
    p.nO = r - 3;
    long long nslabs = 1;
    for (int k = 0; k < 3; ++k) {
        p.eO[k] = k < p.nO ? (int)d.extent[3 + k] : 1;
        nslabs *= p.eO[k];
    }
    if (nslabs > (1LL << 22)) return cudaSuccess;
    p.slab_elems = ds[2] * d.extent[2];
    // outer-permutation classes
    std::map<std::vector<int>, int> classes;
    const int q[3] = {1, T6, T6 * T6};
    for (int t = 0; t < d.nterms; ++t) {
        std::vector<int> key;
        for (int k = 0; k < p.nO; ++k) key.push_back(pos[t][3 + k]);
        auto it = classes.find(key);
        if (it == classes.end()) {
            if ((int)classes.size() == kMaxTau) return cudaSuccess;
            const int u = (int)classes.size();
            it = classes.emplace(key, u).first;
            for (int k = 0; k < 3; ++k) p.xsO[u][k] = k < p.nO ? d.xstride[t][3 + k] : 0;
        }
        p.tau[t] = (unsigned char)it->second;
        for (int k = 0; k < 3; ++k) p.sstr[t][k] = q[pos[t][k]];
    }
    for (int t = d.nterms; t < kOrbTerms; ++t) {
        p.tau[t] = 0;
        for (int k = 0; k < 3; ++k) p.sstr[t][k] = 0;
    }
    p.ntau = (int)classes.size();
    for (int u = p.ntau; u < kMaxTau; ++u)
        for (int k = 0; k < 3; ++k) p.xsO[u][k] = 0;
    const size_t stage_bytes = (size_t)kMaxOmega * p.ntau * kCubeBytes;
    const size_t budget = 227 * 1024 - 4096;                       // static: barriers, stage tables
    p.dbufs = getenv("TCB_ORBIT_DBUFS") ? std::max(2, std::min(kMaxDBufs, atoi(getenv("TCB_ORBIT_DBUFS")))) : 2;
    const size_t dbufs = (size_t)p.dbufs * kMaxOmega * kCubeBytes;
    p.stages = (int)std::min<size_t>(kMaxStages, (budget - dbufs) / stage_bytes);
    if (getenv("TCB_ORBIT_STAGES")) p.stages = std::min(p.stages, atoi(getenv("TCB_ORBIT_STAGES")));
    if (p.stages < 2) return cudaSuccess;
    plan.smem = dbufs + stage_bytes * p.stages;
    // ---- orbits of the cube coordinates under the terms ------------------------------------------------------------
    const int ncubes = nb * nb * nb;
    auto decode = [&](int id, int *c) { for (int k = 0; k < 3; ++k) { c[k] = id % nb; id /= nb; } };
    auto encode = [&](const int *c) { return (c[2] * nb + c[1]) * nb + c[0]; };
    auto image = [&](int id, int t) {          // cube of X that term t reads for cube `id` of D
        int c[3], g[3];
        decode(id, c);
        for (int k = 0; k < 3; ++k) g[pos[t][k]] = c[k];
        return encode(g);
    };
    std::vector<int> orbit_of((size_t)ncubes, -1);
    std::vector<OrbitEntry> orbits;
    for (int id = 0; id < ncubes; ++id) {
        if (orbit_of[(size_t)id] >= 0) continue;
        std::vector<int> members = {id};
        orbit_of[(size_t)id] = (int)orbits.size();
        for (size_t h = 0; h < members.size(); ++h)
            for (int t = 0; t < d.nterms; ++t) {
                const int g = image(members[h], t);
                if (orbit_of[(size_t)g] < 0) {
                    if ((int)members.size() == kMaxOmega) return cudaSuccess;
                    orbit_of[(size_t)g] = (int)orbits.size();
                    members.push_back(g);
                }
            }
        OrbitEntry e;
        std::fill((unsigned char *)&e, (unsigned char *)&e + sizeof e, (unsigned char)0);
        e.n = (unsigned char)members.size();
        for (size_t w = 0; w < members.size(); ++w) {
            int c[3];
            decode(members[w], c);
            for (int k = 0; k < 3; ++k) e.coord[w][k] = (unsigned char)c[k];
            for (int t = 0; t < d.nterms; ++t) {
                const int g = image(members[w], t);
                e.src[w][t] = (unsigned char)(std::find(members.begin(), members.end(), g) - members.begin());
            }
        }
        orbits.push_back(e);
    }
    // ---- groups of outer slabs that are permutations of one another (union-find over the outer classes) --------------
    std::vector<unsigned> order((size_t)nslabs), parent((size_t)nslabs);
    std::iota(order.begin(), order.end(), 0u);
    std::iota(parent.begin(), parent.end(), 0u);
    auto find = [&](unsigned a) {
        while (parent[a] != a) { parent[a] = parent[parent[a]]; a = parent[a]; }
        return a;
    };
    for (unsigned s = 0; s < (unsigned)nslabs; ++s) {
        long long v[3] = {0, 0, 0};
        unsigned rem = s;
        for (int k = 0; k < p.nO; ++k) { v[k] = rem % (unsigned)p.eO[k]; rem /= (unsigned)p.eO[k]; }
        for (int u = 0; u < p.ntau; ++u) {
            long long xo = 0;
            for (int k = 0; k < p.nO; ++k) xo += v[k] * p.xsO[u][k];
            const unsigned a = find(s), b = find((unsigned)(xo / p.slab_elems));
            if (a != b) parent[std::max(a, b)] = std::min(a, b);
        }
    }
    std::vector<unsigned> root((size_t)nslabs);
    for (unsigned s = 0; s < (unsigned)nslabs; ++s) root[s] = find(s);
    std::stable_sort(order.begin(), order.end(), [&](unsigned a, unsigned b) { return root[a] < root[b]; });
    std::vector<unsigned> group_start;
    for (unsigned i = 0; i < (unsigned)nslabs; ++i)
        if (i == 0 || root[order[i]] != root[order[i - 1]]) group_start.push_back(i);
    p.ngroups = (unsigned)group_start.size();
    group_start.push_back((unsigned)nslabs);
    p.norbits = (unsigned)orbits.size();
    // ---- tables to the device, kept for the life of the process ----------------------------------------------------
    const size_t b0 = orbits.size() * sizeof(OrbitEntry), b1 = order.size() * 4, b2 = group_start.size() * 4;
    const size_t o1 = (b0 + 15) / 16 * 16, o2 = o1 + (b1 + 15) / 16 * 16;
    char *tables = nullptr;
    cudaError_t e = cudaMalloc((void **)&tables, o2 + b2);
    if (e != cudaSuccess) return e;
    e = cudaMemcpy(tables, orbits.data(), b0, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(tables + o1, order.data(), b1, cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(tables + o2, group_start.data(), b2, cudaMemcpyHostToDevice);
    // the sources are pageable: cudaMemcpy may return once they are staged, before the DMA has landed, and the kernel runs on
    // a non-blocking stream that the legacy stream does not order -- wait for the copies here (once per shape and term set)
    if (e == cudaSuccess) e = cudaStreamSynchronize(0);
    if (e != cudaSuccess) { cudaFree(tables); return e; }
    p.orbits = reinterpret_cast<const OrbitEntry *>(tables);
    p.slab_order = reinterpret_cast<const unsigned *>(tables + o1);
    p.group_start = reinterpret_cast<const unsigned *>(tables + o2);
    plan.nslabs = nslabs;
    plan.grid = (int)std::min<unsigned long long>((unsigned long long)p.ngroups * p.norbits, (unsigned long long)sm_count());
    plan.eligible = true;
    return cudaSuccess;
}

}  // namespace

// Returns cudaSuccess with *handled = false when the call is not of this kernel's kind (the caller then runs the
// gather kernels).
cudaError_t launch_permsum_orbit(const PermSumDesc &d, cudaStream_t stream, int64_t *launches, bool *handled)
{
    *handled = false;
    if (getenv("TCB_PERMSUM_GENERIC") || getenv("TCB_PERMSUM_NO_ORBIT")) return cudaSuccess;
    EncodeTiledFn fn = orbit_encode_fn();
    if (!fn) return cudaSuccess;
    static std::mutex mu;
    static std::map<std::vector<long long>, OrbitPlan> plans;
    OrbitPlan plan;
    {
        std::lock_guard<std::mutex> lock(mu);
        const std::vector<long long> key = plan_key(d);
        auto it = plans.find(key);
        if (it == plans.end()) {
            OrbitPlan fresh;
            cudaError_t e = build_plan(d, fresh);
            if (e != cudaSuccess) return e;
            it = plans.emplace(key, fresh).first;
        }
        plan = it->second;
    }
    if (!plan.eligible) return cudaSuccess;
    OrbitParams p = plan.p;
    if ((reinterpret_cast<uintptr_t>(d.X) & 15) != 0) return cudaSuccess;
    for (int t = 0; t < kOrbTerms; ++t) {
        p.cr[t] = t < d.nterms ? d.coef_re[t] : 0.0;
        p.ci[t] = t < d.nterms ? d.coef_im[t] : 0.0;
    }
    p.br = d.beta_re; p.bi = d.beta_im;
    p.beta_zero = (d.beta_re == 0.0 && d.beta_im == 0.0) ? 1 : 0;
    p.D = (double2 *)d.D;
    if ((reinterpret_cast<uintptr_t>(d.D) & 15) != 0) return cudaSuccess;
    CUtensorMap tmX, tmD;
    static const CUtensorMapL2promotion kPromo = getenv("TCB_ORBIT_PROMO") ? (CUtensorMapL2promotion)atoi(getenv("TCB_ORBIT_PROMO")) : CU_TENSOR_MAP_L2_PROMOTION_L2_128B;
    {
        const cuuint64_t e = (cuuint64_t)p.eI;
        cuuint64_t dims[4] = {2 * e, e, e, (cuuint64_t)plan.nslabs};
        cuuint64_t strides[3] = {e * 16, e * e * 16, e * e * e * 16};
        cuuint32_t box[4] = {2 * T6, T6, T6, 1}, estr[4] = {1, 1, 1, 1};
        CUresult r = fn(&tmX, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, const_cast<void *>(d.X), dims, strides, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, kPromo,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r == CUDA_SUCCESS)
            r = fn(&tmD, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, d.D, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                   CU_TENSOR_MAP_SWIZZLE_NONE, kPromo, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
        if (r != CUDA_SUCCESS) return cudaSuccess;              // a shape the maps cannot express: the gather kernels
    }
    if (first_use_on_device((const void *)permsum_orbit_kernel)) {
        cudaError_t e = cudaFuncSetAttribute(permsum_orbit_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024 - 4096);
        if (e != cudaSuccess) return e;
    }
    permsum_orbit_kernel<<<plan.grid, kThreads, plan.smem, stream>>>(tmX, tmD, p);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    if (launches) ++*launches;
    *handled = true;
    return cudaSuccess;
}

}  // namespace tcb
