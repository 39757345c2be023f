// zgemm.cu -- S4 + S5: complex FP64 GEMM on the FP64 tensor cores with the permute-and-accumulate epilogue.
//
//   C[m,n] = sum_k A[m,k] B[k,n]     ("Use GEMM to execute the contraction")
//   D[offM[m] + offN[n]] (+)= alpha * C[m,n]   ("Transpose result array to obtain C", PAPER.md:91 -- done
//                                               here as a scatter through offset tables, no extra pass)
//
// B200 facts this design rests on (measured, profiles/r1_fp64_peak.txt): tcgen05 has no FP64 kind, the
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
//   * split-K (skinny M,N with huge K): grid.z slices of K write raw partial tiles, a second kernel sums
//     them in fixed order (deterministic, no atomics) and applies the same scatter.
#include "kernels.h"

#include <mutex>

namespace tcb {

namespace {

constexpr int BM = kGemmBM, BN = kGemmBN, BK = kGemmBK;
constexpr int STAGES = 4;
constexpr int A_BYTES = BM * BK * 16;   // 8 KB
constexpr int B_BYTES = BN * BK * 16;   // 8 KB
constexpr int STAGE_BYTES = A_BYTES + B_BYTES;
constexpr int SMEM_BYTES = STAGES * STAGE_BYTES + 1024 /*alignment slack*/ + 128 /*barriers*/;
constexpr int NTHREADS = 128;

struct GemmParams {
    long long M, N, K;
    int mt, nt, gn;
    int ktiles, splits, ktiles_per_split;
    double2 *D;
    const long long *offM;
    const long long *offN;
    double alpha_re, alpha_im;
    int accumulate;
    double2 *partial;
};

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "LAB_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra DONE;\n"
        "bra LAB_WAIT;\n"
        "DONE:\n"
        "}\n" ::"r"(bar),
        "r"(parity)
        : "memory");
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap *tm, int c0, int c1, uint32_t bar)
{
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
        ::"r"(dst), "l"(tm), "r"(c0), "r"(c1), "r"(bar)
        : "memory");
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
__device__ __forceinline__ double2 lds128(uint32_t addr)
{
    double2 v;
    asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
    return v;
}

template <bool A_KMAJOR, bool B_KMAJOR>
__global__ void __launch_bounds__(NTHREADS, 2)
zgemm_dmma_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB,
                  const GemmParams p)
{
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t bar_base = smem_base + STAGES * STAGE_BYTES;   // full[s] at +8s, empty[s] at +8(STAGES+s)

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int warp_m = warp & 1, warp_n = warp >> 1;

    // tile coordinates: groups of `gn` tile-columns, n fastest inside a group (concurrent CTAs form a
    // near-square block of the output so that A row panels and B column panels are shared through L2)
    int tile_m, tile_n;
    {
        const int group_sz = p.gn * p.mt;
        const int g = blockIdx.x / group_sz, rem = blockIdx.x % group_sz;
        const int n0t = g * p.gn;
        const int gw = min(p.gn, p.nt - n0t);
        tile_m = rem / gw;
        tile_n = n0t + rem % gw;
    }
    const int m0 = tile_m * BM, n0 = tile_n * BN;
    const int kt_begin = blockIdx.z * p.ktiles_per_split;
    const int kt_end = min(p.ktiles, kt_begin + p.ktiles_per_split);
    const int KT = kt_end - kt_begin;

    if (tid == 0) {
        for (int s = 0; s < STAGES; ++s) {
            mbar_init(bar_base + 8 * s, 1);
            mbar_init(bar_base + 8 * (STAGES + s), NTHREADS / 32);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmA) : "memory");
        asm volatile("prefetch.tensormap [%0];" ::"l"(&tmB) : "memory");
    }
    __syncthreads();

    auto issue = [&](int kt_local, int s) {
        const uint32_t bar = bar_base + 8 * s;
        const uint32_t sA = smem_base + s * STAGE_BYTES, sB = sA + A_BYTES;
        const int k0 = (kt_begin + kt_local) * BK;
        mbar_expect_tx(bar, STAGE_BYTES);
        if (A_KMAJOR) {
            tma_load_2d(sA, &tmA, 2 * k0, m0, bar);
        } else {
#pragma unroll
            for (int j = 0; j < BM / 8; ++j) tma_load_2d(sA + j * 1024, &tmA, 2 * (m0 + 8 * j), k0, bar);
        }
        if (B_KMAJOR) {
            tma_load_2d(sB, &tmB, 2 * k0, n0, bar);
        } else {
#pragma unroll
            for (int j = 0; j < BN / 8; ++j) tma_load_2d(sB + j * 1024, &tmB, 2 * (n0 + 8 * j), k0, bar);
        }
    };

    if (tid == 0) {
        const int npro = min(STAGES, KT);
        for (int s = 0; s < npro; ++s) issue(s, s);
    }

    // per-lane fragment offsets inside a 1 KB atom, for the two k-steps of a stage
    const int r = lane >> 2, c = lane & 3;
    const int rowmap = (r >> 1) + 4 * (r & 1);
    uint32_t offA[2], offB[2];
#pragma unroll
    for (int ks = 0; ks < 2; ++ks) {
        const int k = ks * 4 + c;
        offA[ks] = A_KMAJOR ? (rowmap * 128 + ((k ^ rowmap) * 16)) : (k * 128 + ((rowmap ^ k) * 16));
        offB[ks] = B_KMAJOR ? (rowmap * 128 + ((k ^ rowmap) * 16)) : (k * 128 + ((rowmap ^ k) * 16));
    }

    double cr[4][4][2], ci[4][4][2];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            cr[i][j][0] = cr[i][j][1] = 0.0;
            ci[i][j][0] = ci[i][j][1] = 0.0;
        }

    for (int kt = 0; kt < KT; ++kt) {
        const int s = kt % STAGES;
        if (tid == 0 && kt >= 1 && kt - 1 + STAGES < KT) {
            // refill the stage consumed in the previous iteration (the other warps had a whole stage to release it)
            const int sp = (kt - 1) % STAGES;
            mbar_wait(bar_base + 8 * (STAGES + sp), ((kt - 1) / STAGES) & 1);
            issue(kt - 1 + STAGES, sp);
        }
        mbar_wait(bar_base + 8 * s, (kt / STAGES) & 1);
        const uint32_t sA = smem_base + s * STAGE_BYTES + (warp_m * 4) * 1024;
        const uint32_t sB = smem_base + s * STAGE_BYTES + A_BYTES + (warp_n * 4) * 1024;
#pragma unroll
        for (int ks = 0; ks < 2; ++ks) {
            double2 a[4], b[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) a[i] = lds128(sA + i * 1024 + offA[ks]);
#pragma unroll
            for (int j = 0; j < 4; ++j) b[j] = lds128(sB + j * 1024 + offB[ks]);
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const double nai = neg_exact(a[i].y);
#pragma unroll
                for (int j = 0; j < 4; ++j) {
                    dmma(cr[i][j][0], cr[i][j][1], a[i].x, b[j].x);
                    dmma(ci[i][j][0], ci[i][j][1], a[i].x, b[j].y);
                    dmma(cr[i][j][0], cr[i][j][1], nai, b[j].y);
                    dmma(ci[i][j][0], ci[i][j][1], a[i].y, b[j].x);
                }
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_base + 8 * (STAGES + s));
    }

    // ---- epilogue: lane holds C[m = mb*8 + rowmap][n = nb*8 + c (+4)] for its 4x4 blocks -----------------
    const long long mw = (long long)m0 + warp_m * 32 + rowmap;
    const long long nw = (long long)n0 + warp_n * 32 + c;
    if (p.splits > 1) {
        double2 *P = p.partial + (long long)blockIdx.z * p.M * p.N;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const long long m = mw + i * 8;
            if (m >= p.M) continue;
#pragma unroll
            for (int j = 0; j < 4; ++j)
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    const long long n = nw + j * 8 + h * 4;
                    if (n < p.N) P[n * p.M + m] = make_double2(cr[i][j][h], ci[i][j][h]);
                }
        }
        return;
    }
    long long om[4], on[4][2];
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const long long m = mw + i * 8;
        om[i] = (m < p.M) ? p.offM[m] : -1;
    }
#pragma unroll
    for (int j = 0; j < 4; ++j)
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            const long long n = nw + j * 8 + h * 4;
            on[j][h] = (n < p.N) ? p.offN[n] : -1;
        }
    const double ar = p.alpha_re, ai = p.alpha_im;
#pragma unroll
    for (int j = 0; j < 4; ++j)
#pragma unroll
        for (int h = 0; h < 2; ++h) {
            if (on[j][h] < 0) continue;
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                if (om[i] < 0) continue;
                double2 *dst = p.D + om[i] + on[j][h];
                const double xr = cr[i][j][h], xi = ci[i][j][h];
                double2 v = make_double2(ar * xr - ai * xi, ar * xi + ai * xr);
                if (p.accumulate) {
                    const double2 d = *dst;
                    v.x += d.x;
                    v.y += d.y;
                }
                *dst = v;
            }
        }
}

// deterministic split-K reduction + scatter: D[offM[m]+offN[n]] (+)= alpha * sum_z P[z][n][m]  (z ascending)
__global__ void __launch_bounds__(256)
splitk_reduce_kernel(const double2 *__restrict__ P, int splits, long long M, long long N, double2 *D,
                     const long long *__restrict__ offM, const long long *__restrict__ offN, double ar, double ai,
                     int accumulate)
{
    const long long total = M * N;
    for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < total;
         e += (long long)gridDim.x * blockDim.x) {
        double sr = 0.0, si = 0.0;
        for (int z = 0; z < splits; ++z) {
            const double2 v = P[(long long)z * total + e];
            sr += v.x;
            si += v.y;
        }
        const long long m = e % M, n = e / M;
        double2 *dst = D + offM[m] + offN[n];
        double2 v = make_double2(ar * sr - ai * si, ar * si + ai * sr);
        if (accumulate) {
            const double2 d = *dst;
            v.x += d.x;
            v.y += d.y;
        }
        *dst = v;
    }
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
                           int box_rows)
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
        box[1] = 8;
    }
    strides[0] = (cuuint64_t)ld * 16;
    CUresult r = fn(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, const_cast<void *>(ptr), dims, strides, box, estr,
                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                    CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

template <bool AK, bool BK_>
cudaError_t launch_variant(const GemmTensorMaps &maps, const GemmParams &p, dim3 grid, cudaStream_t stream)
{
    auto kern = zgemm_dmma_kernel<AK, BK_>;
    static bool configured = false;
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    kern<<<grid, NTHREADS, SMEM_BYTES, stream>>>(maps.a, maps.b, p);
    return cudaGetLastError();
}

}  // namespace

cudaError_t encode_gemm_maps(const GemmDesc &g, GemmTensorMaps *maps)
{
    // a strided dimension of extent 1 still needs a legal stride: ld >= 1 always holds here
    cudaError_t e = encode_operand(&maps->a, g.A, g.M, g.K, g.lda, g.a_kmajor, BM);
    if (e != cudaSuccess) return e;
    return encode_operand(&maps->b, g.B, g.N, g.K, g.ldb, g.b_kmajor, BN);
}

cudaError_t launch_zgemm_with_maps(const GemmDesc &g, const GemmTensorMaps &maps, cudaStream_t stream,
                                   int64_t *launches)
{
    GemmParams p;
    p.M = g.M; p.N = g.N; p.K = g.K;
    p.mt = (int)((g.M + BM - 1) / BM);
    p.nt = (int)((g.N + BN - 1) / BN);
    p.gn = p.nt <= 24 ? p.nt : 16;
    p.ktiles = (int)((g.K + BK - 1) / BK);
    p.splits = g.splits < 1 ? 1 : g.splits;
    if (p.splits > p.ktiles) p.splits = p.ktiles;
    p.ktiles_per_split = (p.ktiles + p.splits - 1) / p.splits;
    p.splits = (p.ktiles + p.ktiles_per_split - 1) / p.ktiles_per_split;   // no empty slices
    p.D = (double2 *)g.D;
    p.offM = (const long long *)g.offM;
    p.offN = (const long long *)g.offN;
    p.alpha_re = g.alpha_re; p.alpha_im = g.alpha_im;
    p.accumulate = g.accumulate ? 1 : 0;
    p.partial = (double2 *)g.partial;
    if (p.splits > 1 && !p.partial) return cudaErrorInvalidValue;
    dim3 grid((unsigned)((long long)p.mt * p.nt), 1, (unsigned)p.splits);
    cudaError_t e;
    if (g.a_kmajor)
        e = g.b_kmajor ? launch_variant<true, true>(maps, p, grid, stream)
                       : launch_variant<true, false>(maps, p, grid, stream);
    else
        e = g.b_kmajor ? launch_variant<false, true>(maps, p, grid, stream)
                       : launch_variant<false, false>(maps, p, grid, stream);
    if (e != cudaSuccess) return e;
    if (launches) ++*launches;
    if (p.splits > 1) {
        const long long total = g.M * g.N;
        int blocks = (int)((total + 255) / 256);
        if (blocks > 148 * 8) blocks = 148 * 8;
        splitk_reduce_kernel<<<blocks, 256, 0, stream>>>(p.partial, p.splits, p.M, p.N, p.D, p.offM, p.offN,
                                                         p.alpha_re, p.alpha_im, p.accumulate);
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
