// kernels.h -- internal launch interface between the host-side planner/API and the sm_100a kernels.
// Raw device pointers + stream only; no torch types anywhere in this library.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace tcb {

constexpr int kMaxRank = 6;

// Number of SMs of the current device (cudaDevAttrMultiProcessorCount, cached per device); 148 -- a B200 -- when no
// device can be asked (the host-only planner).  Every persistent grid is sized from this.
int sm_count();
// cudaFuncSetAttribute(MaxDynamicSharedMemorySize) is per device: true when `tag` (one per kernel instantiation) has not
// been configured on the current device yet (and marks it configured)
bool first_use_on_device(const void *tag);

// ---- S4 + S5: complex FP64 GEMM on DMMA with the permute-and-accumulate epilogue ---------------------
// C[m,n] = sum_k A[m,k] * B[k,n];   D[offM[m] + offN[n]] (+)= alpha * C[m,n]
// Operand layouts ("K-major": k has unit stride, element (row,k) at row*ld + k;
//                  "M-major": the row index has unit stride, element (row,k) at k*ld + row).
struct GemmDesc {
    int64_t M, N, K;
    const void *A, *B;       // device, complex128
    int64_t lda, ldb;        // in elements
    bool a_kmajor, b_kmajor;
    void *D;                 // device, complex128
    const int64_t *offM;     // device [M], element offsets into D
    const int64_t *offN;     // device [N]
    double alpha_re, alpha_im;
    bool accumulate;         // true: D += ...; false: D = ...
    int splitk;              // 0 = auto (stream-K on the remainder wave), 1 = off, n > 1 = every tile cut n ways
    void *partial;           // device, gemm_schedule(...).partial_bytes (raw accumulator fragments of cut tiles)
    void *counters = nullptr; // device, kGemmCounterBytes, 8-byte aligned, ZERO on entry (the kernel leaves them zero): work
                              // counters of the dynamic deal (null: static deal)
    // Permutation-free operand loads: when gatherAm is set, A is not a matrix in memory and is read in place
    // as A[m,k] = A[gatherAm[m] + gatherAk[k]] (device tables, element offsets; lda / a_kmajor unused); a_mfast: the operand's
    // unit-stride index is a row (free) index, so lanes run along m, else along k.  Same for B.
    const int64_t *gatherAm = nullptr, *gatherAk = nullptr, *gatherBn = nullptr, *gatherBk = nullptr;
    bool a_mfast = false, b_mfast = false;
    bool m3 = false;         // three real products per complex product, 48 x 48 tiles (zgemm.cu); the maps must be encoded with it
};
constexpr size_t kGemmCounterBytes = 64;
// How the (tile, k-tile) iteration space is dealt to the persistent grid (2 CTAs per SM): whole tiles
// data-parallel, the remainder ("stream-K") cut along K into equal chunks, one per CTA, summed by a fix-up kernel.
struct GemmSchedule {
    int mt, nt, ktiles, grid;
    int64_t dp_tiles, sk_tiles, sk_chunks;
    int sk_q, sk_slots;
    int splits;              // pieces per tile when every tile is cut (reported by the planner), else 1
    size_t partial_bytes;
};
GemmSchedule gemm_schedule(int64_t M, int64_t N, int64_t K, int splitk, bool m3 = false);
constexpr int kGemmBM = 64, kGemmBN = 64, kGemmBK = 8;
cudaError_t launch_zgemm(const GemmDesc &g, cudaStream_t stream, int64_t *launches);
// Encodes the two TMA descriptors; separated so that the planner can cache them.
struct GemmTensorMaps { CUtensorMap a, b; };
cudaError_t encode_gemm_maps(const GemmDesc &g, GemmTensorMaps *maps);
cudaError_t launch_zgemm_with_maps(const GemmDesc &g, const GemmTensorMaps &maps, cudaStream_t stream,
                                   int64_t *launches);

// ---- S2 regime "GEMV": one operand contracted away completely (N = 1); the other is read in place through offset tables
//   D[offD[m]] (+)= alpha * sum_k A[offAm[m] + offAk[k]] * B[offBk[k]]
struct GemvDesc {
    int64_t M, K;
    const void *A, *B;       // device, complex128: the operand with free indices, the fully contracted one
    void *D;
    const int64_t *offAm, *offAk, *offBk, *offD;   // device tables (element offsets)
    bool kfast;              // A's unit-stride index is contracted (warp per row) / free (thread per row)
    double alpha_re, alpha_im;
    bool accumulate;
    void *partial;           // device, gemv_ksplit(M, K, kfast) * M complex128 when the split is > 1
};
int gemv_ksplit(int64_t M, int64_t K, bool kfast);
// regime "outer product" (K = 1):  D[offM[m] + offN[n]] (+)= alpha * A[rowA[m]] * B[rowB[n]]   (device tables, element offsets)
struct OuterDesc {
    int64_t M, N;
    const void *A, *B;
    void *D;
    const int64_t *rowA, *rowB, *offM, *offN;
    double alpha_re, alpha_im;
    bool accumulate;
};
cudaError_t launch_outer(const OuterDesc &g, cudaStream_t stream, int64_t *launches);
cudaError_t launch_gemv(const GemvDesc &g, cudaStream_t stream, int64_t *launches);

// ---- S3: tensor transposition, and the permuted add built on it ------------------------------------------
// out[sum_d idx_d * ostride[d]] (op)= in[sum_d idx_d * istride[d]]  over idx in [0, extent)
// The caller passes dims already canonicalised (extent-1 dropped, fusable neighbours fused), sorted by
// input stride (dim 0 = input unit stride).
enum PermuteOp { kPermCopy = 0, kPermScale = 1, kPermAccumulate = 2 };   // =, = alpha*, += alpha*
struct PermuteDesc {
    int rank;
    int64_t extent[kMaxRank];
    int64_t istride[kMaxRank];
    int64_t ostride[kMaxRank];
    const void *in;
    void *out;
    PermuteOp op;
    double alpha_re, alpha_im;
};
// dry_run: only decide whether the shape can be tiled (cudaErrorNotSupported if not) -- nothing is launched
cudaError_t launch_permute(const PermuteDesc &p, cudaStream_t stream, int64_t *launches, bool dry_run = false);

// ---- S6: fused permute-sum -------------------------------------------------------------------------------
constexpr int kMaxTerms = 36;
struct PermSumDesc {
    int rank;
    int64_t extent[kMaxRank];             // of D
    int nterms;
    int64_t xstride[kMaxTerms][kMaxRank]; // stride in X (elements) of D's index k, per term
    double coef_re[kMaxTerms], coef_im[kMaxTerms];
    double beta_re, beta_im;
    const void *X;
    void *D;
};
cudaError_t launch_permsum(const PermSumDesc &p, cudaStream_t stream, int64_t *launches);
// fast path (permsum_orbit.cu): terms that permute three leading indices of equal extent among themselves; *handled =
// false when the call is of another kind
cudaError_t launch_permsum_orbit(const PermSumDesc &p, cudaStream_t stream, int64_t *launches, bool *handled);

// ---- index-permutation-symmetric packed storage (sympack.cu) ---------------------------------
// pack: out[packed linear index] = in[sum_d tab[d][i_d]]  (tab[d]: device table over the values of packed index d)
struct PackDesc {
    int rank;
    int64_t extent[kMaxRank];
    const int64_t *tab[kMaxRank];
    const void *in;
    void *out;
};
cudaError_t launch_pack(const PackDesc &d, cudaStream_t stream, int64_t *launches);
// unpack: out[dense index] (+)= alpha * sign * in[sum_g p(sorted labels of group g) * pstride[g]]
struct UnpackDesc {
    int rank;                       // dense rank
    int64_t extent[kMaxRank];       // dense extents
    int ngroups;                    // = rank of the packed tensor
    int glen[kMaxRank];             // labels per group (1..3)
    int gpos[kMaxRank][3];          // dense positions of the group's labels, in the group's order
    int64_t pstride[kMaxRank];      // stride of the packed index in the packed tensor
    double alpha_re, alpha_im;
    bool accumulate;
    const void *in;
    void *out;
};
cudaError_t launch_unpack(const UnpackDesc &d, cudaStream_t stream, int64_t *launches);
// symmap: both tensors packed.  An element of D fixes a strictly increasing tuple per D index; term t hands the tuple's
// components to the index's labels in the order perm[t]; L is read at the sorted values of its groups' labels:
//   out[e] (+)= alpha * sum_t sign[t] * sortsign * in[sum_g p(sorted labels of L group g) * lstride[g]]
// one identity term: tcb_unpack onto a packed D ("split"); the shuffles of the D groups: tcb_antisym_pack ("merge")
constexpr int kMaxSymTerms = 36;
struct SymTuple { unsigned short v[4]; };   // one strictly increasing tuple (k = 2, 3), first label first
struct SymMapDesc {
    int nd;                                  // rank of D
    int64_t dext[kMaxRank];                  // extents of D (packed)
    int dlen[kMaxRank];                      // labels per D index
    const SymTuple *dtab[kMaxRank];          // device: tuple of packed value i of D index d (nullptr when dlen == 1)
    int nl;                                  // rank of L
    int llen[kMaxRank];
    int lsrc_dim[kMaxRank][3];               // label s of L group g takes its value from D index lsrc_dim, slot lsrc_slot
    int lsrc_slot[kMaxRank][3];
    int64_t lstride[kMaxRank];
    int nterms;
    unsigned char perm[kMaxSymTerms][kMaxRank][3];
    signed char sign[kMaxSymTerms];
    double alpha_re, alpha_im;
    bool accumulate;
    const void *in;
    void *out;
};
cudaError_t launch_symmap(const SymMapDesc &d, cudaStream_t stream, int64_t *launches);

// ---- S7: elementwise --------------------------------------------------------------------------------------
cudaError_t launch_fill(void *D, int64_t n, double re, double im, cudaStream_t stream, int64_t *launches);
cudaError_t launch_scale(void *D, int64_t n, double re, double im, cudaStream_t stream, int64_t *launches);
cudaError_t launch_axpy(void *D, const void *L, int64_t n, double re, double im, bool accumulate,
                        cudaStream_t stream, int64_t *launches);

// D[0] = alpha * sum_i (conj_x ? conj(X[i]) : X[i]) * Y[i]; partial: device, nblocks complex128 (nblocks <= kDotBlocks)
constexpr int kDotBlocks = 1024;      // upper bound of the first-stage grid (4 blocks per SM)
cudaError_t launch_dot(void *D, const void *X, const void *Y, int64_t n, bool conj_x, double re, double im, void *partial,
                       int nblocks, cudaStream_t stream, int64_t *launches);
// The same inner product with its partial sums in a file-scope device array instead of an allocation (dot_noalloc.cu):
// at most kNoAllocMaxElems elements; launches on `stream`; calls that overlap on the GPU race on the array.
constexpr int kNoAllocMaxBlocks = 8192;                                  // partial sums the array holds (131 328 bytes with its header)
constexpr int64_t kNoAllocMaxElems = (int64_t)kNoAllocMaxBlocks * 65536;  // 536 870 912 elements (8.6 GB per operand)
cudaError_t launch_dot_noalloc(void *D, const void *X, const void *Y, int64_t n, bool conj_x, double re, double im,
                               cudaStream_t stream, int64_t *launches);
// T[idx] (+)= alpha * R[idx] / (sum_k eps[eps_at[k] + idx_k]) over the dims with eps_at[k] >= 0 (eps: device doubles)
cudaError_t launch_denominator_update(void *T, const void *R, int rank, const int64_t *extent, const double *eps_dev,
                                      const int *eps_at, double re, double im, bool accumulate, cudaStream_t stream,
                                      int64_t *launches);

// ---- measurement -------------------------------------------------------------------------------------------
cudaError_t run_dmma_peak(double milliseconds, double *tflops, cudaStream_t stream, int64_t *launches);
cudaError_t run_dfma_peak(double milliseconds, double *tflops, cudaStream_t stream, int64_t *launches);

}  // namespace tcb
