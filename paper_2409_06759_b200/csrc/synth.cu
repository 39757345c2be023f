// synth.cu -- device twin of paper_2409_06759_b200/synth.py (seeded input tensors; none of the method's
// arithmetic).  Compiled with -fmad=false: every operation is rounded on its own, exactly as numpy does, so the
// two generators agree bit for bit (tests/test_gpu_synth.py).
#include "../../include/tcb200_synth.h"

#include <cuda_runtime.h>

#include "kernels.h"

// internals of api.cpp that the helper needs
extern "C" int tcbx_internal_stream(tcb_ctx *ctx, void **stream, int64_t **launches);

namespace {

typedef unsigned long long u64;

__device__ __forceinline__ u64 splitmix64(u64 x)
{
    u64 z = x + 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

__constant__ double SIN_C[12] = {0x1.0000000000000p+0, -0x1.5555555555555p-3, 0x1.1111111111111p-7, -0x1.a01a01a01a01ap-13,
                                 0x1.71de3a556c734p-19, -0x1.ae64567f544e4p-26, 0x1.6124613a86d09p-33, -0x1.ae7f3e733b81fp-41,
                                 0x1.952c77030ad4ap-49, -0x1.2f49b46814157p-57, 0x1.71b8ef6dcf572p-66, -0x1.761b413163819p-75};
__constant__ double COS_C[12] = {0x1.0000000000000p+0, -0x1.0000000000000p-1, 0x1.5555555555555p-5, -0x1.6c16c16c16c17p-10,
                                 0x1.a01a01a01a01ap-16, -0x1.27e4fb7789f5cp-22, 0x1.1eed8eff8d898p-29, -0x1.93974a8c07c9dp-37,
                                 0x1.ae7f3e733b81fp-45, -0x1.6827863b97d97p-53, 0x1.e542ba4020225p-62, -0x1.0ce396db7f853p-70};
__constant__ double LOG_C[12] = {0x1.0000000000000p+0, 0x1.5555555555555p-2, 0x1.999999999999ap-3, 0x1.2492492492492p-3,
                                 0x1.c71c71c71c71cp-4, 0x1.745d1745d1746p-4, 0x1.3b13b13b13b14p-4, 0x1.1111111111111p-4,
                                 0x1.e1e1e1e1e1e1ep-5, 0x1.af286bca1af28p-5, 0x1.8618618618618p-5, 0x1.642c8590b2164p-5};

__device__ double ln_unit(u64 k53)
{
    const double x = (double)(k53 + 1ull);
    int e;
    double m = frexp(x, &e);
    if (m < 0x1.6a09e667f3bcdp-1) { m = __dmul_rn(m, 2.0); e -= 1; }
    e -= 53;
    const double s = __ddiv_rn(__dsub_rn(m, 1.0), __dadd_rn(m, 1.0));
    const double s2 = __dmul_rn(s, s);
    double p = LOG_C[11];
#pragma unroll
    for (int k = 10; k >= 0; --k) p = __dadd_rn(__dmul_rn(p, s2), LOG_C[k]);
    const double lnm = __dmul_rn(__dmul_rn(2.0, s), p);
    return __dadd_rn(__dmul_rn((double)e, 0x1.62e42fefa39efp-1), lnm);
}

__device__ void cos_sin_turn(u64 k53, double *c, double *s)
{
    const int q = (int)(k53 >> 51);
    const double frac = __dmul_rn((double)(k53 & ((1ull << 51) - 1ull)), 0x1p-51);
    const double phi = __dmul_rn(frac, 0x1.921fb54442d18p+0);
    const double p2 = __dmul_rn(phi, phi);
    double sp = SIN_C[11], cp = COS_C[11];
#pragma unroll
    for (int k = 10; k >= 0; --k) {
        sp = __dadd_rn(__dmul_rn(sp, p2), SIN_C[k]);
        cp = __dadd_rn(__dmul_rn(cp, p2), COS_C[k]);
    }
    sp = __dmul_rn(sp, phi);
    switch (q) {
    case 0: *c = cp; *s = sp; break;
    case 1: *c = -sp; *s = cp; break;
    case 2: *c = -cp; *s = -sp; break;
    default: *c = sp; *s = -cp; break;
    }
}

__device__ double2 normal_c128(u64 key, u64 idx)
{
    const u64 a = splitmix64(key + 2ull * idx), b = splitmix64(key + 2ull * idx + 1ull);
    const double r = __dsqrt_rn(__dmul_rn(-2.0, ln_unit(a >> 11)));
    double c, s;
    cos_sin_turn(b >> 11, &c, &s);
    return make_double2(__dmul_rn(r, c), __dmul_rn(r, s));
}

struct SynthParams {
    int rank, n_pairs, hermitian;
    int pairs[4];
    long long ext[6], loff[6], lext[6];
    long long n;
    u64 key;
    double sigma;
    double2 *out;
};

__device__ double2 g_at(const SynthParams &p, const long long *ix)
{
    u64 lin = 0, stride = 1;
#pragma unroll
    for (int d = 0; d < 6; ++d) {
        lin += (u64)ix[d] * stride;
        stride *= (u64)p.lext[d];
    }
    return normal_c128(p.key, lin);
}

__device__ double2 antisym_at(const SynthParams &p, const long long *ix)
{
    auto sub = [](double2 a, double2 b) { return make_double2(__dsub_rn(a.x, b.x), __dsub_rn(a.y, b.y)); };
    auto half = [](double2 a) { return make_double2(__dmul_rn(a.x, 0.5), __dmul_rn(a.y, 0.5)); };
    if (p.n_pairs == 0) return g_at(p, ix);
    long long a[6], b[6], c[6];
#pragma unroll
    for (int d = 0; d < 6; ++d) a[d] = b[d] = c[d] = ix[d];
    { const long long t = a[p.pairs[0]]; a[p.pairs[0]] = a[p.pairs[1]]; a[p.pairs[1]] = t; }     // p<->q
    if (p.n_pairs == 1) return half(sub(g_at(p, ix), g_at(p, a)));
    { const long long t = b[p.pairs[2]]; b[p.pairs[2]] = b[p.pairs[3]]; b[p.pairs[3]] = t; }     // r<->s
#pragma unroll
    for (int d = 0; d < 6; ++d) c[d] = a[d];
    { const long long t = c[p.pairs[2]]; c[p.pairs[2]] = c[p.pairs[3]]; c[p.pairs[3]] = t; }     // both
    const double2 t1 = sub(g_at(p, ix), g_at(p, a));
    const double2 t2 = sub(g_at(p, b), g_at(p, c));
    return half(sub(t1, t2));
}

__global__ void __launch_bounds__(256) synth_normal_kernel(const SynthParams p)
{
    for (long long i = blockIdx.x * 256LL + threadIdx.x; i < p.n; i += gridDim.x * 256LL) {
        long long ix[6], rem = i;
#pragma unroll
        for (int d = 0; d < 6; ++d) {
            ix[d] = rem % p.ext[d] + p.loff[d];
            rem /= p.ext[d];
        }
        double2 v = antisym_at(p, ix);
        if (p.hermitian) {
            long long jx[6] = {ix[2], ix[3], ix[0], ix[1], 0, 0};
            const double2 w = antisym_at(p, jx);
            v = make_double2(__dmul_rn(__dadd_rn(v.x, w.x), 0.5), __dmul_rn(__dadd_rn(v.y, -w.y), 0.5));
        }
        if (p.sigma != 1.0) v = make_double2(__dmul_rn(v.x, p.sigma), __dmul_rn(v.y, p.sigma));
        p.out[i] = v;
    }
}

__global__ void __launch_bounds__(256) synth_linear_kernel(double2 *out, long long n)
{
    for (long long i = blockIdx.x * 256LL + threadIdx.x; i < n; i += gridDim.x * 256LL)
        out[i] = make_double2((double)i, __dsub_rn(-(double)i, 0.5));
}

__global__ void __launch_bounds__(256)
synth_mp2_kernel(double2 *T, const double2 *__restrict__ W, const double *__restrict__ eo, const double *__restrict__ ev,
                 long long o, long long v)
{
    const long long n = v * v * o * o;
    for (long long e = blockIdx.x * 256LL + threadIdx.x; e < n; e += gridDim.x * 256LL) {
        const long long a = e % v, b = (e / v) % v, i = (e / (v * v)) % o, j = e / (v * v * o);
        const double den = __dsub_rn(__dadd_rn(eo[i], eo[j]), __dadd_rn(ev[a], ev[b]));
        const double2 w = W[e];
        T[e] = make_double2(__ddiv_rn(w.x, den), __ddiv_rn(w.y, den));
    }
}

int grid_for(long long n)
{
    long long b = (n + 255) / 256;
    if (b > tcb::sm_count() * 16LL) b = tcb::sm_count() * 16LL;
    return b < 1 ? 1 : (int)b;
}

}  // namespace

extern "C" {

int tcbx_synth_normal(tcb_ctx *ctx, tcb_tensor *t, uint64_t seed, uint64_t tensor_id, int n_pairs,
                      const int32_t *pairs, double sigma, int hermitian, const int64_t *label_offset,
                      const int64_t *label_extents)
{
    void *stream;
    int64_t *launches;
    int rc = tcbx_internal_stream(ctx, &stream, &launches);
    if (rc) return rc;
    if (!t || n_pairs < 0 || n_pairs > 2 || (n_pairs && !pairs)) return TCB_EINVAL;
    int rank;
    int64_t ext[TCB_MAX_RANK];
    void *ptr;
    tcb_tensor_info(t, &rank, ext, &ptr);
    if (hermitian && rank != 4) return TCB_EINVAL;
    SynthParams p;
    p.rank = rank; p.n_pairs = n_pairs; p.hermitian = hermitian ? 1 : 0;
    for (int k = 0; k < 4; ++k) p.pairs[k] = k < 2 * n_pairs ? pairs[k] : 0;
    p.n = 1;
    for (int d = 0; d < 6; ++d) {
        p.ext[d] = d < rank ? ext[d] : 1;
        p.loff[d] = (d < rank && label_offset) ? label_offset[d] : 0;
        p.lext[d] = d < rank ? (label_extents ? label_extents[d] : ext[d]) : 1;
        p.n *= p.ext[d];
    }
    // key = splitmix64(seed * M1 + tensor_id), as in synth.py
    {
        unsigned long long x = (unsigned long long)seed * 0x9E3779B97F4A7C15ull + (unsigned long long)tensor_id;
        unsigned long long z = x + 0x9E3779B97F4A7C15ull;
        z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
        z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
        p.key = z ^ (z >> 31);
    }
    p.sigma = sigma;
    p.out = (double2 *)ptr;
    synth_normal_kernel<<<grid_for(p.n), 256, 0, (cudaStream_t)stream>>>(p);
    if (cudaGetLastError() != cudaSuccess) return TCB_ECUDA;
    ++*launches;
    return TCB_OK;
}

int tcbx_synth_index_linear(tcb_ctx *ctx, tcb_tensor *t)
{
    void *stream;
    int64_t *launches;
    int rc = tcbx_internal_stream(ctx, &stream, &launches);
    if (rc) return rc;
    if (!t) return TCB_EINVAL;
    int rank;
    int64_t ext[TCB_MAX_RANK];
    void *ptr;
    tcb_tensor_info(t, &rank, ext, &ptr);
    long long n = 1;
    for (int d = 0; d < rank; ++d) n *= ext[d];
    synth_linear_kernel<<<grid_for(n), 256, 0, (cudaStream_t)stream>>>((double2 *)ptr, n);
    if (cudaGetLastError() != cudaSuccess) return TCB_ECUDA;
    ++*launches;
    return TCB_OK;
}

int tcbx_synth_mp2_amplitudes(tcb_ctx *ctx, tcb_tensor *T, const tcb_tensor *vvoo, const double *eo, int64_t o,
                              const double *ev, int64_t v)
{
    void *stream;
    int64_t *launches;
    int rc = tcbx_internal_stream(ctx, &stream, &launches);
    if (rc) return rc;
    if (!T || !vvoo || !eo || !ev) return TCB_EINVAL;
    int rank;
    int64_t ext[TCB_MAX_RANK];
    void *pT, *pW;
    tcb_tensor_info(T, &rank, ext, &pT);
    if (rank != 4 || ext[0] != v || ext[1] != v || ext[2] != o || ext[3] != o) return TCB_ESHAPE;
    tcb_tensor_info(vvoo, &rank, ext, &pW);
    if (rank != 4 || ext[0] != v || ext[1] != v || ext[2] != o || ext[3] != o) return TCB_ESHAPE;
    double *d_e = nullptr;
    if (cudaMallocAsync((void **)&d_e, (size_t)(o + v) * 8, (cudaStream_t)stream) != cudaSuccess) return TCB_ENOMEM;
    cudaMemcpyAsync(d_e, eo, (size_t)o * 8, cudaMemcpyHostToDevice, (cudaStream_t)stream);
    cudaMemcpyAsync(d_e + o, ev, (size_t)v * 8, cudaMemcpyHostToDevice, (cudaStream_t)stream);
    synth_mp2_kernel<<<grid_for(v * v * o * o), 256, 0, (cudaStream_t)stream>>>((double2 *)pT, (const double2 *)pW,
                                                                                  d_e, d_e + o, o, v);
    cudaError_t e = cudaGetLastError();
    cudaFreeAsync(d_e, (cudaStream_t)stream);
    if (e != cudaSuccess) return TCB_ECUDA;
    ++*launches;
    // eo / ev are pageable host arrays: the copies above have been staged by the time the calls return
    return TCB_OK;
}

}  // extern "C"
