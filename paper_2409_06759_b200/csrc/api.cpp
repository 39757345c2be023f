// api.cpp -- the C ABI of include/tcb200.h: contexts, tensors, argument validation, plan cache, workspace pool,
// and the sequencing of kernels for each call.  Everything a call computes runs in this library's own sm_100a
// kernels; there is no CPU fallback (without a device every compute call returns TCB_ECUDA).
#include "../../include/tcb200.h"

#include <cuda_runtime.h>
#include <nvtx3/nvToolsExt.h>

#include <algorithm>
#include <cstdio>
#include <cstring>
#include <map>
#include <memory>
#include <string>
#include <vector>

#include "kernels.h"
#include "parse.h"
#include "plan.h"

using namespace tcb;

struct CachedPlan {
    ContractPlan plan;
    int64_t *d_tables = nullptr;   // device: offM[M], offN[N], then the GEMV tables or the gather tables of A and B
    const int64_t *d_aux[4] = {nullptr, nullptr, nullptr, nullptr};   // gemv: offAm, offAk, offBk; gemm: gather row/k of A, of B
    // the two TMA descriptors of the GEMM, valid for operands at map_a / map_b (re-encoded when a pointer changes)
    GemmTensorMaps maps;
    const void *map_a = nullptr, *map_b = nullptr;
    bool maps_valid = false;
};

// A lane = one stream with its own workspace (permuted operands, split-K partials, the GEMM's work counters).  Lane 0 is the
// context's stream; independent branches of a call list go to other lanes (tcb_lane_set / tcb_lane_wait).
constexpr int kMaxLanes = 4;
struct Lane {
    cudaStream_t stream = nullptr;
    bool owns_stream = false;
    void *ws = nullptr;
    size_t ws_bytes = 0;
    cudaEvent_t ev = nullptr;        // records "everything enqueued on this lane so far" for tcb_lane_wait
    bool in_capture = false;         // forked into the open capture
};

struct SymTables {
    std::vector<int64_t> host;      // the tables of all packed dims, one after the other
    int64_t *dev = nullptr;
    size_t at[kMaxRank] = {0, 0, 0, 0, 0, 0};
};

struct tcb_ctx {
    int device = 0;
    Lane lanes[kMaxLanes];
    int cur = 0;                     // the lane calls are enqueued on
    uint64_t ws_generation = 0;      // bumped whenever a workspace block is reallocated (captured graphs bake addresses in)
    std::string last_error;
    bool sticky_cuda = false;
    int64_t launches = 0;
    PlanOptions opt;
    std::map<std::string, std::unique_ptr<CachedPlan>> plans;
    std::map<std::string, std::unique_ptr<struct SymTables>> sym_tables;   // tcb_pack offset tables per (spec, extents)
    std::map<std::pair<int64_t, int>, SymTuple *> sym_tuples;              // device: the increasing k-tuples of range(n)
    cudaEvent_t ev0 = nullptr, ev1 = nullptr;
    int64_t live_tensors = 0;
    // per-kernel-class device timing ("kernel_timing" = "on"): event pairs around every launch, summed on query
    bool kernel_timing = false;
    bool capturing = false;                  // between tcb_capture_begin and tcb_capture_end
    bool capture_failed = false;             // a call inside the capture was refused: tcb_capture_end returns no graph
    int64_t capture_l0 = 0;
    struct Span { int cls; cudaEvent_t a, b; double flops, bytes; };
    std::vector<Span> spans;
    std::vector<cudaEvent_t> free_events;
    tcb_kernel_stat acc[4];
};

enum KernelClass { kClsZgemm = 0, kClsPermute = 1, kClsPermsum = 2, kClsElementwise = 3 };

struct tcb_tensor {
    tcb_ctx *ctx = nullptr;
    Shape shape;
    void *ptr = nullptr;
    bool owns = false;
    int64_t elems() const { return shape.volume(); }
};

namespace {

int set_error(tcb_ctx *ctx, int code, const std::string &msg)
{
    if (ctx) ctx->last_error = msg;
    return code;
}

inline cudaStream_t cur_stream(tcb_ctx *ctx) { return ctx->lanes[ctx->cur].stream; }

bool is_capture_error(cudaError_t e)
{
    return e >= cudaErrorStreamCaptureUnsupported && e <= cudaErrorStreamCaptureWrongThread;
}

int cuda_fail(tcb_ctx *ctx, cudaError_t e, const char *where)
{
    if (e == cudaErrorNotSupported) {
        // a launcher refused a shape it cannot tile: decided on the host before anything was enqueued; the context lives on
        cudaGetLastError();
        if (ctx) ctx->last_error = std::string(where) + ": shape not supported by this kernel";
        return TCB_EUNSUPPORTED;
    }
    if (ctx && is_capture_error(e)) {
        // an operation that cannot be recorded was issued inside tcb_capture_begin/end: the capture is lost, the context
        // is not (tcb_capture_end returns TCB_EUNSUPPORTED and the list can be issued call by call)
        cudaGetLastError();
        ctx->capture_failed = true;
        ctx->last_error = std::string(where) + ": " + cudaGetErrorString(e);
        return TCB_EUNSUPPORTED;
    }
    if (ctx) {
        ctx->sticky_cuda = true;
        ctx->last_error = std::string(where) + ": " + cudaGetErrorString(e);
    }
    return TCB_ECUDA;
}

// calls that copy from host memory, synchronise, allocate with cudaMalloc or plan for the first time cannot be recorded
int refuse_in_capture(tcb_ctx *ctx, const char *what)
{
    if (!ctx->capturing) return TCB_OK;
    ctx->capture_failed = true;
    ctx->last_error = std::string(what) + " is not allowed between tcb_capture_begin and tcb_capture_end";
    return TCB_EUNSUPPORTED;
}

struct NvtxRange {                          // one NVTX range per ABI call (tracing)
    explicit NvtxRange(const char *name) { nvtxRangePushA(name); }
    ~NvtxRange() { nvtxRangePop(); }
};

#define TCB_CUDA(ctx, call)                                        \
    do {                                                           \
        cudaError_t e__ = (call);                                  \
        if (e__ != cudaSuccess) return cuda_fail(ctx, e__, #call); \
    } while (0)

int enter(tcb_ctx *ctx)
{
    if (!ctx) return TCB_EINVAL;
    if (ctx->sticky_cuda) return TCB_ECUDA;
    cudaError_t e = cudaSetDevice(ctx->device);
    if (e != cudaSuccess) return cuda_fail(ctx, e, "cudaSetDevice");
    return TCB_OK;
}

size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

constexpr size_t kWsHeader = 8192;      // head of the workspace: persistent work counters (kGemmCounterBytes, see zgemm.cu)
static_assert(kWsHeader >= kGemmCounterBytes, "workspace header too small for the GEMM counters");

int workspace(tcb_ctx *ctx, size_t bytes, void **out)
{
    Lane &ln = ctx->lanes[ctx->cur];
    bytes += kWsHeader;
    if (bytes > ln.ws_bytes) {
        int rc = refuse_in_capture(ctx, "growing the workspace (run the call list once before capturing it)");
        if (rc) return rc;
        TCB_CUDA(ctx, cudaStreamSynchronize(ln.stream));
        if (ln.ws) cudaFree(ln.ws);
        ln.ws = nullptr;
        ln.ws_bytes = 0;
        ++ctx->ws_generation;
        void *p = nullptr;
        const size_t want = align_up(bytes, (size_t)1 << 21);
        cudaError_t e = cudaMalloc(&p, want);
        if (e != cudaSuccess) {
            cudaGetLastError();
            return set_error(ctx, TCB_ENOMEM, "workspace allocation of " + std::to_string(want) + " bytes failed");
        }
        ln.ws = p;
        ln.ws_bytes = want;
        // the first kWsHeader bytes hold the GEMM's work counters: zero once here, every kernel leaves them zero
        TCB_CUDA(ctx, cudaMemsetAsync(p, 0, kWsHeader, ln.stream));
    }
    *out = (char *)ln.ws + kWsHeader;
    return TCB_OK;
}

cudaEvent_t take_event(tcb_ctx *ctx)
{
    cudaEvent_t e = nullptr;
    if (!ctx->free_events.empty()) { e = ctx->free_events.back(); ctx->free_events.pop_back(); }
    else cudaEventCreate(&e);
    return e;
}

// RAII bracket of one kernel-class launch (no-op unless kernel timing is on)
struct TimedLaunch {
    tcb_ctx *ctx;
    tcb_ctx::Span span;
    bool on;
    TimedLaunch(tcb_ctx *c, int cls, double flops, double bytes) : ctx(c), on(c->kernel_timing)
    {
        if (!on) return;
        span.cls = cls; span.flops = flops; span.bytes = bytes;
        span.a = take_event(ctx); span.b = take_event(ctx);
        cudaEventRecord(span.a, cur_stream(ctx));
    }
    ~TimedLaunch()
    {
        if (!on) return;
        cudaEventRecord(span.b, cur_stream(ctx));
        ctx->spans.push_back(span);
    }
};

void fold_spans(tcb_ctx *ctx)
{
    if (ctx->spans.empty()) return;
    for (Lane &ln : ctx->lanes) if (ln.stream) cudaStreamSynchronize(ln.stream);
    for (const tcb_ctx::Span &s : ctx->spans) {
        float ms = 0.f;
        if (cudaEventElapsedTime(&ms, s.a, s.b) == cudaSuccess) {
            tcb_kernel_stat &k = ctx->acc[s.cls];
            k.launches += 1; k.milliseconds += ms; k.flops += s.flops; k.bytes += s.bytes;
        }
        ctx->free_events.push_back(s.a);
        ctx->free_events.push_back(s.b);
    }
    ctx->spans.clear();
}

bool overlaps(const tcb_tensor *a, const tcb_tensor *b)
{
    const char *a0 = (const char *)a->ptr, *a1 = a0 + a->elems() * 16;
    const char *b0 = (const char *)b->ptr, *b1 = b0 + b->elems() * 16;
    return a0 < b1 && b0 < a1;
}

std::string shape_key(const Shape &s)
{
    std::string k = "[";
    for (int i = 0; i < s.rank; ++i) k += std::to_string(s.ext[i]) + ",";
    return k + "]";
}

void strides_of(const Shape &s, int64_t *st)
{
    int64_t x = 1;
    for (int k = 0; k < s.rank; ++k) { st[k] = x; x *= s.ext[k]; }
}

int find_label(const std::vector<std::string> &v, const std::string &n)
{
    for (size_t i = 0; i < v.size(); ++i) if (v[i] == n) return (int)i;
    return -1;
}

bool has_dup(const std::vector<std::string> &v)
{
    for (size_t a = 0; a < v.size(); ++a)
        for (size_t b = a + 1; b < v.size(); ++b)
            if (v[a] == v[b]) return true;
    return false;
}

PermuteDesc make_desc(const PermuteShape &s, const void *in, void *out, PermuteOp op, double ar, double ai)
{
    PermuteDesc d;
    d.rank = s.rank;
    for (int k = 0; k < kMaxRank; ++k) {
        d.extent[k] = k < s.rank ? s.extent[k] : 1;
        d.istride[k] = k < s.rank ? s.istride[k] : 0;
        d.ostride[k] = k < s.rank ? s.ostride[k] : 0;
    }
    d.in = in; d.out = out; d.op = op; d.alpha_re = ar; d.alpha_im = ai;
    return d;
}

int get_plan(tcb_ctx *ctx, const char *expr, const tcb_tensor *D, const tcb_tensor *L, const tcb_tensor *R,
             CachedPlan **out)
{
    std::string key = std::string(expr) + "|" + shape_key(D->shape) + shape_key(L->shape) + shape_key(R->shape) +
                      "|" + std::to_string(ctx->opt.splitk) + "," + std::to_string(ctx->opt.epilogue) + "," +
                      (ctx->opt.permute_always ? "1" : "0") + "," + std::to_string(ctx->opt.operand_loads) + "," +
                      std::to_string(ctx->opt.complex_product);
    auto it = ctx->plans.find(key);
    if (it != ctx->plans.end()) { *out = it->second.get(); return TCB_OK; }
    {
        int rcc = refuse_in_capture(ctx, "planning a contraction for the first time (run the call list once before capturing it)");
        if (rcc) return rcc;
    }
    ParsedExpr e;
    if (!parse_expression(expr, &e)) return set_error(ctx, TCB_EINVAL_EXPR, std::string("cannot parse: ") + expr);
    std::unique_ptr<CachedPlan> cp(new CachedPlan());
    std::string why;
    int rc = plan_contraction(e, D->shape, L->shape, R->shape, ctx->opt, &cp->plan, &why);
    if (rc != TCB_OK) return set_error(ctx, rc, why + ": " + expr);
    const ContractPlan &pl = cp->plan;
    // one device block: offM, offN, then the GEMV tables (offAm, offAk, offBk) or the gather tables (row, k of A; row, k of B).
    // The host vectors live as long as the cache entry, so the stream-ordered copies are safe.
    const std::vector<int64_t> *aux[4] = {&pl.offAm, &pl.offAk, &pl.offBk, nullptr};
    if (!pl.gemv) { aux[0] = &pl.a.gather_row; aux[1] = &pl.a.gather_k; aux[2] = &pl.b.gather_row; aux[3] = &pl.b.gather_k; }
    size_t n = pl.offM.size() + pl.offN.size();
    for (const std::vector<int64_t> *t : aux) if (t) n += t->size();
    TCB_CUDA(ctx, cudaMalloc((void **)&cp->d_tables, n * sizeof(int64_t)));
    size_t at = 0;
    auto put = [&](const std::vector<int64_t> &t) -> cudaError_t {
        cudaError_t e = t.empty() ? cudaSuccess
                                  : cudaMemcpyAsync(cp->d_tables + at, t.data(), t.size() * sizeof(int64_t),
                                                    cudaMemcpyHostToDevice, cur_stream(ctx));
        at += t.size();
        return e;
    };
    TCB_CUDA(ctx, put(pl.offM));
    TCB_CUDA(ctx, put(pl.offN));
    for (int q = 0; q < 4; ++q) {
        if (!aux[q]) continue;
        cp->d_aux[q] = aux[q]->empty() ? nullptr : cp->d_tables + at;
        TCB_CUDA(ctx, put(*aux[q]));
    }
    // the tables were enqueued on the CURRENT lane's stream; the plan may next be used on another lane: wait once, here
    TCB_CUDA(ctx, cudaStreamSynchronize(cur_stream(ctx)));
    *out = cp.get();
    ctx->plans[key] = std::move(cp);
    return TCB_OK;
}

}  // namespace

extern "C" {

const char *tcb_strerror(int code)
{
    switch (code) {
    case TCB_OK: return "ok";
    case TCB_EINVAL_EXPR: return "invalid expression";
    case TCB_ESHAPE: return "rank or extent mismatch";
    case TCB_ERANK: return "rank above 6 or extent below 1";
    case TCB_EALIAS: return "output overlaps an input";
    case TCB_ENOMEM: return "out of device memory";
    case TCB_ECUDA: return "CUDA error";
    case TCB_EUNSUPPORTED: return "unsupported contraction form";
    case TCB_EINVAL: return "invalid argument";
    default: return "unknown error";
    }
}

const char *tcb_last_error(const tcb_ctx *ctx) { return ctx ? ctx->last_error.c_str() : "null context"; }

int64_t tcb_launch_count(const tcb_ctx *ctx) { return ctx ? ctx->launches : 0; }

int tcb_ctx_create(tcb_ctx **out, int device, void *cuda_stream, size_t workspace_bytes)
{
    if (!out) return TCB_EINVAL;
    *out = nullptr;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) {
        cudaGetLastError();
        return TCB_ECUDA;                       // no device: this library has no other way to compute
    }
    if (cudaSetDevice(device) != cudaSuccess) return TCB_ECUDA;
    std::unique_ptr<tcb_ctx> ctx(new tcb_ctx());
    ctx->device = device;
    if (const char *cp_env = getenv("TCB_COMPLEX_PRODUCT")) {          // A/B runs of whole test suites: the context's default
        const std::string v = cp_env;
        ctx->opt.complex_product = v == "3m" ? 2 : v == "4m" ? 1 : 0;
    }
    for (int c = 0; c < 4; ++c) ctx->acc[c] = tcb_kernel_stat{0, 0.0, 0.0, 0.0};
    if (cuda_stream) {
        ctx->lanes[0].stream = (cudaStream_t)cuda_stream;
    } else {
        if (cudaStreamCreateWithFlags(&ctx->lanes[0].stream, cudaStreamNonBlocking) != cudaSuccess) return TCB_ECUDA;
        ctx->lanes[0].owns_stream = true;
    }
    if (cudaEventCreateWithFlags(&ctx->lanes[0].ev, cudaEventDisableTiming) != cudaSuccess) return TCB_ECUDA;
    {   // tensors are created and destroyed every iteration by generated code: keep freed
        // blocks in the stream-ordered pool instead of returning them to the driver at every sync
        cudaMemPool_t pool;
        if (cudaDeviceGetDefaultMemPool(&pool, device) == cudaSuccess) {
            unsigned long long keep = ~0ull;
            cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &keep);
        }
    }
    if (cudaEventCreate(&ctx->ev0) != cudaSuccess || cudaEventCreate(&ctx->ev1) != cudaSuccess) return TCB_ECUDA;
    if (workspace_bytes) {
        void *p;
        int rc = workspace(ctx.get(), workspace_bytes, &p);
        if (rc != TCB_OK) return rc;
    }
    *out = ctx.release();
    return TCB_OK;
}

int tcb_ctx_destroy(tcb_ctx *ctx)
{
    if (!ctx) return TCB_OK;
    cudaSetDevice(ctx->device);
    for (Lane &ln : ctx->lanes) if (ln.stream) cudaStreamSynchronize(ln.stream);
    for (auto &kv : ctx->plans)
        if (kv.second->d_tables) cudaFree(kv.second->d_tables);
    for (auto &kv : ctx->sym_tuples) cudaFree(kv.second);
    for (auto &kv : ctx->sym_tables)
        if (kv.second->dev) cudaFree(kv.second->dev);
    for (Lane &ln : ctx->lanes) if (ln.ws) cudaFree(ln.ws);
    if (ctx->ev0) cudaEventDestroy(ctx->ev0);
    if (ctx->ev1) cudaEventDestroy(ctx->ev1);
    fold_spans(ctx);
    for (cudaEvent_t e : ctx->free_events) cudaEventDestroy(e);
    for (Lane &ln : ctx->lanes) {
        if (ln.ev) cudaEventDestroy(ln.ev);
        if (ln.owns_stream && ln.stream) cudaStreamDestroy(ln.stream);
    }
    delete ctx;
    return TCB_OK;
}

static int apply_option(PlanOptions &opt, const std::string &k, const std::string &v, std::string *why);

int tcb_ctx_set_option(tcb_ctx *ctx, const char *key, const char *value)
{
    if (!ctx || !key || !value) return TCB_EINVAL;
    std::string why;
    if (std::string(key) == "kernel_timing") {
        const std::string v = value;
        if (v != "on" && v != "off") return set_error(ctx, TCB_EINVAL, "kernel_timing: expected on or off");
        ctx->kernel_timing = (v == "on");
        return TCB_OK;
    }
    int rc = apply_option(ctx->opt, key, value, &why);
    return rc ? set_error(ctx, rc, why) : TCB_OK;
}

int tcb_sync(tcb_ctx *ctx)
{
    int rc = enter(ctx);
    if (rc) return rc;
    rc = refuse_in_capture(ctx, "tcb_sync");
    if (rc) return rc;
    for (Lane &ln : ctx->lanes)
        if (ln.stream) TCB_CUDA(ctx, cudaStreamSynchronize(ln.stream));
    return TCB_OK;
}

// ---- lanes: concurrency between independent contractions (DLTC layers; the barrier after every
// tensor operation is the measured serial fraction of PAPER.md:400) --------------------------------------------------------
static int lane_ready(tcb_ctx *ctx, int lane)
{
    Lane &ln = ctx->lanes[lane];
    if (!ln.stream) {
        int rc = refuse_in_capture(ctx, "the first use of a lane (use every lane once before capturing)");
        if (rc) return rc;
        TCB_CUDA(ctx, cudaStreamCreateWithFlags(&ln.stream, cudaStreamNonBlocking));
        ln.owns_stream = true;
        TCB_CUDA(ctx, cudaEventCreateWithFlags(&ln.ev, cudaEventDisableTiming));
    }
    return TCB_OK;
}

// inside a capture a lane joins the graph by depending on the capture's origin (lane 0): done once, at its first use
static int lane_fork_into_capture(tcb_ctx *ctx, int lane)
{
    Lane &ln = ctx->lanes[lane];
    if (!ctx->capturing || lane == 0 || ln.in_capture) return TCB_OK;
    TCB_CUDA(ctx, cudaEventRecord(ctx->lanes[0].ev, ctx->lanes[0].stream));
    TCB_CUDA(ctx, cudaStreamWaitEvent(ln.stream, ctx->lanes[0].ev, 0));
    ln.in_capture = true;
    return TCB_OK;
}

int tcb_lane_count(void) { return kMaxLanes; }

int tcb_lane_set(tcb_ctx *ctx, int lane)
{
    int rc = enter(ctx);
    if (rc) return rc;
    if (lane < 0 || lane >= kMaxLanes) return set_error(ctx, TCB_EINVAL, "lane outside 0..3");
    rc = lane_ready(ctx, lane);
    if (rc) return rc;
    rc = lane_fork_into_capture(ctx, lane);
    if (rc) return rc;
    ctx->cur = lane;
    return TCB_OK;
}

int tcb_lane_wait(tcb_ctx *ctx, int lane, int on_lane)
{
    int rc = enter(ctx);
    if (rc) return rc;
    if (lane < 0 || lane >= kMaxLanes || on_lane < 0 || on_lane >= kMaxLanes)
        return set_error(ctx, TCB_EINVAL, "lane outside 0..3");
    if (lane == on_lane) return TCB_OK;
    rc = lane_ready(ctx, lane);
    if (!rc) rc = lane_ready(ctx, on_lane);
    if (!rc) rc = lane_fork_into_capture(ctx, on_lane);
    if (rc) return rc;
    Lane &a = ctx->lanes[lane], &b = ctx->lanes[on_lane];
    TCB_CUDA(ctx, cudaEventRecord(b.ev, b.stream));
    TCB_CUDA(ctx, cudaStreamWaitEvent(a.stream, b.ev, 0));
    if (ctx->capturing) a.in_capture = true;
    return TCB_OK;
}

// ---- tensors ---------------------------------------------------------------------------------------------

static int make_tensor(tcb_ctx *ctx, tcb_tensor **out, int rank, const int64_t *extents, void *borrowed,
                       bool zero = true)
{
    if (!out) return TCB_EINVAL;
    *out = nullptr;
    int rc = enter(ctx);
    if (rc) return rc;
    if (rank < 0 || rank > TCB_MAX_RANK) return set_error(ctx, TCB_ERANK, "rank outside 0..6");
    if (rank > 0 && !extents) return TCB_EINVAL;
    std::unique_ptr<tcb_tensor> t(new tcb_tensor());
    t->ctx = ctx;
    t->shape.rank = rank;
    for (int k = 0; k < rank; ++k) {
        if (extents[k] < 1) return set_error(ctx, TCB_ERANK, "extent below 1");
        t->shape.ext[k] = extents[k];
    }
    const size_t bytes = (size_t)t->shape.volume() * 16;
    if (borrowed) {
        if (((uintptr_t)borrowed & 15) != 0) return set_error(ctx, TCB_EINVAL, "device pointer not 16-byte aligned");
        t->ptr = borrowed;
        t->owns = false;
    } else {
        void *p = nullptr;
        cudaError_t e = cudaMallocAsync(&p, bytes, cur_stream(ctx));
        if (e != cudaSuccess) {
            cudaGetLastError();
            return set_error(ctx, TCB_ENOMEM, "tensor allocation of " + std::to_string(bytes) + " bytes failed");
        }
        t->ptr = p;
        t->owns = true;
        if (zero) TCB_CUDA(ctx, cudaMemsetAsync(p, 0, bytes, cur_stream(ctx)));
    }
    ++ctx->live_tensors;
    *out = t.release();
    return TCB_OK;
}

int tcb_tensor_create(tcb_ctx *ctx, tcb_tensor **t, int rank, const int64_t *extents)
{
    return make_tensor(ctx, t, rank, extents, nullptr);
}

int tcb_tensor_alloc(tcb_ctx *ctx, tcb_tensor **t, int rank, const int64_t *extents)
{
    return make_tensor(ctx, t, rank, extents, nullptr, false);
}

int tcb_tensor_wrap(tcb_ctx *ctx, tcb_tensor **t, int rank, const int64_t *extents, void *device_ptr)
{
    if (!device_ptr) return TCB_EINVAL;
    return make_tensor(ctx, t, rank, extents, device_ptr);
}

int tcb_tensor_destroy(tcb_tensor *t)
{
    if (!t) return TCB_OK;
    tcb_ctx *ctx = t->ctx;
    if (t->owns && t->ptr) {
        cudaSetDevice(ctx->device);
        cudaFreeAsync(t->ptr, cur_stream(ctx));      // stream-ordered: pending kernels still see the memory
    }
    --ctx->live_tensors;
    delete t;
    return TCB_OK;
}

int tcb_tensor_info(const tcb_tensor *t, int *rank, int64_t extents[TCB_MAX_RANK], void **device_ptr)
{
    if (!t) return TCB_EINVAL;
    if (rank) *rank = t->shape.rank;
    if (extents) for (int k = 0; k < t->shape.rank; ++k) extents[k] = t->shape.ext[k];
    if (device_ptr) *device_ptr = t->ptr;
    return TCB_OK;
}

int tcb_tensor_upload(tcb_ctx *ctx, tcb_tensor *t, const tcb_c128 *host)
{
    int rc = enter(ctx);
    if (rc) return rc;
    if (!t || !host) return TCB_EINVAL;
    rc = refuse_in_capture(ctx, "tcb_tensor_upload");
    if (rc) return rc;
    TCB_CUDA(ctx, cudaMemcpyAsync(t->ptr, host, (size_t)t->elems() * 16, cudaMemcpyHostToDevice, cur_stream(ctx)));
    return TCB_OK;
}

int tcb_tensor_download(tcb_ctx *ctx, const tcb_tensor *t, tcb_c128 *host)
{
    int rc = enter(ctx);
    if (rc) return rc;
    if (!t || !host) return TCB_EINVAL;
    rc = refuse_in_capture(ctx, "tcb_tensor_download");
    if (rc) return rc;
    TCB_CUDA(ctx, cudaMemcpyAsync(host, t->ptr, (size_t)t->elems() * 16, cudaMemcpyDeviceToHost, cur_stream(ctx)));
    TCB_CUDA(ctx, cudaStreamSynchronize(cur_stream(ctx)));
    return TCB_OK;
}

int tcb_tensor_fill(tcb_ctx *ctx, tcb_tensor *t, tcb_c128 value)
{
    NvtxRange nvtx_range("tcb_tensor_fill");
    int rc = enter(ctx);
    if (rc) return rc;
    if (!t) return TCB_EINVAL;
    TimedLaunch tl(ctx, kClsElementwise, 0.0, 16.0 * (double)t->elems());
    TCB_CUDA(ctx, launch_fill(t->ptr, t->elems(), value.re, value.im, cur_stream(ctx), &ctx->launches));
    return TCB_OK;
}

// ---- hot path --------------------------------------------------------------------------------------------

int tcb_contract(tcb_ctx *ctx, const char *expr, tcb_tensor *D, const tcb_tensor *L, const tcb_tensor *R,
                 tcb_c128 alpha)
{
    NvtxRange nvtx_range("tcb_contract");
    int rc = enter(ctx);
    if (rc) return rc;
    if (!expr || !D || !L || !R) return set_error(ctx, TCB_EINVAL, "null argument");
    if (overlaps(D, L) || overlaps(D, R)) return set_error(ctx, TCB_EALIAS, "D overlaps L or R");
    CachedPlan *cp = nullptr;
    rc = get_plan(ctx, expr, D, L, R, &cp);
    if (rc) return rc;
    const ContractPlan &P = cp->plan;
    const tcb_tensor *TA = P.swapped ? R : L, *TB = P.swapped ? L : R;
    if (P.gemv) {
        const size_t bytesPg = align_up(P.partial_bytes, 1024);
        void *wsg = nullptr;
        if (bytesPg) {
            rc = workspace(ctx, bytesPg, &wsg);
            if (rc) return rc;
        }
        GemvDesc g;
        g.M = P.M; g.K = P.K;
        g.A = TA->ptr; g.B = TB->ptr; g.D = D->ptr;
        g.offD = cp->d_tables;
        g.offAm = cp->d_tables + P.offM.size() + P.offN.size();
        g.offAk = g.offAm + P.offAm.size();
        g.offBk = g.offAk + P.offAk.size();
        g.kfast = P.gemv_kfast;
        g.alpha_re = alpha.re; g.alpha_im = alpha.im;
        g.accumulate = P.accumulate;
        g.partial = wsg;
        TimedLaunch tl(ctx, kClsZgemm, P.flops, P.bytes);
        TCB_CUDA(ctx, launch_gemv(g, cur_stream(ctx), &ctx->launches));
        return TCB_OK;
    }

    if (P.outer) {
        OuterDesc g;
        g.M = P.M; g.N = P.N;
        g.A = TA->ptr; g.B = TB->ptr; g.D = D->ptr;
        g.offM = cp->d_tables;
        g.offN = cp->d_tables + P.offM.size();
        g.rowA = cp->d_aux[0]; g.rowB = cp->d_aux[2];
        g.alpha_re = alpha.re; g.alpha_im = alpha.im;
        g.accumulate = P.accumulate;
        TimedLaunch tl(ctx, kClsZgemm, P.flops, P.bytes);
        TCB_CUDA(ctx, launch_outer(g, cur_stream(ctx), &ctx->launches));
        return TCB_OK;
    }
    const size_t bytesA = P.a.permuted ? align_up((size_t)P.a.elems * 16, 1024) : 0;
    const size_t bytesB = P.b.permuted ? align_up((size_t)P.b.elems * 16, 1024) : 0;
    const size_t bytesP = align_up(P.partial_bytes, 1024);
    const size_t bytesC = P.twopass ? align_up((size_t)P.M * (size_t)P.N * 16, 1024) : 0;
    // everything that can refuse is decided before the first launch (on an error return nothing has been enqueued)
    PermuteDesc dA, dB, dC;
    if (P.a.permuted) {
        dA = make_desc(P.a.perm, TA->ptr, nullptr, kPermCopy, 1.0, 0.0);
        TCB_CUDA(ctx, launch_permute(dA, nullptr, nullptr, true));
    }
    if (P.b.permuted) {
        dB = make_desc(P.b.perm, TB->ptr, nullptr, kPermCopy, 1.0, 0.0);
        TCB_CUDA(ctx, launch_permute(dB, nullptr, nullptr, true));
    }
    if (P.twopass) {
        dC = make_desc(P.c_perm, nullptr, D->ptr, P.accumulate ? kPermAccumulate : kPermScale, alpha.re, alpha.im);
        TCB_CUDA(ctx, launch_permute(dC, nullptr, nullptr, true));
    }
    char *ws = nullptr;
    {
        void *p;
        rc = workspace(ctx, bytesA + bytesB + bytesP + bytesC, &p);
        if (rc) return rc;
        ws = (char *)p;
    }
    const void *Aptr = TA->ptr, *Bptr = TB->ptr;
    if (P.a.permuted) {
        dA.out = ws;
        TimedLaunch tl(ctx, kClsPermute, 0.0, 32.0 * (double)P.a.elems);
        TCB_CUDA(ctx, launch_permute(dA, cur_stream(ctx), &ctx->launches));
        Aptr = ws;
    }
    if (P.b.permuted) {
        dB.out = ws + bytesA;
        TimedLaunch tl(ctx, kClsPermute, 0.0, 32.0 * (double)P.b.elems);
        TCB_CUDA(ctx, launch_permute(dB, cur_stream(ctx), &ctx->launches));
        Bptr = ws + bytesA;
    }
    char *Cws = ws + bytesA + bytesB + bytesP;
    GemmDesc g;
    g.M = P.M; g.N = P.N; g.K = P.K;
    g.A = Aptr; g.B = Bptr;
    g.lda = P.a.ld; g.ldb = P.b.ld;
    g.a_kmajor = P.a.kmajor; g.b_kmajor = P.b.kmajor;
    if (P.a.gather) { g.gatherAm = cp->d_aux[0]; g.gatherAk = cp->d_aux[1]; g.a_mfast = P.a.mfast; }
    if (P.b.gather) { g.gatherBn = cp->d_aux[2]; g.gatherBk = cp->d_aux[3]; g.b_mfast = P.b.mfast; }
    g.D = P.twopass ? (void *)Cws : D->ptr;
    g.offM = cp->d_tables;
    g.offN = cp->d_tables + P.offM.size();
    g.alpha_re = P.twopass ? 1.0 : alpha.re; g.alpha_im = P.twopass ? 0.0 : alpha.im;
    g.accumulate = P.twopass ? false : P.accumulate;
    g.splitk = P.splitk;
    g.m3 = P.m3;
    g.partial = bytesP ? ws + bytesA + bytesB : nullptr;
    g.counters = ctx->opt.static_deal ? nullptr : ctx->lanes[ctx->cur].ws;      // the workspace header
    // the two TMA descriptors are kept beside the plan: re-encoded only when an operand sits somewhere else
    if (!cp->maps_valid || cp->map_a != Aptr || cp->map_b != Bptr) {
        TCB_CUDA(ctx, encode_gemm_maps(g, &cp->maps));
        cp->map_a = Aptr; cp->map_b = Bptr; cp->maps_valid = true;
    }
    {
        TimedLaunch tl(ctx, kClsZgemm, P.flops, P.bytes);
        TCB_CUDA(ctx, launch_zgemm_with_maps(g, cp->maps, cur_stream(ctx), &ctx->launches));
    }
    if (P.twopass) {
        dC.in = Cws;
        TimedLaunch tl(ctx, kClsPermute, 0.0, 16.0 * (double)P.M * (double)P.N * (P.accumulate ? 3.0 : 2.0));
        TCB_CUDA(ctx, launch_permute(dC, cur_stream(ctx), &ctx->launches));
    }
    return TCB_OK;
}

int tcb_plan_describe(tcb_ctx *ctx, const char *expr, const tcb_tensor *D, const tcb_tensor *L,
                      const tcb_tensor *R, char *buf, size_t buflen)
{
    int rc = enter(ctx);
    if (rc) return rc;
    if (!expr || !D || !L || !R || !buf || !buflen) return TCB_EINVAL;
    CachedPlan *cp = nullptr;
    rc = get_plan(ctx, expr, D, L, R, &cp);
    if (rc) return rc;
    const std::string s = cp->plan.describe();
    std::snprintf(buf, buflen, "%s", s.c_str());
    return TCB_OK;
}

static int apply_option(PlanOptions &opt, const std::string &k, const std::string &v, std::string *why)
{
    if (k == "splitk") {
        if (v == "auto") opt.splitk = 0;
        else if (v == "off") opt.splitk = 1;
        else {
            const int n = atoi(v.c_str());
            if (n < 1) { *why = "splitk: expected auto, off or a positive integer"; return TCB_EINVAL; }
            opt.splitk = n;
        }
        return TCB_OK;
    }
    if (k == "epilogue") {
        if (v == "auto") opt.epilogue = 0;
        else if (v == "fused") opt.epilogue = 1;
        else if (v == "twopass") opt.epilogue = 2;
        else { *why = "epilogue: expected auto, fused or twopass"; return TCB_EINVAL; }
        return TCB_OK;
    }
    if (k == "permute_operands") {
        if (v == "auto") opt.permute_always = false;
        else if (v == "always") opt.permute_always = true;
        else { *why = "permute_operands: expected auto or always"; return TCB_EINVAL; }
        return TCB_OK;
    }
    if (k == "operand_loads") {
        if (v == "auto") opt.operand_loads = 0;
        else if (v == "gather") opt.operand_loads = 1;
        else if (v == "permute") opt.operand_loads = 2;
        else { *why = "operand_loads: expected auto, gather or permute"; return TCB_EINVAL; }
        return TCB_OK;
    }
    if (k == "complex_product") {
        if (v == "auto") opt.complex_product = 0;
        else if (v == "4m") opt.complex_product = 1;
        else if (v == "3m") opt.complex_product = 2;
        else { *why = "complex_product: expected auto, 4m or 3m"; return TCB_EINVAL; }
        return TCB_OK;
    }
    if (k == "gemm_deal") {
        if (v == "dynamic") opt.static_deal = false;
        else if (v == "static") opt.static_deal = true;
        else { *why = "gemm_deal: expected dynamic or static"; return TCB_EINVAL; }
        return TCB_OK;
    }
    *why = "unknown option " + k;
    return TCB_EINVAL;
}

int tcb_plan_describe_host(const char *expr, int rank_d, const int64_t *ext_d, int rank_l, const int64_t *ext_l,
                           int rank_r, const int64_t *ext_r, const char *options, char *buf, size_t buflen,
                           int64_t *offM, size_t cap_m, int64_t *offN, size_t cap_n)
{
    if (!expr || !buf || !buflen) return TCB_EINVAL;
    Shape sh[3];
    const int ranks[3] = {rank_d, rank_l, rank_r};
    const int64_t *exts[3] = {ext_d, ext_l, ext_r};
    for (int t = 0; t < 3; ++t) {
        if (ranks[t] < 0 || ranks[t] > TCB_MAX_RANK) return TCB_ERANK;
        sh[t].rank = ranks[t];
        for (int k = 0; k < ranks[t]; ++k) {
            if (!exts[t] || exts[t][k] < 1) return TCB_ERANK;
            sh[t].ext[k] = exts[t][k];
        }
    }
    PlanOptions opt;
    std::string why;
    if (options) {
        std::string o = options;
        size_t pos = 0;
        while (pos < o.size()) {
            size_t end = o.find(';', pos);
            if (end == std::string::npos) end = o.size();
            const std::string kv = o.substr(pos, end - pos);
            pos = end + 1;
            if (kv.empty()) continue;
            const size_t eq = kv.find('=');
            if (eq == std::string::npos) return TCB_EINVAL;
            int rc = apply_option(opt, kv.substr(0, eq), kv.substr(eq + 1), &why);
            if (rc) { std::snprintf(buf, buflen, "%s", why.c_str()); return rc; }
        }
    }
    ParsedExpr e;
    if (!parse_expression(expr, &e)) { std::snprintf(buf, buflen, "cannot parse"); return TCB_EINVAL_EXPR; }
    ContractPlan P;
    int rc = plan_contraction(e, sh[0], sh[1], sh[2], opt, &P, &why);
    if (rc) { std::snprintf(buf, buflen, "%s", why.c_str()); return rc; }
    std::snprintf(buf, buflen, "%s", P.describe().c_str());
    if (offM) {
        if (cap_m < P.offM.size()) return TCB_EINVAL;
        std::memcpy(offM, P.offM.data(), P.offM.size() * sizeof(int64_t));
    }
    if (offN) {
        if (cap_n < P.offN.size()) return TCB_EINVAL;
        std::memcpy(offN, P.offN.data(), P.offN.size() * sizeof(int64_t));
    }
    return TCB_OK;
}

// shared by tcb_add and tcb_permute
static int permuted_op(tcb_ctx *ctx, const char *expr, tcb_tensor *D, const tcb_tensor *L, tcb_c128 alpha,
                       bool pure_copy)
{
    NvtxRange nvtx_range(pure_copy ? "tcb_permute" : "tcb_add");
    int rc = enter(ctx);
    if (rc) return rc;
    if (!expr || !D || !L) return set_error(ctx, TCB_EINVAL, "null argument");
    ParsedExpr e;
    if (!parse_expression(expr, &e) || e.has_r)
        return set_error(ctx, TCB_EINVAL_EXPR, std::string("cannot parse as D(..)(+)=L(..): ") + expr);
    if (pure_copy && e.accumulate) return set_error(ctx, TCB_EINVAL_EXPR, "tcb_permute takes '=', not '+='");
    if ((int)e.d.size() != D->shape.rank || (int)e.l.size() != L->shape.rank || D->shape.rank != L->shape.rank)
        return set_error(ctx, TCB_ESHAPE, "rank mismatch");
    if (has_dup(e.d) || has_dup(e.l)) return set_error(ctx, TCB_EUNSUPPORTED, "label repeated inside one tensor");
    int64_t sD[kMaxRank], sL[kMaxRank], ext[kMaxRank], is[kMaxRank], os[kMaxRank];
    strides_of(D->shape, sD);
    strides_of(L->shape, sL);
    const int r = L->shape.rank;
    for (int k = 0; k < r; ++k) {
        const int pd = find_label(e.d, e.l[k]);
        if (pd < 0) return set_error(ctx, TCB_EUNSUPPORTED, "label of L missing in D");
        if (D->shape.ext[pd] != L->shape.ext[k]) return set_error(ctx, TCB_ESHAPE, "extent mismatch");
        ext[k] = L->shape.ext[k]; is[k] = sL[k]; os[k] = sD[pd];
    }
    if (overlaps(D, L)) return set_error(ctx, TCB_EALIAS, "D overlaps L");
    const PermuteShape ps = canonical_permutation(r, ext, is, os);
    const double n16 = 16.0 * (double)D->elems();
    if (pure_copy) {
        TimedLaunch tl(ctx, kClsPermute, 0.0, 2 * n16);
        PermuteDesc d = make_desc(ps, L->ptr, D->ptr, kPermCopy, 1.0, 0.0);
        TCB_CUDA(ctx, launch_permute(d, cur_stream(ctx), &ctx->launches));
    } else if (ps.identity) {
        TimedLaunch tl(ctx, kClsElementwise, 0.0, (e.accumulate ? 3 : 2) * n16);
        TCB_CUDA(ctx, launch_axpy(D->ptr, L->ptr, D->elems(), alpha.re, alpha.im, e.accumulate, cur_stream(ctx),
                                  &ctx->launches));
    } else {
        TimedLaunch tl(ctx, kClsPermute, 0.0, (e.accumulate ? 3 : 2) * n16);
        PermuteDesc d = make_desc(ps, L->ptr, D->ptr, e.accumulate ? kPermAccumulate : kPermScale, alpha.re, alpha.im);
        TCB_CUDA(ctx, launch_permute(d, cur_stream(ctx), &ctx->launches));
    }
    return TCB_OK;
}

int tcb_add(tcb_ctx *ctx, const char *expr, tcb_tensor *D, const tcb_tensor *L, tcb_c128 alpha)
{
    return permuted_op(ctx, expr, D, L, alpha, false);
}

int tcb_permute(tcb_ctx *ctx, const char *expr, tcb_tensor *D, const tcb_tensor *L)
{
    tcb_c128 one = {1.0, 0.0};
    return permuted_op(ctx, expr, D, L, one, true);
}

int tcb_scale(tcb_ctx *ctx, tcb_tensor *D, tcb_c128 alpha)
{
    NvtxRange nvtx_range("tcb_scale");
    int rc = enter(ctx);
    if (rc) return rc;
    if (!D) return TCB_EINVAL;
    TimedLaunch tl(ctx, kClsElementwise, 0.0, 32.0 * (double)D->elems());
    TCB_CUDA(ctx, launch_scale(D->ptr, D->elems(), alpha.re, alpha.im, cur_stream(ctx), &ctx->launches));
    return TCB_OK;
}

int tcb_dot(tcb_ctx *ctx, tcb_tensor *D, const tcb_tensor *X, const tcb_tensor *Y, int conjugate_x, tcb_c128 alpha)
{
    NvtxRange nvtx_range("tcb_dot");
    int rc = enter(ctx);
    if (rc) return rc;
    if (!D || !X || !Y) return set_error(ctx, TCB_EINVAL, "null argument");
    if (D->shape.rank != 0) return set_error(ctx, TCB_ESHAPE, "D must have rank 0");
    if (X->shape.rank != Y->shape.rank) return set_error(ctx, TCB_ESHAPE, "rank mismatch");
    for (int k = 0; k < X->shape.rank; ++k)
        if (X->shape.ext[k] != Y->shape.ext[k]) return set_error(ctx, TCB_ESHAPE, "X and Y differ in shape");
    if (overlaps(D, X) || overlaps(D, Y)) return set_error(ctx, TCB_EALIAS, "D overlaps X or Y");
    const int64_t n = X->elems();
    const int nblocks = (int)std::max<int64_t>(1, std::min<int64_t>(std::min(kDotBlocks, 4 * sm_count()), (n + 255) / 256));
    void *partial = nullptr;
    TCB_CUDA(ctx, cudaMallocAsync(&partial, (size_t)nblocks * 16, cur_stream(ctx)));
    cudaError_t e;
    {
        TimedLaunch tl(ctx, kClsElementwise, 8.0 * (double)n, 32.0 * (double)n);
        e = launch_dot(D->ptr, X->ptr, Y->ptr, n, conjugate_x != 0, alpha.re, alpha.im, partial, nblocks, cur_stream(ctx),
                       &ctx->launches);
    }
    cudaFreeAsync(partial, cur_stream(ctx));
    TCB_CUDA(ctx, e);
    return TCB_OK;
}

static_assert(TCB_DOT_NOALLOC_MAX_ELEMS == kNoAllocMaxElems, "the header states the limit of dot_noalloc.cu");

int tcb_dot_noalloc(tcb_ctx *ctx, tcb_tensor *D, const tcb_tensor *X, const tcb_tensor *Y, int conjugate_x, tcb_c128 alpha)
{
    NvtxRange nvtx_range("tcb_dot_noalloc");
    int rc = enter(ctx);
    if (rc) return rc;
    if (!D || !X || !Y) return set_error(ctx, TCB_EINVAL, "null argument");
    if (D->shape.rank != 0) return set_error(ctx, TCB_ESHAPE, "D must have rank 0");
    if (X->shape.rank != Y->shape.rank) return set_error(ctx, TCB_ESHAPE, "rank mismatch");
    for (int k = 0; k < X->shape.rank; ++k)
        if (X->shape.ext[k] != Y->shape.ext[k]) return set_error(ctx, TCB_ESHAPE, "X and Y differ in shape");
    if (overlaps(D, X) || overlaps(D, Y)) return set_error(ctx, TCB_EALIAS, "D overlaps X or Y");
    const int64_t n = X->elems();
    if (n > kNoAllocMaxElems)
        return set_error(ctx, TCB_EUNSUPPORTED, "tcb_dot_noalloc: " + std::to_string(n) + " elements exceed the fixed scratch array's " +
                                                    std::to_string(kNoAllocMaxElems) + " (TCB_DOT_NOALLOC_MAX_ELEMS); use tcb_dot");
    TimedLaunch tl(ctx, kClsElementwise, 8.0 * (double)n, 32.0 * (double)n);
    TCB_CUDA(ctx, launch_dot_noalloc(D->ptr, X->ptr, Y->ptr, n, conjugate_x != 0, alpha.re, alpha.im, cur_stream(ctx), &ctx->launches));
    return TCB_OK;
}

static int denominator_op(tcb_ctx *ctx, tcb_tensor *T, const tcb_tensor *R, const double *const *eps, tcb_c128 alpha,
                          bool accumulate)
{
    NvtxRange nvtx_range("tcb_denominator_update/divide");
    int rc = enter(ctx);
    if (rc) return rc;
    if (!T || !R || !eps) return set_error(ctx, TCB_EINVAL, "null argument");
    rc = refuse_in_capture(ctx, "tcb_denominator_update / tcb_denominator_divide (they copy the energies from host memory)");
    if (rc) return rc;
    const int r = T->shape.rank;
    if (R->shape.rank != r) return set_error(ctx, TCB_ESHAPE, "rank mismatch");
    for (int k = 0; k < r; ++k)
        if (R->shape.ext[k] != T->shape.ext[k]) return set_error(ctx, TCB_ESHAPE, "T and R differ in shape");
    if (overlaps(T, R)) return set_error(ctx, TCB_EALIAS, "T overlaps R");
    std::vector<double> host;
    int at[kMaxRank];
    bool any = false;
    for (int k = 0; k < kMaxRank; ++k) {
        at[k] = -1;
        if (k < r && eps[k]) {
            at[k] = (int)host.size();
            host.insert(host.end(), eps[k], eps[k] + T->shape.ext[k]);
            any = true;
        }
    }
    if (!any) return set_error(ctx, TCB_EINVAL, "no index carries orbital energies: the denominator would be zero");
    // the energies travel with the call: a few hundred doubles, stream-ordered allocation (pageable source: the copy
    // is staged before cudaMemcpyAsync returns)
    double *dev = nullptr;
    TCB_CUDA(ctx, cudaMallocAsync((void **)&dev, host.size() * sizeof(double), cur_stream(ctx)));
    cudaError_t e = cudaMemcpyAsync(dev, host.data(), host.size() * sizeof(double), cudaMemcpyHostToDevice, cur_stream(ctx));
    if (e == cudaSuccess) {
        TimedLaunch tl(ctx, kClsElementwise, 0.0, (accumulate ? 48.0 : 32.0) * (double)T->elems());
        e = launch_denominator_update(T->ptr, R->ptr, r, T->shape.ext, dev, at, alpha.re, alpha.im, accumulate,
                                      cur_stream(ctx), &ctx->launches);
    }
    cudaFreeAsync(dev, cur_stream(ctx));
    TCB_CUDA(ctx, e);
    return TCB_OK;
}

int tcb_denominator_update(tcb_ctx *ctx, tcb_tensor *T, const tcb_tensor *R, const double *const *eps, tcb_c128 alpha)
{
    return denominator_op(ctx, T, R, eps, alpha, true);
}

int tcb_denominator_divide(tcb_ctx *ctx, tcb_tensor *T, const tcb_tensor *R, const double *const *eps, tcb_c128 alpha)
{
    return denominator_op(ctx, T, R, eps, alpha, false);
}

int tcb_permsum(tcb_ctx *ctx, tcb_tensor *D, const tcb_tensor *X, int nterms, const int32_t *perms,
                const tcb_c128 *coefs, tcb_c128 beta)
{
    NvtxRange nvtx_range("tcb_permsum");
    int rc = enter(ctx);
    if (rc) return rc;
    if (!D || !X || !perms || !coefs) return set_error(ctx, TCB_EINVAL, "null argument");
    if (nterms < 1 || nterms > kMaxTerms) return set_error(ctx, TCB_EINVAL, "nterms outside 1..36");
    const int r = D->shape.rank;
    if (X->shape.rank != r) return set_error(ctx, TCB_ESHAPE, "rank mismatch");
    int64_t sX[kMaxRank];
    strides_of(X->shape, sX);
    PermSumDesc d;
    d.rank = r;
    d.nterms = nterms;
    for (int k = 0; k < kMaxRank; ++k) d.extent[k] = k < r ? D->shape.ext[k] : 1;
    for (int t = 0; t < nterms; ++t) {
        bool seen[kMaxRank] = {false, false, false, false, false, false};
        for (int k = 0; k < kMaxRank; ++k) d.xstride[t][k] = 0;
        for (int m = 0; m < r; ++m) {
            const int s = perms[t * r + m];          // position m of X is indexed by D's index s
            if (s < 0 || s >= r || seen[s]) return set_error(ctx, TCB_EINVAL, "perms is not a permutation table");
            seen[s] = true;
            if (X->shape.ext[m] != D->shape.ext[s]) return set_error(ctx, TCB_ESHAPE, "extent mismatch under a term");
            d.xstride[t][s] = sX[m];
        }
        d.coef_re[t] = coefs[t].re;
        d.coef_im[t] = coefs[t].im;
    }
    if (overlaps(D, X)) return set_error(ctx, TCB_EALIAS, "D overlaps X");
    d.beta_re = beta.re; d.beta_im = beta.im;
    d.X = X->ptr; d.D = D->ptr;
    const bool reads_d = !(beta.re == 0.0 && beta.im == 0.0);
    TimedLaunch tl(ctx, kClsPermsum, 0.0, 16.0 * (double)D->elems() * (reads_d ? 3.0 : 2.0));
    TCB_CUDA(ctx, launch_permsum(d, cur_stream(ctx), &ctx->launches));
    return TCB_OK;
}

int tcb_antisymmetrize(tcb_ctx *ctx, const char *spec, tcb_tensor *D, const tcb_tensor *X, tcb_c128 alpha)
{
    NvtxRange nvtx_range("tcb_antisymmetrize");
    int rc = enter(ctx);
    if (rc) return rc;
    if (!spec || !D || !X) return set_error(ctx, TCB_EINVAL, "null argument");
    std::vector<PermOperator> ops;
    ParsedExpr e;
    if (!parse_antisym_spec(spec, &ops, &e)) return set_error(ctx, TCB_EINVAL_EXPR, std::string("cannot parse: ") + spec);
    const int r = D->shape.rank;
    if ((int)e.d.size() != r || (int)e.l.size() != r || X->shape.rank != r)
        return set_error(ctx, TCB_ESHAPE, "rank mismatch");
    if (has_dup(e.d) || has_dup(e.l)) return set_error(ctx, TCB_EUNSUPPORTED, "label repeated inside one tensor");
    // operators must act on disjoint label sets (they then commute; all CC operators do)
    std::vector<std::string> used;
    for (const PermOperator &op : ops) {
        std::vector<std::string> mine = op.others;
        mine.push_back(op.pivot);
        for (const std::string &s : mine) {
            if (find_label(e.d, s) < 0) return set_error(ctx, TCB_EINVAL_EXPR, "operator label " + s + " not in D");
            if (find_label(used, s) >= 0) return set_error(ctx, TCB_EUNSUPPORTED, "operators share label " + s);
            used.push_back(s);
        }
    }
    // expand the product, first operator outermost
    struct Term { std::vector<std::string> xl; double sign; };
    std::vector<Term> terms = {{e.l, 1.0}};
    for (const PermOperator &op : ops) {
        std::vector<Term> next;
        for (const Term &t : terms) {
            next.push_back(t);
            for (const std::string &o : op.others) {
                Term s = t;
                for (std::string &lab : s.xl) {
                    if (lab == op.pivot) lab = o;
                    else if (lab == o) lab = op.pivot;
                }
                s.sign = -t.sign;
                next.push_back(s);
            }
        }
        terms.swap(next);
    }
    if ((int)terms.size() > kMaxTerms) return set_error(ctx, TCB_EUNSUPPORTED, "more than 36 terms");
    std::vector<int32_t> perms(terms.size() * (size_t)std::max(r, 1));
    std::vector<tcb_c128> coefs(terms.size());
    for (size_t t = 0; t < terms.size(); ++t) {
        for (int m = 0; m < r; ++m) {
            const int s = find_label(e.d, terms[t].xl[m]);
            if (s < 0) return set_error(ctx, TCB_EUNSUPPORTED, "label of X missing in D");
            perms[t * r + m] = s;
        }
        coefs[t].re = alpha.re * terms[t].sign;
        coefs[t].im = alpha.im * terms[t].sign;
    }
    tcb_c128 beta = {e.accumulate ? 1.0 : 0.0, 0.0};
    return tcb_permsum(ctx, D, X, (int)terms.size(), perms.data(), coefs.data(), beta);
}

// ---- index-permutation-symmetric packed storage ------------------------------------------------------------
namespace {

int64_t choose(int64_t n, int k)
{
    if (k == 1) return n;
    if (k == 2) return n * (n - 1) / 2;
    return n * (n - 1) * (n - 2) / 6;
}

// validates a pack / unpack spec against the two handles; dense_pos[g][s] = position in the dense tensor of label s of group g
int bind_sym_spec(tcb_ctx *ctx, const std::vector<std::vector<std::string>> &packed, const std::vector<std::vector<std::string>> &dense,
                  const tcb_tensor *P, const tcb_tensor *Dn, int dense_pos[kMaxRank][3])
{
    if ((int)packed.size() != P->shape.rank || (int)dense.size() != Dn->shape.rank)
        return set_error(ctx, TCB_ESHAPE, "rank of a handle differs from the spec");
    std::vector<std::string> dl;
    for (const auto &g : dense) {
        if (g.size() != 1) return set_error(ctx, TCB_EINVAL_EXPR, "a<b groups on both sides");
        dl.push_back(g[0]);
    }
    if (has_dup(dl)) return set_error(ctx, TCB_EUNSUPPORTED, "label repeated inside the dense tensor");
    size_t used = 0;
    bool any_group = false;
    for (size_t g = 0; g < packed.size(); ++g) {
        const auto &grp = packed[g];
        if (grp.size() > 3) return set_error(ctx, TCB_EUNSUPPORTED, "groups of more than three labels");
        any_group = any_group || grp.size() > 1;
        int64_t n = -1;
        for (size_t s = 0; s < grp.size(); ++s) {
            const int pos = find_label(dl, grp[s]);
            if (pos < 0) return set_error(ctx, TCB_EINVAL_EXPR, "label " + grp[s] + " missing in the dense tensor");
            for (size_t g2 = 0; g2 <= g; ++g2)
                for (size_t s2 = 0; s2 < (g2 == g ? s : packed[g2].size()); ++s2)
                    if (packed[g2][s2] == grp[s]) return set_error(ctx, TCB_EUNSUPPORTED, "label repeated inside the packed tensor");
            dense_pos[g][s] = pos;
            if (n >= 0 && Dn->shape.ext[pos] != n) return set_error(ctx, TCB_ESHAPE, "labels of one group differ in extent");
            n = Dn->shape.ext[pos];
            ++used;
        }
        if (P->shape.ext[g] != choose(n, (int)grp.size()))
            return set_error(ctx, TCB_ESHAPE, "packed extent is not n(n-1)/2 (n(n-1)(n-2)/6) of the group's dense extent");
    }
    if (used != dl.size()) return set_error(ctx, TCB_EINVAL_EXPR, "a dense label is missing in the packed tensor");
    if (!any_group) return set_error(ctx, TCB_EINVAL_EXPR, "no a<b group in the spec (use tcb_permute)");
    return TCB_OK;
}


// inverse of choose: the n with choose(n, k) == e, or -1
int64_t unchoose(int64_t e, int k)
{
    for (int64_t n = k; n < 70000; ++n) {
        const int64_t c = choose(n, k);
        if (c == e) return n;
        if (c > e) break;
    }
    return -1;
}

// A spec with a<b groups on BOTH sides: labels, their extents, and which (index, slot) of each side a label sits in.
struct SymBinding {
    std::vector<std::string> labels;
    std::vector<int64_t> ext;
    std::vector<std::vector<int>> dg, lg;         // per index of D / L: the label ids of its group, in the group's order
};

int bind_sym_general(tcb_ctx *ctx, const SymSpec &sp, const tcb_tensor *D, const tcb_tensor *L, SymBinding *b)
{
    if ((int)sp.lhs.size() != D->shape.rank || (int)sp.rhs.size() != L->shape.rank)
        return set_error(ctx, TCB_ESHAPE, "rank of a handle differs from the spec");
    auto side = [&](const std::vector<std::vector<std::string>> &groups, std::vector<std::vector<int>> *out, bool first) -> int {
        size_t seen = 0;
        for (const auto &grp : groups) {
            if (grp.size() > 3) return set_error(ctx, TCB_EUNSUPPORTED, "groups of more than three labels");
            std::vector<int> ids;
            for (const auto &lab : grp) {
                int id = find_label(b->labels, lab);
                if (first) {
                    if (id >= 0) return set_error(ctx, TCB_EUNSUPPORTED, "label repeated inside a tensor");
                    id = (int)b->labels.size();
                    b->labels.push_back(lab);
                } else if (id < 0) return set_error(ctx, TCB_EINVAL_EXPR, "label " + lab + " is on one side only");
                for (const auto &g2 : *out) for (int x : g2) if (x == id) return set_error(ctx, TCB_EUNSUPPORTED, "label repeated inside a tensor");
                for (int x : ids) if (x == id) return set_error(ctx, TCB_EUNSUPPORTED, "label repeated inside a tensor");
                ids.push_back(id);
                ++seen;
            }
            out->push_back(ids);
        }
        if (!first && seen != b->labels.size()) return set_error(ctx, TCB_EINVAL_EXPR, "a label is on one side only");
        return TCB_OK;
    };
    int rc = side(sp.lhs, &b->dg, true);
    if (rc) return rc;
    rc = side(sp.rhs, &b->lg, false);
    if (rc) return rc;
    b->ext.assign(b->labels.size(), -1);
    auto extents = [&](const std::vector<std::vector<int>> &groups, const tcb_tensor *T) -> int {
        for (size_t g = 0; g < groups.size(); ++g) {
            const int k = (int)groups[g].size();
            const int64_t n = k == 1 ? T->shape.ext[g] : unchoose(T->shape.ext[g], k);
            if (n < 0) return set_error(ctx, TCB_ESHAPE, "packed extent is not n(n-1)/2 (n(n-1)(n-2)/6) of any n");
            if (k > 1 && n > 65535) return set_error(ctx, TCB_EUNSUPPORTED, "group labels of extent above 65535");
            for (int id : groups[g]) {
                if (b->ext[id] >= 0 && b->ext[id] != n) return set_error(ctx, TCB_ESHAPE, "a label has two extents (or a group mixes extents)");
                b->ext[id] = n;
            }
        }
        return TCB_OK;
    };
    rc = extents(b->dg, D);
    if (rc) return rc;
    return extents(b->lg, L);
}

// the device table of the strictly increasing k-tuples of range(n), first label fastest (built once per (n, k))
int sym_tuple_table(tcb_ctx *ctx, int64_t n, int k, const SymTuple **out)
{
    auto it = ctx->sym_tuples.find({n, k});
    if (it == ctx->sym_tuples.end()) {
        int rc = refuse_in_capture(ctx, "the first use of an a<b group of this extent (run the call list once before capturing it)");
        if (rc) return rc;
        std::vector<SymTuple> host;
        host.reserve((size_t)choose(n, k));
        if (k == 2) { for (int64_t y = 0; y < n; ++y) for (int64_t x = 0; x < y; ++x) host.push_back(SymTuple{{(unsigned short)x, (unsigned short)y, 0, 0}}); }
        else for (int64_t z = 0; z < n; ++z) for (int64_t y = 0; y < z; ++y) for (int64_t x = 0; x < y; ++x)
                 host.push_back(SymTuple{{(unsigned short)x, (unsigned short)y, (unsigned short)z, 0}});
        SymTuple *dev = nullptr;
        TCB_CUDA(ctx, cudaMalloc((void **)&dev, std::max<size_t>(1, host.size()) * sizeof(SymTuple)));
        cudaError_t e = cudaMemcpyAsync(dev, host.data(), host.size() * sizeof(SymTuple), cudaMemcpyHostToDevice, cur_stream(ctx));
        if (e == cudaSuccess) e = cudaStreamSynchronize(cur_stream(ctx));   // host vector dies here; usable from every lane
        if (e != cudaSuccess) { cudaFree(dev); return cuda_fail(ctx, e, "cudaMemcpyAsync(tuple table)"); }
        it = ctx->sym_tuples.emplace(std::make_pair(n, k), dev).first;
    }
    *out = it->second;
    return TCB_OK;
}

// fills the descriptor's structure (not the terms) from a binding
int symmap_structure(tcb_ctx *ctx, const SymBinding &b, const tcb_tensor *D, const tcb_tensor *L, SymMapDesc *d)
{
    d->nd = D->shape.rank;
    d->nl = L->shape.rank;
    int64_t sL[kMaxRank];
    strides_of(L->shape, sL);
    std::vector<int> ldim(b.labels.size()), lslot(b.labels.size());
    for (int k = 0; k < kMaxRank; ++k) {
        d->dext[k] = k < d->nd ? D->shape.ext[k] : 1;
        d->dlen[k] = k < d->nd ? (int)b.dg[k].size() : 1;
        d->dtab[k] = nullptr;
        if (k < d->nd) {
            for (size_t s = 0; s < b.dg[k].size(); ++s) { ldim[b.dg[k][s]] = k; lslot[b.dg[k][s]] = (int)s; }
            if (d->dlen[k] > 1) {
                int rc = sym_tuple_table(ctx, b.ext[b.dg[k][0]], d->dlen[k], &d->dtab[k]);
                if (rc) return rc;
            }
        }
    }
    for (int g = 0; g < kMaxRank; ++g) {
        d->llen[g] = g < d->nl ? (int)b.lg[g].size() : 1;
        d->lstride[g] = g < d->nl ? sL[g] : 0;
        for (int s = 0; s < 3; ++s) {
            const bool on = g < d->nl && s < d->llen[g];
            d->lsrc_dim[g][s] = on ? ldim[b.lg[g][s]] : 0;
            d->lsrc_slot[g][s] = on ? lslot[b.lg[g][s]] : 0;
        }
    }
    for (int t = 0; t < kMaxSymTerms; ++t) {
        d->sign[t] = 1;
        for (int k = 0; k < kMaxRank; ++k) for (int s = 0; s < 3; ++s) d->perm[t][k][s] = (unsigned char)s;
    }
    d->nterms = 1;
    return TCB_OK;
}

}  // namespace

int tcb_pack(tcb_ctx *ctx, const char *spec, tcb_tensor *D, const tcb_tensor *L)
{
    NvtxRange nvtx_range("tcb_pack");
    int rc = enter(ctx);
    if (rc) return rc;
    if (!spec || !D || !L) return set_error(ctx, TCB_EINVAL, "null argument");
    SymSpec sp;
    if (!parse_sym_spec(spec, &sp)) return set_error(ctx, TCB_EINVAL_EXPR, std::string("cannot parse: ") + spec);
    if (sp.accumulate) return set_error(ctx, TCB_EINVAL_EXPR, "tcb_pack takes '=', not '+='");
    int pos[kMaxRank][3];
    rc = bind_sym_spec(ctx, sp.lhs, sp.rhs, D, L, pos);
    if (rc) return rc;
    if (overlaps(D, L)) return set_error(ctx, TCB_EALIAS, "D overlaps L");
    const std::string key = std::string(spec) + "|" + shape_key(D->shape) + shape_key(L->shape);
    auto it = ctx->sym_tables.find(key);
    if (it == ctx->sym_tables.end()) {
        rc = refuse_in_capture(ctx, "the first tcb_pack of a spec (run the call list once before capturing it)");
        if (rc) return rc;
        std::unique_ptr<SymTables> st(new SymTables());
        int64_t sL[kMaxRank];
        strides_of(L->shape, sL);
        for (size_t g = 0; g < sp.lhs.size(); ++g) {
            st->at[g] = st->host.size();
            const int k = (int)sp.lhs[g].size();
            const int64_t n = L->shape.ext[pos[g][0]];
            const int64_t s0 = sL[pos[g][0]], s1 = k > 1 ? sL[pos[g][1]] : 0, s2 = k > 2 ? sL[pos[g][2]] : 0;
            // strictly increasing tuples, first label fastest
            if (k == 1) for (int64_t a = 0; a < n; ++a) st->host.push_back(a * s0);
            else if (k == 2) { for (int64_t b = 0; b < n; ++b) for (int64_t a = 0; a < b; ++a) st->host.push_back(a * s0 + b * s1); }
            else for (int64_t c = 0; c < n; ++c) for (int64_t b = 0; b < c; ++b) for (int64_t a = 0; a < b; ++a)
                     st->host.push_back(a * s0 + b * s1 + c * s2);
        }
        TCB_CUDA(ctx, cudaMalloc((void **)&st->dev, std::max<size_t>(1, st->host.size()) * sizeof(int64_t)));
        TCB_CUDA(ctx, cudaMemcpyAsync(st->dev, st->host.data(), st->host.size() * sizeof(int64_t), cudaMemcpyHostToDevice,
                                      cur_stream(ctx)));
        TCB_CUDA(ctx, cudaStreamSynchronize(cur_stream(ctx)));     // usable from every lane from here on
        it = ctx->sym_tables.emplace(key, std::move(st)).first;
    }
    PackDesc d;
    d.rank = D->shape.rank;
    for (int k = 0; k < kMaxRank; ++k) {
        d.extent[k] = k < d.rank ? D->shape.ext[k] : 1;
        d.tab[k] = k < d.rank ? it->second->dev + it->second->at[k] : nullptr;
    }
    d.in = L->ptr; d.out = D->ptr;
    TimedLaunch tl(ctx, kClsPermute, 0.0, 32.0 * (double)D->elems());
    TCB_CUDA(ctx, launch_pack(d, cur_stream(ctx), &ctx->launches));
    return TCB_OK;
}

int tcb_unpack(tcb_ctx *ctx, const char *spec, tcb_tensor *D, const tcb_tensor *L, tcb_c128 alpha)
{
    NvtxRange nvtx_range("tcb_unpack");
    int rc = enter(ctx);
    if (rc) return rc;
    if (!spec || !D || !L) return set_error(ctx, TCB_EINVAL, "null argument");
    SymSpec sp;
    if (!parse_sym_spec(spec, &sp)) return set_error(ctx, TCB_EINVAL_EXPR, std::string("cannot parse: ") + spec);
    bool d_groups = false;
    for (const auto &g : sp.lhs) d_groups = d_groups || g.size() > 1;
    if (d_groups) {
        // a<b groups on D as well: a packed view of a packed tensor, "Tq(d<e,c,i<j<k)=T(d<e<c,i<j<k)" -- one signed read each
        SymBinding b;
        rc = bind_sym_general(ctx, sp, D, L, &b);
        if (rc) return rc;
        if (overlaps(D, L)) return set_error(ctx, TCB_EALIAS, "D overlaps L");
        SymMapDesc m;
        rc = symmap_structure(ctx, b, D, L, &m);
        if (rc) return rc;
        m.alpha_re = alpha.re; m.alpha_im = alpha.im;
        m.accumulate = sp.accumulate;
        m.in = L->ptr; m.out = D->ptr;
        TimedLaunch tl(ctx, kClsPermute, 0.0, 16.0 * (double)D->elems() * (sp.accumulate ? 3.0 : 2.0));
        TCB_CUDA(ctx, launch_symmap(m, cur_stream(ctx), &ctx->launches));
        return TCB_OK;
    }
    int pos[kMaxRank][3];
    rc = bind_sym_spec(ctx, sp.rhs, sp.lhs, L, D, pos);
    if (rc) return rc;
    if (overlaps(D, L)) return set_error(ctx, TCB_EALIAS, "D overlaps L");
    UnpackDesc d;
    d.rank = D->shape.rank;
    d.ngroups = L->shape.rank;
    int64_t sP[kMaxRank];
    strides_of(L->shape, sP);
    for (int k = 0; k < kMaxRank; ++k) d.extent[k] = k < d.rank ? D->shape.ext[k] : 1;
    for (int g = 0; g < kMaxRank; ++g) {
        d.glen[g] = g < d.ngroups ? (int)sp.rhs[g].size() : 1;
        d.pstride[g] = g < d.ngroups ? sP[g] : 0;
        for (int s = 0; s < 3; ++s) d.gpos[g][s] = (g < d.ngroups && s < d.glen[g]) ? pos[g][s] : 0;
    }
    d.alpha_re = alpha.re; d.alpha_im = alpha.im;
    d.accumulate = sp.accumulate;
    d.in = L->ptr; d.out = D->ptr;
    TimedLaunch tl(ctx, kClsPermute, 0.0, 16.0 * ((double)D->elems() * (sp.accumulate ? 2.0 : 1.0) + (double)L->elems()));
    TCB_CUDA(ctx, launch_unpack(d, cur_stream(ctx), &ctx->launches));
    return TCB_OK;
}

int tcb_antisym_pack(tcb_ctx *ctx, const char *spec, tcb_tensor *D, const tcb_tensor *L, tcb_c128 alpha)
{
    NvtxRange nvtx_range("tcb_antisym_pack");
    int rc = enter(ctx);
    if (rc) return rc;
    if (!spec || !D || !L) return set_error(ctx, TCB_EINVAL, "null argument");
    SymSpec sp;
    if (!parse_sym_spec(spec, &sp)) return set_error(ctx, TCB_EINVAL_EXPR, std::string("cannot parse: ") + spec);
    SymBinding b;
    rc = bind_sym_general(ctx, sp, D, L, &b);
    if (rc) return rc;
    if (overlaps(D, L)) return set_error(ctx, TCB_EALIAS, "D overlaps L");
    // every group of L must lie inside one group of D: D's groups are unions of L's
    std::vector<int> dim_of(b.labels.size()), slot_of(b.labels.size());
    for (size_t k = 0; k < b.dg.size(); ++k)
        for (size_t s = 0; s < b.dg[k].size(); ++s) { dim_of[b.dg[k][s]] = (int)k; slot_of[b.dg[k][s]] = (int)s; }
    for (const auto &g : b.lg)
        for (int id : g)
            if (dim_of[id] != dim_of[g[0]]) return set_error(ctx, TCB_EINVAL_EXPR, "a group of L is spread over two groups of D");
    SymMapDesc m;
    rc = symmap_structure(ctx, b, D, L, &m);
    if (rc) return rc;
    // the shuffles: per group of D, the assignments slot -> tuple component under which every block (a group of L, its
    // labels taken in D's slot order) receives increasing components; sign = parity of the assignment
    struct Choice { unsigned char perm[3]; int sign; };
    std::vector<std::vector<Choice>> per_dim(b.dg.size());
    for (size_t k = 0; k < b.dg.size(); ++k) {
        const int n = (int)b.dg[k].size();
        int block[3] = {0, 0, 0};
        for (size_t g = 0; g < b.lg.size(); ++g)
            for (int id : b.lg[g]) if (dim_of[id] == (int)k) block[slot_of[id]] = (int)g;
        int perm[3] = {0, 1, 2};
        do {
            bool ok = true;
            for (int s1 = 0; s1 < n && ok; ++s1)
                for (int s2 = s1 + 1; s2 < n && ok; ++s2)
                    if (block[s1] == block[s2] && perm[s1] > perm[s2]) ok = false;
            if (ok) {
                int inv = 0;
                for (int s1 = 0; s1 < n; ++s1) for (int s2 = s1 + 1; s2 < n; ++s2) inv += perm[s1] > perm[s2] ? 1 : 0;
                Choice c;
                for (int s1 = 0; s1 < 3; ++s1) c.perm[s1] = (unsigned char)(s1 < n ? perm[s1] : s1);
                c.sign = inv % 2 ? -1 : 1;
                per_dim[k].push_back(c);
            }
        } while (std::next_permutation(perm, perm + n));
    }
    size_t nterms = 1;
    for (const auto &v : per_dim) nterms *= v.size();
    if (nterms > (size_t)kMaxSymTerms) return set_error(ctx, TCB_EUNSUPPORTED, "more than 36 signed terms");
    m.nterms = (int)nterms;
    for (size_t t = 0; t < nterms; ++t) {            // first group of D fastest
        size_t r = t;
        int sign = 1;
        for (size_t k = 0; k < per_dim.size(); ++k) {
            const Choice &c = per_dim[k][r % per_dim[k].size()];
            r /= per_dim[k].size();
            for (int s1 = 0; s1 < 3; ++s1) m.perm[t][k][s1] = c.perm[s1];
            sign *= c.sign;
        }
        m.sign[t] = (signed char)sign;
    }
    m.alpha_re = alpha.re; m.alpha_im = alpha.im;
    m.accumulate = sp.accumulate;
    m.in = L->ptr; m.out = D->ptr;
    TimedLaunch tl(ctx, kClsPermute, 0.0, 16.0 * (double)D->elems() * ((double)nterms + (sp.accumulate ? 2.0 : 1.0)));
    TCB_CUDA(ctx, launch_symmap(m, cur_stream(ctx), &ctx->launches));
    return TCB_OK;
}

int64_t tcb_packed_extent(int64_t n, int k)
{
    if (n < 0 || k < 1 || k > 3) return -1;
    return choose(n, k);
}

// used by synth.cu (same shared object): validates the context and exposes its stream and launch counter
int tcbx_internal_stream(tcb_ctx *ctx, void **stream, int64_t **launches)
{
    int rc = enter(ctx);
    if (rc) return rc;
    *stream = (void *)cur_stream(ctx);
    *launches = &ctx->launches;
    return TCB_OK;
}

// ---- measurement -------------------------------------------------------------------------------------------

int tcb_measure_fp64_tensor_peak(tcb_ctx *ctx, double milliseconds, double *tflops)
{
    int rc = enter(ctx);
    if (rc) return rc;
    if (!tflops) return TCB_EINVAL;
    TCB_CUDA(ctx, run_dmma_peak(milliseconds, tflops, cur_stream(ctx), &ctx->launches));
    return TCB_OK;
}

int tcb_measure_fp64_vector_peak(tcb_ctx *ctx, double milliseconds, double *tflops)
{
    int rc = enter(ctx);
    if (rc) return rc;
    if (!tflops) return TCB_EINVAL;
    TCB_CUDA(ctx, run_dfma_peak(milliseconds, tflops, cur_stream(ctx), &ctx->launches));
    return TCB_OK;
}

int tcb_kernel_stats(tcb_ctx *ctx, const char *kernel, tcb_kernel_stat *out)
{
    int rc = enter(ctx);
    if (rc) return rc;
    if (!kernel || !out) return TCB_EINVAL;
    static const char *names[4] = {"zgemm", "permute", "permsum", "elementwise"};
    fold_spans(ctx);
    for (int c = 0; c < 4; ++c)
        if (std::strcmp(kernel, names[c]) == 0) { *out = ctx->acc[c]; return TCB_OK; }
    return set_error(ctx, TCB_EINVAL, std::string("unknown kernel class ") + kernel);
}

int tcb_kernel_stats_reset(tcb_ctx *ctx)
{
    int rc = enter(ctx);
    if (rc) return rc;
    fold_spans(ctx);
    for (int c = 0; c < 4; ++c) ctx->acc[c] = tcb_kernel_stat{0, 0.0, 0.0, 0.0};
    return TCB_OK;
}

// ---- CUDA graph capture of a call list ---------------------------------------------------------------------------
struct tcb_graph {
    cudaGraph_t graph = nullptr;
    cudaGraphExec_t exec = nullptr;
    int64_t launches = 0;
    uint64_t ws_generation = 0;      // the workspace blocks whose addresses the kernels of this graph carry
    size_t nodes = 0, edges = 0, depth = 0;   // depth: nodes on the longest dependency path (= nodes for a chain)
};

int tcb_capture_begin(tcb_ctx *ctx)
{
    int rc = enter(ctx);
    if (rc) return rc;
    if (ctx->capturing) return set_error(ctx, TCB_EINVAL, "a capture is already open");
    if (ctx->kernel_timing) return set_error(ctx, TCB_EINVAL, "kernel_timing must be off during a capture");
    if (ctx->cur != 0) return set_error(ctx, TCB_EINVAL, "a capture starts on lane 0");
    TCB_CUDA(ctx, cudaStreamBeginCapture(ctx->lanes[0].stream, cudaStreamCaptureModeThreadLocal));
    ctx->capturing = true;
    ctx->capture_failed = false;
    for (Lane &ln : ctx->lanes) ln.in_capture = false;
    ctx->lanes[0].in_capture = true;
    ctx->capture_l0 = ctx->launches;
    return TCB_OK;
}

int tcb_capture_end(tcb_ctx *ctx, tcb_graph **out)
{
    if (!ctx || !out) return TCB_EINVAL;
    *out = nullptr;
    if (!ctx->capturing) return set_error(ctx, TCB_EINVAL, "no capture is open");
    cudaSetDevice(ctx->device);
    // every lane that was forked into the capture joins lane 0 again (a capture must end with one open path)
    for (int l = 1; l < kMaxLanes && !ctx->capture_failed; ++l) {
        Lane &ln = ctx->lanes[l];
        if (!ln.in_capture) continue;
        if (cudaEventRecord(ln.ev, ln.stream) != cudaSuccess ||
            cudaStreamWaitEvent(ctx->lanes[0].stream, ln.ev, 0) != cudaSuccess) {
            cudaGetLastError();
            ctx->capture_failed = true;
        }
    }
    ctx->capturing = false;
    ctx->cur = 0;
    for (Lane &ln : ctx->lanes) ln.in_capture = false;
    std::unique_ptr<tcb_graph> g(new tcb_graph);
    cudaError_t e = cudaStreamEndCapture(ctx->lanes[0].stream, &g->graph);
    if (e != cudaSuccess || !g->graph || ctx->capture_failed) {
        cudaGetLastError();
        if (g->graph) cudaGraphDestroy(g->graph);
        const std::string why = ctx->capture_failed ? ctx->last_error : std::string(cudaGetErrorString(e));
        ctx->capture_failed = false;
        return set_error(ctx, TCB_EUNSUPPORTED, "the call list could not be captured: " + why);
    }
    e = cudaGraphInstantiate(&g->exec, g->graph, 0);
    if (e != cudaSuccess) {
        cudaGraphDestroy(g->graph);
        cudaGetLastError();
        return set_error(ctx, TCB_EUNSUPPORTED, std::string("cudaGraphInstantiate: ") + cudaGetErrorString(e));
    }
    cudaGraphGetNodes(g->graph, nullptr, &g->nodes);
    cudaGraphGetEdges(g->graph, nullptr, nullptr, &g->edges);
    {   // longest dependency path, in nodes
        std::vector<cudaGraphNode_t> nd(g->nodes), from(g->edges), to(g->edges);
        size_t nn = g->nodes, ne = g->edges;
        if (nn && cudaGraphGetNodes(g->graph, nd.data(), &nn) == cudaSuccess &&
            (!ne || cudaGraphGetEdges(g->graph, from.data(), to.data(), &ne) == cudaSuccess)) {
            std::map<cudaGraphNode_t, size_t> len;
            for (size_t i = 0; i < nn; ++i) len[nd[i]] = 1;
            for (size_t pass = 0; pass < nn; ++pass) {           // relax until stable (graphs here have tens of nodes)
                bool moved = false;
                for (size_t k = 0; k < ne; ++k)
                    if (len[to[k]] < len[from[k]] + 1) { len[to[k]] = len[from[k]] + 1; moved = true; }
                if (!moved) break;
            }
            for (auto &kv : len) g->depth = std::max(g->depth, kv.second);
        }
        cudaGetLastError();
    }
    g->launches = ctx->launches - ctx->capture_l0;
    g->ws_generation = ctx->ws_generation;
    *out = g.release();
    return TCB_OK;
}

int tcb_graph_launch(tcb_ctx *ctx, tcb_graph *g)
{
    NvtxRange nvtx_range("tcb_graph_launch");
    int rc = enter(ctx);
    if (rc) return rc;
    if (!g || !g->exec) return TCB_EINVAL;
    if (ctx->capturing) return set_error(ctx, TCB_EINVAL, "graph launch inside a capture");
    if (g->ws_generation != ctx->ws_generation)
        return set_error(ctx, TCB_EINVAL, "the workspace was reallocated after this graph was captured (a later call needed a "
                                          "larger one): capture the call list again");
    TCB_CUDA(ctx, cudaGraphLaunch(g->exec, ctx->lanes[0].stream));
    ctx->launches += g->launches;
    return TCB_OK;
}

int tcb_graph_info(const tcb_graph *g, int64_t *nodes, int64_t *edges, int64_t *kernel_launches, int64_t *depth)
{
    if (!g) return TCB_EINVAL;
    if (depth) *depth = (int64_t)g->depth;
    if (nodes) *nodes = (int64_t)g->nodes;
    if (edges) *edges = (int64_t)g->edges;
    if (kernel_launches) *kernel_launches = g->launches;
    return TCB_OK;
}

int tcb_graph_destroy(tcb_graph *g)
{
    if (!g) return TCB_EINVAL;
    if (g->exec) cudaGraphExecDestroy(g->exec);
    if (g->graph) cudaGraphDestroy(g->graph);
    delete g;
    return TCB_OK;
}

int tcb_timer_start(tcb_ctx *ctx)
{
    int rc = enter(ctx);
    if (rc) return rc;
    TCB_CUDA(ctx, cudaEventRecord(ctx->ev0, cur_stream(ctx)));
    return TCB_OK;
}

int tcb_timer_stop(tcb_ctx *ctx, double *milliseconds)
{
    int rc = enter(ctx);
    if (rc) return rc;
    if (!milliseconds) return TCB_EINVAL;
    TCB_CUDA(ctx, cudaEventRecord(ctx->ev1, cur_stream(ctx)));
    TCB_CUDA(ctx, cudaEventSynchronize(ctx->ev1));
    float ms = 0.f;
    TCB_CUDA(ctx, cudaEventElapsedTime(&ms, ctx->ev0, ctx->ev1));
    *milliseconds = ms;
    return TCB_OK;
}

}  // extern "C"
