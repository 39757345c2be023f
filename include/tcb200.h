/*
 * tcb200.h -- C ABI of the B200 tensor-contraction backend (libtcb200.so).
 *
 * What this boundary is: the calls a tenpi-generated coupled-cluster driver issues to its tensor
 * library: create / destroy tensors, contract two tensors into a third with a scalar
 * factor, add, scale, and a barrier.  "Contraction ... includes a list of tensors, a scalar factor and
 * optionally permutation operators and an output tensor"; only two tensors are
 * contracted per instruction.  How a contraction is evaluated is the library's business;
 * the reference scheme is TTGT: bring the operands to matrix form, GEMM, bring the
 * result to the output's index order.
 *
 * Conventions (readings #1, #7, #8, #11, #12)
 *   - element: complex128 = interleaved (re, im) IEEE doubles, 16 bytes, 16-byte aligned.
 *   - layout: dense, generalised column-major: in T(a,b,i,j) the FIRST listed index has unit stride
 *     ("unit-stride index"; tenpi emits Fortran).  offset = sum_k idx_k * prod_{m<k} ext_m.
 *   - rank 0..6, every extent >= 1.  All tensor data lives in DEVICE memory.
 *   - expression grammar (white space ignored):
 *         name '(' [label {',' label}] ')' ('+=' | '=') name '(' ... ')' [ '*' name '(' ... ')' ]
 *     label = [A-Za-z][A-Za-z0-9_]*  (tenpi prints a,b,i,j or p1,p2,h1,h2 -- PAPER.md:232);
 *     tensor names are ignored, operands bind by position (D, L, R).  '+=' accumulates into D,
 *     '=' overwrites D.
 *   - a valid contraction: every label occurs exactly twice over D, L, R and at most once per tensor
 *     (no batch/Hadamard index, no trace, no broadcast -> TCB_EUNSUPPORTED).  K = 1 (outer product)
 *     and fully contracted R (N = 1) are valid.
 *   - execution: every call validates its arguments, then enqueues work on the context's stream and
 *     returns; calls execute in issue order (the paper's barrier after each operation, PAPER.md:400,
 *     becomes stream order).  tcb_sync and tcb_tensor_download block.  On any error return nothing has
 *     been enqueued and D is untouched.
 *   - ownership: handles are created and destroyed by the library.  tcb_tensor_wrap borrows caller
 *     memory and never frees it.  D must not overlap L or R (TCB_EALIAS).
 *   - no CPU fallback exists: without a CUDA device every compute call returns TCB_ECUDA.
 *   - not thread-safe per context.
 *
 * All functions return 0 (TCB_OK) or a negative tcb_status.
 */
#ifndef TCB200_H
#define TCB200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define TCB_MAX_RANK 6

typedef enum {
    TCB_OK = 0,
    TCB_EINVAL_EXPR = -1,   /* expression does not parse, or operand count / op does not fit the call */
    TCB_ESHAPE = -2,        /* ranks or extents of the handles disagree with the expression */
    TCB_ERANK = -3,         /* rank > TCB_MAX_RANK, or extent < 1 */
    TCB_EALIAS = -4,        /* D overlaps L or R */
    TCB_ENOMEM = -5,        /* device allocation or workspace exhausted */
    TCB_ECUDA = -6,         /* a CUDA call failed (sticky per context); text via tcb_last_error */
    TCB_EUNSUPPORTED = -7,  /* batch / trace / broadcast index, conjugation, ... */
    TCB_EINVAL = -8         /* NULL handle, bad option, bad permutation table, ... */
} tcb_status;

typedef struct tcb_ctx tcb_ctx;       /* device, stream, workspace pool, plan cache */
typedef struct tcb_tensor tcb_tensor; /* rank, extents, device pointer, owns-memory flag */
typedef struct { double re, im; } tcb_c128;

/* ---- context ------------------------------------------------------------------------------------ */

/* device: CUDA ordinal.  cuda_stream: a cudaStream_t to enqueue on, or NULL for a stream the context
 * creates and owns.  workspace_bytes: initial size of the workspace pool used for permuted operands and
 * split-K partials (0 = grow on demand; growth synchronises the stream). */
int tcb_ctx_create(tcb_ctx **ctx, int device, void *cuda_stream, size_t workspace_bytes);
int tcb_ctx_destroy(tcb_ctx *ctx);
/* keys: "splitk" = "auto" | "off" | <integer number of splits>;
 *       "epilogue" = "auto" | "fused" (alpha*C scattered into D's index order by the GEMM epilogue: no third TTGT pass)
 *                  | "twopass" (PAPER.md:91 literally: the GEMM writes a plain M x N matrix into workspace, a
 *                    permute-accumulate pass brings it into D; kept for A/B tests, "auto" never picks it);
 *       "operand_loads" = "auto" (cost model: per operand the cheapest of reading it in place by TMA, reading it in place
 *                    through offset tables, or permuting it into workspace first) | "gather" (never permute) | "permute"
 *                    (never gather: TTGT as in PAPER.md:88-89);
 *       "permute_operands" = "auto" | "always"  (A/B testing of plans: both operands always permuted);
 *       "complex_product" = "auto" | "4m" | "3m": how the GEMM forms a complex product from real tensor-core products.
 *                    "4m": Re = ArBr - AiBi, Im = ArBi + AiBr (four).  "3m": P1 = ArBr, P2 = AiBi, P3 = (Ar+Ai)(Br+Bi),
 *                    Re = P1 - P2, Im = P3 - P1 - P2 (three: 25 % less tensor work, 8 ... 27 % faster).  Both meet the 1e-11 * snorm tolerance with orders of magnitude to spare; 3m gives up
 *                    bit-exact products of exactly representable operands (a delta tensor returns its partner to within
 *                    2^-52 (|re| + |im|), not bit for bit) -- real operands still give an exactly real result.  "auto": 3m
 *                    when both operands are TMA-fed (not gathered) and K >= 32; 4m otherwise;
 *       "gemm_deal" = "dynamic" | "static" (how the GEMM's tiles and stream-K chunks reach the CTAs: claimed from a counter,
 *                    or dealt round-robin; the result is the same bit for bit);
 *       "kernel_timing" = "on" | "off" (see tcb_kernel_stats);   unknown key -> TCB_EINVAL. */
int tcb_ctx_set_option(tcb_ctx *ctx, const char *key, const char *value);
/* Blocks until everything enqueued so far -- on every lane -- has finished (the paper's barrier). */
int tcb_sync(tcb_ctx *ctx);
/* Lanes: concurrency between independent contractions.  Generated code puts a barrier after every tensor
 * operation, which the paper measures as its serial fraction; DLTC-style layering lets
 * operations without a data dependence run side by side.  A context has tcb_lane_count() lanes; each is a stream with its
 * own workspace.  Lane 0 is the context's stream and the default.
 *   tcb_lane_set(ctx, l)      : every following call (tensor creation and destruction included) is enqueued on lane l;
 *   tcb_lane_wait(ctx, l, m)  : what is enqueued on lane l from now on starts after everything enqueued on lane m so far.
 * Calls on ONE lane execute in issue order; calls on different lanes are unordered unless a tcb_lane_wait orders them --
 * that is the caller's statement that they are independent (no output of one is an operand or output of the other, and a
 * tensor is destroyed on a lane that has waited for its last user).  Inside tcb_capture_begin/end the lanes become
 * parallel branches of the graph: a lane joins the capture at its first use there (it then starts after what lane 0 held
 * at that point) and is joined back into lane 0 by tcb_capture_end.  Errors: TCB_EINVAL (lane out of range), TCB_ECUDA. */
int tcb_lane_count(void);
int tcb_lane_set(tcb_ctx *ctx, int lane);
int tcb_lane_wait(tcb_ctx *ctx, int lane, int on_lane);
/* Text of the last error recorded on this context (valid until the next call on it). */
const char *tcb_last_error(const tcb_ctx *ctx);
const char *tcb_strerror(int code);
/* Number of kernels this context has launched so far (all of them this library's own). */
int64_t tcb_launch_count(const tcb_ctx *ctx);

/* ---- tensors ------------------------------------------------------------------------------------ */

/* Library-owned, zero-filled device tensor.  extents[rank], copied. */
int tcb_tensor_create(tcb_ctx *ctx, tcb_tensor **t, int rank, const int64_t *extents);
/* The same without the zero fill: contents are undefined until written.  For intermediates whose first use is an '='
 * operation (generated code creates and destroys them around every use); a 6 GB tensor saves 1 ms. */
int tcb_tensor_alloc(tcb_ctx *ctx, tcb_tensor **t, int rank, const int64_t *extents);
/* Borrow caller-owned device memory (e.g. torch storage), 16-byte aligned, prod(extents)*16 bytes. */
int tcb_tensor_wrap(tcb_ctx *ctx, tcb_tensor **t, int rank, const int64_t *extents, void *device_ptr);
/* Stream-ordered free of library-owned memory; borrowed memory is left alone.  NULL is accepted. */
int tcb_tensor_destroy(tcb_tensor *t);
/* Any of rank / extents / device_ptr may be NULL. */
int tcb_tensor_info(const tcb_tensor *t, int *rank, int64_t extents[TCB_MAX_RANK], void **device_ptr);
/* HOST <-> device copies of the whole tensor in the layout above.  upload is stream-ordered (the host
 * buffer must stay valid until tcb_sync unless it is pageable); download blocks until the data is there. */
int tcb_tensor_upload(tcb_ctx *ctx, tcb_tensor *t, const tcb_c128 *host);
int tcb_tensor_download(tcb_ctx *ctx, const tcb_tensor *t, tcb_c128 *host);
/* D[...] = value */
int tcb_tensor_fill(tcb_ctx *ctx, tcb_tensor *t, tcb_c128 value);

/* ---- the hot path ------------------------------------------------------------------------------- */

/* S1-S5: D(d..) (+)= alpha * L(l..) * R(r..), e.g.
 *     "R(a,b,i,j)+=V(a,b,c,d)*T(c,d,i,j)".
 * The planner picks the index grouping (M, N, K), which operands to permute into matrix form (workspace),
 * the GEMM variant, and scatters alpha*C into D's own index order in the GEMM epilogue. */
int tcb_contract(tcb_ctx *ctx, const char *expr, tcb_tensor *D, const tcb_tensor *L, const tcb_tensor *R,
                 tcb_c128 alpha);
/* Permuted add, "D(a,b,i,j)+=L(b,a,i,j)":  D = D + alpha * permuted L  ('=' : D = alpha * permuted L). */
int tcb_add(tcb_ctx *ctx, const char *expr, tcb_tensor *D, const tcb_tensor *L, tcb_c128 alpha);
/* D *= alpha */
int tcb_scale(tcb_ctx *ctx, tcb_tensor *D, tcb_c128 alpha);
/* Next row 8(f)-3, the solver around the residual: the Jacobi step with orbital-energy denominators ("adding energy
 * denominators to selected terms"; one such step per CC iteration):
 *     T[i0,i1,..] += alpha * R[i0,i1,..] / (eps[0][i0] + eps[1][i1] + ...)      energies summed in index order
 * eps: HOST array of rank pointers; eps[k] = extent_k real doubles, or NULL when index k does not enter the
 * denominator (at least one must be given).  For t_ij^ab stored T(a,b,i,j): eps = {-e_virt, -e_virt, +e_occ, +e_occ}.
 * T and R have the same shape and must not overlap.  The energies are copied before the call returns.  A zero
 * denominator is not detected (the quotient is IEEE inf/nan).  Errors: TCB_EINVAL, TCB_ESHAPE, TCB_EALIAS, TCB_ECUDA. */
int tcb_denominator_update(tcb_ctx *ctx, tcb_tensor *T, const tcb_tensor *R, const double *const *eps, tcb_c128 alpha);
/* The '=' form of the same operation:  T[i0,i1,..] = alpha * R[i0,i1,..] / (eps[0][i0] + eps[1][i1] + ...); T is not
 * read (first-order amplitudes from a residual, e.g. t3 = R3 / D3 of the triples correction).  Same arguments, same errors. */
int tcb_denominator_divide(tcb_ctx *ctx, tcb_tensor *T, const tcb_tensor *R, const double *const *eps, tcb_c128 alpha);
/* Inner product into a rank-0 tensor (what a DIIS extrapolation around the iteration needs; the bilinear form is also
 * reachable as a full contraction "E()=X(..)*Y(..)", the sesquilinear one only here):
 *     D = alpha * sum_i (conjugate_x ? conj(X[i]) : X[i]) * Y[i]
 * X and Y have the same shape (any rank), D has rank 0 and overlaps neither.  Deterministic (fixed summation order).
 * Stream-ordered like every other call: download D to read it.  Errors: TCB_EINVAL, TCB_ESHAPE, TCB_EALIAS, TCB_ECUDA. */
int tcb_dot(tcb_ctx *ctx, tcb_tensor *D, const tcb_tensor *X, const tcb_tensor *Y, int conjugate_x, tcb_c128 alpha);
/* The same inner product for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc): tcb_dot keeps its per-block partial sums in a stream-ordered allocation made for the call; this
 * entry point keeps them in ONE fixed device array inside the library (131 328 bytes, held by every GPU that loads the
 * library until the process exits) and calls no cudaMalloc / cudaMallocAsync / cudaFree or allocating routine: one
 * 4-byte cudaMemsetAsync and one kernel launch on the context's current lane.  Same arguments and checks as tcb_dot.
 *   Limit: X and Y hold at most TCB_DOT_NOALLOC_MAX_ELEMS = 536 870 912 elements (8.6 GB each); more is refused with
 *          TCB_EUNSUPPORTED (nothing enqueued, D untouched) -- use tcb_dot.
 *   Result: deterministic; the grid depends on the element count alone, so the bits do not depend on the GPU model either.
 *          It differs from tcb_dot's by summation order only (both round every product and sum separately; <x|x> has an
 *          exactly zero imaginary part).
 *   Sharing: every call on a device uses the same array, which keeps the last call's contents (the call clears the counter
 *          it needs at zero itself).  Calls that OVERLAP on the GPU -- other lanes, streams, contexts or host threads on
 *          the same device -- race on it: keep them on one stream or order them with events.
 * Errors: TCB_EINVAL, TCB_ESHAPE, TCB_EALIAS, TCB_EUNSUPPORTED (too many elements), TCB_ECUDA. */
#define TCB_DOT_NOALLOC_MAX_ELEMS 536870912LL
int tcb_dot_noalloc(tcb_ctx *ctx, tcb_tensor *D, const tcb_tensor *X, const tcb_tensor *Y, int conjugate_x, tcb_c128 alpha);
/* S3, tensor transposition: "D(i,j,a,b)=L(a,b,i,j)", pure data movement, bit-exact. */
int tcb_permute(tcb_ctx *ctx, const char *expr, tcb_tensor *D, const tcb_tensor *L);
/* S6, fused permute-sum (the generator's unrolled permutation operators):
 *     D[i] = beta * D[i] + sum_{t<nterms} coefs[t] * X[i_{s_t(0)}, i_{s_t(1)}, ...],   terms added in order t;
 * perms[t*rank + k] = s_t(k): position k of X is indexed by D's index number s_t(k), so
 * "D(a,b,i,j) += -1 * X(b,a,i,j)" is s = (1,0,2,3), c = -1.  beta = 0 does not read D.
 * X must not overlap D.  Each product and each sum is rounded on its own (no FMA contraction). */
int tcb_permsum(tcb_ctx *ctx, tcb_tensor *D, const tcb_tensor *X, int nterms, const int32_t *perms,
                const tcb_c128 *coefs, tcb_c128 beta);
/* Sugar over tcb_permsum: spec = "P(a/bc)P(k/ij):D(a,b,c,i,j,k)+=X(a,b,c,i,j,k)".  Each P(x/yz..) stands
 * for 1 - (x<->y) - (x<->z) - ...; P(xy) for 1 - (x<->y); the product is expanded into signed terms
 * (first operator outermost).  D = D + alpha * sum of terms. */
int tcb_antisymmetrize(tcb_ctx *ctx, const char *spec, tcb_tensor *D, const tcb_tensor *X, tcb_c128 alpha);
/* Index-permutation-symmetric (antisymmetric) packed storage, SURVEY 8(f)-2.  The paper lists index-permutation symmetry as
 * what its generated code does not exploit yet (outlook 440, 452); it gives no storage scheme, so this is
 * a reading (reading 16): a group a<b (or a<b<c) of labels of equal extent n, in which the tensor is antisymmetric,
 * is stored as ONE packed index running over the strictly increasing tuples, first label fastest:
 *     pairs (0,1) (0,2) (1,2) (0,3) ..   p = b(b-1)/2 + a;      triples (0,1,2) (0,1,3) (0,2,3) (1,2,3) ..
 * of extent tcb_packed_extent(n, 2) = n(n-1)/2, tcb_packed_extent(n, 3) = n(n-1)(n-2)/6.  A packed tensor is an ordinary
 * handle (create it with those extents); contractions over whole groups are plain tcb_contract calls on the packed indices:
 *     Vp(a<b,c<d) = V(a,b,c,d);  Tp(c<d,i<j) = T(c,d,i,j);  "Rp(x,y)+=Vp(x,z)*Tp(z,y)" with alpha = 1;  R(a,b,i,j) += Rp(a<b,i<j)
 * is the pp ladder R += 1/2 V T at 1/8 of the flops (the c<d sum visits each unordered pair once: no factor 1/2).
 *   tcb_pack   spec "Vp(a<b,c<d)=V(a,b,c,d)": Dp[.., p, ..] = L[.., a, .., b, ..]; pure data movement, bit-exact; groups of
 *              1..3 labels, in any order and at any dense positions; '=' only.
 *   tcb_unpack spec "R(a,b,i,j)+=Rp(a<b,i<j)" (or '='): D[.., a, .., b, ..] (+)= alpha * sign * Lp[.., p(sorted a, b), ..],
 *              sign = parity of the sorting permutation, 0 when two labels of a group coincide.  With alpha = 1 and '=' an
 *              exactly antisymmetric tensor comes back bit for bit.
 *              D may carry groups too -- a packed view of a packed tensor, "Tq(d<e,c,i<j<k)=T(d<e<c,i<j<k)": an element of D
 *              fixes the values of all labels (increasing inside D's groups), and L is read at them by the same rule, one
 *              signed read per element.  Any two groupings of the same labels are allowed.
 *   tcb_antisym_pack spec "R(a<b<c,i<j<k)+=X(a,i,b<c,j<k)" (or '='): the permutation operator P(a/bc)P(i/jk) of the paper's
 *              notation evaluated on packed storage.  Every group of L must lie inside one group of D.  For
 *              an element of D (one increasing tuple per group) the sum runs over the SHUFFLES of each tuple: the ways to
 *              hand its components to the group's labels such that the labels of one L group, in D's order, receive
 *              increasing components -- 3 for (a | b<c), 6 for (a | b | c), 1 for (a<b<c); sign = parity of the assignment:
 *                  D[tuples] (+)= alpha * sum_shuffles sign * L[at those label values],
 *              terms added in a fixed order (first group of D fastest), then one multiplication by alpha.  With L dense this
 *              is the full antisymmetriser (36 terms for two triples) restricted to a<b<c, i<j<k.  At most 36 terms.
 * Errors: TCB_EINVAL_EXPR (syntax, no group, '+=' in tcb_pack, labels not matching, an L group spread over two D groups in
 * tcb_antisym_pack), TCB_ESHAPE (ranks, unequal extents in a group, packed extent not n choose k), TCB_EUNSUPPORTED (groups
 * of more than 3 labels, repeated label, group labels of extent above 65535 when both sides are packed), TCB_EALIAS.  The
 * first call that meets a new (extent, group size) builds a tuple table on the device: like a first plan, it is refused
 * inside a stream capture. */
int tcb_pack(tcb_ctx *ctx, const char *spec, tcb_tensor *D, const tcb_tensor *L);
int tcb_unpack(tcb_ctx *ctx, const char *spec, tcb_tensor *D, const tcb_tensor *L, tcb_c128 alpha);
int tcb_antisym_pack(tcb_ctx *ctx, const char *spec, tcb_tensor *D, const tcb_tensor *L, tcb_c128 alpha);
int64_t tcb_packed_extent(int64_t n, int k);      /* n choose k for k = 1, 2, 3; -1 otherwise */
/* JSON description of the plan tcb_contract would use: M, N, K, which operands are permuted, GEMM variant,
 * split-K, estimated flops and bytes.  Truncated to buflen-1 characters. */
int tcb_plan_describe(tcb_ctx *ctx, const char *expr, const tcb_tensor *D, const tcb_tensor *L,
                      const tcb_tensor *R, char *buf, size_t buflen);

/* Host-only planning (no device, no context): the same planner on bare shapes.  options: NULL or
 * "key=value;key=value" with the keys of tcb_ctx_set_option.  offM / offN (may be NULL) receive the epilogue
 * offset tables: C[m,n] of the matricised product lands at D[offM[m] + offN[n]]; cap_m / cap_n are the
 * capacities of the two arrays (TCB_EINVAL if too small). */
int tcb_plan_describe_host(const char *expr, int rank_d, const int64_t *ext_d, int rank_l, const int64_t *ext_l,
                           int rank_r, const int64_t *ext_r, const char *options, char *buf, size_t buflen,
                           int64_t *offM, size_t cap_m, int64_t *offN, size_t cap_n);

/* ---- measurement helpers (not part of the hot path) ----------------------------------------------- */

/* Register-resident mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4) loop on every SM for about `milliseconds`;
 * returns achieved TFLOP/s (512 flop per warp instruction).  The roofline denominator of the contraction. */
int tcb_measure_fp64_tensor_peak(tcb_ctx *ctx, double milliseconds, double *tflops);
/* The same for the plain FP64 pipe (register-resident DFMA chains, 2 flop per FMA and lane): on B200 the vector and
 * the tensor FP64 rates are nominally equal; the pair of numbers shows what the tensor path buys. */
int tcb_measure_fp64_vector_peak(tcb_ctx *ctx, double milliseconds, double *tflops);
/* CUDA graph of a call list (a whole residual evaluation: "capture launch-bound inner loops", the paper's barrier per
 * operation, becomes graph edges).  Between tcb_capture_begin and tcb_capture_end every call on the
 * context is RECORDED instead of executed -- kernels, stream-ordered creation and destruction of intermediates --
 * and tcb_graph_launch replays the list on the context's stream (lane 0; calls issued on other lanes inside the capture
 * become parallel branches).  Requirements: the same call list has run at least once before (plans cached, workspace
 * grown, lanes created: none of it may happen inside a capture), "kernel_timing" is off, no upload / download / sync /
 * tcb_denominator_* inside (they copy from host memory).  A call that breaks a requirement returns TCB_EUNSUPPORTED
 * WITHOUT touching the device, the context stays usable, and tcb_capture_end then returns TCB_EUNSUPPORTED and no graph:
 * issue the list call by call instead.  The tensors the list reads and writes must stay alive and at their addresses
 * while the graph is used; so must the context's workspace: tcb_graph_launch returns TCB_EINVAL when a later call has
 * made the workspace grow (its old block, whose address the graph carries, is gone) -- capture again.
 * tcb_launch_count advances by the captured launches per replay.  tcb_graph_info: nodes and dependency edges of the
 * graph, the kernel launches per replay, and depth = the number of nodes on the longest dependency path (a chain has
 * depth = nodes; parallel branches make it smaller).  Any output pointer may be NULL. */
typedef struct tcb_graph tcb_graph;
int tcb_capture_begin(tcb_ctx *ctx);
int tcb_capture_end(tcb_ctx *ctx, tcb_graph **graph);
int tcb_graph_launch(tcb_ctx *ctx, tcb_graph *graph);
int tcb_graph_info(const tcb_graph *graph, int64_t *nodes, int64_t *edges, int64_t *kernel_launches, int64_t *depth);
int tcb_graph_destroy(tcb_graph *graph);
/* Milliseconds between two points of the context's stream: tcb_timer_start / tcb_timer_stop bracket the
 * calls in between with CUDA events on that stream; stop blocks and returns the elapsed time. */
int tcb_timer_start(tcb_ctx *ctx);
int tcb_timer_stop(tcb_ctx *ctx, double *milliseconds);
/* Per-kernel-class device time.  After tcb_ctx_set_option(ctx, "kernel_timing", "on") every kernel launch of
 * the library is bracketed by a CUDA event pair on the context's stream; tcb_kernel_stats synchronises the
 * stream and returns the sums since the last reset for kernel = "zgemm" (the GEMM + epilogue launch, with its
 * split-K reduction when there is one), "permute" (S3 and permuted adds), "permsum" (S6) or "elementwise" (S7).
 * flops / bytes are the ALGORITHMIC counts of those launches (8 M N K; operands read once, D written once and
 * read once more for '+='; a transposition moves 2*16 bytes per element). */
typedef struct { int64_t launches; double milliseconds; double flops; double bytes; } tcb_kernel_stat;
int tcb_kernel_stats(tcb_ctx *ctx, const char *kernel, tcb_kernel_stat *out);
int tcb_kernel_stats_reset(tcb_ctx *ctx);

#ifdef __cplusplus
}
#endif
#endif /* TCB200_H */
