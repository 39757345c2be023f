// plan.cpp -- S2 (host).  "There are different approaches of dealing with tensor transposition ... required
// for the usage of BLAS GEMM, which depends on a unit-stride index": the planner decides which
// transpositions of TTGT are really needed.
//
//  (i)   extent-1 indices are dropped;
//  (ii)  the operand that owns D's unit-stride index becomes the GEMM's row side A (its rows run along the
//        lanes of the epilogue stores), otherwise L and R swap roles;
//  (iii) an operand is fed IN PLACE when its memory order is [free..][contracted..] ("M-major") or
//        [contracted..][free..] ("K-major"), in whatever order inside each group: the order of the free
//        indices is absorbed by the epilogue offset tables offM/offN, and the order of the contracted indices
//        only has to be common to both operands;
//  (iv)  otherwise it is permuted into workspace as [contracted in the common order][free in D's order];
//        if both operands are matrix-shaped but disagree on the contracted order the smaller one is permuted;
//  (v)   an in-place row operand whose fastest free index is not D's unit-stride index would scatter 16-byte
//        stores; it is permuted too when it is no larger than D;
//  (vi)  the result permutation is never a separate pass: alpha*C is scattered by the GEMM epilogue to
//        D[offM[m] + offN[n]];
//  (vii) few output tiles and a long K -> split-K with a deterministic second-stage reduction.
#include "plan.h"

#include <algorithm>
#include <cstdio>
#include <map>
#include <numeric>

#include "../../include/tcb200.h"

namespace tcb {

PermuteShape canonical_permutation(int rank, const int64_t *extent, const int64_t *istride, const int64_t *ostride)
{
    struct Dim { int64_t e, is, os; };
    std::vector<Dim> d;
    for (int k = 0; k < rank; ++k)
        if (extent[k] > 1) d.push_back({extent[k], istride[k], ostride[k]});
    std::sort(d.begin(), d.end(), [](const Dim &a, const Dim &b) { return a.is < b.is; });
    std::vector<Dim> f;
    for (const Dim &x : d) {
        if (!f.empty() && x.is == f.back().is * f.back().e && x.os == f.back().os * f.back().e)
            f.back().e *= x.e;
        else
            f.push_back(x);
    }
    PermuteShape p;
    p.rank = (int)f.size();
    p.identity = true;
    p.volume = 1;
    for (int k = 0; k < p.rank; ++k) {
        p.extent[k] = f[k].e; p.istride[k] = f[k].is; p.ostride[k] = f[k].os;
        if (f[k].is != f[k].os) p.identity = false;
        p.volume *= f[k].e;
    }
    return p;
}

namespace {

struct Lab {
    std::string name;
    int64_t ext = 1;
    int inD = -1, inL = -1, inR = -1;     // positions
    int64_t sD = 0, sL = 0, sR = 0;       // strides (elements)
};

void strides_of(const Shape &s, int64_t *st)
{
    int64_t x = 1;
    for (int k = 0; k < s.rank; ++k) { st[k] = x; x *= s.ext[k]; }
}

bool has_dup(const std::vector<std::string> &v)
{
    for (size_t a = 0; a < v.size(); ++a)
        for (size_t b = a + 1; b < v.size(); ++b)
            if (v[a] == v[b]) return true;
    return false;
}

// offsets of the multi-index enumerated over `order` (first label fastest) in the tensor whose strides `which` picks:
// 0 = D, 1 = L, 2 = R
std::vector<int64_t> offset_table(const std::vector<const Lab *> &order, int which = 0)
{
    auto stride = [which](const Lab *l) { return which == 0 ? l->sD : which == 1 ? l->sL : l->sR; };
    int64_t n = 1;
    for (const Lab *l : order) n *= l->ext;
    std::vector<int64_t> t((size_t)n);
    std::vector<int64_t> idx(order.size(), 0);
    int64_t off = 0;
    for (int64_t i = 0; i < n; ++i) {
        t[(size_t)i] = off;
        for (size_t q = 0; q < order.size(); ++q) {
            off += stride(order[q]);
            if (++idx[q] < order[q]->ext) break;
            off -= stride(order[q]) * order[q]->ext;
            idx[q] = 0;
        }
    }
    return t;
}

std::string join(const std::vector<std::string> &v)
{
    std::string s;
    for (size_t i = 0; i < v.size(); ++i) { if (i) s += ","; s += v[i]; }
    return s;
}

}  // namespace

int plan_contraction(const ParsedExpr &e, const Shape &D, const Shape &L, const Shape &R, const PlanOptions &opt,
                     ContractPlan *out, std::string *why)
{
    auto fail = [&](int code, const char *msg) { if (why) *why = msg; return code; };
    if (!e.has_r) return fail(TCB_EINVAL_EXPR, "contraction needs two operands");
    if ((int)e.d.size() != D.rank || (int)e.l.size() != L.rank || (int)e.r.size() != R.rank)
        return fail(TCB_ESHAPE, "rank of a handle differs from the expression");
    if (has_dup(e.d) || has_dup(e.l) || has_dup(e.r))
        return fail(TCB_EUNSUPPORTED, "label repeated inside one tensor (trace / diagonal)");

    int64_t stD[kMaxRank], stL[kMaxRank], stR[kMaxRank];
    strides_of(D, stD); strides_of(L, stL); strides_of(R, stR);
    std::vector<Lab> labs;
    auto find = [&](const std::string &n) -> Lab * {
        for (Lab &l : labs) if (l.name == n) return &l;
        labs.push_back(Lab());
        labs.back().name = n;
        return &labs.back();
    };
    labs.reserve(3 * kMaxRank);
    for (int k = 0; k < D.rank; ++k) { Lab *l = find(e.d[k]); l->inD = k; l->sD = stD[k]; l->ext = D.ext[k]; }
    for (int k = 0; k < L.rank; ++k) {
        Lab *l = find(e.l[k]);
        if (l->inD >= 0 && l->ext != L.ext[k]) return fail(TCB_ESHAPE, "extent of an index differs between D and L");
        l->inL = k; l->sL = stL[k]; l->ext = L.ext[k];
    }
    for (int k = 0; k < R.rank; ++k) {
        Lab *l = find(e.r[k]);
        if ((l->inD >= 0 || l->inL >= 0) && l->ext != R.ext[k])
            return fail(TCB_ESHAPE, "extent of an index differs between R and D or L");
        l->inR = k; l->sR = stR[k]; l->ext = R.ext[k];
    }
    for (const Lab &l : labs) {
        const int n = (l.inD >= 0) + (l.inL >= 0) + (l.inR >= 0);
        if (n == 3) return fail(TCB_EUNSUPPORTED, "index in D, L and R (batch / Hadamard index)");
        if (n == 1) return fail(TCB_EUNSUPPORTED, "index in only one tensor (trace / broadcast)");
    }

    // (ii) row side = owner of D's unit-stride (first non-trivial) index
    bool swapped = false;
    for (int k = 0; k < D.rank; ++k) {
        const Lab *l = find(e.d[k]);
        if (l->ext > 1) { swapped = (l->inR >= 0); break; }
    }
    const std::vector<std::string> &la = swapped ? e.r : e.l, &lb = swapped ? e.l : e.r;
    auto posA = [&](const Lab *l) { return swapped ? l->inR : l->inL; };
    auto posB = [&](const Lab *l) { return swapped ? l->inL : l->inR; };
    auto strA = [&](const Lab *l) { return swapped ? l->sR : l->sL; };
    auto strB = [&](const Lab *l) { return swapped ? l->sL : l->sR; };

    // memory-order label sequences without extent-1 indices
    std::vector<const Lab *> seqA, seqB, seqD;
    for (const std::string &n : la) { const Lab *l = find(n); if (l->ext > 1) seqA.push_back(l); }
    for (const std::string &n : lb) { const Lab *l = find(n); if (l->ext > 1) seqB.push_back(l); }
    for (const std::string &n : e.d) { const Lab *l = find(n); if (l->ext > 1) seqD.push_back(l); }
    auto is_con = [&](const Lab *l) { return l->inD < 0; };

    struct Shape2 { bool mmajor, kmajor; std::vector<const Lab *> free, con; };
    auto analyse = [&](const std::vector<const Lab *> &seq) {
        Shape2 s;
        for (const Lab *l : seq) (is_con(l) ? s.con : s.free).push_back(l);
        size_t i = 0;
        while (i < seq.size() && !is_con(seq[i])) ++i;
        size_t j = i;
        while (j < seq.size() && is_con(seq[j])) ++j;
        s.mmajor = (j == seq.size());                 // [free..][con..]
        i = 0;
        while (i < seq.size() && is_con(seq[i])) ++i;
        j = i;
        while (j < seq.size() && !is_con(seq[j])) ++j;
        s.kmajor = (j == seq.size());                 // [con..][free..]
        return s;
    };
    Shape2 sa = analyse(seqA), sb = analyse(seqB);

    ContractPlan P;
    P.swapped = swapped;
    P.accumulate = e.accumulate;
    P.M = P.N = P.K = 1;
    for (const Lab *l : sa.free) P.M *= l->ext;
    for (const Lab *l : sb.free) P.N *= l->ext;
    for (const Lab *l : sa.con) P.K *= l->ext;
    int64_t sizeA = P.M * P.K, sizeB = P.N * P.K, sizeD = P.M * P.N;
    if (P.M >= (1LL << 30) || P.N >= (1LL << 30) || P.K >= (1LL << 30))
        return fail(TCB_EUNSUPPORTED, "a matricised extent exceeds 2^30");

    // (vii) GEMV route: B is contracted away completely.  A tensor's offset is a sum over its indices, so A is a matrix
    // with a row table and a column table whatever its index order: no operand is permuted, A is read once in place.
    // Both operands contracted away (rank-0 D: the correlation energy E = 1/4 <ij||ab> t_ij^ab, the 11th CCD diagram of
    // PAPER.md:276) is the same route with a single row.
    if (sb.free.empty() && P.K > 1 && (P.M > 1 || sa.free.empty()) && !seqA.empty() && !opt.permute_always) {
        P.gemv = true;
        P.gemv_kfast = is_con(seqA[0]);
        const int wa = swapped ? 2 : 1, wb = swapped ? 1 : 2;
        P.offM = offset_table(sa.free, 0);              // rows enumerated in A's own memory order
        P.offAm = offset_table(sa.free, wa);
        P.offAk = offset_table(sa.con, wa);
        P.offBk = offset_table(sa.con, wb);
        P.offN.assign(1, 0);
        P.a.permuted = P.b.permuted = false;
        P.a.rows = P.M; P.b.rows = 1; P.a.elems = sizeA; P.b.elems = sizeB;
        P.a.kmajor = P.gemv_kfast; P.b.kmajor = true;
        for (const Lab *l : sa.free) P.m_labels.push_back(l->name);
        for (const Lab *l : sa.con) P.k_labels.push_back(l->name);
        P.splitk = opt.splitk;
        P.splits = gemv_ksplit(P.M, P.K, P.gemv_kfast);
        P.partial_bytes = P.splits > 1 ? (size_t)P.splits * (size_t)P.M * 16 : 0;
        P.flops = 8.0 * (double)P.M * (double)P.K;
        P.bytes = 16.0 * ((double)sizeA + (double)sizeB + (double)sizeD * (e.accumulate ? 2.0 : 1.0));
        P.est_seconds = std::max(P.flops / (37.2e12 * 0.92), P.bytes / 6.0e12) + 4e-6;
        *out = std::move(P);
        return TCB_OK;
    }

    // (vii) regime "outer product": nothing is contracted (tt(a,b,i,j) = T1(a,i) T1(b,j)) -- a store stream, no tensor work:
    // both operands are read through row tables in D's order of their indices
    if (P.K == 1 && !opt.permute_always) {
        std::vector<const Lab *> fa_, fb_;
        for (const Lab *l : seqD) (posA(l) >= 0 ? fa_ : fb_).push_back(l);
        P.outer = true;
        P.offM = offset_table(fa_);
        P.offN = offset_table(fb_);
        P.a.gather_row = offset_table(fa_, swapped ? 2 : 1);
        P.b.gather_row = offset_table(fb_, swapped ? 1 : 2);
        P.a.rows = P.M; P.b.rows = P.N; P.a.elems = sizeA; P.b.elems = sizeB;
        for (const Lab *l : fa_) P.m_labels.push_back(l->name);
        for (const Lab *l : fb_) P.n_labels.push_back(l->name);
        P.splitk = opt.splitk;
        P.flops = 8.0 * (double)P.M * (double)P.N;
        P.bytes = 16.0 * ((double)sizeA + (double)sizeB + (double)sizeD * (e.accumulate ? 2.0 : 1.0));
        P.est_seconds = P.bytes / 6.0e12 + 4e-6;
        *out = std::move(P);
        return TCB_OK;
    }

    // (iii)-(viii) how each operand reaches the GEMM, decided by a cost model.  Per operand three feeds exist:
    //   tma     : read in place by 2-D TMA boxes -- needs a matrix-shaped memory order whose contracted order is the common one;
    //   gather  : read in place through a row table and a column table (any index order);
    //   permute : copied into workspace as [contracted in the common order][free in D's order] first (TTGT).
    // The common contracted order is A's or B's own.  A candidate costs  sum over passes of max(flops / peak, bytes / BW)
    // (SURVEY 8(a) S2 (viii)); bytes count twice where only 16 of a 32-byte sector are used (no contiguous direction for the
    // lanes of a gathered operand; epilogue stores that do not run along D's unit-stride index).
    auto same_order = [&](const std::vector<const Lab *> &x, const std::vector<const Lab *> &y) {
        if (x.size() != y.size()) return false;
        for (size_t i = 0; i < x.size(); ++i) if (x[i] != y[i]) return false;
        return true;
    };
    std::vector<const Lab *> dorderA, dorderB;            // the free labels in D's order
    for (const Lab *l : seqD) if (posA(l) >= 0) dorderA.push_back(l);
    for (const Lab *l : seqD) if (posB(l) >= 0) dorderB.push_back(l);
    struct Feed { int kind; std::vector<const Lab *> forder; bool mfast; double waste; };   // kind: 0 tma, 1 gather, 2 permute
    auto feeds_of = [&](const Shape2 &s, const std::vector<const Lab *> &seq, const std::vector<const Lab *> &dorder,
                        const std::vector<const Lab *> &corder, bool is_a) {
        std::vector<Feed> f;
        const bool matrix = (s.mmajor || s.kmajor) && same_order(s.con, corder);
        if (matrix && !opt.permute_always) f.push_back({0, s.free, false, 1.0});
        if (!opt.permute_always && opt.operand_loads != 2) {
            const Lab *u = seq.empty() ? nullptr : seq[0];           // the operand's unit-stride index
            auto gather = [&](const std::vector<const Lab *> &forder) {
                bool mfast = false;
                int64_t run = 1;
                if (u && !is_con(u)) { mfast = !forder.empty() && forder[0] == u; run = mfast ? u->ext : 1; }
                else if (u) run = (!corder.empty() && corder[0] == u) ? std::min<int64_t>(u->ext, 8) : 1;
                f.push_back({1, forder, mfast, run >= 2 ? 1.0 : 2.0});
            };
            gather(is_a ? dorder : s.free);                          // A: rows in D's order (contiguous epilogue stores)
            if (is_a && !same_order(dorder, s.free)) gather(s.free);  //    or in its own (contiguous loads)
        }
        if (opt.operand_loads != 1 || opt.permute_always) f.push_back({2, dorder, false, 1.0});
        return f;
    };
    // achievable rates on a B200: 0.92 of the FP64 tensor peak, 5.5 TB/s for a transposition pass
    const double kPeak = 37.2e12 * 0.92, kBw = 6.0e12, kBwPerm = 5.5e12, kLaunch = 4e-6;
    // what a gathered operand costs the tensor pipe (table loads, address arithmetic and 4 x LDGSTS per thread and k-tile
    // are issued by the warps that also issue the DMMAs; a gathered operand also keeps the GEMM on four real products).
    // Measured against 0.92 of the peak: 4500^3 and 1600^3 ring terms with both operands gathered 1.34 (1.16 per operand),
    // 100 x 12000 x 79200 with a gathered 15 GB view of T3 1.28, 79200 x 100 x 12000 1.19 (profiles/r2_gemm_ab.md,
    // profiles/r2_ccsdt_packed.md): +18 % per operand whose lanes run along contiguous memory, +30 % when every lane
    // fetches its own 32-byte sector
    // -- in the tensor-bound regime (K >= 256).  A short-K GEMM leaves the issue slots the gather needs idle anyway: there the
    // first calibration stands (+4.5 % / +26 %; R2 += vvvo T1, K = 150: 1.51 ms transposed first, 1.20 ms gathered)
    const double kGatherCost = P.K >= 256 ? 1.18 : 1.045, kGatherScattered = P.K >= 256 ? 1.30 : 1.26;
    const double flops = 8.0 * (double)P.M * (double)P.N * (double)P.K;
    const double bytesD = 16.0 * (double)sizeD * (e.accumulate ? 2.0 : 1.0);
    std::vector<std::vector<const Lab *>> corders;
    corders.push_back(sa.con);
    if (!same_order(sa.con, sb.con)) corders.push_back(sb.con);
    double best = -1.0;
    Feed fa, fb;
    std::vector<const Lab *> corder;
    for (const auto &co : corders)
        for (const Feed &ca : feeds_of(sa, seqA, dorderA, co, true))
            for (const Feed &cb : feeds_of(sb, seqB, dorderB, co, false)) {
                const double wd = (seqD.empty() || (!ca.forder.empty() && ca.forder[0] == seqD[0])) ? 1.0 : 2.0;
                double fl = flops / kPeak;
                // TMA-fed candidates run with three real products per complex product (vii-a): measured 0.80 of the 4M time
                if (opt.complex_product != 1 && ca.kind != 1 && cb.kind != 1 && P.K >= 32) fl *= 0.80;
                if (ca.kind == 1) fl *= ca.waste > 1.0 ? kGatherScattered : kGatherCost;
                if (cb.kind == 1) fl *= cb.waste > 1.0 ? kGatherScattered : kGatherCost;
                const double by = (16.0 * (double)sizeA * ca.waste + 16.0 * (double)sizeB * cb.waste + bytesD * wd) / kBw;
                double t = std::max(fl, by) + kLaunch;
                // 16-byte scattered epilogue stores are not hidden behind the tensor work (one sector per lane instead of
                // four lines per warp instruction): they cost their traffic on top (measured in round 1: permuting a row
                // operand no larger than D first paid off)
                if (wd > 1.0) t += bytesD / kBw;
                if (ca.kind == 2) t += 32.0 * (double)sizeA / kBwPerm + kLaunch;
                if (cb.kind == 2) t += 32.0 * (double)sizeB / kBwPerm + kLaunch;
                if (best < 0 || t < best * (1.0 - 1e-9)) { best = t; fa = ca; fb = cb; corder = co; }
            }
    if (best < 0) return fail(TCB_EUNSUPPORTED, "no way to feed the operands under the given options");
    P.est_seconds = best;
    const std::vector<const Lab *> &forderA = fa.forder, &forderB = fb.forder;

    auto fill_operand = [&](OperandPlan &o, const Feed &f, const Shape2 &s, const std::vector<const Lab *> &seq,
                            int64_t rows, auto strX, int which) {
        o.rows = rows;
        o.elems = rows * P.K;
        o.permuted = f.kind == 2;
        o.gather = f.kind == 1;
        o.mfast = f.mfast;
        if (f.kind == 0) {
            // K = 1: rows contiguous -> M-major; otherwise prefer what the memory order says
            if (s.con.empty()) { o.kmajor = false; o.ld = rows; }
            else if (s.free.empty()) { o.kmajor = true; o.ld = P.K; }
            else if (s.kmajor) { o.kmajor = true; o.ld = P.K; }
            else { o.kmajor = false; o.ld = rows; }
        } else if (f.kind == 1) {
            o.kmajor = true;                   // the layout the gathered k-tile has in shared memory
            o.ld = P.K;
            o.gather_row = offset_table(f.forder, which);
            o.gather_k = offset_table(corder, which);
        } else {
            o.kmajor = true;
            o.ld = P.K;
            int64_t ext[2 * kMaxRank], is[2 * kMaxRank], os[2 * kMaxRank];
            int n = 0;
            int64_t st = 1;
            std::map<const Lab *, int64_t> target;
            for (const Lab *l : corder) { target[l] = st; st *= l->ext; }
            for (const Lab *l : f.forder) { target[l] = st; st *= l->ext; }
            for (const Lab *l : seq) { ext[n] = l->ext; is[n] = strX(l); os[n] = target[l]; ++n; }
            o.perm = canonical_permutation(n, ext, is, os);
        }
    };
    fill_operand(P.a, fa, sa, seqA, P.M, strA, swapped ? 2 : 1);
    fill_operand(P.b, fb, sb, seqB, P.N, strB, swapped ? 1 : 2);

    // (vi) epilogue: fused scatter (default), or -- "epilogue" = "twopass", the third pass of TTGT kept for
    // A/B tests -- the GEMM writes a plain M x N matrix into workspace and a permute-accumulate pass brings it into D
    P.twopass = opt.epilogue == 2;
    if (P.twopass) {
        int64_t ext[2 * kMaxRank], is[2 * kMaxRank], os[2 * kMaxRank];
        int n = 0;
        int64_t st = 1;
        for (const Lab *l : forderA) { ext[n] = l->ext; is[n] = st; os[n] = l->sD; st *= l->ext; ++n; }
        for (const Lab *l : forderB) { ext[n] = l->ext; is[n] = st; os[n] = l->sD; st *= l->ext; ++n; }
        P.c_perm = canonical_permutation(n, ext, is, os);
    }

    P.offM = offset_table(forderA);
    P.offN = offset_table(forderB);
    if (P.twopass) {                       // C[m + n * M]
        for (size_t m = 0; m < P.offM.size(); ++m) P.offM[m] = (int64_t)m;
        for (size_t n = 0; n < P.offN.size(); ++n) P.offN[n] = (int64_t)n * P.M;
    }
    for (const Lab *l : forderA) P.m_labels.push_back(l->name);
    for (const Lab *l : forderB) P.n_labels.push_back(l->name);
    for (const Lab *l : corder) P.k_labels.push_back(l->name);

    // (vii) schedule: whole tiles data-parallel over the persistent grid, the remainder wave (or, for skinny
    // M x N with long K, everything) cut along K -- see gemm_schedule in zgemm.cu
    // (vii-a) complex products from three real ones (3M) where both operands are TMA-fed (in place or after a transposition):
    // measured faster from K = 32 up in every layout pair (+8 % at K = 32, +15 % at 64, +20 ... +27 % from 512 up,
    // profiles/r2_gemm_3m.md); K = 16 loses 6 % (one 16-deep k-tile: no pipelining), a gathered operand makes the gather the
    // bound (0 ... -5 %).  "complex_product" = "3m" / "4m" forces either.
    constexpr int64_t kM3MinK = 32;
    P.m3 = opt.complex_product == 2 || (opt.complex_product == 0 && !P.a.gather && !P.b.gather && P.K >= kM3MinK);
    P.splitk = opt.splitk;
    const GemmSchedule sc = gemm_schedule(P.M, P.N, P.K, opt.splitk, P.m3);
    P.splits = sc.splits;
    P.partial_bytes = sc.partial_bytes;

    P.flops = 8.0 * (double)P.M * (double)P.N * (double)P.K;
    P.bytes = 16.0 * ((double)sizeA + (double)sizeB + (double)sizeD * (e.accumulate ? 2.0 : 1.0));
    *out = std::move(P);
    return TCB_OK;
}

std::string ContractPlan::describe() const
{
    char buf[1280];
    auto feed = [&](const OperandPlan &o) { return (gemv || outer) ? "table" : o.permuted ? "permute" : o.gather ? "gather" : "tma"; };
    std::snprintf(buf, sizeof buf,
                  "{\"M\": %lld, \"N\": %lld, \"K\": %lld, \"m_labels\": \"%s\", \"n_labels\": \"%s\", "
                  "\"k_labels\": \"%s\", \"row_operand\": \"%s\", \"permute_A\": %s, \"permute_B\": %s, "
                  "\"A_layout\": \"%s\", \"B_layout\": \"%s\", \"feed_A\": \"%s\", \"feed_B\": \"%s\", \"splits\": %d, "
                  "\"route\": \"%s\", \"epilogue\": \"%s\", \"accumulate\": %s, \"flops\": %.6g, \"bytes\": %.6g, "
                  "\"est_us\": %.4g, \"complex_product\": \"%s\"}",
                  (long long)M, (long long)N, (long long)K, join(m_labels).c_str(), join(n_labels).c_str(),
                  join(k_labels).c_str(), swapped ? "R" : "L", a.permuted ? "true" : "false",
                  b.permuted ? "true" : "false", a.kmajor ? "K-major" : "M-major", b.kmajor ? "K-major" : "M-major",
                  feed(a), feed(b), splits, gemv ? "gemv" : outer ? "outer" : "gemm", twopass ? "twopass" : "fused-scatter",
                  accumulate ? "true" : "false", flops, bytes, est_seconds * 1e6, (gemv || outer) ? "fma" : m3 ? "3m" : "4m");
    return buf;
}

}  // namespace tcb
