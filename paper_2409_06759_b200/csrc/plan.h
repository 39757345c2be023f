// plan.h -- S2: the contraction planner (host).  Chooses the index grouping (M, N, K), which operands are
// permuted into matrix form, the GEMM variant, split-K, and the epilogue offset tables.
#pragma once
#include <stdint.h>

#include <string>
#include <vector>

#include "kernels.h"
#include "parse.h"

namespace tcb {

struct Shape {
    int rank = 0;
    int64_t ext[kMaxRank] = {1, 1, 1, 1, 1, 1};
    int64_t volume() const { int64_t v = 1; for (int k = 0; k < rank; ++k) v *= ext[k]; return v; }
};

struct PlanOptions {
    int splitk = 0;               // 0 = auto, 1 = off, n > 1 = forced
    int epilogue = 0;             // 0 = auto, 1 = fused, 2 = two-pass (GEMM into workspace + permute-accumulate pass)
    int operand_loads = 0;        // 0 = auto (cost model), 1 = never permute (gather whatever TMA cannot read), 2 = never gather
    int complex_product = 0;      // 0 = auto, 1 = "4m" (four real products per complex product), 2 = "3m" (three; see zgemm.cu)
    bool permute_always = false;  // A/B testing: permute both operands even when they are matrix-shaped
    bool static_deal = false;     // A/B testing: GEMM work dealt statically (tile c + w * grid) instead of claimed
};

// canonical transposition descriptor without pointers (extent-1 dropped, neighbours fused, sorted by input stride)
struct PermuteShape {
    int rank = 0;
    int64_t extent[kMaxRank], istride[kMaxRank], ostride[kMaxRank];
    bool identity = true;        // output order == input order (plain copy)
    int64_t volume = 1;
};
PermuteShape canonical_permutation(int rank, const int64_t *extent, const int64_t *istride, const int64_t *ostride);

struct OperandPlan {
    bool permuted = false;   // copied into workspace in K-major matrix form first
    bool gather = false;     // read in place through gather_row / gather_k (element offsets into the operand)
    bool mfast = false;      // gather: lanes run along the rows (the operand's unit-stride index leads the row order)
    std::vector<int64_t> gather_row, gather_k;
    bool kmajor = false;     // layout the GEMM reads
    int64_t rows = 1, ld = 1, elems = 1;
    PermuteShape perm;       // valid when permuted
};

struct ContractPlan {
    bool swapped = false;    // A := R, B := L (D's unit-stride index lives in R)
    bool accumulate = false;
    int64_t M = 1, N = 1, K = 1;
    OperandPlan a, b;
    std::vector<int64_t> offM, offN;
    // GEMV route (N = 1: one operand fully contracted): the other operand is read in place through these tables
    bool outer = false;      // K = 1 (nothing contracted): the store-stream kernel, rows / columns through a.gather_row / b.gather_row
    bool gemv = false, gemv_kfast = false;
    std::vector<int64_t> offAm, offAk, offBk;
    int splits = 1;          // pieces per tile when every tile is cut along K (skinny shapes), else 1
    int splitk = 0;          // the option the schedule was made with
    size_t partial_bytes = 0; // workspace for the raw fragments of tiles cut along K
    std::vector<std::string> m_labels, n_labels, k_labels;
    double flops = 0, bytes = 0;
    double est_seconds = 0;   // the cost model's estimate for the chosen candidate
    bool m3 = false;          // the GEMM forms complex products from three real ones (3M); decided here, see plan.cpp
    bool twopass = false;     // epilogue: GEMM into a plain M x N workspace matrix, then c_perm brings it into D
    PermuteShape c_perm;
    std::string describe() const;
};

// returns a tcb_status value (0 = ok)
int plan_contraction(const ParsedExpr &e, const Shape &D, const Shape &L, const Shape &R, const PlanOptions &opt,
                     ContractPlan *out, std::string *why);

}  // namespace tcb
