// parse.h -- S1: expression strings -> label lists (host).  Grammar in include/tcb200.h.
#pragma once
#include <string>
#include <vector>

namespace tcb {

struct ParsedExpr {
    std::vector<std::string> d, l, r;
    bool has_r = false;
    bool accumulate = false;
};

// false on any syntax error
bool parse_expression(const char *text, ParsedExpr *out);

// "P(a/bc)P(k/ij):D(a,b,c,i,j,k)+=X(a,b,c,i,j,k)" -> operators + expression
struct PermOperator {
    std::string pivot;                  // x in P(x/yz); for P(xy): pivot = x, others = {y}
    std::vector<std::string> others;
};
bool parse_antisym_spec(const char *text, std::vector<PermOperator> *ops, ParsedExpr *expr);

// "Vp(a<b,c<d)=V(a,b,c,d)" / "R(a,b,i,j)+=Rp(a<b,i<j)": each index position is a group of one or more labels joined by '<'
// (index-permutation-symmetric packed storage, tcb_pack / tcb_unpack)
struct SymSpec {
    std::vector<std::vector<std::string>> lhs, rhs;
    bool accumulate = false;
};
bool parse_sym_spec(const char *text, SymSpec *out);

}  // namespace tcb
