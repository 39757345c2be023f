// parse.cpp -- S1 (host): the symbolic form in which generated code hands a contraction to the library
// (tensors with index lists + a scalar factor; two tensors per instruction).
#include "parse.h"

#include <cctype>

namespace tcb {

namespace {

struct Cursor {
    const char *p;
    void ws() { while (*p && std::isspace((unsigned char)*p)) ++p; }
    bool eat(char c) { ws(); if (*p == c) { ++p; return true; } return false; }
};

bool ident(Cursor &c, std::string *out)
{
    c.ws();
    if (!std::isalpha((unsigned char)*c.p) && *c.p != '_') return false;
    const char *b = c.p;
    while (std::isalnum((unsigned char)*c.p) || *c.p == '_') ++c.p;
    if (out) out->assign(b, c.p);
    return true;
}

bool tensor(Cursor &c, std::vector<std::string> *labels)
{
    if (!ident(c, nullptr)) return false;          // tensor name: ignored, binding is positional
    if (!c.eat('(')) return false;
    labels->clear();
    if (c.eat(')')) return true;
    for (;;) {
        std::string lab;
        c.ws();
        if (!std::isalpha((unsigned char)*c.p)) return false;
        if (!ident(c, &lab)) return false;
        labels->push_back(lab);
        if (c.eat(',')) continue;
        return c.eat(')');
    }
}

bool sym_tensor(Cursor &c, std::vector<std::vector<std::string>> *items)
{
    if (!ident(c, nullptr)) return false;
    if (!c.eat('(')) return false;
    items->clear();
    if (c.eat(')')) return true;
    for (;;) {
        std::vector<std::string> group;
        for (;;) {
            std::string lab;
            c.ws();
            if (!std::isalpha((unsigned char)*c.p)) return false;
            if (!ident(c, &lab)) return false;
            group.push_back(lab);
            if (!c.eat('<')) break;
        }
        items->push_back(group);
        if (c.eat(',')) continue;
        return c.eat(')');
    }
}

bool expression(Cursor &c, ParsedExpr *e)
{
    if (!tensor(c, &e->d)) return false;
    c.ws();
    if (c.p[0] == '+' && c.p[1] == '=') { e->accumulate = true; c.p += 2; }
    else if (c.p[0] == '=') { e->accumulate = false; c.p += 1; }
    else return false;
    if (!tensor(c, &e->l)) return false;
    e->has_r = false;
    if (c.eat('*')) {
        if (!tensor(c, &e->r)) return false;
        e->has_r = true;
    }
    c.ws();
    return *c.p == 0;
}

}  // namespace

bool parse_expression(const char *text, ParsedExpr *out)
{
    if (!text || !out) return false;
    Cursor c{text};
    return expression(c, out);
}

bool parse_antisym_spec(const char *text, std::vector<PermOperator> *ops, ParsedExpr *expr)
{
    if (!text) return false;
    Cursor c{text};
    ops->clear();
    for (;;) {
        c.ws();
        if (*c.p == ':') { ++c.p; break; }
        if (*c.p != 'P') return false;
        ++c.p;
        if (!c.eat('(')) return false;
        // labels inside an operator are single letters optionally followed by digits: P(ab), P(a/bc), P(p1/p2p3)
        std::vector<std::string> first, second;
        std::vector<std::string> *cur = &first;
        for (;;) {
            c.ws();
            if (*c.p == ')') { ++c.p; break; }
            if (*c.p == '/') { ++c.p; if (cur == &second) return false; cur = &second; continue; }
            if (*c.p == ',') { ++c.p; continue; }
            if (!std::isalpha((unsigned char)*c.p)) return false;
            std::string lab(1, *c.p++);
            while (std::isdigit((unsigned char)*c.p)) lab.push_back(*c.p++);
            cur->push_back(lab);
        }
        PermOperator op;
        if (second.empty()) {                      // P(xy) == P(x/y)
            if (first.size() != 2) return false;
            op.pivot = first[0];
            op.others = {first[1]};
        } else {
            if (first.size() != 1) return false;
            op.pivot = first[0];
            op.others = second;
        }
        ops->push_back(op);
    }
    return expression(c, expr) && !expr->has_r;
}

bool parse_sym_spec(const char *text, SymSpec *out)
{
    if (!text || !out) return false;
    Cursor c{text};
    if (!sym_tensor(c, &out->lhs)) return false;
    c.ws();
    if (c.p[0] == '+' && c.p[1] == '=') { out->accumulate = true; c.p += 2; }
    else if (c.p[0] == '=') { out->accumulate = false; c.p += 1; }
    else return false;
    if (!sym_tensor(c, &out->rhs)) return false;
    c.ws();
    return *c.p == 0;
}

}  // namespace tcb
