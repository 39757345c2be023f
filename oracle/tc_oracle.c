/*
 * oracle/tc_oracle.c -- TEST INFRASTRUCTURE ONLY (CPU oracle, "order A").
 *
 * Plain nested-loop definition of what the hot path computes.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may call this.  It shares no code with paper_2409_06759_b200/csrc (own
 * parser, own index arithmetic) and never touches a GPU.
 *
 * What it follows:
 *   PAPER.md:87-91 (sec. I.C): a tensor library evaluates C = A x B; TTGT
 *   (transpose, transpose, GEMM, transpose) is only one way to REACH that
 *   result.  The result itself is the plain sum over the contracted indices,
 *   which is what is written here, the way the paper's own checker does it
 *   ("brute-force test code with contractions expressed in
 *   nested for loops").  A term is "a list of tensors, a scalar factor ... and
 *   an output tensor", binary only.
 *
 * Layout (reading #1): generalised column-major -- the FIRST listed
 * index has unit stride ("unit-stride index"; tenpi emits Fortran,
 * PAPER.md:224); element = interleaved (re, im) doubles.
 *
 *   offset(idx) = sum_k idx_k * prod_{m<k} extent_m
 *
 * No blocking, no reordering: D index outermost, contracted index innermost.
 * Build: gcc -O2 -fopenmp -ffp-contract=off -shared -fPIC (see oracle/build.py).
 */
#include <ctype.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORC_MAXRANK 8
#define ORC_MAXLAB 24
#define ORC_LABLEN 16

typedef struct {
    int rank;
    char lab[ORC_MAXRANK][ORC_LABLEN];
} orc_ilist;

typedef struct {
    orc_ilist d, l, r;
    int has_r;
    int accumulate; /* 1: "+=", 0: "=" */
} orc_expr;

/* ---- parser: name '(' [label {',' label}] ')' ('+='|'=') name '(' .. ')' ['*' name '(' .. ')'] ---- */
static const char *skip_ws(const char *p) { while (*p && isspace((unsigned char)*p)) ++p; return p; }

static const char *parse_tensor(const char *p, orc_ilist *t)
{
    p = skip_ws(p);
    if (!isalpha((unsigned char)*p) && *p != '_') return NULL;
    while (isalnum((unsigned char)*p) || *p == '_') ++p;      /* tensor name: ignored */
    p = skip_ws(p);
    if (*p != '(') return NULL;
    ++p;
    t->rank = 0;
    p = skip_ws(p);
    if (*p == ')') return p + 1;
    for (;;) {
        p = skip_ws(p);
        if (!isalpha((unsigned char)*p)) return NULL;
        int n = 0;
        if (t->rank >= ORC_MAXRANK) return NULL;
        while (isalnum((unsigned char)*p) || *p == '_') {
            if (n >= ORC_LABLEN - 1) return NULL;
            t->lab[t->rank][n++] = *p++;
        }
        t->lab[t->rank][n] = 0;
        t->rank++;
        p = skip_ws(p);
        if (*p == ',') { ++p; continue; }
        if (*p == ')') return p + 1;
        return NULL;
    }
}

static int parse_expr(const char *s, orc_expr *e)
{
    const char *p = parse_tensor(s, &e->d);
    if (!p) return -1;
    p = skip_ws(p);
    if (p[0] == '+' && p[1] == '=') { e->accumulate = 1; p += 2; }
    else if (p[0] == '=') { e->accumulate = 0; p += 1; }
    else return -1;
    p = parse_tensor(p, &e->l);
    if (!p) return -1;
    p = skip_ws(p);
    e->has_r = 0;
    if (*p == '*') {
        p = parse_tensor(p + 1, &e->r);
        if (!p) return -1;
        e->has_r = 1;
        p = skip_ws(p);
    }
    return *p == 0 ? 0 : -1;
}

static int find_label(const orc_ilist *t, const char *lab)
{
    for (int k = 0; k < t->rank; ++k)
        if (strcmp(t->lab[k], lab) == 0) return k;
    return -1;
}

static void col_major_strides(int rank, const int64_t *ext, int64_t *str)
{
    int64_t s = 1;
    for (int k = 0; k < rank; ++k) { str[k] = s; s *= ext[k]; }
}

static int64_t volume(int rank, const int64_t *ext)
{
    int64_t v = 1;
    for (int k = 0; k < rank; ++k) v *= ext[k];
    return v;
}

/*
 * D(d..) (+)= alpha * L(l..) * R(r..)
 *
 *   for every multi-index d of D:
 *       s = sum over contracted multi-index c of L[l(d,c)] * R[r(d,c)]      (complex)
 *       S = sum over c of |L[l(d,c)]| * |R[r(d,c)]|
 *       D[d] = (accumulate ? D[d] : 0) + alpha * s
 *       snorm[d] = |alpha| * S + |D_in[d]|          (the parity normaliser of north_star)
 *
 * use_long_double = 1: 80-bit accumulators (parity runs); 0: double (timed baseline).
 * snorm may be NULL.  Returns 0, or a negative code for a malformed / inconsistent expression.
 * Rules: every label occurs exactly twice over D, L, R and at most once per tensor.
 */
int orc_contract(const char *expr, double *D, const int64_t *extD, const double *L, const int64_t *extL,
                 const double *R, const int64_t *extR, double alpha_re, double alpha_im,
                 int use_long_double, double *snorm)
{
    orc_expr e;
    if (parse_expr(expr, &e) != 0 || !e.has_r) return -1;
    int rd = e.d.rank, rl = e.l.rank, rr = e.r.rank;
    int64_t sD[ORC_MAXRANK], sL[ORC_MAXRANK], sR[ORC_MAXRANK];
    col_major_strides(rd, extD, sD);
    col_major_strides(rl, extL, sL);
    col_major_strides(rr, extR, sR);

    /* no label twice inside one tensor */
    const orc_ilist *ts[3] = {&e.d, &e.l, &e.r};
    for (int t = 0; t < 3; ++t)
        for (int a = 0; a < ts[t]->rank; ++a)
            for (int b = a + 1; b < ts[t]->rank; ++b)
                if (strcmp(ts[t]->lab[a], ts[t]->lab[b]) == 0) return -2;

    /* per D index: stride in L and in R (exactly one of them holds it) */
    int64_t dL[ORC_MAXRANK], dR[ORC_MAXRANK];
    for (int k = 0; k < rd; ++k) {
        int il = find_label(&e.l, e.d.lab[k]), ir = find_label(&e.r, e.d.lab[k]);
        if ((il >= 0) == (ir >= 0)) return -3;               /* in both (batch) or in neither */
        dL[k] = il >= 0 ? sL[il] : 0;
        dR[k] = ir >= 0 ? sR[ir] : 0;
        if (il >= 0 && extL[il] != extD[k]) return -4;
        if (ir >= 0 && extR[ir] != extD[k]) return -4;
    }
    /* contracted indices: labels of L not in D; must be in R */
    int nc = 0;
    int64_t cext[ORC_MAXRANK], cL[ORC_MAXRANK], cR[ORC_MAXRANK];
    for (int k = 0; k < rl; ++k) {
        if (find_label(&e.d, e.l.lab[k]) >= 0) continue;
        int ir = find_label(&e.r, e.l.lab[k]);
        if (ir < 0) return -3;                                 /* trace / broadcast index */
        if (extR[ir] != extL[k]) return -4;
        cext[nc] = extL[k]; cL[nc] = sL[k]; cR[nc] = sR[ir]; ++nc;
    }
    for (int k = 0; k < rr; ++k)                              /* every R label is in D or in L */
        if (find_label(&e.d, e.r.lab[k]) < 0 && find_label(&e.l, e.r.lab[k]) < 0) return -3;

    int64_t nD = volume(rd, extD), K = volume(nc, cext);
    double abs_alpha = hypot(alpha_re, alpha_im);
    int acc = e.accumulate;

#pragma omp parallel for schedule(static)
    for (int64_t dlin = 0; dlin < nD; ++dlin) {
        int64_t rem = dlin, offL = 0, offR = 0;
        for (int k = 0; k < rd; ++k) {
            int64_t ik = rem % extD[k];
            rem /= extD[k];
            offL += ik * dL[k];
            offR += ik * dR[k];
        }
        int64_t cidx[ORC_MAXRANK] = {0};
        double din_re = acc ? D[2 * dlin] : 0.0, din_im = acc ? D[2 * dlin + 1] : 0.0;
        double out_re, out_im, S;
        if (use_long_double) {
            long double sre = 0, sim = 0, SS = 0;
            for (int64_t c = 0; c < K; ++c) {
                long double xr = L[2 * offL], xi = L[2 * offL + 1], yr = R[2 * offR], yi = R[2 * offR + 1];
                sre += xr * yr - xi * yi;
                sim += xr * yi + xi * yr;
                if (snorm) SS += hypotl(xr, xi) * hypotl(yr, yi);
                for (int q = 0; q < nc; ++q) {              /* odometer over the contracted multi-index */
                    offL += cL[q]; offR += cR[q];
                    if (++cidx[q] < cext[q]) break;
                    offL -= cL[q] * cext[q]; offR -= cR[q] * cext[q]; cidx[q] = 0;
                }
            }
            long double ar = alpha_re, ai = alpha_im;
            out_re = (double)((long double)din_re + (ar * sre - ai * sim));
            out_im = (double)((long double)din_im + (ar * sim + ai * sre));
            S = (double)SS;
        } else {
            double sre = 0, sim = 0, SS = 0;
            for (int64_t c = 0; c < K; ++c) {
                double xr = L[2 * offL], xi = L[2 * offL + 1], yr = R[2 * offR], yi = R[2 * offR + 1];
                sre += xr * yr - xi * yi;
                sim += xr * yi + xi * yr;
                if (snorm) SS += hypot(xr, xi) * hypot(yr, yi);
                for (int q = 0; q < nc; ++q) {
                    offL += cL[q]; offR += cR[q];
                    if (++cidx[q] < cext[q]) break;
                    offL -= cL[q] * cext[q]; offR -= cR[q] * cext[q]; cidx[q] = 0;
                }
            }
            out_re = din_re + (alpha_re * sre - alpha_im * sim);
            out_im = din_im + (alpha_re * sim + alpha_im * sre);
            S = SS;
        }
        D[2 * dlin] = out_re;
        D[2 * dlin + 1] = out_im;
        if (snorm) snorm[dlin] = abs_alpha * S + hypot(din_re, din_im);
    }
    return 0;
}

/*
 * Permutation / permuted add ("tensor transposition (reshape)"):
 *   expr "D(i,j,a,b)=L(a,b,i,j)"  :  D[off_D(idx)] = L[off_L(idx)]            (pure copy, bit-exact)
 *   expr "D(..)+=L(..)"           :  D[...] = D[...] + alpha * L[...]
 * With '=', alpha must be 1+0i and elements are moved as bytes (NaN payloads, -0.0 preserved).
 */
int orc_permute_add(const char *expr, double *D, const int64_t *extD, const double *L, const int64_t *extL,
                    double alpha_re, double alpha_im)
{
    orc_expr e;
    if (parse_expr(expr, &e) != 0 || e.has_r) return -1;
    int rank = e.d.rank;
    if (e.l.rank != rank) return -3;
    int64_t sL[ORC_MAXRANK], mapL[ORC_MAXRANK];
    col_major_strides(rank, extL, sL);
    for (int k = 0; k < rank; ++k) {
        for (int b = k + 1; b < rank; ++b) if (strcmp(e.d.lab[k], e.d.lab[b]) == 0) return -2;
        int il = find_label(&e.l, e.d.lab[k]);
        if (il < 0) return -3;
        if (extL[il] != extD[k]) return -4;
        mapL[k] = sL[il];
    }
    int copy = !e.accumulate;
    if (copy && !(alpha_re == 1.0 && alpha_im == 0.0)) return -5;
    int64_t n = volume(rank, extD);
#pragma omp parallel for schedule(static)
    for (int64_t dlin = 0; dlin < n; ++dlin) {
        int64_t rem = dlin, off = 0;
        for (int k = 0; k < rank; ++k) { off += (rem % extD[k]) * mapL[k]; rem /= extD[k]; }
        if (copy) {
            memcpy(&D[2 * dlin], &L[2 * off], 16);
        } else {
            double xr = L[2 * off], xi = L[2 * off + 1];
            double pr = alpha_re * xr - alpha_im * xi, pi = alpha_re * xi + alpha_im * xr;
            D[2 * dlin] = D[2 * dlin] + pr;
            D[2 * dlin + 1] = D[2 * dlin + 1] + pi;
        }
    }
    return 0;
}

/*
 * Permute-sum (O3; the generator unrolls permutation operators into signed terms,
 * PAPER.md:194, 230, 284):
 *
 *   D[i] = beta * D[i] + sum_{t=0..nterms-1} c_t * X[pi_t(i)],    terms added in order t = 0,1,...
 *
 * perms[t*rank + k] = s_t(k): position k of X is indexed by D's index number s_t(k), i.e.
 *   pi_t(i) = (i_{s_t(0)}, i_{s_t(1)}, ..., i_{s_t(rank-1)}),
 * so "D(a,b,i,j) += -1 * X(b,a,i,j)" is the term s = (1,0,2,3), c = -1.
 * Each multiply and each add is rounded separately (-ffp-contract=off), complex multiply written out.
 * beta == 0 means D_in is not read (so NaNs in D_in do not propagate).
 */
int orc_permsum(double *D, const int64_t *extD, int rank, const double *X, const int64_t *extX, int nterms,
                const int32_t *perms, const double *coefs /* 2*nterms */, double beta_re, double beta_im)
{
    if (rank < 0 || rank > ORC_MAXRANK) return -3;
    int64_t sX[ORC_MAXRANK];
    col_major_strides(rank, extX, sX);
    for (int t = 0; t < nterms; ++t) {
        int seen[ORC_MAXRANK] = {0};
        for (int k = 0; k < rank; ++k) {
            int p = perms[t * rank + k];
            if (p < 0 || p >= rank || seen[p]) return -2;
            seen[p] = 1;
            if (extX[k] != extD[p]) return -4;
        }
    }
    int64_t n = volume(rank, extD);
    int beta_zero = (beta_re == 0.0 && beta_im == 0.0);
#pragma omp parallel for schedule(static)
    for (int64_t dlin = 0; dlin < n; ++dlin) {
        int64_t idx[ORC_MAXRANK], rem = dlin;
        for (int k = 0; k < rank; ++k) { idx[k] = rem % extD[k]; rem /= extD[k]; }
        double are = 0.0, aim = 0.0;
        if (!beta_zero) {
            double dr = D[2 * dlin], di = D[2 * dlin + 1];
            are = beta_re * dr - beta_im * di;
            aim = beta_re * di + beta_im * dr;
        }
        for (int t = 0; t < nterms; ++t) {
            int64_t off = 0;
            for (int k = 0; k < rank; ++k) off += idx[perms[t * rank + k]] * sX[k];
            double xr = X[2 * off], xi = X[2 * off + 1], cr = coefs[2 * t], ci = coefs[2 * t + 1];
            are = are + (cr * xr - ci * xi);
            aim = aim + (cr * xi + ci * xr);
        }
        D[2 * dlin] = are;
        D[2 * dlin + 1] = aim;
    }
    return 0;
}

/* D *= alpha (north_star "tensor add/scale"; the scalar factor of PAPER.md:230) */
int orc_scale(double *D, int64_t n, double alpha_re, double alpha_im)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < n; ++i) {
        double dr = D[2 * i], di = D[2 * i + 1];
        D[2 * i] = alpha_re * dr - alpha_im * di;
        D[2 * i + 1] = alpha_re * di + alpha_im * dr;
    }
    return 0;
}

int orc_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
