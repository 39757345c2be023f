"""oracle.sym -- index-permutation-symmetric (antisymmetric) packed storage, CPU oracle.  TEST INFRASTRUCTURE ONLY.

What it follows: the paper names "index-permutation symmetry" of tensors as the feature its production code does not exploit
yet (PAPER.md:202 feature list, 264 "work in progress", 440 and 452 outlook: the main stated limitation).  The paper gives
no storage scheme, so this is a reading (reading 16), the plainest one:

  * a GROUP  a<b  (or a<b<c) of labels of equal extent n, in which the tensor is antisymmetric, is stored as ONE packed index
    that runs over the strictly increasing tuples only: n(n-1)/2 pairs, n(n-1)(n-2)/6 triples;
  * tuples are enumerated with the FIRST label fastest (the library's column-major convention):
        pairs   (0,1) (0,2) (1,2) (0,3) (1,3) (2,3) ...          p = b(b-1)/2 + a
        triples (0,1,2) (0,1,3) (0,2,3) (1,2,3) (0,1,4) ...      p = c(c-1)(c-2)/6 + b(b-1)/2 + a
  * pack   : Dp[.., p(a<b), ..] = L[.., a, .., b, ..]     (a copy of the stored elements: bit-exact)
  * unpack : D[.., a, .., b, ..] (+)= alpha * sign * Lp[.., p(sorted a,b), ..];  sign = parity of the sorting permutation,
             0 when two labels of a group coincide.  With alpha = 1 and '=' an exactly antisymmetric tensor is reproduced
             bit for bit (negation is exact).

  * a packed VIEW of a packed tensor (groups on both sides of `unpack`, e.g. 'Tq(d<e,c,i<j<k)=T(d<e<c,i<j<k)'): an element
    of D fixes the value of every label; L is read at those values by the same sort-and-sign rule.
  * antisym_pack 'R(a<b<c,i<j<k)+=X(a,i,b<c,j<k)': the paper's permutation operator P(a/bc)P(i/jk) (operators
    "P(a/bc)" are what the generator unrolls into signed permuted terms) with the result kept only on increasing tuples.
    Every group of L lies inside one group of D; for one element of D the sum runs over the shuffles of each tuple -- the
    assignments of its components to the group's labels under which the labels of one L group (in D's order) receive
    increasing components -- each with the parity of the assignment as its sign.

Everything here is explicit Python loops over index tuples (tiny sizes) or numpy `take` on index lists built by those
loops; no closed-form index arithmetic is shared with the CUDA side.
"""
import itertools
import re

import numpy as np


def tuples(n, k):
    """strictly increasing k-tuples of range(n), FIRST element fastest: built by explicit enumeration + sort key"""
    tl = [t for t in itertools.combinations(range(n), k)]
    tl.sort(key=lambda t: tuple(reversed(t)))          # last element slowest ... first element fastest
    return tl


def packed_extent(n, k):
    return len(tuples(n, k))


def _parse_side(text):
    m = re.fullmatch(r"\s*\w+\s*\(([^()]*)\)\s*", text)
    if not m:
        raise ValueError(f"cannot parse {text!r}")
    items = [x.strip() for x in m.group(1).split(",")] if m.group(1).strip() else []
    return [[y.strip() for y in it.split("<")] for it in items]


def parse_both(spec):
    """'R(a<b<c,i<j<k)+=X(a,i,b<c,j<k)' -> (groups of D, groups of L, accumulate); groups allowed on both sides"""
    m = re.fullmatch(r"(.*?)(\+=|=)(.*)", spec)
    if not m:
        raise ValueError(f"cannot parse {spec!r}")
    lhs, rhs = _parse_side(m.group(1)), _parse_side(m.group(3))
    flat_l, flat_r = [x for g in lhs for x in g], [x for g in rhs for x in g]
    if len(set(flat_l)) != len(flat_l) or len(set(flat_r)) != len(flat_r) or set(flat_l) != set(flat_r):
        raise ValueError("every label exactly once on each side")
    if any(len(g) > 3 for g in lhs + rhs):
        raise ValueError("groups of at most three labels")
    return lhs, rhs, m.group(2) == "+="


def parse(spec):
    """'Vp(a<b,c<d)=V(a,b,c,d)' -> (packed items, dense labels, accumulate, packed_on_left)"""
    m = re.fullmatch(r"(.*?)(\+=|=)(.*)", spec)
    if not m:
        raise ValueError(f"cannot parse {spec!r}")
    lhs, rhs = _parse_side(m.group(1)), _parse_side(m.group(3))
    acc = m.group(2) == "+="
    lhs_packed = any(len(it) > 1 for it in lhs)
    rhs_packed = any(len(it) > 1 for it in rhs)
    if lhs_packed == rhs_packed:
        raise ValueError("exactly one side must carry a<b groups")
    return lhs, rhs, acc, lhs_packed


def _sort_sign(vals):
    """(sorted tuple, sign of the sorting permutation), sign 0 when two values coincide -- by bubble sort, counting swaps"""
    v = list(vals)
    if len(set(v)) < len(v):
        return tuple(sorted(v)), 0
    sign = 1
    for i in range(len(v)):
        for j in range(len(v) - 1 - i):
            if v[j] > v[j + 1]:
                v[j], v[j + 1] = v[j + 1], v[j]
                sign = -sign
    return tuple(v), sign


def pack(spec, L):
    """spec 'Vp(a<b,c<d)=V(a,b,c,d)': returns the packed tensor (Fortran order)."""
    items, dense, acc, lhs_packed = parse(spec)
    if not lhs_packed or acc:
        raise ValueError("pack: 'P(a<b,..)=D(a,b,..)'")
    labs = [d[0] for d in dense]
    L = np.asarray(L, dtype=np.complex128)
    ext = dict(zip(labs, L.shape))
    lists = []
    for it in items:
        n = ext[it[0]]
        assert all(ext[x] == n for x in it), "labels of a group need equal extents"
        lists.append(tuples(n, len(it)))
    out = np.zeros([len(t) for t in lists], dtype=np.complex128, order="F")
    for pidx in itertools.product(*[range(len(t)) for t in lists]):
        val = {}
        for it, t, p in zip(items, lists, pidx):
            for lab, x in zip(it, t[p]):
                val[lab] = x
        out[pidx] = L[tuple(val[x] for x in labs)]
    return out


def unpack(spec, Lp, D=None, alpha=1.0, extents=None):
    """spec 'R(a,b,i,j)+=Rp(a<b,i<j)': returns D (+)= alpha * sign * Lp[packed position]; D=None starts from zeros of
    `extents` (dict label -> extent, or taken from the packed extents when unambiguous)."""
    if any("<" in part for part in re.split(r"\+=|=", spec, maxsplit=1)[0].split(",")):
        return _unpack_view(spec, Lp, D, alpha, extents)
    dense, items, acc, lhs_packed = parse(spec)
    if lhs_packed:
        raise ValueError("unpack: 'D(a,b,..)(+)=P(a<b,..)'")
    labs = [d[0] for d in dense]
    Lp = np.asarray(Lp, dtype=np.complex128)
    if D is not None:
        D = np.array(D, dtype=np.complex128, order="F")
        ext = dict(zip(labs, D.shape))
    else:
        ext = dict(extents)
        D = np.zeros([ext[x] for x in labs], dtype=np.complex128, order="F")
    where = []
    for it, pe in zip(items, Lp.shape):
        tl = tuples(ext[it[0]], len(it))
        assert len(tl) == pe, "packed extent does not match the dense extents"
        where.append({t: p for p, t in enumerate(tl)})
    a = complex(alpha)
    for idx in itertools.product(*[range(ext[x]) for x in labs]):
        val = dict(zip(labs, idx))
        sign, pidx = 1, []
        for it, w in zip(items, where):
            srt, sg = _sort_sign([val[x] for x in it])
            sign *= sg
            pidx.append(w.get(srt, 0))
        term = 0.0 if sign == 0 else a * Lp[tuple(pidx)] * sign
        D[idx] = (D[idx] if acc else 0.0) + term
    return D


def _label_extents(groups, shape, ext):
    """fills ext[label] from a tensor's groups and shape: a group of k labels on an index of extent e has the n with
    n-choose-k = e (found by counting tuples)"""
    if len(groups) != len(shape):
        raise ValueError("rank of a tensor differs from the spec")
    for g, e in zip(groups, shape):
        n = len(g)
        while packed_extent(n, len(g)) < e:
            n += 1
        if packed_extent(n, len(g)) != e:
            raise ValueError("an extent is not n-choose-k")
        for x in g:
            if ext.setdefault(x, n) != n:
                raise ValueError("a label has two extents")
    return ext


def _read(groups, where, val, Lp):
    """Lp at the label values `val`: per group sort the values, look the sorted tuple up; (value, sign)"""
    sign, pidx = 1, []
    for g, w in zip(groups, where):
        srt, sg = _sort_sign([val[x] for x in g])
        sign *= sg
        pidx.append(w.get(srt, 0))
    return (0.0 if sign == 0 else Lp[tuple(pidx)]), sign


def _unpack_view(spec, Lp, D, alpha, extents):
    """groups on both sides: D[element] (+)= alpha * sign * Lp[at the label values the element of D fixes]"""
    dg, lg, acc = parse_both(spec)
    Lp = np.asarray(Lp, dtype=np.complex128)
    ext = _label_extents(lg, Lp.shape, dict(extents or {}))
    dl = [tuples(ext[g[0]], len(g)) for g in dg]
    if D is None:
        D = np.zeros([len(t) for t in dl], dtype=np.complex128, order="F")
    else:
        D = np.array(D, dtype=np.complex128, order="F")
    _label_extents(dg, D.shape, ext)
    where = [{t: p for p, t in enumerate(tuples(ext[g[0]], len(g)))} for g in lg]
    a = complex(alpha)
    for pidx in itertools.product(*[range(len(t)) for t in dl]):
        val = {}
        for g, t, p in zip(dg, dl, pidx):
            for lab, x in zip(g, t[p]):
                val[lab] = x
        w, sign = _read(lg, where, val, Lp)
        term = 0.0 if sign == 0 else a * (w * sign)
        D[pidx] = (D[pidx] if acc else 0.0) + term
    return D


def shuffles(group, blocks):
    """the assignments (a tuple: slot -> component) of k components to the k labels of `group` under which, for every block
    (a set of labels), the labels of the block in the group's order receive increasing components; with their parities"""
    k = len(group)
    out = []
    for perm in itertools.permutations(range(k)):
        ok = all(perm[s1] < perm[s2] for s1 in range(k) for s2 in range(s1 + 1, k)
                 if any(group[s1] in b and group[s2] in b for b in blocks))
        if ok:
            inv = sum(1 for s1 in range(k) for s2 in range(s1 + 1, k) if perm[s1] > perm[s2])
            out.append((perm, -1 if inv % 2 else 1))
    return out


def antisym_pack(spec, L, D=None, alpha=1.0, extents=None, magnitudes=False):
    """spec 'R(a<b<c,i<j<k)+=X(a,i,b<c,j<k)': D[tuples] (+)= alpha * sum over the shuffles of sign * L[at the label values];
    the terms are summed with the FIRST group of D running fastest, then multiplied by alpha once.
    magnitudes=True (for the tests' normaliser): every term enters as |L[..]| with sign +."""
    dg, lg, acc = parse_both(spec)
    for g in lg:
        if not any(all(x in d for x in g) for d in dg):
            raise ValueError("a group of L is spread over two groups of D")
    L = np.asarray(L, dtype=np.complex128)
    ext = _label_extents(lg, L.shape, dict(extents or {}))
    dl = [tuples(ext[g[0]], len(g)) for g in dg]
    if D is None:
        D = np.zeros([len(t) for t in dl], dtype=np.complex128, order="F")
    else:
        D = np.array(D, dtype=np.complex128, order="F")
    _label_extents(dg, D.shape, ext)
    where = [{t: p for p, t in enumerate(tuples(ext[g[0]], len(g)))} for g in lg]
    per_group = [shuffles(g, [set(b) for b in lg]) for g in dg]
    # first group fastest: itertools.product runs its LAST argument fastest
    terms = [tuple(reversed(c)) for c in itertools.product(*reversed(per_group))]
    a = complex(alpha)
    for pidx in itertools.product(*[range(len(t)) for t in dl]):
        total = 0.0
        for choice in terms:
            val, sign = {}, 1
            for g, t, p, (perm, sg) in zip(dg, dl, pidx, choice):
                sign *= sg
                for slot, lab in enumerate(g):
                    val[lab] = t[p][perm[slot]]
            w, s2 = _read(lg, where, val, L)
            if sign * s2 != 0:
                total = total + (abs(w) if magnitudes else w * (sign * s2))
        D[pidx] = (D[pidx] if acc else 0.0) + a * total
    return D
