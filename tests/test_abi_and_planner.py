"""-m "not gpu": the C-ABI library loads and exports every symbol include/*.h declares, and the host planner
(S1 + S2, no device needed) makes the choices DESIGN.md describes.  No compute call is made here."""
import ctypes
import glob
import os
import re

import numpy as np
import pytest

import paper_2409_06759_b200 as pkg
from paper_2409_06759_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    names = set()
    for h in glob.glob(os.path.join(ROOT, "include", "*.h")):
        text = re.sub(r"/\*.*?\*/", "", open(h).read(), flags=re.S)
        names |= set(re.findall(r"\b(tcbx?_[a-z0-9_]+)\s*\(", text))
    return names


def test_library_exports_every_declared_symbol():
    lib = pkg.load_library()
    decl = declared_symbols()
    assert len(decl) >= 28
    for name in decl:
        assert hasattr(lib, name), name
    assert decl == set(binding.ABI_SYMBOLS), decl ^ set(binding.ABI_SYMBOLS)


def test_strerror_and_null_handling():
    lib = pkg.load_library()
    assert lib.tcb_strerror(0) == b"ok"
    assert lib.tcb_strerror(-7) == b"unsupported contraction form"
    assert lib.tcb_tensor_destroy(None) == 0
    assert lib.tcb_ctx_destroy(None) == 0
    assert lib.tcb_sync(None) == binding.TCB_EINVAL


def test_no_cpu_fallback_without_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    with pytest.raises(pkg.TcbError) as ei:
        pkg.Context(0)
    assert ei.value.code == binding.TCB_ECUDA


def plan(expr, d, l, r, options=None, tables=False):
    return binding.plan_describe_host(expr, d, l, r, options, want_tables=tables)


def test_config3_ladder_needs_no_permutation():
    o, v = 40, 200
    p = plan("R(a,b,i,j)+=V(a,b,c,d)*T(c,d,i,j)", (v, v, o, o), (v, v, v, v), (v, v, o, o))
    assert (p["M"], p["N"], p["K"]) == (40000, 1600, 40000)
    assert not p["permute_A"] and not p["permute_B"] and p["splits"] == 1
    assert p["A_layout"] == "M-major" and p["B_layout"] == "K-major" and p["row_operand"] == "L"
    assert p["flops"] == 8.0 * 40000 * 1600 * 40000
    # V given as V(c,d,a,b): still in place, K-major
    p = plan("R(a,b,i,j)+=V(c,d,a,b)*T(c,d,i,j)", (v, v, o, o), (v, v, v, v), (v, v, o, o))
    assert not p["permute_A"] and p["A_layout"] == "K-major"
    # T given as T(i,j,c,d): N-major B, still no permutation
    p = plan("R(a,b,i,j)+=V(a,b,c,d)*T(i,j,c,d)", (v, v, o, o), (v, v, v, v), (o, o, v, v))
    assert not p["permute_A"] and not p["permute_B"] and p["B_layout"] == "M-major"


def test_row_operand_is_owner_of_unit_stride_index_of_D():
    p = plan("X(a,b,i,j)=I(a,d)*T(d,b,i,j)", (9, 9, 4, 4), (9, 9), (9, 9, 4, 4))
    assert p["row_operand"] == "L" and p["M"] == 9 and p["N"] == 9 * 16
    p = plan("X(a,b,i,j)=T(d,b,i,j)*I(a,d)", (9, 9, 4, 4), (9, 9, 4, 4), (9, 9))
    assert p["row_operand"] == "R" and p["M"] == 9


def test_ring_term_reads_both_operands_in_place_through_offset_tables():
    """neither operand of the ring term is matrix-shaped; TTGT would transpose both, the
    cost model reads both in place (gather); "operand_loads=permute" gives the TTGT plan back for A/B tests."""
    o, v = 6, 14
    e, shapes = "X(a,b,i,j)=T(a,c,i,k)*I(k,b,c,j)", ((v, v, o, o), (v, v, o, o), (o, v, v, o))
    p = plan(e, *shapes)
    assert (p["M"], p["N"], p["K"]) == (o * v, o * v, o * v)
    assert not p["permute_A"] and not p["permute_B"] and p["feed_A"] == "gather" and p["feed_B"] == "gather"
    assert p["m_labels"] == "a,i"                          # rows in D's order: contiguous epilogue stores
    p = plan(e, *shapes, "operand_loads=permute")
    assert p["permute_A"] and p["permute_B"] and p["feed_A"] == "permute"
    q = plan(e, *shapes, "operand_loads=gather")
    assert q["feed_A"] == "gather" and q["est_us"] < p["est_us"]


def test_cost_model_picks_per_operand_feeds():
    """S2 (viii): candidates cost max(flops / peak, bytes / BW) per pass.  At CC sizes (o=30, v=150): matrix-shaped operands
    stay on TMA; a non-matrix operand of a short-K call (where a transposition pass would cost as much as the GEMM) is
    gathered; the tensor-bound 4500^3 ring terms transpose both operands first (a 0.1 ms pass each against a 21 ms GEMM
    that gathering would slow by more); "operand_loads=gather" removes every transposition."""
    from paper_2409_06759_b200 import ccsd_contractions as cl
    o, v = 30, 150
    seen = set()
    for e, sign, sd, sl, sr in cl.all_calls(o, v):
        p = plan(e, sd, sl, sr)
        assert p["est_us"] > 0
        seen.add((p["feed_A"], p["feed_B"]))
        q = plan(e, sd, sl, sr, "operand_loads=gather")
        assert not q["permute_A"] and not q["permute_B"], (e, q)
        assert q["est_us"] >= p["est_us"] * (1 - 1e-6)        # "auto" never costs more than a forced choice
        big = max(np.prod(sl), np.prod(sr))
        if big >= o * v ** 3 and p["K"] <= 150:                # a v^3 o operand in front of a short-K GEMM: never transposed
            assert not p["permute_A"] and not p["permute_B"], (e, p)
    assert ("tma", "tma") in seen and ("permute", "permute") in seen and any("gather" in fb for fb in seen)
    ring = plan("R2(a,b,i,j)+=T2(a,e,i,m)*Wmbej(m,b,e,j)", (v, v, o, o), (v, v, o, o), (o, v, v, o))
    assert ring["feed_A"] == "permute" and ring["feed_B"] == "permute"
    short = plan("R2(a,b,i,j)+=vvvo(a,b,e,j)*T1(e,i)", (v, v, o, o), (v, v, v, o), (v, o))
    assert short["feed_A"] == "gather" and short["feed_B"] == "tma" and short["m_labels"] == "a,b,j"
    # pp ladder: both in place by TMA, cost = the tensor-bound GEMM
    p = plan("R(a,b,i,j)+=V(a,b,c,d)*T(c,d,i,j)", (v, v, o, o), (v, v, v, v), (v, v, o, o))
    assert p["feed_A"] == "tma" and p["feed_B"] == "tma"
    # ... run with three real products per complex product (0.80 of the four-product time); "4m" costs the full time
    assert p["complex_product"] == "3m"
    assert abs(p["est_us"] - 0.80 * 8.0 * 22500 * 900 * 22500 / (37.2e12 * 0.92) * 1e6) < 0.02 * p["est_us"]
    p4 = plan("R(a,b,i,j)+=V(a,b,c,d)*T(c,d,i,j)", (v, v, o, o), (v, v, v, v), (v, v, o, o), "complex_product=4m")
    assert p4["complex_product"] == "4m"
    assert abs(p4["est_us"] - 8.0 * 22500 * 900 * 22500 / (37.2e12 * 0.92) * 1e6) < 0.02 * p4["est_us"]
    # the two-pass epilogue is an option, never the default
    assert p["epilogue"] == "fused-scatter"
    assert plan("R(a,b,i,j)+=V(a,b,c,d)*T(c,d,i,j)", (v, v, o, o), (v, v, v, v), (v, v, o, o), "epilogue=twopass")["epilogue"] == "twopass"


def test_offset_tables_reproduce_the_contraction():
    """C[m,n] scattered through offM/offN must land where the index string says: checked with numpy on the host."""
    rng = np.random.default_rng(0)
    ext = dict(a=5, b=4, c=3, i=2, j=3, k=2)
    expr = "X(b,i,a,j)=T(a,c,i,k)*I(k,b,c,j)"
    shp = lambda s: tuple(ext[x] for x in s)
    p, offM, offN = plan(expr, shp("biaj"), shp("acik"), shp("kbcj"), tables=True)
    T = rng.standard_normal(shp("acik")) + 1j * rng.standard_normal(shp("acik"))
    I = rng.standard_normal(shp("kbcj")) + 1j * rng.standard_normal(shp("kbcj"))
    ref = np.einsum("acik,kbcj->biaj", T, I)
    m_lab, n_lab, k_lab = p["m_labels"].split(","), p["n_labels"].split(","), p["k_labels"].split(",")
    rowT, colI = (T, I) if p["row_operand"] == "L" else (I, T)
    rl, cl = ("acik", "kbcj") if p["row_operand"] == "L" else ("kbcj", "acik")
    # matricise by hand in the planner's label orders (first label fastest)
    A = np.transpose(rowT, [rl.index(x) for x in m_lab + k_lab]).reshape(p["M"], p["K"], order="F")
    Bm = np.transpose(colI, [cl.index(x) for x in k_lab + n_lab]).reshape(p["K"], p["N"], order="F")
    C = A @ Bm
    flat = np.zeros(ref.size, dtype=np.complex128)
    flat[offM[:, None] + offN[None, :]] = C
    assert np.allclose(flat.reshape(ref.shape, order="F"), ref, atol=1e-12)
    assert len(set((offM[:, None] + offN[None, :]).ravel().tolist())) == ref.size     # a bijection onto D


def test_skinny_contraction_gets_split_k_and_options_override():
    o, v = 30, 150
    p = plan("I(l,i)=W(k,l,c,d)*T(d,c,i,k)", (o, o), (o, o, v, v), (v, v, o, o))
    assert (p["M"], p["N"], p["K"]) == (30, 30, 675000) and p["splits"] > 1
    p = plan("I(l,i)=W(k,l,c,d)*T(d,c,i,k)", (o, o), (o, o, v, v), (v, v, o, o), "splitk=off")
    assert p["splits"] == 1
    p = plan("I(l,i)=W(k,l,c,d)*T(d,c,i,k)", (o, o), (o, o, v, v), (v, v, o, o), "splitk=7")
    assert p["splits"] == 7


@pytest.mark.parametrize("expr,shapes,code", [
    ("D(m,n)+=L(m,k)*R(k,n", [(2, 2)] * 3, binding.TCB_EINVAL_EXPR),
    ("D(m,n)+=L(m,k)", [(2, 2)] * 3, binding.TCB_EINVAL_EXPR),
    ("D(m,n)+=L(m,k)*R(k,n)", [(2, 3), (2, 4), (5, 3)], binding.TCB_ESHAPE),
    ("D(m,n)+=L(m,k,q)*R(k,n)", [(2, 2)] * 3, binding.TCB_ESHAPE),
    ("D(m,n)+=L(m,k)*R(k,q)", [(2, 2)] * 3, binding.TCB_EUNSUPPORTED),       # n, q in one tensor only
    ("D(m,n)+=L(m,n)*R(m,n)", [(2, 2)] * 3, binding.TCB_EUNSUPPORTED),       # Hadamard
    ("D(m,n)+=L(m,k)*R(k,k)", [(2, 2)] * 3, binding.TCB_EUNSUPPORTED),       # trace
])
def test_invalid_contractions_are_rejected(expr, shapes, code):
    with pytest.raises(pkg.TcbError) as ei:
        plan(expr, *shapes)
    assert ei.value.code == code


def test_extent_one_indices_are_dropped_and_labels_may_be_long():
    p = plan("R(p1,x,h1)+=T(p1,e_1,y,h1)*F(e_1,x,y)", (70, 1, 9), (70, 40, 1, 9), (40, 1, 1))
    assert (p["M"], p["N"], p["K"]) == (630, 1, 40)
    # [free][contracted][free] is not matrix-shaped, but N = 1 takes the GEMV route: T is read in place through its row
    # and column offset tables, nothing is permuted
    assert p["route"] == "gemv" and not p["permute_A"] and not p["permute_B"]
    p = plan("R(p1,x,h1,q)+=T(p1,e_1,y,h1)*F(e_1,x,q,y)", (70, 1, 9, 3), (70, 40, 1, 9), (40, 1, 3, 1))
    assert (p["M"], p["N"], p["K"]) == (630, 3, 40) and p["route"] == "gemm" and p["feed_A"] == "gather"
    p = plan("R(p1,x,h1)+=T(p1,y,h1,e_1)*F(e_1,x,y)", (70, 1, 9), (70, 1, 9, 40), (40, 1, 1))
    assert (p["M"], p["N"], p["K"]) == (630, 1, 40) and not p["permute_A"] and p["A_layout"] == "M-major"


class _RecordingContext:
    """Duck-typed stand-in for Context: records the library calls a driver of ccd.py issues (no device, no arithmetic)."""

    class _T:
        def __init__(self, extents):
            self.extents = tuple(int(e) for e in extents)

        def destroy(self):
            pass

    def __init__(self):
        self.contractions, self.antisym, self.adds, self.other = [], [], [], []

    def tensor_create(self, extents, zero=True):
        return self._T(extents)

    def contract(self, expr, D, L, R, alpha=1.0):
        self.contractions.append((expr, D.extents, L.extents, R.extents))

    def antisymmetrize(self, spec, D, X, alpha=1.0):
        assert D.extents == X.extents
        self.antisym.append(spec)

    def add(self, expr, D, L, alpha=1.0):
        self.adds.append(expr)

    def denominator_divide(self, T, R, eps, alpha=1.0):
        assert T.extents == R.extents and len(eps) == len(T.extents)
        self.other.append("divide")

    def dot(self, D, X, Y, conj=True, alpha=1.0):
        assert D.extents == () and X.extents == Y.extents
        self.other.append("dot")


def test_every_contraction_of_the_driver_programs_is_planned_on_the_host():
    """The CCD, CCSD and (T) programs of ccd.py, replayed against a recording context: every contraction string goes
    through the host planner (tcb_plan_describe_host, no device) with the shapes the program gives it; the counts are the
    documented ones and the big operands are never permuted."""
    from paper_2409_06759_b200 import ccd
    o, v = 6, 14
    ext = lambda name: tuple(o if c == "o" else v for c in name)
    rec = _RecordingContext()
    B = {k: rec._T(ext(k[-2:]) if k[0] == "f" else ext(k)) for k in ccd.CCSD_BLOCKS}
    T1, T2 = rec._T((v, o)), rec._T((v, v, o, o))
    ccd.ccd_residual(rec, B, T2)
    n_ccd = len(rec.contractions)
    assert (n_ccd, len(rec.antisym), len(rec.adds)) == (11, 5, 3)
    ccd.ccsd_residual(rec, B, T1, T2)
    assert len(rec.contractions) - n_ccd == 34 and len(rec.antisym) - 5 == 9
    n_before = len(rec.contractions)
    ccd.triples_correction(rec, rec._T((v, v, v, o)), rec._T((o, v, o, o)), T2, [0.0] * o, [0.0] * v,
                           T1=T1, oovv=B["oovv"])
    assert len(rec.contractions) - n_before == 3 and rec.other == ["divide", "dot", "dot"]
    routes = {}
    for expr, d, l, r in rec.contractions:
        p = plan(expr, d, l, r)
        flops = 8.0 * p["M"] * p["N"] * p["K"]
        assert abs(p["flops"] - flops) <= 1e-5 * flops          # the description prints six significant digits
        routes[p["route"]] = routes.get(p["route"], 0) + 1
        big = max(np.prod(l), np.prod(r))
        if np.prod(l) == big and big >= v ** 4:
            assert not p["permute_A" if p["row_operand"] == "L" else "permute_B"], expr     # vvvv-sized operands in place
    assert routes.get("gemv", 0) >= 6 and routes.get("gemm", 0) >= 35
