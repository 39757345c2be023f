"""oracle -- CPU oracle of the tensor-contraction hot path.  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package.  It shares no code with paper_2409_06759_b200 and never imports it.

Contents
  contract / permute / add / permsum / scale : ctypes wrappers over oracle/tc_oracle.c ("order A":
      plain nested loops, D index outermost, contracted index innermost).
  contract_order_b : an independent second implementation (own parser, numpy, contracted index
      OUTERMOST, scatter-accumulate into D) used only to pin order A.
  cc : Fock-space (tier 0) and spin-orbital CCD equations (tier 1a / 1b), see oracle/cc.py.

Arrays are numpy complex128 in Fortran order (first index fastest = unit stride), shape = extents.

Pins (tests/test_oracle_*.py, all `-m "not gpu"`): brute-force python loops on tiny extents, order A
vs order B, numpy.einsum / matmul special cases, delta-tensor identity, exact power-of-two scaling,
antisymmetry carried through, closed-form linear-index permutation check, permutation group
identities, antisymmetriser idempotence, Fock-space evaluation of PAPER Eqs. (2)-(4) for the CCD
residual.  Unpinned: the molecular energies of PAPER Tables III/IV (need DIRAC integrals) --
"parity unpinned", out of scope.
"""
import ctypes
import re

import numpy as np

from . import build as _build

_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(_build.build())
        i64p = ctypes.POINTER(ctypes.c_int64)
        dp = ctypes.POINTER(ctypes.c_double)
        lib.orc_contract.argtypes = [ctypes.c_char_p, dp, i64p, dp, i64p, dp, i64p,
                                     ctypes.c_double, ctypes.c_double, ctypes.c_int, dp]
        lib.orc_contract.restype = ctypes.c_int
        lib.orc_permute_add.argtypes = [ctypes.c_char_p, dp, i64p, dp, i64p, ctypes.c_double, ctypes.c_double]
        lib.orc_permute_add.restype = ctypes.c_int
        lib.orc_permsum.argtypes = [dp, i64p, ctypes.c_int, dp, i64p, ctypes.c_int,
                                    ctypes.POINTER(ctypes.c_int32), dp, ctypes.c_double, ctypes.c_double]
        lib.orc_permsum.restype = ctypes.c_int
        lib.orc_scale.argtypes = [dp, ctypes.c_int64, ctypes.c_double, ctypes.c_double]
        lib.orc_scale.restype = ctypes.c_int
        lib.orc_num_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def _dptr(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _ext(a):
    return (ctypes.c_int64 * max(a.ndim, 1))(*a.shape)


def _f(a):
    """complex128, Fortran-contiguous view/copy."""
    a = np.asarray(a, dtype=np.complex128)
    return np.asfortranarray(a)


class OracleError(ValueError):
    pass


def num_threads() -> int:
    return _load().orc_num_threads()


def contract(expr, D, L, R, alpha=1.0, long_double=True, want_snorm=True):
    """D(d..) (+)= alpha*L(l..)*R(r..), order A.  Returns (D_out, snorm); D is not modified.

    snorm[d] = |alpha| * sum_c |L||R| + |D_in[d]| is the normaliser of the parity metric
    (BASELINE.json north_star: "error normalised by sum|L||R| over the contracted indices").
    """
    lib = _load()
    Dw = _f(D).copy(order="F")
    Lf, Rf = _f(L), _f(R)
    sn = np.zeros(Dw.shape, dtype=np.float64, order="F") if want_snorm else None
    a = complex(alpha)
    rc = lib.orc_contract(expr.encode(), _dptr(Dw), _ext(Dw), _dptr(Lf), _ext(Lf), _dptr(Rf), _ext(Rf),
                          a.real, a.imag, 1 if long_double else 0,
                          _dptr(sn) if want_snorm else None)
    if rc != 0:
        raise OracleError(f"orc_contract({expr!r}) -> {rc}")
    return Dw, sn


def contract_inplace_double(expr, D, L, R, alpha=1.0):
    """The timed CPU baseline: order A, double accumulators, no snorm, D (Fortran complex128) updated in place."""
    lib = _load()
    assert D.flags.f_contiguous and L.flags.f_contiguous and R.flags.f_contiguous
    a = complex(alpha)
    rc = lib.orc_contract(expr.encode(), _dptr(D), _ext(D), _dptr(L), _ext(L), _dptr(R), _ext(R),
                          a.real, a.imag, 0, None)
    if rc != 0:
        raise OracleError(f"orc_contract({expr!r}) -> {rc}")
    return D


def permute(expr, L, shapeD):
    """expr "D(i,j,a,b)=L(a,b,i,j)": pure data movement, bit-exact."""
    lib = _load()
    Lf = _f(L)
    Dw = np.zeros(tuple(shapeD), dtype=np.complex128, order="F")
    rc = lib.orc_permute_add(expr.encode(), _dptr(Dw), _ext(Dw), _dptr(Lf), _ext(Lf), 1.0, 0.0)
    if rc != 0:
        raise OracleError(f"orc_permute_add({expr!r}) -> {rc}")
    return Dw


def add(expr, D, L, alpha=1.0):
    """expr "D(a,b,i,j)+=L(b,a,i,j)": D + alpha * permuted L.  Returns a new array."""
    lib = _load()
    Dw = _f(D).copy(order="F")
    Lf = _f(L)
    a = complex(alpha)
    rc = lib.orc_permute_add(expr.encode(), _dptr(Dw), _ext(Dw), _dptr(Lf), _ext(Lf), a.real, a.imag)
    if rc != 0:
        raise OracleError(f"orc_permute_add({expr!r}) -> {rc}")
    return Dw


def permsum(D, X, perms, coefs, beta=1.0):
    """D[i] = beta*D[i] + sum_t coefs[t] * X[i_{perms[t][0]}, i_{perms[t][1]}, ...], terms in order."""
    lib = _load()
    Dw = _f(D).copy(order="F")
    Xf = _f(X)
    perms = np.ascontiguousarray(np.asarray(perms, dtype=np.int32).reshape(len(coefs), Dw.ndim))
    cf = np.ascontiguousarray(np.asarray(coefs, dtype=np.complex128))
    b = complex(beta)
    rc = lib.orc_permsum(_dptr(Dw), _ext(Dw), Dw.ndim, _dptr(Xf), _ext(Xf), len(cf),
                         perms.ctypes.data_as(ctypes.POINTER(ctypes.c_int32)),
                         cf.view(np.float64).ctypes.data_as(ctypes.POINTER(ctypes.c_double)), b.real, b.imag)
    if rc != 0:
        raise OracleError(f"orc_permsum -> {rc}")
    return Dw


def scale(D, alpha):
    lib = _load()
    Dw = _f(D).copy(order="F")
    a = complex(alpha)
    lib.orc_scale(_dptr(Dw), Dw.size, a.real, a.imag)
    return Dw


# ---------------------------------------------------------------------------------------------
# Order B: an independent implementation used only to pin order A ("two independent
# loop orders").  Own parser (regex), contracted multi-index OUTERMOST (and walked in REVERSED
# order), whole-D scatter-accumulate per contracted value via numpy broadcasting.
# ---------------------------------------------------------------------------------------------
_TENSOR_RE = re.compile(r"\s*[A-Za-z_][A-Za-z0-9_]*\s*\(([^()]*)\)\s*")


def _parse_b(expr):
    m = re.fullmatch(r"(.*?)(\+=|=)(.*?)\*(.*)", expr)
    if not m:
        raise OracleError(f"order B cannot parse {expr!r}")
    out = []
    for part in (m.group(1), m.group(3), m.group(4)):
        mm = _TENSOR_RE.fullmatch(part)
        if not mm:
            raise OracleError(f"order B cannot parse {part!r}")
        labs = [s.strip() for s in mm.group(1).split(",")] if mm.group(1).strip() else []
        out.append(labs)
    return out[0], out[1], out[2], m.group(2) == "+="


def contract_order_b(expr, D, L, R, alpha=1.0):
    import itertools
    dl, ll, rl, acc = _parse_b(expr)
    D = np.asarray(D, dtype=np.complex128)
    L = np.asarray(L, dtype=np.complex128)
    R = np.asarray(R, dtype=np.complex128)
    con = [x for x in ll if x not in dl]
    if sorted(con) != sorted(x for x in rl if x not in dl):
        raise OracleError("order B: contracted labels differ between L and R")
    cext = [L.shape[ll.index(x)] for x in con]
    accum = np.zeros(D.shape, dtype=np.clongdouble)
    # move L's free axes / R's free axes into D's axis order with broadcasting singleton axes
    for cidx in reversed(list(itertools.product(*[range(e) for e in cext]))):
        fix = dict(zip(con, cidx))
        Ls = L[tuple(fix.get(x, slice(None)) for x in ll)]
        Rs = R[tuple(fix.get(x, slice(None)) for x in rl)]
        lfree = [x for x in ll if x in dl]
        rfree = [x for x in rl if x in dl]
        Lb = np.transpose(Ls, [lfree.index(x) for x in dl if x in lfree]) if lfree else Ls
        Rb = np.transpose(Rs, [rfree.index(x) for x in dl if x in rfree]) if rfree else Rs
        Lb = Lb.reshape([D.shape[k] if dl[k] in lfree else 1 for k in range(len(dl))])
        Rb = Rb.reshape([D.shape[k] if dl[k] in rfree else 1 for k in range(len(dl))])
        accum += Lb.astype(np.clongdouble) * Rb.astype(np.clongdouble)
    res = np.clongdouble(complex(alpha)) * accum
    if acc:
        res = res + D.astype(np.clongdouble)
    return np.asfortranarray(res.astype(np.complex128))
