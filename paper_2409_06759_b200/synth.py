"""Seeded synthetic inputs (host side, numpy).  Holds NONE of the method's arithmetic.

This module is the one piece shared by the oracle-side tests and the CUDA-side tests/bench: it only
produces input tensors.  It imports neither `oracle` nor the CUDA library.  The device twin is
csrc/synth.cu (same counter-based generator, bit-identical results -- checked by a gpu test), used
where a tensor is too large to generate on the host (config 3: V is 25.6 GB).

Generator:
  key   = splitmix64(seed * 0x9E3779B97F4A7C15 + tensor_id)
  a, b  = splitmix64(key + 2*idx), splitmix64(key + 2*idx + 1)        idx = canonical linear index
  u1    = ((a >> 11) + 1) * 2^-53  in (0, 1]
  z     = sqrt(-2 ln u1) * (cos t + i sin t),  t = 2 pi * (b >> 11) * 2^-53      (Box-Muller)
so ONE draw gives one complex number with Re, Im i.i.d. N(0,1).  ln / sin / cos are evaluated by
fixed polynomial recipes using only IEEE +, *, /, sqrt with every operation rounded on its own
(no FMA), so that numpy and the CUDA kernel agree bit for bit.

Antisymmetrisation (reading #4): for index pairs (p,q),(r,s)
  V = 1/2 [ (g - g(p<->q)) - (g(r<->s) - g(p<->q, r<->s)) ]   evaluated in exactly this order, which makes
  V(p<->q) = -V and V(r<->s) = -V hold bit for bit (x - y == -(y - x) in IEEE arithmetic).
Hermitian-consistent integrals (reading #5): W(pqrs) = 1/2 [A(pqrs) + conj A(rspq)], A antisymmetrised.
"""
import numpy as np

U64 = np.uint64
_M1 = U64(0x9E3779B97F4A7C15)
_M2 = U64(0xBF58476D1CE4E5B9)
_M3 = U64(0x94D049BB133111EB)
LN2 = 0.6931471805599453
HALF_PI = 1.5707963267948966
SQRT_HALF = 0.7071067811865476
N_LOG_TERMS = 12     # atanh series terms: s^(2k)/(2k+1), k = 0..11
N_TRIG_TERMS = 12    # Taylor terms in phi^2


def splitmix64(x):
    with np.errstate(over="ignore"):
        z = (np.asarray(x, dtype=U64) + _M1).astype(U64)
        z = (z ^ (z >> U64(30))) * _M2
        z = (z ^ (z >> U64(27))) * _M3
        return z ^ (z >> U64(31))


def tensor_key(seed, tensor_id):
    with np.errstate(over="ignore"):
        return splitmix64(U64(seed) * _M1 + U64(tensor_id))


def _ln_unit(k53):
    """ln((k53+1) * 2^-53) with a fixed recipe: frexp, fold to [sqrt(.5), sqrt(2)), atanh series (Horner)."""
    x = (k53 + U64(1)).astype(np.float64)                 # exact: <= 2^53
    m, e = np.frexp(x)                                     # x = m * 2^e, m in [0.5, 1)
    small = m < SQRT_HALF
    m = np.where(small, m * 2.0, m)
    e = np.where(small, e - 1, e) - 53
    s = (m - 1.0) / (m + 1.0)
    s2 = s * s
    p = np.full_like(s, _LOG_C[-1])
    for k in range(N_LOG_TERMS - 2, -1, -1):
        p = p * s2 + _LOG_C[k]
    lnm = (2.0 * s) * p
    return e.astype(np.float64) * LN2 + lnm


# hex-float literals; csrc/synth.cu carries the same ones
_SIN_C = [float.fromhex(x) for x in (
    "0x1.0000000000000p+0", "-0x1.5555555555555p-3", "0x1.1111111111111p-7", "-0x1.a01a01a01a01ap-13",
    "0x1.71de3a556c734p-19", "-0x1.ae64567f544e4p-26", "0x1.6124613a86d09p-33", "-0x1.ae7f3e733b81fp-41",
    "0x1.952c77030ad4ap-49", "-0x1.2f49b46814157p-57", "0x1.71b8ef6dcf572p-66", "-0x1.761b413163819p-75")]
_COS_C = [float.fromhex(x) for x in (
    "0x1.0000000000000p+0", "-0x1.0000000000000p-1", "0x1.5555555555555p-5", "-0x1.6c16c16c16c17p-10",
    "0x1.a01a01a01a01ap-16", "-0x1.27e4fb7789f5cp-22", "0x1.1eed8eff8d898p-29", "-0x1.93974a8c07c9dp-37",
    "0x1.ae7f3e733b81fp-45", "-0x1.6827863b97d97p-53", "0x1.e542ba4020225p-62", "-0x1.0ce396db7f853p-70")]
_LOG_C = [float.fromhex(x) for x in (
    "0x1.0000000000000p+0", "0x1.5555555555555p-2", "0x1.999999999999ap-3", "0x1.2492492492492p-3",
    "0x1.c71c71c71c71cp-4", "0x1.745d1745d1746p-4", "0x1.3b13b13b13b14p-4", "0x1.1111111111111p-4",
    "0x1.e1e1e1e1e1e1ep-5", "0x1.af286bca1af28p-5", "0x1.8618618618618p-5", "0x1.642c8590b2164p-5")]


def _cos_sin_turn(k53):
    """(cos, sin) of 2*pi*k53*2^-53: quadrant from the top 2 bits (exact), Taylor in [0, pi/2)."""
    q = (k53 >> U64(51)).astype(np.int64)
    frac = (k53 & U64((1 << 51) - 1)).astype(np.float64) * (2.0 ** -51)
    phi = frac * HALF_PI
    p2 = phi * phi
    sp = np.full_like(phi, _SIN_C[-1])
    cp = np.full_like(phi, _COS_C[-1])
    for k in range(N_TRIG_TERMS - 2, -1, -1):
        sp = sp * p2 + _SIN_C[k]
        cp = cp * p2 + _COS_C[k]
    sp = sp * phi
    c = np.choose(q, [cp, -sp, -cp, sp])
    s = np.choose(q, [sp, cp, -sp, -cp])
    return c, s


def normal_c128(key, idx):
    """One complex N(0,1)+iN(0,1) draw per canonical index (uint64 array)."""
    idx = np.asarray(idx, dtype=U64)
    with np.errstate(over="ignore"):
        a = splitmix64(key + U64(2) * idx)
        b = splitmix64(key + U64(2) * idx + U64(1))
    r = np.sqrt(-2.0 * _ln_unit(a >> U64(11)))
    c, s = _cos_sin_turn(b >> U64(11))
    out = np.empty(idx.shape, dtype=np.complex128)
    out.real = r * c
    out.imag = r * s
    return out


def _scale(z, s):
    """complex * real, component by component (one rounding each)."""
    out = np.empty_like(z)
    out.real = z.real * s
    out.imag = z.imag * s
    return out


def uniform01(key, idx):
    """u in [0,1) with 53 bits, one per index."""
    idx = np.asarray(idx, dtype=U64)
    with np.errstate(over="ignore"):
        a = splitmix64(key + idx)
    return (a >> U64(11)).astype(np.float64) * (2.0 ** -53)


def _grid(sub):
    """list of 1-D index arrays -> broadcastable uint64 index arrays (first index varies fastest in F order)."""
    r = len(sub)
    return [np.asarray(s, dtype=U64).reshape([-1 if k == d else 1 for k in range(r)]) for d, s in enumerate(sub)]


def _linear(idx, label_extents):
    lin = np.zeros((), dtype=U64)
    stride = 1
    with np.errstate(over="ignore"):
        for i, e in zip(idx, label_extents):
            lin = lin + i * U64(stride)
            stride *= int(e)
    return lin


def tensor(seed, tensor_id, extents, antisym=(), sigma=1.0, sub=None, hermitian=False, label_offset=None,
           label_extents=None):
    """Seeded complex tensor, Fortran order.

    extents        : shape of the returned tensor when sub is None.
    label_extents  : extents of the index space the canonical linear index runs over (default: extents);
                     with label_offset (per dim) a block of a larger label space is produced (config 2:
                     blocks of <pq||rs> over all o+v spinors).
    antisym        : up to two index pairs, e.g. ((0,1),(2,3)).
    hermitian      : W(pqrs) = 1/2 [A(pqrs) + conj A(rspq)]   (rank 4 only, all label extents equal).
    sub            : per-dimension index arrays (in LOCAL indices) selecting a sub-tensor; the values are
                     exactly those of the full tensor at those indices.
    """
    rank = len(extents)
    key = tensor_key(seed, tensor_id)
    if label_extents is None:
        label_extents = list(extents)
    if label_offset is None:
        label_offset = [0] * rank
    if sub is None:
        sub = [np.arange(e) for e in extents]
    idx = [g + U64(o) for g, o in zip(_grid(sub), label_offset)]

    def g_at(ix):
        return normal_c128(key, _linear(ix, label_extents))

    def swapped(ix, pair):
        ix = list(ix)
        ix[pair[0]], ix[pair[1]] = ix[pair[1]], ix[pair[0]]
        return ix

    def antisymmetrised(ix):
        if len(antisym) == 0:
            return g_at(ix)
        if len(antisym) == 1:
            return _scale(g_at(ix) - g_at(swapped(ix, antisym[0])), 0.5)
        p, q = antisym
        t1 = g_at(ix) - g_at(swapped(ix, p))
        t2 = g_at(swapped(ix, q)) - g_at(swapped(swapped(ix, p), q))
        return _scale(t1 - t2, 0.5)

    if hermitian:
        assert rank == 4
        A = antisymmetrised(idx)
        Ad = np.conj(antisymmetrised([idx[2], idx[3], idx[0], idx[1]]))
        val = _scale(A + Ad, 0.5)
    else:
        val = antisymmetrised(idx)
    if sigma != 1.0:
        val = _scale(val, sigma)
    shape = [len(s) for s in sub]
    return np.asfortranarray(np.broadcast_to(val, shape)).copy(order="F")


def orbital_energies(seed, o, v):
    """e_occ ~ U(-2,-0.5), e_virt ~ U(0.5,3)   (config 2)."""
    key = tensor_key(seed, 9001)
    u = uniform01(key, np.arange(o + v, dtype=np.uint64))
    eo = -2.0 + 1.5 * u[:o]
    ev = 0.5 + 2.5 * u[o:]
    return eo, ev


def index_linear_tensor(extents):
    """re = canonical linear index, im = -(index) - 0.5: every element distinct, closed-form checkable."""
    n = int(np.prod(extents))
    lin = np.arange(n, dtype=np.float64)
    out = np.empty(n, dtype=np.complex128)
    out.real = lin
    out.imag = -lin - 0.5
    return out.reshape(extents, order="F")


# ---- the BASELINE.json workloads ----------------------------------------------------------------
SEED0 = 20240906


def config_ladder(o, v, config_no, sub_ab=None, sub_ij=None):
    """V(a,b,c,d) antisym (a,b),(c,d); T(c,d,i,j) antisym (c,d),(i,j)  (configs 1, 3)."""
    seed = SEED0 + config_no
    subV = None if sub_ab is None else [sub_ab[0], sub_ab[1], np.arange(v), np.arange(v)]
    subT = None if sub_ij is None else [np.arange(v), np.arange(v), sub_ij[0], sub_ij[1]]
    V = tensor(seed, 1, [v, v, v, v], antisym=((0, 1), (2, 3)), sub=subV)
    T = tensor(seed, 2, [v, v, o, o], antisym=((0, 1), (2, 3)), sub=subT)
    return V, T


def config_ccd(o, v, config_no=2):
    """f (diagonal, stored full), blocks of <pq||rs> ~ complex N(0, 0.1^2) antisymmetric + Hermitian-consistent,
    T2 = <ab||ij> / ((e_i + e_j) - (e_a + e_b))  [this bracketing keeps T2 exactly antisymmetric]."""
    seed = SEED0 + config_no
    n = o + v
    eo, ev = orbital_energies(seed, o, v)
    O, V = (0, o), (o, v)

    def blk(*rng):
        return tensor(seed, 1, [r[1] for r in rng], antisym=((0, 1), (2, 3)), sigma=0.1, hermitian=True,
                      label_offset=[r[0] for r in rng], label_extents=[n] * 4)

    B = {"vvoo": blk(V, V, O, O), "oovv": blk(O, O, V, V), "oooo": blk(O, O, O, O),
         "vvvv": blk(V, V, V, V), "ovvo": blk(O, V, V, O)}
    B["foo"] = np.asfortranarray(np.diag(eo).astype(np.complex128))
    B["fvv"] = np.asfortranarray(np.diag(ev).astype(np.complex128))
    den = (eo[None, None, :, None] + eo[None, None, None, :]) - (ev[:, None, None, None] + ev[None, :, None, None])
    T = np.empty(B["vvoo"].shape, dtype=np.complex128, order="F")
    T.real = B["vvoo"].real / den
    T.imag = B["vvoo"].imag / den
    return B, T, eo, ev


def config_t3(o, v, config_no=4):
    """W(b,c,d,k) antisym (b,c); T2(a,d,i,j) antisym (a,d),(i,j); R3 dense N(0,1)."""
    seed = SEED0 + config_no
    W = tensor(seed, 1, [v, v, v, o], antisym=((0, 1),))
    T2 = tensor(seed, 2, [v, v, o, o], antisym=((0, 1), (2, 3)))
    return W, T2


def config_t3_r3(o, v, config_no=4, sub=None):
    return tensor(SEED0 + config_no, 3, [v, v, v, o, o, o], sub=sub)
