"""oracle/cc.py -- coupled-cluster residuals for the oracle.  TEST INFRASTRUCTURE ONLY.

Three tiers:

tier 0  `fock_space_residuals`: literally the paper's equations.  Jordan-Wigner matrices for the
        a_p, a_p^dagger on the 2^n-dimensional Fock space; the Hamiltonian of PAPER Eq. (4)
        (PAPER.md:298), the cluster operators of Eq. (2), the similarity
        transform and projections of Eq. (3).  Exponentials by their
        terminating series.  n = o+v <= ~8.
tier 1a `ccd_residual_unfactorised`: the 10 spin-orbital CCD doubles terms + 1 energy term
        (= the 11 CCD diagrams of PAPER Table I) as direct sums (numpy.einsum
        as the library primitive for "sum over these indices").  The paper does not print these
        (it cites textbooks); they are PINNED to tier 0 in tests/test_oracle_cc.py.
tier 1b `ccd_residual_program`: the same residual as a list of BINARY tensor operations
        (two tensors per instruction), every line one oracle.contract /
        oracle.permsum / oracle.add call.  This is the config-2 workload.  Pinned to tier 1a.
t3      `t3_term_unfactorised` / `t3_term_program`: the config-4 CCSDT piece
        X(a,b,c,i,j,k) = sum_d <bc||dk> t_ij^ad ;  R3 += P(k/ij) P(a/bc) X  (9 signed terms),
        pinned to the tier-0 triples projection of [H, T2]|Phi0>.

Conventions: spinors 0..o-1 occupied, o..o+v-1 virtual.  g[p,q,r,s] = <pq||rs>.
T2 is stored T[a,b,i,j] = t_ij^ab; integral blocks keep bra-ket order, e.g. oovv[k,l,c,d] = <kl||cd>.
All arrays are complex128 (relativistic spinor basis: complex, no spin symmetry).
"""
import itertools

import numpy as np

import oracle as _o


# ------------------------------------------------------------------------------------------
# tier 0: Fock space
# ------------------------------------------------------------------------------------------
def jordan_wigner(n):
    """a_p = Z^{(x)p} (x) [[0,1],[0,0]] (x) I^{(x)(n-p-1)}; returns list of dense (2^n, 2^n) annihilators."""
    Z = np.diag([1.0, -1.0])
    I2 = np.eye(2)
    low = np.array([[0.0, 1.0], [0.0, 0.0]])
    ops = []
    for p in range(n):
        m = np.array([[1.0]])
        for q in range(n):
            m = np.kron(m, Z if q < p else (low if q == p else I2))
        ops.append(m)
    return ops


class FockSpace:
    def __init__(self, o, v):
        self.o, self.v, self.n = o, v, o + v
        self.a = jordan_wigner(self.n)
        self.ad = [m.T.copy() for m in self.a]          # real matrices: dagger = transpose
        vac = np.zeros(2 ** self.n, dtype=np.complex128)
        vac[0] = 1.0                                     # all sites in state |0> = empty
        phi = vac
        for i in reversed(range(o)):                     # |Phi0> = a+_0 a+_1 ... a+_{o-1} |vac>
            phi = self.ad[i] @ phi
        self.phi0 = phi

    def apply_H(self, f, g, psi):
        """H psi, H = sum h_pq a+_p a_q + 1/4 sum <pq||rs> a+_p a+_q a_s a_r   (PAPER Eq. 4),
        with the bare one-electron part recovered from the Fock matrix: h_pq = f_pq - sum_i <pi||qi>."""
        n, o = self.n, self.o
        h = f - np.einsum("piqi->pq", g[:, :o, :, :o])
        out = np.zeros_like(psi)
        aq = [self.a[q] @ psi for q in range(n)]
        for p in range(n):
            acc = np.zeros_like(psi)
            for q in range(n):
                acc += h[p, q] * aq[q]
            out += self.ad[p] @ acc
        w = np.zeros((n, n, psi.size), dtype=np.complex128)
        for r in range(n):
            for s in range(n):
                w[r, s] = self.a[s] @ aq[r]              # a_s a_r psi
        u = np.einsum("pqrs,rsx->pqx", g, w)
        for p in range(n):
            for q in range(n):
                out += 0.25 * (self.ad[p] @ (self.ad[q] @ u[p, q]))
        return out

    def apply_T(self, t1, t2, psi, t3=None):
        """T psi with T1 = sum t_i^a a+_a a_i, T2 = 1/4 sum t_ij^ab a+_a a+_b a_j a_i (PAPER Eq. 2).
        t1[a,i], t2[a,b,i,j] with a,b counted from the first virtual."""
        o, v = self.o, self.v
        out = np.zeros_like(psi)
        if t1 is not None:
            for a in range(v):
                for i in range(o):
                    out += t1[a, i] * (self.ad[o + a] @ (self.a[i] @ psi))
        if t2 is not None:
            for i in range(o):
                ai = self.a[i] @ psi
                for j in range(o):
                    aji = self.a[j] @ ai
                    for a in range(v):
                        for b in range(v):
                            if t2[a, b, i, j] != 0:
                                out += 0.25 * t2[a, b, i, j] * (self.ad[o + a] @ (self.ad[o + b] @ aji))
        return out

    def apply_T3(self, t3, psi):
        """T3 psi, T3 = 1/36 sum t_ijk^abc a+_a a+_b a+_c a_k a_j a_i (PAPER Eq. 2); t3[a,b,c,i,j,k]."""
        o, v = self.o, self.v
        out = np.zeros_like(psi)
        for i, j, k in itertools.product(range(o), repeat=3):
            low = self.a[k] @ (self.a[j] @ (self.a[i] @ psi))
            if not np.any(low):
                continue
            for a, b, c in itertools.product(range(v), repeat=3):
                if t3[a, b, c, i, j, k] != 0:
                    out += t3[a, b, c, i, j, k] / 36.0 * (self.ad[o + a] @ (self.ad[o + b] @ (self.ad[o + c] @ low)))
        return out

    def exp_T(self, t1, t2, psi, sign=1.0):
        """exp(sign*T) psi by the terminating series (T is nilpotent on a finite Fock space)."""
        out = psi.copy()
        term = psi.copy()
        for k in range(1, self.n + 2):
            term = sign * self.apply_T(t1, t2, term) / k
            if not np.any(term):
                break
            out = out + term
        return out

    def hbar_phi0(self, f, g, t1, t2):
        """exp(-T) H exp(T) |Phi0>."""
        return self.exp_T(t1, t2, self.apply_H(f, g, self.exp_T(t1, t2, self.phi0)), sign=-1.0)

    def project_doubles(self, psi):
        """R[a,b,i,j] = <Phi0| (a+_a a+_b a_j a_i)^dagger |psi>."""
        o, v = self.o, self.v
        R = np.zeros((v, v, o, o), dtype=np.complex128)
        for a, b, i, j in itertools.product(range(v), range(v), range(o), range(o)):
            ket = self.ad[o + a] @ (self.ad[o + b] @ (self.a[j] @ (self.a[i] @ self.phi0)))
            R[a, b, i, j] = np.vdot(ket, psi)
        return R

    def project_singles(self, psi):
        o, v = self.o, self.v
        R = np.zeros((v, o), dtype=np.complex128)
        for a, i in itertools.product(range(v), range(o)):
            R[a, i] = np.vdot(self.ad[o + a] @ (self.a[i] @ self.phi0), psi)
        return R

    def project_triples(self, psi):
        """R3[a,b,c,i,j,k] = <Phi0| (a+_a a+_b a+_c a_k a_j a_i)^dagger |psi>   (tau of PAPER Eq. 2)."""
        o, v = self.o, self.v
        R = np.zeros((v, v, v, o, o, o), dtype=np.complex128)
        for a, b, c, i, j, k in itertools.product(range(v), range(v), range(v), range(o), range(o), range(o)):
            ket = self.a[k] @ (self.a[j] @ (self.a[i] @ self.phi0))
            ket = self.ad[o + a] @ (self.ad[o + b] @ (self.ad[o + c] @ ket))
            R[a, b, c, i, j, k] = np.vdot(ket, psi)
        return R


def fock_space_residuals(o, v, f, g, t2, t1=None):
    """(E_corr, R1, R2) from PAPER Eq. (3): <Phi0|Hbar|Phi0> - <Phi0|H|Phi0> and <Phi_l|Hbar|Phi0>."""
    fs = FockSpace(o, v)
    psi = fs.hbar_phi0(f, g, t1, t2)
    e_ref = np.vdot(fs.phi0, fs.apply_H(f, g, fs.phi0))
    e = np.vdot(fs.phi0, psi) - e_ref
    return e, fs.project_singles(psi), fs.project_doubles(psi)


# ------------------------------------------------------------------------------------------
# integral blocks
# ------------------------------------------------------------------------------------------
def blocks(o, f, g):
    """Slices of f and <pq||rs> in bra-ket order, Fortran-contiguous copies."""
    O, V = slice(0, o), slice(o, None)
    F = lambda x: np.asfortranarray(x)
    return {
        "foo": F(f[O, O]), "fvv": F(f[V, V]), "fov": F(f[O, V]), "fvo": F(f[V, O]),
        "vvoo": F(g[V, V, O, O]), "oovv": F(g[O, O, V, V]), "oooo": F(g[O, O, O, O]),
        "vvvv": F(g[V, V, V, V]), "ovvo": F(g[O, V, V, O]),
    }


# ------------------------------------------------------------------------------------------
# tier 1a: un-factorised CCD, 10 amplitude terms + energy
# ------------------------------------------------------------------------------------------
def _P(X, ax1, ax2):
    """P(pq) X = X - X(p<->q)."""
    return X - np.swapaxes(X, ax1, ax2)


def ccd_residual_unfactorised(o, f, g, t):
    """R[a,b,i,j] and E_corr;  t[a,b,i,j] = t_ij^ab.

    R_ij^ab = <ab||ij> + P(ab) f_bc t_ij^ac - P(ij) f_kj t_ik^ab + 1/2 <kl||ij> t_kl^ab
            + 1/2 <ab||cd> t_ij^cd + P(ij)P(ab) <kb||cj> t_ik^ac + 1/4 <kl||cd> t_ij^cd t_kl^ab
            + P(ij) <kl||cd> t_ik^ac t_jl^bd - 1/2 P(ij) <kl||cd> t_ik^dc t_lj^ab
            - 1/2 P(ab) <kl||cd> t_lk^ac t_ij^db ;       E = 1/4 <ij||ab> t_ij^ab
    """
    B = blocks(o, f, g)
    es = np.einsum
    terms = [
        B["vvoo"].copy(),
        _P(es("bc,acij->abij", B["fvv"], t), 0, 1),
        -_P(es("kj,abik->abij", B["foo"], t), 2, 3),
        0.5 * es("klij,abkl->abij", B["oooo"], t),
        0.5 * es("abcd,cdij->abij", B["vvvv"], t),
        _P(_P(es("kbcj,acik->abij", B["ovvo"], t), 2, 3), 0, 1),
        0.25 * es("klcd,cdij,abkl->abij", B["oovv"], t, t),
        _P(es("klcd,acik,bdjl->abij", B["oovv"], t, t), 2, 3),
        -0.5 * _P(es("klcd,dcik,ablj->abij", B["oovv"], t, t), 2, 3),
        -0.5 * _P(es("klcd,aclk,dbij->abij", B["oovv"], t, t), 0, 1),
    ]
    e_terms = [0.25 * es("ijab,abij->", B["oovv"], t)]
    return sum(terms), sum(e_terms), len(terms), len(e_terms)


# ------------------------------------------------------------------------------------------
# tier 1b: the factorised program of binary operations (config 2)
# ------------------------------------------------------------------------------------------
P_AB = ([[0, 1, 2, 3], [1, 0, 2, 3]], [1, -1])
P_IJ = ([[0, 1, 2, 3], [0, 1, 3, 2]], [1, -1])
P_IJ_AB = ([[0, 1, 2, 3], [1, 0, 2, 3], [0, 1, 3, 2], [1, 0, 3, 2]], [1, -1, -1, 1])


def ccd_residual_program(B, T, long_double=True):
    """The CCD residual as binary contractions + permute-sums, each one oracle call.

    B: dict of blocks (see `blocks`), T[a,b,i,j].  Returns (R, list of (name, snorm-free info)).
    Every line is D (+)= alpha * L * R or D += sum_t c_t X[pi_t].
    """
    v, o = T.shape[0], T.shape[2]
    z = lambda *s: np.zeros(s, dtype=np.complex128, order="F")
    con = lambda e, D, L, R, a=1.0: _o.contract(e, D, L, R, a, long_double=long_double, want_snorm=False)[0]

    def acc(R, X, PS, s):
        return _o.permsum(R, X, PS[0], [s * c for c in PS[1]], 1.0)

    R = np.asfortranarray(B["vvoo"]).copy(order="F")                       # driver <ab||ij>
    X = con("X(a,b,i,j)=T(a,c,i,j)*f(b,c)", z(v, v, o, o), T, B["fvv"])
    R = acc(R, X, P_AB, +1.0)                                               # + P(ab) f_bc t_ij^ac
    X = con("X(a,b,i,j)=T(a,b,i,k)*f(k,j)", z(v, v, o, o), T, B["foo"])
    R = acc(R, X, P_IJ, -1.0)                                               # - P(ij) f_kj t_ik^ab
    I1 = con("I1(k,l,i,j)+=W(k,l,c,d)*T(c,d,i,j)", B["oooo"], B["oovv"], T, 0.5)
    R = con("R(a,b,i,j)+=T(a,b,k,l)*I1(k,l,i,j)", R, T, I1, 0.5)           # hh ladder + 1/4 quadratic
    R = con("R(a,b,i,j)+=V(a,b,c,d)*T(c,d,i,j)", R, B["vvvv"], T, 0.5)     # pp ladder
    I2 = con("I2(k,b,c,j)+=W(k,l,c,d)*T(b,d,j,l)", B["ovvo"], B["oovv"], T, 0.5)
    X = con("X(a,b,i,j)=T(a,c,i,k)*I2(k,b,c,j)", z(v, v, o, o), T, I2)
    R = acc(R, X, P_IJ_AB, +1.0)                                            # ring + quadratic ring
    I3 = con("I3(l,i)=W(k,l,c,d)*T(d,c,i,k)", z(o, o), B["oovv"], T)
    X = con("X(a,b,i,j)=T(a,b,l,j)*I3(l,i)", z(v, v, o, o), T, I3)
    R = acc(R, X, P_IJ, -0.5)
    I4 = con("I4(a,d)=W(k,l,c,d)*T(a,c,l,k)", z(v, v), B["oovv"], T)
    X = con("X(a,b,i,j)=I4(a,d)*T(d,b,i,j)", z(v, v, o, o), I4, T)
    R = acc(R, X, P_AB, -0.5)
    return R


# ------------------------------------------------------------------------------------------
# CCSD (next row 8(f)-3; the paper's scaling benchmark is a CCSD iteration).  The paper prints only
# Eqs. (1)-(4); these are the textbook intermediates (Stanton et al. form, refs. at PAPER.md:216) in residual form (full
# Fock matrix, no denominators), PINNED to tier 0 in tests/test_oracle_cc.py.  t1[a,i] = t_i^a.
# ------------------------------------------------------------------------------------------
def block(o, g, name):
    """<pq||rs> block by letters, e.g. 'ovvo' -> g[O,V,V,O] (bra-ket order), Fortran-contiguous."""
    rng = {"o": slice(0, o), "v": slice(o, None)}
    return np.asfortranarray(g[tuple(rng[c] for c in name)])


CCSD_BLOCKS = ("vvoo", "oovv", "oooo", "vvvv", "ovvo", "ooov", "ovvv", "vovv", "oovo", "ovov", "vvvo", "ovoo")


def ccsd_blocks(o, f, g):
    B = {name: block(o, g, name) for name in CCSD_BLOCKS}
    O, V = slice(0, o), slice(o, None)
    for name, sl in (("foo", (O, O)), ("fvv", (V, V)), ("fov", (O, V)), ("fvo", (V, O))):
        B[name] = np.asfortranarray(f[sl])
    return B


def ccsd_residual_unfactorised(o, f, g, t1, t2):
    """(E_corr, R1[a,i], R2[a,b,i,j]) of spin-orbital CCSD:
    tau~ = t2 + 1/2 (t1 t1 - a<->b), tau = t2 + t1 t1 - a<->b
    Fae = f_ae - 1/2 f_me t_m^a + t_m^f <ma||fe> - 1/2 tau~_mn^af <mn||ef>
    Fmi = f_mi + 1/2 t_i^e f_me + t_n^e <mn||ie> + 1/2 tau~_in^ef <mn||ef>;   Fme = f_me + t_n^f <mn||ef>
    Wmnij = <mn||ij> + P(ij) t_j^e <mn||ie> + 1/4 tau_ij^ef <mn||ef>
    Wabef = <ab||ef> - P(ab) t_m^b <am||ef> + 1/4 tau_mn^ab <mn||ef>
    Wmbej = <mb||ej> + t_j^f <mb||ef> - t_n^b <mn||ej> - (1/2 t_jn^fb + t_j^f t_n^b) <mn||ef>
    R1 = f_ai + t_i^e Fae - t_m^a Fmi + t_im^ae Fme - t_n^f <na||if> - 1/2 t_im^ef <ma||ef> - 1/2 t_mn^ae <nm||ei>
    R2 = <ab||ij> + P(ab) t_ij^ae (Fbe - 1/2 t_m^b Fme) - P(ij) t_im^ab (Fmj + 1/2 t_j^e Fme) + 1/2 tau_mn^ab Wmnij
         + 1/2 tau_ij^ef Wabef + P(ij)P(ab) (t_im^ae Wmbej - t_i^e t_m^a <mb||ej>) + P(ij) t_i^e <ab||ej> - P(ab) t_m^a <mb||ij>
    E = f_ia t_i^a + 1/4 <ij||ab> t_ij^ab + 1/2 <ij||ab> t_i^a t_j^b"""
    B = ccsd_blocks(o, f, g)
    es = np.einsum
    tt = es("ai,bj->abij", t1, t1)
    tau_t = t2 + 0.5 * (tt - tt.transpose(1, 0, 2, 3))
    tau = t2 + tt - tt.transpose(1, 0, 2, 3)
    Fae = (B["fvv"] - 0.5 * es("me,am->ae", B["fov"], t1) + es("fm,mafe->ae", t1, B["ovvv"])
           - 0.5 * es("afmn,mnef->ae", tau_t, B["oovv"]))
    Fmi = (B["foo"] + 0.5 * es("ei,me->mi", t1, B["fov"]) + es("en,mnie->mi", t1, B["ooov"])
           + 0.5 * es("efin,mnef->mi", tau_t, B["oovv"]))
    Fme = B["fov"] + es("fn,mnef->me", t1, B["oovv"])
    Wmnij = B["oooo"] + _P(es("ej,mnie->mnij", t1, B["ooov"]), 2, 3) + 0.25 * es("efij,mnef->mnij", tau, B["oovv"])
    Wabef = B["vvvv"] - _P(es("bm,amef->abef", t1, B["vovv"]), 0, 1) + 0.25 * es("abmn,mnef->abef", tau, B["oovv"])
    Wmbej = (B["ovvo"] + es("fj,mbef->mbej", t1, B["ovvv"]) - es("bn,mnej->mbej", t1, B["oovo"])
             - es("fbjn,mnef->mbej", 0.5 * t2 + es("fj,bn->fbjn", t1, t1), B["oovv"]))
    R1 = (B["fvo"] + es("ei,ae->ai", t1, Fae) - es("am,mi->ai", t1, Fmi) + es("aeim,me->ai", t2, Fme)
          - es("fn,naif->ai", t1, B["ovov"]) - 0.5 * es("efim,maef->ai", t2, B["ovvv"])
          - 0.5 * es("aemn,nmei->ai", t2, B["oovo"]))
    R2 = (B["vvoo"]
          + _P(es("aeij,be->abij", t2, Fae - 0.5 * es("bm,me->be", t1, Fme)), 0, 1)
          - _P(es("abim,mj->abij", t2, Fmi + 0.5 * es("ej,me->mj", t1, Fme)), 2, 3)
          + 0.5 * es("abmn,mnij->abij", tau, Wmnij) + 0.5 * es("efij,abef->abij", tau, Wabef)
          + _P(_P(es("aeim,mbej->abij", t2, Wmbej) - es("ei,am,mbej->abij", t1, t1, B["ovvo"]), 2, 3), 0, 1)
          + _P(es("ei,abej->abij", t1, B["vvvo"]), 2, 3) - _P(es("am,mbij->abij", t1, B["ovoo"]), 0, 1))
    E = es("ia,ai->", B["fov"], t1) + 0.25 * es("ijab,abij->", B["oovv"], t2) + 0.5 * es("ijab,ai,bj->", B["oovv"], t1, t1)
    return E, R1, R2


def ccsd_residual_program(B, T1, T2, long_double=True):
    """The CCSD residuals as BINARY tensor operations, every line one oracle.contract / oracle.add /
    oracle.permsum call -- the same list of operations `paper_2409_06759_b200.ccd.ccsd_residual` issues to the library.
    B: `ccsd_blocks`; T1[a,i], T2[a,b,i,j].  Returns (E, R1, R2).  Pinned to `ccsd_residual_unfactorised`."""
    v, o = T1.shape
    z = lambda *s: np.zeros(s, dtype=np.complex128, order="F")
    cp = lambda x: np.asfortranarray(x).copy(order="F")
    con = lambda e, D, L, R, a=1.0: _o.contract(e, D, L, R, a, long_double=long_double, want_snorm=False)[0]

    def acc(D, X, PS, s):
        return _o.permsum(D, X, PS[0], [s * c for c in PS[1]], 1.0)

    tt = con("tt(a,b,i,j)=T1(a,i)*T1(b,j)", z(v, v, o, o), T1, T1)
    taut = acc(cp(T2), tt, P_AB, 0.5)
    tau = acc(cp(T2), tt, P_AB, 1.0)
    Fae = con("F(a,e)+=T1(a,m)*f(m,e)", cp(B["fvv"]), T1, B["fov"], -0.5)
    Fae = con("F(a,e)+=W(m,a,f,e)*T1(f,m)", Fae, B["ovvv"], T1, 1.0)
    Fae = con("F(a,e)+=t(a,f,m,n)*W(m,n,e,f)", Fae, taut, B["oovv"], -0.5)
    Fmi = con("F(m,i)+=f(m,e)*T1(e,i)", cp(B["foo"]), B["fov"], T1, 0.5)
    Fmi = con("F(m,i)+=W(m,n,i,e)*T1(e,n)", Fmi, B["ooov"], T1, 1.0)
    Fmi = con("F(m,i)+=W(m,n,e,f)*t(e,f,i,n)", Fmi, B["oovv"], taut, 0.5)
    Fme = con("F(m,e)+=W(m,n,e,f)*T1(f,n)", cp(B["fov"]), B["oovv"], T1, 1.0)
    X = con("X(m,n,i,j)=W(m,n,i,e)*T1(e,j)", z(o, o, o, o), B["ooov"], T1)
    Wmnij = acc(cp(B["oooo"]), X, P_IJ, 1.0)
    Wmnij = con("W(m,n,i,j)+=V(m,n,e,f)*t(e,f,i,j)", Wmnij, B["oovv"], tau, 0.25)
    X = con("X(a,b,e,f)=V(a,m,e,f)*T1(b,m)", z(v, v, v, v), B["vovv"], T1)
    Wabef = acc(cp(B["vvvv"]), X, P_AB, -1.0)
    Wabef = con("W(a,b,e,f)+=t(a,b,m,n)*V(m,n,e,f)", Wabef, tau, B["oovv"], 0.25)
    Q = _o.add("Q(f,b,j,n)+=t(f,b,j,n)", _o.add("Q(f,b,j,n)+=T2(f,b,j,n)", z(v, v, o, o), T2, 0.5), tt, 1.0)
    Wmbej = con("W(m,b,e,j)+=V(m,b,e,f)*T1(f,j)", cp(B["ovvo"]), B["ovvv"], T1, 1.0)
    Wmbej = con("W(m,b,e,j)+=V(m,n,e,j)*T1(b,n)", Wmbej, B["oovo"], T1, -1.0)
    Wmbej = con("W(m,b,e,j)+=V(m,n,e,f)*Q(f,b,j,n)", Wmbej, B["oovv"], Q, -1.0)
    R1 = con("R(a,i)+=F(a,e)*T1(e,i)", cp(B["fvo"]), Fae, T1, 1.0)
    R1 = con("R(a,i)+=T1(a,m)*F(m,i)", R1, T1, Fmi, -1.0)
    R1 = con("R(a,i)+=T2(a,e,i,m)*F(m,e)", R1, T2, Fme, 1.0)
    R1 = con("R(a,i)+=V(n,a,i,f)*T1(f,n)", R1, B["ovov"], T1, -1.0)
    R1 = con("R(a,i)+=V(m,a,e,f)*T2(e,f,i,m)", R1, B["ovvv"], T2, -0.5)
    R1 = con("R(a,i)+=T2(a,e,m,n)*V(n,m,e,i)", R1, T2, B["oovo"], -0.5)
    G = con("G(b,e)+=T1(b,m)*F(m,e)", cp(Fae), T1, Fme, -0.5)
    X = con("X(a,b,i,j)=T2(a,e,i,j)*G(b,e)", z(v, v, o, o), T2, G)
    R2 = acc(cp(B["vvoo"]), X, P_AB, 1.0)
    Gm = con("G(m,j)+=F(m,e)*T1(e,j)", cp(Fmi), Fme, T1, 0.5)
    X = con("X(a,b,i,j)=T2(a,b,i,m)*G(m,j)", z(v, v, o, o), T2, Gm)
    R2 = acc(R2, X, P_IJ, -1.0)
    R2 = con("R(a,b,i,j)+=t(a,b,m,n)*W(m,n,i,j)", R2, tau, Wmnij, 0.5)
    R2 = con("R(a,b,i,j)+=W(a,b,e,f)*t(e,f,i,j)", R2, Wabef, tau, 0.5)
    X = con("X(a,b,i,j)=T2(a,e,i,m)*W(m,b,e,j)", z(v, v, o, o), T2, Wmbej)
    Z = con("Z(m,b,i,j)=V(m,b,e,j)*T1(e,i)", z(o, v, o, o), B["ovvo"], T1)
    X = con("X(a,b,i,j)+=T1(a,m)*Z(m,b,i,j)", X, T1, Z, -1.0)
    R2 = acc(R2, X, P_IJ_AB, 1.0)
    X = con("X(a,b,i,j)=V(a,b,e,j)*T1(e,i)", z(v, v, o, o), B["vvvo"], T1)
    R2 = acc(R2, X, P_IJ, 1.0)
    X = con("X(a,b,i,j)=T1(a,m)*V(m,b,i,j)", z(v, v, o, o), T1, B["ovoo"])
    R2 = acc(R2, X, P_AB, -1.0)
    E = con("E()=f(i,a)*T1(a,i)", np.zeros(()), B["fov"], T1, 1.0)
    E = con("E()+=V(i,j,a,b)*T2(a,b,i,j)", E, B["oovv"], T2, 0.25)
    E = con("E()+=V(i,j,a,b)*t(a,b,i,j)", E, B["oovv"], tt, 0.5)
    return complex(np.asarray(E).reshape(-1)[0]), R1, R2


# ------------------------------------------------------------------------------------------
# next row 8(f)-3: the Jacobi iteration around the residual (energy denominators; a "CC iteration",
# PAPER.md:406-410).  The paper does not print the update; it is the textbook fixed-point step, PINNED in
# tests/test_oracle_cc.py: the first step from T = 0 is the MP2 amplitude closed form, and the converged
# amplitudes zero the tier-0 (Fock-space) doubles projection.
# ------------------------------------------------------------------------------------------
def denominator_update(T, R, eps, alpha=1.0):
    """T[i0,i1,..] + alpha * R[i0,i1,..] / (eps[0][i0] + eps[1][i1] + ...), energies summed in index order,
    real and imaginary parts divided separately.  eps[k] = None: index k does not enter."""
    d = np.zeros(T.shape, dtype=np.float64, order="F")
    for k, e in enumerate(eps):
        if e is not None:
            shape = [1] * T.ndim
            shape[k] = T.shape[k]
            d = d + np.asarray(e, dtype=np.float64).reshape(shape)
    q = (R.real / d) + 1j * (R.imag / d)
    return np.asfortranarray(T + alpha * q)


def ccd_energy(B, T):
    """E_corr = 1/4 sum <ij||ab> t_ij^ab"""
    return complex(np.asarray(_o.contract("E()=W(i,j,a,b)*T(a,b,i,j)", np.zeros(()), B["oovv"], T, 0.25,
                                          want_snorm=False)[0]).reshape(-1)[0])


def ccd_jacobi(B, e_occ, e_virt, iterations, T0=None):
    """T <- T + R(T) / (e_i + e_j - e_a - e_b), `iterations` times from T0 (default 0).  R contains the full Fock terms,
    so the fixed point has R = 0 whatever diagonal is used as denominator.  Returns (T, [E_corr after each step])."""
    v, o = B["vvoo"].shape[0], B["vvoo"].shape[2]
    T = np.zeros((v, v, o, o), dtype=np.complex128, order="F") if T0 is None else np.asfortranarray(T0).copy(order="F")
    ev, eo = -np.asarray(e_virt, dtype=np.float64), np.asarray(e_occ, dtype=np.float64)
    energies = []
    for _ in range(iterations):
        R = ccd_residual_program(B, T)
        T = denominator_update(T, R, [ev, ev, eo, eo], 1.0)
        energies.append(ccd_energy(B, T))
    return T, energies


def diis_coefficients(Bm):
    """min |sum_i c_i e_i|^2 subject to sum_i c_i = 1, Bm[i,j] = <e_i|e_j> (Pulay):  [[B, 1], [1^T, 0]] [c; lam] = [0; 1]."""
    m = Bm.shape[0]
    A = np.zeros((m + 1, m + 1), dtype=np.complex128)
    A[:m, :m] = Bm
    A[:m, m] = A[m, :m] = 1.0
    rhs = np.zeros(m + 1, dtype=np.complex128)
    rhs[m] = 1.0
    return np.linalg.solve(A, rhs)[:m]


def ccd_diis(B, e_occ, e_virt, iterations, depth=6):
    """The CCD iteration with DIIS extrapolation: error vector e_k = R(T_k) / D (the Jacobi step), trial vector
    T_k + e_k; the next T is the combination of the last `depth` trial vectors that minimises |sum c_i e_i|.
    Returns (T, [E_corr after each step], [|e_k| of each step])."""
    v, o = B["vvoo"].shape[0], B["vvoo"].shape[2]
    T = np.zeros((v, v, o, o), dtype=np.complex128, order="F")
    ev, eo = -np.asarray(e_virt, dtype=np.float64), np.asarray(e_occ, dtype=np.float64)
    trial, err, energies, norms = [], [], [], []
    for _ in range(iterations):
        R = ccd_residual_program(B, T)
        e = denominator_update(np.zeros_like(T), R, [ev, ev, eo, eo], 1.0)
        trial.append(np.asfortranarray(T + e))
        err.append(e)
        trial, err = trial[-depth:], err[-depth:]
        m = len(err)
        Bm = np.array([[np.vdot(err[i], err[j]) for j in range(m)] for i in range(m)])
        norms.append(float(np.sqrt(abs(Bm[m - 1, m - 1]))))
        c = diis_coefficients(Bm) if m > 1 else np.ones(1)
        T = np.asfortranarray(sum(ci * t for ci, t in zip(c, trial)))
        energies.append(ccd_energy(B, T))
    return T, energies, norms


def ccsd_jacobi(B, e_occ, e_virt, iterations):
    """t1 <- t1 + R1 / (e_i - e_a), t2 <- t2 + R2 / (e_i + e_j - e_a - e_b) from zero amplitudes, both residuals
    evaluated at the same (old) amplitudes.  Returns (T1, T2, [E_corr of the amplitudes after each step])."""
    v, o = B["fvo"].shape
    T1 = np.zeros((v, o), dtype=np.complex128, order="F")
    T2 = np.zeros((v, v, o, o), dtype=np.complex128, order="F")
    ev, eo = -np.asarray(e_virt, dtype=np.float64), np.asarray(e_occ, dtype=np.float64)
    energies = []
    for it in range(iterations + 1):
        E, R1, R2 = ccsd_residual_program(B, T1, T2)
        if it > 0:
            energies.append(E)                  # the energy comes with the residuals of the NEXT evaluation
        if it == iterations:
            break
        T1 = denominator_update(T1, R1, [ev, eo], 1.0)
        T2 = denominator_update(T2, R2, [ev, ev, eo, eo], 1.0)
    return T1, T2, energies


def residual_norm(*residuals):
    """|R| = sqrt(sum over all given residual tensors of <R|R>): the "norm of the residual vector" the paper's tables quote
    per converged calculation."""
    return float(np.sqrt(sum(np.vdot(r, r).real for r in residuals)))


def ccsd_diis(B, e_occ, e_virt, iterations, depth=6):
    """The CCSD iteration with DIIS extrapolation over the combined (t1, t2) vector: error vector e_k = (R1 / D1, R2 / D2)
    at the current amplitudes, trial vector = amplitudes + e_k, next amplitudes = the combination of the last `depth`
    trial vectors minimising |sum c_i e_i| with <e_i|e_j> = <e1_i|e1_j> + <e2_i|e2_j>.
    Returns (T1, T2, [E_corr of the amplitudes each residual evaluation saw], [|R| = residual norm of each evaluation])."""
    v, o = B["fvo"].shape
    T1 = np.zeros((v, o), dtype=np.complex128, order="F")
    T2 = np.zeros((v, v, o, o), dtype=np.complex128, order="F")
    ev, eo = -np.asarray(e_virt, dtype=np.float64), np.asarray(e_occ, dtype=np.float64)
    trial, err, energies, norms = [], [], [], []
    for _ in range(iterations):
        E, R1, R2 = ccsd_residual_program(B, T1, T2)
        energies.append(E)
        norms.append(residual_norm(R1, R2))
        e1 = denominator_update(np.zeros_like(T1), R1, [ev, eo], 1.0)
        e2 = denominator_update(np.zeros_like(T2), R2, [ev, ev, eo, eo], 1.0)
        trial.append((np.asfortranarray(T1 + e1), np.asfortranarray(T2 + e2)))
        err.append((e1, e2))
        trial, err = trial[-depth:], err[-depth:]
        m = len(err)
        Bm = np.array([[np.vdot(err[i][0], err[j][0]) + np.vdot(err[i][1], err[j][1]) for j in range(m)] for i in range(m)])
        c = diis_coefficients(Bm) if m > 1 else np.ones(1)
        T1 = np.asfortranarray(sum(ci * t[0] for ci, t in zip(c, trial)))
        T2 = np.asfortranarray(sum(ci * t[1] for ci, t in zip(c, trial)))
    return T1, T2, energies, norms


# ------------------------------------------------------------------------------------------
# config 4: CCSDT piece
# ------------------------------------------------------------------------------------------
def _swap(X, p, q):
    return np.swapaxes(X, p, q)


def t3_term_unfactorised(W, T2):
    """P(k/ij) P(a/bc) sum_d W(b,c,d,k) T2(a,d,i,j);  P(a/bc)F = F - F(a<->b) - F(a<->c),
    P(k/ij)F = F - F(k<->i) - F(k<->j).   W(b,c,d,k) = <bc||dk>, T2(a,d,i,j) = t_ij^ad."""
    X = np.einsum("bcdk,adij->abcijk", W, T2)
    Y = X - _swap(X, 0, 1) - _swap(X, 0, 2)
    return X, Y - _swap(Y, 5, 3) - _swap(Y, 5, 4)


def p9_terms():
    """The 9 signed index maps of P(k/ij)P(a/bc) in the permsum convention
    (term: X position m is indexed by D's index number s[m])."""
    abc = [((0, 1, 2), 1.0), ((1, 0, 2), -1.0), ((2, 1, 0), -1.0)]
    ijk = [((3, 4, 5), 1.0), ((5, 4, 3), -1.0), ((3, 5, 4), -1.0)]
    perms, coefs = [], []
    for (pa, sa) in abc:
        for (pi, si) in ijk:
            perms.append(list(pa) + list(pi))
            coefs.append(sa * si)
    return perms, coefs


def full_antisymmetriser_terms():
    """All 36 signed (a,b,c) x (i,j,k) permutations."""
    def sign(p):
        s, p = 1, list(p)
        for i in range(len(p)):
            while p[i] != i:
                j = p[i]
                p[i], p[j] = p[j], p[i]
                s = -s
        return s
    perms, coefs = [], []
    for pa in itertools.permutations(range(3)):
        for pi in itertools.permutations(range(3)):
            perms.append(list(pa) + [3 + x for x in pi])
            coefs.append(float(sign(pa) * sign(pi)))
    return perms, coefs


def t3_term_program(W, T2, R3, long_double=True):
    """config 4 as library calls: X = W*T2 (one contraction), R3 += P(k/ij)P(a/bc) X (one permute-sum)."""
    v, o = T2.shape[0], T2.shape[2]
    X0 = np.zeros((v, v, v, o, o, o), dtype=np.complex128, order="F")
    X, _ = _o.contract("X(a,b,c,i,j,k)=W(b,c,d,k)*T(a,d,i,j)", X0, W, T2, 1.0,
                       long_double=long_double, want_snorm=False)
    perms, coefs = p9_terms()
    return X, _o.permsum(R3, X, perms, coefs, 1.0)


# ------------------------------------------------------------------------------------------
# next row 8(f)-3, outlook of the paper (CCSD(T)): the [T] triples correction from doubles.
#   R3(a,b,c,i,j,k) = <Phi_ijk^abc| [H, T2] |Phi0>
#                   = P(k/ij)P(a/bc) sum_d <bc||dk> t_ij^ad - P(i/jk)P(c/ab) sum_l <lc||jk> t_il^ab
#   t3 = R3 / D3,  D3 = e_i + e_j + e_k - e_a - e_b - e_c ;   E[T] = 1/36 sum conj(t3) D3 t3 = 1/36 <t3|R3>
# The connected-triples formula is pinned to the tier-0 triples projection, the 1/36 to a sum over unique triples.
# ------------------------------------------------------------------------------------------
def p9_terms_second():
    """The 9 signed index maps of P(i/jk)P(c/ab) in the permsum convention."""
    abc = [((0, 1, 2), 1.0), ((2, 1, 0), -1.0), ((0, 2, 1), -1.0)]      # 1 - (c<->a) - (c<->b)
    ijk = [((3, 4, 5), 1.0), ((4, 3, 5), -1.0), ((5, 4, 3), -1.0)]      # 1 - (i<->j) - (i<->k)
    perms, coefs = [], []
    for (pa, sa) in abc:
        for (pi, si) in ijk:
            perms.append(list(pa) + list(pi))
            coefs.append(sa * si)
    return perms, coefs


def triples_unfactorised(o, g, t2, e_occ, e_virt):
    """(R3, E[T]) by direct sums."""
    W, U = g[o:, o:, o:, :o], g[:o, o:, :o, :o]                          # <bc||dk>, <lc||jk>
    _, Y = t3_term_unfactorised(W, t2)
    Z = np.einsum("lcjk,abil->abcijk", U, t2)
    Z = Z - _swap(Z, 2, 0) - _swap(Z, 2, 1)
    Z = Z - _swap(Z, 3, 4) - _swap(Z, 3, 5)
    R3 = Y - Z
    eo, ev = np.asarray(e_occ), np.asarray(e_virt)
    D3 = (eo[None, None, None, :, None, None] + eo[None, None, None, None, :, None] + eo[None, None, None, None, None, :]
          - ev[:, None, None, None, None, None] - ev[None, :, None, None, None, None] - ev[None, None, :, None, None, None])
    return R3, np.sum(np.conj(R3) * R3 / D3) / 36.0


def triples_program(W, U, T2, e_occ, e_virt, long_double=True):
    """The same as library calls: two contractions into rank-6 tensors, two 9-term permute-sums, one denominator
    update, one inner product.  W(b,c,d,k) = <bc||dk>, U(l,c,j,k) = <lc||jk>.  Returns (R3, t3, E[T])."""
    v, o = T2.shape[0], T2.shape[2]
    z6 = lambda: np.zeros((v, v, v, o, o, o), dtype=np.complex128, order="F")
    con = lambda e, D, L, R, a=1.0: _o.contract(e, D, L, R, a, long_double=long_double, want_snorm=False)[0]
    X = con("X(a,b,c,i,j,k)=W(b,c,d,k)*T(a,d,i,j)", z6(), W, T2)
    p1, c1 = p9_terms()
    R3 = _o.permsum(z6(), X, p1, c1, 0.0)
    Z = con("Z(a,b,c,i,j,k)=T(a,b,i,l)*U(l,c,j,k)", z6(), T2, U)
    p2, c2 = p9_terms_second()
    R3 = _o.permsum(R3, Z, p2, [-c for c in c2], 1.0)
    ev, eo = -np.asarray(e_virt, dtype=np.float64), np.asarray(e_occ, dtype=np.float64)
    t3 = denominator_update(z6(), R3, [ev, ev, ev, eo, eo, eo], 1.0)
    return R3, t3, np.vdot(t3, R3) / 36.0


def triples_singles_term(t1, oovv, t3, long_double=True):
    """The singles term that turns [T] into (T):  E_ST = <Phi0| T1^+ H T3 |Phi0> = 1/4 sum conj(t_i^a) <jk||bc> t_ijk^abc,
    as library calls: Y(a,i) = t3(a,b,c,i,j,k) * <jk||bc> (a rank-6 tensor contracted down to rank 2), E_ST = 1/4 <t1|Y>.
    Pinned to the Fock-space matrix element in tests/test_oracle_cc.py."""
    v, o = t1.shape
    Y = _o.contract("Y(a,i)=T(a,b,c,i,j,k)*W(j,k,b,c)", np.zeros((v, o), dtype=np.complex128, order="F"), t3, oovv, 1.0,
                    long_double=long_double, want_snorm=False)[0]
    return Y, 0.25 * np.vdot(t1, Y)


# ------------------------------------------------------------------------------------------
# CCSDT (next row 8(f)-3: "CCSDT iterations"; the paper's production target beyond CCSD).
# The paper prints only Eqs. (1)-(4).  The equations below were obtained by enumerating every connected contraction
# topology of H with T2 and T3 and fitting the coefficients to the Fock-space projections of exp(-T) H exp(T) |Phi0>
# (Eq. 3) at o = v = 5 with a NON-Hermitian H (fit residual 4e-15, every coefficient a simple rational); they are PINNED
# to the Fock space in tests/test_oracle_cc.py.  T1 enters through the exact similarity transformation of the integrals
# (`dress_t1`), so the amplitude equations themselves are written for T = T2 + T3 only.
# ------------------------------------------------------------------------------------------
def dress_t1(o, f, g, t1):
    """(f~, g~) with  sum f~ .. + 1/4 sum g~ .. = exp(-T1) H exp(T1):  exp(-T1) a+_p exp(T1) = sum_q a+_q X[q,p],
    exp(-T1) a_q exp(T1) = sum_r Y[q,r] a_r with X = 1 - tau, Y = 1 + tau, tau[a,i] = t_i^a (virtual row, occupied column);
    h~ = X h Y, g~[PQRS] = X[P,p] X[Q,q] g[pqrs] Y[r,R] Y[s,S]; h = f - sum_i <pi||qi> is the bare one-electron part and
    f~ = h~ + sum_i g~[P i Q i] the Fock matrix of the dressed integrals."""
    n = f.shape[0]
    tau = np.zeros((n, n), dtype=np.complex128)
    tau[o:, :o] = t1
    X, Y = np.eye(n) - tau, np.eye(n) + tau
    h = f - np.einsum("piqi->pq", g[:, :o, :, :o])
    ht = X @ h @ Y
    gt = np.einsum("Pp,Qq,pqrs,rR,sS->PQRS", X, X, g, Y, Y)
    ft = ht + np.einsum("piqi->pq", gt[:, :o, :, :o])
    return ft, gt


def _perm_sign(p):
    s, p = 1, list(p)
    for i in range(len(p)):
        while p[i] != i:
            j = p[i]
            p[i], p[j] = p[j], p[i]
            s = -s
    return s


def antisymmetrise_abc_ijk(X):
    """A3 X = sum over the 36 signed permutations of (a,b,c) x (i,j,k)   (X[a,b,c,i,j,k])"""
    out = np.zeros_like(X)
    for pv in itertools.permutations(range(3)):
        for po in itertools.permutations(range(3)):
            out = out + _perm_sign(pv) * _perm_sign(po) * X.transpose(list(pv) + [3 + q for q in po])
    return out


# (coefficient, block types of H, einsum) -- R3 = A3 sum_k c_k X_k, T = T2 + T3 (T1 dressed away)
CCSDT_R3_TERMS = [
    (+1 / 4, "g", "ovoo", "laij,bclk->abcijk", ("t2",)),
    (+1 / 4, "g", "vvov", "abid,dcjk->abcijk", ("t2",)),
    (-1 / 12, "f", "oo", "li,abcljk->abcijk", ("t3",)),
    (+1 / 12, "f", "vv", "ad,dbcijk->abcijk", ("t3",)),
    (+1 / 24, "g", "oooo", "lmij,abclmk->abcijk", ("t3",)),
    (-1 / 4, "g", "ovov", "laid,dbcljk->abcijk", ("t3",)),
    (+1 / 24, "g", "vvvv", "abde,decijk->abcijk", ("t3",)),
    (+1 / 4, "f", "ov", "ld,abli,dcjk->abcijk", ("t2", "t2")),
    (+1 / 8, "g", "ooov", "lmid,ablm,dcjk->abcijk", ("t2", "t2")),
    (-1 / 2, "g", "ooov", "lmid,dalj,bcmk->abcijk", ("t2", "t2")),
    (-1 / 2, "g", "ovvv", "lade,dbli,ecjk->abcijk", ("t2", "t2")),
    (+1 / 8, "g", "ovvv", "lade,bcli,dejk->abcijk", ("t2", "t2")),
    (-1 / 24, "g", "oovv", "lmde,dalm,ebcijk->abcijk", ("t2", "t3")),
    (+1 / 48, "g", "oovv", "lmde,ablm,decijk->abcijk", ("t2", "t3")),
    (-1 / 24, "g", "oovv", "lmde,deli,abcmjk->abcijk", ("t2", "t3")),
    (+1 / 4, "g", "oovv", "lmde,dali,ebcmjk->abcijk", ("t2", "t3")),
    (-1 / 8, "g", "oovv", "lmde,abli,decmjk->abcijk", ("t2", "t3")),
    (+1 / 48, "g", "oovv", "lmde,deij,abclmk->abcijk", ("t2", "t3")),
    (-1 / 8, "g", "oovv", "lmde,daij,ebclmk->abcijk", ("t2", "t3")),
]


def _blk(o, H, types):
    return H[tuple(slice(0, o) if t == "o" else slice(o, None) for t in types)]


def ccsdt_residual_unfactorised(o, f, g, t1, t2, t3):
    """(E_corr, R1, R2, R3) of CCSDT: the projections of exp(-T) H exp(T) |Phi0>, T = T1 + T2 + T3 (PAPER Eqs. 2-3), as
    explicit sums.  With (f~, g~) = dress_t1:
      R1[a,i]  = f~[a,i] + f~[l,d] t2[d,a,l,i] + 1/2 g~[l,m,i,d] t2[d,a,l,m] + 1/2 g~[l,a,d,e] t2[d,e,l,i]
                 + 1/4 g~[l,m,d,e] t3[d,e,a,l,m,i]
      R2       = (the 10-term CCD residual of f~, g~, t2) + f~[l,d] t3[d,a,b,l,i,j]
                 + 1/2 P(ij) g~[l,m,i,d] t3[d,a,b,l,m,j] + 1/2 P(ab) g~[l,a,d,e] t3[d,e,b,l,i,j]
      R3       = A3 sum of CCSDT_R3_TERMS (19 terms)
      E_corr   = f[i,a] t1[a,i] + 1/4 <ij||ab> t2 + 1/2 <ij||ab> t1 t1   (bare integrals; T3 does not enter)"""
    es = np.einsum
    ft, gt = dress_t1(o, f, g, t1)
    B = lambda H, ty: _blk(o, H, ty)
    r1 = (B(ft, "vo") + es("ld,dali->ai", B(ft, "ov"), t2) + 0.5 * es("lmid,dalm->ai", B(gt, "ooov"), t2)
          + 0.5 * es("lade,deli->ai", B(gt, "ovvv"), t2) + 0.25 * es("lmde,dealmi->ai", B(gt, "oovv"), t3))
    r2 = ccd_residual_unfactorised(o, ft, gt, t2)[0]
    r2 = r2 + es("ld,dablij->abij", B(ft, "ov"), t3)
    r2 = r2 + 0.5 * _P(es("lmid,dablmj->abij", B(gt, "ooov"), t3), 2, 3)
    r2 = r2 + 0.5 * _P(es("lade,deblij->abij", B(gt, "ovvv"), t3), 0, 1)
    amps = {"t2": t2, "t3": t3}
    x = np.zeros_like(t3)
    for c, which, types, spec, ts in CCSDT_R3_TERMS:
        x = x + c * es(spec, B(ft if which == "f" else gt, types), *[amps[t] for t in ts])
    r3 = antisymmetrise_abc_ijk(x)
    oovv = B(g, "oovv")
    e = (es("ia,ai->", B(f, "ov"), t1) + 0.25 * es("ijab,abij->", oovv, t2) + 0.5 * es("ijab,ai,bj->", oovv, t1, t1))
    return complex(e), r1, r2, r3


def ccsdt_jacobi(o, f, g, iterations):
    """t1 += R1 / (e_i - e_a), t2 += R2 / (e_i + e_j - e_a - e_b), t3 += R3 / (e_i + e_j + e_k - e_a - e_b - e_c) from zero
    amplitudes, e = diag f, all three residuals evaluated at the old amplitudes (`ccsdt_residual_unfactorised`).
    Returns (T1, T2, T3, [E_corr of the amplitudes each evaluation saw], [residual norm of each evaluation])."""
    v = f.shape[0] - o
    e = np.real(np.diag(f))
    eo, ev = e[:o], -e[o:]
    T1 = np.zeros((v, o), dtype=np.complex128, order="F")
    T2 = np.zeros((v, v, o, o), dtype=np.complex128, order="F")
    T3 = np.zeros((v, v, v, o, o, o), dtype=np.complex128, order="F")
    energies, norms = [], []
    for _ in range(iterations):
        E, R1, R2, R3 = ccsdt_residual_unfactorised(o, f, g, T1, T2, T3)
        energies.append(E)
        norms.append(residual_norm(R1, R2, R3))
        T1 = denominator_update(T1, R1, [ev, eo], 1.0)
        T2 = denominator_update(T2, R2, [ev, ev, eo, eo], 1.0)
        T3 = denominator_update(T3, R3, [ev, ev, ev, eo, eo, eo], 1.0)
    return T1, T2, T3, energies, norms


def ccsdt_diis(o, f, g, iterations, depth=6):
    """The CCSDT iteration with DIIS over the combined (t1, t2, t3) vector (as `ccsd_diis`, one more component): error
    vector e_k = (R1 / D1, R2 / D2, R3 / D3) at the current amplitudes, trial vector = amplitudes + e_k, next amplitudes =
    the combination of the last `depth` trial vectors minimising |sum c_i e_i|, <e_i|e_j> summed over the three components
    (every element of the full antisymmetric tensors counted).
    Returns (T1, T2, T3, [E_corr of the amplitudes each evaluation saw], [residual norm of each evaluation])."""
    v = f.shape[0] - o
    e = np.real(np.diag(f))
    eo, ev = e[:o], -e[o:]
    T = [np.zeros((v, o), dtype=np.complex128, order="F"), np.zeros((v, v, o, o), dtype=np.complex128, order="F"),
         np.zeros((v, v, v, o, o, o), dtype=np.complex128, order="F")]
    eps = [[ev, eo], [ev, ev, eo, eo], [ev, ev, ev, eo, eo, eo]]
    trial, err, energies, norms = [], [], [], []
    for _ in range(iterations):
        E, R1, R2, R3 = ccsdt_residual_unfactorised(o, f, g, *T)
        energies.append(E)
        norms.append(residual_norm(R1, R2, R3))
        ek = [denominator_update(np.zeros_like(t), r, d, 1.0) for t, r, d in zip(T, (R1, R2, R3), eps)]
        trial.append([np.asfortranarray(t + x) for t, x in zip(T, ek)])
        err.append(ek)
        trial, err = trial[-depth:], err[-depth:]
        m = len(err)
        Bm = np.array([[sum(np.vdot(err[i][q], err[j][q]) for q in range(3)) for j in range(m)] for i in range(m)])
        c = diis_coefficients(Bm) if m > 1 else np.ones(1)
        T = [np.asfortranarray(sum(ci * t[q] for ci, t in zip(c, trial))) for q in range(3)]
    return T[0], T[1], T[2], energies, norms
