"""The 'generated driver' stand-in: a spin-orbital CCD doubles residual as the list of binary tensor operations a
tenpi-generated program would issue to its tensor library, each line one C-ABI call.
Everything is computed by libtcb200.so; this file only sequences calls and owns the intermediates' lifetimes
(tenpi emits create/destroy around every intermediate).

Equations (config 2): t_ij^ab stored T(a,b,i,j); integral blocks in bra-ket order.
"""

PROGRAM_DOC = """
R(a,b,i,j)  = vvoo(a,b,i,j)
X(a,b,i,j)  = T(a,c,i,j)*fvv(b,c)              ; R += P(ab) X
X(a,b,i,j)  = T(a,b,i,k)*foo(k,j)              ; R -= P(ij) X
I1(k,l,i,j) = oooo(k,l,i,j) + 1/2 oovv(k,l,c,d)*T(c,d,i,j)
R(a,b,i,j) += 1/2 T(a,b,k,l)*I1(k,l,i,j)
R(a,b,i,j) += 1/2 vvvv(a,b,c,d)*T(c,d,i,j)
I2(k,b,c,j) = ovvo(k,b,c,j) + 1/2 oovv(k,l,c,d)*T(b,d,j,l)
X(a,b,i,j)  = T(a,c,i,k)*I2(k,b,c,j)           ; R += P(ij)P(ab) X
I3(l,i)     = oovv(k,l,c,d)*T(d,c,i,k) ; X(a,b,i,j) = T(a,b,l,j)*I3(l,i) ; R -= 1/2 P(ij) X
I4(a,d)     = oovv(k,l,c,d)*T(a,c,l,k) ; X(a,b,i,j) = I4(a,d)*T(d,b,i,j) ; R -= 1/2 P(ab) X
"""


def ccd_residual(ctx, B, T, R=None, lanes=True, packed=None):
    """B: dict name -> Tensor for foo, fvv, vvoo, oovv, oooo, vvvv, ovvo;  T: Tensor (v,v,o,o).
    Returns the residual tensor R (v,v,o,o); all work is enqueued on the context (lane 0 holds the result).

    lanes: the intermediates that do not depend on one another are built side by side (DLTC layers,
    PAPER.md:79, instead of the barrier after every operation of PAPER.md:400): lane 1 builds I3, I4 and their X tensors
    (skinny, long-K contractions that leave most of the tensor pipe idle), lane 2 builds I2 and the ring term's X, lane 0
    does the Fock terms, the two ladders, and every update of R (updates of one tensor stay on one lane, in order).
    packed: a dict (start with {}) runs the particle-particle ladder on packed storage (`pp_ladder_packed`: 1/8 of the flops)
    and keeps the packed <ab||cd> under "vvvv" between calls; destroy its values when done."""
    v, _, o, _ = T.extents
    use_lanes = lanes and hasattr(ctx, "lane_set")
    lane = ctx.lane_set if use_lanes else (lambda l: None)
    wait = ctx.lane_wait if use_lanes else (lambda l, m: None)
    new = lambda shape: ctx.tensor_create(shape, zero=False)   # every intermediate below is first written by an '=' call
    if R is None:
        R = new((v, v, o, o))
    wait(1, 0)
    wait(2, 0)
    # ---- lane 2: I2 and the ring term ------------------------------------------------------------------------------------
    lane(2)
    I2 = new((o, v, v, o))
    ctx.add("I2(k,b,c,j)=W(k,b,c,j)", I2, B["ovvo"], 1.0)
    ctx.contract("I2(k,b,c,j)+=W(k,l,c,d)*T(b,d,j,l)", I2, B["oovv"], T, 0.5)
    X2 = new((v, v, o, o))
    ctx.contract("X(a,b,i,j)=T(a,c,i,k)*I2(k,b,c,j)", X2, T, I2, 1.0)
    I2.destroy()
    # ---- lane 1: the two skinny intermediates and their terms ------------------------------------------------------------
    lane(1)
    I3 = new((o, o))
    ctx.contract("I3(l,i)=W(k,l,c,d)*T(d,c,i,k)", I3, B["oovv"], T, 1.0)
    X3 = new((v, v, o, o))
    ctx.contract("X(a,b,i,j)=T(a,b,l,j)*I3(l,i)", X3, T, I3, 1.0)
    I3.destroy()
    I4 = new((v, v))
    ctx.contract("I4(a,d)=W(k,l,c,d)*T(a,c,l,k)", I4, B["oovv"], T, 1.0)
    X4 = new((v, v, o, o))
    ctx.contract("X(a,b,i,j)=I4(a,d)*T(d,b,i,j)", X4, I4, T, 1.0)
    I4.destroy()
    # ---- lane 0: driver, Fock terms, ladders, and every update of R ------------------------------------------------------
    lane(0)
    X = new((v, v, o, o))
    ctx.add("R(a,b,i,j)=W(a,b,i,j)", R, B["vvoo"], 1.0)
    ctx.contract("X(a,b,i,j)=T(a,c,i,j)*f(b,c)", X, T, B["fvv"], 1.0)
    ctx.antisymmetrize("P(ab):R(a,b,i,j)+=X(a,b,i,j)", R, X, 1.0)
    ctx.contract("X(a,b,i,j)=T(a,b,i,k)*f(k,j)", X, T, B["foo"], 1.0)
    ctx.antisymmetrize("P(ij):R(a,b,i,j)+=X(a,b,i,j)", R, X, -1.0)
    X.destroy()
    I1 = new((o, o, o, o))
    ctx.add("I1(k,l,i,j)=W(k,l,i,j)", I1, B["oooo"], 1.0)
    ctx.contract("I1(k,l,i,j)+=W(k,l,c,d)*T(c,d,i,j)", I1, B["oovv"], T, 0.5)
    ctx.contract("R(a,b,i,j)+=T(a,b,k,l)*I1(k,l,i,j)", R, T, I1, 0.5)
    I1.destroy()
    if packed is None:
        ctx.contract("R(a,b,i,j)+=V(a,b,c,d)*T(c,d,i,j)", R, B["vvvv"], T, 0.5)
    else:
        packed["vvvv"] = pp_ladder_packed(ctx, R, B["vvvv"], T, Vp=packed.get("vvvv"), alpha=0.5)
    wait(0, 2)
    ctx.antisymmetrize("P(ij)P(ab):R(a,b,i,j)+=X(a,b,i,j)", R, X2, 1.0)
    X2.destroy()
    wait(0, 1)
    ctx.antisymmetrize("P(ij):R(a,b,i,j)+=X(a,b,i,j)", R, X3, -0.5)
    ctx.antisymmetrize("P(ab):R(a,b,i,j)+=X(a,b,i,j)", R, X4, -0.5)
    X3.destroy()
    X4.destroy()
    return R


def pp_ladder_packed(ctx, R, V, T, Vp=None, alpha=0.5):
    """R(a,b,i,j) += alpha sum_cd V(a,b,c,d) T(c,d,i,j) for V antisymmetric in (a,b) and (c,d) and T in (c,d) and (i,j), on
    index-permutation-symmetric packed storage: with c<d, a<b, i<j the contraction
    is a plain GEMM at 1/2 of M, of N and of K -- 1/8 of the flops -- and the sum over c<d visits every unordered pair once,
    so alpha doubles.  Vp: V already packed (v(v-1)/2 squared: 6.3 GB instead of 25.6 GB at v = 200), reusable across
    iterations; built from V when None.  Returns Vp."""
    v, _, o, _ = T.extents
    nv, no = ctx.packed_extent(v, 2), ctx.packed_extent(o, 2)
    if Vp is None:
        Vp = ctx.tensor_create((nv, nv), zero=False)
        ctx.pack("Vp(a<b,c<d)=V(a,b,c,d)", Vp, V)
    Tp = ctx.tensor_create((nv, no), zero=False)
    ctx.pack("Tp(c<d,i<j)=T(c,d,i,j)", Tp, T)
    Rp = ctx.tensor_create((nv, no), zero=False)
    ctx.contract("Rp(x,y)=Vp(x,z)*Tp(z,y)", Rp, Vp, Tp, 2.0 * alpha)
    ctx.unpack("R(a,b,i,j)+=Rp(a<b,i<j)", R, Rp, 1.0)
    Tp.destroy()
    Rp.destroy()
    return Vp


def ccd_energy(ctx, B, T):
    """E_corr = 1/4 sum_ijab <ij||ab> t_ij^ab -- the energy diagram (the 11th of the paper's 11 CCD diagrams,
    PAPER.md:276), a contraction into a rank-0 tensor.  Returns the rank-0 device tensor E (download it to read it)."""
    E = ctx.tensor_create(())
    ctx.contract("E()=W(i,j,a,b)*T(a,b,i,j)", E, B["oovv"], T, 0.25)
    return E


CCSD_BLOCKS = ("vvoo", "oovv", "oooo", "vvvv", "ovvo", "ooov", "ovvv", "vovv", "oovo", "ovov", "vvvo", "ovoo",
               "foo", "fvv", "fov", "fvo")


def ccsd_residual(ctx, B, T1, T2, R1=None, R2=None, packed=None):
    """Spin-orbital CCSD residuals (the paper's benchmark iteration) as the binary tensor operations a
    generated driver issues: 34 contractions, 9 permute-sums, 12 adds; intermediates are created and destroyed around
    their use.  B: dict of device tensors `CCSD_BLOCKS` (<pq||rs> blocks in bra-ket order, f blocks);
    T1 (v,o) = t_i^a, T2 (v,v,o,o) = t_ij^ab.  Returns (E rank-0 tensor, R1, R2).  Equations: DESIGN.md / oracle/cc.py
    `ccsd_residual_unfactorised` (pinned to PAPER Eq. (3) on the Fock space).
    packed: a dict (start with {}) switches the particle-particle ladder to index-permutation-symmetric packed storage
    (SURVEY 8(f)-2): W_abef is built and used only as Wp(a<b, e<f) -- the v^4 o^2 ladder at 1/8 of the flops, its T1 term at
    1/2, P(ab) as a `tcb_antisym_pack`.  The dict keeps the packed integral blocks (<ab||ef>, <am||ef>) between
    calls; destroy its values when done."""
    v, o = T1.extents
    new = lambda shape: ctx.tensor_create(shape, zero=False)      # every tensor below is first written by an '=' call
    con, add, asym = ctx.contract, ctx.add, ctx.antisymmetrize

    def copy(src, shape, label):
        D = new(shape)
        add(f"D({label})=S({label})", D, src, 1.0)
        return D

    tt = new((v, v, o, o))
    con("tt(a,b,i,j)=T1(a,i)*T1(b,j)", tt, T1, T1, 1.0)
    taut = copy(T2, (v, v, o, o), "a,b,i,j")
    asym("P(ab):t(a,b,i,j)+=tt(a,b,i,j)", taut, tt, 0.5)
    tau = copy(T2, (v, v, o, o), "a,b,i,j")
    asym("P(ab):t(a,b,i,j)+=tt(a,b,i,j)", tau, tt, 1.0)
    Fae = copy(B["fvv"], (v, v), "a,e")
    con("F(a,e)+=T1(a,m)*f(m,e)", Fae, T1, B["fov"], -0.5)
    con("F(a,e)+=W(m,a,f,e)*T1(f,m)", Fae, B["ovvv"], T1, 1.0)
    con("F(a,e)+=t(a,f,m,n)*W(m,n,e,f)", Fae, taut, B["oovv"], -0.5)
    Fmi = copy(B["foo"], (o, o), "m,i")
    con("F(m,i)+=f(m,e)*T1(e,i)", Fmi, B["fov"], T1, 0.5)
    con("F(m,i)+=W(m,n,i,e)*T1(e,n)", Fmi, B["ooov"], T1, 1.0)
    con("F(m,i)+=W(m,n,e,f)*t(e,f,i,n)", Fmi, B["oovv"], taut, 0.5)
    taut.destroy()
    Fme = copy(B["fov"], (o, v), "m,e")
    con("F(m,e)+=W(m,n,e,f)*T1(f,n)", Fme, B["oovv"], T1, 1.0)
    X = new((o, o, o, o))
    con("X(m,n,i,j)=W(m,n,i,e)*T1(e,j)", X, B["ooov"], T1, 1.0)
    Wmnij = copy(B["oooo"], (o, o, o, o), "m,n,i,j")
    asym("P(ij):W(m,n,i,j)+=X(m,n,i,j)", Wmnij, X, 1.0)
    X.destroy()
    # The quadratic term 1/4 tau V tau of R2 enters through W_mnij alone (coefficient 1/2 here instead of 1/4 here and 1/4
    # in W_abef): o^4 v^2 work instead of v^4 o^2 -- the same residual; neither intermediate is used anywhere else.
    con("W(m,n,i,j)+=V(m,n,e,f)*t(e,f,i,j)", Wmnij, B["oovv"], tau, 0.5)
    if packed is None:
        X = new((v, v, v, v))
        con("X(a,b,e,f)=V(a,m,e,f)*T1(b,m)", X, B["vovv"], T1, 1.0)
        Wabef = copy(B["vvvv"], (v, v, v, v), "a,b,e,f")
        asym("P(ab):W(a,b,e,f)+=X(a,b,e,f)", Wabef, X, -1.0)
        X.destroy()
    else:
        nv2, no2 = ctx.packed_extent(v, 2), ctx.packed_extent(o, 2)
        for name, shape, spec in (("vvvv", (nv2, nv2), "P(a<b,e<f)=V(a,b,e,f)"), ("vovv", (v, o, nv2), "P(a,m,e<f)=V(a,m,e,f)")):
            if name not in packed:
                packed[name] = new(shape)
                ctx.pack(spec, packed[name], B[name])
        X = new((v, v, nv2))
        con("X(a,b,z)=V(a,m,z)*T1(b,m)", X, packed["vovv"], T1, 1.0)
        Wabef = copy(packed["vvvv"], (nv2, nv2), "x,z")
        ctx.antisym_pack("W(a<b,z)+=X(a,b,z)", Wabef, X, -1.0)                 # P(ab) on packed storage
        X.destroy()
        taup = new((nv2, no2))
        ctx.pack("P(e<f,i<j)=t(e,f,i,j)", taup, tau)
    Q = new((v, v, o, o))
    add("Q(f,b,j,n)=T2(f,b,j,n)", Q, T2, 0.5)
    add("Q(f,b,j,n)+=t(f,b,j,n)", Q, tt, 1.0)
    Wmbej = copy(B["ovvo"], (o, v, v, o), "m,b,e,j")
    con("W(m,b,e,j)+=V(m,b,e,f)*T1(f,j)", Wmbej, B["ovvv"], T1, 1.0)
    con("W(m,b,e,j)+=V(m,n,e,j)*T1(b,n)", Wmbej, B["oovo"], T1, -1.0)
    con("W(m,b,e,j)+=V(m,n,e,f)*Q(f,b,j,n)", Wmbej, B["oovv"], Q, -1.0)
    Q.destroy()
    if R1 is None:
        R1 = new((v, o))
    add("R(a,i)=f(a,i)", R1, B["fvo"], 1.0)
    con("R(a,i)+=F(a,e)*T1(e,i)", R1, Fae, T1, 1.0)
    con("R(a,i)+=T1(a,m)*F(m,i)", R1, T1, Fmi, -1.0)
    con("R(a,i)+=T2(a,e,i,m)*F(m,e)", R1, T2, Fme, 1.0)
    con("R(a,i)+=V(n,a,i,f)*T1(f,n)", R1, B["ovov"], T1, -1.0)
    con("R(a,i)+=V(m,a,e,f)*T2(e,f,i,m)", R1, B["ovvv"], T2, -0.5)
    con("R(a,i)+=T2(a,e,m,n)*V(n,m,e,i)", R1, T2, B["oovo"], -0.5)
    if R2 is None:
        R2 = new((v, v, o, o))
    add("R(a,b,i,j)=W(a,b,i,j)", R2, B["vvoo"], 1.0)
    X = new((v, v, o, o))
    con("G(b,e)+=T1(b,m)*F(m,e)", Fae, T1, Fme, -0.5)                 # Fae is not needed any more: it becomes G
    con("X(a,b,i,j)=T2(a,e,i,j)*G(b,e)", X, T2, Fae, 1.0)
    asym("P(ab):R(a,b,i,j)+=X(a,b,i,j)", R2, X, 1.0)
    Fae.destroy()
    con("G(m,j)+=F(m,e)*T1(e,j)", Fmi, Fme, T1, 0.5)                   # likewise Fmi becomes Gm
    con("X(a,b,i,j)=T2(a,b,i,m)*G(m,j)", X, T2, Fmi, 1.0)
    asym("P(ij):R(a,b,i,j)+=X(a,b,i,j)", R2, X, -1.0)
    Fmi.destroy()
    Fme.destroy()
    con("R(a,b,i,j)+=t(a,b,m,n)*W(m,n,i,j)", R2, tau, Wmnij, 0.5)
    Wmnij.destroy()
    if packed is None:
        con("R(a,b,i,j)+=W(a,b,e,f)*t(e,f,i,j)", R2, Wabef, tau, 0.5)
    else:
        Rp = new((nv2, no2))
        con("R(x,y)=W(x,z)*t(z,y)", Rp, Wabef, taup, 1.0)                      # 1/2 sum_ef = sum_{e<f}
        ctx.unpack("R(a,b,i,j)+=P(a<b,i<j)", R2, Rp, 1.0)
        Rp.destroy()
        taup.destroy()
    Wabef.destroy()
    tau.destroy()
    con("X(a,b,i,j)=T2(a,e,i,m)*W(m,b,e,j)", X, T2, Wmbej, 1.0)
    Wmbej.destroy()
    Z = new((o, v, o, o))
    con("Z(m,b,i,j)=V(m,b,e,j)*T1(e,i)", Z, B["ovvo"], T1, 1.0)
    con("X(a,b,i,j)+=T1(a,m)*Z(m,b,i,j)", X, T1, Z, -1.0)
    Z.destroy()
    asym("P(ij)P(ab):R(a,b,i,j)+=X(a,b,i,j)", R2, X, 1.0)
    con("X(a,b,i,j)=V(a,b,e,j)*T1(e,i)", X, B["vvvo"], T1, 1.0)
    asym("P(ij):R(a,b,i,j)+=X(a,b,i,j)", R2, X, 1.0)
    con("X(a,b,i,j)=T1(a,m)*V(m,b,i,j)", X, T1, B["ovoo"], 1.0)
    asym("P(ab):R(a,b,i,j)+=X(a,b,i,j)", R2, X, -1.0)
    X.destroy()
    E = new(())
    con("E()=f(i,a)*T1(a,i)", E, B["fov"], T1, 1.0)
    con("E()+=V(i,j,a,b)*T2(a,b,i,j)", E, B["oovv"], T2, 0.25)
    con("E()+=V(i,j,a,b)*t(a,b,i,j)", E, B["oovv"], tt, 0.5)
    tt.destroy()
    return E, R1, R2


def ccd_solve(ctx, B, e_occ, e_virt, iterations, T=None, norms=None, packed=False):
    """Jacobi iterations of the CCD amplitude equations (PAPER.md:212 energy denominators, 406-410 "CC
    iteration"):  T <- T + R(T) / (e_i + e_j - e_a - e_b), from T (default: a zero tensor, whose first step is the MP2
    guess).  Every step is `ccd_residual` + one `tcb_denominator_update` + the rank-0 energy contraction; only the
    16-byte energy comes back to the host per iteration.  norms: a list that receives the residual norm |R(T)| each
    iteration started from (one `tcb_dot`).  packed=True: the pp ladder on packed storage, <ab||cd>
    packed once for all iterations.  Returns (T, [E_corr after each step])."""
    import numpy as np
    v, _, o, _ = B["vvoo"].extents
    if T is None:
        T = ctx.tensor_create((v, v, o, o))
    ev, eo = -np.asarray(e_virt, dtype=np.float64), np.asarray(e_occ, dtype=np.float64)
    R = ctx.tensor_create((v, v, o, o))
    energies = []
    cache = {} if packed else None
    for _ in range(iterations):
        ccd_residual(ctx, B, T, R, packed=cache)
        if norms is not None:
            norms.append(residual_norm(ctx, R))     # |R(T)| of the amplitudes this iteration started from
        ctx.denominator_update(T, R, [ev, ev, eo, eo], 1.0)
        E = ccd_energy(ctx, B, T)
        energies.append(complex(ctx.tensor_download(E)))
        E.destroy()
    for t in [R] + list((cache or {}).values()):
        t.destroy()
    return T, energies


def triples_correction(ctx, W, U, T2, e_occ, e_virt, keep=False, T1=None, oovv=None):
    """The [T] triples correction from doubles (the paper's outlook, CCSD(T): PAPER.md:386, 452), all rank-6 work on the
    device:  R3 = P(k/ij)P(a/bc) sum_d <bc||dk> t_ij^ad - P(i/jk)P(c/ab) sum_l <lc||jk> t_il^ab   (two contractions into
    6 GB-class tensors, two 9-term antisymmetrisers),  t3 = R3 / (e_i + e_j + e_k - e_a - e_b - e_c)
    (`tcb_denominator_divide`),  E[T] = 1/36 <t3|R3> (`tcb_dot`).  W (v,v,v,o) = <bc||dk>, U (o,v,o,o) = <lc||jk>.
    With T1 (v,o) and oovv given, also the singles term of (T):  Y(a,i) = t3(a,b,c,i,j,k) <jk||bc> (the rank-6 tensor
    read once, in place), E_ST = 1/4 <t1|Y>.
    Returns the rank-0 tensor E[T]; with T1, (E[T], E_ST); with keep=True, additionally R3 and t3."""
    import numpy as np
    v, _, o, _ = T2.extents
    shape = (v, v, v, o, o, o)
    X, R3 = ctx.tensor_create(shape, zero=False), ctx.tensor_create(shape, zero=False)    # both first written by '='
    ctx.contract("X(a,b,c,i,j,k)=W(b,c,d,k)*T(a,d,i,j)", X, W, T2, 1.0)
    ctx.antisymmetrize("P(a/bc)P(k/ij):R(a,b,c,i,j,k)=X(a,b,c,i,j,k)", R3, X, 1.0)
    ctx.contract("X(a,b,c,i,j,k)=T(a,b,i,l)*U(l,c,j,k)", X, T2, U, 1.0)
    ctx.antisymmetrize("P(c/ab)P(i/jk):R(a,b,c,i,j,k)+=X(a,b,c,i,j,k)", R3, X, -1.0)
    ev, eo = -np.asarray(e_virt, dtype=np.float64), np.asarray(e_occ, dtype=np.float64)
    ctx.denominator_divide(X, R3, [ev, ev, ev, eo, eo, eo], 1.0)       # X becomes t3
    E = ctx.tensor_create(())
    ctx.dot(E, X, R3, True, 1.0 / 36.0)
    out = [E]
    if T1 is not None:
        Y, Est = ctx.tensor_create((v, o)), ctx.tensor_create(())
        ctx.contract("Y(a,i)=T(a,b,c,i,j,k)*W(j,k,b,c)", Y, X, oovv, 1.0)
        ctx.dot(Est, T1, Y, True, 0.25)
        Y.destroy()
        out.append(Est)
    if keep:
        return tuple(out) + (R3, X)
    X.destroy()
    R3.destroy()
    return out[0] if T1 is None else tuple(out)


def triples_correction_packed(ctx, W, U, T2, e_occ, e_virt, keep=False, T1=None, oovv=None):
    """`triples_correction` on index-permutation-symmetric packed storage: R3 and t3
    exist only on a<b<c, i<j<k.  W(b,c,d,k) is antisymmetric in (b,c), U(l,c,j,k) in (j,k), T2 in (a,b) and (i,j), so
        X1(a, i<j, b<c, k) = sum_d T2(a,d,i<j) W(b<c,d,k)        X2(a<b, i, c, j<k) = sum_l T2(a<b,i,l) U(l,c,j<k)
    are 1/4 of the dense contractions, and the two 9-term operators P(a/bc)P(k/ij), P(c/ab)P(i/jk) are `tcb_antisym_pack`
    calls straight into R3p(a<b<c, i<j<k):  E[T] = <t3p|R3p> (each unordered triple pair once: the factor 1/36 is gone).
    Singles term: Y(a,i) = 4 sum_{b<c, j<k} t3(b<c, a | j<k, i) <j<k||b<c> on a packed view of t3p, E_ST = 1/4 <t1|Y>.
    Returns as `triples_correction`; with keep=True R3p and t3p (packed).  Needs o >= 3 and v >= 3."""
    import numpy as np
    v, _, o, _ = T2.extents
    if o < 3 or v < 3:
        raise ValueError("triples_correction_packed needs o >= 3 and v >= 3 (a<b<c groups)")
    nv2, nv3, no2, no3 = (ctx.packed_extent(v, 2), ctx.packed_extent(v, 3), ctx.packed_extent(o, 2), ctx.packed_extent(o, 3))
    new = lambda shape: ctx.tensor_create(shape, zero=False)
    T2y, Wp, T2z, Up = new((v, v, no2)), new((nv2, v, o)), new((nv2, o, o)), new((o, v, no2))
    ctx.pack("P(a,d,i<j)=T(a,d,i,j)", T2y, T2)
    ctx.pack("P(b<c,d,k)=W(b,c,d,k)", Wp, W)
    ctx.pack("P(a<b,i,l)=T(a,b,i,l)", T2z, T2)
    ctx.pack("P(l,c,j<k)=U(l,c,j,k)", Up, U)
    X1, X2 = new((v, no2, nv2, o)), new((nv2, o, v, no2))
    ctx.contract("X(a,y,x,k)=T(a,d,y)*W(x,d,k)", X1, T2y, Wp, 1.0)
    ctx.contract("X(x,i,c,y)=T(x,i,l)*U(l,c,y)", X2, T2z, Up, 1.0)
    R3p = new((nv3, no3))
    ctx.antisym_pack("R(a<b<c,i<j<k)=X(a,i<j,b<c,k)", R3p, X1, 1.0)
    ctx.antisym_pack("R(a<b<c,i<j<k)+=X(a<b,i,c,j<k)", R3p, X2, -1.0)
    for t in (T2y, Wp, T2z, Up, X1, X2):
        t.destroy()
    ev, eo = -np.asarray(e_virt, dtype=np.float64), np.asarray(e_occ, dtype=np.float64)
    t3p = new((nv3, no3))
    ctx.denominator_divide(t3p, R3p, [np.asarray(_tuple_sums(ev, 3)), np.asarray(_tuple_sums(eo, 3))], 1.0)
    E = ctx.tensor_create(())
    ctx.dot(E, t3p, R3p, True, 1.0)
    out = [E]
    if T1 is not None:
        V, gp = new((nv2, no2, v, o)), new((no2, nv2))
        ctx.unpack("V(b<c,j<k,a,i)=T(b<c<a,j<k<i)", V, t3p, 1.0)
        ctx.pack("P(j<k,b<c)=g(j,k,b,c)", gp, oovv)
        Y, Est = ctx.tensor_create((v, o)), ctx.tensor_create(())
        ctx.contract("Y(a,i)=T(x,y,a,i)*W(y,x)", Y, V, gp, 4.0)
        ctx.dot(Est, T1, Y, True, 0.25)
        for t in (V, gp, Y):
            t.destroy()
        out.append(Est)
    if keep:
        return tuple(out) + (R3p, t3p)
    R3p.destroy()
    t3p.destroy()
    return out[0] if T1 is None else tuple(out)


def ccd_solve_diis(ctx, B, e_occ, e_virt, iterations, depth=6):
    """The CCD iteration with DIIS extrapolation (Pulay): error vector e_k = R(T_k) / D, trial vector T_k + e_k, next T =
    the combination of the last `depth` trial vectors minimising |sum c_i e_i|.  Tensors, inner products (`tcb_dot`,
    one new row of <e_i|e_j> per iteration) and linear combinations (`tcb_add`) live on the device; only the
    depth x depth system is solved on the host.  Returns (T, [E_corr after each step], [|e_k| of each step])."""
    import numpy as np
    v, _, o, _ = B["vvoo"].extents
    shape = (v, v, o, o)
    T, R = ctx.tensor_create(shape), ctx.tensor_create(shape)
    ev, eo = -np.asarray(e_virt, dtype=np.float64), np.asarray(e_occ, dtype=np.float64)
    trial, err, energies, norms = [], [], [], []
    Bm = np.zeros((0, 0), dtype=np.complex128)
    s = ctx.tensor_create(())
    for _ in range(iterations):
        ccd_residual(ctx, B, T, R)
        if len(err) == depth:                      # the oldest pair leaves; its tensors are reused
            e, t = err.pop(0), trial.pop(0)
            Bm = Bm[1:, 1:]
        else:
            e, t = ctx.tensor_create(shape), ctx.tensor_create(shape)
        ctx.denominator_divide(e, R, [ev, ev, eo, eo], 1.0)
        ctx.add("t(a,b,i,j)=T(a,b,i,j)", t, T, 1.0)
        ctx.add("t(a,b,i,j)+=e(a,b,i,j)", t, e, 1.0)
        err.append(e)
        trial.append(t)
        m = len(err)
        row = np.zeros(m, dtype=np.complex128)
        for i in range(m):                         # <e_i|e_new>; the matrix is Hermitian
            ctx.dot(s, err[i], e, True, 1.0)
            row[i] = complex(ctx.tensor_download(s))
        Bn = np.zeros((m, m), dtype=np.complex128)
        Bn[:m - 1, :m - 1] = Bm
        Bn[:, m - 1] = row
        Bn[m - 1, :] = row.conj()
        Bn[m - 1, m - 1] = row[m - 1]
        Bm = Bn
        norms.append(float(np.sqrt(abs(Bm[m - 1, m - 1]))))
        if m > 1:
            A = np.zeros((m + 1, m + 1), dtype=np.complex128)
            A[:m, :m] = Bm
            A[:m, m] = A[m, :m] = 1.0
            rhs = np.zeros(m + 1, dtype=np.complex128)
            rhs[m] = 1.0
            c = np.linalg.solve(A, rhs)[:m]
        else:
            c = np.ones(1, dtype=np.complex128)
        ctx.add("T(a,b,i,j)=t(a,b,i,j)", T, trial[0], complex(c[0]))
        for ci, ti in zip(c[1:], trial[1:]):
            ctx.add("T(a,b,i,j)+=t(a,b,i,j)", T, ti, complex(ci))
        E = ccd_energy(ctx, B, T)
        energies.append(complex(ctx.tensor_download(E)))
        E.destroy()
    for x in err + trial + [R, s]:
        x.destroy()
    return T, energies, norms


def ccsd_solve(ctx, B, e_occ, e_virt, iterations, packed=False):
    """Jacobi iterations of the CCSD amplitude equations from zero amplitudes: t1 += R1 / (e_i - e_a),
    t2 += R2 / (e_i + e_j - e_a - e_b), both residuals evaluated at the old amplitudes.  One iteration = `ccsd_residual`
    + two `tcb_denominator_update`; the energy of the updated amplitudes is produced by the next residual evaluation
    (so `iterations` updates cost iterations + 1 evaluations).  packed=True: the pp ladder on packed storage, the packed
    integral blocks built once for all iterations.  Returns (T1, T2, [E_corr after each step])."""
    import numpy as np
    v, o = B["fvo"].extents
    T1, T2 = ctx.tensor_create((v, o)), ctx.tensor_create((v, v, o, o))
    R1, R2 = ctx.tensor_create((v, o)), ctx.tensor_create((v, v, o, o))
    ev, eo = -np.asarray(e_virt, dtype=np.float64), np.asarray(e_occ, dtype=np.float64)
    energies = []
    cache = {} if packed else None
    for it in range(iterations + 1):
        E, _, _ = ccsd_residual(ctx, B, T1, T2, R1, R2, cache)
        if it > 0:
            energies.append(complex(ctx.tensor_download(E)))
        E.destroy()
        if it == iterations:
            break
        ctx.denominator_update(T1, R1, [ev, eo], 1.0)
        ctx.denominator_update(T2, R2, [ev, ev, eo, eo], 1.0)
    for t in [R1, R2] + list((cache or {}).values()):
        t.destroy()
    return T1, T2, energies


def residual_norm(ctx, *residuals):
    """|R| = sqrt(sum <R|R>) over the given residual tensors -- the "norm of the residual vector" quoted per calculation in
    the paper: one `tcb_dot` into a rank-0 tensor per residual, read back as one number."""
    import math
    s = ctx.tensor_create(())
    total = 0.0
    for R in residuals:
        ctx.dot(s, R, R, True, 1.0)
        total += complex(ctx.tensor_download(s)).real
    s.destroy()
    return math.sqrt(total)


def ccsd_solve_diis(ctx, B, e_occ, e_virt, iterations, depth=6):
    """The CCSD iteration with DIIS over the combined (t1, t2) vector (oracle: cc.ccsd_diis): per evaluation the residuals,
    their norm, the error vectors e = R / D (`tcb_denominator_divide`), the trial vectors, one new row of
    <e_i|e_j> = <e1_i|e1_j> + <e2_i|e2_j> (`tcb_dot`), and the extrapolated amplitudes (`tcb_add`) -- all on the device;
    the depth x depth system is solved on the host.
    Returns (T1, T2, [E_corr of the amplitudes each evaluation saw], [residual norm |R| of each evaluation])."""
    import numpy as np
    v, o = B["fvo"].extents
    s1, s2 = (v, o), (v, v, o, o)
    T1, T2 = ctx.tensor_create(s1), ctx.tensor_create(s2)
    R1, R2 = ctx.tensor_create(s1), ctx.tensor_create(s2)
    ev, eo = -np.asarray(e_virt, dtype=np.float64), np.asarray(e_occ, dtype=np.float64)
    trial, err, energies, norms = [], [], [], []
    Bm = np.zeros((0, 0), dtype=np.complex128)
    s = ctx.tensor_create(())

    def dot(X, Y):
        ctx.dot(s, X, Y, True, 1.0)
        return complex(ctx.tensor_download(s))

    for _ in range(iterations):
        E, _, _ = ccsd_residual(ctx, B, T1, T2, R1, R2)
        energies.append(complex(ctx.tensor_download(E)))
        E.destroy()
        norms.append(float(np.sqrt(dot(R1, R1).real + dot(R2, R2).real)))
        if len(err) == depth:                      # the oldest pair leaves; its tensors are reused
            (e1, e2), (t1, t2) = err.pop(0), trial.pop(0)
            Bm = Bm[1:, 1:]
        else:
            e1, e2, t1, t2 = (ctx.tensor_create(x, zero=False) for x in (s1, s2, s1, s2))
        ctx.denominator_divide(e1, R1, [ev, eo], 1.0)
        ctx.denominator_divide(e2, R2, [ev, ev, eo, eo], 1.0)
        ctx.add("t(a,i)=T(a,i)", t1, T1, 1.0)
        ctx.add("t(a,i)+=e(a,i)", t1, e1, 1.0)
        ctx.add("t(a,b,i,j)=T(a,b,i,j)", t2, T2, 1.0)
        ctx.add("t(a,b,i,j)+=e(a,b,i,j)", t2, e2, 1.0)
        err.append((e1, e2))
        trial.append((t1, t2))
        m = len(err)
        row = np.array([dot(err[i][0], e1) + dot(err[i][1], e2) for i in range(m)])      # <e_i|e_new>; B is Hermitian
        Bn = np.zeros((m, m), dtype=np.complex128)
        Bn[:m - 1, :m - 1] = Bm
        Bn[:, m - 1] = row
        Bn[m - 1, :] = row.conj()
        Bn[m - 1, m - 1] = row[m - 1]
        Bm = Bn
        if m > 1:
            A = np.zeros((m + 1, m + 1), dtype=np.complex128)
            A[:m, :m] = Bm
            A[:m, m] = A[m, :m] = 1.0
            rhs = np.zeros(m + 1, dtype=np.complex128)
            rhs[m] = 1.0
            c = np.linalg.solve(A, rhs)[:m]
        else:
            c = np.ones(1, dtype=np.complex128)
        for k, (ci, (ta, tb)) in enumerate(zip(c, trial)):
            op = "=" if k == 0 else "+="
            ctx.add(f"T(a,i){op}t(a,i)", T1, ta, complex(ci))
            ctx.add(f"T(a,b,i,j){op}t(a,b,i,j)", T2, tb, complex(ci))
    for pair in err + trial:
        for x in pair:
            x.destroy()
    for x in (R1, R2, s):
        x.destroy()
    return T1, T2, energies, norms


CCD_FLOPS = lambda o, v: 8.0 * (                 # 8 real flop per complex multiply-add
    v * v * o * o * v                            # Fock vv
    + v * v * o * o * o                          # Fock oo
    + o ** 4 * v * v + v * v * o ** 4            # I1 build + hh ladder
    + v ** 4 * o * o                             # pp ladder
    + 2 * (o * v) ** 3                           # I2 build + ring
    + o * o * o * v * v + v * v * o * o * o      # I3 build + use
    + v * v * o * o * v + v * v * o * o * v)     # I4 build + use


def t3_term(ctx, W, T2, R3, X=None):
    """config 4: X(a,b,c,i,j,k) = sum_d W(b,c,d,k) T2(a,d,i,j);  R3 += P(a/bc)P(k/ij) X."""
    v, _, o, _ = T2.extents
    own = X is None
    if own:
        X = ctx.tensor_create((v, v, v, o, o, o))
    ctx.contract("X(a,b,c,i,j,k)=W(b,c,d,k)*T(a,d,i,j)", X, W, T2, 1.0)
    ctx.antisymmetrize("P(a/bc)P(k/ij):R(a,b,c,i,j,k)+=X(a,b,c,i,j,k)", R3, X, 1.0)
    if own:
        X.destroy()
    return R3


# ---- CCSDT ("CCSDT iterations"; the paper's production target beyond CCSD: Tables III-IV) --------
A3_PERMS, A3_SIGNS = [], []
for _pv, _sv in (((0, 1, 2), 1), ((1, 0, 2), -1), ((2, 1, 0), -1), ((0, 2, 1), -1), ((1, 2, 0), 1), ((2, 0, 1), 1)):
    for _po, _so in (((0, 1, 2), 1), ((1, 0, 2), -1), ((2, 1, 0), -1), ((0, 2, 1), -1), ((1, 2, 0), 1), ((2, 0, 1), 1)):
        A3_PERMS.append(list(_pv) + [3 + q for q in _po])
        A3_SIGNS.append(float(_sv * _so))


def t1_dressed_blocks(ctx, o, h, g, T1, names):
    """The blocks `names` (e.g. "ovvv", "fov") of the T1-similarity-transformed integrals, exp(-T1) H exp(T1), built from the
    FULL-range bare one-electron matrix h(p,q) and <pq||rs> = g(p,q,r,s) (device tensors over all n = o + v spinors) by binary
    contractions:  g~[PQRS] = X[P,p] X[Q,q] g[pqrs] Y[r,R] Y[s,S],  X = 1 - tau, Y = 1 + tau, tau[a,i] = t_i^a;
    f~ = X (h + J) Y with J(p,r) = sum_{i occ} sum_s g(p,i,r,s) Y[s,i].  Only the 16-byte-per-element t1 is read back to
    build the four row / column slices of X and Y on the host.  Returns {name: Tensor}."""
    import numpy as np
    n = g.extents[0]
    v = n - o
    t1 = ctx.tensor_download(T1)
    tau = np.zeros((n, n), dtype=np.complex128)
    tau[o:, :o] = t1
    X, Y = np.eye(n) - tau, np.eye(n) + tau
    ext = {"o": o, "v": v}
    rng = {"o": slice(0, o), "v": slice(o, n)}
    Xr = {c: ctx.tensor_from_numpy(np.asfortranarray(X[rng[c], :])) for c in "ov"}      # (|c|, n): rows of X
    Yc = {c: ctx.tensor_from_numpy(np.asfortranarray(Y[:, rng[c]])) for c in "ov"}      # (n, |c|): columns of Y
    Yocc = Y.copy()
    Yocc[:, o:] = 0.0
    Yp = ctx.tensor_from_numpy(np.asfortranarray(Yocc))
    new = lambda shape: ctx.tensor_create(shape, zero=False)
    out = {}
    # ---- f~ blocks
    fnames = [x for x in names if x[0] == "f"]
    if fnames:
        hJ = new((n, n))
        ctx.add("hJ(p,r)=h(p,r)", hJ, h, 1.0)
        ctx.contract("hJ(p,r)+=g(p,q,r,s)*Yp(s,q)", hJ, g, Yp, 1.0)
        for name in fnames:
            P, Q = name[1], name[2]
            F1 = new((n, ext[Q]))
            ctx.contract("F1(p,Q)=hJ(p,r)*Yc(r,Q)", F1, hJ, Yc[Q], 1.0)
            out[name] = new((ext[P], ext[Q]))
            ctx.contract("F(P,Q)=Xr(P,p)*F1(p,Q)", out[name], Xr[P], F1, 1.0)
            F1.destroy()
        hJ.destroy()
    # ---- g~ blocks.  Every step contracts the FIRST (unit-stride) index of its operand and appends the new index last:
    #     G1(q,r,s,P) = g(p,q,r,s) X(P,p);  G2(r,s,P,Q) = G1(q,..) X(Q,q);  G3(s,P,Q,R) = G2(r,..) Y(r,R);  g~(P,Q,R,S) = G3(s,..) Y(s,S)
    # so each operand is a K-major matrix as it lies in memory and each result a plain matrix: four TMA-fed GEMMs per block,
    # no gather tables and no transposition (contracting index 4, 3, 2, 1 in place left the free indices on both sides of the
    # contracted one: three of the four steps ran on gathered operands).  Partial transforms are shared between the blocks
    # that need them.
    gnames = sorted(x for x in names if x[0] != "f")
    for P in "ov":
        needP = [x for x in gnames if x[0] == P]
        if not needP:
            continue
        G1 = new((n, n, n, ext[P]))
        ctx.contract("G1(q,r,s,P)=g(p,q,r,s)*Xr(P,p)", G1, g, Xr[P], 1.0)
        for Q in "ov":
            needQ = [x for x in needP if x[1] == Q]
            if not needQ:
                continue
            G2 = new((n, n, ext[P], ext[Q]))
            ctx.contract("G2(r,s,P,Q)=G1(q,r,s,P)*Xr(Q,q)", G2, G1, Xr[Q], 1.0)
            for Rr in "ov":
                needR = [x for x in needQ if x[2] == Rr]
                if not needR:
                    continue
                G3 = new((n, ext[P], ext[Q], ext[Rr]))
                ctx.contract("G3(s,P,Q,R)=G2(r,s,P,Q)*Yc(r,R)", G3, G2, Yc[Rr], 1.0)
                for name in needR:
                    out[name] = new((ext[P], ext[Q], ext[Rr], ext[name[3]]))
                    ctx.contract("G(P,Q,R,S)=G3(s,P,Q,R)*Yc(s,S)", out[name], G3, Yc[name[3]], 1.0)
                G3.destroy()
            G2.destroy()
        G1.destroy()
    for t in list(Xr.values()) + list(Yc.values()) + [Yp]:
        t.destroy()
    return out


CCSDT_BLOCKS = ("foo", "fvv", "fov", "fvo", "vvoo", "oovv", "oooo", "vvvv", "ovvo", "ooov", "ovvv", "ovoo", "vvov", "ovov")


def ccsdt_residual(ctx, o, h, g, T1, T2, T3, R1=None, R2=None, R3=None):
    """Spin-orbital CCSDT residuals R1, R2, R3 = <Phi_mu| exp(-T) H exp(T) |Phi0>, T = T1 + T2 + T3 (PAPER Eqs. 2-3), as binary
    tensor operations.  T1 is absorbed exactly into the integrals (`t1_dressed_blocks`); with the dressed blocks the
    equations are those of T = T2 + T3 (oracle: cc.ccsdt_residual_unfactorised, 5 + 13 + 19 terms, pinned to the Fock space):
      R1 = f~vo + f~ov.T2 + 1/2 g~ooov.T2 + 1/2 g~ovvv.T2 + 1/4 g~oovv.T3
      R2 = [CCD residual of the dressed blocks] + f~ov.T3 + 1/2 P(ij) g~ooov.T3 + 1/2 P(ab) g~ovvv.T3
      R3 = A3 X,  X = Wovoo.T2 + Wvvov.T2 + Fo.T3 + Fv.T3 + Woooo.T3 + Wvvvv.T3 + Wr.T3  (seven rank-6 contractions into one X,
           the 36-term antisymmetriser as a 4-term and a 9-term permute-sum), the W / F intermediates carrying the quadratic
           T2 T2 and T2 T3 terms.
    h (n,n) bare one-electron matrix, g (n,n,n,n) = <pq||rs>, n = o + v.  Returns (R1, R2, R3)."""
    v = T1.extents[0]
    B = t1_dressed_blocks(ctx, o, h, g, T1, CCSDT_BLOCKS)
    new = lambda shape: ctx.tensor_create(shape, zero=False)
    con, add = ctx.contract, ctx.add
    # ---- singles
    if R1 is None:
        R1 = new((v, o))
    add("R(a,i)=f(a,i)", R1, B["fvo"], 1.0)
    con("R(a,i)+=f(l,d)*T(d,a,l,i)", R1, B["fov"], T2, 1.0)
    con("R(a,i)+=W(l,m,i,d)*T(d,a,l,m)", R1, B["ooov"], T2, 0.5)
    con("R(a,i)+=W(l,a,d,e)*T(d,e,l,i)", R1, B["ovvv"], T2, 0.5)
    con("R(a,i)+=T(d,e,a,l,m,i)*W(l,m,d,e)", R1, T3, B["oovv"], 0.25)
    # ---- doubles: the CCD program on the dressed blocks + the three T3 terms
    R2 = ccd_residual(ctx, B, T2, R2)
    con("R(a,b,i,j)+=T(d,a,b,l,i,j)*f(l,d)", R2, T3, B["fov"], 1.0)
    X2 = new((v, v, o, o))
    con("X(a,b,i,j)=T(d,a,b,l,m,j)*W(l,m,i,d)", X2, T3, B["ooov"], 1.0)
    ctx.antisymmetrize("P(ij):R(a,b,i,j)+=X(a,b,i,j)", R2, X2, 0.5)
    con("X(a,b,i,j)=W(l,a,d,e)*T(d,e,b,l,i,j)", X2, B["ovvv"], T3, 1.0)
    ctx.antisymmetrize("P(ab):R(a,b,i,j)+=X(a,b,i,j)", R2, X2, 0.5)
    X2.destroy()
    # ---- triples: intermediates
    Wovoo = new((o, v, o, o))
    add("W(l,a,i,j)=g(l,a,i,j)", Wovoo, B["ovoo"], 0.25)
    con("W(l,a,i,j)+=f(l,d)*T(d,a,i,j)", Wovoo, B["fov"], T2, 0.25)
    con("W(m,a,i,j)+=g(l,m,i,d)*T(d,a,l,j)", Wovoo, B["ooov"], T2, -0.5)
    con("W(l,a,j,k)+=g(l,a,d,e)*T(d,e,j,k)", Wovoo, B["ovvv"], T2, 0.125)
    con("W(l,a,i,j)+=g(l,m,d,e)*T(d,e,a,m,i,j)", Wovoo, B["oovv"], T3, -0.125)
    Wvvov = new((v, v, o, v))
    add("W(a,b,i,d)=g(a,b,i,d)", Wvvov, B["vvov"], 0.25)
    con("W(a,b,i,d)+=T(a,b,l,m)*g(l,m,i,d)", Wvvov, T2, B["ooov"], 0.125)
    con("W(a,b,i,e)+=g(l,a,d,e)*T(d,b,l,i)", Wvvov, B["ovvv"], T2, -0.5)
    con("W(a,b,i,d)+=g(l,m,d,e)*T(e,a,b,l,m,i)", Wvvov, B["oovv"], T3, -0.125)
    Fo, Fv = new((o, o)), new((v, v))
    add("F(m,i)=f(m,i)", Fo, B["foo"], -1.0 / 12.0)
    con("F(m,i)+=g(l,m,d,e)*T(d,e,l,i)", Fo, B["oovv"], T2, -1.0 / 24.0)
    add("F(a,e)=f(a,e)", Fv, B["fvv"], 1.0 / 12.0)
    con("F(a,e)+=g(l,m,d,e)*T(d,a,l,m)", Fv, B["oovv"], T2, -1.0 / 24.0)
    Woooo, Wvvvv, Wr = new((o, o, o, o)), new((v, v, v, v)), new((o, v, o, v))
    add("W(l,m,i,j)=g(l,m,i,j)", Woooo, B["oooo"], 1.0 / 24.0)
    con("W(l,m,i,j)+=g(l,m,d,e)*T(d,e,i,j)", Woooo, B["oovv"], T2, 1.0 / 48.0)
    add("W(a,b,d,e)=g(a,b,d,e)", Wvvvv, B["vvvv"], 1.0 / 24.0)
    con("W(a,b,d,e)+=T(a,b,l,m)*g(l,m,d,e)", Wvvvv, T2, B["oovv"], 1.0 / 48.0)
    add("W(m,a,i,e)=g(m,a,i,e)", Wr, B["ovov"], -0.25)
    con("W(m,a,i,e)+=g(l,m,d,e)*T(d,a,l,i)", Wr, B["oovv"], T2, 0.25)
    for t in B.values():
        t.destroy()
    # ---- triples: seven contractions into one X, one antisymmetrisation
    X = new((v, v, v, o, o, o))
    con("X(a,b,c,i,j,k)=W(l,a,i,j)*T(b,c,l,k)", X, Wovoo, T2, 1.0)
    con("X(a,b,c,i,j,k)+=W(a,b,i,d)*T(d,c,j,k)", X, Wvvov, T2, 1.0)
    con("X(a,b,c,i,j,k)+=F(m,i)*T(a,b,c,m,j,k)", X, Fo, T3, 1.0)
    con("X(a,b,c,i,j,k)+=F(a,e)*T(e,b,c,i,j,k)", X, Fv, T3, 1.0)
    con("X(a,b,c,i,j,k)+=W(l,m,i,j)*T(a,b,c,l,m,k)", X, Woooo, T3, 1.0)
    con("X(a,b,c,i,j,k)+=W(a,b,d,e)*T(d,e,c,i,j,k)", X, Wvvvv, T3, 1.0)
    con("X(a,b,c,i,j,k)+=W(m,a,i,e)*T(e,b,c,m,j,k)", X, Wr, T3, 1.0)
    for t in (Wovoo, Wvvov, Fo, Fv, Woooo, Wvvvv, Wr):
        t.destroy()
    # A3 = [P(a/bc) P(k/ij)] [P(bc) P(ij)]: (1 - (ab) - (ac))(1 - (bc)) runs over all six signed permutations of (a,b,c), likewise
    # for (i,j,k).  As ONE 36-term tcb_permsum the generic gather kernel took 130 ms on the 6 GB tensors of o=12, v=60; as a
    # 4-term pass (index a stays unit-stride in every term) followed by the 9-term pass of the orbit kernel it takes ~10 ms.
    Y = new((v, v, v, o, o, o))
    ctx.antisymmetrize("P(bc)P(ij):Y(a,b,c,i,j,k)=X(a,b,c,i,j,k)", Y, X, 1.0)
    X.destroy()
    if R3 is None:
        R3 = new((v, v, v, o, o, o))
    ctx.antisymmetrize("P(a/bc)P(k/ij):R(a,b,c,i,j,k)=Y(a,b,c,i,j,k)", R3, Y, 1.0)
    Y.destroy()
    return R1, R2, R3


def ccsdt_residual_packed(ctx, o, h, g, T1, T2, T3p, R1=None, R2=None, R3p=None):
    """`ccsdt_residual` on index-permutation-symmetric packed storage (SURVEY 8(f)-2 applied to 8(f)-3; PAPER.md:202, 440,
    452): the triples amplitudes and the triples residual exist only as T3p, R3p(a<b<c, i<j<k) -- 1/36 of the dense tensor
    (120 MB instead of 6 GB at o = 12, v = 60); no rank-6 dense tensor is ever formed.  T2 must be antisymmetric in (a,b) and
    in (i,j) (it is in `ccsdt_solve`).  T3p is read by three packed views (`tcb_unpack` with groups on both sides),
        Tq(d<e, c, i<j<k)      To(a<b<c, l<m, k)      Tr(b<c, j<k, e, m) = T3(b,c,e,j,k,m)
    (T3(e,b,c,..) = T3(b,c,e,..): a cyclic relabelling has sign +), and the seven rank-6 contractions collapse onto three
    packed accumulators -- the full antisymmetriser A3 that follows does not care which of a, b, c (of i, j, k) a term calls
    its "single" index, and only the antisymmetric part of an intermediate survives it:
        Xq(a<b, c, i<j<k)  = 2 Wvvvv(a<b, d<e) Tq(d<e, c, ijk)          + Tq(a<b, e, ijk) Fv(c, e)
        Xo(a<b<c, i<j, k)  = 2 To(abc, l<m, k) Woooo(l<m, i<j)          + To(abc, i<j, m) Fo(m, k)
        Xr(a, i, b<c, j<k) = Wr(m,a,i,e) Tr(b<c, j<k, e, m) + Wvvov(b<c, i, d) T2(d, a, j<k) + Wovoo(l, a, j<k) T2(b<c, l, i)
    against the dense program: 1/32 of the flops for the vvvv term, 1/4 for the ring term.  On an X antisymmetric in (b,c)
    and (j,k) the 36-term A3 is 4 P(a/bc) P(i/jk), on Xq it is 12 P(c/ab), on Xo 12 P(k/ij): three `tcb_antisym_pack` calls
    (9 + 3 + 3 signed reads per element of R3p).  Returns (R1, R2, R3p); needs o >= 3 and v >= 3."""
    v = T1.extents[0]
    if o < 3 or v < 3:
        raise ValueError("ccsdt_residual_packed needs o >= 3 and v >= 3 (a<b<c groups)")
    B = t1_dressed_blocks(ctx, o, h, g, T1, CCSDT_BLOCKS)
    new = lambda shape: ctx.tensor_create(shape, zero=False)
    con, add, pack, unpack = ctx.contract, ctx.add, ctx.pack, ctx.unpack
    nv2, nv3, no2, no3 = (ctx.packed_extent(v, 2), ctx.packed_extent(v, 3), ctx.packed_extent(o, 2), ctx.packed_extent(o, 3))

    def packed(shape, spec, src):
        t = new(shape)
        pack(spec, t, src)
        return t
    # ---- the three packed views of T3, the packed views of T2 and of the dressed integrals
    Tq, To, Tr = new((nv2, v, no3)), new((nv3, no2, o)), new((nv2, no2, v, o))
    unpack("Tq(d<e,c,i<j<k)=T(d<e<c,i<j<k)", Tq, T3p, 1.0)
    unpack("To(a<b<c,l<m,k)=T(a<b<c,l<m<k)", To, T3p, 1.0)
    unpack("Tr(b<c,j<k,e,m)=T(b<c<e,j<k<m)", Tr, T3p, 1.0)
    T2p = packed((nv2, no2), "P(a<b,l<m)=T(a,b,l,m)", T2)
    T2x = packed((nv2, o, o), "P(b<c,l,i)=T(b,c,l,i)", T2)
    T2y = packed((v, v, no2), "P(d,a,j<k)=T(d,a,j,k)", T2)
    gp = packed((no2, nv2), "P(l<m,d<e)=g(l,m,d,e)", B["oovv"])
    gs = packed((o, o, nv2), "P(l,m,d<e)=g(l,m,d,e)", B["oovv"])
    gt = packed((no2, v, v), "P(l<m,d,e)=g(l,m,d,e)", B["oovv"])
    gq = packed((no2, o, v), "P(l<m,i,d)=g(l,m,i,d)", B["ooov"])
    gr = packed((o, v, nv2), "P(l,a,d<e)=g(l,a,d,e)", B["ovvv"])
    # ---- singles
    if R1 is None:
        R1 = new((v, o))
    add("R(a,i)=f(a,i)", R1, B["fvo"], 1.0)
    con("R(a,i)+=f(l,d)*T(d,a,l,i)", R1, B["fov"], T2, 1.0)
    con("R(a,i)+=W(l,m,i,d)*T(d,a,l,m)", R1, B["ooov"], T2, 0.5)
    con("R(a,i)+=W(l,a,d,e)*T(d,e,l,i)", R1, B["ovvv"], T2, 0.5)
    con("R(a,i)+=T(x,y,a,i)*W(y,x)", R1, Tr, gp, 1.0)                  # 1/4 sum_{de,lm} = sum_{d<e,l<m}
    # ---- doubles: the CCD program on the dressed blocks + the three T3 terms
    R2 = ccd_residual(ctx, B, T2, R2)
    R2p = new((nv2, no2))
    con("R(x,y)=T(x,y,d,l)*f(l,d)", R2p, Tr, B["fov"], 1.0)
    unpack("R(a,b,i,j)+=P(a<b,i<j)", R2, R2p, 1.0)
    R2p.destroy()
    X2, X2a, X2b = new((v, v, o, o)), new((nv2, o, o)), new((v, v, no2))
    con("X(x,i,j)=T(x,z,d,j)*W(z,i,d)", X2a, Tr, gq, 2.0)
    unpack("X(a,b,i,j)=P(a<b,i,j)", X2, X2a, 1.0)
    ctx.antisymmetrize("P(ij):R(a,b,i,j)+=X(a,b,i,j)", R2, X2, 0.5)
    con("X(a,b,y)=W(l,a,z)*T(z,y,b,l)", X2b, gr, Tr, 2.0)
    unpack("X(a,b,i,j)=P(a,b,i<j)", X2, X2b, 1.0)
    ctx.antisymmetrize("P(ab):R(a,b,i,j)+=X(a,b,i,j)", R2, X2, 0.5)
    for t in (X2, X2a, X2b):
        t.destroy()
    # ---- triples: intermediates.  Wovoo and Wvvov: T2 terms dense, their antisymmetric part packed, the T3 term added packed
    Wd, Wa = new((o, v, o, o)), new((o, v, o, o))
    add("W(l,a,i,j)=g(l,a,i,j)", Wd, B["ovoo"], 0.25)
    con("W(l,a,i,j)+=f(l,d)*T(d,a,i,j)", Wd, B["fov"], T2, 0.25)
    con("W(m,a,i,j)+=g(l,m,i,d)*T(d,a,l,j)", Wd, B["ooov"], T2, -0.5)
    con("W(l,a,j,k)+=g(l,a,d,e)*T(d,e,j,k)", Wd, B["ovvv"], T2, 0.125)
    ctx.antisymmetrize("P(ij):A(l,a,i,j)=W(l,a,i,j)", Wa, Wd, 0.5)
    Wovoo = packed((o, v, no2), "P(l,a,i<j)=W(l,a,i,j)", Wa)
    con("W(l,a,y)+=g(l,m,z)*T(z,y,a,m)", Wovoo, gs, Tr, -0.25)
    Wd.destroy()
    Wa.destroy()
    Wd, Wa = new((v, v, o, v)), new((v, v, o, v))
    add("W(a,b,i,d)=g(a,b,i,d)", Wd, B["vvov"], 0.25)
    con("W(a,b,i,d)+=T(a,b,l,m)*g(l,m,i,d)", Wd, T2, B["ooov"], 0.125)
    con("W(a,b,i,e)+=g(l,a,d,e)*T(d,b,l,i)", Wd, B["ovvv"], T2, -0.5)
    ctx.antisymmetrize("P(ab):A(a,b,i,d)=W(a,b,i,d)", Wa, Wd, 0.5)
    Wvvov = packed((nv2, o, v), "P(a<b,i,d)=W(a,b,i,d)", Wa)
    con("W(x,i,d)+=T(x,z,e,i)*g(z,d,e)", Wvvov, Tr, gt, -0.25)
    Wd.destroy()
    Wa.destroy()
    Fo, Fv = new((o, o)), new((v, v))
    add("F(m,i)=f(m,i)", Fo, B["foo"], -1.0 / 12.0)
    con("F(m,i)+=g(l,m,d,e)*T(d,e,l,i)", Fo, B["oovv"], T2, -1.0 / 24.0)
    add("F(a,e)=f(a,e)", Fv, B["fvv"], 1.0 / 12.0)
    con("F(a,e)+=g(l,m,d,e)*T(d,a,l,m)", Fv, B["oovv"], T2, -1.0 / 24.0)
    Woooo, Wvvvv = new((no2, no2)), new((nv2, nv2))
    gpk = packed((no2, no2), "P(l<m,i<j)=g(l,m,i,j)", B["oooo"])
    add("W(z,y)=g(z,y)", Woooo, gpk, 1.0 / 24.0)
    gpk.destroy()
    con("W(z,y)+=g(z,x)*T(x,y)", Woooo, gp, T2p, 1.0 / 24.0)           # 1/48 sum_de = 1/24 sum_{d<e}
    gpk = packed((nv2, nv2), "P(a<b,d<e)=g(a,b,d,e)", B["vvvv"])
    add("W(x,z)=g(x,z)", Wvvvv, gpk, 1.0 / 24.0)
    gpk.destroy()
    con("W(x,z)+=T(x,y)*g(y,z)", Wvvvv, T2p, gp, 1.0 / 24.0)
    Wr = new((o, v, o, v))
    add("W(m,a,i,e)=g(m,a,i,e)", Wr, B["ovov"], -0.25)
    con("W(m,a,i,e)+=g(l,m,d,e)*T(d,a,l,i)", Wr, B["oovv"], T2, 0.25)
    for t in list(B.values()) + [gp, gs, gt, gq, gr, T2p]:
        t.destroy()
    # ---- triples: the three packed accumulators
    Xq, Xo, Xr = new((nv2, v, no3)), new((nv3, no2, o)), new((v, o, nv2, no2))
    con("X(x,c,t)=W(x,z)*T(z,c,t)", Xq, Wvvvv, Tq, 2.0)
    con("X(x,c,t)+=T(x,e,t)*F(c,e)", Xq, Tq, Fv, 1.0)
    con("X(t,y,k)=T(t,z,k)*W(z,y)", Xo, To, Woooo, 2.0)
    con("X(t,y,k)+=T(t,y,m)*F(m,k)", Xo, To, Fo, 1.0)
    con("X(a,i,x,y)=W(m,a,i,e)*T(x,y,e,m)", Xr, Wr, Tr, 1.0)
    con("X(a,i,x,y)+=W(x,i,d)*T(d,a,y)", Xr, Wvvov, T2y, 1.0)
    con("X(a,i,x,y)+=W(l,a,y)*T(x,l,i)", Xr, Wovoo, T2x, 1.0)
    for t in (Wovoo, Wvvov, Fo, Fv, Woooo, Wvvvv, Wr, Tq, To, Tr, T2x, T2y):
        t.destroy()
    if R3p is None:
        R3p = new((nv3, no3))
    ctx.antisym_pack("R(a<b<c,i<j<k)=X(a,i,b<c,j<k)", R3p, Xr, 4.0)
    ctx.antisym_pack("R(a<b<c,i<j<k)+=X(a<b,c,i<j<k)", R3p, Xq, 12.0)
    ctx.antisym_pack("R(a<b<c,i<j<k)+=X(a<b<c,i<j,k)", R3p, Xo, 12.0)
    for t in (Xq, Xo, Xr):
        t.destroy()
    return R1, R2, R3p


_TUPLES = {}


def _tuple_members(n, k):
    """index arrays (a, b[, c]) of the strictly increasing k-tuples of range(n), first label fastest (the packed order);
    the pairs with b < c are the first c(c-1)/2 pairs, so the triples are prefixes of the pair list, one per c"""
    import numpy as np
    if (n, k) not in _TUPLES:
        b = np.repeat(np.arange(n), np.arange(n))
        a = np.concatenate([np.arange(x) for x in range(n)]) if n else np.zeros(0, dtype=np.int64)
        if k == 2:
            _TUPLES[(n, k)] = (a, b)
        else:
            cnt = [c * (c - 1) // 2 for c in range(n)]
            _TUPLES[(n, k)] = (np.concatenate([a[:m] for m in cnt]), np.concatenate([b[:m] for m in cnt]),
                               np.repeat(np.arange(n), cnt))
    return _TUPLES[(n, k)]


def _tuple_sums(e, k):
    """sum of e over the strictly increasing k-tuples of range(len(e)), in the packed order, members added first to last"""
    import numpy as np
    e = np.asarray(e, dtype=np.float64)
    m = _tuple_members(len(e), k)
    out = e[m[0]] + e[m[1]]
    return out if k == 2 else out + e[m[2]]


def ccsdt_solve(ctx, o, h, g, f_diag, iterations, packed=False):
    """Jacobi iterations of the CCSDT amplitude equations from zero amplitudes (oracle: cc.ccsdt_jacobi): per iteration
    `ccsdt_residual`, the residual norm |R|, the energy of the amplitudes the evaluation saw, and three
    `tcb_denominator_update`.  f_diag: the n orbital energies (diagonal of the Fock matrix).
    packed=True: `ccsdt_residual_packed`; T3 and R3 live as (a<b<c, i<j<k) packed tensors (their denominators are the sums
    of the orbital energies over the tuples, |R3|^2 = 36 |R3p|^2) and T3 comes back packed.
    Returns (T1, T2, T3, [E_corr per evaluation], [|R| per evaluation])."""
    import math
    import numpy as np
    n = g.extents[0]
    v = n - o
    e = np.asarray(f_diag, dtype=np.float64)
    eo, ev = e[:o], -e[o:]
    if packed:
        shape3 = (ctx.packed_extent(v, 3), ctx.packed_extent(o, 3))
        eps3 = [np.asarray(_tuple_sums(ev, 3)), np.asarray(_tuple_sums(eo, 3))]
    else:
        shape3 = (v, v, v, o, o, o)
        eps3 = [ev, ev, ev, eo, eo, eo]
    residual = ccsdt_residual_packed if packed else ccsdt_residual
    T1, T2, T3 = ctx.tensor_create((v, o)), ctx.tensor_create((v, v, o, o)), ctx.tensor_create(shape3)
    R1, R2, R3 = ctx.tensor_create((v, o)), ctx.tensor_create((v, v, o, o)), ctx.tensor_create(shape3, zero=False)
    # bare blocks for the energy: E = f_ia t_i^a + 1/4 <ij||ab> t_ij^ab + 1/2 <ij||ab> t_i^a t_j^b
    Bz = t1_dressed_blocks(ctx, o, h, g, T1, ("fov", "oovv"))          # T1 = 0 here: the bare blocks
    energies, norms = [], []
    for _ in range(iterations):
        E = ctx.tensor_create(())
        Y = ctx.tensor_create((o, v), zero=False)
        ctx.contract("E()=f(i,a)*T(a,i)", E, Bz["fov"], T1, 1.0)
        ctx.contract("E()+=W(i,j,a,b)*T(a,b,i,j)", E, Bz["oovv"], T2, 0.25)
        ctx.contract("Y(i,a)=W(i,j,a,b)*T(b,j)", Y, Bz["oovv"], T1, 1.0)
        ctx.contract("E()+=Y(i,a)*T(a,i)", E, Y, T1, 0.5)
        residual(ctx, o, h, g, T1, T2, T3, R1, R2, R3)
        energies.append(complex(ctx.tensor_download(E)))
        if packed:
            norms.append(math.sqrt(residual_norm(ctx, R1, R2) ** 2 + 36.0 * residual_norm(ctx, R3) ** 2))
        else:
            norms.append(residual_norm(ctx, R1, R2, R3))
        E.destroy()
        Y.destroy()
        ctx.denominator_update(T1, R1, [ev, eo], 1.0)
        ctx.denominator_update(T2, R2, [ev, ev, eo, eo], 1.0)
        ctx.denominator_update(T3, R3, eps3, 1.0)
    for t in list(Bz.values()) + [R1, R2, R3]:
        t.destroy()
    return T1, T2, T3, energies, norms


def ccsdt_solve_diis(ctx, o, h, g, f_diag, iterations, depth=6, packed=True):
    """The CCSDT iteration with DIIS over the combined (t1, t2, t3) vector (oracle: cc.ccsdt_diis): per evaluation the three
    residuals, their norm, the error vectors e = R / D (`tcb_denominator_divide`), the trial vectors, one new row of
    <e_i|e_j> (three `tcb_dot` per pair), the extrapolated amplitudes (`tcb_add`) -- all on the device; the depth x depth
    system is solved on the host.  packed=True: t3, R3 and the DIIS history of t3 live as (a<b<c, i<j<k) tensors (each
    history entry 1/36 of a dense one); an inner product over the full antisymmetric tensor is 36 times the packed one.
    Returns (T1, T2, T3, [E_corr of the amplitudes each evaluation saw], [residual norm of each evaluation])."""
    import numpy as np
    n = g.extents[0]
    v = n - o
    e = np.asarray(f_diag, dtype=np.float64)
    eo, ev = e[:o], -e[o:]
    if packed:
        shape3, lab3, w3 = (ctx.packed_extent(v, 3), ctx.packed_extent(o, 3)), "x,y", 36.0
        eps3 = [np.asarray(_tuple_sums(ev, 3)), np.asarray(_tuple_sums(eo, 3))]
    else:
        shape3, lab3, w3 = (v, v, v, o, o, o), "a,b,c,i,j,k", 1.0
        eps3 = [ev, ev, ev, eo, eo, eo]
    shapes = [(v, o), (v, v, o, o), shape3]
    labels = ["a,i", "a,b,i,j", lab3]
    eps = [[ev, eo], [ev, ev, eo, eo], eps3]
    weight = [1.0, 1.0, w3]
    residual = ccsdt_residual_packed if packed else ccsdt_residual
    T = [ctx.tensor_create(s_) for s_ in shapes]
    R = [ctx.tensor_create(s_) for s_ in shapes]
    Bz = t1_dressed_blocks(ctx, o, h, g, T[0], ("fov", "oovv"))        # T1 = 0 here: the bare blocks, for the energy
    trial, err, energies, norms = [], [], [], []
    Bm = np.zeros((0, 0), dtype=np.complex128)
    s = ctx.tensor_create(())

    def dot(X, Y):
        ctx.dot(s, X, Y, True, 1.0)
        return complex(ctx.tensor_download(s))

    for _ in range(iterations):
        E = ctx.tensor_create(())
        Y = ctx.tensor_create((o, v), zero=False)
        ctx.contract("E()=f(i,a)*T(a,i)", E, Bz["fov"], T[0], 1.0)
        ctx.contract("E()+=W(i,j,a,b)*T(a,b,i,j)", E, Bz["oovv"], T[1], 0.25)
        ctx.contract("Y(i,a)=W(i,j,a,b)*T(b,j)", Y, Bz["oovv"], T[0], 1.0)
        ctx.contract("E()+=Y(i,a)*T(a,i)", E, Y, T[0], 0.5)
        residual(ctx, o, h, g, T[0], T[1], T[2], R[0], R[1], R[2])
        energies.append(complex(ctx.tensor_download(E)))
        E.destroy()
        Y.destroy()
        norms.append(float(np.sqrt(sum(w * dot(r, r).real for w, r in zip(weight, R)))))
        if len(err) == depth:                      # the oldest entry leaves; its tensors are reused
            ek, tk = err.pop(0), trial.pop(0)
            Bm = Bm[1:, 1:]
        else:
            ek = [ctx.tensor_create(s_, zero=False) for s_ in shapes]
            tk = [ctx.tensor_create(s_, zero=False) for s_ in shapes]
        for q in range(3):
            ctx.denominator_divide(ek[q], R[q], eps[q], 1.0)
            ctx.add(f"t({labels[q]})=T({labels[q]})", tk[q], T[q], 1.0)
            ctx.add(f"t({labels[q]})+=e({labels[q]})", tk[q], ek[q], 1.0)
        err.append(ek)
        trial.append(tk)
        m = len(err)
        row = np.array([sum(weight[q] * dot(err[i][q], ek[q]) for q in range(3)) for i in range(m)])   # <e_i|e_new>
        Bn = np.zeros((m, m), dtype=np.complex128)
        Bn[:m - 1, :m - 1] = Bm
        Bn[:, m - 1] = row
        Bn[m - 1, :] = row.conj()
        Bn[m - 1, m - 1] = row[m - 1]
        Bm = Bn
        if m > 1:
            A = np.zeros((m + 1, m + 1), dtype=np.complex128)
            A[:m, :m] = Bm
            A[:m, m] = A[m, :m] = 1.0
            rhs = np.zeros(m + 1, dtype=np.complex128)
            rhs[m] = 1.0
            c = np.linalg.solve(A, rhs)[:m]
        else:
            c = np.ones(1, dtype=np.complex128)
        for k, (ci, tk_) in enumerate(zip(c, trial)):
            op = "=" if k == 0 else "+="
            for q in range(3):
                ctx.add(f"T({labels[q]}){op}t({labels[q]})", T[q], tk_[q], complex(ci))
    for entry in err + trial:
        for x in entry:
            x.destroy()
    for x in R + [s] + list(Bz.values()):
        x.destroy()
    return T[0], T[1], T[2], energies, norms
