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


def ccd_residual(ctx, B, T, R=None):
    """B: dict name -> Tensor for foo, fvv, vvoo, oovv, oooo, vvvv, ovvo;  T: Tensor (v,v,o,o).
    Returns the residual tensor R (v,v,o,o); all work is enqueued on the context's stream."""
    v, _, o, _ = T.extents
    if R is None:
        R = ctx.tensor_create((v, v, o, o))
    X = ctx.tensor_create((v, v, o, o))
    ctx.add("R(a,b,i,j)=W(a,b,i,j)", R, B["vvoo"], 1.0)
    ctx.contract("X(a,b,i,j)=T(a,c,i,j)*f(b,c)", X, T, B["fvv"], 1.0)
    ctx.antisymmetrize("P(ab):R(a,b,i,j)+=X(a,b,i,j)", R, X, 1.0)
    ctx.contract("X(a,b,i,j)=T(a,b,i,k)*f(k,j)", X, T, B["foo"], 1.0)
    ctx.antisymmetrize("P(ij):R(a,b,i,j)+=X(a,b,i,j)", R, X, -1.0)
    I1 = ctx.tensor_create((o, o, o, o))
    ctx.add("I1(k,l,i,j)=W(k,l,i,j)", I1, B["oooo"], 1.0)
    ctx.contract("I1(k,l,i,j)+=W(k,l,c,d)*T(c,d,i,j)", I1, B["oovv"], T, 0.5)
    ctx.contract("R(a,b,i,j)+=T(a,b,k,l)*I1(k,l,i,j)", R, T, I1, 0.5)
    I1.destroy()
    ctx.contract("R(a,b,i,j)+=V(a,b,c,d)*T(c,d,i,j)", R, B["vvvv"], T, 0.5)
    I2 = ctx.tensor_create((o, v, v, o))
    ctx.add("I2(k,b,c,j)=W(k,b,c,j)", I2, B["ovvo"], 1.0)
    ctx.contract("I2(k,b,c,j)+=W(k,l,c,d)*T(b,d,j,l)", I2, B["oovv"], T, 0.5)
    ctx.contract("X(a,b,i,j)=T(a,c,i,k)*I2(k,b,c,j)", X, T, I2, 1.0)
    I2.destroy()
    ctx.antisymmetrize("P(ij)P(ab):R(a,b,i,j)+=X(a,b,i,j)", R, X, 1.0)
    I3 = ctx.tensor_create((o, o))
    ctx.contract("I3(l,i)=W(k,l,c,d)*T(d,c,i,k)", I3, B["oovv"], T, 1.0)
    ctx.contract("X(a,b,i,j)=T(a,b,l,j)*I3(l,i)", X, T, I3, 1.0)
    I3.destroy()
    ctx.antisymmetrize("P(ij):R(a,b,i,j)+=X(a,b,i,j)", R, X, -0.5)
    I4 = ctx.tensor_create((v, v))
    ctx.contract("I4(a,d)=W(k,l,c,d)*T(a,c,l,k)", I4, B["oovv"], T, 1.0)
    ctx.contract("X(a,b,i,j)=I4(a,d)*T(d,b,i,j)", X, I4, T, 1.0)
    I4.destroy()
    ctx.antisymmetrize("P(ab):R(a,b,i,j)+=X(a,b,i,j)", R, X, -0.5)
    X.destroy()
    return R


def ccd_energy(ctx, B, T):
    """E_corr = 1/4 sum_ijab <ij||ab> t_ij^ab -- the energy diagram (the 11th of the paper's 11 CCD diagrams,
    PAPER.md:276), a contraction into a rank-0 tensor.  Returns the rank-0 device tensor E (download it to read it)."""
    E = ctx.tensor_create(())
    ctx.contract("E()=W(i,j,a,b)*T(a,b,i,j)", E, B["oovv"], T, 0.25)
    return E


def ccd_solve(ctx, B, e_occ, e_virt, iterations, T=None):
    """Jacobi iterations of the CCD amplitude equations (PAPER.md:212 energy denominators, 406-410 "CC
    iteration"):  T <- T + R(T) / (e_i + e_j - e_a - e_b), from T (default: a zero tensor, whose first step is the MP2
    guess).  Every step is `ccd_residual` + one `tcb_denominator_update` + the rank-0 energy contraction; only the
    16-byte energy comes back to the host per iteration.  Returns (T, [E_corr after each step])."""
    import numpy as np
    v, _, o, _ = B["vvoo"].extents
    if T is None:
        T = ctx.tensor_create((v, v, o, o))
    ev, eo = -np.asarray(e_virt, dtype=np.float64), np.asarray(e_occ, dtype=np.float64)
    R = ctx.tensor_create((v, v, o, o))
    energies = []
    for _ in range(iterations):
        ccd_residual(ctx, B, T, R)
        ctx.denominator_update(T, R, [ev, ev, eo, eo], 1.0)
        E = ccd_energy(ctx, B, T)
        energies.append(complex(ctx.tensor_download(E)))
        E.destroy()
    R.destroy()
    return T, energies


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
