"""-m gpu: the CC 'generated driver' programs (config 2 CCD residual, config 4 T3 term) run call by call through the
C ABI, against the same programs evaluated by the oracle, and against the un-factorised equations."""
import numpy as np
import pytest

from oracle import cc
import paper_2409_06759_b200 as pkg
from paper_2409_06759_b200 import synth, ccd

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ctx():
    c = pkg.Context(0)
    yield c
    c.destroy()


@pytest.mark.parametrize("o,v", [(3, 5), (6, 14)])
def test_ccd_residual_program(ctx, o, v):
    B, T, eo, ev = synth.config_ccd(o, v)
    dB = {k: ctx.tensor_from_numpy(x) for k, x in B.items()}
    dT = ctx.tensor_from_numpy(T)
    dR = ccd.ccd_residual(ctx, dB, dT)
    R = ctx.tensor_download(dR)
    ref = cc.ccd_residual_program(B, T)
    scale = np.abs(ref).max()
    assert np.max(np.abs(R - ref)) <= 1e-11 * max(scale, np.abs(B["vvoo"]).max())
    # invariants: residual antisymmetry (to rounding), driver + Fock terms cancel for the MP2 guess
    assert np.max(np.abs(R + R.transpose(1, 0, 2, 3))) <= 1e-12 * scale
    assert np.max(np.abs(R + R.transpose(0, 1, 3, 2))) <= 1e-12 * scale
    if o <= 3:
        n = o + v
        f = np.zeros((n, n), dtype=np.complex128)
        f[:o, :o], f[o:, o:] = B["foo"], B["fvv"]
        g = synth.tensor(synth.SEED0 + 2, 1, [n] * 4, antisym=((0, 1), (2, 3)), sigma=0.1, hermitian=True)
        ref_unf = cc.ccd_residual_unfactorised(o, f, g, T)[0]
        assert np.max(np.abs(R - ref_unf)) <= 1e-11 * max(np.abs(ref_unf).max(), np.abs(B["vvoo"]).max())


@pytest.mark.parametrize("o,v,lanes", [(3, 5, True), (6, 14, True), (6, 14, False)])
def test_ccd_residual_program_call_by_call_with_each_calls_own_snorm(ctx, o, v, lanes):
    """north_star's metric is per element and per contraction: every one of the program's 19 calls (11 contractions, 5
    permute-sums, 3 adds) is compared with the oracle's evaluation of the same call, normalised by that call's
    snorm = |alpha| sum|L||R| + |D_in| -- an element that is small by cancellation cannot hide behind max|ref|."""
    from gpu_util import ShadowContext
    B, T, eo, ev = synth.config_ccd(o, v)
    sh = ShadowContext(ctx)
    sB = {k: sh.wrap(x) for k, x in B.items()}
    sT = sh.wrap(T)
    sR = ccd.ccd_residual(sh, sB, sT, lanes=lanes)
    assert sh.calls == 19 and sh.worst <= 1e-11
    ref = cc.ccd_residual_program(B, T)
    assert np.max(np.abs(sR.host - ref)) <= 1e-12 * np.abs(ref).max()     # the shadow's own chain is the oracle program
    # the pp ladder on packed storage: 2 packs + GEMM on packed indices + unpack instead of the one dense contraction
    sh2 = ShadowContext(ctx)
    cache = {}
    pR = ccd.ccd_residual(sh2, {k: sh2.wrap(x) for k, x in B.items()}, sh2.wrap(T), lanes=lanes, packed=cache)
    assert sh2.calls == 22 and sh2.worst <= 1e-11 and list(cache) == ["vvvv"]
    assert np.max(np.abs(pR.host - ref)) <= 1e-12 * np.abs(ref).max()
    assert np.max(np.abs(ctx.tensor_download(pR.gpu) - ctx.tensor_download(sR.gpu))) <= 1e-11 * np.abs(pR.norm).max()


def test_ccsd_residual_program_call_by_call_with_each_calls_own_snorm(ctx):
    from gpu_util import ShadowContext
    o, v = 4, 7
    n = o + v
    rng = np.random.default_rng(47)
    c = lambda *s: rng.standard_normal(s) + 1j * rng.standard_normal(s)
    g = synth.tensor(synth.SEED0 + 5, 1, [n] * 4, antisym=((0, 1), (2, 3)), sigma=0.1, hermitian=True)
    f = c(n, n) * 0.1
    f = f + f.conj().T + np.diag(np.concatenate([np.linspace(-2, -0.5, o), np.linspace(0.5, 3, v)]))
    t2 = c(v, v, o, o) * 0.2
    t2 = t2 - t2.transpose(1, 0, 2, 3)
    t2 = np.asfortranarray(t2 - t2.transpose(0, 1, 3, 2))
    t1 = np.asfortranarray(c(v, o) * 0.2)
    B = cc.ccsd_blocks(o, f, g)
    sh = ShadowContext(ctx)
    sB = {k: sh.wrap(x) for k, x in B.items()}
    sE, sR1, sR2 = ccd.ccsd_residual(sh, sB, sh.wrap(t1), sh.wrap(t2))
    assert sh.calls == 55 and sh.worst <= 1e-11
    e_ref, r1_ref, r2_ref = cc.ccsd_residual_program(B, t1, t2)
    assert np.max(np.abs(sR2.host - r2_ref)) <= 1e-12 * np.abs(r2_ref).max()
    assert abs(complex(sE.host) - e_ref) <= 1e-12 * abs(e_ref)
    # the same with the pp ladder on packed storage (W_abef only as Wp(a<b,e<f), P(ab) = tcb_antisym_pack)
    sh2 = ShadowContext(ctx)
    sB2 = {k: sh2.wrap(x) for k, x in B.items()}
    cache = {}
    pE, pR1, pR2 = ccd.ccsd_residual(sh2, sB2, sh2.wrap(t1), sh2.wrap(t2), packed=cache)
    assert sh2.calls == 59 and sh2.worst <= 1e-11 and sorted(cache) == ["vovv", "vvvv"]
    assert np.max(np.abs(pR2.host - r2_ref)) <= 1e-12 * np.abs(r2_ref).max()
    assert np.max(np.abs(ctx.tensor_download(pR2.gpu) - ctx.tensor_download(sR2.gpu))) <= 1e-11 * np.abs(pR2.norm).max()
    assert np.max(np.abs(ctx.tensor_download(pR1.gpu) - ctx.tensor_download(sR1.gpu))) <= 1e-11 * np.abs(pR1.norm).max()


def test_t3_term_program(ctx):
    o, v = 4, 9
    W, T2 = synth.config_t3(o, v)
    R3 = synth.config_t3_r3(o, v)
    dW, dT, dR = ctx.tensor_from_numpy(W), ctx.tensor_from_numpy(T2), ctx.tensor_from_numpy(R3)
    dX = ctx.tensor_create((v, v, v, o, o, o))
    ccd.t3_term(ctx, dW, dT, dR, dX)
    X, ref = cc.t3_term_program(W, T2, R3)
    gotX, got = ctx.tensor_download(dX), ctx.tensor_download(dR)
    assert np.max(np.abs(gotX - X)) <= 1e-11 * v * np.abs(W).max() * np.abs(T2).max()
    assert np.max(np.abs(got - ref)) <= 1e-11 * (np.abs(R3).max() + 9 * np.abs(X).max())


@pytest.mark.parametrize("o,v", [(3, 5), (20, 80)])
def test_ccd_energy_is_a_rank0_contraction(ctx, o, v):
    """E = 1/4 sum <ij||ab> t_ij^ab (the 11th CCD diagram): both operands contracted away, D of rank 0.
    At (20, 80) -- the bench size -- the inputs come from the device twin of the generator and are downloaded."""
    import oracle
    if o <= 6:
        B, T, eo, ev = synth.config_ccd(o, v)
        W, Th = B["oovv"], T
        dW, dT = ctx.tensor_from_numpy(W), ctx.tensor_from_numpy(Th)
    else:
        dW, dT = ctx.tensor_create((o, o, v, v)), ctx.tensor_create((v, v, o, o))
        ctx.synth_normal(dW, synth.SEED0 + 2, 1, antisym=((0, 1), (2, 3)), sigma=0.1)
        ctx.synth_normal(dT, synth.SEED0 + 2, 2, antisym=((0, 1), (2, 3)))
        W, Th = ctx.tensor_download(dW), ctx.tensor_download(dT)
    dE = ccd.ccd_energy(ctx, {"oovv": dW}, dT)
    got = ctx.tensor_download(dE)
    ref, sn = oracle.contract("E()=W(i,j,a,b)*T(a,b,i,j)", np.zeros(()), W, Th, 0.25)
    assert got.shape == ()
    assert abs(complex(got) - complex(np.asarray(ref).reshape(-1)[0])) <= 1e-11 * float(np.asarray(sn).reshape(-1)[0])
    plan = ctx.plan_describe("E()=W(i,j,a,b)*T(a,b,i,j)", dE, dW, dT)
    assert plan["route"] == "gemv" and (plan["M"], plan["N"]) == (1, 1) and not plan["permute_A"] and not plan["permute_B"]
    # accumulate form and determinism
    ctx.contract("E()+=W(i,j,a,b)*T(a,b,i,j)", dE, dW, dT, 0.25)
    twice = complex(ctx.tensor_download(dE))
    assert abs(twice - 2 * complex(got)) <= 1e-11 * float(np.asarray(sn).reshape(-1)[0])
    if o <= 6:
        # and it is the oracle's CCD energy (tier 1a)
        n = o + v
        f = np.zeros((n, n), dtype=np.complex128)
        f[:o, :o], f[o:, o:] = B["foo"], B["fvv"]
        g = synth.tensor(synth.SEED0 + 2, 1, [n] * 4, antisym=((0, 1), (2, 3)), sigma=0.1, hermitian=True)
        e_ref = cc.ccd_residual_unfactorised(o, f, g, T)[1]
        assert abs(complex(got) - complex(e_ref)) <= 1e-11 * float(np.asarray(sn).reshape(-1)[0])


@pytest.mark.parametrize("shape,eps_on,alpha", [
    ((5, 5, 3, 3), (1, 1, 1, 1), 1.0),
    ((7, 3, 5), (1, 0, 1), 0.5 - 2.0j),
    ((4, 4, 4, 3, 3, 3), (1, 1, 1, 1, 1, 1), -1.0),
    ((300, 7), (0, 1), 1.0j),
])
def test_denominator_update_matches_the_oracle(ctx, shape, eps_on, alpha):
    """tcb_denominator_update: T += alpha * R / (sum_k eps_k[i_k]), energies summed in index order, components divided
    separately -- the same roundings as the oracle, so the bound is a few ulp."""
    rng = np.random.default_rng(sum(shape))
    T = np.asfortranarray(rng.standard_normal(shape) + 1j * rng.standard_normal(shape))
    R = np.asfortranarray(rng.standard_normal(shape) + 1j * rng.standard_normal(shape))
    eps = [rng.uniform(0.5, 2.0, e) if on else None for e, on in zip(shape, eps_on)]
    dT, dR = ctx.tensor_from_numpy(T), ctx.tensor_from_numpy(R)
    ctx.denominator_update(dT, dR, eps, alpha)
    got, ref = ctx.tensor_download(dT), cc.denominator_update(T, R, eps, alpha)
    assert np.max(np.abs(got - ref)) <= 4e-16 * (np.abs(T).max() + abs(alpha) * np.abs(R).max() / 0.5)
    ctx.denominator_divide(dT, dR, eps, alpha)                            # the '=' form does not read T
    ref0 = cc.denominator_update(np.zeros_like(T), R, eps, alpha)
    assert np.max(np.abs(ctx.tensor_download(dT) - ref0)) <= 4e-16 * abs(alpha) * np.abs(R).max() / 0.5
    with pytest.raises(pkg.TcbError):
        ctx.denominator_update(dT, dR, [None] * len(shape), 1.0)          # no energies at all
    with pytest.raises(pkg.TcbError):
        ctx.denominator_update(dT, dT, eps, 1.0)                           # T aliases R
    for t in (dT, dR):
        t.destroy()


def test_ccd_jacobi_iterations_follow_the_oracle(ctx):
    """Five CC iterations (residual program + denominator update + rank-0 energy) on the GPU against the same five on
    the oracle; the converged run zeroes the residual (whose Fock-space pin is in tests/test_oracle_cc.py)."""
    o, v = 3, 5
    B, T_mp2, eo, ev = synth.config_ccd(o, v)
    dB = {k: ctx.tensor_from_numpy(x) for k, x in B.items()}
    dT, energies = ccd.ccd_solve(ctx, dB, eo, ev, 5)
    T_ref, e_ref = cc.ccd_jacobi(B, eo, ev, 5)
    assert np.max(np.abs(ctx.tensor_download(dT) - T_ref)) <= 1e-11 * np.abs(T_ref).max()
    for e, r in zip(energies, e_ref):
        assert abs(e - r) <= 1e-11 * abs(r)
    dT, energies = ccd.ccd_solve(ctx, dB, eo, ev, 35, dT)
    dR = ccd.ccd_residual(ctx, dB, dT)
    assert np.max(np.abs(ctx.tensor_download(dR))) <= 1e-11 * np.abs(B["vvoo"]).max()
    assert abs(energies[-1] - energies[-2]) <= 1e-12 * abs(energies[-1])
    assert abs(energies[-1] - cc.ccd_jacobi(B, eo, ev, 40)[1][-1]) <= 1e-11 * abs(energies[-1])


@pytest.mark.parametrize("o,v", [(3, 4), (5, 11)])
def test_ccsd_residual_program(ctx, o, v):
    """The CCSD residuals (singles, doubles, energy) as 55 ABI calls against the oracle's program of the same binary
    operations; at (3,4) also against the unfactorised tier (itself pinned to the Fock space)."""
    n = o + v
    rng = np.random.default_rng(o * 100 + v)
    c = lambda *s: rng.standard_normal(s) + 1j * rng.standard_normal(s)
    g = synth.tensor(synth.SEED0 + 5, 1, [n] * 4, antisym=((0, 1), (2, 3)), sigma=0.1, hermitian=True)
    f = c(n, n) * 0.1
    f = f + f.conj().T + np.diag(np.concatenate([np.linspace(-2, -0.5, o), np.linspace(0.5, 3, v)]))
    t2 = c(v, v, o, o) * 0.2
    t2 = t2 - t2.transpose(1, 0, 2, 3)
    t2 = np.asfortranarray(t2 - t2.transpose(0, 1, 3, 2))
    t1 = np.asfortranarray(c(v, o) * 0.2)
    B = cc.ccsd_blocks(o, f, g)
    assert set(B) == set(ccd.CCSD_BLOCKS)
    dB = {k: ctx.tensor_from_numpy(x) for k, x in B.items()}
    dT1, dT2 = ctx.tensor_from_numpy(t1), ctx.tensor_from_numpy(t2)
    live = ctx.launch_count()
    dE, dR1, dR2 = ccd.ccsd_residual(ctx, dB, dT1, dT2)
    assert ctx.launch_count() - live >= 55          # 55 ABI calls, at least one launch each
    E, R1, R2 = complex(ctx.tensor_download(dE)), ctx.tensor_download(dR1), ctx.tensor_download(dR2)
    e_ref, r1_ref, r2_ref = cc.ccsd_residual_program(B, t1, t2)
    assert abs(E - e_ref) <= 1e-11 * abs(e_ref)
    assert np.max(np.abs(R1 - r1_ref)) <= 1e-11 * np.abs(r1_ref).max()
    assert np.max(np.abs(R2 - r2_ref)) <= 1e-11 * np.abs(r2_ref).max()
    assert np.max(np.abs(R2 + R2.transpose(1, 0, 2, 3))) <= 1e-12 * np.abs(r2_ref).max()
    if o <= 3:
        e_u, r1_u, r2_u = cc.ccsd_residual_unfactorised(o, f, g, t1, t2)
        assert abs(E - e_u) <= 1e-11 * abs(e_u)
        assert np.max(np.abs(R1 - r1_u)) <= 1e-11 * np.abs(r1_u).max()
        assert np.max(np.abs(R2 - r2_u)) <= 1e-11 * np.abs(r2_u).max()
    for t in list(dB.values()) + [dT1, dT2, dE, dR1, dR2]:
        t.destroy()


def test_ccsd_jacobi_iterations_follow_the_oracle(ctx):
    """Four CCSD iterations on the GPU (residual program + two denominator updates each) against the oracle's."""
    o, v = 3, 4
    rng = np.random.default_rng(77)
    n = o + v
    c = lambda *s: rng.standard_normal(s) + 1j * rng.standard_normal(s)
    g = synth.tensor(synth.SEED0 + 6, 1, [n] * 4, antisym=((0, 1), (2, 3)), sigma=0.05, hermitian=True)
    e = np.concatenate([np.linspace(-2.0, -0.5, o), np.linspace(0.5, 3.0, v)])
    f = 0.05 * c(n, n)
    f = f + f.conj().T
    f[np.diag_indices(n)] = e
    B = cc.ccsd_blocks(o, f, g)
    dB = {k: ctx.tensor_from_numpy(x) for k, x in B.items()}
    dT1, dT2, energies = ccd.ccsd_solve(ctx, dB, e[:o], e[o:], 4)
    T1, T2, e_ref = cc.ccsd_jacobi(B, e[:o], e[o:], 4)
    assert np.max(np.abs(ctx.tensor_download(dT1) - T1)) <= 1e-11 * np.abs(T1).max()
    assert np.max(np.abs(ctx.tensor_download(dT2) - T2)) <= 1e-11 * np.abs(T2).max()
    assert len(energies) == 4
    for x, y in zip(energies, e_ref):
        assert abs(x - y) <= 1e-11 * abs(y)
    for t in list(dB.values()) + [dT1, dT2]:
        t.destroy()


@pytest.mark.parametrize("shape,conj", [((7, 5, 3), True), ((7, 5, 3), False), ((300, 41, 9), True), ((), True)])
def test_dot_matches_numpy(ctx, shape, conj):
    rng = np.random.default_rng(len(shape) + int(conj))
    X = np.asfortranarray(rng.standard_normal(shape) + 1j * rng.standard_normal(shape))
    Y = np.asfortranarray(rng.standard_normal(shape) + 1j * rng.standard_normal(shape))
    dX, dY, dD = ctx.tensor_from_numpy(X), ctx.tensor_from_numpy(Y), ctx.tensor_create(())
    alpha = 0.5 - 1.5j
    ctx.dot(dD, dX, dY, conj, alpha)
    ref = alpha * (np.vdot(X, Y) if conj else np.sum(X * Y))
    assert abs(complex(ctx.tensor_download(dD)) - ref) <= 1e-13 * abs(alpha) * np.sum(np.abs(X) * np.abs(Y))
    ctx.dot(dD, dX, dX, True, 1.0)
    got = complex(ctx.tensor_download(dD))
    assert got.imag == 0.0 and abs(got.real - np.sum(np.abs(X) ** 2)) <= 1e-13 * np.sum(np.abs(X) ** 2)
    with pytest.raises(pkg.TcbError):
        ctx.dot(dX, dX, dY, True, 1.0) if len(shape) else ctx.dot(dD, dD, dY, True, 1.0)
    for t in (dX, dY, dD):
        t.destroy()


def test_ccd_diis_follows_the_oracle_and_converges(ctx):
    o, v = 3, 5
    B, T_mp2, eo, ev = synth.config_ccd(o, v)
    dB = {k: ctx.tensor_from_numpy(x) for k, x in B.items()}
    dT, energies, norms = ccd.ccd_solve_diis(ctx, dB, eo, ev, 4)
    T_ref, e_ref, n_ref = cc.ccd_diis(B, eo, ev, 4)
    # the small linear system amplifies rounding differences of the inner products: 1e-9, not 1e-11
    assert np.max(np.abs(ctx.tensor_download(dT) - T_ref)) <= 1e-9 * np.abs(T_ref).max()
    for x, y in zip(energies, e_ref):
        assert abs(x - y) <= 1e-9 * abs(y)
    dT2, energies2, norms2 = ccd.ccd_solve_diis(ctx, dB, eo, ev, 16)
    dR = ccd.ccd_residual(ctx, dB, dT2)
    assert np.max(np.abs(ctx.tensor_download(dR))) <= 1e-11 * np.abs(B["vvoo"]).max()
    assert norms2[-1] <= 1e-11 * norms2[0]
    # same fixed point as the plain iteration
    assert abs(energies2[-1] - cc.ccd_jacobi(B, eo, ev, 40)[1][-1]) <= 1e-11 * abs(energies2[-1])


@pytest.mark.parametrize("o,v", [(3, 4), (4, 12)])
def test_triples_correction_program(ctx, o, v):
    """[T] from doubles: two rank-6 contractions, two 9-term antisymmetrisers (the second one is P(c/ab)P(i/jk)), the
    rank-6 denominator update and the inner product, against the oracle's program of the same calls."""
    n = o + v
    g = synth.tensor(synth.SEED0 + 7, 1, [n] * 4, antisym=((0, 1), (2, 3)), sigma=0.3, hermitian=True)
    rng = np.random.default_rng(o + v)
    t2 = rng.standard_normal((v, v, o, o)) + 1j * rng.standard_normal((v, v, o, o))
    t2 = t2 - t2.transpose(1, 0, 2, 3)
    t2 = np.asfortranarray(t2 - t2.transpose(0, 1, 3, 2))
    eo, ev = np.linspace(-2.0, -0.5, o), np.linspace(0.5, 3.0, v)
    W, U = np.asfortranarray(g[o:, o:, o:, :o]), np.asfortranarray(g[:o, o:, :o, :o])
    dW, dU, dT = ctx.tensor_from_numpy(W), ctx.tensor_from_numpy(U), ctx.tensor_from_numpy(t2)
    dE, dR3, dt3 = ccd.triples_correction(ctx, dW, dU, dT, eo, ev, keep=True)
    R3, t3, E = cc.triples_program(W, U, t2, eo, ev)
    scale = np.abs(R3).max()
    assert np.max(np.abs(ctx.tensor_download(dR3) - R3)) <= 1e-11 * scale
    assert np.max(np.abs(ctx.tensor_download(dt3) - t3)) <= 1e-11 * np.abs(t3).max()
    got = complex(ctx.tensor_download(dE))
    assert abs(got - E) <= 1e-11 * abs(E) and got.real < 0
    if o == 3:
        R3u, Eu = cc.triples_unfactorised(o, g, t2, eo, ev)
        assert abs(got - Eu) <= 1e-11 * abs(Eu)
    # (T): the singles term, the rank-6 amplitudes contracted down to rank 2 in place (GEMV route)
    t1 = np.asfortranarray(rng.standard_normal((v, o)) + 1j * rng.standard_normal((v, o)))
    oovv = np.asfortranarray(g[:o, :o, o:, o:])
    dT1, dV = ctx.tensor_from_numpy(t1), ctx.tensor_from_numpy(oovv)
    dE2, dEst = ccd.triples_correction(ctx, dW, dU, dT, eo, ev, T1=dT1, oovv=dV)
    _, est_ref = cc.triples_singles_term(t1, oovv, t3)
    assert abs(complex(ctx.tensor_download(dEst)) - est_ref) <= 1e-11 * abs(est_ref)
    assert complex(ctx.tensor_download(dE2)) == got                       # deterministic: the same bits twice
    plan = ctx.plan_describe("Y(a,i)=T(a,b,c,i,j,k)*W(j,k,b,c)", dT1, dt3, dV)
    assert plan["route"] == "gemv" and not plan["permute_A"]
    for t in (dW, dU, dT, dE, dR3, dt3, dT1, dV, dE2, dEst):
        t.destroy()


def test_cuda_graph_of_the_residual_call_list_replays_bit_identically(ctx):
    """tcb_capture_begin/end around a warm CCD residual evaluation: 35 kernel nodes plus the stream-ordered creation and
    destruction of its intermediates; a replay gives the same bits as the call-by-call evaluation and counts its launches."""
    o, v = 6, 14
    B, T, eo, ev = synth.config_ccd(o, v)
    dB = {k: ctx.tensor_from_numpy(x) for k, x in B.items()}
    dT = ctx.tensor_from_numpy(T)
    dR, dR2 = ctx.tensor_create((v, v, o, o)), ctx.tensor_create((v, v, o, o))
    for _ in range(2):
        ccd.ccd_residual(ctx, dB, dT, dR)
    ref = ctx.tensor_download(dR)
    l0 = ctx.launch_count()
    ctx.capture_begin()
    with pytest.raises(pkg.TcbError):
        ctx.capture_begin()                                     # one capture at a time
    ccd.ccd_residual(ctx, dB, dT, dR2)
    g = ctx.capture_end()
    per_list = ctx.launch_count() - l0
    assert per_list >= 19
    assert not np.any(ctx.tensor_download(dR2))                 # recorded, not executed
    for _ in range(2):
        l1 = ctx.launch_count()
        ctx.graph_launch(g)
        assert ctx.launch_count() - l1 == per_list
        assert ctx.tensor_download(dR2).tobytes() == ref.tobytes()
    ctx.graph_destroy(g)
    ctx.set_option("kernel_timing", "on")
    with pytest.raises(pkg.TcbError):
        ctx.capture_begin()                                     # event pairs cannot live inside a graph
    ctx.set_option("kernel_timing", "off")
    with pytest.raises(pkg.TcbError):
        ctx.capture_end()                                       # nothing open


def test_ccsd_diis_and_residual_norms_follow_the_oracle(ctx):
    """DIIS around the CCSD iteration and the residual norm per evaluation, every tensor
    operation on the device, against oracle cc.ccsd_diis (pinned to the Fock-space projections in tests/test_oracle_cc.py)."""
    o, v = 3, 4
    rng = np.random.default_rng(46)
    n = o + v
    c = lambda *s: rng.standard_normal(s) + 1j * rng.standard_normal(s)
    A = c(n, n, n, n)
    A = A - A.transpose(1, 0, 2, 3)
    A = A - A.transpose(0, 1, 3, 2)
    g = 0.05 * 0.5 * (A + A.transpose(2, 3, 0, 1).conj())
    e = np.concatenate([np.linspace(-2.0, -0.5, o), np.linspace(0.5, 3.0, v)])
    f = 0.05 * c(n, n)
    f = f + f.conj().T
    f[np.diag_indices(n)] = e
    B = cc.ccsd_blocks(o, f, g)
    dB = {k: ctx.tensor_from_numpy(x) for k, x in B.items()}
    its = 10
    dT1, dT2, energies, norms = ccd.ccsd_solve_diis(ctx, dB, e[:o], e[o:], its)
    T1, T2, e_ref, n_ref = cc.ccsd_diis(B, e[:o], e[o:], its)
    assert np.max(np.abs(ctx.tensor_download(dT1) - T1)) <= 1e-10 * np.abs(T1).max()
    assert np.max(np.abs(ctx.tensor_download(dT2) - T2)) <= 1e-10 * np.abs(T2).max()
    for k in range(its):
        assert abs(energies[k] - e_ref[k]) <= 1e-10 * max(abs(e_ref[-1]), 1e-300)
        assert abs(norms[k] - n_ref[k]) <= 1e-10 * n_ref[0]
    assert norms[-1] < 1e-6 * norms[0]                          # it converges; |R| is what the paper's tables quote
    # the CCD Jacobi solver reports its residual norms the same way
    B2, T_mp2, eo, ev = synth.config_ccd(3, 5)
    dB2 = {k: ctx.tensor_from_numpy(x) for k, x in B2.items()}
    got = []
    ccd.ccd_solve(ctx, dB2, eo, ev, 3, norms=got)
    Tr = np.zeros_like(T_mp2)
    for k in range(3):
        R = cc.ccd_residual_program(B2, Tr)
        assert abs(got[k] - cc.residual_norm(R)) <= 1e-11 * cc.residual_norm(cc.ccd_residual_program(B2, np.zeros_like(T_mp2)))
        Tr = cc.denominator_update(Tr, R, [-ev, -ev, eo, eo], 1.0)


def _ccsdt_inputs(o, v, seed, scale=0.3):
    rng = np.random.default_rng(seed)
    n = o + v
    c = lambda *s: rng.standard_normal(s) + 1j * rng.standard_normal(s)
    g = c(n, n, n, n)
    g = g - g.transpose(1, 0, 2, 3)
    g = scale * (g - g.transpose(0, 1, 3, 2))
    f = scale * c(n, n)
    t1 = scale * c(v, o)
    t2 = c(v, v, o, o)
    t2 = t2 - t2.transpose(1, 0, 2, 3)
    t2 = scale * (t2 - t2.transpose(0, 1, 3, 2))
    t3 = 0.1 * cc.antisymmetrise_abc_ijk(c(v, v, v, o, o, o))
    h = f - np.einsum("piqi->pq", g[:, :o, :, :o])
    return f, g, h, t1, t2, t3


@pytest.mark.parametrize("o,v", [(3, 4), (4, 6)])
def test_ccsdt_residual_call_by_call_and_against_the_fock_space_pinned_equations(ctx, o, v):
    """SURVEY 8(f)-3, CCSDT: the driver's 88 library calls (T1 dressing of the integrals, CCD program on the dressed blocks,
    intermediates, seven rank-6 contractions, the 36-term antisymmetriser as a 4-term and a 9-term permute-sum), each compared with the oracle's evaluation of
    the same call under its own carried snorm; the three residuals against cc.ccsdt_residual_unfactorised (pinned to the
    Fock-space projections in tests/test_oracle_cc.py), H general complex and not Hermitian."""
    from gpu_util import ShadowContext
    f, g, h, t1, t2, t3 = _ccsdt_inputs(o, v, 100 * o + v)
    sh = ShadowContext(ctx)
    R1, R2, R3 = ccd.ccsdt_residual(sh, o, sh.wrap(h), sh.wrap(g), sh.wrap(t1), sh.wrap(t2), sh.wrap(t3))
    assert sh.calls == 88 and sh.worst <= 1e-11
    e, r1, r2, r3 = cc.ccsdt_residual_unfactorised(o, f, g, t1, t2, t3)
    for got, ref in ((R1, r1), (R2, r2), (R3, r3)):
        dev = ctx.tensor_download(got.gpu)
        assert np.abs(dev - ref).max() <= 1e-11 * np.abs(got.norm).max()
        assert np.abs(got.host - ref).max() <= 1e-12 * np.abs(got.norm).max()
    gR3 = ctx.tensor_download(R3.gpu)
    assert np.abs(gR3 + gR3.transpose(1, 0, 2, 3, 4, 5)).max() <= 1e-12 * np.abs(R3.norm).max()


@pytest.mark.parametrize("o,v", [(3, 4), (4, 12), (6, 9)])
def test_packed_triples_correction_program(ctx, o, v):
    """(T) on packed storage: R3p, t3p against the pack of the oracle program's dense R3, t3; E[T] and E_ST against the
    oracle's and against the dense driver on the same inputs."""
    from oracle import sym
    n = o + v
    g = synth.tensor(synth.SEED0 + 7, 1, [n] * 4, antisym=((0, 1), (2, 3)), sigma=0.3, hermitian=True)
    rng = np.random.default_rng(o + v)
    t2 = rng.standard_normal((v, v, o, o)) + 1j * rng.standard_normal((v, v, o, o))
    t2 = t2 - t2.transpose(1, 0, 2, 3)
    t2 = np.asfortranarray(t2 - t2.transpose(0, 1, 3, 2))
    t1 = np.asfortranarray(rng.standard_normal((v, o)) + 1j * rng.standard_normal((v, o)))
    eo, ev = np.linspace(-2.0, -0.5, o), np.linspace(0.5, 3.0, v)
    W, U = np.asfortranarray(g[o:, o:, o:, :o]), np.asfortranarray(g[:o, o:, :o, :o])
    oovv = np.asfortranarray(g[:o, :o, o:, o:])
    dW, dU, dT, dT1, dV = (ctx.tensor_from_numpy(x) for x in (W, U, t2, t1, oovv))
    dE, dEst, dR3p, dt3p = ccd.triples_correction_packed(ctx, dW, dU, dT, eo, ev, keep=True, T1=dT1, oovv=dV)
    R3, t3, E = cc.triples_program(W, U, t2, eo, ev)
    _, est_ref = cc.triples_singles_term(t1, oovv, t3)
    assert np.max(np.abs(ctx.tensor_download(dR3p) - sym.pack("P(a<b<c,i<j<k)=R(a,b,c,i,j,k)", R3))) <= 1e-11 * np.abs(R3).max()
    assert np.max(np.abs(ctx.tensor_download(dt3p) - sym.pack("P(a<b<c,i<j<k)=T(a,b,c,i,j,k)", t3))) <= 1e-11 * np.abs(t3).max()
    got, got_st = complex(ctx.tensor_download(dE)), complex(ctx.tensor_download(dEst))
    assert abs(got - E) <= 1e-11 * abs(E) and got.real < 0
    assert abs(got_st - est_ref) <= 1e-11 * abs(est_ref)
    eE, eEst = ccd.triples_correction(ctx, dW, dU, dT, eo, ev, T1=dT1, oovv=dV)
    assert abs(got - complex(ctx.tensor_download(eE))) <= 1e-11 * abs(E)
    assert abs(got_st - complex(ctx.tensor_download(eEst))) <= 1e-11 * abs(est_ref)
    with pytest.raises(ValueError):
        ccd.triples_correction_packed(ctx, dW, dU, ctx.tensor_create((v, v, 2, 2)), eo, ev)
    for t in (dW, dU, dT, dT1, dV, dE, dEst, dR3p, dt3p, eE, eEst):
        t.destroy()


@pytest.mark.parametrize("o,v", [(3, 4), (4, 6), (5, 5)])
def test_packed_ccsdt_residual_call_by_call_and_against_the_fock_space_pinned_equations(ctx, o, v):
    """SURVEY 8(f)-2 applied to 8(f)-3: ccd.ccsdt_residual_packed -- T3 and R3 only as (a<b<c, i<j<k) packed tensors, every
    contraction with T3 on packed views -- call by call against the oracle (tcb_pack bit-exact; packed views, contractions
    and tcb_antisym_pack under their carried snorm), the residuals against the unfactorised equations, and against the dense
    driver."""
    from gpu_util import ShadowContext
    from oracle import sym
    f, g, h, t1, t2, t3 = _ccsdt_inputs(o, v, 100 * o + v)
    t3p = sym.pack("P(a<b<c,i<j<k)=T(a,b,c,i,j,k)", t3)
    sh = ShadowContext(ctx)
    R1, R2, R3p = ccd.ccsdt_residual_packed(sh, o, sh.wrap(h), sh.wrap(g), sh.wrap(t1), sh.wrap(t2), sh.wrap(t3p))
    assert sh.calls == 109 and sh.worst <= 1e-11
    e, r1, r2, r3 = cc.ccsdt_residual_unfactorised(o, f, g, t1, t2, t3)
    W = ctx.tensor_from_numpy
    D1, D2, D3 = ccd.ccsdt_residual(ctx, o, W(h), W(g), W(t1), W(t2), W(t3))
    R3 = ctx.tensor_create((v, v, v, o, o, o), zero=False)
    ctx.unpack("R(a,b,c,i,j,k)=P(a<b<c,i<j<k)", R3, R3p.gpu, 1.0)
    scale3 = np.abs(R3p.norm).max()
    for got, scale, ref, dense in ((R1.gpu, np.abs(R1.norm).max(), r1, D1), (R2.gpu, np.abs(R2.norm).max(), r2, D2), (R3, scale3, r3, D3)):
        dev = ctx.tensor_download(got)
        assert np.abs(dev - ref).max() <= 1e-11 * scale
        assert np.abs(dev - ctx.tensor_download(dense)).max() <= 1e-11 * scale
    assert np.abs(R3p.host - sym.pack("P(a<b<c,i<j<k)=R(a,b,c,i,j,k)", r3)).max() <= 1e-12 * scale3


@pytest.mark.parametrize("packed", [False, True])
def test_ccsdt_iterations_follow_the_oracle_and_converge(ctx, packed):
    o, v = 3, 3
    rng = np.random.default_rng(52)
    n = o + v
    c = lambda *s: rng.standard_normal(s) + 1j * rng.standard_normal(s)
    A = c(n, n, n, n)
    A = A - A.transpose(1, 0, 2, 3)
    A = A - A.transpose(0, 1, 3, 2)
    g = 0.05 * 0.5 * (A + A.transpose(2, 3, 0, 1).conj())
    e = np.concatenate([np.linspace(-2.0, -0.5, o), np.linspace(0.5, 3.0, v)])
    f = 0.05 * c(n, n)
    f = f + f.conj().T
    f[np.diag_indices(n)] = e
    h = f - np.einsum("piqi->pq", g[:, :o, :, :o])
    its = 12
    dh, dg = ctx.tensor_from_numpy(h), ctx.tensor_from_numpy(g)
    T1, T2, T3, energies, norms = ccd.ccsdt_solve(ctx, o, dh, dg, e, its, packed=packed)
    r1, r2, r3, e_ref, n_ref = cc.ccsdt_jacobi(o, f, g, its)
    if packed:
        T3p, T3 = T3, ctx.tensor_create((v, v, v, o, o, o), zero=False)
        ctx.unpack("T(a,b,c,i,j,k)=P(a<b<c,i<j<k)", T3, T3p, 1.0)
    for got, ref in ((T1, r1), (T2, r2), (T3, r3)):
        assert np.abs(ctx.tensor_download(got) - ref).max() <= 1e-10 * max(np.abs(ref).max(), 1e-300)
    for k in range(its):
        assert abs(energies[k] - e_ref[k]) <= 1e-10 * abs(e_ref[-1]) and abs(norms[k] - n_ref[k]) <= 1e-10 * n_ref[0]
    assert norms[-1] < 1e-4 * norms[0]


@pytest.mark.parametrize("packed", [False, True])
def test_ccsdt_diis_follows_the_oracle_and_converges(ctx, packed):
    """DIIS over (t1, t2, t3) around the CCSDT residual, dense and with t3 / R3 / the t3 history packed (inner products
    weighted by 36): amplitudes, energies and residual norms of every evaluation against cc.ccsdt_diis."""
    o, v = 3, 3
    rng = np.random.default_rng(52)
    n = o + v
    c = lambda *s: rng.standard_normal(s) + 1j * rng.standard_normal(s)
    A = c(n, n, n, n)
    A = A - A.transpose(1, 0, 2, 3)
    A = A - A.transpose(0, 1, 3, 2)
    g = 0.05 * 0.5 * (A + A.transpose(2, 3, 0, 1).conj())
    e = np.concatenate([np.linspace(-2.0, -0.5, o), np.linspace(0.5, 3.0, v)])
    f = 0.05 * c(n, n)
    f = f + f.conj().T
    f[np.diag_indices(n)] = e
    h = f - np.einsum("piqi->pq", g[:, :o, :, :o])
    its = 9
    dh, dg = ctx.tensor_from_numpy(h), ctx.tensor_from_numpy(g)
    T1, T2, T3, energies, norms = ccd.ccsdt_solve_diis(ctx, o, dh, dg, e, its, packed=packed)
    r1, r2, r3, e_ref, n_ref = cc.ccsdt_diis(o, f, g, its)
    if packed:
        T3p, T3 = T3, ctx.tensor_create((v, v, v, o, o, o), zero=False)
        ctx.unpack("T(a,b,c,i,j,k)=P(a<b<c,i<j<k)", T3, T3p, 1.0)
    for got, ref in ((T1, r1), (T2, r2), (T3, r3)):
        assert np.abs(ctx.tensor_download(got) - ref).max() <= 1e-9 * max(np.abs(ref).max(), 1e-300)
    for k in range(its):
        assert abs(energies[k] - e_ref[k]) <= 1e-9 * abs(e_ref[-1]) and abs(norms[k] - n_ref[k]) <= 1e-9 * n_ref[0]
    assert norms[-1] < 1e-5 * norms[0]
