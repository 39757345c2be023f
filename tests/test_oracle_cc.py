"""Pins for oracle/cc.py.  Tier 0 evaluates PAPER Eqs. (2)-(4) literally on
the Fock space; the spin-orbital CCD equations (tier 1a) and the factorised binary program (tier 1b,
config 2) must reproduce it for complex, non-diagonal, Hermitian-consistent inputs."""
import numpy as np
import pytest

import oracle
from oracle import cc


def rand_inputs(o, v, seed):
    rng = np.random.default_rng(seed)
    n = o + v
    c = lambda *s: rng.standard_normal(s) + 1j * rng.standard_normal(s)
    A = c(n, n, n, n)
    A = A - A.transpose(1, 0, 2, 3)
    A = A - A.transpose(0, 1, 3, 2)
    g = 0.5 * (A + A.transpose(2, 3, 0, 1).conj())
    f = c(n, n)
    f = f + f.conj().T                         # general (non-diagonal) Hermitian Fock matrix
    t = c(v, v, o, o)
    t = t - t.transpose(1, 0, 2, 3)
    t = t - t.transpose(0, 1, 3, 2)
    return f, g, t


def test_jordan_wigner_anticommutators():
    a = cc.jordan_wigner(4)
    for p in range(4):
        for q in range(4):
            assert np.array_equal(a[p] @ a[q].T + a[q].T @ a[p], np.eye(16) * (p == q))
            assert not np.any(a[p] @ a[q] + a[q] @ a[p])


@pytest.mark.parametrize("o,v", [(2, 3), (3, 3), (2, 4)])
def test_ccd_tiers_agree_with_fock_space(o, v):
    f, g, t = rand_inputs(o, v, 100 * o + v)
    e0, _, r0 = cc.fock_space_residuals(o, v, f, g, t)
    r1a, e1a, n_amp, n_en = cc.ccd_residual_unfactorised(o, f, g, t)
    assert n_amp + n_en == 11                                   # PAPER Table I: CCD = 11 diagrams
    scale = np.abs(r0).max()
    assert np.abs(r1a - r0).max() <= 1e-13 * scale
    assert abs(e1a - e0) <= 1e-13 * abs(e0)
    r1b = cc.ccd_residual_program(cc.blocks(o, f, g), np.asfortranarray(t))
    assert np.abs(r1b - r1a).max() <= 1e-13 * scale
    # residual antisymmetry R(a,b,i,j) = -R(b,a,i,j) = -R(a,b,j,i)
    assert np.abs(r1b + r1b.transpose(1, 0, 2, 3)).max() <= 1e-13 * scale
    assert np.abs(r1b + r1b.transpose(0, 1, 3, 2)).max() <= 1e-13 * scale


def test_mp2_guess_cancels_driver_and_fock_terms_and_energy_closed_form():
    o, v = 3, 4
    _, g, _ = rand_inputs(o, v, 9)
    rng = np.random.default_rng(10)
    eo, ev = -2 + 1.5 * rng.random(o), 0.5 + 2.5 * rng.random(v)
    f = np.diag(np.concatenate([eo, ev])).astype(np.complex128)
    den = eo[None, None, :, None] + eo[None, None, None, :] - ev[:, None, None, None] - ev[None, :, None, None]
    vvoo = g[o:, o:, :o, :o]
    t = vvoo / den
    # linear-in-f part of the residual + driver vanishes:  <ab||ij> + (e_a+e_b-e_i-e_j) t = 0
    gz = np.zeros_like(g)
    gz[o:, o:, :o, :o] = vvoo
    r, e, _, _ = cc.ccd_residual_unfactorised(o, f, gz, t)
    assert np.abs(r).max() <= 1e-14 * np.abs(vvoo).max()
    # MP2 energy: 1/4 sum <ij||ab> t = 1/4 sum |<ab||ij>|^2 / den : real and negative
    _, e, _, _ = cc.ccd_residual_unfactorised(o, f, g, t)
    closed = 0.25 * np.sum(np.abs(vvoo) ** 2 / den)
    assert abs(e - closed) <= 1e-13 * abs(closed) and closed < 0 and abs(e.imag) <= 1e-14 * abs(closed)


def test_t3_term_against_fock_space_triples_projection():
    """<Phi_ijk^abc| [H, T2] |Phi0> = P(k/ij)P(a/bc) sum_d <bc||dk> t_ij^ad - P(i/jk)P(c/ab) sum_l <lc||jk> t_il^ab."""
    o = v = 3
    f, g, t = rand_inputs(o, v, 7)
    fs = cc.FockSpace(o, v)
    psi = fs.apply_H(f, g, fs.apply_T(None, t, fs.phi0)) - fs.apply_T(None, t, fs.apply_H(f, g, fs.phi0))
    R3 = fs.project_triples(psi)
    W = g[o:, o:, o:, :o]
    X, Y = cc.t3_term_unfactorised(W, t)
    Z = np.einsum("lcjk,abil->abcijk", g[:o, o:, :o, :o], t)
    Z = Z - np.swapaxes(Z, 2, 0) - np.swapaxes(Z, 2, 1)
    Z = Z - np.swapaxes(Z, 3, 4) - np.swapaxes(Z, 3, 5)
    assert np.abs(R3 - (Y - Z)).max() <= 1e-13 * np.abs(R3).max()
    # the library-call form (one contraction + one 9-term permute-sum) reproduces the particle part
    Xp, R3p = cc.t3_term_program(np.asfortranarray(W), np.asfortranarray(t), np.zeros_like(X))
    assert np.abs(Xp - X).max() <= 1e-13 * np.abs(X).max()
    assert np.abs(R3p - Y).max() <= 1e-13 * np.abs(Y).max()


def _ccd_problem(o, v):
    """config_ccd blocks plus the full f and g they were cut from (the generator is keyed by global spinor labels)"""
    from paper_2409_06759_b200 import synth
    B, T_mp2, eo, ev = synth.config_ccd(o, v)
    n = o + v
    f = np.zeros((n, n), dtype=np.complex128)
    f[:o, :o], f[o:, o:] = B["foo"], B["fvv"]
    g = synth.tensor(synth.SEED0 + 2, 1, [n] * 4, antisym=((0, 1), (2, 3)), sigma=0.1, hermitian=True)
    return B, T_mp2, eo, ev, f, g


def test_jacobi_first_step_from_zero_is_the_mp2_closed_form():
    """T = 0: R = <ab||ij>, so one step gives t = <ab||ij> / (e_i + e_j - e_a - e_b) -- the generator's own MP2
    amplitudes, written there from the closed form -- and E = 1/4 sum |<ab||ij>|^2 / (e_i + e_j - e_a - e_b) < 0."""
    B, T_mp2, eo, ev, f, g = _ccd_problem(3, 4)
    T, energies = cc.ccd_jacobi(B, eo, ev, 1)
    assert np.abs(T - T_mp2).max() <= 1e-14 * np.abs(T_mp2).max()
    d = eo[None, None, :, None] + eo[None, None, None, :] - ev[:, None, None, None] - ev[None, :, None, None]
    e_closed = 0.25 * np.sum(np.abs(B["vvoo"]) ** 2 / d)
    assert e_closed < 0 and abs(energies[0] - e_closed) <= 1e-13 * abs(e_closed)
    assert abs(energies[0].imag) <= 1e-15 * abs(e_closed)


def test_denominator_update_closed_form_and_skipped_indices():
    rng = np.random.default_rng(5)
    T = np.asfortranarray(rng.standard_normal((3, 4, 2)) + 1j * rng.standard_normal((3, 4, 2)))
    R = np.asfortranarray(rng.standard_normal((3, 4, 2)) + 1j * rng.standard_normal((3, 4, 2)))
    e0, e2 = rng.uniform(1, 2, 3), rng.uniform(1, 2, 2)
    got = cc.denominator_update(T, R, [e0, None, e2], 0.5 - 2j)
    for i in range(3):
        for j in range(4):
            for k in range(2):
                assert abs(got[i, j, k] - (T[i, j, k] + (0.5 - 2j) * R[i, j, k] / (e0[i] + e2[k]))) <= 1e-15 * 8


@pytest.mark.parametrize("o,v", [(2, 3), (3, 3)])
def test_converged_jacobi_amplitudes_zero_the_fock_space_projection(o, v):
    """The fixed point of the iteration solves PAPER Eq. (3): <Phi_ij^ab| exp(-T) H exp(T) |Phi0> = 0, evaluated on the
    Fock space (tier 0) -- which shares nothing with the factorised program the iteration runs on -- and the energy of
    the last step is the tier-0 <Phi0| exp(-T) H exp(T) |Phi0> - <Phi0|H|Phi0>."""
    B, T_mp2, eo, ev, f, g = _ccd_problem(o, v)
    T, energies = cc.ccd_jacobi(B, eo, ev, 40)
    e0, _, r0 = cc.fock_space_residuals(o, v, f, g, T)
    assert np.abs(r0).max() <= 1e-12 * np.abs(B["vvoo"]).max()
    assert abs(energies[-1] - e0) <= 1e-12 * abs(e0)
    assert abs(energies[-1] - energies[-2]) <= 1e-13 * abs(e0)
    assert np.abs(T - T_mp2).max() > 1e-3 * np.abs(T_mp2).max()          # it did move away from the MP2 guess


@pytest.mark.parametrize("o,v", [(2, 3), (3, 3), (2, 4)])
def test_ccsd_unfactorised_agrees_with_fock_space(o, v):
    """The textbook CCSD intermediates, in residual form with a general complex non-diagonal Hermitian f, against
    PAPER Eq. (3) on the Fock space: singles and doubles projections and the energy."""
    f, g, t2 = rand_inputs(o, v, 300 * o + v)
    rng = np.random.default_rng(7 * o + v)
    t1 = rng.standard_normal((v, o)) + 1j * rng.standard_normal((v, o))
    t2, t1 = 0.3 * t2, 0.3 * t1
    e0, r1_0, r2_0 = cc.fock_space_residuals(o, v, f, g, t2, t1)
    e, r1, r2 = cc.ccsd_residual_unfactorised(o, f, g, t1, t2)
    assert abs(e - e0) <= 1e-13 * abs(e0)
    assert np.abs(r1 - r1_0).max() <= 1e-13 * np.abs(r1_0).max()
    assert np.abs(r2 - r2_0).max() <= 1e-13 * np.abs(r2_0).max()
    # t1 = 0 reduces to CCD
    e_d, r1_d, r2_d = cc.ccsd_residual_unfactorised(o, f, g, 0 * t1, t2)
    assert np.abs(r2_d - cc.ccd_residual_unfactorised(o, f, g, t2)[0]).max() <= 1e-13 * np.abs(r2_d).max()


@pytest.mark.parametrize("o,v", [(2, 3), (3, 4), (4, 5)])
def test_ccsd_driver_with_the_packed_pp_ladder_equals_the_unfactorised_tier(o, v):
    """ccd.ccsd_residual(packed={}): W_abef only as Wp(a<b, e<f), P(ab) as antisym_pack, the ladder at 1/8 of the flops --
    run on the host through the oracle's primitives (tests/oracle_ctx.py) against the Fock-space-pinned direct sums, and
    against the same driver with the dense ladder."""
    from oracle_ctx import OracleContext
    from paper_2409_06759_b200 import ccd
    f, g, t2 = rand_inputs(o, v, 500 * o + v)
    rng = np.random.default_rng(11 * o + v)
    t1 = np.asfortranarray(0.3 * (rng.standard_normal((v, o)) + 1j * rng.standard_normal((v, o))))
    t2 = np.asfortranarray(0.3 * t2)
    e, r1, r2 = cc.ccsd_residual_unfactorised(o, f, g, t1, t2)
    out = {}
    for mode in ("dense", "packed"):
        oc = OracleContext()
        B = {k: oc.tensor_from_numpy(x) for k, x in cc.ccsd_blocks(o, f, g).items()}
        cache = {} if mode == "packed" else None
        E, R1, R2 = ccd.ccsd_residual(oc, B, oc.tensor_from_numpy(t1), oc.tensor_from_numpy(t2), packed=cache)
        assert abs(E.host.ravel()[0] - e) <= 1e-13 * abs(e)
        assert np.abs(R1.host - r1).max() <= 1e-13 * np.abs(r1).max()
        assert np.abs(R2.host - r2).max() <= 1e-13 * np.abs(r2).max()
        out[mode] = (oc.calls, cache)
    assert out["dense"][0] == 55 and out["packed"][0] == 55 + 4      # 2 packs (once per solve), pack tau, unpack Rp
    assert sorted(out["packed"][1]) == ["vovv", "vvvv"]


@pytest.mark.parametrize("o,v", [(2, 3), (3, 4)])
def test_ccsd_program_of_binary_operations_agrees_with_the_unfactorised_tier(o, v):
    f, g, t2 = rand_inputs(o, v, 500 * o + v)
    rng = np.random.default_rng(11 * o + v)
    t1 = np.asfortranarray(0.3 * (rng.standard_normal((v, o)) + 1j * rng.standard_normal((v, o))))
    t2 = np.asfortranarray(0.3 * t2)
    e, r1, r2 = cc.ccsd_residual_unfactorised(o, f, g, t1, t2)
    ep, r1p, r2p = cc.ccsd_residual_program(cc.ccsd_blocks(o, f, g), t1, t2)
    assert abs(ep - e) <= 1e-13 * abs(e)
    assert np.abs(r1p - r1).max() <= 1e-13 * np.abs(r1).max()
    assert np.abs(r2p - r2).max() <= 1e-13 * np.abs(r2).max()
    assert np.abs(r2p + r2p.transpose(1, 0, 2, 3)).max() <= 1e-13 * np.abs(r2).max()
    assert np.abs(r2p + r2p.transpose(0, 1, 3, 2)).max() <= 1e-13 * np.abs(r2).max()


def _ccsd_problem(o, v, seed):
    """weakly coupled Hermitian problem with a non-zero occupied-virtual Fock block (so that t1 does not vanish)"""
    rng = np.random.default_rng(seed)
    n = o + v
    c = lambda *s: rng.standard_normal(s) + 1j * rng.standard_normal(s)
    A = c(n, n, n, n)
    A = A - A.transpose(1, 0, 2, 3)
    A = A - A.transpose(0, 1, 3, 2)
    g = 0.05 * 0.5 * (A + A.transpose(2, 3, 0, 1).conj())
    f = 0.05 * c(n, n)
    e = np.concatenate([np.linspace(-2.0, -0.5, o), np.linspace(0.5, 3.0, v)])
    f = f + f.conj().T
    f[np.diag_indices(n)] = e
    return f, g, e[:o], e[o:]


@pytest.mark.parametrize("o,v", [(2, 3), (3, 3)])
def test_converged_ccsd_jacobi_zeroes_the_fock_space_singles_and_doubles(o, v):
    f, g, eo, ev = _ccsd_problem(o, v, 40 + o + v)
    T1, T2, energies = cc.ccsd_jacobi(cc.ccsd_blocks(o, f, g), eo, ev, 60)
    e0, r1, r2 = cc.fock_space_residuals(o, v, f, g, T2, T1)
    scale = np.abs(g).max()
    assert np.abs(r1).max() <= 1e-12 * scale and np.abs(r2).max() <= 1e-12 * scale
    assert abs(energies[-1] - e0) <= 1e-12 * abs(e0)
    assert np.abs(T1).max() > 1e-3 and np.abs(T2).max() > 1e-3


def test_diis_reaches_the_same_fixed_point_in_fewer_steps():
    """DIIS changes the path, not the solution: its amplitudes zero the Fock-space projection as well, the error vector of
    the 6th DIIS step is far below that of the 6th Jacobi step, and the coefficients sum to one."""
    o, v = 3, 3
    B, T_mp2, eo, ev, f, g = _ccd_problem(o, v)
    T, energies, norms = cc.ccd_diis(B, eo, ev, 14)
    e0, _, r0 = cc.fock_space_residuals(o, v, f, g, T)
    assert np.abs(r0).max() <= 1e-12 * np.abs(B["vvoo"]).max()
    assert abs(energies[-1] - e0) <= 1e-12 * abs(e0)
    Tj, _ = cc.ccd_jacobi(B, eo, ev, 5)
    rj = cc.ccd_residual_program(B, Tj)
    d = eo[None, None, :, None] + eo[None, None, None, :] - ev[:, None, None, None] - ev[None, :, None, None]
    assert norms[5] < 0.1 * np.linalg.norm(rj / d)
    assert abs(norms[0] - np.linalg.norm(B["vvoo"] / d)) <= 1e-13 * norms[0]      # first error vector = MP2 amplitudes
    Bm = np.array([[2.0, 0.5j], [-0.5j, 1.0]])
    c = cc.diis_coefficients(Bm)
    assert abs(c.sum() - 1) <= 1e-15
    # the constrained minimum: any other c' with sum 1 gives a larger c'^H B c'
    best = np.vdot(c, Bm @ c).real
    for t in (-0.3, 0.2, 0.7, 1.4):
        cp = np.array([t, 1 - t])
        assert np.vdot(cp, Bm @ cp).real >= best - 1e-15


def test_triples_correction_against_the_fock_space_and_unique_triples():
    """R3 of the [T] correction is the tier-0 projection <Phi_ijk^abc|[H,T2]|Phi0>; the energy's 1/36 is checked by
    summing |R3|^2 / D3 over unique triples a<b<c, i<j<k; the program of library calls reproduces both."""
    o = v = 3
    f, g, t = rand_inputs(o, v, 21)
    eo, ev = np.linspace(-2.0, -0.5, o), np.linspace(0.5, 3.0, v)
    fs = cc.FockSpace(o, v)
    psi = fs.apply_H(f, g, fs.apply_T(None, t, fs.phi0)) - fs.apply_T(None, t, fs.apply_H(f, g, fs.phi0))
    R3_0 = fs.project_triples(psi)
    R3, E = cc.triples_unfactorised(o, g, t, eo, ev)
    assert np.abs(R3 - R3_0).max() <= 1e-13 * np.abs(R3_0).max()
    e_unique = 0.0
    for a in range(v):
        for b in range(a + 1, v):
            for c in range(b + 1, v):
                for i in range(o):
                    for j in range(i + 1, o):
                        for k in range(j + 1, o):
                            e_unique += abs(R3_0[a, b, c, i, j, k]) ** 2 / (eo[i] + eo[j] + eo[k] - ev[a] - ev[b] - ev[c])
    assert e_unique < 0 and abs(E - e_unique) <= 1e-13 * abs(e_unique) and abs(E.imag) <= 1e-15 * abs(e_unique)
    W = np.asfortranarray(g[o:, o:, o:, :o])
    U = np.asfortranarray(g[:o, o:, :o, :o])
    R3p, t3p, Ep = cc.triples_program(W, U, np.asfortranarray(t), eo, ev)
    assert np.abs(R3p - R3).max() <= 1e-13 * np.abs(R3).max()
    assert abs(Ep - E) <= 1e-13 * abs(E)
    # antisymmetry of the triples amplitudes in (a,b,c) and (i,j,k)
    assert np.abs(t3p + t3p.transpose(1, 0, 2, 3, 4, 5)).max() <= 1e-13 * np.abs(t3p).max()
    assert np.abs(t3p + t3p.transpose(0, 1, 2, 3, 5, 4)).max() <= 1e-13 * np.abs(t3p).max()


@pytest.mark.parametrize("o,v", [(3, 3), (3, 4), (4, 5)])
def test_packed_triples_correction_driver_equals_the_unfactorised_sums(o, v):
    """ccd.triples_correction_packed (R3, t3 only on a<b<c, i<j<k; contractions at 1/4 of the flops; tcb_antisym_pack for both
    9-term operators; no factor 1/36) run on the host through the oracle's primitives: R3p is the pack of the direct sums,
    E[T] and the singles term E_ST are those of the dense oracle programs (pinned above and below to the Fock space)."""
    from oracle import sym
    from oracle_ctx import OracleContext
    from paper_2409_06759_b200 import ccd
    f, g, t2 = rand_inputs(o, v, 50 + o + v)
    t2 = np.asfortranarray(t2)
    eo, ev = np.linspace(-2.0, -0.5, o), np.linspace(0.5, 3.0, v)
    rng = np.random.default_rng(o * v)
    t1 = np.asfortranarray(rng.standard_normal((v, o)) + 1j * rng.standard_normal((v, o)))
    W, U = np.asfortranarray(g[o:, o:, o:, :o]), np.asfortranarray(g[:o, o:, :o, :o])
    oovv = np.asfortranarray(g[:o, :o, o:, o:])
    oc = OracleContext()
    Wr = oc.tensor_from_numpy
    E, Est, R3p, t3p = ccd.triples_correction_packed(oc, Wr(W), Wr(U), Wr(t2), eo, ev, keep=True, T1=Wr(t1), oovv=Wr(oovv))
    R3u, Eu = cc.triples_unfactorised(o, g, t2, eo, ev)
    _, t3, _ = cc.triples_program(W, U, t2, eo, ev)
    _, est_ref = cc.triples_singles_term(t1, oovv, t3)
    assert np.abs(R3p.host - sym.pack("P(a<b<c,i<j<k)=R(a,b,c,i,j,k)", R3u)).max() <= 1e-13 * np.abs(R3u).max()
    assert np.abs(t3p.host - sym.pack("P(a<b<c,i<j<k)=T(a,b,c,i,j,k)", t3)).max() <= 1e-13 * np.abs(t3).max()
    assert abs(E.host.ravel()[0] - Eu) <= 1e-13 * abs(Eu)
    assert abs(Est.host.ravel()[0] - est_ref) <= 1e-13 * abs(est_ref)
    assert oc.calls == 14


def test_triples_singles_term_against_the_fock_space_matrix_element():
    """E_ST = <T1 Phi0| H |T3 Phi0> on the Fock space (T3 from PAPER Eq. 2) against 1/4 sum conj(t1) <jk||bc> t3."""
    o = v = 3
    f, g, t2 = rand_inputs(o, v, 33)
    eo, ev = np.linspace(-2.0, -0.5, o), np.linspace(0.5, 3.0, v)
    rng = np.random.default_rng(3)
    t1 = np.asfortranarray(rng.standard_normal((v, o)) + 1j * rng.standard_normal((v, o)))
    W, U = np.asfortranarray(g[o:, o:, o:, :o]), np.asfortranarray(g[:o, o:, :o, :o])
    _, t3, _ = cc.triples_program(W, U, np.asfortranarray(t2), eo, ev)
    fs = cc.FockSpace(o, v)
    e0 = np.vdot(fs.apply_T(t1, None, fs.phi0), fs.apply_H(f, g, fs.apply_T3(t3, fs.phi0)))
    Y, e = cc.triples_singles_term(t1, cc.block(o, g, "oovv"), t3)
    assert abs(e - e0) <= 1e-13 * abs(e0)
    assert abs(e - 0.25 * np.einsum("ai,jkbc,abcijk->", t1.conj(), g[:o, :o, o:, o:], t3)) <= 1e-13 * abs(e0)
    # T3 Phi0 has the right norm: 1/36 of the sum over all index tuples = sum over unique triples
    assert abs(np.vdot(fs.apply_T3(t3, fs.phi0), fs.apply_T3(t3, fs.phi0)) - np.sum(np.abs(t3) ** 2) / 36.0) <= 1e-13 * np.sum(np.abs(t3) ** 2)


def test_ccsd_diis_fixed_point_is_the_fock_space_solution_and_residual_norm_is_the_vector_norm():
    """DIIS around the CCSD iteration (combined t1, t2 error vector): the amplitudes it converges to zero the Fock-space
    singles and doubles projections of e^-T H e^T (PAPER Eq. 3) -- the same fixed point as the Jacobi iteration, reached in
    fewer evaluations; the residual norm it reports is the 2-norm of the Fock-space projections at the
    amplitudes of that evaluation, and its first value is that of the bare driver terms (f_ai, <ab||ij>)."""
    o, v = 3, 3
    f, g, eo, ev = _ccsd_problem(o, v, 46)
    B = cc.ccsd_blocks(o, f, g)
    T1, T2, energies, norms = cc.ccsd_diis(B, eo, ev, 16)
    e0, r1, r2 = cc.fock_space_residuals(o, v, f, g, T2, T1)
    scale = np.abs(g).max()
    assert np.abs(r1).max() <= 1e-12 * scale and np.abs(r2).max() <= 1e-12 * scale
    # energies[k] belongs to the amplitudes evaluation k saw: one more evaluation at the converged amplitudes gives e0
    e_last, r1p, r2p = cc.ccsd_residual_program(B, T1, T2)
    assert abs(e_last - e0) <= 1e-12 * abs(e0)
    assert abs(cc.residual_norm(r1p, r2p) - np.sqrt(np.sum(np.abs(r1) ** 2) + np.sum(np.abs(r2) ** 2))) <= 1e-13 * scale
    assert abs(norms[0] - np.sqrt(np.sum(np.abs(B["fvo"]) ** 2) + np.sum(np.abs(B["vvoo"]) ** 2))) <= 1e-14 * norms[0]
    assert energies[0] == 0
    # fewer evaluations than Jacobi: after 8 evaluations the DIIS residual norm is far below the Jacobi one
    Tj1, Tj2, _ = cc.ccsd_jacobi(B, eo, ev, 7)
    _, j1, j2 = cc.ccsd_residual_program(B, Tj1, Tj2)
    assert norms[7] < 0.1 * cc.residual_norm(j1, j2)
    assert all(norms[k + 1] < norms[k] for k in range(8))


def _ccsdt_problem(o, v, seed, hermitian=False, scale=0.3):
    rng = np.random.default_rng(seed)
    n = o + v
    c = lambda *s: rng.standard_normal(s) + 1j * rng.standard_normal(s)
    g = c(n, n, n, n)
    g = g - g.transpose(1, 0, 2, 3)
    g = scale * (g - g.transpose(0, 1, 3, 2))
    f = scale * c(n, n)
    if hermitian:
        g = 0.5 * (g + g.transpose(2, 3, 0, 1).conj())
        f = 0.5 * (f + f.conj().T)
    t1 = scale * c(v, o)
    t2 = c(v, v, o, o)
    t2 = t2 - t2.transpose(1, 0, 2, 3)
    t2 = scale * (t2 - t2.transpose(0, 1, 3, 2))
    t3 = 0.1 * cc.antisymmetrise_abc_ijk(c(v, v, v, o, o, o))
    return f, g, t1, t2, t3


def _fock_ccsdt(o, v, f, g, t1, t2, t3):
    """exp(-T) H exp(T) |Phi0> with T = T1 + T2 + T3 on the Fock space: E, singles, doubles, triples projections"""
    fs = cc.FockSpace(o, v)

    def exp_t(psi, sign):
        out, term = psi.copy(), psi.copy()
        for k in range(1, o + v + 2):
            term = sign * (fs.apply_T(t1, t2, term) + fs.apply_T3(t3, term)) / k
            if not np.any(term):
                break
            out = out + term
        return out
    psi = exp_t(fs.apply_H(f, g, exp_t(fs.phi0, 1.0)), -1.0)
    e = np.vdot(fs.phi0, psi) - np.vdot(fs.phi0, fs.apply_H(f, g, fs.phi0))
    return e, fs.project_singles(psi), fs.project_doubles(psi), fs.project_triples(psi), fs


def test_t1_dressing_is_the_similarity_transformation_on_the_fock_space():
    """H~ built from dress_t1's integrals IS exp(-T1) H exp(T1) as an operator: applied to a random Fock-space vector"""
    o, v = 2, 3
    f, g, t1, _, _ = _ccsdt_problem(o, v, 5)
    ft, gt = cc.dress_t1(o, f, g, t1)
    fs = cc.FockSpace(o, v)
    rng = np.random.default_rng(1)
    psi = rng.standard_normal(2 ** (o + v)) + 1j * rng.standard_normal(2 ** (o + v))
    lhs = fs.exp_T(t1, None, fs.apply_H(f, g, fs.exp_T(t1, None, psi)), sign=-1.0)
    rhs = fs.apply_H(ft, gt, psi)
    assert np.abs(lhs - rhs).max() <= 1e-12 * np.abs(lhs).max()
    ft0, gt0 = cc.dress_t1(o, f, g, np.zeros_like(t1))
    assert np.array_equal(gt0, g) and np.abs(ft0 - f).max() <= 1e-15


@pytest.mark.parametrize("o,v,hermitian", [(3, 4, False), (4, 4, False), (3, 5, True)])
def test_ccsdt_residuals_equal_the_fock_space_projections(o, v, hermitian):
    """CCSDT: 5 + 13 + 19 terms against Eq. (3) evaluated literally, random complex t1, t2, t3, H general (non-Hermitian: the
    T1-dressed integrals are not Hermitian either) -- a dropped term, a wrong sign, factor or index placement in any of the
    three equations fails this (sizes beyond o = 3 matter: at o = 3 the occupied part of T3 is one-dimensional)"""
    f, g, t1, t2, t3 = _ccsdt_problem(o, v, 10 * o + v, hermitian)
    e0, s0, d0, t0, _ = _fock_ccsdt(o, v, f, g, t1, t2, t3)
    e, r1, r2, r3 = cc.ccsdt_residual_unfactorised(o, f, g, t1, t2, t3)
    assert abs(e - e0) <= 1e-12 * abs(e0)
    for got, ref in ((r1, s0), (r2, d0), (r3, t0)):
        assert np.abs(got - ref).max() <= 1e-12 * np.abs(ref).max()
    assert len(cc.CCSDT_R3_TERMS) == 19
    # each of the 19 triples terms matters: dropping any one changes R3 by far more than the tolerance (from o = v = 4 on:
    # with three occupied spinors some topologies vanish under the antisymmetriser)
    amps = {"t2": t2, "t3": t3}
    ft, gt = cc.dress_t1(o, f, g, t1)
    for cf, which, types, spec, ts in (cc.CCSDT_R3_TERMS if min(o, v) >= 4 else []):
        x = cf * np.einsum(spec, cc._blk(o, ft if which == "f" else gt, types), *[amps[t] for t in ts])
        assert np.abs(cc.antisymmetrise_abc_ijk(x)).max() >= 1e-6 * np.abs(t0).max(), spec
    # t3 = 0, t1 = 0: the doubles equation is the CCD tier, the triples equation the (T) driver terms
    e_, r1_, r2_, r3_ = cc.ccsdt_residual_unfactorised(o, f, g, 0 * t1, t2, 0 * t3)
    assert np.abs(r2_ - cc.ccd_residual_unfactorised(o, f, g, t2)[0]).max() <= 1e-13 * np.abs(r2_).max()


def test_ccsdt_driver_call_list_is_the_unfactorised_equations():
    """The product's CCSDT driver (ccd.ccsdt_residual: T1 dressing by binary contractions, intermediates, seven rank-6
    contractions into one X, the antisymmetriser in two passes) run on the host with every tensor operation done by the oracle:
    its result is the unfactorised 37-term evaluation (pinned above to the Fock space)."""
    from oracle_ctx import OracleContext
    from paper_2409_06759_b200 import ccd
    o, v = 3, 4
    f, g, t1, t2, t3 = _ccsdt_problem(o, v, 77)
    h = f - np.einsum("piqi->pq", g[:, :o, :, :o])
    oc = OracleContext()
    W = oc.tensor_from_numpy
    R1, R2, R3 = ccd.ccsdt_residual(oc, o, W(h), W(g), W(t1), W(t2), W(t3))
    e, r1, r2, r3 = cc.ccsdt_residual_unfactorised(o, f, g, t1, t2, t3)
    for got, ref in ((R1.host, r1), (R2.host, r2), (R3.host, r3)):
        assert np.abs(got - ref).max() <= 1e-12 * np.abs(ref).max()
    assert oc.calls == 88


@pytest.mark.parametrize("o,v", [(3, 3), (3, 4), (4, 4)])
def test_packed_ccsdt_driver_call_list_is_the_unfactorised_equations(o, v):
    """ccd.ccsdt_residual_packed (T3 and R3 exist only packed, (a<b<c, i<j<k); three packed views of T3, three packed
    accumulators, three packed permutation operators) run on the host with the oracle's contract / add / permsum / sym.*:
    R3p unpacked equals the unfactorised 37-term evaluation."""
    from oracle import sym
    from oracle_ctx import OracleContext
    from paper_2409_06759_b200 import ccd
    f, g, t1, t2, t3 = _ccsdt_problem(o, v, 78 + o + v)
    h = f - np.einsum("piqi->pq", g[:, :o, :, :o])
    oc = OracleContext()
    W = oc.tensor_from_numpy
    t3p = sym.pack("P(a<b<c,i<j<k)=T(a,b,c,i,j,k)", t3)
    R1, R2, R3p = ccd.ccsdt_residual_packed(oc, o, W(h), W(g), W(t1), W(t2), W(t3p))
    e, r1, r2, r3 = cc.ccsdt_residual_unfactorised(o, f, g, t1, t2, t3)
    R3 = sym.unpack("R(a,b,c,i,j,k)=P(a<b<c,i<j<k)", R3p.host, extents=dict(a=v, b=v, c=v, i=o, j=o, k=o))
    for got, ref in ((R1.host, r1), (R2.host, r2), (R3, r3)):
        assert np.abs(got - ref).max() <= 1e-12 * np.abs(ref).max()
    assert oc.calls == 109
    with pytest.raises(ValueError):
        ccd.ccsdt_residual_packed(oc, 2, W(h), W(g), W(t1[:, :2]), W(t2), W(t3p))


def test_converged_ccsdt_iteration_zeroes_all_three_fock_space_projections():
    """Jacobi iterations of the CCSDT equations on a weakly coupled Hermitian problem (non-zero occupied-virtual Fock block,
    so t1 != 0): at the fixed point the singles, doubles AND triples projections of exp(-T) H exp(T)|Phi0> vanish and the
    energy is the Fock-space one; the residual norm falls monotonically."""
    o, v = 3, 3
    f, g, eo, ev = _ccsd_problem(o, v, 52)
    T1, T2, T3, energies, norms = cc.ccsdt_jacobi(o, f, g, 45)
    e0, s0, d0, t0, _ = _fock_ccsdt(o, v, f, g, T1, T2, T3)
    scale = np.abs(g).max()
    assert max(np.abs(s0).max(), np.abs(d0).max(), np.abs(t0).max()) <= 1e-12 * scale
    assert abs(cc.ccsdt_residual_unfactorised(o, f, g, T1, T2, T3)[0] - e0) <= 1e-12 * abs(e0)
    assert np.abs(T3).max() > 1e-6 and np.abs(T1).max() > 1e-4
    assert all(norms[k + 1] < norms[k] for k in range(20))
    # triples change the energy: CCSD's fixed point differs
    _, _, e_sd = cc.ccsd_jacobi(cc.ccsd_blocks(o, f, g), eo, ev, 45)
    assert abs(e_sd[-1] - e0) > 1e-9 * abs(e0)


def test_ccsdt_diis_reaches_the_fock_space_fixed_point_in_fewer_evaluations():
    """DIIS over (t1, t2, t3): the amplitudes it converges to zero all three Fock-space projections (the Jacobi fixed point),
    the first residual norm is that of the driver terms, and after 10 evaluations the norm is far below Jacobi's."""
    o, v = 3, 3
    f, g, eo, ev = _ccsd_problem(o, v, 52)
    T1, T2, T3, energies, norms = cc.ccsdt_diis(o, f, g, 18)
    e0, s0, d0, t0, _ = _fock_ccsdt(o, v, f, g, T1, T2, T3)
    scale = np.abs(g).max()
    assert max(np.abs(s0).max(), np.abs(d0).max(), np.abs(t0).max()) <= 1e-12 * scale
    assert abs(cc.ccsdt_residual_unfactorised(o, f, g, T1, T2, T3)[0] - e0) <= 1e-12 * abs(e0)
    _, _, _, ej, nj = cc.ccsdt_jacobi(o, f, g, 11)
    assert norms[0] == nj[0] and energies[0] == 0 and abs(norms[1] - nj[1]) <= 1e-14 * nj[0]    # the first step is a Jacobi step
    assert norms[10] < 0.05 * nj[10]
    assert np.abs(T3).max() > 1e-6
