"""The seeded input generator: determinism, sub-tensor consistency, exact symmetries, moments."""
import numpy as np

from paper_2409_06759_b200 import synth


def test_reference_accuracy_of_fixed_recipes():
    k53 = np.random.default_rng(0).integers(0, 2**53, 50000).astype(np.uint64)
    ref = np.log((k53.astype(np.float64) + 1) * 2.0**-53)
    assert np.abs(synth._ln_unit(k53) - ref).max() < 1e-14
    c, s = synth._cos_sin_turn(k53)
    th = 2 * np.pi * k53.astype(np.float64) * 2.0**-53
    assert np.abs(c - np.cos(th)).max() < 1e-14 and np.abs(s - np.sin(th)).max() < 1e-14


def test_moments_and_determinism():
    key = synth.tensor_key(1, 2)
    z = synth.normal_c128(key, np.arange(400000, dtype=np.uint64))
    assert abs(z.real.mean()) < 0.01 and abs(z.imag.mean()) < 0.01
    assert abs(z.real.std() - 1) < 0.01 and abs(z.imag.std() - 1) < 0.01
    assert abs((z.real * z.imag).mean()) < 0.01
    assert np.array_equal(z[1000:1010], synth.normal_c128(key, np.arange(1000, 1010, dtype=np.uint64)))
    assert not np.array_equal(z[:10], synth.normal_c128(synth.tensor_key(1, 3), np.arange(10, dtype=np.uint64)))


def test_ladder_inputs_exact_antisymmetry_and_subtensors():
    V, T = synth.config_ladder(4, 6, 1)
    assert V.flags.f_contiguous and V.shape == (6, 6, 6, 6) and T.shape == (6, 6, 4, 4)
    assert not np.any(V + V.transpose(1, 0, 2, 3)) and not np.any(V + V.transpose(0, 1, 3, 2))
    assert not np.any(T + T.transpose(1, 0, 2, 3)) and not np.any(T + T.transpose(0, 1, 3, 2))
    Vs, Ts = synth.config_ladder(4, 6, 1, sub_ab=([1, 3], [0, 5]), sub_ij=([2], [0, 3]))
    assert np.array_equal(Vs, V[np.ix_([1, 3], [0, 5], range(6), range(6))])
    assert np.array_equal(Ts, T[np.ix_(range(6), range(6), [2], [0, 3])])


def test_ccd_inputs_hermitian_consistent():
    B, T, eo, ev = synth.config_ccd(3, 5)
    assert np.array_equal(B["oovv"], B["vvoo"].transpose(2, 3, 0, 1).conj())
    assert np.array_equal(B["vvvv"], B["vvvv"].transpose(2, 3, 0, 1).conj())
    for k in ("oovv", "vvvv", "oooo"):
        assert not np.any(B[k] + B[k].transpose(1, 0, 2, 3)) and not np.any(B[k] + B[k].transpose(0, 1, 3, 2))
    assert np.all((eo >= -2) & (eo < -0.5)) and np.all((ev >= 0.5) & (ev < 3))
    assert not np.any(T + T.transpose(1, 0, 2, 3))


def test_index_linear_tensor():
    x = synth.index_linear_tensor((2, 3, 4))
    assert x[1, 2, 3].real == 1 + 2 * 2 + 3 * 6 and x[1, 2, 3].imag == -(1 + 4 + 18) - 0.5
