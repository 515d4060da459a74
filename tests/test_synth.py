"""The seeded generator: deterministic, counter-based (any sub-range regenerates identically), right statistics."""
import numpy as np

from paper_2303_11557_b200 import synth


def test_subrange_regeneration_is_identical():
    spec = synth.GaussSpec(8, 5000, 128, sigma=16.0, rho=0.05, tones=[synth.Tone(5, 4.0, 1)], seed=123)
    full = synth.gauss_voltages(spec)
    part = synth.gauss_voltages(spec, inputs=(3, 6), samples=(1000, 1700))
    assert np.array_equal(part, full[3:6, 1000:1700])
    assert np.array_equal(full, synth.gauss_voltages(spec))


def test_statistics_and_clipping():
    spec = synth.GaussSpec(4, 200000, 128, sigma=16.0, rho=0.3, seed=9)
    v = synth.gauss_voltages(spec).astype(np.float64)
    assert abs(v.std() - np.sqrt(16.0 ** 2 + 1 / 12)) < 0.1 and abs(v.mean()) < 0.1
    z = v[..., 0] + 1j * v[..., 1]
    r = (z[0] * np.conj(z[1])).mean() / (np.abs(z[0]) ** 2).mean()
    assert abs(r.real - 0.3) < 0.01 and abs(r.imag) < 0.01
    big = synth.gauss_voltages(synth.GaussSpec(1, 10000, 64, sigma=100.0, seed=1))
    assert big.max() == 127 and big.min() == -127


def test_uniform_recipe():
    z = synth.uniform_voltages(4, 100, 80, n_shared=64, seed=3)
    assert z[:, :, 64:].min() >= -8 and z[:, :, 64:].max() <= 7
    assert z[:, :, :64].min() >= -16 and z[:, :, :64].max() <= 14
    assert np.array_equal(z, synth.uniform_voltages(4, 100, 80, n_shared=64, seed=3))
    assert not np.array_equal(z, synth.uniform_voltages(4, 100, 80, n_shared=64, seed=4))


def test_config_shapes():
    c3, c4, c5 = synth.CONFIGS["C3"], synth.CONFIGS["C4"], synth.CONFIGS["C5"]
    assert c3.samples_per_input == 1_280_000 and c3.seconds_of_data == 1.0
    assert c4.samples_per_input == 2_560_000 and c4.n_keep // c4.f_avg == 128
    assert c5.samples_per_input == 640_000 and c5.n_coarse == 8
