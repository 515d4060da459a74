"""Pins for the float64 oracle: what the paper and the mathematics fix.

Every check here compares the oracle against something OTHER than itself: a brute-force sum written
out in numpy, numpy.fft as a library routine on special cases, closed forms, invariants stated in the
paper, values printed in the paper (tests/golden/), or statistical expectations.
"""
import os

import numpy as np
import pytest

from oracle import oracle
from paper_2303_11557_b200 import synth

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
rng = np.random.default_rng(20231157)


def _rand_c(n):
    return rng.standard_normal(n) + 1j * rng.standard_normal(n)


def _brute_dft(x):
    N = x.size
    k = np.arange(N)
    # definition with exact integer phase reduction
    ph = (np.outer(k, k) % N) / N
    return (x[None, :] * np.exp(-2j * np.pi * ph)).sum(axis=1)


def _volt_from_complex(x):
    """complex array [n][m] with integer parts -> int8 [n][m][2]"""
    v = np.empty(x.shape + (2,), dtype=np.int8)
    v[..., 0] = np.rint(x.real)
    v[..., 1] = np.rint(x.imag)
    return v


# ------------------------------------------------------------------ P1: DFT routine
@pytest.mark.parametrize("N", [1, 2, 3, 4, 5, 7, 8, 10, 16, 20, 25, 50, 64, 100, 125, 128, 256, 320, 625, 1000])
def test_p1_fft_equals_bruteforce(N):
    x = _rand_c(N)
    ref = _brute_dft(x)
    scale = np.abs(ref).max()
    assert np.abs(oracle.fft(x) - ref).max() <= 1e-10 * scale
    assert np.abs(oracle.dft_naive(x) - ref).max() <= 1e-10 * scale


def test_p1_fft_6400_vs_library_and_sampled_bruteforce():
    N = 6400
    x = _rand_c(N)
    got = oracle.fft(x)
    lib = np.fft.fft(x)  # library routine, same sign/scale convention (reading Q1)
    assert np.abs(got - lib).max() <= 1e-10 * np.abs(lib).max()
    q = np.arange(N)
    for k in [0, 1, 5, 175, 3199, 3200, 4793, 6399]:
        bf = (x * np.exp(-2j * np.pi * ((k * q) % N) / N)).sum()
        assert abs(got[k] - bf) <= 1e-9 * np.abs(lib).max()


def test_p1_impulse_and_linearity():
    N = 100
    e = np.zeros(N, complex)
    e[0] = 1
    assert np.allclose(oracle.fft(e), np.ones(N), atol=1e-13)
    e[:] = 0
    e[3] = 1  # shifted impulse -> pure phase ramp exp(-2 pi i 3k/N)
    assert np.allclose(oracle.fft(e), np.exp(-2j * np.pi * 3 * np.arange(N) / N), atol=1e-12)
    a, b = _rand_c(N), _rand_c(N)
    assert np.allclose(oracle.fft(2 * a - 3j * b), 2 * oracle.fft(a) - 3j * oracle.fft(b), atol=1e-10)


# ------------------------------------------------------------------ P2: sign + channel map
@pytest.mark.parametrize("N,K", [(64, 64), (128, 128), (100, 50), (25, 25), (25, 11), (6400, 6400)])
def test_p2_tone_lands_in_expected_position(N, K):
    T, A = 2, 20.0
    q = np.arange(N * T)
    for k0 in [3, -3, 0]:
        if abs(k0) > (K - 1) // 2:
            continue
        x = A * np.exp(2j * np.pi * ((k0 * q) % N) / N)
        # exact integer voltages are needed for the int8 interface: use a tone whose samples are integers
        # only when k0 == 0; otherwise feed the rounded tone and check the dominant position and its phase.
        Y = oracle.spectra(_volt_from_complex(x[None, :]), N, K, T)
        p = np.unravel_index(np.abs(Y[:, 0, 0]).argmax(), (K,))[0]
        assert p == k0 + K // 2  # DC at floor(K/2); +k0 above it; -k0 mirrors below
        assert abs(Y[p, 0, 0] - A * N) <= 0.02 * A * N  # value A*N up to int8 rounding noise
    # constant input -> DC position only, exact
    x = np.full(N * T, 7 + 3j)
    Y = oracle.spectra(_volt_from_complex(x[None, :]), N, K, T)
    assert np.allclose(Y[K // 2, :, 0], (7 + 3j) * N, atol=1e-9)
    Y[K // 2] = 0
    assert np.abs(Y).max() < 1e-9


def test_p2_keep_selects_centre_channels_in_signed_order():
    N, K, T = 20, 7, 1
    x = np.rint(10 * _rand_c(N))
    full = np.fft.fft(x)  # library routine
    Y = oracle.spectra(_volt_from_complex(x[None, :]), N, K, T)[:, 0, 0]
    expect = np.array([full[u % N] for u in range(-(K // 2), K - K // 2)])
    assert np.allclose(Y, expect, atol=1e-10)
    # even K: the extra channel is on the negative side (reading Q3)
    K = 8
    Y = oracle.spectra(_volt_from_complex(x[None, :]), N, K, T)[:, 0, 0]
    expect = np.array([full[u % N] for u in range(-4, 4)])
    assert np.allclose(Y, expect, atol=1e-10)


# ------------------------------------------------------------------ P3: Parseval
@pytest.mark.parametrize("N", [64, 128, 50])
def test_p3_parseval_total_power(N):
    n, T = 3, 5
    x = np.rint(16 * (rng.standard_normal((n, N * T)) + 1j * rng.standard_normal((n, N * T))))
    V = oracle.fx(_volt_from_complex(x), N, N, T, 1)
    for i in range(n):
        total = V[:, oracle.baseline_index(i, i)].real.sum()
        assert abs(total - N * (np.abs(x[i]) ** 2).sum()) <= 1e-9 * total


# ------------------------------------------------------------------ P4: correlation structure
def test_p4_hermitian_autos_and_bruteforce_pairs():
    n, N, T = 4, 16, 6
    x = np.rint(16 * (rng.standard_normal((n, N * T)) + 1j * rng.standard_normal((n, N * T))))
    volt = _volt_from_complex(x)
    V = oracle.fx(volt, N, N, T, 1)
    # brute force with numpy.fft (library) + explicit products
    S = np.fft.fftshift(np.fft.fft(x.reshape(n, T, N), axis=2), axes=2)  # [n][T][p]
    for i in range(n):
        for j in range(i + 1):
            ref = (S[i] * np.conj(S[j])).sum(axis=0)  # over T -> [p]
            got = V[:, oracle.baseline_index(i, j)]
            assert np.abs(got - ref).max() <= 1e-9 * np.abs(ref).max()
    for i in range(n):
        a = V[:, oracle.baseline_index(i, i)]
        assert np.all(a.imag == 0.0) and np.all(a.real >= 0.0)
    # V_ji = conj(V_ij): compute with the input order reversed
    Vr = oracle.fx(volt, N, N, T, 1, sel=np.arange(n)[::-1])
    for i in range(n):
        for j in range(i):
            # in the reversed selection, input j sits at index n-1-j > n-1-i
            vji = Vr[:, oracle.baseline_index(n - 1 - j, n - 1 - i)]
            assert np.allclose(vji, np.conj(V[:, oracle.baseline_index(i, j)]), rtol=1e-12, atol=1e-9)


def test_p4_tone_phase_and_amplitude_closure():
    """§3.1 method: per-input tones of known amplitude/phase -> arg V_ij = phi_i - phi_j and
    |V_ij| = T N^2 a_i a_j."""
    n, N, T, k0 = 4, 64, 4, 5
    amps = np.array([10.0, 20.0, 30.0, 40.0])
    phis = np.array([0.1, 1.3, -2.0, 2.9])
    q = np.arange(N * T)
    x = amps[:, None] * np.exp(1j * (2 * np.pi * ((k0 * q) % N) / N + phis[:, None]))
    V = oracle.fx(_volt_from_complex(x), N, N, T, 1)
    p = k0 + N // 2
    for i in range(n):
        for j in range(i + 1):
            v = V[p, oracle.baseline_index(i, j)]
            assert abs(abs(v) - T * N * N * amps[i] * amps[j]) <= 0.03 * T * N * N * amps[i] * amps[j]
            d = np.angle(v * np.exp(-1j * (phis[i] - phis[j])))
            assert abs(d) < 0.03


def test_p4_additivity_over_time():
    n, N, T = 3, 20, 4
    x = np.rint(16 * (rng.standard_normal((n, N * 2 * T)) + 1j * rng.standard_normal((n, N * 2 * T))))
    volt = _volt_from_complex(x)
    whole = oracle.fx(volt, N, N, 2 * T, 1)
    parts = oracle.fx(volt, N, N, T, 1, dump=0) + oracle.fx(volt, N, N, T, 1, dump=1)
    assert np.allclose(whole, parts, rtol=1e-12, atol=1e-9)


# ------------------------------------------------------------------ P5: common-signal recovery
def test_p5_common_signal_correlation_coefficient():
    cfg = synth.CONFIGS["C1"]
    spec = cfg.spec()
    spec.tones = []  # exclude tones (an off-bin or strong tone biases r-hat)
    volt = synth.gauss_voltages(spec)
    V = oracle.fx(volt, cfg.n_fft, cfg.n_keep, cfg.t_int, 1)
    n = cfg.n_inputs
    sigma2 = cfg.sigma ** 2
    expect = cfg.rho * sigma2 / (sigma2 + 1.0 / 12.0)  # integer rounding adds 1/12 variance per component
    M = cfg.t_int * cfg.n_keep
    rs = []
    for i in range(n):
        for j in range(i):
            v = V[:, oracle.baseline_index(i, j)].sum()
            ai = V[:, oracle.baseline_index(i, i)].real.sum()
            aj = V[:, oracle.baseline_index(j, j)].real.sum()
            rs.append(v / np.sqrt(ai * aj))
    rs = np.array(rs)
    tol = 5.0 / np.sqrt(M)  # conservative 5 sigma; all baselines share s so they do not average down
    assert np.all(np.abs(rs.real - expect) < tol)
    assert np.all(np.abs(rs.imag) < tol)
    assert abs(rs.real.mean() - expect) < tol


# ------------------------------------------------------------------ P6-P8: averaging weights
def test_weights_golden_K8_F2():
    tab = np.loadtxt(os.path.join(GOLDEN, "weights_K8_F2.txt"))
    W = oracle.weights(8, 2)
    assert np.array_equal(W * 2, tab)  # table is before the division by F


@pytest.mark.parametrize("K,F", [(8, 2), (256, 2), (6400, 25), (6400, 50), (6400, 256), (6400, 5), (100, 4), (75, 3)])
def test_p7_partition_of_unity_and_symmetry(K, F):
    W = oracle.weights(K, F)
    C = K // F
    c0, dc = C // 2, K // 2
    assert np.allclose(W.sum(axis=1), 1.0)  # rows are means
    assert np.all(W[:, dc] == 0.0)  # DC column excluded (L290)
    col = W.sum(axis=0) * F
    centre_taps = np.nonzero(W[c0])[0]
    others = np.setdiff1d(np.arange(K), np.concatenate([centre_taps, [dc]]))
    # "energy at every frequency contributes equally" (L306): total weight 1 outside the re-scaled centre group
    assert np.allclose(col[others], 1.0)
    # ends of the centre group are shared with a neighbour at weight 1/2 each side when F is even
    # mirror symmetry about the centre channel (L296, L302): taps of c0+m mirror those of c0-m about DC
    for m in range(1, min(c0, C - 1 - c0) + 1):
        up, dn = W[c0 + m], W[c0 - m]
        for p in np.nonzero(up)[0]:
            pm = (2 * dc - p) % K
            assert dn[pm] == up[p]
    # tap counts (L298)
    ntaps = (W[(c0 + 1) % C] != 0).sum() if C > 1 else None
    if C > 1:
        assert ntaps == (F if F % 2 else F + 1)


def test_p6_boundary_tone_splits_50_50():
    """An on-bin tone exactly on an output-channel boundary appears at 50 % in each neighbour — 'precisely 3 dB
    down at the channel boundaries'."""
    N = K = 400
    F, T, A = 50, 1, 30.0
    u = 25 + 50 * 2  # boundary between output channels c0+2 and c0+3
    q = np.arange(N * T)
    x = A * np.exp(2j * np.pi * ((u * q) % N) / N)
    V = oracle.fx(_volt_from_complex(x[None, :]), N, K, T, F)[:, 0].real
    full = oracle.fx(_volt_from_complex(x[None, :]), N, K, T, 1)[:, 0].real
    tone_power = full[u + K // 2]
    c0 = (K // F) // 2
    lo, hi = V[c0 + 2] * F, V[c0 + 3] * F  # undo the mean
    assert abs(lo / tone_power - 0.5) < 0.01 and abs(hi / tone_power - 0.5) < 0.01
    assert abs(10 * np.log10(lo / tone_power) + 3.0103) < 0.1


def test_p8_dc_tone_vanishes_and_white_noise_is_flat():
    N = K = 64
    F, T = 4, 2000
    x = np.full(N * 4, 50.0 + 0j)
    V = oracle.fx(_volt_from_complex(x[None, :]), N, K, 4, F)[:, 0]
    assert np.abs(V).max() < 1e-6  # a pure DC offset leaves no trace anywhere
    # white noise: every output channel, including the re-scaled centre one, has the same expected power
    spec = synth.GaussSpec(1, N * T, N, sigma=16.0, rho=0.0, seed=77)
    V = oracle.fx(synth.gauss_voltages(spec), N, K, T, F)[:, 0].real
    expect = T * N * 2 * (16.0 ** 2 + 1 / 12)
    # relative std of a channel ~ 1/sqrt(T*F) ~ 1.1 % (centre channel: 1/sqrt(T*(F-1)))
    assert np.all(np.abs(V / expect - 1.0) < 0.06)
    c0 = (K // F) // 2
    assert abs(V[c0] / np.delete(V, c0).mean() - 1.0) < 0.05


@pytest.mark.parametrize("K,F", [(8, 2), (64, 4), (75, 3), (6400, 50)])
def test_keep_dc_mode_weights(K, F):
    """MWAX_OPT_DC_EXCLUDE = 0: the exclusion of PAPER.md L290-294 left out.  Every fine channel then
    has total weight exactly 1 across the outputs (partition of unity with NO exception), every row is a mean, the
    centre row is the mirror-symmetric F (odd) / F + 1 (even, half-weight ends) tap window around DC written out here,
    and all other rows equal those of the default mode."""
    W = oracle.weights(K, F, oracle.AVG_KEEP_DC)
    Wd = oracle.weights(K, F)
    C, dc = K // F, K // 2
    c0 = C // 2
    assert np.allclose(W.sum(axis=1), 1.0) and np.allclose(W.sum(axis=0) * F, 1.0)
    expect = np.zeros(K)
    dmax = (F - 1) // 2 if F % 2 else F // 2
    for d in range(-dmax, dmax + 1):
        expect[(dc + d) % K] += (0.5 if (F % 2 == 0 and abs(d) == dmax) else 1.0) / F
    assert np.allclose(W[c0], expect)
    assert np.array_equal(np.delete(W, c0, axis=0), np.delete(Wd, c0, axis=0))


def test_keep_dc_mode_dc_tone_survives():
    """The pair to test_p8: with the exclusion off a DC offset of amplitude A appears in the centre channel only, at
    its closed-form power T (A N)^2 / F (one of the F taps of the mean holds it); with it on (default) it vanishes."""
    N = K = 64
    F, T, A = 4, 4, 50.0
    x = np.full(N * T, A + 0j)
    volt = _volt_from_complex(x[None, :])
    V = oracle.fx(volt, N, K, T, F, oracle.AVG_KEEP_DC)[:, 0].real
    c0 = (K // F) // 2
    assert abs(V[c0] / (T * (A * N) ** 2 / F) - 1.0) < 1e-12
    assert np.abs(np.delete(V, c0)).max() < 1e-6
    assert np.abs(oracle.fx(volt, N, K, T, F)[:, 0]).max() < 1e-6


def test_block_mode_weights():
    W = oracle.weights(12, 3, oracle.AVG_BLOCK)
    for c in range(4):
        expect = np.zeros(12)
        expect[3 * c:3 * c + 3] = 1 / 3
        assert np.allclose(W[c], expect)
    assert np.array_equal(oracle.weights(16, 1), np.eye(16))  # F = 1: identity, no DC exclusion (reading Q7)


def test_average_equals_weight_table_product():
    n, K, F = 3, 24, 4
    B = n * (n + 1) // 2
    R = _rand_c(K * B).reshape(K, B)
    V = oracle.average(R, n, F)
    W = oracle.weights(K, F)
    ref = W @ R
    for a in range(n):
        ref[:, oracle.baseline_index(a, a)] = ref[:, oracle.baseline_index(a, a)].real
    assert np.allclose(V, ref, rtol=1e-13, atol=1e-13)


# ------------------------------------------------------------------ P9: output sizes printed in the paper
def test_p9_fig14_data_rates():
    rows = np.loadtxt(os.path.join(GOLDEN, "fig14_rates.txt"))
    n = 256  # 128 tiles x 2 polarisations
    for fscrunch, count, tres, rate in rows:
        assert 6400 // int(fscrunch) == int(count)
        W = oracle.weights(6400, int(fscrunch)) if fscrunch in (25, 50) else None
        C = W.shape[0] if W is not None else 6400 // int(fscrunch)
        nbytes = C * (n * (n + 1) // 2) * 8  # complex fp32 lower triangle incl. autos (Fig 8: "complex single-precision")
        got = nbytes / tres * 24 / 1e9
        assert abs(got - rate) <= 0.0051 + 1e-9, (fscrunch, tres, got, rate)


def test_fig8_baseline_count():
    n, rows = np.loadtxt(os.path.join(GOLDEN, "fig8_baseline_rows.txt"), dtype=int)
    x = np.rint(5 * _rand_c(n * 8)).reshape(n, 8)
    V = oracle.fx(_volt_from_complex(x), 8, 8, 1, 1)
    assert V.shape[1] == rows
    assert oracle.baseline_index(n - 1, n - 1) == rows - 1


# ------------------------------------------------------------------ P10: integer path
def test_p10_int_path_bruteforce_trace_hermitian_and_float_equality():
    n_chan, n_time, n = 3, 37, 6
    z = synth.uniform_voltages(n_chan, n_time, n, n_shared=2, seed=5)
    vis = oracle.xcorr_i8(z)
    zc = z[..., 0].astype(np.int64) + 1j * z[..., 1].astype(np.int64)  # [c][t][i]
    for c in range(n_chan):
        for i in range(n):
            for j in range(i + 1):
                ref = (zc[c, :, i] * np.conj(zc[c, :, j])).sum()
                got = vis[c, oracle.baseline_index(i, j)]
                assert got[0] == int(ref.real) and got[1] == int(ref.imag)
        trace = sum(int(vis[c, oracle.baseline_index(i, i), 0]) for i in range(n))
        assert trace == int((np.abs(zc[c]) ** 2).sum().round())
        assert all(vis[c, oracle.baseline_index(i, i), 1] == 0 for i in range(n))
    # equals the float64 step-4 oracle on the same integers, exactly
    R = oracle.correlate(np.ascontiguousarray(zc.astype(np.complex128)))
    assert np.array_equal(R.real.astype(np.int64), vis[..., 0]) and np.array_equal(R.imag.astype(np.int64), vis[..., 1])
    # swapping the two inputs conjugates
    v01 = oracle.xcorr_i8(z, sel=[0, 1])[:, 1]
    v10 = oracle.xcorr_i8(z, sel=[1, 0])[:, 1]
    assert np.array_equal(v01[:, 0], v10[:, 0]) and np.array_equal(v01[:, 1], -v10[:, 1])


# ------------------------------------------------------------------ C1 worked expectation
def test_c1_tone_position_and_phase_gradient():
    """BASELINE.json configs[0]: tone at bin +5 -> position 37; arg V_jk = 2 pi (j - k)/16."""
    cfg = synth.CONFIGS["C1"]
    volt = synth.gauss_voltages(cfg.spec())
    V = oracle.fx(volt, cfg.n_fft, cfg.n_keep, cfg.t_int, cfg.f_avg)
    autos = np.array([V[:, oracle.baseline_index(i, i)].real for i in range(cfg.n_inputs)])
    assert np.all(autos.argmax(axis=1) == 37)
    # expected value at the tone position: tone term T N^2 a^2 e^{i dphi} plus the (real) common-signal term
    T, N, a = cfg.t_int, cfg.n_fft, cfg.tones[0].amp
    common = cfg.rho * 2 * cfg.sigma ** 2 * N * T
    for j, k in [(1, 0), (5, 2), (15, 3), (9, 8), (12, 4)]:
        expect = T * N * N * a * a * np.exp(2j * np.pi * (j - k) / 16) + common
        got = V[37, oracle.baseline_index(j, k)]
        assert abs(np.angle(got * np.conj(expect))) < 0.03
        assert abs(abs(got) / abs(expect) - 1.0) < 0.05


# ------------------------------------------------------------------------------------------------------------------
# Step 3b: fractional-delay / phase correction (PAPER.md 2.5.1 L266-272; reading Q19)
# ------------------------------------------------------------------------------------------------------------------
def test_delay_integer_shift_theorem_against_numpy_roll():
    """A frame circularly DELAYED by m samples (numpy.roll, nothing of the oracle's formula) has spectrum
    X(u) exp(-2 pi i u m / N); applying a delay of -m must give back the undelayed spectrum, bin by bin."""
    rng = np.random.default_rng(5)
    N, T, m = 100, 3, 7
    x = rng.integers(-100, 100, size=(T, N, 2)).astype(np.int8)
    volt = np.stack([x.reshape(T * N, 2), np.roll(x, m, axis=1).reshape(T * N, 2)]).copy()
    Y = oracle.spectra(volt, N, N, T)
    delay = np.zeros((2, T))
    delay[1, :] = -m
    Yc = oracle.apply_delays(Y, N, delay=delay)
    scale = np.abs(Y).max()
    assert np.abs(Yc[:, :, 1] - Y[:, :, 0]).max() <= 1e-10 * scale
    assert np.abs(Yc[:, :, 0] - Y[:, :, 0]).max() == 0.0
    # the opposite sign must NOT work (guards the sign convention of reading Q19)
    delay[1, :] = +m
    assert np.abs(oracle.apply_delays(Y, N, delay=delay)[:, :, 1] - Y[:, :, 0]).max() > 0.1 * scale


def test_delay_keep_uses_signed_bins():
    """With K < N the gradient must be taken at the SIGNED bin u = p - floor(K/2), not at the position p."""
    rng = np.random.default_rng(6)
    N, K, T, m = 64, 20, 2, 3
    x = rng.integers(-100, 100, size=(T, N, 2)).astype(np.int8)
    volt = np.stack([x.reshape(T * N, 2), np.roll(x, m, axis=1).reshape(T * N, 2)]).copy()
    Y = oracle.spectra(volt, N, K, T)
    delay = np.array([[0.0] * T, [-float(m)] * T])
    Yc = oracle.apply_delays(Y, N, delay=delay)
    assert np.abs(Yc[:, :, 1] - Y[:, :, 0]).max() <= 1e-10 * np.abs(Y).max()


def test_phase_offset_rotates_cross_products_and_leaves_autos():
    spec = synth.GaussSpec(4, 32 * 6, 32, sigma=16.0, rho=0.3, tones=[], seed=77)
    volt = synth.gauss_voltages(spec)
    T = 6
    phase = np.array([[0.3] * T, [-1.1] * T, [2.0] * T, [0.0] * T])
    V0 = oracle.fx(volt, 32, 32, T, 1)
    V1 = oracle.fx(volt, 32, 32, T, 1, phase=phase)
    for i in range(4):
        for j in range(i + 1):
            rot = np.exp(1j * (phase[i, 0] - phase[j, 0]))
            b = oracle.baseline_index(i, j)
            assert np.abs(V1[:, b] - V0[:, b] * rot).max() <= 1e-9 * np.abs(V0[:, b]).max()
    # per-frame values are honoured: a phase that flips sign every frame cancels in pairs for a stationary tone
    # only if it is applied frame by frame (here: simply check frame dependence changes the result)
    phase2 = phase.copy()
    phase2[0, ::2] += np.pi
    V2 = oracle.fx(volt, 32, 32, T, 1, phase=phase2)
    assert np.abs(V2[:, oracle.baseline_index(1, 0)] - V1[:, oracle.baseline_index(1, 0)]).max() > 0


def test_fractional_delay_flattens_the_phase_of_a_delayed_copy():
    """Input 1 = input 0 delayed by tau = 0.37 samples (band-limited construction in the frequency domain with
    numpy.fft, independent of the oracle): uncorrected, arg V_10(u) = -2 pi u tau / N; after applying delay -tau to
    input 1 the phase is flat ('the resulting visibilities having flat phase as a function of
    frequency')."""
    rng = np.random.default_rng(9)
    N, T, tau = 64, 40, 0.37
    u = np.fft.fftfreq(N, d=1.0 / N)                       # signed bins
    frames0, frames1 = [], []
    for _ in range(T):
        S = (rng.normal(size=N) + 1j * rng.normal(size=N)) * 60.0
        S[N // 2] = 0                                        # no Nyquist bin: its fractional delay is ambiguous
        frames0.append(np.fft.ifft(S) * np.sqrt(N))
        frames1.append(np.fft.ifft(S * np.exp(-2j * np.pi * u * tau / N)) * np.sqrt(N))
    def q(fr):
        z = np.concatenate(fr)
        return np.stack([np.clip(np.rint(z.real), -127, 127), np.clip(np.rint(z.imag), -127, 127)], axis=-1).astype(np.int8)
    volt = np.stack([q(frames0), q(frames1)]).copy()
    b = oracle.baseline_index(1, 0)
    V = oracle.fx(volt, N, N, T, 1)[:, b]
    useed = np.arange(N) - N // 2
    sel = np.abs(useed) < N // 2 - 1
    slope = np.angle(V[sel] * np.exp(2j * np.pi * useed[sel] * tau / N))
    assert np.abs(slope).max() < 0.05                        # uncorrected: the expected gradient
    Vc = oracle.fx(volt, N, N, T, 1, delay=np.array([[0.0] * T, [-tau] * T]))[:, b]
    assert np.abs(np.angle(Vc[sel])).max() < 0.05            # corrected: flat
    assert np.abs(np.angle(V[sel])).max() > 0.5


# ------------------------------------------------------------------------------------------------------------------
# Step 7: MWAX_ORDER (PAPER.md 2.7 L318-326, Figs 8-9)
# ------------------------------------------------------------------------------------------------------------------
def test_mwax_order_fig8_rows_and_bruteforce_products():
    """Fig. 8's example: 4 tiles, 2 channels -> 10 baseline rows in the printed order, channel faster than baseline,
    xx xy yx yy fastest; every element equals the product sum formed directly from the spectra with numpy."""
    n_tiles, want_rows = [int(x) for x in np.loadtxt(os.path.join(GOLDEN, "fig8_baseline_rows.txt"), dtype=int)]
    assert (n_tiles, want_rows) == (4, 10)
    n, N, K, T = 2 * n_tiles, 8, 2, 5
    spec = synth.GaussSpec(n, N * T, N, sigma=16.0, rho=0.4, tones=[], seed=808)
    volt = synth.gauss_voltages(spec)
    Y = oracle.spectra(volt, N, K, T)                      # [K][T][n]
    V = oracle.average(oracle.correlate(Y), n, 1)
    M, W = oracle.mwax_order(V, n)
    assert M.shape == (want_rows, K, 4) and W.shape == (want_rows, 4) and np.all(W == 1.0)
    rows = [(a, b) for a in range(n_tiles) for b in range(a, n_tiles)]
    assert rows == [(0, 0), (0, 1), (0, 2), (0, 3), (1, 1), (1, 2), (1, 3), (2, 2), (2, 3), (3, 3)]   # as printed in Fig. 8
    for r, (a, b) in enumerate(rows):
        for ch in range(K):
            for p in range(2):
                for q in range(2):
                    direct = np.sum(Y[ch, :, 2 * a + p] * np.conj(Y[ch, :, 2 * b + q]))
                    assert abs(M[r, ch, 2 * p + q] - direct) <= 1e-9 * max(1.0, abs(direct))
    # autos: xx and yy real, xy = conj(yx)
    for r, (a, b) in enumerate(rows):
        if a == b:
            assert np.all(M[r, :, 0].imag == 0) and np.all(M[r, :, 3].imag == 0)
            assert np.allclose(M[r, :, 1], np.conj(M[r, :, 2]))


def test_mwax_order_value_count_matches_the_paper():
    """128 tiles: 8256 baselines x 4 polarisation products = 33 024 values per channel (Fig. 8's format; DESIGN Q16)."""
    nt = 128
    assert nt * (nt + 1) // 2 * 4 == 33024


# ------------------------------------------------------------------------------------------------------------------
# Step 8: occupancy weights from the zeroing flags (PAPER.md 4.1 L557-559)
# ------------------------------------------------------------------------------------------------------------------
def test_occupancy_weights_bruteforce_and_special_cases():
    rng = np.random.default_rng(12)
    nt, S = 5, 16
    flags = (rng.random((2 * nt, S)) < 0.3).astype(np.uint8)
    flags[4, :] = 1                                          # a signal path zeroed for the whole integration
    flags[7, :] = 0                                          # a signal path that lost nothing
    W = oracle.occupancy(flags)
    valid = 1 - flags.astype(np.int64)
    row = 0
    for a in range(nt):
        for b in range(a, nt):
            for p in range(2):
                for q in range(2):
                    want = np.mean(valid[2 * a + p] & valid[2 * b + q])      # numpy, nothing of the oracle's loop
                    assert W[row, 2 * p + q] == want
            row += 1
    assert np.all((W >= 0) & (W <= 1))
    assert np.all(oracle.occupancy(np.zeros((2 * nt, S), np.uint8)) == 1.0)          # "all values are set to 1.0" today (L328)
    rows = {(a, b): r for r, (a, b) in enumerate((a, b) for a in range(nt) for b in range(a, nt))}
    assert np.all(W[rows[(2, 2)], 0] == 0) and np.all(W[rows[(0, 2)], [0, 2]] == 0)  # everything with path 4 = (tile 2, x)
    assert W[rows[(3, 3)], 3] == 1.0                                                # path 7 with itself


def test_occupancy_normalisation_restores_visibility_magnitudes():
    """Zero a quarter of the integration on one signal path: its cross products drop to ~75 %; dividing by the weight
    brings them back (L559: 'such that missing packets do not cause variations in visibility magnitudes')."""
    n, N, T, S = 4, 32, 400, 8
    spec = synth.GaussSpec(n, N * T, N, sigma=16.0, rho=0.6, tones=[], seed=99)
    volt = synth.gauss_voltages(spec)
    full, _ = oracle.mwax_order(oracle.fx(volt, N, N, T, N), n)       # one output channel (all fine channels averaged)
    flags = np.zeros((n, S), np.uint8)
    flags[1, :2] = 1                                                   # path 1 = (tile 0, y): first quarter zeroed
    vz = volt.copy()
    vz[1, : N * T // 4] = 0
    M, _ = oracle.mwax_order(oracle.fx(vz, N, N, T, N), n)
    W, Mn = oracle.occupancy(flags, M, normalise=True)
    r01 = 1                                                            # row (antA 0, antB 1)
    assert W[r01, 2] == 0.75 and W[r01, 0] == 1.0                      # yx involves path 1, xx does not
    ratio_raw = abs(M[r01, 0, 2]) / abs(full[r01, 0, 2])
    ratio_norm = abs(Mn[r01, 0, 2]) / abs(full[r01, 0, 2])
    assert abs(ratio_raw - 0.75) < 0.05 and abs(ratio_norm - 1.0) < 0.05
    assert np.array_equal(Mn[r01, :, 0], M[r01, :, 0])                 # weight 1.0: untouched


# ------------------------------------------------------------------ step 3c: per-channel magnitude gains (PFB de-ripple, PAPER.md 4.2)
def test_channel_gains_scale_each_fine_channel_by_gain_squared():
    """F = 1: V'[p] = gain[p]^2 V[p] (both operands of every product carry the gain); the expected values are the
    UNGAINED oracle output scaled in numpy.  An un-squared gain, a gain on one operand only, or a gain indexed in FFT
    order instead of centre order all fail here."""
    n, N, K, T = 3, 16, 12, 5
    volt = rng.integers(-100, 100, size=(n, T * N, 2)).astype(np.int8)
    gain = 0.5 + rng.random(K)
    V0 = oracle.fx(volt, N, K, T, 1)
    V1 = oracle.fx(volt, N, K, T, 1, gain=gain)
    np.testing.assert_allclose(V1, V0 * (gain ** 2)[:, None], rtol=1e-12, atol=1e-9)
    np.testing.assert_array_equal(oracle.fx(volt, N, K, T, 1, gain=np.ones(K)), V0)


def test_channel_gains_tone_power_follows_its_own_channel():
    """A tone on signed bin u0 sits at position u0 + K/2: only THAT entry of the gain table changes its power."""
    N = K = 32
    T, u0, a = 4, -7, 20.0
    m = np.arange(T * N)
    x = a * np.exp(2j * np.pi * u0 * m / N)
    volt = _volt_from_complex(x[None, :])
    base = oracle.fx(volt, N, K, T, 1)[:, 0].real
    for p_changed in (u0 + K // 2, (u0 % N)):                  # the right index, and the FFT-order index (wrong one)
        gain = np.ones(K)
        gain[p_changed] = 3.0
        got = oracle.fx(volt, N, K, T, 1, gain=gain)[:, 0].real
        ratio = got[u0 + K // 2] / base[u0 + K // 2]
        assert np.isclose(ratio, 9.0 if p_changed == u0 + K // 2 else 1.0, rtol=1e-9)


def test_channel_gains_with_averaging_equal_numpy_scaled_fine_channels():
    """F > 1: the gained dump equals the paper's weighted mean (weights() is pinned by P6-P8 and the golden table) of
    the numpy-scaled fine-channel products."""
    n, N, K, T, F = 2, 40, 40, 3, 4
    volt = rng.integers(-60, 60, size=(n, T * N, 2)).astype(np.int8)
    gain = 0.8 + 0.4 * rng.random(K)
    R = oracle.correlate(oracle.spectra(volt, N, K, T))        # [K][B]
    W = oracle.weights(K, F)                                   # [C][K]
    expect = W @ (R * (gain ** 2)[:, None])
    expect[:, [0, 2]] = expect[:, [0, 2]].real                 # autos (baselines 0 and 2 of n = 2)
    np.testing.assert_allclose(oracle.fx(volt, N, K, T, F, gain=gain), expect, rtol=1e-11, atol=1e-7)


def test_deripple_flattens_a_known_passband_ripple():
    """PAPER.md 4.2 L567: gains equal to the inverse of the passband magnitude response give 'a flattened overall
    frequency response'.  White noise is given a known ripple H(u) per frame with numpy.fft (a library routine, circular
    filtering), quantised to int8, and correlated with gain = 1 / H: the auto spectrum must come out flat, and without
    the gains it must follow H^2."""
    N = K = 64
    T, sigma = 600, 20.0
    u = np.arange(K) - K // 2                                  # signed bin of position p
    H_pos = 1.0 + 0.3 * np.cos(2 * np.pi * u / K) - 0.15 * np.sin(6 * np.pi * u / K)   # deliberately not symmetric in u
    H_fft = np.fft.ifftshift(H_pos)                            # FFT order (bin k = u mod N)
    g = sigma * (rng.standard_normal((T, N)) + 1j * rng.standard_normal((T, N)))
    x = np.fft.ifft(np.fft.fft(g, axis=1) * H_fft[None, :], axis=1).reshape(1, T * N)
    volt = _volt_from_complex(x)
    raw = oracle.fx(volt, N, K, T, 1)[:, 0].real
    flat = oracle.fx(volt, N, K, T, 1, gain=1.0 / H_pos)[:, 0].real
    level = 2 * sigma ** 2 * N * T                             # E|X[k]|^2 summed over T spectra
    # chi-square scatter of a T-spectrum sum: 1/sqrt(T) = 4 %; int8 rounding adds 1/6 to 800 (0.02 %)
    assert np.all(np.abs(flat / level - 1.0) < 5 / np.sqrt(T))
    assert np.all(np.abs(raw / (level * H_pos ** 2) - 1.0) < 5 / np.sqrt(T))
    assert np.std(raw / level) > 5 * np.std(flat / level)      # the ripple was really there, and is gone
