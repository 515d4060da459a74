"""GPU parity: the CUDA path (through the C ABI) against the float64 oracle on the same seeded inputs.

Bars (BASELINE.json north star): int8 X-only path bit-exact; float path |V_gpu - V_ref| <= 2e-3 * sqrt(A_i A_j) per
visibility, A = the oracle's autocorrelation in the same (dump, channel); no absolute floor (all-zero data must
give exact zeros).  Small cases are compared element by element; BASELINE.json's full-size configs are compared
on sampled inputs (every pair among a selection that straddles the tile boundaries) which the oracle computes
one by one, in the launch configuration bench.py times.
"""
import numpy as np
import pytest
import torch

from oracle import oracle
from paper_2303_11557_b200 import corr, synth

pytestmark = pytest.mark.gpu

TOL = 2e-3   # north star: |V_gpu - V_ref| <= 2e-3 sqrt(A_i A_j)


def _complex(vis_f32):
    v = vis_f32.astype(np.float64)
    return v[..., 0] + 1j * v[..., 1]


def _norm_err(got, ref, n_sel):
    """got, ref complex [C][B_sel] over the same selection; returns max |got-ref| / sqrt(A_i A_j)."""
    A = np.array([ref[:, oracle.baseline_index(i, i)].real for i in range(n_sel)])     # [n_sel][C]
    ii, jj = np.tril_indices(n_sel)
    norm = np.sqrt(A[ii] * A[jj]).T
    d = np.abs(got - ref)
    assert np.all(d[norm == 0] == 0), "non-zero output where the oracle's autocorrelations vanish"
    with np.errstate(invalid="ignore", divide="ignore"):
        e = np.where(norm > 0, d / norm, 0.0)
    return float(e.max())


def _gather_sel(full, sel):
    """full [..., B_full] -> [..., B_sel] for sorted selection sel (pairs (a >= b) -> inputs (sel[a], sel[b]))."""
    sel = np.asarray(sel)
    a, b = np.tril_indices(len(sel))
    idx = sel[a] * (sel[a] + 1) // 2 + sel[b]
    return full[..., idx]


def _run_fx(volt, n, N, K, T, F, mode=0, n_dumps=1, options=()):
    h = corr.MwaxCorr(n, N, K, T, F, avg_mode=mode)
    for key, value in options:
        h.set_option(key, value)
    v = torch.from_numpy(volt).cuda()
    out = h.new_output(n_dumps=n_dumps)
    out.fill_(float("nan"))
    if n_dumps == 1 and volt.shape[1] == T * N:
        h.process(v, out[0, 0])
    else:
        h.process_batch(v[None], out, n_dumps)
    torch.cuda.synchronize()
    got = _complex(out.cpu().numpy()[0])
    h.destroy()
    return got     # [D][C][B]


# ---------------------------------------------------------------------------------------------- int8 X-only
@pytest.mark.parametrize("n,n_chan,n_time", [
    (8, 1, 1), (8, 2, 31), (16, 3, 128), (64, 2, 129), (72, 3, 300), (136, 2, 257), (200, 5, 1000), (512, 2, 2000),
])
def test_int8_bit_exact_elementwise(n, n_chan, n_time):
    z = synth.uniform_voltages(n_chan, n_time, n, n_shared=min(64, n), seed=100 + n)
    h = corr.MwaxXcorrI8(n, n_chan, n_time)
    out = h.new_output()
    out.fill_(-12345)
    h.process(torch.from_numpy(z).cuda(), out)
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy(), oracle.xcorr_i8(z))
    h.destroy()


@pytest.mark.parametrize("n,n_chan,n_time", [(72, 9, 300), (13, 5, 129), (200, 3, 64)])
def test_int8_host_buffer_entry_bit_exact(n, n_chan, n_time):
    """mwax_xcorr_i8_process_host: channel ranges pipelined over three streams (fewer channels than ranges included),
    rows padded to 16 bytes on the way in when n % 8 != 0."""
    z = synth.uniform_voltages(n_chan, n_time, n, n_shared=min(64, n), seed=300 + n)
    h = corr.MwaxXcorrI8(n, n_chan, n_time)
    hz = torch.from_numpy(z).contiguous().pin_memory()
    hout = torch.full((n_chan, n * (n + 1) // 2, 2), -7, dtype=torch.int32).pin_memory()
    for _ in range(2):      # the second call reuses the staging buffers
        h.process_host(hz, hout)
    assert np.array_equal(hout.numpy(), oracle.xcorr_i8(z))
    h.destroy()


def test_int8_extreme_values_bit_exact():
    """-128 and +127 everywhere it hurts: accumulator magnitude 2*128^2*T stays exact in int32."""
    n, n_chan, n_time = 24, 2, 4000
    rng = np.random.default_rng(5)
    z = rng.choice(np.array([-128, -127, 127, 0, 1], dtype=np.int8), size=(n_chan, n_time, n, 2))
    z[0, :, 0, :] = -128
    z[0, :, 1, :] = 127
    h = corr.MwaxXcorrI8(n, n_chan, n_time)
    out = h.new_output()
    h.process(torch.from_numpy(z).cuda(), out)
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy(), oracle.xcorr_i8(z))
    h.destroy()


def test_int8_config2_full_size_sampled():
    """BASELINE.json configs[1]: 512 inputs x 1024 channels x 2000 samples; the oracle computes every pair among
    a selection of inputs straddling all tile boundaries, for every channel."""
    n, n_chan, n_time = 512, 1024, 2000
    z = synth.uniform_voltages(n_chan, n_time, n)          # recipe: U{-8..7} + shared component on inputs 0-63
    h = corr.MwaxXcorrI8(n, n_chan, n_time)
    out = h.new_output()
    h.process(torch.from_numpy(z).cuda(), out)
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    sel = np.array([0, 1, 31, 63, 64, 65, 127, 128, 129, 191, 255, 256, 300, 383, 384, 448, 510, 511])
    ref = oracle.xcorr_i8(z, sel=sel)
    a, b = np.tril_indices(len(sel))
    idx = sel[a] * (sel[a] + 1) // 2 + sel[b]
    assert np.array_equal(got[:, idx, :], ref)
    # properties that hold at any size: autos real, non-negative, equal to the summed power
    ii = np.arange(n)
    autos = got[:, ii * (ii + 1) // 2 + ii, :]
    assert np.all(autos[..., 1] == 0) and np.all(autos[..., 0] >= 0)
    power = (z.astype(np.int64) ** 2).sum(axis=(1, 3))      # [chan][input]
    assert np.array_equal(autos[..., 0].astype(np.int64), power)
    h.destroy()


# ---------------------------------------------------------------------------------------------- float FX path
def test_config1_tiny_fx_elementwise():
    """BASELINE.json configs[0]: 16 inputs, N = K = 64, 256 spectra, rho = 0.3, tone at bin +5."""
    cfg = synth.CONFIGS["C1"]
    volt = synth.gauss_voltages(cfg.spec())
    ref = oracle.fx(volt, cfg.n_fft, cfg.n_keep, cfg.t_int, cfg.f_avg)
    got = _run_fx(volt, cfg.n_inputs, cfg.n_fft, cfg.n_keep, cfg.t_int, cfg.f_avg)[0]
    assert _norm_err(got, ref, cfg.n_inputs) <= TOL
    # the library counts the kernels it enqueues (bench.py's gpu_launches): one F + one X per integration, one for MWAX_ORDER
    h = corr.MwaxCorr(cfg.n_inputs, cfg.n_fft, cfg.n_keep, cfg.t_int, cfg.f_avg)
    assert h.launch_count() == 0
    out = h.new_output()
    h.process(torch.from_numpy(volt).cuda(), out[0, 0])
    assert h.launch_count() == 2
    h.to_mwax_order(out[0, 0])
    assert h.launch_count() == 3
    torch.cuda.synchronize()
    h.destroy()
    # the tone lands at position 5 + 32 with phase 2 pi (i - j) / 16 (reading Q18)
    p = 37
    n = cfg.n_inputs
    auto = np.array([got[:, oracle.baseline_index(i, i)].real for i in range(n)])
    assert np.all(auto.argmax(axis=1) == p)
    v = got[p, oracle.baseline_index(9, 4)]
    assert abs(np.angle(v * np.exp(-2j * np.pi * (9 - 4) / 16))) < 0.05


@pytest.mark.parametrize("n,N,K,T,F,mode", [
    (1, 64, 64, 8, 1, 0),          # a single input: one auto per channel
    (3, 5, 5, 7, 1, 0),            # tiny odd everything, scalar-load path
    (16, 64, 64, 40, 2, 0),        # even F: F+1 taps, half-weight edges, cyclic wrap of channel 0
    (16, 64, 64, 40, 2, 1),        # BLOCK mode
    (24, 100, 50, 33, 5, 0),       # radix-5, K < N, odd F, DC exclusion
    (40, 250, 250, 17, 25, 0),     # 2 * 5^3
    (70, 128, 96, 65, 4, 0),       # ragged inputs (pad columns), T one past a 64-row block
    (130, 128, 128, 100, 1, 0),    # inputs straddle a 128-input tile
    (200, 256, 256, 20, 2, 0),     # config-5 shape cut down
    (33, 512, 512, 9, 4, 0),       # largest register-kernel length
    (33, 64, 48, 9, 1, 0),         # keep < fft in the register kernel
    (40, 2048, 2048, 3, 1, 0),     # power of two beyond the register kernel (generic Stockham path)
    (12, 1024, 1000, 6, 8, 0),
    (8, 6400, 6400, 4, 50, 0),     # the paper's mode, cut down
    (8, 6400, 6400, 3, 256, 0),    # odd number of output channels (25)
    (20, 6400, 6400, 2, 1, 0),     # no averaging at N = 6400
    (10, 6400, 6400, 3, 50, 0),    # inputs not a multiple of the 4-input group of the 80 x 80 kernel
    (6, 6400, 5000, 2, 50, 0),     # keep < fft at N = 6400 (oversampled coarse channel, L611)
    (7, 6400, 6400, 2, 50, 1),     # BLOCK mode at N = 6400
    (16, 6400, 6400, 60, 50, 0),   # 120 work items on 148 CTAs: one item each, every row leaves in the kernel's final flush
    (48, 6400, 6400, 37, 50, 0),   # 222 work items on 148 CTAs: half the CTAs store one item during the next item's passes
                                   # 1-2 and flush the second, the others flush their only one
    (48, 6400, 4000, 37, 50, 0),   # the same with keep < fft: the deferred stores carry the row-range predicate
])
def test_fx_elementwise_shapes(n, N, K, T, F, mode):
    tones = [synth.Tone(min(3, K // 2 - 1), 6.0, 1)] if K > 8 else []
    spec = synth.GaussSpec(n, N * T, N, sigma=16.0, rho=0.2, tones=tones, seed=1000 + n + N)
    volt = synth.gauss_voltages(spec)
    ref = oracle.fx(volt, N, K, T, F, mode)
    got = _run_fx(volt, n, N, K, T, F, mode)[0]
    assert not np.isnan(got.view(np.float64)).any()
    assert _norm_err(got, ref, n) <= TOL
    ii = np.arange(n)
    autos = got[:, ii * (ii + 1) // 2 + ii]
    assert np.all(autos.imag == 0.0) and np.all(autos.real >= 0.0)


def test_fx_all_zero_input_gives_exact_zeros():
    n, N, T = 16, 64, 10
    volt = np.zeros((n, N * T, 2), dtype=np.int8)
    got = _run_fx(volt, n, N, N, T, 2)[0]
    assert np.all(got == 0)


def test_fx_full_scale_tone_does_not_overflow_fp16():
    """+-127 full-scale tone at N = 6400: |X| = 127 sqrt(2) N would overflow fp16 without the F-stage scaling."""
    n, N, T, F = 8, 6400, 2, 50
    q = np.arange(N * T)
    x = 127.0 * np.exp(2j * np.pi * ((1010 * q) % N) / N)
    volt = np.empty((n, N * T, 2), dtype=np.int8)
    volt[..., 0] = np.rint(x.real)
    volt[..., 1] = np.rint(x.imag)
    volt[3] = np.random.default_rng(3).choice(np.array([-128, 127], dtype=np.int8), size=(N * T, 2))
    ref = oracle.fx(volt, N, N, T, F)
    got = _run_fx(volt, n, N, N, T, F)[0]
    assert np.isfinite(got.view(np.float64)).all()
    assert _norm_err(got, ref, n) <= TOL


@pytest.mark.parametrize("n,N,K,T,F", [
    (40, 128, 128, 6, 1),       # register kernel, N = 128, every bin kept
    (40, 256, 256, 5, 2),       # register kernel, N = 256, FULL + SCALE variant
    (40, 256, 200, 5, 4),       # register kernel, N = 256, keep < fft
    (40, 64, 64, 7, 1),         # register kernel, N = 64
    (12, 100, 100, 6, 5),       # generic Stockham kernel
    (12, 6400, 6400, 2, 50),    # N = 6400 kernel (byte-permute promotion since round 2)
])
def test_fx_minus_128_and_plus_127_samples(n, N, K, T, F):
    """-128 is a legal sample (reading Q9) that the seeded generator never makes (it clips to +-127): rows of nothing but
    {-128, +127}, a row that is -128 seven times out of ten and an alternating row with random flips go through every F
    kernel's int8 -> fp32 promotion.  (Exactly constant or exactly alternating rows would have exactly-zero channels,
    where the normalised error is 0/0.)"""
    rng = np.random.default_rng(128 + N)
    volt = synth.gauss_voltages(synth.GaussSpec(n, N * T, N, sigma=16.0, rho=0.2, tones=[], seed=128 + n + N))
    volt[1] = rng.choice(np.array([-128, 127], dtype=np.int8), size=(N * T, 2))
    volt[2] = np.where(rng.random((N * T, 2)) < 0.7, -128, rng.integers(-128, 128, size=(N * T, 2))).astype(np.int8)
    alt = np.where(np.arange(N * T)[:, None] % 2 == 0, -128, 127) * np.where(rng.random((N * T, 2)) < 0.1, 0, 1)
    volt[5] = alt.astype(np.int8)
    volt[n - 1] = rng.choice(np.array([-128, -127, 0, 127], dtype=np.int8), size=(N * T, 2))
    ref = oracle.fx(volt, N, K, T, F)
    got = _run_fx(volt, n, N, K, T, F)[0]
    assert np.isfinite(got.view(np.float64)).all()
    assert _norm_err(got, ref, n) <= TOL


@pytest.mark.parametrize("n,N,K,T,F", [(16, 64, 64, 40, 4), (20, 128, 96, 9, 3), (10, 6400, 6400, 3, 50), (33, 256, 256, 70, 2)])
def test_dc_exclude_option(n, N, K, T, F):
    """MWAX_OPT_DC_EXCLUDE: 1 (default) removes the DC fine channel from the centre output channel and
    re-scales it, 0 leaves the step out; both against the oracle's weight tables, with a DC offset on every input so that
    the two differ by far more than the tolerance."""
    spec = synth.GaussSpec(n, N * T, N, sigma=16.0, rho=0.2, tones=[synth.Tone(0, 12.0, 0)], seed=600 + n + N)
    volt = synth.gauss_voltages(spec)
    ref_on = oracle.fx(volt, N, K, T, F)
    ref_off = oracle.fx(volt, N, K, T, F, oracle.AVG_KEEP_DC)
    got_on = _run_fx(volt, n, N, K, T, F)[0]
    got_off = _run_fx(volt, n, N, K, T, F, options=[(corr.MWAX_OPT_DC_EXCLUDE, 0)])[0]
    back_on = _run_fx(volt, n, N, K, T, F, options=[(corr.MWAX_OPT_DC_EXCLUDE, 0), (corr.MWAX_OPT_DC_EXCLUDE, 1)])[0]
    assert _norm_err(got_on, ref_on, n) <= TOL
    assert _norm_err(got_off, ref_off, n) <= TOL
    assert np.array_equal(back_on, got_on)
    c0 = (K // F) // 2
    assert got_off[c0, 0].real > 3.0 * got_on[c0, 0].real, "with the exclusion off the DC offset must show in the centre channel"


def test_fx_additivity_over_dumps_and_batch_layout():
    """process_batch with a row pitch longer than one integration: dump d uses samples [dTN, (d+1)TN) of every
    row; an integration over 2T equals the sum of the two integrations over T."""
    n, N, T = 48, 128, 30
    spec = synth.GaussSpec(n, N * 2 * T, N, sigma=16.0, rho=0.1, seed=77)
    volt = synth.gauss_voltages(spec)
    two = _run_fx(volt, n, N, N, T, 1, n_dumps=2)
    whole = _run_fx(volt, n, N, N, 2 * T, 1)[0]
    ref0 = oracle.fx(volt, N, N, T, 1, dump=0)
    ref1 = oracle.fx(volt, N, N, T, 1, dump=1)
    assert _norm_err(two[0], ref0, n) <= TOL and _norm_err(two[1], ref1, n) <= TOL
    assert _norm_err(two[0] + two[1], ref0 + ref1, n) <= TOL
    assert _norm_err(whole, ref0 + ref1, n) <= TOL


SEL = [0, 1, 62, 63, 64, 127, 128, 129, 255, 256, 383, 384, 510, 511]


@pytest.mark.parametrize("name", ["C3", "C4"])
def test_fx_full_size_configs_sampled(name):
    """BASELINE.json configs[2]/[3] at full size through process_batch (the launch configuration bench.py times);
    the oracle computes every pair among SEL (inputs on both sides of every 64/128-input tile edge), all channels,
    both dumps."""
    cfg = synth.CONFIGS[name]
    n, N, K, T, F, D = cfg.n_inputs, cfg.n_fft, cfg.n_keep, cfg.t_int, cfg.f_avg, cfg.n_dumps
    host = torch.empty((1, n, cfg.samples_per_input, 2), dtype=torch.int8)
    volt = host.numpy()[0]
    synth.gauss_voltages(cfg.spec(), out=volt)
    h = corr.MwaxCorr(n, N, K, T, F)
    out = h.new_output(n_dumps=D)
    h.process_batch(host.cuda(), out, D)
    torch.cuda.synchronize()
    got = _complex(out.cpu().numpy()[0])
    h.destroy()
    for d in range(D):
        ref = oracle.fx(volt, N, K, T, F, dump=d, sel=np.array(SEL))
        assert _norm_err(_gather_sel(got[d], SEL), ref, len(SEL)) <= TOL
    # a seeded-random selection as well (SEL sits on tile edges; a wrong store INSIDE a 256 x 256 tile would pass it):
    # 16 inputs on dump 0, and 64 inputs = 2080 baselines on every channel of dump 1
    rng = np.random.default_rng(20260 + len(name) + N)
    for d, m in ((0, 16), (1, 64)):
        rsel = np.sort(rng.choice(n, size=m, replace=False))
        ref = oracle.fx(volt, N, K, T, F, dump=d, sel=rsel)
        assert _norm_err(_gather_sel(got[d], rsel), ref, m) <= TOL
    ii = np.arange(n)
    autos = got[..., ii * (ii + 1) // 2 + ii]
    assert np.all(autos.imag == 0.0) and np.all(autos.real >= 0.0)
    if name == "C4":
        # the DC tone (amplitude 10 on every input) must vanish from the centre output channel:
        # that channel's autos stay at the noise level of its neighbours
        c0 = (K // F) // 2
        assert np.all(autos[:, c0] < 1.5 * autos[:, c0 + 1])


def test_fx_config5_shape_two_coarse_channels_sampled():
    """BASELINE.json configs[4] cut to 2 of its 8 coarse channels (same per-channel sizes: 1024 inputs, N = 256,
    F = 2, 2 dumps of 1250 spectra), [coarse][input][time] layout through process_batch."""
    cfg = synth.CONFIGS["C5"]
    n, N, K, T, F, D = cfg.n_inputs, cfg.n_fft, cfg.n_keep, cfg.t_int, cfg.f_avg, cfg.n_dumps
    n_coarse = 2
    host = torch.empty((n_coarse, n, cfg.samples_per_input, 2), dtype=torch.int8)
    for c in range(n_coarse):
        synth.gauss_voltages(cfg.spec(coarse=c), out=host.numpy()[c])
    h = corr.MwaxCorr(n, N, K, T, F)
    out = h.new_output(n_dumps=D, n_coarse=n_coarse)
    h.process_batch(host.cuda(), out, D, n_coarse)
    torch.cuda.synchronize()
    got = _complex(out.cpu().numpy())
    h.destroy()
    sel = [0, 63, 64, 127, 128, 511, 512, 767, 768, 1023]
    for c in range(n_coarse):
        for d in range(D):
            ref = oracle.fx(host.numpy()[c], N, K, T, F, dump=d, sel=np.array(sel))
            assert _norm_err(_gather_sel(got[c, d], sel), ref, len(sel)) <= TOL


def test_fx_config5_full_batch_last_coarse_channel():
    """BASELINE.json configs[4] WHOLE: 8 coarse channels x 1024 inputs x 0.5 s through one process_batch call (10.5 GB in,
    8.6 GB out: byte offsets beyond 4 GiB on both sides); the oracle checks coarse channel 7, dump 1 and coarse channel 0,
    dump 0 on a 10-input selection.  Coarse channels 1..6 reuse channel 0's samples (generation time), 7 has its own."""
    cfg = synth.CONFIGS["C5"]
    n, N, K, T, F, D = cfg.n_inputs, cfg.n_fft, cfg.n_keep, cfg.t_int, cfg.f_avg, cfg.n_dumps
    NCO = 8
    dev = torch.empty((NCO, n, cfg.samples_per_input, 2), dtype=torch.int8, device="cuda")
    host = torch.empty((n, cfg.samples_per_input, 2), dtype=torch.int8).pin_memory()
    synth.gauss_voltages(cfg.spec(coarse=0), out=host.numpy())
    first = host.numpy().copy()
    for c in range(NCO - 1):
        dev[c].copy_(host)
    synth.gauss_voltages(cfg.spec(coarse=7), out=host.numpy())
    dev[NCO - 1].copy_(host)
    h = corr.MwaxCorr(n, N, K, T, F)
    out = h.new_output(n_dumps=D, n_coarse=NCO)
    assert dev.numel() > 2 ** 32 and out.numel() * 4 > 2 ** 32
    h.process_batch(dev, out, D, NCO)
    torch.cuda.synchronize()
    sel = [0, 1, 63, 64, 500, 511, 512, 767, 1000, 1023]
    for (c, d, volt) in ((NCO - 1, 1, host.numpy()), (0, 0, first)):
        got = _complex(out[c, d].cpu().numpy())
        ref = oracle.fx(volt, N, K, T, F, dump=d, sel=np.array(sel))
        assert _norm_err(_gather_sel(got, sel), ref, len(sel)) <= TOL
    # channels 1..6 saw channel 0's samples: same bits
    assert torch.equal(out[3].view(torch.int32), out[0].view(torch.int32))
    h.destroy()


def test_host_buffer_entry_full_config3_against_oracle():
    """The e2e leg of bench.py: mwax_corr_process_host at BASELINE.json configs[2]'s full size (two dumps, the last one
    leaving in four channel ranges) against the oracle on SEL, and bit-identical to the device entry."""
    cfg = synth.CONFIGS["C3"]
    n, N, K, T, F, D = cfg.n_inputs, cfg.n_fft, cfg.n_keep, cfg.t_int, cfg.f_avg, cfg.n_dumps
    hv = torch.empty((1, n, cfg.samples_per_input, 2), dtype=torch.int8).pin_memory()
    synth.gauss_voltages(cfg.spec(), out=hv.numpy()[0])
    h = corr.MwaxCorr(n, N, K, T, F)
    hout = torch.full((1, D, K // F, n * (n + 1) // 2, 2), float("nan"), dtype=torch.float32).pin_memory()
    h.process_host(hv, hout, D, 1)
    dev = h.new_output(n_dumps=D)
    h.process_batch(hv.cuda(), dev, D)
    torch.cuda.synchronize()
    assert torch.equal(hout.view(torch.int32), dev.cpu().view(torch.int32))
    got = _complex(hout.numpy()[0])
    for d in range(D):
        ref = oracle.fx(hv.numpy()[0], N, K, T, F, dump=d, sel=np.array(SEL))
        assert _norm_err(_gather_sel(got[d], SEL), ref, len(SEL)) <= TOL
    # streaming accumulation has no host entry (the sum would live in the staging buffer): refused, nothing enqueued
    h.set_accumulate(True)
    with pytest.raises(corr.MwaxError):
        h.process_host(hv, hout, D, 1)
    h.destroy()


def test_two_live_handles_of_different_lengths_alternate():
    """Several handles may be alive at once (include/mwax_corr.h).  Kernel attributes are per device, not per handle: a
    generic-kernel plan with a large shared tile (N = 2048), one with a small tile (N = 100) and a specialised one
    (N = 6400, given a misaligned buffer so that it falls back to the generic kernel with ITS tile) keep working in any order."""
    shapes = [(12, 2048, 2048, 3, 1), (12, 100, 100, 6, 5), (8, 6400, 6400, 2, 50)]
    hs, vs, refs = [], [], []
    for k, (n, N, K, T, F) in enumerate(shapes):
        volt = synth.gauss_voltages(synth.GaussSpec(n, N * T, N, sigma=16.0, rho=0.2, tones=[], seed=50 + k))
        refs.append(oracle.fx(volt, N, K, T, F))
        hs.append(corr.MwaxCorr(n, N, K, T, F))
        if N == 6400:
            buf = torch.empty(volt.size + 2, dtype=torch.int8, device="cuda")
            v = buf[2:].view(volt.shape)       # 2 bytes off 16-byte alignment: scalar-load generic kernel
            v.copy_(torch.from_numpy(volt))
        else:
            v = torch.from_numpy(volt).cuda()
        vs.append(v)
    for order in ((0, 1, 2), (2, 0, 1), (1, 2, 0), (0, 2, 1)):
        for k in order:
            n, N, K, T, F = shapes[k]
            out = hs[k].new_output()
            out.fill_(float("nan"))
            if N == 6400:
                hs[k].process_batch(vs[k][None], out, 1)
            else:
                hs[k].process(vs[k], out[0, 0])
            torch.cuda.synchronize()
            assert _norm_err(_complex(out.cpu().numpy()[0, 0]), refs[k], n) <= TOL
    for h in hs:
        h.destroy()


@pytest.mark.parametrize("n,N,K,T,F,D,NCO", [
    (32, 128, 128, 20, 2, 2, 1),
    (70, 320, 300, 6, 3, 1, 2),      # two coarse channels through the reused staging; 100 output channels in 4 uneven ranges
    (300, 64, 64, 40, 1, 3, 1),      # pair tiles; the last dump leaves in channel ranges (mwax_api.cu: process_host)
    (20, 64, 6, 12, 1, 2, 1),        # fewer than 8 output channels: no ranges
])
def test_host_buffer_entry_matches_device_entry(n, N, K, T, F, D, NCO):
    volt = np.stack([synth.gauss_voltages(synth.GaussSpec(n, N * T * D, N, sigma=16.0, rho=0.1, seed=9 + c))
                     for c in range(NCO)])
    h = corr.MwaxCorr(n, N, K, T, F)
    dev = h.new_output(n_dumps=D, n_coarse=NCO)
    h.process_batch(torch.from_numpy(volt).cuda(), dev, D, NCO)
    hv = torch.from_numpy(volt).contiguous().pin_memory()
    hout = torch.full(dev.shape, float("nan"), dtype=torch.float32).pin_memory()
    h.process_host(hv, hout, D, NCO)
    torch.cuda.synchronize()
    assert torch.equal(hout, dev.cpu())
    h.destroy()


# ------------------------------------------------------------------------------------------------------------------
# fractional-delay / phase correction fused into the F kernels (PAPER.md 2.5.1 L266-272)
# ------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n,N,K,T,F", [
    (16, 64, 64, 12, 1),        # register kernel, every bin kept
    (20, 128, 96, 9, 4),        # register kernel, keep < fft, averaging weights
    (33, 256, 256, 5, 2),       # ragged input group, shared edge taps
    (12, 100, 100, 7, 5),       # generic Stockham kernel
    (10, 6400, 6400, 3, 50),    # the paper's mode: three-pass cluster kernel, ragged group
    (6, 6400, 5000, 2, 50),     # keep < fft at N = 6400
    (300, 128, 128, 20, 1),     # several pair tiles and ten 32-input F groups
    (40, 6400, 6400, 2, 50),    # five 8-input work items of the N = 6400 kernel
])
def test_delay_phase_correction_elementwise(n, N, K, T, F):
    rng = np.random.default_rng(100 + n + N)
    spec = synth.GaussSpec(n, N * T, N, sigma=16.0, rho=0.3, tones=[synth.Tone(min(3, K // 2 - 1), 6.0, 1)], seed=2000 + n + N)
    volt = synth.gauss_voltages(spec)
    delay = rng.uniform(-0.5, 0.5, size=(n, T)).astype(np.float32)       # a different value every frame (fringe stopping)
    phase = rng.uniform(-np.pi, np.pi, size=(n, T)).astype(np.float32)
    ref = oracle.fx(volt, N, K, T, F, delay=delay.astype(np.float64), phase=phase.astype(np.float64))
    plain = oracle.fx(volt, N, K, T, F)
    h = corr.MwaxCorr(n, N, K, T, F)
    v = torch.from_numpy(volt).cuda()
    out = h.new_output()
    h.set_delays(torch.from_numpy(delay).cuda(), torch.from_numpy(phase).cuda())
    h.process(v, out[0, 0])
    torch.cuda.synchronize()
    got = _complex(out.cpu().numpy()[0, 0])
    assert _norm_err(got, ref, n) <= TOL
    assert _norm_err(got, plain, n) > 0.05, "the correction must change the cross products"
    # delay only / phase only / off again
    h.set_delays(torch.from_numpy(delay).cuda(), None)
    h.process(v, out[0, 0])
    torch.cuda.synchronize()
    assert _norm_err(_complex(out.cpu().numpy()[0, 0]), oracle.fx(volt, N, K, T, F, delay=delay.astype(np.float64)), n) <= TOL
    h.set_delays(None, None)
    h.process(v, out[0, 0])
    torch.cuda.synchronize()
    assert _norm_err(_complex(out.cpu().numpy()[0, 0]), plain, n) <= TOL
    h.destroy()


# SURVEY.md 8(f) NEXT #1, second half: per-channel magnitude gains ("PFB de-ripple", PAPER.md 4.2 L561-567) folded
# into the F kernels' per-channel factor
@pytest.mark.parametrize("n,N,K,T,F,mode", [
    (16, 64, 64, 12, 1, 0),        # register kernel, F = 1 (the unscaled variant becomes the scaled one)
    (20, 128, 96, 9, 4, 0),        # keep < fft, centre-symmetric weights times gains
    (33, 256, 256, 5, 2, 0),       # shared edge taps (sqrt(1/2) times gain)
    (12, 100, 100, 7, 5, 1),       # generic Stockham kernel, BLOCK mode
    (10, 6400, 6400, 3, 50, 0),    # the paper's mode: the three-pass kernel leaves its 2-bit weight codes for the table
    (6, 6400, 5000, 2, 50, 0),     # keep < fft at N = 6400
    (300, 256, 256, 10, 2, 0),     # several pair tiles and ten 32-input F groups
])
def test_channel_gains_elementwise(n, N, K, T, F, mode):
    rng = np.random.default_rng(300 + n + N)
    spec = synth.GaussSpec(n, N * T, N, sigma=16.0, rho=0.3, tones=[synth.Tone(min(3, K // 2 - 1), 6.0, 1)], seed=3000 + n + N)
    volt = synth.gauss_voltages(spec)
    u = np.arange(K) - K // 2
    gain = (1.0 + 0.25 * np.cos(2 * np.pi * u / K) + 0.1 * rng.standard_normal(K)).astype(np.float32)   # a ripple's inverse
    ref = oracle.fx(volt, N, K, T, F, mode=mode, gain=gain.astype(np.float64))
    plain = oracle.fx(volt, N, K, T, F, mode=mode)
    h = corr.MwaxCorr(n, N, K, T, F, avg_mode=mode)
    v = torch.from_numpy(volt).cuda()
    out = h.new_output()
    h.set_channel_gains(gain)
    h.process(v, out[0, 0])
    torch.cuda.synchronize()
    got = _complex(out.cpu().numpy()[0, 0])
    assert _norm_err(got, ref, n) <= TOL
    assert _norm_err(got, plain, n) > 0.05, "the gains must change the visibilities"
    # together with the delay / phase correction (the paper's combined look-up table)
    delay = rng.uniform(-0.5, 0.5, size=(n, T)).astype(np.float32)
    phase = rng.uniform(-np.pi, np.pi, size=(n, T)).astype(np.float32)
    h.set_delays(torch.from_numpy(delay).cuda(), torch.from_numpy(phase).cuda())
    h.process(v, out[0, 0])
    torch.cuda.synchronize()
    both = oracle.fx(volt, N, K, T, F, mode=mode, delay=delay.astype(np.float64), phase=phase.astype(np.float64),
                     gain=gain.astype(np.float64))
    assert _norm_err(_complex(out.cpu().numpy()[0, 0]), both, n) <= TOL
    # off again: back to the plain path (and, at N = 6400, to the 2-bit weight codes)
    h.set_delays(None, None)
    h.set_channel_gains(None)
    h.process(v, out[0, 0])
    torch.cuda.synchronize()
    assert _norm_err(_complex(out.cpu().numpy()[0, 0]), plain, n) <= TOL
    # out-of-range gains are refused
    bad = gain.copy()
    bad[K // 3] = 5.0
    with pytest.raises(corr.MwaxError):
        h.set_channel_gains(bad)
    bad[K // 3] = np.nan
    with pytest.raises(corr.MwaxError):
        h.set_channel_gains(bad)
    h.destroy()


def test_delay_tables_follow_dumps_and_coarse_channels():
    n, N, T, D, NC = 8, 64, 6, 2, 2
    rng = np.random.default_rng(3)
    volt = np.stack([synth.gauss_voltages(synth.GaussSpec(n, N * T * D, N, sigma=16.0, rho=0.2, tones=[], seed=31, coarse=c))
                     for c in range(NC)])
    delay = rng.uniform(-0.5, 0.5, size=(NC, n, T * D)).astype(np.float32)
    phase = rng.uniform(-3, 3, size=(NC, n, T * D)).astype(np.float32)
    h = corr.MwaxCorr(n, N, N, T, 1)
    out = h.new_output(n_dumps=D, n_coarse=NC)
    h.set_delays(torch.from_numpy(delay).cuda(), torch.from_numpy(phase).cuda())
    h.process_batch(torch.from_numpy(volt).cuda(), out, D, NC)
    torch.cuda.synchronize()
    got = _complex(out.cpu().numpy())
    for c in range(NC):
        for d in range(D):
            ref = oracle.fx(volt[c], N, N, T, 1, dump=d, delay=delay[c].astype(np.float64), phase=phase[c].astype(np.float64))
            assert _norm_err(got[c, d], ref, n) <= TOL
    # a table shorter than the frames of the batch is refused
    short = torch.zeros((n, T), dtype=torch.float32, device="cuda")
    h.set_delays(short, None)
    with pytest.raises(corr.MwaxError):
        h.process_batch(torch.from_numpy(volt).cuda(), out, D, NC)
    h.destroy()


# ------------------------------------------------------------------------------------------------------------------
# MWAX_ORDER emitter (PAPER.md 2.7 L318-326, Figs 8-9) — index work, bit-exact
# ------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n,C", [(8, 2), (70, 5), (34, 25), (512, 128)])
def test_mwax_order_reindexing_is_bit_exact(n, C):
    """Host-made native array (not from the CUDA path) -> device re-index vs the oracle's step 7, element for element."""
    rng = np.random.default_rng(n * 1000 + C)
    B = n * (n + 1) // 2
    nat = rng.standard_normal((C, B, 2)).astype(np.float32)
    ii = np.arange(n)
    nat[:, ii * (ii + 1) // 2 + ii, 1] = 0.0                 # autos are real
    h = corr.MwaxCorr(n, C, C, 1, 1)                         # the call only uses (n, C) of the plan
    assert h.n_out == C
    nt = n // 2
    out = torch.full((nt * (nt + 1) // 2, C, 4, 2), float("nan"), dtype=torch.float32, device="cuda")
    wts = torch.zeros((nt * (nt + 1) // 2, 4), dtype=torch.float32, device="cuda")
    h.to_mwax_order(torch.from_numpy(nat).cuda(), out, wts)
    torch.cuda.synchronize()
    M, W = oracle.mwax_order(nat[..., 0].astype(np.float64) + 1j * nat[..., 1].astype(np.float64), n)
    got = out.cpu().numpy()
    assert np.array_equal(got[..., 0], M.real.astype(np.float32)) and np.array_equal(got[..., 1], M.imag.astype(np.float32))
    assert np.array_equal(wts.cpu().numpy(), W.astype(np.float32))
    h.destroy()


def test_fx_then_mwax_order_matches_oracle():
    n, N, T = 12, 64, 20
    spec = synth.GaussSpec(n, N * T, N, sigma=16.0, rho=0.3, tones=[synth.Tone(7, 5.0, 1)], seed=4242)
    volt = synth.gauss_voltages(spec)
    ref = oracle.fx(volt, N, N, T, 4)
    Mref, _ = oracle.mwax_order(ref, n)
    h = corr.MwaxCorr(n, N, N, T, 4)
    vis = h.new_output()[0, 0]
    h.process(torch.from_numpy(volt).cuda(), vis)
    out = h.to_mwax_order(vis)
    torch.cuda.synchronize()
    got = _complex(out.cpu().numpy())                        # [rows][C][4]
    A = np.array([ref[:, oracle.baseline_index(i, i)].real for i in range(n)])      # [n][C]
    row = 0
    for a in range(n // 2):
        for b in range(a, n // 2):
            for p in range(2):
                for q in range(2):
                    norm = np.sqrt(A[2 * a + p] * A[2 * b + q])
                    assert np.all(np.abs(got[row, :, 2 * p + q] - Mref[row, :, 2 * p + q]) <= TOL * norm)
            row += 1
    h.destroy()


# ------------------------------------------------------------------------------------------------------------------
# occupancy weights from zeroing flags + optional normalisation (PAPER.md 4.1 L557-559)
# ------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n,C,S", [(8, 2, 4), (70, 5, 20), (512, 128, 10)])
def test_occupancy_weights_and_normalisation(n, C, S):
    rng = np.random.default_rng(n + C + S)
    B = n * (n + 1) // 2
    nat = rng.standard_normal((C, B, 2)).astype(np.float32)
    ii = np.arange(n)
    nat[:, ii * (ii + 1) // 2 + ii, 1] = 0.0
    flags = (rng.random((n, S)) < 0.2).astype(np.uint8)
    flags[3, :] = 1                                          # a path lost for the whole integration: weight 0
    h = corr.MwaxCorr(n, C, C, 1, 1)
    nt = n // 2
    wts = torch.zeros((nt * (nt + 1) // 2, 4), dtype=torch.float32, device="cuda")
    M, _ = oracle.mwax_order(nat[..., 0].astype(np.float64) + 1j * nat[..., 1].astype(np.float64), n)
    W, Mn = oracle.occupancy(flags, M, normalise=True)
    # weights only: values stay bit copies
    out = h.to_mwax_order(torch.from_numpy(nat).cuda(), weights=wts, flags=torch.from_numpy(flags).cuda(), normalise=False)
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    assert np.array_equal(wts.cpu().numpy(), W.astype(np.float32))             # k/S in fp32 == fp32(k/S in fp64)
    assert np.array_equal(got[..., 0], M.real.astype(np.float32)) and np.array_equal(got[..., 1], M.imag.astype(np.float32))
    # normalised: one fp32 division per component
    out = h.to_mwax_order(torch.from_numpy(nat).cuda(), weights=wts, flags=torch.from_numpy(flags).cuda(), normalise=True)
    torch.cuda.synchronize()
    got = _complex(out.cpu().numpy())
    assert np.all(np.abs(got - Mn) <= 2e-7 * np.abs(Mn))
    h.destroy()


# ------------------------------------------------------------------------------------------------------------------
# streaming integration over the paper's block structure (PAPER.md 2.5 L258, 2.5.2 L280)
# ------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("n,N,F,spb,blocks", [
    (16, 64, 1, 8, 5),           # five blocks of 8 spectra
    (12, 6400, 50, 10, 3),       # the paper's shape: 50 ms blocks of 10 x 6400-point frames, fscrunch 50
])
def test_streaming_accumulation_over_blocks_equals_one_integration(n, N, F, spb, blocks):
    """Subfile-shaped input [block][input][spb*N] fed one block per call with MWAX_OPT_ACCUMULATE equals the oracle's
    single integration over all blocks (the oracle's additivity over time is pinned in test_p4_additivity_over_time)."""
    T = spb * blocks
    spec = synth.GaussSpec(n, N * T, N, sigma=16.0, rho=0.25, tones=[synth.Tone(3, 5.0, 1)], seed=555 + N)
    volt = synth.gauss_voltages(spec)                                        # [n][T*N][2]
    ref = oracle.fx(volt, N, N, T, F)
    sub = np.ascontiguousarray(volt.reshape(n, blocks, spb * N, 2).transpose(1, 0, 2, 3))   # [block][input][spb*N][2] (L258-260)
    h = corr.MwaxCorr(n, N, N, spb, F)
    vis = h.new_output()[0, 0]
    vis.fill_(float("nan"))
    dsub = torch.from_numpy(sub).cuda()
    for b in range(blocks):
        h.set_accumulate(b > 0)
        h.process(dsub[b], vis)
    torch.cuda.synchronize()
    got = _complex(vis.cpu().numpy())
    assert _norm_err(got, ref, n) <= TOL
    ii = np.arange(n)
    assert np.all(got[:, ii * (ii + 1) // 2 + ii].imag == 0.0)
    h.destroy()


@pytest.mark.parametrize("n,N,T,F", [(20, 128, 6, 1), (8, 6400, 2, 50)])
def test_misaligned_voltage_buffer_takes_the_scalar_load_path(n, N, T, F):
    """A buffer that is only 2-byte aligned (samples are 2 bytes) is legal: the plan routes it to the generic kernel
    instead of the 16-byte-load kernels; results must not change."""
    spec = synth.GaussSpec(n, N * T, N, sigma=16.0, rho=0.2, tones=[synth.Tone(3, 6.0, 1)], seed=321 + N)
    volt = synth.gauss_voltages(spec)
    ref = oracle.fx(volt, N, N, T, F)
    flat = torch.zeros(volt.size + 64, dtype=torch.int8, device="cuda")
    view = flat[2:2 + volt.size].view(n, N * T, 2)
    view.copy_(torch.from_numpy(volt))
    assert view.data_ptr() % 16 == 2 and view.is_contiguous()
    h = corr.MwaxCorr(n, N, N, T, F)
    out = h.new_output()[0, 0]
    h.process(view, out)
    torch.cuda.synchronize()
    assert _norm_err(_complex(out.cpu().numpy()), ref, n) <= TOL
    h.destroy()


def test_caller_owned_workspace_gives_the_same_result():
    n, N, T, F = 24, 128, 30, 4
    spec = synth.GaussSpec(n, N * T, N, sigma=16.0, rho=0.2, tones=[], seed=77)
    volt = synth.gauss_voltages(spec)
    ref = oracle.fx(volt, N, N, T, F)
    h = corr.MwaxCorr(n, N, N, T, F)
    ws = torch.full((h.workspace_bytes() + 512,), 0x7F, dtype=torch.uint8, device="cuda")     # garbage: must be zeroed by the call
    off = (-ws.data_ptr()) % 256
    h.set_workspace(ws[off:off + h.workspace_bytes()])
    out = h.new_output()[0, 0]
    h.process(torch.from_numpy(volt).cuda(), out)
    torch.cuda.synchronize()
    assert _norm_err(_complex(out.cpu().numpy()), ref, n) <= TOL
    with pytest.raises(corr.MwaxError):
        h.set_workspace(ws[off:off + 16])                                                      # too small
    h.destroy()


@pytest.mark.parametrize("n,N,K,T,F,runs", [
    (16, 64, 64, 80, 2, 5),        # 32 output channels in 5 uneven runs; channel 0's lower edge wraps to position K - 1
    (16, 64, 64, 64, 2, 32),       # one channel per run: every unit is INIT, ADD, OUT
    (70, 128, 96, 65, 4, 3),       # F = 4: three interior taps per channel, T one past a 64-row block, ragged inputs
    (200, 256, 256, 70, 2, 1),     # config-5 shape cut down, several pair tiles, the whole band as one run
    (8, 6400, 6400, 64, 50, 7),    # the paper's mode: 49 interior taps per channel
])
def test_shared_edge_schedule_matches_oracle(n, N, K, T, F, runs):
    """Even F, centre-symmetric averaging: the pair kernel's shared-edge schedule (each half-weight edge channel contracted
    once per run of adjacent output channels) against the oracle, and against the plain schedule."""
    spec = synth.GaussSpec(n, N * T, N, sigma=16.0, rho=0.2, tones=[synth.Tone(3, 6.0, 1)], seed=4000 + n + N + runs)
    volt = synth.gauss_voltages(spec)
    ref = oracle.fx(volt, N, K, T, F, 0)
    got = _run_fx(volt, n, N, K, T, F, 0, options=[(corr.MWAX_OPT_X_EDGE_RUNS, runs)])[0]
    plain = _run_fx(volt, n, N, K, T, F, 0, options=[(corr.MWAX_OPT_X_EDGE_RUNS, 0)])[0]
    assert not np.isnan(got.view(np.float64)).any()
    assert _norm_err(got, ref, n) <= TOL
    assert _norm_err(plain, ref, n) <= TOL
    assert _norm_err(got, plain, n) <= 1e-5        # same products, another summation order
    ii = np.arange(n)
    assert np.all(got[:, ii * (ii + 1) // 2 + ii].imag == 0.0)


def test_shared_edge_schedule_with_streaming_accumulation():
    """MWAX_OPT_ACCUMULATE under the shared-edge schedule: two blocks added equal one integration."""
    n, N, K, T, F = 16, 64, 64, 64, 2
    spec = synth.GaussSpec(n, N * 2 * T, N, sigma=16.0, rho=0.2, tones=[], seed=4242)
    volt = synth.gauss_voltages(spec)
    ref = oracle.fx(volt, N, K, 2 * T, F, 0)
    h = corr.MwaxCorr(n, N, K, T, F)
    h.set_option(corr.MWAX_OPT_X_EDGE_RUNS, 3)
    assert h.x_edge_runs() == 3
    v = torch.from_numpy(volt).cuda()
    out = h.new_output()
    out.fill_(float("nan"))
    for b in range(2):
        h.set_accumulate(b > 0)
        h.process(v[:, b * T * N:(b + 1) * T * N].contiguous(), out[0, 0])
    torch.cuda.synchronize()
    got = _complex(out.cpu().numpy()[0, 0])
    h.destroy()
    assert _norm_err(got, ref, n) <= TOL


@pytest.mark.parametrize("n,N,K,T,F", [
    (512, 128, 128, 600, 1),     # C3 kernels (pow2 F, pair X, every SM busy for several waves)
    (70, 6400, 6400, 6, 50),     # C4 kernels (three-pass F, both sub-items parked in tensor memory, stores deferred)
    (300, 256, 256, 96, 2),      # C5 kernels (shared-edge X schedule where the chooser picks it)
    (40, 320, 300, 9, 3),        # generic F kernel, one ragged pair tile
])
def test_repeated_runs_are_bit_identical_and_do_not_depend_on_earlier_calls(n, N, K, T, F):
    """The path has a fixed summation order (no atomics): the same input must give the same BITS on every launch, into
    NaN-filled outputs, also after a different input went through the same handle (stale workspace / TMEM / shared-memory
    reuse and missing barriers show up here as run-to-run differences; compute-sanitizer is not available on the GPU pool)."""
    a = synth.gauss_voltages(synth.GaussSpec(n, N * T, N, sigma=20.0, rho=0.3, tones=[], seed=4242 + n))
    b = synth.gauss_voltages(synth.GaussSpec(n, N * T, N, sigma=35.0, rho=0.0, tones=[], seed=977 + N))
    h = corr.MwaxCorr(n, N, K, T, F)
    va, vb = torch.from_numpy(a).cuda(), torch.from_numpy(b).cuda()
    outs = []
    for v in (va, va, vb, va, va, va):
        out = h.new_output()
        out.fill_(float("nan"))
        h.process(v, out[0, 0])
        outs.append(out)
    torch.cuda.synchronize()
    first = outs[0].view(torch.int32)
    assert not torch.isnan(outs[0]).any()
    for k in (1, 3, 4, 5):
        assert torch.equal(first, outs[k].view(torch.int32)), f"launch {k} differs from launch 0 on the same input"
    assert not torch.equal(first, outs[2].view(torch.int32))
    # and the repeated result is the right one (a sampled check keeps the oracle's work small at n = 512)
    sel = sorted(set([0, 1, n // 2 - 1, n // 2, n - 2, n - 1]))
    ref = oracle.fx(a[sel], N, K, T, F)
    got = _gather_sel(_complex(outs[5].cpu().numpy()[0, 0]), sel)
    assert _norm_err(got, ref, len(sel)) <= TOL
    h.destroy()
