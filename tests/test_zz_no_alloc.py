"""mwax_corr_process_static: the allocation-free entry point (static device scratch) against the handle path.

Collected last on purpose (the suite runs with `pytest -x`).  The reference here is mwax_corr_create + mwax_corr_process,
which tests/test_parity_gpu.py holds to the oracle; the bar is the same one, |dV| <= 2e-3 sqrt(A_i A_j) per visibility.
Consecutive calls use DIFFERENT shapes, with and without pad columns, so that what one call leaves in the shared array
lies where the next one needs zeros.
"""
import numpy as np
import pytest
import torch

from paper_2303_11557_b200 import corr, synth

pytestmark = pytest.mark.gpu

TOL = 2e-3

# (n_inputs, n_fft, t_int, f_avg): pad columns (2n % 64 != 0) / none, every register kernel, with and without averaging
SHAPES = [(48, 128, 96, 2), (20, 64, 40, 1), (64, 256, 33, 4), (130, 512, 17, 8), (48, 128, 96, 2)]


def _volt(n, N, T, seed):
    return synth.gauss_voltages(synth.GaussSpec(n, N * T, N, sigma=16.0, rho=0.2, tones=[], seed=seed))


def _handle_path(volt, n, N, T, F):
    h = corr.MwaxCorr(n, N, N, T, F)
    out = h.new_output()
    out.fill_(float("nan"))
    h.process(torch.from_numpy(volt).cuda(), out[0, 0])
    torch.cuda.synchronize()
    ref = out[0, 0].cpu().numpy().astype(np.float64)
    h.destroy()
    return ref


def _norm_err(got, ref, n):
    """max |got - ref| / sqrt(A_i A_j), A = the reference's autocorrelations in the same channel"""
    g = got[..., 0] + 1j * got[..., 1]
    r = ref[..., 0] + 1j * ref[..., 1]
    ii, jj = np.tril_indices(n)
    i = np.arange(n)
    A = r[:, i * (i + 1) // 2 + i].real                                        # [C][n]
    norm = np.sqrt(A[:, ii] * A[:, jj])
    d = np.abs(g - r)
    assert np.all(d[norm == 0] == 0)
    return float(np.where(norm > 0, d / np.where(norm > 0, norm, 1.0), 0.0).max())


def test_static_entry_matches_the_handle_path_on_consecutive_calls():
    refs, volts, outs = [], [], []
    for q, (n, N, T, F) in enumerate(SHAPES):
        v = _volt(n, N, T, seed=4100 + q)
        refs.append(_handle_path(v, n, N, T, F))
        volts.append(torch.from_numpy(v).cuda())
        outs.append(torch.full((N // F, n * (n + 1) // 2, 2), float("nan"), dtype=torch.float32, device="cuda"))
    # calls in a row on one stream, nothing in between; then the same sequence again with the outputs re-poisoned
    for rep in range(2):
        for o in outs:
            o.fill_(float("nan"))
        torch.cuda.synchronize()
        if rep == 1:
            free_before = torch.cuda.mem_get_info()[0]
        for (n, N, T, F), v, o in zip(SHAPES, volts, outs):
            corr.process_static(v, o, n, N, T, F)
        torch.cuda.synchronize()
        if rep == 1:
            assert torch.cuda.mem_get_info()[0] == free_before, "device memory was allocated during the calls"
        for (n, N, T, F), o, ref in zip(SHAPES, outs, refs):
            got = o.cpu().numpy().astype(np.float64)
            assert np.isfinite(got).all()
            err = _norm_err(got, ref, n)
            assert err <= TOL, f"shape {(n, N, T, F)} call round {rep}: normalised error {err:.3e}"


def test_static_entry_rejects_what_does_not_fit():
    n, N, F = 128, 128, 1
    limit = corr.static_workspace_max()
    assert limit == 32 * 1024 * 1024
    t_fit = limit // (N * 2 * n * 2)                                            # 512 spectra: exactly the limit
    L = corr.lib()
    v = torch.zeros((n, (t_fit + 1) * N, 2), dtype=torch.int8, device="cuda")
    o = torch.zeros((N, n * (n + 1) // 2, 2), dtype=torch.float32, device="cuda")
    rc = L.mwax_corr_process_static(v.data_ptr(), o.data_ptr(), n, N, t_fit + 1, F, None)
    assert rc == -7 and b"static workspace" in L.mwax_corr_strerror(rc)
    with pytest.raises(corr.MwaxError):
        corr.process_static(v, o, n, N, t_fit + 1, F)
    # the largest problem that fits runs, and equals the handle path
    volt = _volt(n, N, t_fit, seed=4200)
    ref = _handle_path(volt, n, N, t_fit, F)
    o.fill_(float("nan"))
    corr.process_static(torch.from_numpy(volt).cuda(), o, n, N, t_fit, F)
    torch.cuda.synchronize()
    assert _norm_err(o.cpu().numpy().astype(np.float64), ref, n) <= TOL
    # unsupported lengths and misaligned input are refused before anything is enqueued
    assert L.mwax_corr_process_static(v.data_ptr(), o.data_ptr(), n, 6400, 1, 1, None) == -3
    assert L.mwax_corr_process_static(v.data_ptr() + 2, o.data_ptr(), n, N, 4, 1, None) == -2
