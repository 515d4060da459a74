"""ctypes wrapper of the float64 CPU oracle (oracle/mwax_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
--impl reference legs.  Nothing under paper_2303_11557_b200/ imports it, and it imports nothing from there.
All arithmetic is in the C file; this module only marshals numpy arrays.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mwax_oracle.c")
_LIB = os.path.join(_HERE, "libmwax_oracle.so")
_lib = None

AVG_CENTRE_SYMMETRIC = 0
AVG_BLOCK = 1
AVG_KEEP_DC = 2   # flag on the centre-symmetric mode: the DC ultra-fine channel is NOT excluded (PAPER.md L290-294 left out)


def build(force: bool = False) -> str:
    """gcc -O2 (no fast-math) -fopenmp; building the checker is not using it."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-std=c99", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int)
        i8p = ctypes.POINTER(ctypes.c_int8)
        i32p = ctypes.POINTER(ctypes.c_int32)
        lib.mwax_oracle_dft_naive.argtypes = [ctypes.c_int, dp, dp]
        lib.mwax_oracle_fft.argtypes = [ctypes.c_int, dp, dp]
        lib.mwax_oracle_weights.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, dp]
        lib.mwax_oracle_spectra.argtypes = [ctypes.c_int, ip, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                            i8p, ctypes.c_int64, dp]
        lib.mwax_oracle_correlate.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, dp, dp]
        lib.mwax_oracle_average.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, dp, dp]
        lib.mwax_oracle_fx.argtypes = [ctypes.c_int, ip, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                       ctypes.c_int, ctypes.c_int, i8p, ctypes.c_int64, dp]
        lib.mwax_oracle_apply_delays.argtypes = [ctypes.c_int, ip, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                                 dp, dp, ctypes.c_int64, dp]
        lib.mwax_oracle_fx_delay.argtypes = [ctypes.c_int, ip, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                             ctypes.c_int, ctypes.c_int, i8p, ctypes.c_int64, dp, dp, ctypes.c_int64, dp]
        lib.mwax_oracle_apply_channel_gains.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, dp, dp]
        lib.mwax_oracle_fx_gain.argtypes = [ctypes.c_int, ip, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                            ctypes.c_int, ctypes.c_int, i8p, ctypes.c_int64, dp, dp, ctypes.c_int64, dp, dp]
        lib.mwax_oracle_mwax_order.argtypes = [ctypes.c_int, ctypes.c_int, dp, dp, dp]
        lib.mwax_oracle_occupancy.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.POINTER(ctypes.c_uint8), ctypes.c_int,
                                              ctypes.c_int, dp, dp]
        lib.mwax_oracle_xcorr_i8.argtypes = [ctypes.c_int, ip, ctypes.c_int, ctypes.c_int, ctypes.c_int, i8p, i32p]
        lib.mwax_oracle_threads.argtypes = []
        lib.mwax_oracle_set_threads.argtypes = [ctypes.c_int]
        lib.mwax_oracle_set_threads.restype = None
        _lib = lib
    return _lib


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _check(rc, what):
    if rc != 0:
        raise RuntimeError(f"oracle {what} failed with code {rc}")


def _sel(sel, n_inputs):
    s = np.ascontiguousarray(np.arange(n_inputs) if sel is None else sel, dtype=np.int32)
    return s, s.ctypes.data_as(ctypes.POINTER(ctypes.c_int))


def threads() -> int:
    return int(_load().mwax_oracle_threads())


def set_threads(n: int) -> None:
    """OpenMP threads of the following calls (timing infrastructure: bench.py's single-thread run of config C1)."""
    _load().mwax_oracle_set_threads(int(n))


def dft_naive(x: np.ndarray) -> np.ndarray:
    x = np.ascontiguousarray(x, dtype=np.complex128)
    out = np.empty_like(x)
    _check(_load().mwax_oracle_dft_naive(x.size, _dp(x.view(np.float64)), _dp(out.view(np.float64))), "dft_naive")
    return out


def fft(x: np.ndarray) -> np.ndarray:
    x = np.ascontiguousarray(x, dtype=np.complex128)
    out = np.empty_like(x)
    _check(_load().mwax_oracle_fft(x.size, _dp(x.view(np.float64)), _dp(out.view(np.float64))), "fft")
    return out


def weights(K: int, F: int, mode: int = AVG_CENTRE_SYMMETRIC) -> np.ndarray:
    W = np.empty((K // F, K), dtype=np.float64)
    _check(_load().mwax_oracle_weights(K, F, mode, _dp(W)), "weights")
    return W


def spectra(volt: np.ndarray, N: int, K: int, T: int, dump: int = 0, sel=None) -> np.ndarray:
    """volt int8 [n][samples][2] -> Y complex128 [K][T][n_sel] (steps 1-3)."""
    assert volt.dtype == np.int8 and volt.ndim == 3 and volt.shape[2] == 2 and volt.flags.c_contiguous
    assert volt.shape[1] >= (dump + 1) * T * N
    s, sp = _sel(sel, volt.shape[0])
    Y = np.empty((K, T, s.size), dtype=np.complex128)
    _check(_load().mwax_oracle_spectra(s.size, sp, N, K, T, dump, volt.ctypes.data_as(ctypes.POINTER(ctypes.c_int8)),
                                       volt.shape[1], _dp(Y.view(np.float64))), "spectra")
    return Y


def correlate(Y: np.ndarray) -> np.ndarray:
    """Y complex128 [K][T][n] -> R complex128 [K][n(n+1)/2] (step 4)."""
    Y = np.ascontiguousarray(Y, dtype=np.complex128)
    K, T, n = Y.shape
    R = np.empty((K, n * (n + 1) // 2), dtype=np.complex128)
    _check(_load().mwax_oracle_correlate(n, K, T, _dp(Y.view(np.float64)), _dp(R.view(np.float64))), "correlate")
    return R


def average(R: np.ndarray, n: int, F: int, mode: int = AVG_CENTRE_SYMMETRIC) -> np.ndarray:
    """R complex128 [K][B] -> V complex128 [K/F][B] (steps 5-6)."""
    R = np.ascontiguousarray(R, dtype=np.complex128)
    K, B = R.shape
    assert B == n * (n + 1) // 2
    V = np.empty((K // F, B), dtype=np.complex128)
    _check(_load().mwax_oracle_average(n, K, F, mode, _dp(R.view(np.float64)), _dp(V.view(np.float64))), "average")
    return V


def _tab(a, n_inputs):
    if a is None:
        return None, None
    a = np.ascontiguousarray(a, dtype=np.float64)
    assert a.ndim == 2 and a.shape[0] == n_inputs
    return a, _dp(a)


def apply_delays(Y: np.ndarray, N: int, delay=None, phase=None, dump: int = 0, sel=None, n_inputs=None) -> np.ndarray:
    """Step 3b: Y complex128 [K][T][n_sel] times exp(i (phase - 2 pi u delay / N)); tables [n_inputs][frames]."""
    Y = np.array(Y, dtype=np.complex128, order="C")
    K, T, n_sel = Y.shape
    n_inputs = n_inputs if n_inputs is not None else (delay if delay is not None else phase).shape[0]
    s, sp = _sel(sel, n_inputs)
    assert s.size == n_sel
    d, dpp = _tab(delay, n_inputs)
    ph, php = _tab(phase, n_inputs)
    stride = (d if d is not None else ph).shape[1]
    assert stride >= (dump + 1) * T and (d is None or ph is None or d.shape == ph.shape)
    _check(_load().mwax_oracle_apply_delays(n_sel, sp, N, K, T, dump, dpp, php, stride, _dp(Y.view(np.float64))),
           "apply_delays")
    return Y


def apply_channel_gains(Y: np.ndarray, gain) -> np.ndarray:
    """Step 3c: Y complex128 [K][T][n_sel] times the real per-channel magnitude gain[K] (PFB de-ripple)."""
    Y = np.array(Y, dtype=np.complex128, order="C")
    K, T, n_sel = Y.shape
    g = np.ascontiguousarray(gain, dtype=np.float64)
    assert g.shape == (K,)
    _check(_load().mwax_oracle_apply_channel_gains(n_sel, K, T, _dp(g), _dp(Y.view(np.float64))), "apply_channel_gains")
    return Y


def fx(volt: np.ndarray, N: int, K: int, T: int, F: int, mode: int = AVG_CENTRE_SYMMETRIC, dump: int = 0,
       sel=None, delay=None, phase=None, gain=None) -> np.ndarray:
    """Whole float path, one dump: int8 [n][samples][2] -> V complex128 [K/F][n_sel(n_sel+1)/2].
    delay / phase: optional [n][frames] tables of the fractional-delay correction (step 3b);
    gain: optional [K] per-channel magnitudes (step 3c)."""
    assert volt.dtype == np.int8 and volt.ndim == 3 and volt.shape[2] == 2 and volt.flags.c_contiguous
    assert volt.shape[1] >= (dump + 1) * T * N
    s, sp = _sel(sel, volt.shape[0])
    V = np.empty((K // F, s.size * (s.size + 1) // 2), dtype=np.complex128)
    d, dpp = _tab(delay, volt.shape[0])
    ph, php = _tab(phase, volt.shape[0])
    stride = 0
    if d is not None or ph is not None:
        stride = (d if d is not None else ph).shape[1]
        assert stride >= (dump + 1) * T and (d is None or ph is None or d.shape == ph.shape)
    g = None
    if gain is not None:
        g = np.ascontiguousarray(gain, dtype=np.float64)
        assert g.shape == (K,)
    _check(_load().mwax_oracle_fx_gain(s.size, sp, N, K, T, F, mode, dump,
                                       volt.ctypes.data_as(ctypes.POINTER(ctypes.c_int8)), volt.shape[1],
                                       dpp, php, stride, _dp(g) if g is not None else None,
                                       _dp(V.view(np.float64))), "fx")
    return V


def mwax_order(V: np.ndarray, n_inputs: int):
    """Step 7: native V complex128 [C][n(n+1)/2] -> (M complex128 [n_tiles(n_tiles+1)/2][C][4], W float64 [..][4])."""
    V = np.ascontiguousarray(V, dtype=np.complex128)
    C, B = V.shape
    assert n_inputs % 2 == 0 and B == n_inputs * (n_inputs + 1) // 2
    nt = n_inputs // 2
    M = np.empty((nt * (nt + 1) // 2, C, 4), dtype=np.complex128)
    W = np.empty((nt * (nt + 1) // 2, 4), dtype=np.float64)
    _check(_load().mwax_oracle_mwax_order(nt, C, _dp(V.view(np.float64)), _dp(M.view(np.float64)), _dp(W)), "mwax_order")
    return M, W


def occupancy(flags: np.ndarray, M: np.ndarray | None = None, normalise: bool = False):
    """Step 8: zeroing flags uint8 [n][S] (1 = zeroed) -> weights float64 [n_tiles(n_tiles+1)/2][4]; with M (MWAX_ORDER,
    complex128 [rows][C][4]) and normalise=True also returns M divided by its weights."""
    flags = np.ascontiguousarray(flags, dtype=np.uint8)
    n, S = flags.shape
    assert n % 2 == 0
    nt = n // 2
    W = np.empty((nt * (nt + 1) // 2, 4), dtype=np.float64)
    Mo, C, mp = None, 0, None
    if M is not None:
        Mo = np.array(M, dtype=np.complex128, order="C")
        C = Mo.shape[1]
        mp = _dp(Mo.view(np.float64))
    _check(_load().mwax_oracle_occupancy(nt, S, flags.ctypes.data_as(ctypes.POINTER(ctypes.c_uint8)), C,
                                         1 if normalise else 0, _dp(W), mp), "occupancy")
    return (W, Mo) if M is not None else W


def xcorr_i8(z: np.ndarray, sel=None) -> np.ndarray:
    """z int8 [chan][time][input][2] -> int32 [chan][n_sel(n_sel+1)/2][2], exact."""
    assert z.dtype == np.int8 and z.ndim == 4 and z.shape[3] == 2 and z.flags.c_contiguous
    n_chan, n_time, n_inputs, _ = z.shape
    s, sp = _sel(sel, n_inputs)
    vis = np.empty((n_chan, s.size * (s.size + 1) // 2, 2), dtype=np.int32)
    _check(_load().mwax_oracle_xcorr_i8(s.size, sp, n_inputs, n_chan, n_time,
                                        z.ctypes.data_as(ctypes.POINTER(ctypes.c_int8)),
                                        vis.ctypes.data_as(ctypes.POINTER(ctypes.c_int32))), "xcorr_i8")
    return vis


def baseline_index(i: int, j: int) -> int:
    """Packed lower-triangle index of pair (i >= j)."""
    assert i >= j >= 0
    return i * (i + 1) // 2 + j
