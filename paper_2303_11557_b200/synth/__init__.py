"""Seeded synthetic MWA-like voltages (generator only — none of the correlator's arithmetic lives here).

Stand-in for the paper's telescope subfiles, which are not available; recipe in
DESIGN.md §4.  The C source `mwax_synth.c` is compiled in-tree with gcc on first use.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass, field

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mwax_synth.c")
_LIB = os.path.join(_HERE, "libmwax_synth.so")
_lib = None

BASE_SEED = 0x4D574158  # "MWAX"


def build(force: bool = False) -> str:
    """Compile libmwax_synth.so next to its source (gcc, OpenMP)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O3", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        i8p = ctypes.POINTER(ctypes.c_int8)
        lib.mwax_synth_gauss.restype = None
        lib.mwax_synth_gauss.argtypes = [
            ctypes.c_uint64, ctypes.c_uint32, ctypes.c_int, ctypes.c_int, ctypes.c_int,
            ctypes.c_int64, ctypes.c_int64, ctypes.c_int64, ctypes.c_double, ctypes.c_double,
            ctypes.c_int, ctypes.POINTER(ctypes.c_int), ctypes.POINTER(ctypes.c_double),
            ctypes.POINTER(ctypes.c_int), ctypes.c_int, i8p]
        lib.mwax_synth_uniform.restype = None
        lib.mwax_synth_uniform.argtypes = [ctypes.c_uint64, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                           ctypes.c_int, i8p]
        _lib = lib
    return _lib


@dataclass
class Tone:
    bin: int          # signed DFT bin k (for frame length n_fft)
    amp: float        # amplitude per component
    phase_mult: int   # phase of input i = 2*pi*phase_mult*i/n_inputs


@dataclass
class GaussSpec:
    """One coarse channel of Gaussian voltages, layout [input][time][re,im] int8."""
    n_inputs: int
    n_samples: int            # per input
    n_fft: int                # frame length the tone bins refer to
    sigma: float = 16.0
    rho: float = 0.0
    tones: list = field(default_factory=list)
    seed: int = BASE_SEED
    coarse: int = 0


def gauss_voltages(spec: GaussSpec, out: np.ndarray | None = None, inputs: tuple[int, int] | None = None,
                   samples: tuple[int, int] | None = None) -> np.ndarray:
    """Fill (or allocate) an int8 array [n_gen][n_samp][2]; `inputs`/`samples` select a sub-range."""
    i0, i1 = inputs if inputs is not None else (0, spec.n_inputs)
    s0, s1 = samples if samples is not None else (0, spec.n_samples)
    n_gen, n_samp = i1 - i0, s1 - s0
    if out is None:
        out = np.empty((n_gen, n_samp, 2), dtype=np.int8)
    assert out.dtype == np.int8 and out.flags.c_contiguous and out.shape == (n_gen, n_samp, 2)
    nt = len(spec.tones)
    bins = (ctypes.c_int * max(nt, 1))(*[t.bin for t in spec.tones])
    amps = (ctypes.c_double * max(nt, 1))(*[t.amp for t in spec.tones])
    mults = (ctypes.c_int * max(nt, 1))(*[t.phase_mult for t in spec.tones])
    _load().mwax_synth_gauss(spec.seed, spec.coarse, i0, n_gen, spec.n_inputs, s0, n_samp, n_samp,
                             spec.sigma, spec.rho, nt, bins, amps, mults, spec.n_fft,
                             out.ctypes.data_as(ctypes.POINTER(ctypes.c_int8)))
    return out


def uniform_voltages(n_chan: int, n_time: int, n_inputs: int, n_shared: int = 64, seed: int = BASE_SEED + 1,
                     out: np.ndarray | None = None) -> np.ndarray:
    """Pre-channelised integer samples [chan][time][input][re,im] int8 (BASELINE.json configs[1])."""
    if out is None:
        out = np.empty((n_chan, n_time, n_inputs, 2), dtype=np.int8)
    assert out.dtype == np.int8 and out.flags.c_contiguous and out.shape == (n_chan, n_time, n_inputs, 2)
    _load().mwax_synth_uniform(seed, n_chan, n_time, n_inputs, n_shared,
                               out.ctypes.data_as(ctypes.POINTER(ctypes.c_int8)))
    return out


# ---------------------------------------------------------------------------------------------------
# BASELINE.json configs (shapes and value recipes)
# ---------------------------------------------------------------------------------------------------
@dataclass
class FxConfig:
    name: str
    n_inputs: int
    n_fft: int
    n_keep: int
    t_int: int
    f_avg: int
    n_dumps: int
    n_coarse: int
    sigma: float
    rho: float
    tones: list
    seed: int

    @property
    def samples_per_input(self) -> int:
        return self.n_fft * self.t_int * self.n_dumps

    @property
    def seconds_of_data(self) -> float:
        return self.samples_per_input / 1.28e6

    def spec(self, coarse: int = 0) -> GaussSpec:
        return GaussSpec(self.n_inputs, self.samples_per_input, self.n_fft, self.sigma, self.rho, self.tones,
                         self.seed, coarse)


CONFIGS = {
    # C1: 16 inputs, N=64, 256 spectra, common signal rho=0.3, tone at bin +5 with phase 2*pi*j/16
    "C1": FxConfig("C1-tiny", 16, 64, 64, 256, 1, 1, 1, 16.0, 0.3, [Tone(5, 8.0, 1)], BASE_SEED + 0),
    # C3: 512 inputs, N=128, 0.5 s integrations (5000 spectra), 1 s of data
    "C3": FxConfig("C3-10kHz", 512, 128, 128, 5000, 1, 2, 1, 16.0, 0.05,
                   [Tone(5, 4.0, 1), Tone(-37, 8.0, 3), Tone(60, 2.0, 7)], BASE_SEED + 2),
    # C4: 512 inputs, N=6400, 1 s integrations (200 spectra), fscrunch 50, 2 s of data; tones: inside a
    # channel, exactly on an output-channel boundary (u = 25 + 50*3 = 175), and at DC (must vanish)
    "C4": FxConfig("C4-highres", 512, 6400, 6400, 200, 50, 2, 1, 16.0, 0.05,
                   [Tone(1010, 4.0, 1), Tone(175, 8.0, 3), Tone(0, 10.0, 0), Tone(-1607, 2.0, 7)], BASE_SEED + 3),
    # C5: 1024 inputs, 8 coarse channels, N=256, 0.25 s integrations (1250 spectra), fscrunch 2, 0.5 s of data
    "C5": FxConfig("C5-batch", 1024, 256, 256, 1250, 2, 2, 8, 16.0, 0.02, [], BASE_SEED + 4),
}
