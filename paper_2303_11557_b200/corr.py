"""Thin Python binding of the C ABI in include/mwax_corr.h (argument marshalling only).

Every step of the path runs in the CUDA kernels of libmwax_corr.so; this module converts torch tensors to raw
pointers and checks return codes.  There is no CPU fallback: if the native library is missing or cannot be
built, importing a function from here raises.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_HERE, "csrc")
_LIB = os.path.join(_HERE, "libmwax_corr.so")
_SOURCES = ["mwax_api.cu", "mwax_order.cuh", "f_stage.cuh", "f_stage_pow2.cuh", "f_stage_6400.cuh", "x_stage.cuh", "x_stage2.cuh", "ptx.cuh"]
_HEADER = os.path.join(os.path.dirname(_HERE), "include", "mwax_corr.h")
_lib = None

MWAX_OK = 0
MWAX_OPT_AVG_MODE = 1
MWAX_OPT_ACCUMULATE = 2
MWAX_OPT_DC_EXCLUDE = 3
MWAX_OPT_X_EDGE_RUNS = 4
MWAX_AVG_CENTRE_SYMMETRIC = 0
MWAX_AVG_BLOCK = 1

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared"]


class MwaxError(RuntimeError):
    pass


def _stale() -> bool:
    if not os.path.exists(_LIB):
        return True
    t = os.path.getmtime(_LIB)
    deps = [os.path.join(_CSRC, s) for s in _SOURCES] + [_HEADER]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile libmwax_corr.so in-tree for sm_100a (nvcc cross-compiles without a GPU)."""
    if force or _stale():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        tmp = _LIB + f".tmp{os.getpid()}"
        cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp, os.path.join(_CSRC, "mwax_api.cu")]
        subprocess.check_call(cmd)
        os.replace(tmp, _LIB)
    return _LIB


def lib() -> ctypes.CDLL:
    """Load the native library (building it if the sources are newer); raises if that is impossible."""
    global _lib
    if _lib is None:
        try:
            path = build()
        except Exception as e:  # no nvcc on this machine: use the shipped .so if there is one
            if not os.path.exists(_LIB):
                raise MwaxError(f"libmwax_corr.so is missing and could not be built: {e}") from e
            path = _LIB
        L = ctypes.CDLL(path)
        vp, i32, sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_size_t
        L.mwax_corr_create.restype = vp
        L.mwax_corr_create.argtypes = [i32] * 5
        L.mwax_corr_last_error.restype = i32
        L.mwax_corr_set_option.argtypes = [vp, i32, i32]
        L.mwax_corr_process.argtypes = [vp, vp, vp, vp]
        L.mwax_corr_process_batch.argtypes = [vp, vp, sz, sz, i32, i32, vp, vp]
        L.mwax_corr_process_host.argtypes = [vp, vp, sz, sz, i32, i32, vp, vp]
        L.mwax_corr_f_stage.argtypes = [vp, vp, sz, vp]
        L.mwax_corr_set_delays.argtypes = [vp, vp, vp, sz, sz]
        L.mwax_corr_set_workspace.argtypes = [vp, vp, sz]
        L.mwax_corr_x_edge_runs.argtypes = [vp]
        L.mwax_corr_set_channel_gains.argtypes = [vp, vp]
        L.mwax_corr_to_mwax_order.argtypes = [vp, vp, vp, vp, vp]
        L.mwax_corr_to_mwax_order_weighted.argtypes = [vp, vp, vp, i32, i32, vp, vp, vp]
        L.mwax_corr_mwax_order_bytes.restype = sz
        L.mwax_corr_mwax_order_bytes.argtypes = [vp]
        L.mwax_corr_x_stage.argtypes = [vp, vp, vp]
        for f in ("input_bytes", "output_bytes", "workspace_bytes"):
            getattr(L, "mwax_corr_" + f).restype = sz
            getattr(L, "mwax_corr_" + f).argtypes = [vp]
        L.mwax_corr_launch_count.restype = ctypes.c_longlong
        L.mwax_corr_launch_count.argtypes = [vp]
        L.mwax_corr_last_cuda_error.argtypes = [vp]
        L.mwax_corr_destroy.argtypes = [vp]
        L.mwax_xcorr_i8_create.restype = vp
        L.mwax_xcorr_i8_create.argtypes = [i32] * 3
        L.mwax_xcorr_i8_process.argtypes = [vp, vp, vp, vp]
        L.mwax_xcorr_i8_process_host.argtypes = [vp, vp, vp, vp]
        L.mwax_xcorr_i8_destroy.argtypes = [vp]
        L.mwax_corr_static_workspace_max.restype = sz
        L.mwax_corr_static_workspace_max.argtypes = []
        L.mwax_corr_process_static.argtypes = [vp, vp, i32, i32, i32, i32, vp]
        L.mwax_corr_strerror.restype = ctypes.c_char_p
        L.mwax_corr_strerror.argtypes = [i32]
        L.mwax_corr_version.restype = ctypes.c_char_p
        _lib = L
    return _lib


def _check(rc: int, what: str, handle=None):
    if rc != MWAX_OK:
        msg = lib().mwax_corr_strerror(rc).decode()
        extra = ""
        if handle is not None:
            extra = f" (cuda error {lib().mwax_corr_last_cuda_error(handle)})"
        raise MwaxError(f"{what}: {msg} [{rc}]{extra}")


def _stream_ptr(stream) -> int:
    if stream is None:
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream)


class MwaxCorr:
    """mwax_corr_create / process / destroy with torch tensors for device memory."""

    def __init__(self, n_inputs: int, n_fft: int, n_keep: int, t_int: int, f_avg: int, avg_mode: int | None = None):
        L = lib()
        self._h = L.mwax_corr_create(n_inputs, n_fft, n_keep, t_int, f_avg)
        if not self._h:
            rc = L.mwax_corr_last_error()
            raise MwaxError(f"mwax_corr_create: {L.mwax_corr_strerror(rc).decode()} [{rc}]")
        self.n_inputs, self.n_fft, self.n_keep, self.t_int, self.f_avg = n_inputs, n_fft, n_keep, t_int, f_avg
        self.n_out = n_keep // f_avg
        self.n_baselines = n_inputs * (n_inputs + 1) // 2
        if avg_mode is not None:
            _check(L.mwax_corr_set_option(self._h, MWAX_OPT_AVG_MODE, avg_mode), "mwax_corr_set_option")

    def set_workspace(self, ws: torch.Tensor):
        """Use a caller-owned CUDA tensor (>= workspace_bytes(), 256-byte aligned) as the fp16 spectra workspace."""
        assert ws.is_cuda and ws.is_contiguous()
        self._ws_ref = ws
        _check(lib().mwax_corr_set_workspace(self._h, ws.data_ptr(), ws.numel() * ws.element_size()), "mwax_corr_set_workspace",
               self._h)

    def x_edge_runs(self) -> int:
        """Runs per tile of the X stage's shared-edge schedule (even f_avg), 0 = plain schedule."""
        r = lib().mwax_corr_x_edge_runs(self._h)
        if r < 0:
            _check(r, "mwax_corr_x_edge_runs", self._h)
        return r

    def set_accumulate(self, on: bool):
        """Streaming integration: with True, process() adds into `vis` instead of overwriting it."""
        _check(lib().mwax_corr_set_option(self._h, MWAX_OPT_ACCUMULATE, 1 if on else 0), "mwax_corr_set_option", self._h)

    # sizes
    def input_bytes(self) -> int:
        return lib().mwax_corr_input_bytes(self._h)

    def output_bytes(self) -> int:
        return lib().mwax_corr_output_bytes(self._h)

    def workspace_bytes(self) -> int:
        return lib().mwax_corr_workspace_bytes(self._h)

    def launch_count(self) -> int:
        """Kernels this handle has enqueued since it was created."""
        return int(lib().mwax_corr_launch_count(self._h))

    def set_option(self, key: int, value: int):
        """mwax_corr_set_option: MWAX_OPT_AVG_MODE, MWAX_OPT_ACCUMULATE, MWAX_OPT_DC_EXCLUDE, MWAX_OPT_X_EDGE_RUNS."""
        _check(lib().mwax_corr_set_option(self._h, key, value), "mwax_corr_set_option", self._h)

    def new_output(self, n_dumps: int = 1, n_coarse: int = 1, device="cuda") -> torch.Tensor:
        return torch.empty((n_coarse, n_dumps, self.n_out, self.n_baselines, 2), dtype=torch.float32, device=device)

    def process(self, volt: torch.Tensor, vis: torch.Tensor, stream=None) -> torch.Tensor:
        """volt int8 cuda [n][T*N][2]; vis float32 cuda [C][B][2] (written)."""
        assert volt.is_cuda and volt.dtype == torch.int8 and volt.is_contiguous()
        assert vis.is_cuda and vis.dtype == torch.float32 and vis.is_contiguous()
        assert volt.numel() == self.input_bytes() and vis.numel() * 4 == self.output_bytes()
        _check(lib().mwax_corr_process(self._h, volt.data_ptr(), vis.data_ptr(), _stream_ptr(stream)),
               "mwax_corr_process", self._h)
        return vis

    def process_batch(self, volt: torch.Tensor, vis: torch.Tensor, n_dumps: int, n_coarse: int = 1, stream=None):
        """volt int8 cuda [n_coarse][n][row_pitch][2]; vis float32 cuda [n_coarse][n_dumps][C][B][2]."""
        assert volt.is_cuda and volt.dtype == torch.int8 and volt.is_contiguous() and volt.dim() == 4
        assert vis.is_cuda and vis.dtype == torch.float32 and vis.is_contiguous()
        assert volt.shape[0] == n_coarse and volt.shape[1] == self.n_inputs
        row_pitch = volt.shape[2]
        assert vis.numel() * 4 == self.output_bytes() * n_dumps * n_coarse
        _check(lib().mwax_corr_process_batch(self._h, volt.data_ptr(), row_pitch, row_pitch * self.n_inputs, n_dumps,
                                             n_coarse, vis.data_ptr(), _stream_ptr(stream)),
               "mwax_corr_process_batch", self._h)
        return vis

    def process_host(self, volt: torch.Tensor, vis: torch.Tensor, n_dumps: int, n_coarse: int = 1, stream=None):
        """Host (ideally pinned) tensors in and out; H2D and D2H copies happen inside the call."""
        assert (not volt.is_cuda) and volt.dtype == torch.int8 and volt.is_contiguous() and volt.dim() == 4
        assert (not vis.is_cuda) and vis.dtype == torch.float32 and vis.is_contiguous()
        row_pitch = volt.shape[2]
        assert vis.numel() * 4 == self.output_bytes() * n_dumps * n_coarse
        _check(lib().mwax_corr_process_host(self._h, volt.data_ptr(), row_pitch, row_pitch * self.n_inputs, n_dumps,
                                            n_coarse, vis.data_ptr(), _stream_ptr(stream)),
               "mwax_corr_process_host", self._h)
        return vis

    def set_delays(self, delay: torch.Tensor | None, phase: torch.Tensor | None):
        """delay (samples) / phase (radians): float32 cuda [n][frames] or [n_coarse][n][frames]; None = zeros; both
        None switches the correction off.  The tensors are kept alive by this object."""
        ref = delay if delay is not None else phase
        if ref is None:
            self._delay_refs = None
            _check(lib().mwax_corr_set_delays(self._h, None, None, 0, 0), "mwax_corr_set_delays", self._h)
            return
        for t in (delay, phase):
            assert t is None or (t.is_cuda and t.dtype == torch.float32 and t.is_contiguous() and t.shape == ref.shape)
        assert ref.dim() in (2, 3) and ref.shape[-2] == self.n_inputs
        row_stride = ref.shape[-1]
        self._delay_refs = (delay, phase)
        _check(lib().mwax_corr_set_delays(self._h, delay.data_ptr() if delay is not None else None,
                                          phase.data_ptr() if phase is not None else None, row_stride,
                                          row_stride * self.n_inputs), "mwax_corr_set_delays", self._h)

    def set_channel_gains(self, gain):
        """gain: float32 host array-like [n_keep] of per-channel magnitudes in [0, 4] (PFB de-ripple, PAPER.md 4.2);
        None switches them off.  The library copies the values."""
        if gain is None:
            _check(lib().mwax_corr_set_channel_gains(self._h, None), "mwax_corr_set_channel_gains", self._h)
            return
        g = torch.as_tensor(gain, dtype=torch.float32, device="cpu").contiguous()
        assert g.numel() == self.n_keep
        _check(lib().mwax_corr_set_channel_gains(self._h, g.data_ptr()), "mwax_corr_set_channel_gains", self._h)

    def to_mwax_order(self, vis: torch.Tensor, out: torch.Tensor | None = None, weights: torch.Tensor | None = None,
                      stream=None, flags: torch.Tensor | None = None, normalise: bool = False):
        """vis float32 cuda [C][B][2] (one dump) -> out float32 cuda [n_tiles(n_tiles+1)/2][C][4][2] (+ weights [..][4])."""
        assert vis.is_cuda and vis.dtype == torch.float32 and vis.is_contiguous() and vis.numel() * 4 == self.output_bytes()
        nt = self.n_inputs // 2
        if out is None:
            out = torch.empty((nt * (nt + 1) // 2, self.n_out, 4, 2), dtype=torch.float32, device=vis.device)
        assert out.is_cuda and out.dtype == torch.float32 and out.is_contiguous()
        assert out.numel() * 4 == lib().mwax_corr_mwax_order_bytes(self._h)
        if weights is not None:
            assert weights.is_cuda and weights.dtype == torch.float32 and weights.numel() == nt * (nt + 1) // 2 * 4
        n_sub = 0
        if flags is not None:
            assert flags.is_cuda and flags.dtype == torch.uint8 and flags.is_contiguous() and flags.shape[0] == self.n_inputs
            n_sub = flags.shape[1]
        _check(lib().mwax_corr_to_mwax_order_weighted(self._h, vis.data_ptr(), flags.data_ptr() if flags is not None else None,
                                                      n_sub, 1 if normalise else 0, out.data_ptr(),
                                                      weights.data_ptr() if weights is not None else None,
                                                      _stream_ptr(stream)), "mwax_corr_to_mwax_order_weighted", self._h)
        return out

    def f_stage(self, volt: torch.Tensor, row_pitch: int | None = None, stream=None):
        assert volt.is_cuda and volt.dtype == torch.int8 and volt.is_contiguous()
        if row_pitch is None:
            row_pitch = self.t_int * self.n_fft
        _check(lib().mwax_corr_f_stage(self._h, volt.data_ptr(), row_pitch, _stream_ptr(stream)), "mwax_corr_f_stage",
               self._h)

    def x_stage(self, vis: torch.Tensor, stream=None):
        assert vis.is_cuda and vis.dtype == torch.float32 and vis.is_contiguous()
        _check(lib().mwax_corr_x_stage(self._h, vis.data_ptr(), _stream_ptr(stream)), "mwax_corr_x_stage", self._h)

    def destroy(self):
        if getattr(self, "_h", None):
            lib().mwax_corr_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def static_workspace_max() -> int:
    """Bytes of fp16 spectra (n_fft * t_int * roundup(2 n_inputs, 64) * 2) that process_static() can hold."""
    return int(lib().mwax_corr_static_workspace_max())


def process_static(volt: torch.Tensor, vis: torch.Tensor, n_inputs: int, n_fft: int, t_int: int, f_avg: int, stream=None):
    """mwax_corr_process_static: one integration without a handle and without any device allocation inside the library
    (its scratch is a static device array; calls that overlap on the GPU race).  volt int8 cuda [n][T*N][2]; vis float32
    cuda [N/F][n(n+1)/2][2] (written).  Raises MwaxError (MWAX_ERR_TOO_LARGE) beyond static_workspace_max()."""
    assert volt.is_cuda and volt.dtype == torch.int8 and volt.is_contiguous()
    assert vis.is_cuda and vis.dtype == torch.float32 and vis.is_contiguous()
    assert volt.numel() == n_inputs * t_int * n_fft * 2
    assert f_avg >= 1 and vis.numel() == (n_fft // f_avg) * (n_inputs * (n_inputs + 1) // 2) * 2
    _check(lib().mwax_corr_process_static(volt.data_ptr(), vis.data_ptr(), n_inputs, n_fft, t_int, f_avg, _stream_ptr(stream)),
           "mwax_corr_process_static")
    return vis


class MwaxXcorrI8:
    """mwax_xcorr_i8_create / process / destroy: exact integer X stage on pre-channelised int8 samples."""

    def __init__(self, n_inputs: int, n_chan: int, n_time: int):
        L = lib()
        self._h = L.mwax_xcorr_i8_create(n_inputs, n_chan, n_time)
        if not self._h:
            rc = L.mwax_corr_last_error()
            raise MwaxError(f"mwax_xcorr_i8_create: {L.mwax_corr_strerror(rc).decode()} [{rc}]")
        self.n_inputs, self.n_chan, self.n_time = n_inputs, n_chan, n_time
        self.n_baselines = n_inputs * (n_inputs + 1) // 2

    def new_output(self, device="cuda") -> torch.Tensor:
        return torch.empty((self.n_chan, self.n_baselines, 2), dtype=torch.int32, device=device)

    def process(self, z: torch.Tensor, vis: torch.Tensor, stream=None) -> torch.Tensor:
        assert z.is_cuda and z.dtype == torch.int8 and z.is_contiguous()
        assert z.numel() == self.n_chan * self.n_time * self.n_inputs * 2
        assert vis.is_cuda and vis.dtype == torch.int32 and vis.is_contiguous()
        assert vis.numel() == self.n_chan * self.n_baselines * 2
        _check(lib().mwax_xcorr_i8_process(self._h, z.data_ptr(), vis.data_ptr(), _stream_ptr(stream)),
               "mwax_xcorr_i8_process")
        return vis

    def process_host(self, z: torch.Tensor, vis: torch.Tensor, stream=None) -> torch.Tensor:
        assert (not z.is_cuda) and z.dtype == torch.int8 and z.is_contiguous()
        assert (not vis.is_cuda) and vis.dtype == torch.int32 and vis.is_contiguous()
        _check(lib().mwax_xcorr_i8_process_host(self._h, z.data_ptr(), vis.data_ptr(), _stream_ptr(stream)),
               "mwax_xcorr_i8_process_host")
        return vis

    def destroy(self):
        if getattr(self, "_h", None):
            lib().mwax_xcorr_i8_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass
