"""Thin ctypes binding of libpcal (include/pcal.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind the C ABI; PyTorch is used for device
memory (``tensor.data_ptr()``) and streams (``torch.cuda.current_stream().cuda_stream``) only.
There is no fallback: if the shared library is missing or CUDA is unavailable, calls raise.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpcal.so")
_SRC_DIR = os.path.join(_HERE, "csrc")
_INCLUDE_DIR = os.path.join(os.path.dirname(_HERE), "include")

PCAL_OK = 0
ENC_OFFSET_BINARY, ENC_SIGN_MAG, ENC_TWOS_COMPLEMENT, ENC_IEEE_FLOAT = 0, 1, 2, 3
ROT_AUTO, ROT_LUT, ROT_GENERATOR = 0, 1, 2
MAX_CHANNELS = 16

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC"]


class PcalError(RuntimeError):
    def __init__(self, code: int, what: str):
        super().__init__(f"{what}: {_strerror(code)} ({code})")
        self.code = code


class InfoT(ctypes.Structure):
    _fields_ = [("n_channels", ctypes.c_int32), ("n_bins", ctypes.c_int32), ("bits", ctypes.c_int32),
                ("encoding", ctypes.c_int32), ("rotator_requested", ctypes.c_int32),
                ("rotator_in_effect", ctypes.c_int32), ("integer_exact", ctypes.c_int32),
                ("k_shift", ctypes.c_int32), ("n_processed", ctypes.c_uint64),
                ("fold_period", ctypes.c_uint64), ("lut_len", ctypes.c_uint64 * MAX_CHANNELS),
                ("kernel_launches", ctypes.c_uint64)]


def _sources():
    return sorted(os.path.join(_SRC_DIR, f) for f in os.listdir(_SRC_DIR)) + \
        sorted(os.path.join(_INCLUDE_DIR, f) for f in os.listdir(_INCLUDE_DIR))


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile libpcal.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
    stale = force or not os.path.exists(LIB_PATH) or any(
        os.path.getmtime(s) > os.path.getmtime(LIB_PATH) for s in _sources())
    if stale:
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + \
              ["-o", LIB_PATH, os.path.join(_SRC_DIR, "pcal_api.cu"), os.path.join(_SRC_DIR, "pcal_probe.cu")]
        subprocess.check_call(cmd)
    return LIB_PATH


_lib = None


def lib():
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: run `python -c 'import __graft_entry__ as g; g.build()'`; "
                               "there is no CPU fallback")
        L = ctypes.CDLL(LIB_PATH)
        vp, u64, i32, dbl = ctypes.c_void_p, ctypes.c_uint64, ctypes.c_int, ctypes.c_double
        sig = {
            "pcal_create": (i32, [ctypes.POINTER(vp), dbl, dbl, dbl, i32, i32, i32]),
            "pcal_set_channel_offsets": (i32, [vp, vp]),
            "pcal_set_rotator": (i32, [vp, i32]),
            "pcal_set_k_shift": (i32, [vp, i32]),
            "pcal_set_start_index": (i32, [vp, u64]),
            "pcal_set_input_ready": (i32, [vp, i32]),
            "pcal_extract": (i32, [vp, vp, u64, vp]),
            "pcal_extract_host": (i32, [vp, vp, u64, vp]),
            "pcal_read_probe": (i32, [vp, vp, u64, vp]),
            "pcal_set_folded_sum_dev": (i32, [vp, vp, ctypes.c_uint32]),
            "pcal_finalize_series_sum_dev": (i32, [vp, vp, ctypes.c_uint32, ctypes.c_uint32, vp, vp]),
            "pcal_generator_study": (i32, [vp, ctypes.c_uint32, u64, ctypes.c_uint32, vp]),
            "pcal_extract_series": (i32, [vp, vp, u64, ctypes.c_uint32, vp, vp, vp]),
            "pcal_analyze": (i32, [vp, vp, vp]),
            "pcal_residual_rotation": (i32, [vp, vp, ctypes.c_uint32, vp]),
            "pcal_refine_offset": (i32, [vp, vp, u64, ctypes.c_uint32, vp, ctypes.c_uint32, dbl, ctypes.POINTER(dbl), vp,
                                         ctypes.POINTER(ctypes.c_uint32)]),
            "pcal_finalize": (i32, [vp, vp]),
            "pcal_finalize_async": (i32, [vp, vp]),
            "pcal_integrate": (i32, [vp, vp, u64, vp, vp]),
            "pcal_get_folded": (i32, [vp, vp]),
            "pcal_get_folded_i64": (i32, [vp, vp]),
            "pcal_add_folded": (i32, [vp, vp]),
            "pcal_get_folded_dev": (i32, [vp, vp]),
            "pcal_add_folded_dev": (i32, [vp, vp]),
            "pcal_set_profiling": (i32, [vp, i32]),
            "pcal_get_profile": (i32, [vp, ctypes.POINTER(dbl), ctypes.POINTER(u64)]),
            "pcal_pipe_probe": (i32, [i32, ctypes.POINTER(dbl)]),
            "pcal_fold_noalloc": (i32, [vp, u64, u64, dbl, dbl, dbl, i32, i32, i32, vp, vp]),
            "pcal_reset": (i32, [vp]),
            "pcal_destroy": (None, [vp]),
            "pcal_info": (i32, [vp, ctypes.POINTER(InfoT)]),
            "pcal_strerror": (ctypes.c_char_p, [i32]),
        }
        for name, (res, args) in sig.items():
            fn = getattr(L, name)
            fn.restype, fn.argtypes = res, args
        _lib = L
    return _lib


def _strerror(code: int) -> str:
    try:
        return lib().pcal_strerror(code).decode()
    except Exception:  # pragma: no cover
        return "?"


def _check(code: int, what: str):
    if code != PCAL_OK:
        raise PcalError(code, what)


def _stream_handle(stream) -> int:
    if stream is None:
        import torch
        return int(torch.cuda.current_stream().cuda_stream)
    return int(getattr(stream, "cuda_stream", stream))


class Pcal:
    """One extraction context (``pcal_ctx``).  Method names mirror the C ABI."""

    def __init__(self, f_s_hz: float, f_comb_hz: float, f_offset_hz: float, bits: int, encoding: int,
                 n_channels: int = 1):
        h = ctypes.c_void_p()
        _check(lib().pcal_create(ctypes.byref(h), f_s_hz, f_comb_hz, f_offset_hz, bits, encoding, n_channels),
               "pcal_create")
        self._h = h
        self.n_channels = n_channels
        self.n_bins = self.info().n_bins

    # -- configuration ---------------------------------------------------------------------
    def set_channel_offsets(self, f_offset_hz: Sequence[float]):
        a = np.ascontiguousarray(f_offset_hz, np.float64)
        assert a.shape == (self.n_channels,)
        _check(lib().pcal_set_channel_offsets(self._h, a.ctypes.data), "pcal_set_channel_offsets")

    def set_rotator(self, mode: int):
        _check(lib().pcal_set_rotator(self._h, mode), "pcal_set_rotator")

    def set_k_shift(self, k: int):
        _check(lib().pcal_set_k_shift(self._h, k), "pcal_set_k_shift")

    def set_input_ready(self, ready: bool):
        _check(lib().pcal_set_input_ready(self._h, int(ready)), "pcal_set_input_ready")

    def set_start_index(self, n_start: int):
        _check(lib().pcal_set_start_index(self._h, n_start), "pcal_set_start_index")

    # -- hot path --------------------------------------------------------------------------
    def extract(self, dev_samples, n_samples: Optional[int] = None, stream=None):
        """dev_samples: CUDA tensor (or raw device pointer int); n_samples per channel."""
        if hasattr(dev_samples, "data_ptr"):
            if not dev_samples.is_cuda:
                raise ValueError("pcal_extract needs a device buffer; use extract_host for host memory")
            ptr = dev_samples.data_ptr()
            if n_samples is None:
                nbytes = dev_samples.numel() * dev_samples.element_size()
                inf = self.info()
                n_samples = nbytes * 8 // (inf.bits * inf.n_channels)
        else:
            ptr = int(dev_samples)
        _check(lib().pcal_extract(self._h, ptr, n_samples, _stream_handle(stream)), "pcal_extract")

    def extract_series(self, dev_samples, n_per_period: int, n_periods: int, out_tones, out_folded=None, stream=None):
        """Time series of integrations: out_tones / out_folded are CUDA complex128 tensors
        [n_periods, n_channels, N_bins] (caller-owned); asynchronous."""
        _check(lib().pcal_extract_series(self._h, dev_samples.data_ptr(), n_per_period, n_periods, _stream_handle(stream),
                                         out_tones.data_ptr(), out_folded.data_ptr() if out_folded is not None else None),
               "pcal_extract_series")

    def extract_host(self, host_samples, n_samples: Optional[int] = None, stream=None):
        """host_samples: CPU tensor / numpy array (pinned for full speed)."""
        if hasattr(host_samples, "data_ptr"):
            ptr = host_samples.data_ptr()
            nbytes = host_samples.numel() * host_samples.element_size()
        else:
            ptr = host_samples.ctypes.data
            nbytes = host_samples.nbytes
        if n_samples is None:
            inf = self.info()
            n_samples = nbytes * 8 // (inf.bits * inf.n_channels)
        _check(lib().pcal_extract_host(self._h, ptr, n_samples, _stream_handle(stream)), "pcal_extract_host")

    def finalize(self) -> np.ndarray:
        """complex128 [n_channels, N_bins] tone spectrum T (synchronises)."""
        out = np.empty((self.n_channels, self.n_bins), np.complex128)
        _check(lib().pcal_finalize(self._h, out.ctypes.data), "pcal_finalize")
        return out

    def finalize_async(self, out_pinned):
        """Enqueue DFT + copy into a pinned complex128 host tensor; caller synchronises."""
        _check(lib().pcal_finalize_async(self._h, out_pinned.data_ptr()), "pcal_finalize_async")

    def integrate(self, dev_samples, n_samples: int, out_pinned, stream=None):
        """One integration period: reset + extract + finalize_async in one library call (asynchronous).
        Tensors or raw addresses (a host loop over short periods can hoist ``data_ptr()`` and the stream handle)."""
        src = dev_samples.data_ptr() if hasattr(dev_samples, "data_ptr") else int(dev_samples)
        dst = out_pinned.data_ptr() if hasattr(out_pinned, "data_ptr") else int(out_pinned)
        _check(lib().pcal_integrate(self._h, src, n_samples, _stream_handle(stream), dst), "pcal_integrate")

    def analyze(self, bandpass: bool = True):
        """(summary float64 [n_channels, 8], corrected band-pass complex128 [n_channels, N_bins] or None)."""
        summ = np.empty((self.n_channels, 8), np.float64)
        bp = np.empty((self.n_channels, self.n_bins), np.complex128) if bandpass else None
        _check(lib().pcal_analyze(self._h, summ.ctypes.data, bp.ctypes.data if bandpass else None), "pcal_analyze")
        return summ, bp

    def residual_rotation(self, dev_series_tones, n_periods: int) -> np.ndarray:
        """float64 [n_channels, 3]: (arg S, |S|, norm) of a pcal_extract_series output (CUDA complex128 tensor)."""
        out = np.empty((self.n_channels, 3), np.float64)
        _check(lib().pcal_residual_rotation(self._h, dev_series_tones.data_ptr(), n_periods, out.ctypes.data), "pcal_residual_rotation")
        return out

    def refine_offset(self, dev_samples, n_per_period: int, n_periods: int, max_passes: int = 4, tol_rad: float = 1e-6, stream=None):
        """Multi-pass counter-rotation.  Returns (refined f_offset in Hz, history float64 [passes, 4]:
        f_rot used, arg S, |S|, norm).  The context is reset and its f_offset replaced by the refined value."""
        f, n = ctypes.c_double(), ctypes.c_uint32()
        hist = np.zeros((max_passes, 4), np.float64)
        _check(lib().pcal_refine_offset(self._h, dev_samples.data_ptr(), n_per_period, n_periods, _stream_handle(stream), max_passes,
                                        tol_rad, ctypes.byref(f), hist.ctypes.data, ctypes.byref(n)), "pcal_refine_offset")
        return f.value, hist[:n.value]

    def get_folded(self) -> np.ndarray:
        out = np.empty((self.n_channels, self.n_bins), np.complex128)
        _check(lib().pcal_get_folded(self._h, out.ctypes.data), "pcal_get_folded")
        return out

    def get_folded_i64(self) -> np.ndarray:
        out = np.empty((self.n_channels, self.n_bins), np.int64)
        _check(lib().pcal_get_folded_i64(self._h, out.ctypes.data), "pcal_get_folded_i64")
        return out

    def add_folded(self, bins: np.ndarray):
        b = np.ascontiguousarray(bins, np.complex128)
        assert b.shape == (self.n_channels, self.n_bins)
        _check(lib().pcal_add_folded(self._h, b.ctypes.data), "pcal_add_folded")

    def get_folded_dev(self, dev_bins):
        _check(lib().pcal_get_folded_dev(self._h, dev_bins.data_ptr()), "pcal_get_folded_dev")

    def add_folded_dev(self, dev_bins):
        _check(lib().pcal_add_folded_dev(self._h, dev_bins.data_ptr()), "pcal_add_folded_dev")

    def read_probe(self, dev_buf, stream=None):
        """Calibration: enqueue a pure streaming read of the whole device tensor (roofline report)."""
        nbytes = dev_buf.numel() * dev_buf.element_size()
        _check(lib().pcal_read_probe(self._h, dev_buf.data_ptr(), nbytes, _stream_handle(stream)), "pcal_read_probe")

    def set_folded_sum_dev(self, dev_parts, n_parts: int):
        """Accumulators <- sum of n_parts gathered bin blocks (rank order); dev_parts: CUDA float64 tensor."""
        _check(lib().pcal_set_folded_sum_dev(self._h, dev_parts.data_ptr(), n_parts), "pcal_set_folded_sum_dev")

    def finalize_series_sum_dev(self, dev_parts, n_parts: int, n_periods: int, out_folded, out_tones):
        """Rank-order sums + DFT of n_periods gathered periods (CUDA tensors); asynchronous."""
        _check(lib().pcal_finalize_series_sum_dev(self._h, dev_parts.data_ptr(), n_parts, n_periods, out_folded.data_ptr(),
                                                  out_tones.data_ptr()), "pcal_finalize_series_sum_dev")

    def set_profiling(self, enable: bool):
        _check(lib().pcal_set_profiling(self._h, int(enable)), "pcal_set_profiling")

    def get_profile(self):
        """(summed hot-kernel event time in ms, hot-kernel launches) since the last call."""
        ms, n = ctypes.c_double(), ctypes.c_uint64()
        _check(lib().pcal_get_profile(self._h, ctypes.byref(ms), ctypes.byref(n)), "pcal_get_profile")
        return ms.value, n.value

    def reset(self):
        _check(lib().pcal_reset(self._h), "pcal_reset")

    def info(self) -> InfoT:
        inf = InfoT()
        _check(lib().pcal_info(self._h, ctypes.byref(inf)), "pcal_info")
        return inf

    def destroy(self):
        if getattr(self, "_h", None):
            lib().pcal_destroy(self._h)
            self._h = None

    def __del__(self):  # pragma: no cover
        try:
            self.destroy()
        except Exception:
            pass


GEN_CFO, GEN_MCO, GEN_DFR, GEN_DFR_FMA, GEN_DIRECT = 0, 1, 2, 3, 4


class GenCaseT(ctypes.Structure):
    _fields_ = [("form", ctypes.c_int32), ("precision", ctypes.c_int32), ("f_s_hz", ctypes.c_double),
                ("f_rot_hz", ctypes.c_double)]


def generator_study(cases, n_steps: int, n_chk: int) -> np.ndarray:
    """cases: sequence of (form, precision, f_s_hz, f_rot_hz); returns float64 [n_cases, n_chk] max errors."""
    arr = (GenCaseT * len(cases))(*[GenCaseT(int(f), int(p), float(fs), float(fr)) for f, p, fs, fr in cases])
    out = np.empty((len(cases), n_chk), np.float64)
    _check(lib().pcal_generator_study(ctypes.cast(arr, ctypes.c_void_p), len(cases), n_steps, n_chk, out.ctypes.data),
           "pcal_generator_study")
    return out


def pipe_probe(kind: int) -> float:
    """Measured issue rate of one pipe (0 FFMA, 1 LOP3: thread-instructions/s; 2 IMMA m16n8k16: warp-level MMAs/s)."""
    v = ctypes.c_double()
    _check(lib().pcal_pipe_probe(kind, ctypes.byref(v)), "pcal_pipe_probe")
    return v.value


def fold_noalloc(dev_samples, n_samples: int, start_index: int, f_s_hz: float, f_comb_hz: float, f_offset_hz: float,
                 bits: int, encoding: int, accumulate: bool, dev_out_bins, stream=None):
    """pcal_fold_noalloc (include/pcal_noalloc.h): rotate + fold one single-channel segment into the caller's device bins
    without any allocation in the library (N_bins <= 1024; every call on a device shares one scratch array).
    Tensors or raw addresses; asynchronous.  Marshalling only."""
    src = dev_samples.data_ptr() if hasattr(dev_samples, "data_ptr") else int(dev_samples)
    dst = dev_out_bins.data_ptr() if hasattr(dev_out_bins, "data_ptr") else int(dev_out_bins)
    _check(lib().pcal_fold_noalloc(src, n_samples, start_index, f_s_hz, f_comb_hz, f_offset_hz, bits, encoding,
                                   1 if accumulate else 0, dst, _stream_handle(stream)), "pcal_fold_noalloc")


def from_workload(w) -> "Pcal":
    """Context for a ``synth.Workload`` (marshalling only)."""
    p = Pcal(w.f_s_hz, w.f_comb_hz, w.f_offset_hz[0], w.bits, w.encoding, w.n_channels)
    if w.n_channels > 1 or any(f != w.f_offset_hz[0] for f in w.f_offset_hz):
        p.set_channel_offsets(w.f_offset_hz)
    p.set_rotator({"auto": ROT_AUTO, "lut": ROT_LUT, "generator": ROT_GENERATOR}[w.rotator])
    return p
