"""TEST INFRASTRUCTURE, NOT THE PRODUCT -- ctypes front end of ``oracle/pcal_oracle.c``.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It never imports
``paper_2501_05993_b200`` and that package never imports it.

The arithmetic lives in the C file (each function there cites the passage of
/root/reference/PAPER.md it restates).  This module only marshals arguments, snaps
frequencies to the 1 micro-hertz grid (reading R16) and, for long streams, splits the
sample range into contiguous pieces that are summed *in range order* in long double
(SURVEY.md section 8(d) "Oracle timing") -- the per-sample arithmetic is untouched.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from concurrent.futures import ThreadPoolExecutor

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pcal_oracle.c")
_LIB = os.path.join(_HERE, "libpcal_oracle.so")

F32, I8, TWO_BIT_OFFSET_BINARY, TWO_BIT_SIGN_MAG, F64 = 0, 1, 2, 3, 4


def build(force: bool = False) -> str:
    """Compile the C oracle with gcc (building the checker is not using it)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"])
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = ctypes.CDLL(build())
        u64, i32, vp = ctypes.c_uint64, ctypes.c_int, ctypes.c_void_p
        L.orc_decode.restype = ctypes.c_double
        L.orc_decode.argtypes = [vp, i32, i32, i32, u64]
        L.orc_phase_num.restype = u64
        L.orc_phase_num.argtypes = [u64, u64, u64]
        L.orc_rotator_len.restype = u64
        L.orc_rotator_len.argtypes = [u64, u64]
        L.orc_direct.restype = None
        L.orc_direct.argtypes = [vp, i32, i32, i32, u64, u64, u64, u64, u64, u64, vp, vp]
        L.orc_fold.restype = None
        L.orc_fold.argtypes = [vp, i32, i32, i32, u64, u64, u64, u64, u64, u64, u64, vp, vp]
        L.orc_fold_tabulated.restype = None
        L.orc_fold_tabulated.argtypes = [vp, i32, i32, i32, u64, u64, u64, u64, u64, u64, u64, vp, vp, vp, vp]
        L.orc_fold_i64.restype = i32
        L.orc_fold_i64.argtypes = [vp, i32, i32, i32, u64, u64, u64, u64, u64, vp]
        L.orc_dft.restype = None
        L.orc_dft.argtypes = [vp, vp, u64, vp]
        _lib = L
    return _lib


def to_uhz(f_hz: float) -> int:
    """Snap a frequency in Hz to the integer micro-hertz grid (R16)."""
    return int(round(float(f_hz) * 1e6))


def _ptr(a: np.ndarray) -> int:
    assert a.flags["C_CONTIGUOUS"]
    return a.ctypes.data


def decode(buf: np.ndarray, fmt: int, n_channels: int, c: int, m: int) -> float:
    return lib().orc_decode(_ptr(buf), fmt, n_channels, c, m)


def rotator_len(f_s_hz: float, f_offset_hz: float) -> int:
    return lib().orc_rotator_len(to_uhz(f_s_hz), to_uhz(f_offset_hz))


def direct(buf, fmt, n_channels, c, m0, count, n_abs0, f_s_hz, f_comb_hz, f_offset_hz) -> np.ndarray:
    """O-direct: complex128[N_bins] per-tone correlations (eq. 2.1-2.3)."""
    Fs, Fc, Fo = to_uhz(f_s_hz), to_uhz(f_comb_hz), to_uhz(f_offset_hz)
    nb = Fs // Fc
    tr = np.zeros(nb, np.longdouble)
    ti = np.zeros(nb, np.longdouble)
    lib().orc_direct(_ptr(buf), fmt, n_channels, c, m0, count, n_abs0, Fs, Fc, Fo, _ptr(tr), _ptr(ti))
    return tr.astype(np.float64) + 1j * ti.astype(np.float64)


def fold_ld(buf, fmt, n_channels, c, m_first, m_step, m_end, n_abs0, f_s_hz, f_comb_hz, f_offset_hz,
            tabulated: bool = False, threads: int = 1):
    """O-fold, first half: (P_re, P_im) as long double[N_bins] (eq. 2.3 then eq. 2.2).

    ``threads`` > 1 splits [m_first, m_end) into that many contiguous ranges evaluated
    concurrently by the same C routine and added in range order."""
    Fs, Fc, Fo = to_uhz(f_s_hz), to_uhz(f_comb_hz), to_uhz(f_offset_hz)
    nb = Fs // Fc
    L = lib()

    def piece(lo, hi):
        pr = np.zeros(nb, np.longdouble)
        pi = np.zeros(nb, np.longdouble)
        if hi > lo:
            nrot = L.orc_rotator_len(Fs, Fo)
            # tabulate only a rotator vector of practical length ("impractically long
            # vector"); otherwise every phasor is computed directly -- the values are identical
            if tabulated and Fo != 0 and nrot <= (1 << 24):
                tc = np.empty(nrot, np.float64)
                ts = np.empty(nrot, np.float64)
                L.orc_fold_tabulated(_ptr(buf), fmt, n_channels, c, lo, m_step, hi, n_abs0, Fs, Fc, Fo,
                                     _ptr(tc), _ptr(ts), _ptr(pr), _ptr(pi))
            else:
                L.orc_fold(_ptr(buf), fmt, n_channels, c, lo, m_step, hi, n_abs0, Fs, Fc, Fo, _ptr(pr), _ptr(pi))
        return pr, pi

    if threads <= 1:
        return piece(m_first, m_end)
    n_steps = (max(m_end - m_first, 0) + m_step - 1) // m_step
    per = (n_steps + threads - 1) // threads
    bounds = [(m_first + k * per * m_step, min(m_first + (k + 1) * per * m_step, m_end)) for k in range(threads)]
    with ThreadPoolExecutor(threads) as ex:
        parts = list(ex.map(lambda b: piece(*b), bounds))
    pr = np.zeros(nb, np.longdouble)
    pi = np.zeros(nb, np.longdouble)
    for a, b in parts:  # range order
        pr += a
        pi += b
    return pr, pi


def fold_i64(buf, fmt, n_channels, c, m_first, m_step, m_end, n_abs0, n_bins) -> np.ndarray:
    """O-int: exact int64 bins (eq. 2.2, f_offset = 0, integer samples)."""
    p = np.zeros(n_bins, np.int64)
    rc = lib().orc_fold_i64(_ptr(buf), fmt, n_channels, c, m_first, m_step, m_end, n_abs0, n_bins, _ptr(p))
    if rc != 0:
        raise ValueError("orc_fold_i64: float input has no integer bins")
    return p


def dft(p_re: np.ndarray, p_im: np.ndarray) -> np.ndarray:
    """O-fold, second half: forward unnormalised DFT of the folded period."""
    p_re = np.ascontiguousarray(p_re, np.longdouble)
    p_im = np.ascontiguousarray(p_im, np.longdouble)
    n = p_re.shape[0]
    t = np.empty(2 * n, np.float64)
    lib().orc_dft(_ptr(p_re), _ptr(p_im), n, _ptr(t))
    return t[0::2] + 1j * t[1::2]


def extract(buf, fmt, n_channels, c, n_samples, n_abs0, f_s_hz, f_comb_hz, f_offset_hz,
            tabulated: bool = False, threads: int = 1) -> np.ndarray:
    """O-fold end to end: tones T[i], complex128[N_bins], for channel c."""
    pr, pi = fold_ld(buf, fmt, n_channels, c, 0, 1, n_samples, n_abs0, f_s_hz, f_comb_hz, f_offset_hz,
                     tabulated=tabulated, threads=threads)
    return dft(pr, pi)
