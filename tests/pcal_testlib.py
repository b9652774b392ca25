"""Shared helpers of the GPU parity tests: run a workload through the C ABI and through the oracle."""
import numpy as np

from paper_2501_05993_b200 import synth

REL_TOL = 1e-5      # north_star: each tone within 1e-5 relative ...
PHASE_TOL = 1e-5    # ... and its phase within 1e-5 rad of the oracle


def oracle_fmt(orc, w):
    if w.bits == 32:
        return orc.F32
    if w.bits == 8:
        return orc.I8
    return orc.TWO_BIT_OFFSET_BINARY if w.encoding == synth.ENC_OFFSET_BINARY else orc.TWO_BIT_SIGN_MAG


def oracle_folded(orc, w, host_buf, c, n_abs0=0, threads=1, tabulated=True, bins=None):
    """P[c] as complex128 via the oracle; ``bins`` = list of bins to visit only (others left 0)."""
    fmt = oracle_fmt(orc, w)
    nb = w.n_bins
    if bins is None:
        pr, pi = orc.fold_ld(host_buf, fmt, w.n_channels, c, 0, 1, w.n_samples, n_abs0,
                             w.f_s_hz, w.f_comb_hz, w.f_offset_hz[c], tabulated=tabulated, threads=threads)
        return pr, pi
    pr = np.zeros(nb, np.longdouble)
    pi = np.zeros(nb, np.longdouble)
    for b in bins:
        m_first = (b - n_abs0) % nb
        r, i = orc.fold_ld(host_buf, fmt, w.n_channels, c, m_first, nb, w.n_samples, n_abs0,
                           w.f_s_hz, w.f_comb_hz, w.f_offset_hz[c], tabulated=tabulated, threads=threads)
        pr[b], pi[b] = r[b], i[b]
    return pr, pi


def oracle_tones(orc, w, host_buf, c, n_abs0=0, threads=1):
    pr, pi = oracle_folded(orc, w, host_buf, c, n_abs0, threads)
    return orc.dft(pr, pi)


def gpu_run(w, dev_buf, splits=(), k_shift=0, rotator=None, start=0):
    """Extract ``dev_buf`` (optionally in segments cut at the given time-sample indices)."""
    from paper_2501_05993_b200 import binding
    if rotator is not None:
        w = synth.replace(w, rotator=rotator)
    p = binding.from_workload(w)
    if k_shift:
        p.set_k_shift(k_shift)
    if start:
        p.set_start_index(start)
    bytes_per_t = w.bits * w.n_channels / 8.0
    flat = dev_buf.view(-1).view(dtype=__import__("torch").uint8)
    edges = [0] + list(splits) + [w.n_samples]
    for a, b in zip(edges[:-1], edges[1:]):
        lo, hi = int(a * bytes_per_t), int(b * bytes_per_t)
        assert lo % 16 == 0, "segment start must stay 16-byte aligned"
        if hi > lo:
            p.extract(flat[lo:hi], b - a)
        else:
            p.extract(flat[lo:lo], 0)
    T = p.finalize()
    P = p.get_folded()
    return p, T, P


def assert_close(got, want, what="", floor_frac=0.0):
    """north_star's bar, per output.  ``floor_frac`` > 0 (short integrations only, where a noise bin
    can fall near zero by chance and its relative error is ill-conditioned) measures the error of
    such a bin against floor_frac * median |want| instead of its own magnitude."""
    got = np.asarray(got)
    want = np.asarray(want)
    err = np.abs(got - want)
    rel = err / np.maximum(np.maximum(np.abs(want), floor_frac * np.median(np.abs(want))), 1e-300)
    worst = int(np.argmax(rel))
    assert rel.max() <= REL_TOL, f"{what}: rel err {rel.max():.3e} at {worst} (|want|={abs(want.flat[worst]):.3e})"
    dphi = np.angle(got * np.conj(want))
    if floor_frac:
        dphi = dphi[np.abs(want) >= floor_frac * np.median(np.abs(want))]
    assert np.abs(dphi).max() <= PHASE_TOL, f"{what}: phase err {np.abs(dphi).max():.3e} rad"
    return float(rel.max()), float(err.max() / np.abs(want).max())
