"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times: the whole resident buffer in
one period, once as pcal_extract + pcal_finalize and once exactly as bench.py's step issues it (pcal_set_input_ready +
pcal_integrate into a pinned buffer, twice back to back so that the launches overlap).

Configs 1-4: every folded bin and every tone against the oracle (rotator tabulated, host threads over
contiguous ranges).  Config 5 (4e9 samples, offset without a practical table): first six sampled folded bins the
oracle can compute one by one (a bin only needs the 1/1024 of the samples that land in it) as a fast pre-check,
then ALL 1024 bins and tones against the un-tabulated oracle on every host thread (~200 core-seconds).
"""
import os

import numpy as np
import pytest
import torch

from paper_2501_05993_b200 import synth
from pcal_testlib import assert_close, gpu_run, oracle_folded

pytestmark = pytest.mark.gpu
THREADS = min(32, os.cpu_count() or 1)


def bench_step_agrees(p, w, dev, T):
    """bench.py's step on the same context: two overlapping periods; both must reproduce T (already held to the oracle)."""
    outs = [torch.zeros((w.n_channels, w.n_bins), dtype=torch.complex128).pin_memory() for _ in range(2)]
    p.set_input_ready(True)
    for o in outs:
        p.integrate(dev, w.n_samples, o)
    torch.cuda.synchronize()
    for o in outs:
        assert np.abs(o.numpy() - T).max() <= 1e-12 * np.abs(T).max()


@pytest.mark.parametrize("idx,rot", [(1, None), (2, None), (3, "lut"), (3, "generator")])
def test_fullsize_single_channel(oracle, idx, rot):
    w = synth.config(idx)
    dev = synth.generate(w, "cuda")
    host = dev.cpu().numpy()
    p, T, P = gpu_run(w, dev, rotator=rot)
    assert p.info().n_processed == w.n_samples
    pr, pi = oracle_folded(oracle, w, host, 0, threads=THREADS)
    rel, _ = assert_close(P[0], pr.astype(np.float64) + 1j * pi.astype(np.float64), f"cfg{idx} {rot} folded")
    assert_close(T[0], oracle.dft(pr, pi), f"cfg{idx} {rot} tones")
    print(f"cfg{idx} {rot}: worst-bin relative error {rel:.3e}")
    bench_step_agrees(p, w, dev, T)


def test_fullsize_cfg4_sixteen_channels(oracle):
    w = synth.config(4)
    dev = synth.generate(w, "cuda")
    host = dev.cpu().numpy()
    p, T, P = gpu_run(w, dev)
    assert p.info().fold_period == 6400
    for c in (0, 5, 10, 15):
        pr, pi = oracle_folded(oracle, w, host, c, threads=THREADS)
        assert_close(P[c], pr.astype(np.float64) + 1j * pi.astype(np.float64), f"cfg4 ch{c} folded")
        assert_close(T[c], oracle.dft(pr, pi), f"cfg4 ch{c} tones")
    bench_step_agrees(p, w, dev, T)


def test_fullsize_cfg5_all_bins(oracle):
    w = synth.config(5)
    dev = synth.generate(w, "cuda")
    p, T, P = gpu_run(w, dev)
    assert p.info().rotator_in_effect == 2 and p.info().n_processed == w.n_samples
    bench_step_agrees(p, w, dev, T)
    host = dev.cpu().numpy()
    del dev
    torch.cuda.empty_cache()
    bins = [0, 1, 511, 512, 777, 1023]
    pr, pi = oracle_folded(oracle, w, host, 0, threads=THREADS, tabulated=False, bins=bins)
    want = pr.astype(np.float64) + 1j * pi.astype(np.float64)
    assert_close(P[0][bins], want[bins], "cfg5 sampled folded bins")
    # every bin and every tone: the oracle's own fold (exactly reduced phase + sincos per sample) and its own DFT
    pr, pi = oracle_folded(oracle, w, host, 0, threads=THREADS, tabulated=False)
    rel, _ = assert_close(P[0], pr.astype(np.float64) + 1j * pi.astype(np.float64), "cfg5 folded, all bins")
    assert_close(T[0], oracle.dft(pr, pi), "cfg5 tones, all bins")
    print(f"cfg5: worst-bin relative error {rel:.3e}")
    # the comb must be visible.  (Its pulses peak at K*A = 512 >> 127, so the int8 clip of
    # BASELINE.json config 5 compresses the tone amplitudes below the closed form's A N / 2.)
    amp = 2 * np.abs(T[0][1:500]) / w.n_samples
    assert np.all((amp > 0.3 * w.amp) & (amp < 1.05 * w.amp)), (amp.min(), amp.max())
    # (No "upper bins are noise-only" check here: the clip's odd-order intermodulation products
    # f_a + f_b - f_c = (a+b-c) f_comb + f_offset fall exactly on comb bins, including the aliased
    # ones above N_bins/2, so those bins legitimately hold power for this input.)
