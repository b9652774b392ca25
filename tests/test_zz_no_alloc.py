"""pcal_fold_noalloc (include/pcal_noalloc.h): the entry point that allocates nothing -- its scratch is a file-scope
``static __device__`` array of the library -- against the existing context path (``Pcal.extract`` + ``get_folded``) on the
same bytes, within the tolerance of the other GPU tests (pcal_testlib.assert_close: 1e-5 relative, 1e-5 rad per bin).

Collected last on purpose (the suite runs with ``pytest -x``).  Every test makes its calls back to back on one stream
WITHOUT a synchronisation in between: all calls share the scratch array, which keeps the previous call's contents.
"""
import numpy as np
import pytest
import torch

from paper_2501_05993_b200 import synth
from pcal_testlib import assert_close

pytestmark = pytest.mark.gpu

DEV = "cuda"
PCAL_ERR_LIMIT = -7


def existing_path(w, dev, start=0):
    """Folded bins of channel 0 through a context (the path every other test holds to the oracle)."""
    from paper_2501_05993_b200 import binding
    p = binding.from_workload(w)
    if start:
        p.set_start_index(start)
    p.extract(dev, w.n_samples)
    P = p.get_folded()[0]
    p.destroy()
    return P


def noalloc(w, dev, out, start=0, accumulate=False, n=None, byte_offset=0):
    from paper_2501_05993_b200 import binding
    n = w.n_samples if n is None else n
    binding.fold_noalloc(dev.view(-1).view(torch.uint8).data_ptr() + byte_offset, n, start, w.f_s_hz, w.f_comb_hz, w.f_offset_hz[0],
                         w.bits, w.encoding, accumulate, out)


def small_args(w):
    # reading R28: float32 input may have a few "small" bins on a short integration
    return dict(max_small=max(1, w.n_bins // 64), small_bin=1e-2) if w.bits == 32 else dict(max_small=1)


# (config, samples): float32 with rotation (N_bins 16), 2-bit (N_bins 32), int8 with the non-rational offset (N_bins 1024 = the limit)
CASES = [(8, 1_300_001), (2, 1_300_004), (5, 2_600_003)]


@pytest.mark.parametrize("first,second", [(CASES[0], CASES[1]), (CASES[2], CASES[0]), (CASES[1], CASES[2])])
def test_two_calls_in_a_row_match_the_context_path(first, second):
    """Two different problems back to back (different sample type, N_bins and grid of partial bins): the second call must not
    see anything of the first in the shared scratch, and the first must not be disturbed by the second starting."""
    ws, devs, outs = [], [], []
    for idx, n in (first, second):
        w = synth.replace(synth.config(idx).scaled(n), rotator="generator")
        ws.append(w)
        devs.append(synth.generate(w, DEV))
        outs.append(torch.full((w.n_bins,), float("nan"), dtype=torch.complex128, device=DEV))     # overwritten, not added to
    for w, dev, out in zip(ws, devs, outs):
        noalloc(w, dev, out)                     # no synchronisation between the two calls
    torch.cuda.synchronize()
    for w, dev, out in zip(ws, devs, outs):
        assert_close(out.cpu().numpy(), existing_path(w, dev), f"{w.name} noalloc vs context", **small_args(w))


def test_same_problem_twice_and_accumulate():
    """The same call twice gives bit-identical bins (nothing of call 1 leaks into call 2); a stream cut in two segments with
    accumulate = 1 and the second segment's start index equals the one-call result to rounding."""
    w = synth.replace(synth.config(8).scaled(2_000_004), rotator="generator")
    dev = synth.generate(w, DEV)
    a = torch.empty(w.n_bins, dtype=torch.complex128, device=DEV)
    b = torch.empty_like(a)
    c = torch.empty_like(a)
    noalloc(w, dev, a)
    noalloc(w, dev, b)
    cut = 1_000_000                              # float32: 4 bytes per sample, the cut stays 16-byte aligned
    noalloc(w, dev, c, n=cut)
    noalloc(w, dev, c, start=cut, accumulate=True, n=w.n_samples - cut, byte_offset=4 * cut)
    torch.cuda.synchronize()
    assert torch.equal(a.view(torch.float64), b.view(torch.float64))
    want = existing_path(w, dev)
    assert_close(a.cpu().numpy(), want, "noalloc vs context", **small_args(w))
    assert_close(c.cpu().numpy(), want, "noalloc, two segments", **small_args(w))


def test_start_index_and_tiny_segments():
    """A start index in the middle of a period, and segments shorter than one load (tail-only) / than one CTA iteration."""
    for n in (3, 16, 1028):
        w = synth.replace(synth.config(8).scaled(n), rotator="generator")
        dev = synth.generate(w, DEV)
        buf = dev if dev.numel() * dev.element_size() >= 16 else torch.cat([dev.view(-1), torch.zeros(4, dtype=dev.dtype, device=DEV)])
        out = torch.empty(w.n_bins, dtype=torch.complex128, device=DEV)
        noalloc(w, buf, out, start=12_345)
        torch.cuda.synchronize()
        want = existing_path(w, buf, start=12_345)
        got = out.cpu().numpy()
        empty = want == 0                         # bins no sample fell into: exactly zero on both sides
        assert not got[empty].any()
        if (~empty).any():
            assert_close(got[~empty], want[~empty], f"n={n}")


def test_sizes_beyond_the_scratch_are_refused():
    """N_bins above PCAL_NOALLOC_MAX_BINS -> PCAL_ERR_LIMIT with a message that names the limit; nothing is launched."""
    from paper_2501_05993_b200 import binding
    x = torch.zeros(4096, dtype=torch.float32, device=DEV)
    out = torch.zeros(2048, dtype=torch.complex128, device=DEV)
    with pytest.raises(binding.PcalError) as e:
        binding.fold_noalloc(x, 4096, 0, 2048e6, 1e6, 10e3, 32, binding.ENC_IEEE_FLOAT, False, out)
    assert e.value.code == PCAL_ERR_LIMIT and "1024" in str(e.value)
    torch.cuda.synchronize()
    assert not out.view(torch.float64).any()
    with pytest.raises(binding.PcalError) as e:          # a sample type that does not exist: PCAL_ERR_INVALID
        binding.fold_noalloc(x, 4096, 0, 32e6, 1e6, 0.0, 16, binding.ENC_IEEE_FLOAT, False, out)
    assert e.value.code == -1


def test_free_device_memory_does_not_move(monkeypatch):
    """After the first call on the device (set-up), further calls leave cudaMemGetInfo's free figure where it was: nothing is
    allocated or freed -- also when a call needs several launches (PCAL_SMALL_PIECES=1: 2 tiles per CTA and launch, three
    pieces here, the later ones added to the bins the first one has overwritten)."""
    monkeypatch.setenv("PCAL_SMALL_PIECES", "1")
    w = synth.replace(synth.config(8).scaled(40_000_004), rotator="generator")
    dev = synth.generate(w, DEV)
    out = torch.full((w.n_bins,), float("nan"), dtype=torch.complex128, device=DEV)
    noalloc(w, dev, out, n=4096)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        noalloc(w, dev, out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0
    monkeypatch.delenv("PCAL_SMALL_PIECES")
    assert_close(out.cpu().numpy(), existing_path(w, dev), "40e6 samples in three pieces", **small_args(w))
