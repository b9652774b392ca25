"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same seeded bytes.  Sizes span many tiles / super-rows and end in a ragged tail.

Bar (north_star): int64 folded bins bit-exact for integer input with f_offset = 0; every tone
within 1e-5 relative and 1e-5 rad otherwise (R17: every one of the N_bins outputs).
"""
import numpy as np
import pytest
import torch

from paper_2501_05993_b200 import synth
from pcal_testlib import assert_close, gpu_run, oracle_fmt, oracle_folded, oracle_tones

pytestmark = pytest.mark.gpu

DEV = "cuda"

# (config index, n_samples) -- ragged: not a multiple of a 16-byte vector, of L, or of a tile
SMALL = [
    (1, 1_300_001),      # float32, f_offset 0
    (2, 1_300_004),      # 2-bit offset-binary, L = 3200 (LUT)
    (3, 2_600_036),      # 2-bit, N_bins 512, L = 51200 (LUT)
    (4, 200_003),        # 16 channels, sign-magnitude, per-channel offsets
    (5, 1_300_003),      # int8, irrational offset -> generator
    (6, 1_300_004),      # cfg 2', f_offset 0: integer-exact
    (7, 1_300_003),      # cfg 5', int8 f_offset 0: integer-exact
    (8, 1_300_001),      # the paper's benchmark shape: float32 with rotation, L = 1600
]


def make(idx, n):
    w = synth.config(idx).scaled(n)
    dev = synth.generate(w, DEV)
    host = dev.cpu().numpy()
    return w, dev, host


@pytest.mark.parametrize("idx,n", SMALL)
def test_parity_every_config_small(oracle, idx, n):
    w, dev, host = make(idx, n)
    p, T, P = gpu_run(w, dev)
    inf = p.info()
    assert inf.n_processed == n
    for c in range(w.n_channels):
        pr, pi = oracle_folded(oracle, w, host, c)
        want_P = pr.astype(np.float64) + 1j * pi.astype(np.float64)
        assert_close(P[c], want_P, f"cfg{idx} ch{c} folded")
        assert_close(T[c], oracle.dft(pr, pi), f"cfg{idx} ch{c} tones")
    if idx in (6, 7):
        assert inf.integer_exact == 1
        got = p.get_folded_i64()
        want = oracle.fold_i64(host, oracle_fmt(oracle, w), 1, 0, 0, 1, n, 0, w.n_bins)
        assert np.array_equal(got[0], want)          # bit-exact
        assert np.array_equal(P[0].real, want.astype(np.float64)) and not P[0].imag.any()


def test_zero_offset_channel_of_cfg4_is_integer_exact(oracle):
    """R20: force one zero-offset channel among rotated ones; its bins must be exact integers."""
    w = synth.config(4).scaled(100_001)
    w.f_offset_hz[3] = 0.0
    dev = synth.generate(w, DEV)
    host = dev.cpu().numpy()
    p, T, P = gpu_run(w, dev)
    want = oracle.fold_i64(host, oracle.TWO_BIT_SIGN_MAG, 16, 3, 0, 1, w.n_samples, 0, w.n_bins)
    assert np.array_equal(P[3].real, want.astype(np.float64)) and not P[3].imag.any()
    for c in (0, 3, 15):
        assert_close(T[c], oracle_tones(oracle, w, host, c), f"ch{c}")


@pytest.mark.parametrize("rot", ["lut", "generator"])
def test_cfg3_both_rotator_variants(oracle, rot):
    w, dev, host = make(3, 3_000_004)
    p, T, P = gpu_run(w, dev, rotator=rot)
    assert p.info().rotator_in_effect == (1 if rot == "lut" else 2)
    assert_close(T[0], oracle_tones(oracle, w, host, 0), f"cfg3 {rot}")


@pytest.mark.parametrize("idx,n", [(2, 700_004), (8, 500_003), (7, 400_001)])
def test_generator_on_every_sample_type(oracle, idx, n):
    """2-bit (both encodings), float32 and int8 through the generator kernel."""
    w, dev, host = make(idx, n)
    if idx == 7:
        w = synth.replace(w, f_offset_hz=[1234.567])
    p, T, P = gpu_run(w, dev, rotator="generator")
    assert p.info().rotator_in_effect == 2
    assert_close(T[0], oracle_tones(oracle, w, host, 0), f"gen cfg{idx}")
    if idx == 2:
        w2 = synth.replace(w, encoding=synth.ENC_SIGN_MAG)
        p, T, P = gpu_run(w2, dev, rotator="generator")
        assert_close(T[0], oracle_tones(oracle, w2, host, 0), "gen sign-mag")


@pytest.mark.parametrize("idx,n,k_shift", [(1, 1_300_001, 0), (2, 1_300_004, 0), (2, 1_300_004, 5), (4, 200_003, 0), (6, 600_004, 0),
                                           (3, 2_600_036, 0), (5, 1_300_003, 0), (8, 500_001, 0), (2, 60, 0)])
def test_integrate_is_reset_extract_finalize(oracle, idx, n, k_shift):
    """pcal_integrate = pcal_reset + pcal_extract + pcal_finalize_async in one call.  On the LUT path and on the 2-bit
    generator paths the last CTA of the extract kernel takes the DFT itself (two stages) and writes T straight into the
    pinned buffer: one launch per period.  Repeated periods on one context, against the oracle and against the three calls."""
    from paper_2501_05993_b200 import binding
    w, dev, host = make(idx, n)
    p = binding.from_workload(w)
    if k_shift:
        p.set_k_shift(k_shift)
    out = torch.empty((w.n_channels, w.n_bins), dtype=torch.complex128).pin_memory()
    l0 = p.info().kernel_launches
    for _ in range(3):                      # the context keeps integrating period after period
        out.zero_()
        p.integrate(dev, n, out)
    torch.cuda.synchronize()
    per_period = (p.info().kernel_launches - l0) // 3
    T1 = out.numpy().copy()
    p.reset(); p.extract(dev, n); T2 = p.finalize()
    # (config 5: 296 CTAs x 1024 bins keep the separate post and DFT kernels; a period shorter than one vector: tail kernel + DFT kernel)
    assert per_period == (3 if idx == 5 else (1 if n > 1000 else 2)), per_period
    for c in range(0, w.n_channels, 5):
        if n > 1000:
            assert_close(T1[c], oracle_tones(oracle, w, host, c), f"integrate cfg{idx} ch{c}")
    assert np.abs(T1 - T2).max() <= 1e-12 * np.abs(T2).max()
    p.destroy()


@pytest.mark.parametrize("idx,n,enc", [(5, 1_300_003, None), (7, 700_001, None), (2, 900_004, 0), (2, 900_004, 1), (3, 2_000_004, 0),
                                       (5, 2047, None), (5, 2048 * 33 + 5, None), (2, 8192 * 3 + 64, 0)])
def test_both_generator_kernels(oracle, idx, n, enc, monkeypatch):
    """Integer samples run the tensor-core generator kernels (pcal_gen2.cuh for 2-bit, pcal_gen_mma.cuh for int8: integer
    MMAs over 31-bit fixed-point phasor digits); PCAL_GEN_MMA=0 selects the FFMA2 kernel of pcal_gen.cuh (the path of
    float32 input).  Both must match the oracle; lengths around one row and one 2^16-sample tile included."""
    w, dev, host = make(idx, n)
    if idx == 7:
        w = synth.replace(w, f_offset_hz=[1234.567])
    if enc is not None:
        w = synth.replace(w, encoding=enc)
    want = oracle_tones(oracle, w, host, 0)
    p1, T1, _ = gpu_run(w, dev, rotator="generator")
    assert p1.info().rotator_in_effect == 2
    assert_close(T1[0], want, f"mma generator cfg{idx}")
    monkeypatch.setenv("PCAL_GEN_MMA", "0")
    p2, T2, _ = gpu_run(w, dev, rotator="generator")
    monkeypatch.delenv("PCAL_GEN_MMA")
    # (the FFMA2 kernel multiplies in fp32: ~1e-7 of a typical tone, which a tone of a very short integration
    #  that happens to be small cannot meet per bin -- reading R28)
    assert_close(T2[0], want, f"ffma2 generator cfg{idx}", max_small=1 if n < 100_000 else 0)
    assert np.abs(T1 - T2).max() <= 2e-6 * np.abs(want).max()


@pytest.mark.parametrize("idx,n,splits", [
    (2, 1_000_004, [64, 64 * 1000, 64 * 9001]),
    (5, 800_003, [16, 16 * 4099, 16 * 30000]),
    (1, 500_001, [4, 4 * 77777]),
    (4, 90_001, [4, 4 * 10001]),
    (6, 600_004, [64 * 3, 64 * 5000]),
])
def test_split_point_invariance(oracle, idx, n, splits):
    """Successive pcal_extract calls are one continuous stream (R7, R8)."""
    w, dev, host = make(idx, n)
    p1, T1, P1 = gpu_run(w, dev)
    p2, T2, P2 = gpu_run(w, dev, splits=splits)
    if idx == 6:
        assert np.array_equal(p1.get_folded_i64(), p2.get_folded_i64())
    scale = np.abs(P1).max()
    # integer fold + fp64 rotate: only fp64 rounding may differ; fp32-run paths (generator, float32
    # input) regroup their short fp32 runs when the tiling shifts
    tol = 1e-6 if (idx in (1, 5)) else 1e-11
    assert np.abs(P1 - P2).max() <= tol * scale
    for c in range(0, w.n_channels, 5):
        assert_close(T2[c], oracle_tones(oracle, w, host, c), f"split cfg{idx} ch{c}")


def test_start_index_and_add_folded_time_sharding(oracle):
    """Two contexts each take half of the stream at its absolute index; summing P gives the whole."""
    from paper_2501_05993_b200 import binding
    w, dev, host = make(2, 1_000_000)
    half = 64 * 7000
    flat = dev.view(torch.uint8)
    a = binding.from_workload(w)
    a.extract(flat[: half // 4], half)
    b = binding.from_workload(w)
    b.set_start_index(half)
    b.extract(flat[half // 4:], w.n_samples - half)
    a.add_folded(b.get_folded())
    assert_close(a.finalize()[0], oracle_tones(oracle, w, host, 0), "time-sharded")


@pytest.mark.parametrize("idx,rot", [(2, None), (5, None), (2, "generator"), (3, "generator")])
def test_k_shift_unshifts_to_natural_order(oracle, idx, rot):
    """rotate by w_off + k w_comb, reorder the bins back."""
    w, dev, host = make(idx, 500_000 if idx == 5 else 600_004)
    p, T, P = gpu_run(w, dev, k_shift=w.n_bins // 4, rotator=rot)
    assert p.info().k_shift == w.n_bins // 4
    pr, pi = oracle_folded(oracle, w, host, 0)
    assert_close(T[0], oracle.dft(pr, pi), f"k-shift cfg{idx}")
    assert_close(P[0], pr.astype(np.float64) + 1j * pi.astype(np.float64), f"k-shift folded cfg{idx}")


def test_bitwise_determinism():
    w = synth.config(3).scaled(4_000_000)
    dev = synth.generate(w, DEV)
    for rot in ("lut", "generator"):
        _, T1, P1 = gpu_run(w, dev, rotator=rot)
        _, T2, P2 = gpu_run(w, dev, rotator=rot)
        assert np.array_equal(T1.view(np.uint64), T2.view(np.uint64))
        assert np.array_equal(P1.view(np.uint64), P2.view(np.uint64))


def test_bitwise_determinism_under_dynamic_tile_claims():
    """pcal_gen2.cuh hands a quarter of its tiles out through a device counter: which CTA gets which tile differs from run to
    run, the result must not (the per-position sums are exact integers, added with integer atomics).  60e6 samples = 915
    tiles = 229 batches, 81 of them claimed; also with the stream cut where the second piece starts in the middle of a row,
    and with other work keeping some SMs busy when the kernel starts."""
    w = synth.config(3).scaled(60_000_004)
    dev = synth.generate(w, DEV)
    ref = None
    for trial in range(4):
        if trial >= 2:      # unrelated kernels in flight on another stream: some CTAs start late and claim fewer tiles
            side = torch.cuda.Stream()
            with torch.cuda.stream(side):
                junk = torch.randn(64 << 20, device=DEV)
                for _ in range(3):
                    junk = junk * 1.0001 + 1.0
        _, T, P = gpu_run(w, dev, rotator="generator", splits=(20_000_128 + 64 * trial * 0,))
        torch.cuda.synchronize()
        if ref is None:
            ref = (T.copy(), P.copy())
        assert np.array_equal(T.view(np.uint64), ref[0].view(np.uint64)), trial
        assert np.array_equal(P.view(np.uint64), ref[1].view(np.uint64)), trial


@pytest.mark.parametrize("idx,n,rot", [(2, 4, None), (2, 60, None), (2, 64, None), (2, 68, None), (5, 1, None), (5, 15, None), (5, 16, None),
                                       (5, 17, None), (1, 1, None), (1, 3, None), (1, 4, None), (1, 5, None), (4, 1, None), (4, 3, None),
                                       (4, 4, None), (4, 5, None), (3, 2052, None),
                                       (3, 4, "generator"), (3, 508, "generator"), (3, 512, "generator"), (3, 516, "generator"),
                                       (3, 512 * 128 - 4, "generator"), (3, 512 * 128 + 4, "generator"), (2, 60, "generator"), (2, 516, "generator"),
                                       (8, 1, "generator"), (8, 3, "generator"), (8, 1020, "generator"), (8, 1024, "generator"), (8, 1028, "generator"),
                                       (8, 1024 * 147 + 8, "generator"), (8, 1024 * 148, "generator"), (8, 1024 * 149 - 4, "generator"),
                                       (8, 1024 * 64 * 148 + 1024 * 3 + 4, "generator")])
def test_tiny_and_ragged_lengths(oracle, idx, n, rot):
    """Segments shorter than / equal to / just above one 16-byte vector (tail-only and 1-vector paths); for the generator
    kernel of 2-bit samples: around one row (512 samples) and one tile (128 rows); for the float32 generator kernel: around
    one CTA iteration (1024 samples), one iteration per CTA (fewer iterations than CTAs, exactly as many, one more) and a
    little more than one full tile per CTA."""
    w, dev, host = make(idx, n)
    if rot:
        w = synth.replace(w, rotator=rot)
    if dev.numel() * dev.element_size() < 16:  # keep the device buffer 16-byte aligned & readable
        pad = torch.zeros(16, dtype=torch.uint8, device=DEV)
        pad[: dev.numel() * dev.element_size()] = dev.view(torch.uint8)
        dev = pad
    p, T, P = gpu_run(w, dev)
    for c in range(w.n_channels):
        pr, pi = oracle_folded(oracle, w, host, c)
        want = pr.astype(np.float64) + 1j * pi.astype(np.float64)
        empty = want == 0                                    # bins no sample fell into: exactly zero on both sides
        assert not P[c][empty].any(), (idx, n, c)
        if (~empty).any():
            assert_close(P[c][~empty], want[~empty], f"cfg{idx} n={n} ch{c} folded")
        wt = oracle.dft(pr, pi)
        small = 1e-2 if w.bits == 32 else 1e-3               # reading R28: "small" tones, float32 input: 1e-2 of the largest
        assert np.abs(T[c] - wt).max() <= 1e-5 * np.abs(wt).max() * small + 1e-300, (idx, n, c)    # every tone to 1e-8 (1e-7) of the largest ...
        big = np.abs(wt) >= small * np.abs(wt).max()
        assert_close(T[c][big], wt[big], f"cfg{idx} n={n} ch{c} tones")                              # ... and per tone where it is not a cancellation


def test_impulse_and_reset(oracle):
    """x = delta[n - n1] (float32): T[i] = e^{-j(i w_comb + w_off) n1}; reset restarts the index."""
    from paper_2501_05993_b200 import binding
    n1, N = 123_457, 200_000
    x = torch.zeros(N, dtype=torch.float32, device=DEV)
    x[n1] = 1.0
    for rot in (binding.ROT_LUT, binding.ROT_GENERATOR):
        p = binding.Pcal(32e6, 1e6, 10e3, 32, binding.ENC_IEEE_FLOAT, 1)
        p.set_rotator(rot)
        p.extract(x)
        T = p.finalize()[0]
        want = oracle.extract(x.cpu().numpy(), oracle.F32, 1, 0, N, 0, 32e6, 1e6, 10e3)
        assert np.abs(T - want).max() < 1e-6
        assert abs(abs(T[5]) - 1.0) < 1e-6
        p.reset()
        assert p.info().n_processed == 0
        p.extract(x)
        assert np.abs(p.finalize()[0] - want).max() < 1e-6
        p.extract(x)  # continues the stream: second copy starts at absolute index N
        want2 = want + oracle.extract(x.cpu().numpy(), oracle.F32, 1, 0, N, N, 32e6, 1e6, 10e3)
        assert np.abs(p.finalize()[0] - want2).max() < 1e-6


def test_extract_host_matches_device_path():
    from paper_2501_05993_b200 import binding
    w = synth.config(2).scaled(3_000_004)
    dev = synth.generate(w, DEV)
    _, T, _ = gpu_run(w, dev)
    pinned = dev.cpu().pin_memory()
    p = binding.from_workload(w)
    p.extract_host(pinned, w.n_samples)
    assert np.array_equal(p.finalize().view(np.uint64), T.view(np.uint64))


def test_error_codes():
    from paper_2501_05993_b200 import binding as B
    for args in [(32e6, 3e6, 0.0, 2, 0, 1), (32e6, 1e6, 0.0, 3, 0, 1), (32e6, 1e6, 0.0, 8, 0, 1),
                 (32e6, 1e6, 0.0, 2, 0, 3), (32e6, 1e6, 0.0, 8, 2, 2), (32e6, 1e6, 40e6, 2, 0, 1)]:
        with pytest.raises(B.PcalError) as e:
            B.Pcal(*args)
        assert e.value.code == -1, args
    p = B.Pcal(32e6, 1e6, 10e3, 2, B.ENC_OFFSET_BINARY, 1)
    buf = torch.zeros(4096, dtype=torch.uint8, device=DEV)
    with pytest.raises(B.PcalError) as e:
        p.extract(buf[1:], 64)                       # misaligned pointer
    assert e.value.code == -2
    p.extract(buf, 0)                                # n = 0 is a no-op
    assert p.info().n_processed == 0
    p.extract(buf, 4096 * 4)
    with pytest.raises(B.PcalError) as e:
        p.set_rotator(B.ROT_GENERATOR)               # after the first extract
    assert e.value.code == -3
    with pytest.raises(B.PcalError) as e:
        p.get_folded_i64()                           # rotated: no integer bins
    assert e.value.code == -3
    q = B.Pcal(1024e6, 1e6, 1234.567, 8, B.ENC_TWOS_COMPLEMENT, 1)
    q.set_rotator(B.ROT_LUT)
    with pytest.raises(B.PcalError) as e:
        q.extract(torch.zeros(4096, dtype=torch.int8, device=DEV))
    assert e.value.code == -4                        # LUT of impractical length


@pytest.mark.parametrize("idx,n,rot", [(2, 250_000_004, None), (4, 14_000_003, None), (5, 90_000_003, None),
                                       (3, 90_000_004, "generator"), (8, 40_000_001, "generator")])
def test_segments_longer_than_one_launch(oracle, idx, n, rot, monkeypatch):
    """A segment that exceeds the per-launch limits (16-bit lanes of the fold kernel, 256-entry resync
    table of the generator kernel) is cut into several launches by the host; PCAL_SMALL_PIECES=1 lowers
    both limits so that this size already needs 2-4 of them.  Result = one continuous stream."""
    monkeypatch.setenv("PCAL_SMALL_PIECES", "1")
    w, dev, host = make(idx, n)
    p, T, P = gpu_run(w, dev, rotator=rot)
    assert p.info().kernel_launches >= 2 + 1, p.info().kernel_launches         # >= 2 pieces (one kernel each) + the DFT
    for c in range(0, w.n_channels, 6):
        assert_close(T[c], oracle_tones(oracle, w, host, c, threads=8), f"cfg{idx} ch{c} multi-launch")
    monkeypatch.delenv("PCAL_SMALL_PIECES")
    p2, T2, _ = gpu_run(w, dev, rotator=rot)
    assert p2.info().kernel_launches < p.info().kernel_launches
    assert_close(T, T2, f"cfg{idx} pieces vs single launch")


@pytest.mark.parametrize("idx,n", [(1, 1_300_001), (2, 1_300_004), (3, 2_600_036), (4, 200_003), (6, 1_300_004),
                                   (7, 1_300_003), (8, 1_300_001), (2, 60), (4, 7)])
def test_unfused_reduction_kernels_agree_with_the_fused_tail(oracle, idx, n, monkeypatch):
    """The LUT path reduces, rotates and accumulates inside the fold kernel (pcal_tail.cuh: the CTAs that
    finish last).  PCAL_NO_FUSED_TAIL=1 selects the separate reduce_replicas/rotate_fold kernels instead
    (also the fall-back for geometries with very many slot groups); both must match the oracle, and each
    other to fp64 rounding (bit-identical integer bins)."""
    w, dev, host = make(idx, n)
    p1, T1, P1 = gpu_run(w, dev)
    monkeypatch.setenv("PCAL_NO_FUSED_TAIL", "1")
    p2, T2, P2 = gpu_run(w, dev)
    monkeypatch.delenv("PCAL_NO_FUSED_TAIL")
    if n > 1000:
        assert p2.info().kernel_launches == p1.info().kernel_launches + 2
        for c in range(0, w.n_channels, 5):
            want = oracle_tones(oracle, w, host, c)
            assert_close(T1[c], want, f"fused cfg{idx} ch{c}")
            assert_close(T2[c], want, f"unfused cfg{idx} ch{c}")
    scale = np.abs(P1).max()
    # float32 input: the fused geometry folds modulo a larger period, which regroups the short fp32 runs
    assert np.abs(P1 - P2).max() <= (1e-6 if idx in (1, 8) else 1e-11) * scale
    if idx in (6, 7):
        assert np.array_equal(p1.get_folded_i64(), p2.get_folded_i64())


@pytest.mark.parametrize("idx,n,rot", [(2, 3_000_004, None), (4, 300_003, None), (5, 2_000_003, None), (3, 2_000_004, "generator")])
def test_input_ready_promise_changes_nothing(oracle, idx, n, rot):
    """pcal_set_input_ready(1) lets the streaming kernel read its input before the previous segment's small
    kernels have finished (programmatic dependent launch); many back-to-back segments and resets must give
    bit-identical results to the conservative order, and match the oracle."""
    w, dev, host = make(idx, n)
    if rot:
        w = synth.replace(w, rotator=rot)
    from paper_2501_05993_b200 import binding
    outs = []
    for ready in (False, True):
        p = binding.from_workload(w)
        p.set_input_ready(ready)
        res = []
        pinned = torch.empty((w.n_channels, w.n_bins), dtype=torch.complex128).pin_memory()
        for rep in range(6):                      # reset + extract + finalize_async back to back, no sync
            p.reset()
            p.extract(dev, n)
            p.finalize_async(pinned)
        torch.cuda.synchronize()
        res.append(pinned.numpy().copy())
        p.reset()
        bytes_per_t = w.bits * w.n_channels // 8 if w.bits * w.n_channels >= 8 else None
        half = (n // 2) // 64 * 64
        flat = dev.view(-1).view(dtype=torch.uint8)
        cut = half * w.bits * w.n_channels // 8
        p.extract(flat[:cut], half)
        p.extract(flat[cut:], n - half)
        res.append(p.finalize())
        outs.append(res)
        p.destroy()
    assert np.array_equal(outs[0][0], outs[1][0]) and np.array_equal(outs[0][1], outs[1][1])
    assert_close(outs[1][0][0], oracle_tones(oracle, w, host, 0), f"cfg{idx} input_ready")


@pytest.mark.parametrize("rot", ["lut", "generator"])
@pytest.mark.parametrize("C,enc", [(2, 0), (4, 1), (8, 0), (16, 1)])
def test_every_power_of_two_channel_count(oracle, C, enc, rot):
    """Demultiplexing ("several baseband channels"): one field of 2C bits per time sample, packed
    LSB-first; channel c in bits 2c..2c+1 of its field.  Random codes.  Table rotation: mixed zero / non-zero
    offsets.  Generator rotation: a different offset with an impractical table per channel, one
    channel left unrotated; two segments, the second one starting in the middle of a row."""
    from paper_2501_05993_b200 import binding
    n = 300_004
    rs = np.random.RandomState(4200 + C)
    codes = rs.randint(0, 4, size=(n, C)).astype(np.uint8)
    flat = codes.reshape(-1, 4)
    packed = (flat[:, 0] | (flat[:, 1] << 2) | (flat[:, 2] << 4) | (flat[:, 3] << 6)).astype(np.uint8)
    gen = rot == "generator"
    if gen:
        offs = [0.0 if c == 1 else 1234.567 + 100321.0123 * c for c in range(C)]
    else:
        offs = [0.0 if c % 3 == 0 else 10e3 * (1 + c) for c in range(C)]
    p = binding.Pcal(64e6, 1e6, 0.0, 2, enc, C)
    p.set_channel_offsets(offs)
    p.set_rotator(binding.ROT_GENERATOR if gen else binding.ROT_LUT)
    dev = torch.from_numpy(packed).cuda()
    if gen:
        cut = 100_032 * 2 * C // 8       # bytes of the first 100 032 time samples (16-byte aligned for every C)
        p.extract(dev[:cut], 100_032)
        p.extract(dev[cut:], n - 100_032)
        assert p.info().rotator_in_effect == binding.ROT_GENERATOR
    else:
        p.extract(dev, n)
    T, P = p.finalize(), p.get_folded()
    fmt = oracle.TWO_BIT_SIGN_MAG if enc else oracle.TWO_BIT_OFFSET_BINARY
    for c in range(C):
        pr, pi = oracle.fold_ld(packed, fmt, C, c, 0, 1, n, 0, 64e6, 1e6, offs[c], tabulated=not gen)
        assert_close(P[c], pr.astype(np.float64) + 1j * pi.astype(np.float64), f"C={C} ch{c} folded")
        assert_close(T[c], oracle.dft(pr, pi), f"C={C} ch{c} tones")
        if offs[c] == 0.0 and not gen:
            want = oracle.fold_i64(packed, fmt, C, c, 0, 1, n, 0, 64)
            assert np.array_equal(P[c].real, want.astype(np.float64)) and not P[c].imag.any()
    p.destroy()


@pytest.mark.parametrize("chunks", [8, 16, 32])
@pytest.mark.parametrize("C,enc", [(1, 0), (2, 1), (4, 0), (16, 1)])
def test_generator_row_lengths(oracle, monkeypatch, C, enc, chunks):
    """The 2-bit generator kernel with rows of 8, 16 and 32 sixteen-byte chunks (PCAL_G2_CHUNKS, read when the context is set
    up): every combination of chunks per consumer warp, generator warps and items per generator lane, with the row table in
    shared memory and without.  A length with a ragged last tile and a ragged tail; tones through the fused DFT."""
    from paper_2501_05993_b200 import binding
    monkeypatch.setenv("PCAL_G2_CHUNKS", str(chunks))
    n = 1_300_004
    rs = np.random.RandomState(4300 + 10 * C + chunks)
    packed = rs.randint(0, 256, size=n * 2 * C // 8).astype(np.uint8)
    offs = [1234.567 + 100321.0123 * c for c in range(C)]
    p = binding.Pcal(64e6, 1e6, 0.0, 2, enc, C)
    p.set_channel_offsets(offs)
    p.set_rotator(binding.ROT_GENERATOR)
    dev = torch.from_numpy(packed).cuda()
    out = torch.empty((C, 64), dtype=torch.complex128).pin_memory()
    p.integrate(dev.data_ptr(), n, out.data_ptr())
    torch.cuda.synchronize()
    assert p.info().rotator_in_effect == binding.ROT_GENERATOR
    P = p.get_folded()
    fmt = oracle.TWO_BIT_SIGN_MAG if enc else oracle.TWO_BIT_OFFSET_BINARY
    for c in range(C):
        pr, pi = oracle.fold_ld(packed, fmt, C, c, 0, 1, n, 0, 64e6, 1e6, offs[c], tabulated=False)
        assert_close(P[c], pr.astype(np.float64) + 1j * pi.astype(np.float64), f"C={C} chunks={chunks} ch{c} folded")
        assert_close(out[c].numpy(), oracle.dft(pr, pi), f"C={C} chunks={chunks} ch{c} tones")
    p.destroy()


@pytest.mark.parametrize("C,ncls", [(8, "1"), (16, "1"), (16, "2")])
def test_generator_byte_classes_per_launch(oracle, monkeypatch, C, ncls):
    """Words of 8 / 16 channels through the 2-bit generator kernel with fewer byte classes per launch than the default (all of
    them in one launch): PCAL_G2_NCLS = 1 (one launch per four channels) and 2 (16 channels in two launches)."""
    from paper_2501_05993_b200 import binding
    monkeypatch.setenv("PCAL_G2_NCLS", ncls)
    n = 700_004
    rs = np.random.RandomState(4400 + C + int(ncls))
    packed = rs.randint(0, 256, size=n * 2 * C // 8).astype(np.uint8)
    offs = [1234.567 + 100321.0123 * c for c in range(C)]
    p = binding.Pcal(64e6, 1e6, 0.0, 2, 1, C)
    p.set_channel_offsets(offs)
    p.set_rotator(binding.ROT_GENERATOR)
    dev = torch.from_numpy(packed).cuda()
    launches0 = p.info().kernel_launches
    p.extract(dev, n)
    assert p.info().kernel_launches - launches0 == C // 4 // int(ncls)
    T, P = p.finalize(), p.get_folded()
    for c in sorted(set(int(x) for x in rs.randint(0, C, size=5))):
        pr, pi = oracle.fold_ld(packed, oracle.TWO_BIT_SIGN_MAG, C, c, 0, 1, n, 0, 64e6, 1e6, offs[c], tabulated=False, threads=8)
        assert_close(P[c], pr.astype(np.float64) + 1j * pi.astype(np.float64), f"C={C} ncls={ncls} ch{c} folded")
        assert_close(T[c], oracle.dft(pr, pi), f"C={C} ncls={ncls} ch{c} tones")
    p.destroy()


def test_exchange_step_in_one_launch(oracle):
    """What bench.py does per step with N ranks, emulated on one GPU: every "rank" folds its time shard at
    its absolute start index, the bins are gathered into one buffer (stand-in for the NCCL all-gather) and
    pcal_set_folded_sum_dev adds them in rank order."""
    from paper_2501_05993_b200 import binding
    w, dev, host = make(2, 1_200_000)
    world, per = 3, 400_000
    flat = dev.view(torch.uint8)
    gathered = torch.empty(world * w.n_bins * 2, dtype=torch.float64, device=DEV)
    ctxs = []
    for r in range(world):
        p = binding.from_workload(w)
        p.set_start_index(r * per)
        p.extract(flat[r * per // 4:(r + 1) * per // 4], per)
        p.get_folded_dev(gathered[r * w.n_bins * 2:(r + 1) * w.n_bins * 2])
        ctxs.append(p)
    torch.cuda.synchronize()
    outs = []
    for p in ctxs:                                  # every rank ends with the same bits
        p.reset()
        p.set_folded_sum_dev(gathered, world)
        outs.append(p.finalize())
    assert all(np.array_equal(outs[0], o) for o in outs[1:])
    assert_close(outs[0][0], oracle_tones(oracle, w, host, 0), "gathered exchange")


@pytest.mark.parametrize("n_bins", [375, 1100, 363])
@pytest.mark.parametrize("unfused", [False, True])
def test_float32_odd_slot_group_counts(oracle, n_bins, unfused, monkeypatch):
    """float32 vectors hold 4 samples, so a slot-group count q that is odd makes q * 4 * 32 replica sums -- not a multiple
    of the 256 threads of reduce_replicas_kernel's CTAs (its last CTA is partly empty).  Both reduction paths."""
    if unfused:
        monkeypatch.setenv("PCAL_NO_FUSED_TAIL", "1")
    w = synth.Workload("f32_odd_q", 1, n_bins * 1e6, 1e6, [0.0], 32, 3, 1_500_003, 0.05, 1.0, [5e-9], 4250)
    dev = synth.generate(w, DEV)
    host = dev.cpu().numpy()
    p, T, P = gpu_run(w, dev)
    pr, pi = oracle_folded(oracle, w, host, 0)
    # (without rotation the bins are REAL sums of ~4000 float32 samples each, of which a few per cent cancel to ~1 % of a typical
    #  bin: the fold kernel adds float32 samples in fp64 for that reason, and no bin needs the rule of reading R28)
    assert_close(P[0], pr.astype(np.float64) + 1j * pi.astype(np.float64), f"N_bins={n_bins} folded")
    assert_close(T[0][1:n_bins // 2], oracle.dft(pr, pi)[1:n_bins // 2], f"N_bins={n_bins} in-band tones")
    p.destroy()


def test_first_call_on_a_side_stream(oracle):
    """Everything a context sets up lazily (tables, counters) is issued on the stream handed to pcal_extract: the very
    first call may be made on a non-blocking side stream (every torch.cuda.Stream is one)."""
    for idx, n, rot in [(2, 2_000_004, None), (3, 2_000_004, "generator"), (4, 300_003, None)]:
        w, dev, host = make(idx, n)
        if rot:
            w = synth.replace(w, rotator=rot)
        torch.cuda.synchronize()
        side = torch.cuda.Stream()
        with torch.cuda.stream(side):
            p = __import__("paper_2501_05993_b200.binding", fromlist=["x"]).from_workload(w)
            p.extract(dev, n)
            T = p.finalize()
        assert_close(T[0], oracle_tones(oracle, w, host, 0), f"cfg{idx} first call on a side stream")
        p.destroy()


def test_exact_integer_bins_survive_the_exchange(oracle):
    """Time-sharded integer input without rotation: after the exchange step (pcal_set_folded_sum_dev, pcal_add_folded_dev,
    pcal_add_folded) pcal_get_folded_i64 still returns the exact bins of the WHOLE stream."""
    from paper_2501_05993_b200 import binding
    w, dev, host = make(6, 1_200_000)                  # config 2 with f_offset = 0
    fmt = oracle.TWO_BIT_OFFSET_BINARY
    want = oracle.fold_i64(host, fmt, 1, 0, 0, 1, w.n_samples, 0, w.n_bins)
    flat = dev.view(torch.uint8)
    world, per = 3, 400_000
    gathered = torch.empty(world * w.n_bins * 2, dtype=torch.float64, device=DEV)
    ctxs = []
    for r in range(world):
        p = binding.from_workload(w)
        p.set_start_index(r * per)
        p.extract(flat[r * per // 4:(r + 1) * per // 4], per)
        p.get_folded_dev(gathered[r * w.n_bins * 2:(r + 1) * w.n_bins * 2])
        ctxs.append(p)
    ctxs[0].set_folded_sum_dev(gathered, world)
    assert np.array_equal(ctxs[0].get_folded_i64()[0], want)
    ctxs[1].add_folded_dev(gathered[0:w.n_bins * 2])                       # rank 1 + rank 0 + rank 2, one at a time
    ctxs[1].add_folded(ctxs[2].get_folded())
    assert np.array_equal(ctxs[1].get_folded_i64()[0], want)
    for p in ctxs:
        p.destroy()


def test_sharding_package_on_one_gpu(oracle):
    """sharding.ShardedIntegrator and sharding.series_sharded (what bench.py --gpus N and the gloo test run) with real
    contexts: three "ranks" in one process, two lanes each, three periods; then a two-period series with one exchange."""
    from paper_2501_05993_b200 import binding, sharding
    w, dev, host = make(2, 1_200_000)
    world, per = 3, 400_000
    flat = dev.view(torch.uint8)
    # every rank's gathered buffers must exist before anybody copies into them: one warm-up round builds them
    want = oracle_tones(oracle, w, host, 0)
    ranks = []
    for r in range(world):
        ctxs = [binding.from_workload(w), binding.from_workload(w)]
        ranks.append({"ctxs": ctxs, "local": [torch.empty(w.n_bins * 2, dtype=torch.float64, device=DEV) for _ in range(3)]})
    n2 = w.n_bins * 2
    outs = [[torch.zeros((1, w.n_bins), dtype=torch.complex128).pin_memory() for _ in range(3)] for _ in range(world)]
    # the exchange, in process: period k of every rank writes into one gathered tensor per period, shared by the ranks
    shared = [torch.empty(world * n2, dtype=torch.float64, device=DEV) for _ in range(3)]

    class Done:
        def wait(self):
            pass

    integ = []
    for r in range(world):
        s = sharding.ShardedIntegrator(ranks[r]["ctxs"], 1, w.n_bins, world, DEV, gather=None)
        integ.append(s)
    for k in range(3):
        for r in range(world):
            s = integ[r]
            lane = s.lanes[s.count % 2]

            def gather(gathered, local, k=k, r=r, lane=lane):
                shared[k][r * n2:(r + 1) * n2].copy_(local)
                lane["gathered"] = shared[k]              # every rank reads the same gathered bins
                return Done()
            s.gather = gather
            s.submit(flat[r * per // 4:(r + 1) * per // 4], per, r * per, outs[r][k])
    for s in integ:
        s.drain()
    torch.cuda.synchronize()
    for r in range(world):
        for k in range(3):
            assert np.array_equal(outs[r][k].numpy(), outs[0][0].numpy())     # every rank, every period: the same bits
    assert_close(outs[0][0].numpy()[0], want, "sharded integrator")
    # series: two periods of 600 000 samples, three ranks, ONE exchange
    half, sh = 600_000, 200_000
    big = torch.zeros(world * 2 * n2, dtype=torch.float64, device=DEV)
    pf = torch.zeros((2, 1, w.n_bins), dtype=torch.complex128, device=DEV)
    pt = torch.zeros_like(pf)
    for r in range(world):
        shards = [flat[(k * half + r * sh) // 4:(k * half + (r + 1) * sh) // 4] for k in range(2)]
        starts = [k * half + r * sh for k in range(2)]

        def gather(gathered, local, r=r):
            big.view(world, -1)[r].copy_(local)
            gathered.copy_(big)
            return Done()
        sharding.series_sharded(ranks[r]["ctxs"][0], shards, sh, starts, 1, w.n_bins, world, DEV, pf, pt, gather=gather)
    torch.cuda.synchronize()                          # (the last rank saw every rank's bins)
    hb = host.reshape(-1).view(np.uint8)
    for k in range(2):
        pr, pi = oracle.fold_ld(hb[k * half // 4:(k + 1) * half // 4], oracle.TWO_BIT_OFFSET_BINARY, 1, 0, 0, 1, half, k * half,
                                w.f_s_hz, w.f_comb_hz, w.f_offset_hz[0])
        assert_close(pf[k, 0].cpu().numpy(), pr.astype(np.float64) + 1j * pi.astype(np.float64), f"series period {k} folded")
        assert_close(pt[k, 0].cpu().numpy(), oracle.dft(pr, pi), f"series period {k} tones")
    for rk in ranks:
        for c in rk["ctxs"]:
            c.destroy()


@pytest.mark.parametrize("idx,n,rot", [(2, 2_000_004, None), (1, 700_001, None), (4, 150_003, None), (3, 1_500_004, None),
                                       (3, 9_000_004, "generator"), (2, 2_000_004, "generator")])
def test_pipelined_launches_stress_and_graph_replay(oracle, idx, n, rot):
    """Consecutive fold launches overlap (device-side sequence numbers instead of grid-wide waits, pcal_tail.cuh).  Many
    back-to-back integration periods over different inputs, each into its own pinned buffer, must equal the result of the
    same period run alone, bit for bit -- launched directly and replayed from a CUDA graph (frozen parameters: the ring
    slot and the ordering are derived on the device)."""
    from dataclasses import replace
    from paper_2501_05993_b200 import binding
    w = synth.config(idx).scaled(n)
    if rot:
        w = replace(w, rotator=rot)
    bufs = [synth.generate(replace(w, seed=w.seed + 31 * k), DEV) for k in range(3)]
    p = binding.from_workload(w)
    alone = []
    ref = torch.zeros((w.n_channels, w.n_bins), dtype=torch.complex128).pin_memory()
    for b in bufs:                                   # reference: the same call, one period at a time, synchronised
        p.integrate(b, n, ref); torch.cuda.synchronize(); alone.append(ref.numpy().copy())
    assert_close(alone[0][0], oracle_tones(oracle, w, bufs[0].cpu().numpy(), 0), f"cfg{idx} alone")
    p.set_input_ready(True)
    reps = 40
    outs = [torch.zeros((w.n_channels, w.n_bins), dtype=torch.complex128).pin_memory() for _ in range(reps)]
    for r in range(reps):
        p.integrate(bufs[r % 3], n, outs[r])
    torch.cuda.synchronize()
    for r in range(reps):
        assert np.array_equal(outs[r].numpy(), alone[r % 3]), f"direct launch {r}"
    # the same through a CUDA graph: 6 periods captured once, replayed 7 times, interleaved with direct launches
    gouts = [torch.zeros((w.n_channels, w.n_bins), dtype=torch.complex128).pin_memory() for _ in range(6)]
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        with torch.cuda.graph(g, stream=side):
            for k in range(6):
                p.integrate(bufs[k % 3], n, gouts[k])
    torch.cuda.current_stream().wait_stream(side)
    for it in range(7):
        for o in gouts:
            o.zero_()
        g.replay()
        if it % 2:
            p.integrate(bufs[1], n, outs[0])
        torch.cuda.synchronize()
        for k in range(6):
            assert np.array_equal(gouts[k].numpy(), alone[k % 3]), f"replay {it} period {k}"
        if it % 2:
            assert np.array_equal(outs[0].numpy(), alone[1])
    p.destroy()


@pytest.mark.parametrize("f_s,f_comb,f_off,bits,enc,n", [
    (50e6, 1e6, 10e3, 2, 0, 1_000_064),      # N_bins = 50 (not a power of two), L = 5000
    (25e6, 1e6, 0.0, 2, 1, 800_000),          # N_bins = 25 (odd), zero offset: integer-exact
    (48e6, 2e6, 30e3, 32, 3, 600_001),        # N_bins = 24, float32, L = 1600
    (96e6, 1e6, 250e3, 8, 2, 900_003),        # N_bins = 96 (> 64: DFT kernel), int8 through the LUT path, L = 384
])
def test_bin_counts_that_are_not_powers_of_two(oracle, f_s, f_comb, f_off, bits, enc, n):
    """The fold geometry, the fused tail and its DFT make no power-of-two assumption about N_bins."""
    from paper_2501_05993_b200 import binding
    w = synth.Workload("odd_bins", 1, f_s, f_comb, [f_off], bits, enc, n, 0.05 if bits != 8 else 1.0, 1.0 if bits != 8 else 20.0, [5e-9], 4242)
    dev = synth.generate(w, DEV)
    host = dev.cpu().numpy()
    p, T, P = gpu_run(w, dev)
    assert p.info().rotator_in_effect == 1
    pr, pi = oracle_folded(oracle, w, host, 0)
    assert_close(P[0], pr.astype(np.float64) + 1j * pi.astype(np.float64), "folded")
    assert_close(T[0], oracle.dft(pr, pi), "tones")
    if f_off == 0.0 and bits != 32:
        want = oracle.fold_i64(host, oracle_fmt(oracle, w), 1, 0, 0, 1, n, 0, w.n_bins)
        assert np.array_equal(p.get_folded_i64()[0], want)
    out = torch.zeros((1, w.n_bins), dtype=torch.complex128).pin_memory()
    p.integrate(dev, n, out)
    torch.cuda.synchronize()
    assert np.abs(out.numpy() - T).max() <= 1e-12 * np.abs(T).max()
    p.destroy()


@pytest.mark.parametrize("f_s,f_comb,f_off,bits,enc,n", [
    (50e6, 1e6, 1234.567, 2, 0, 1_000_064),    # N_bins = 50: rows of 1600 samples (25 sixteen-byte chunks)
    (25e6, 1e6, 777.123456, 2, 1, 800_000),    # N_bins = 25 (odd), SIGN_MAG
    (48e6, 2e6, 30e3 + 0.5, 2, 0, 600_004),    # N_bins = 24: rows of 576 samples (9 chunks)
    (96e6, 1e6, 250e3 + 1e-3, 2, 0, 900_004),  # N_bins = 96
    (2048e6, 1e6, 1234.567, 2, 0, 3_000_004),  # N_bins = 2048: the longest row (32 chunks)
    (1000e6, 1e6, 1234.567, 2, 0, 2_000_004),  # N_bins = 1000: rows of 8000 samples, in column blocks
    (50e6, 1e6, 1234.567, 8, 2, 1_000_003),    # int8, N_bins = 50 does not divide 2048: FFMA2 kernel, 4000 samples per CTA iteration
    (1000e6, 1e6, 777.123456, 8, 2, 2_000_001),  # int8, N_bins = 1000
    (48e6, 2e6, 30e3 + 0.5, 32, 3, 600_001),   # float32, N_bins = 24: 1008 samples per CTA iteration
    (1000e6, 1e6, 1234.567, 32, 3, 1_500_001), # float32, N_bins = 1000
])
def test_generator_bin_counts_that_are_not_powers_of_two(oracle, f_s, f_comb, f_off, bits, enc, n):
    """The generator path needs an integer N_bins only (eq. 2.2): offsets whose table is impractical."""
    from paper_2501_05993_b200 import binding
    w = synth.Workload("odd_bins_gen", 1, f_s, f_comb, [f_off], bits, enc, n, 0.05 if bits != 8 else 1.0, 1.0 if bits != 8 else 20.0,
                       [5e-9], 4243, rotator="generator")
    dev = synth.generate(w, DEV)
    host = dev.cpu().numpy()
    p, T, P = gpu_run(w, dev, splits=(300_032,))
    assert p.info().rotator_in_effect == 2
    pr, pi = oracle_folded(oracle, w, host, 0, tabulated=False)
    assert_close(P[0], pr.astype(np.float64) + 1j * pi.astype(np.float64), "folded")
    assert_close(T[0], oracle.dft(pr, pi), "tones")
    p.destroy()


def test_two_contexts_interleaved_on_one_stream(oracle):
    """Contexts keep their own tickets and progress counters: alternating overlapping periods of two different
    configurations on one stream (what the time-sharded bench does with its two lanes) leaves both exact."""
    from paper_2501_05993_b200 import binding
    wa, da, ha = make(2, 1_500_004)
    wb, db, hb = make(4, 120_003)
    pa, pb = binding.from_workload(wa), binding.from_workload(wb)
    for p_ in (pa, pb):
        p_.set_input_ready(True)
    oa = [torch.zeros((wa.n_channels, wa.n_bins), dtype=torch.complex128).pin_memory() for _ in range(12)]
    ob = [torch.zeros((wb.n_channels, wb.n_bins), dtype=torch.complex128).pin_memory() for _ in range(12)]
    for k in range(12):
        pa.integrate(da, wa.n_samples, oa[k])
        pb.integrate(db, wb.n_samples, ob[k])
        if k % 3 == 2:
            pa.finalize_async(oa[k])              # a DFT kernel of one context between the folds of the other
    torch.cuda.synchronize()
    want_a = oracle_tones(oracle, wa, ha, 0)
    for k in range(12):
        assert np.array_equal(oa[k].numpy(), oa[0].numpy()) or np.abs(oa[k].numpy() - oa[0].numpy()).max() <= 1e-12 * np.abs(want_a).max()
        assert np.array_equal(ob[k].numpy(), ob[0].numpy())
    assert_close(oa[0].numpy()[0], want_a, "context A")
    for c in (0, 7, 15):
        assert_close(ob[0].numpy()[c], oracle_tones(oracle, wb, hb, c), f"context B ch{c}")
    pa.destroy(); pb.destroy()
