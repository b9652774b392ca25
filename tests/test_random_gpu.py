"""Seeded random configurations through the C ABI against the oracle: sample type, channel count, encoding, N_bins (powers
of two and not), per-channel offsets (zero, rational, non-rational), rotator request, length, segment cuts and start index
are all drawn from the seed.  Every folded bin and every tone of the checked channels is held to north_star's bar
(pcal_testlib.assert_close).  The point is the combinations the hand-written cases do not list.
"""
import os

import numpy as np
import pytest
import torch

from paper_2501_05993_b200 import synth
from pcal_testlib import assert_close

pytestmark = pytest.mark.gpu

DEV = "cuda"
N_BINS = [16, 24, 32, 50, 64, 96, 128, 256, 500, 512, 1024]


def draw(seed):
    rs = np.random.RandomState(90_000 + seed)
    kind = ["2bit", "2bit", "2bit", "i8", "f32"][rs.randint(5)]
    C = int([1, 1, 2, 4, 8, 16][rs.randint(6)]) if kind == "2bit" else 1
    bits = {"2bit": 2, "i8": 8, "f32": 32}[kind]
    enc = {"2bit": int(rs.randint(2)), "i8": synth.ENC_TWOS_COMPLEMENT, "f32": synth.ENC_IEEE_FLOAT}[kind]
    n_bins = int(N_BINS[rs.randint(len(N_BINS))])
    f_comb = 1e6
    f_s = n_bins * f_comb
    style = rs.randint(3)                      # 0: rational offsets (some zero), 1: non-rational, 2: all zero
    offs = []
    for c in range(C):
        if style == 2 or (style == 0 and rs.randint(4) == 0):
            offs.append(0.0)
        elif style == 0:
            offs.append(float(10e3 * (1 + rs.randint(99))))
        else:
            offs.append(float(1234.567 + 100321.0123 * c + rs.randint(1000)))
    rot = ["auto", "auto", "generator"][rs.randint(3)] if style != 2 else "auto"
    # whole bytes for one channel, whole 32-bit words for several (include/pcal.h, pcal_extract)
    unit = (4 if C == 1 else 32 // (2 * C)) if bits == 2 else 1
    n = int(rs.randint(1_000, max(2_000, 1_600_000 // C)))
    n -= n % unit
    per16 = 128 // (bits * C)                  # time samples per 16 bytes: cuts must keep the next segment 16-byte aligned
    cuts = sorted(set(int(rs.randint(1, n // per16)) * per16 for _ in range(rs.randint(3)))) if n > 4 * per16 else []
    start = int([0, 0, rs.randint(1, 10**6), rs.randint(1, 2**40)][rs.randint(4)])
    if kind == "f32":
        data = rs.standard_normal(n).astype(np.float32)
    elif kind == "i8":
        data = rs.randint(-127, 128, size=n).astype(np.int8)
    else:
        data = rs.randint(0, 256, size=n * 2 * C // 8).astype(np.uint8)
    return dict(kind=kind, C=C, bits=bits, enc=enc, n_bins=n_bins, f_s=f_s, f_comb=f_comb, offs=offs, rot=rot, n=n, cuts=cuts,
                start=start, data=data, rs=rs)


@pytest.mark.parametrize("seed", range(int(os.environ.get("PCAL_RANDOM_CASES", "28"))))     # (more seeds: a longer search)
def test_random_configuration(oracle, seed):
    from paper_2501_05993_b200 import binding
    d = draw(seed)
    C, n, bits = d["C"], d["n"], d["bits"]
    dev = torch.from_numpy(d["data"]).to(DEV)
    flat = dev.view(-1).view(torch.uint8)
    what = f"seed {seed}: {d['kind']} C={C} enc={d['enc']} N_bins={d['n_bins']} offs={d['offs'][:2]} rot={d['rot']} n={n} cuts={d['cuts']} start={d['start']}"

    def run(rot):
        p = binding.Pcal(d["f_s"], d["f_comb"], d["offs"][0], bits, d["enc"], C)
        if C > 1 or any(f != d["offs"][0] for f in d["offs"]):
            p.set_channel_offsets(d["offs"])
        p.set_rotator({"auto": binding.ROT_AUTO, "generator": binding.ROT_GENERATOR}[rot])
        if d["start"]:
            p.set_start_index(d["start"])
        edges = [0] + d["cuts"] + [n]
        for a, b in zip(edges[:-1], edges[1:]):
            lo, hi = a * bits * C // 8, b * bits * C // 8
            p.extract(flat[lo:hi], b - a)
        T, P = p.finalize(), p.get_folded()
        in_effect = p.info().rotator_in_effect
        # the same data as ONE integration period through pcal_integrate, twice back to back (launches overlap; where the
        # geometry allows, reduction and DFT run inside the hot kernel): tones delivered to pinned host memory
        Ti = None
        if not d["start"]:
            outs = [torch.empty((C, d["n_bins"]), dtype=torch.complex128).pin_memory() for _ in range(2)]
            for o in outs:
                p.integrate(flat, n, o)
            torch.cuda.synchronize()
            assert torch.equal(outs[0].view(torch.float64), outs[1].view(torch.float64)), what
            Ti = outs[1].numpy()
        p.destroy()
        return T, P, in_effect, Ti

    try:
        T, P, in_effect, Ti = run(d["rot"])
    except binding.PcalError as e:             # a generator request the kernels' geometry cannot serve: documented, then AUTO must work
        assert e.code == -4 and d["rot"] == "generator", what
        T, P, in_effect, Ti = run("auto")
    fmt = {"f32": oracle.F32, "i8": oracle.I8}.get(d["kind"], oracle.TWO_BIT_SIGN_MAG if d["enc"] else oracle.TWO_BIT_OFFSET_BINARY)
    chans = list(range(C)) if C <= 4 else sorted(set(int(x) for x in d["rs"].randint(0, C, size=4)))
    # reading R28: a few outputs of a noise-only integration may cancel below 1e-3 of the median (1e-2 where float32
    # samples went through the FFMA2 generator, whose products are fp32): absolute bound there
    f32_gen = d["kind"] == "f32" and in_effect == binding.ROT_GENERATOR
    small = dict(max_small=max(1, d["n_bins"] // 32), small_bin=1e-2 if f32_gen else 1e-3)
    for c in chans:
        pr, pi = oracle.fold_ld(d["data"], fmt, C, c, 0, 1, n, d["start"], d["f_s"], d["f_comb"], d["offs"][c], tabulated=True, threads=8)
        want = pr.astype(np.float64) + 1j * pi.astype(np.float64)
        empty = want == 0
        assert not P[c][empty].any(), what
        if (~empty).any():
            assert_close(P[c][~empty], want[~empty], what + f" ch{c} folded", **small)
        wt = oracle.dft(pr, pi)
        assert_close(T[c], wt, what + f" ch{c} tones", **small)
        if Ti is not None:
            assert_close(Ti[c], wt, what + f" ch{c} tones (pcal_integrate)", **small)
        if d["offs"][c] == 0.0 and d["kind"] != "f32" and in_effect == binding.ROT_LUT:      # (unrotated integer sums: bit-exact)
            wi = oracle.fold_i64(d["data"], fmt, C, c, 0, 1, n, d["start"], d["n_bins"])
            assert np.array_equal(P[c].real, wi.astype(np.float64)) and not P[c].imag.any(), what + f" ch{c} exact integers"
