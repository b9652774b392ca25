"""Reproduce the generator accuracy comparison the paper cites as "Figure 7" (figure not in
the text): max |generated phasor - exact phasor| of the direct method and of the eq. 2.6 / 2.7 recursions,
fp32 and fp64, with and without the k-shift of PAPER.md:97, over six equal intervals of n.

    python -m paper_2501_05993_b200.generator_study [--f-s HZ] [--f-offset HZ] [--f-comb HZ] [--k K] [--steps N]

Everything is computed by pcal_generator_study (CUDA); this module only formats the table.
"""
import argparse

from . import binding as b


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--f-s", type=float, default=1024e6)
    ap.add_argument("--f-offset", type=float, default=1234.567)
    ap.add_argument("--f-comb", type=float, default=1e6)
    ap.add_argument("--k", type=int, default=256, help="k-shift: rotate at f_offset + k f_comb")
    ap.add_argument("--steps", type=int, default=1 << 24)
    a = ap.parse_args()
    fs, fo, fk = a.f_s, a.f_offset, a.f_offset + a.k * a.f_comb
    rows = [("direct fp32", b.GEN_DIRECT, 32, fo), ("CFO fp32", b.GEN_CFO, 32, fo), ("MCO fp32", b.GEN_MCO, 32, fo),
            ("DFR fp32", b.GEN_DFR, 32, fo), ("DFR-FMA fp32", b.GEN_DFR_FMA, 32, fo),
            (f"CFO fp32 k={a.k}", b.GEN_CFO, 32, fk), (f"MCO fp32 k={a.k}", b.GEN_MCO, 32, fk),
            (f"DFR fp32 k={a.k}", b.GEN_DFR, 32, fk), (f"DFR-FMA fp32 k={a.k}", b.GEN_DFR_FMA, 32, fk),
            ("CFO fp64", b.GEN_CFO, 64, fo), ("MCO fp64", b.GEN_MCO, 64, fo), ("DFR fp64", b.GEN_DFR, 64, fo),
            ("DFR-FMA fp64", b.GEN_DFR_FMA, 64, fo)]
    err = b.generator_study([(f, p, fs, fr) for _, f, p, fr in rows], a.steps, 6)
    print(f"f_s = {fs:g} Hz, f_offset = {fo:g} Hz, n = 1..{a.steps} in 6 intervals; max |error| per interval")
    for (name, *_), e in zip(rows, err):
        print(f"{name:22s}" + " ".join(f"{x:9.2e}" for x in e))


if __name__ == "__main__":
    main()
