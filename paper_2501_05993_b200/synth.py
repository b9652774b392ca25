"""Seeded synthetic baseband generator -- the one module both the CUDA path's tests/bench and the
oracle's tests consume.  It holds NONE of the extraction method's arithmetic (no rotation, no
fold, no DFT, no decode): it only *encodes* a signal model into packed sample bytes.

Signal model: eq. 2.1 of the paper
    x[n] = sigma * g[n] + A * sum_{i=0}^{K-1} sin((i w_comb + w_offset) n + phi_i),
    phi_i = (i w_comb + w_offset) t_d f_s,  K = N_bins / 2 in-band tones (R4, R19),
g ~ N(0,1) from ``torch.Generator(device).manual_seed(seed + channel)`` drawn in fixed chunks of
2**22 samples (so the byte stream depends only on (seed, device type)).  The consumer on the GPU
and the oracle on the CPU read the *same bytes*; nothing needs to be reproducible across devices.

Encodings produced (R15, R21; BASELINE.json configs):
  float32            cast once from the fp64 sum
  int8               round-half-even, clip to [-127, 127]
  2-bit              thresholds -0.98, 0, +0.98 (in units of the noise sigma = 1) -> level index
                     0..3 for levels {-3,-1,+1,+3};  OFFSET_BINARY code = level index,
                     SIGN_MAG code: +1->0, +3->1, -1->2, -3->3
  1 channel 2-bit    4 samples per byte, sample m in bits 2(m&3)..2(m&3)+1 (LSB first)
  C channel 2-bit    one little-endian uint32 per time sample, channel c in bits 2c..2c+1

These inputs stand in for the paper's recorded VLBI data, which is not available.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace
from typing import List

import numpy as np
import torch

CHUNK = 1 << 22

# encoding names shared with the C-ABI's PCAL_ENC_* (values restated in include/pcal.h)
ENC_OFFSET_BINARY, ENC_SIGN_MAG, ENC_TWOS_COMPLEMENT, ENC_IEEE_FLOAT = 0, 1, 2, 3


@dataclass
class Workload:
    name: str
    n_channels: int
    f_s_hz: float
    f_comb_hz: float
    f_offset_hz: List[float]          # per channel
    bits: int                          # 2, 8, 32
    encoding: int
    n_samples: int                     # per channel
    amp: float
    sigma: float
    t_d_s: List[float]                 # per channel cable delay
    seed: int
    rotator: str = "auto"              # "auto" | "lut" | "generator"
    tones: int = -1                    # K; -1 -> N_bins/2

    @property
    def n_bins(self) -> int:
        return int(round(self.f_s_hz / self.f_comb_hz))

    @property
    def n_bytes(self) -> int:
        return self.n_samples * self.n_channels * self.bits // 8

    def scaled(self, n_samples: int) -> "Workload":
        return replace(self, n_samples=int(n_samples))


def _cfg4_draws(seed: int):
    rs = np.random.RandomState(seed)
    k = rs.randint(0, 100, size=16)
    td = rs.uniform(0.0, 20e-9, size=16)
    return [float(10e3 * kk) for kk in k], [float(t) for t in td]


def config(idx: int) -> Workload:
    """The five BASELINE.json configs (1-based) plus the parity-only / smoke shapes.

    6 = cfg 2' (cfg 2 with f_offset 0, bit-exact clause, R20); 7 = cfg 5' (int8,
    f_offset 0, 2**28 samples); 8 = the paper's own benchmark shape."""
    if idx == 1:
        return Workload("cfg1_f32_32MHz_off0", 1, 32e6, 1e6, [0.0], 32, ENC_IEEE_FLOAT, 1 << 22, 0.05, 1.0, [5e-9], 1001)
    if idx == 2:
        return Workload("cfg2_2bit_32MHz_10kHz", 1, 32e6, 1e6, [10e3], 2, ENC_OFFSET_BINARY, 1 << 28, 0.05, 1.0, [5e-9], 1002)
    if idx == 3:
        return Workload("cfg3_2bit_512MHz_10kHz", 1, 512e6, 1e6, [10e3], 2, ENC_OFFSET_BINARY, 512_000_000, 0.03, 1.0, [12.5e-9], 1003)
    if idx == 4:
        offs, tds = _cfg4_draws(1004)
        return Workload("cfg4_16ch_2bit_64MHz", 16, 64e6, 1e6, offs, 2, ENC_SIGN_MAG, 64_000_000, 0.05, 1.0, tds, 1004)
    if idx == 5:
        return Workload("cfg5_int8_1024MHz_1234.567Hz", 1, 1024e6, 1e6, [1234.567], 8, ENC_TWOS_COMPLEMENT, 4_000_000_000, 1.0, 20.0, [5e-9], 1005, rotator="generator")
    if idx == 6:
        return replace(config(2), name="cfg2p_2bit_32MHz_off0", f_offset_hz=[0.0], seed=1006)
    if idx == 7:
        return replace(config(5), name="cfg5p_int8_1024MHz_off0", f_offset_hz=[0.0], n_samples=1 << 28, seed=1007, rotator="auto")
    if idx == 8:
        return Workload("paper_bench_f32_16MHz_10kHz", 1, 16e6, 1e6, [10e3], 32, ENC_IEEE_FLOAT, 16_000_000, 0.05, 1.0, [5e-9], 1008)
    raise ValueError(f"no config {idx}")


def tone_phases(w: Workload, c: int = 0) -> np.ndarray:
    """phi_i of eq. 2.1 for channel c (radians, not wrapped), i = 0..K-1."""
    K = w.tones if w.tones >= 0 else w.n_bins // 2
    i = np.arange(K, dtype=np.float64)
    return 2.0 * math.pi * (i * w.f_comb_hz + w.f_offset_hz[c]) * w.t_d_s[c]


def _comb_chunk(w: Workload, c: int, n0: int, length: int, device) -> torch.Tensor:
    """A * sum_i sin((i w_comb + w_off)(n + tau)), fp64, for n = n0 .. n0+length-1.

    Uses sum_i e^{j i w_comb (n+tau)} = B[n mod N_bins] (w_comb N_bins = 2 pi), so the cost is
    O(1) per sample instead of K sines."""
    nb = w.n_bins
    K = w.tones if w.tones >= 0 else nb // 2
    tau = w.t_d_s[c] * w.f_s_hz
    b = torch.arange(nb, dtype=torch.float64, device=device) + tau
    i = torch.arange(K, dtype=torch.float64, device=device)
    ang = (2.0 * math.pi / nb) * torch.outer(b, i)
    B_re = torch.cos(ang).sum(1)
    B_im = torch.sin(ang).sum(1)
    n = torch.arange(n0, n0 + length, dtype=torch.int64, device=device)
    idx = n % nb
    cyc = torch.remainder((n.to(torch.float64) + tau) * (w.f_offset_hz[c] / w.f_s_hz), 1.0)
    ph = 2.0 * math.pi * cyc
    # Im(e^{j ph} * B) = sin(ph) Re B + cos(ph) Im B
    return w.amp * (torch.sin(ph) * B_re[idx] + torch.cos(ph) * B_im[idx])


def _codes_2bit(x: torch.Tensor, encoding: int) -> torch.Tensor:
    lvl = (x >= -0.98).to(torch.uint8) + (x >= 0.0).to(torch.uint8) + (x >= 0.98).to(torch.uint8)
    if encoding == ENC_OFFSET_BINARY:
        return lvl
    # SIGN_MAG: level index 0..3 (-3,-1,+1,+3) -> code 3,2,0,1
    lut = torch.tensor([3, 2, 0, 1], dtype=torch.uint8, device=x.device)
    return lut[lvl.long()]


def generate(w: Workload, device="cpu", noise: bool = True) -> torch.Tensor:
    """Packed sample buffer for workload ``w`` on ``device``.

    Returns float32[n], int8[n], uint8[n/4] (1-channel 2-bit) or int32[n] (multi-channel 2-bit
    words; the bit pattern is the little-endian uint32 described above)."""
    device = torch.device(device)
    n = w.n_samples
    if w.bits == 2 and w.n_channels == 1 and n % 4:
        raise ValueError("2-bit single channel needs n_samples % 4 == 0")
    gens = [torch.Generator(device=device).manual_seed(w.seed + c) for c in range(w.n_channels)]
    if w.bits == 32:
        out = torch.empty(n, dtype=torch.float32, device=device)
    elif w.bits == 8:
        out = torch.empty(n, dtype=torch.int8, device=device)
    elif w.n_channels == 1:
        out = torch.empty(n // 4, dtype=torch.uint8, device=device)
    else:
        out = torch.empty(n, dtype=torch.int32, device=device)
    for n0 in range(0, n, CHUNK):
        ln = min(CHUNK, n - n0)
        word = None
        for c in range(w.n_channels):
            x = _comb_chunk(w, c, n0, ln, device)
            if noise:
                g = torch.randn(ln, generator=gens[c], device=device, dtype=torch.float32)
                x = x + w.sigma * g.to(torch.float64)
            if w.bits == 32:
                out[n0:n0 + ln] = x.to(torch.float32)
            elif w.bits == 8:
                out[n0:n0 + ln] = torch.clamp(torch.round(x), -127, 127).to(torch.int8)
            else:
                code = _codes_2bit(x, w.encoding)
                if w.n_channels == 1:
                    q = code.view(-1, 4)
                    out[n0 // 4:(n0 + ln) // 4] = q[:, 0] | (q[:, 1] << 2) | (q[:, 2] << 4) | (q[:, 3] << 6)
                else:
                    t = code.to(torch.int64) << (2 * c)
                    word = t if word is None else (word | t)
        if word is not None:
            word = torch.where(word >= (1 << 31), word - (1 << 32), word)
            out[n0:n0 + ln] = word.to(torch.int32)
    return out
