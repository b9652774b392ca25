#!/usr/bin/env python
"""bench.py -- PCal extraction throughput on B200 (contract: see the task statement / DESIGN.md section 9).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config IDX] [--rotator lut|generator] [--impl reference]
                    [--no-all] [--quick] [--parity-report]

A *step* is one pass of the whole hot path over one batch: pcal_reset -> pcal_extract (load/demux, decode, rotate,
fold, reduce) -> pcal_finalize (DFT + result to the host), issued as ONE library call (pcal_integrate).  Headline
workload: BASELINE.json configs[4] (config 5: 1024 MHz, int8, 4e9 samples = 4 GB, generator rotation), the largest
configuration that fits one GPU; every other configuration has its own row, with its own roofline object, under
`all_configs`.

One JSON line on stdout (rank 0):
  value        whole-job samples/s, inputs resident in HBM, device-timed over exactly K steps (max over ranks)
  stats        median / best / worst ms per step over further timed regions of the same steps
  e2e          same metric through pcal_extract_host: pinned HOST buffer -> device inside the timed region, result
               read back to the host every step
  roofline     the hot kernel against the slower of its two bounds: algorithmic bytes at the measured HBM peak, and
               thread-instructions per sample (ncu, profiles/r2_kernels.csv) at the measured issue rate of its pipe
  parity       achieved error against the oracle on a bounded sample of the same workload
  cpu_baseline the CPU oracle timed on this box's host cores on a bounded sample of the workload
`--impl reference` times the oracle (the only "reference implementation" this paper-only task has) on the same
configuration, a bounded sample per step.  With N > 1 (torchrun) the stream is time-sharded through
paper_2501_05993_b200.sharding.ShardedIntegrator (weak scaling: per-GPU work fixed).
"""
from __future__ import annotations

import argparse
import csv
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "pcal_extraction_samples_per_s"
UNIT = "samples/s"
L2_BYTES = 126 << 20
KERNEL_TABLE = os.path.join("profiles", "r2_kernels.csv")


def row_key(idx: int, rotator: str) -> str:
    name = {8: "paper_shape"}.get(idx, f"cfg{idx}")
    return f"{name}_{rotator}"


def load_kernel_table():
    """Per workload row: hot kernel, dram bytes per launch and thread-instructions per sample from the committed ncu
    captures (profiles/r2_kernels.csv; profiles/r2_kernels.md names the commands).  {} if the file is missing."""
    out = {}
    try:
        with open(os.path.join(ROOT, KERNEL_TABLE)) as f:
            for r in csv.DictReader(f):
                out[r["row"]] = r
    except Exception:
        pass
    return out


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            d = json.load(open(path))
            return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-i", str(self.index), "-lms", "100"], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=self._pump, daemon=True).start()
        except Exception:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.rows.append([t.strip() for t in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, smax, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); smax = float(r[1])
                for name, v in zip(names, r[4:8]):
                    if v.lower().startswith("active"):
                        reasons.add(name)
            except Exception:
                continue
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": smax, "reasons": sorted(reasons),
                "samples": len(sm)}


def oracle_fmt(orc, w):
    from paper_2501_05993_b200 import synth
    if w.bits == 32:
        return orc.F32
    if w.bits == 8:
        return orc.I8
    return orc.TWO_BIT_OFFSET_BINARY if w.encoding == synth.ENC_OFFSET_BINARY else orc.TWO_BIT_SIGN_MAG


def time_oracle(w, n_sample: int, steps: int = 1, threads: int = 0):
    """The oracle as it stands (O-fold + DFT) on the first n_sample samples of workload w; threads = 0: all host cores."""
    import oracle as orc
    from paper_2501_05993_b200 import synth
    orc.build()
    ws = w.scaled(n_sample)
    buf = synth.generate(ws, "cpu").numpy()
    cores = threads or os.cpu_count() or 1
    fmt = oracle_fmt(orc, ws)
    t0 = time.perf_counter()
    for _ in range(steps):
        for c in range(ws.n_channels):
            orc.extract(buf, fmt, ws.n_channels, c, n_sample, 0, ws.f_s_hz, ws.f_comb_hz, ws.f_offset_hz[c],
                        tabulated=True, threads=cores)
    dt = (time.perf_counter() - t0) / steps
    return n_sample * ws.n_channels / dt, cores, dt


def parity_sample(w, device, n_sample: int):
    """Achieved error of the CUDA path against the oracle on the first n_sample samples of w: every tone of (up to four)
    channels.  north_star's bar is 1e-5 relative and 1e-5 rad per tone; this records the margin."""
    import numpy as np
    import oracle as orc
    from paper_2501_05993_b200 import binding, synth
    orc.build()
    ws = w.scaled(n_sample)
    dev = synth.generate(ws, device)
    p = binding.from_workload(ws)
    p.extract(dev, n_sample)
    T = p.finalize()
    rot = {1: "lut", 2: "generator"}[p.info().rotator_in_effect]
    p.destroy()
    host = dev.cpu().numpy()
    del dev
    chans = sorted(set(range(0, ws.n_channels, max(1, ws.n_channels // 4))))
    worst_rel, worst_ph, worst_scaled, bins = 0.0, 0.0, 0.0, 0
    for c in chans:
        want = orc.extract(host, oracle_fmt(orc, ws), ws.n_channels, c, n_sample, 0, ws.f_s_hz, ws.f_comb_hz, ws.f_offset_hz[c],
                           tabulated=True, threads=os.cpu_count() or 1)
        err = np.abs(T[c] - want)
        worst_rel = max(worst_rel, float((err / np.abs(want)).max()))
        worst_ph = max(worst_ph, float(np.abs(np.angle(T[c] * np.conj(want))).max()))
        worst_scaled = max(worst_scaled, float(err.max() / np.abs(want).max()))
        bins += want.size
    return {"max_rel_err": worst_rel, "max_phase_err_rad": worst_ph, "max_err_over_largest_tone": worst_scaled,
            "tones_compared": bins, "channels": chans, "samples_per_channel": n_sample, "rotator": rot,
            "bar": "1e-5 relative and 1e-5 rad per tone (north_star); oracle: oracle/pcal_oracle.c, O-fold + DFT"}


def roofline_of(key, w, step_s, isolated_us, floor_us, launches_per_step, pipe_peaks, ktab, rotator):
    """The hot kernel of one row against the slower of its two bounds (north_star): input bytes at the measured HBM
    peak, and thread-instructions per sample (ncu) at the measured issue rate of the pipe that executes most of them."""
    peak, peak_src = load_peaks()
    row = ktab.get(key, {})
    samples = w.n_samples * w.n_channels
    hbm_s = w.n_bytes / (peak * 1e9)
    ips = float(row["thread_instr_per_sample"]) if row.get("thread_instr_per_sample") else None
    pipe = row.get("pipe") or "lop3"
    pipe_peak = (pipe_peaks or {}).get(pipe)
    alu_s = samples * ips / pipe_peak if (ips and pipe_peak) else None
    # legacy tensor path of the generator kernels: warp-level IMMA per sample (from the kernels' tiling: gen2_kernel 4 x m16n8k32
    # per 16 bytes x 32 rows = 2048 samples, times the passes over 8 / 16-channel words; gen_mma_kernel one m16n8k16 per 256)
    kname = row.get("kernel") or ""
    mma = None
    if kname.startswith("gen2_kernel"):
        mma = ("imma_k32", (1.0 / 512.0) * max(1, w.n_channels // 4))
    elif kname.startswith("gen_mma_kernel"):
        mma = ("imma_k16", 1.0 / 256.0)
    mma_peak = (pipe_peaks or {}).get(mma[0]) if mma else None
    mma_s = samples * mma[1] / mma_peak if mma_peak else None
    bound = "alu" if (alu_s is not None and alu_s > hbm_s) else "hbm"
    if mma_s is not None and mma_s > max(hbm_s, alu_s or 0.0):
        bound = "tensor"
    achieved_gbs = w.n_bytes / step_s / 1e9
    r = {"bound": bound, "kernel": row.get("kernel") or ("generator kernel" if rotator == "generator" else "fold kernel incl. fused tail"),
         "algorithmic_bytes_per_launch": w.n_bytes, "avg_launch_us": step_s * 1e6, "launches_per_step": launches_per_step,
         "hbm": {"bound_us": hbm_s * 1e6, "achieved_gbs": achieved_gbs, "peak_gbs": peak, "frac": achieved_gbs / peak, "peak_source": peak_src},
         "alu": None if alu_s is None else {
             "thread_instr_per_sample": ips, "pipe": pipe, "pipe_peak_thread_instr_per_s": pipe_peak, "bound_us": alu_s * 1e6,
             "frac": alu_s / step_s, "source": f"{KERNEL_TABLE} (ncu smsp__inst_executed.sum x 32 / samples) and pcal_pipe_probe"},
         "tensor": None if mma_s is None else {
             "warp_mma_per_sample": mma[1], "pipe": mma[0], "pipe_peak_warp_mma_per_s": mma_peak, "bound_us": mma_s * 1e6,
             "frac": mma_s / step_s, "source": "MMA count from the kernel's tiling (DESIGN.md 5.2) and pcal_pipe_probe"},
         "traffic": int(row["dram_bytes_per_launch"]) if row.get("dram_bytes_per_launch") else None,
         "traffic_source": f"{KERNEL_TABLE}: dram__bytes_read.sum + dram__bytes_write.sum of one launch, committed ncu --set full capture "
                           "(profiles/r2_kernels.md), not measured in this run" if row.get("dram_bytes_per_launch") else None,
         "isolated_launch_us": isolated_us,
         "single_integration_frac": (w.n_bytes / (isolated_us * 1e-6) / 1e9 / peak) if isolated_us else None,
         "how": "avg_launch_us = device time of the timed region (CUDA events on the launching stream) / launches of the kernel in it: "
                "consecutive launches overlap (programmatic dependent launch), the step's small kernels are inside.  isolated_launch_us = "
                "the same kernel bracketed by events launch by launch (serialised: the latency of one integration on its own)"}
    if bound == "hbm":
        r.update({"achieved": achieved_gbs, "peak": peak, "unit": "GB/s", "frac": achieved_gbs / peak})
    elif bound == "tensor":
        r.update({"achieved": samples * mma[1] / step_s, "peak": mma_peak, "unit": "warp-MMA/s", "frac": mma_s / step_s})
    else:
        r.update({"achieved": samples * ips / step_s, "peak": pipe_peak, "unit": "thread-instr/s", "frac": alu_s / step_s})
    if floor_us:
        r["read_floor"] = {"us": floor_us, "gbs": w.n_bytes / floor_us / 1e3, "frac_of_floor": floor_us / (step_s * 1e6),
                           "what": "pcal_read_probe: pure streaming read of the same buffers (no decode/fold), back-to-back launches timed like the steps"}
    return r


def measure(idx: int, steps: int, warmup: int, rank: int, world: int, device, do_e2e: bool = True,
            rotator: str | None = None, n_override: int | None = None, min_warm_s: float = 0.5,
            no_graph: bool = False, exchange: bool = False, pipe_peaks=None, ktab=None, regions: int = 5,
            min_region_steps: int = 0):
    """Run config idx on this rank's GPU; returns the measurement dict (device timing is per rank)."""
    import torch
    import torch.distributed as dist
    from dataclasses import replace
    from paper_2501_05993_b200 import binding, sharding, synth

    w = synth.config(idx)
    if n_override:
        w = w.scaled(n_override)
    if rotator:
        w = replace(w, rotator=rotator)
    n, C, nb = w.n_samples, w.n_channels, w.n_bins
    # distinct input copies, at least 2 x L2 in total, so that every step reads from DRAM and not from the 126 MB L2
    ncopies = 1 if w.n_bytes >= 2 * L2_BYTES else min(24, -(-(2 * L2_BYTES + (32 << 20)) // w.n_bytes))
    bufs = [synth.generate(replace(w, seed=w.seed + 100 * i + 7 * rank), device) for i in range(ncopies)]
    exchange = exchange or world > 1
    ctxs = [binding.from_workload(w) for _ in range(2 if exchange else 1)]
    for q_ in ctxs:
        q_.set_input_ready(True)  # inputs are resident in HBM and complete before the timed region starts
    p = ctxs[0]
    out_pinned = torch.empty((C, nb), dtype=torch.complex128).pin_memory()
    # Multi-GPU: the package's time-sharded integrator, two lanes (the all-gather of integration k is in flight on
    # NCCL's stream while integration k+1 is being folded and integration k-1 is being finished)
    shard = sharding.ShardedIntegrator(ctxs, C, nb, world, device) if exchange else None
    shard_outs = [torch.empty((C, nb), dtype=torch.complex128).pin_memory() for _ in range(2)]
    buf_ptrs, out_ptr = [b_.data_ptr() for b_ in bufs], out_pinned.data_ptr()
    cur_stream = int(torch.cuda.current_stream().cuda_stream)

    def step(i, stream=None):
        if shard is None:
            # pcal_reset + pcal_extract + pcal_finalize_async in one call; raw addresses, stream handle hoisted
            p.integrate(buf_ptrs[i % ncopies], n, out_ptr, stream=stream)
        else:
            shard.submit(bufs[i % ncopies], n, rank * n, shard_outs[i % 2])     # time shard of rank r starts at r*n

    def drain():
        if shard is not None:
            shard.drain()

    # clocks are sampled from the start of the warm-up to the end of the timed regions; the warm-up runs >= W steps and
    # >= 0.5 s of the same steps, so the samples are taken under the same load
    sampler = ClockSampler(torch.cuda.current_device())
    if rank == 0:
        sampler.start()
    t_w = time.perf_counter()
    i = 0
    while i < max(warmup, 3) or (rank == 0 and world == 1 and time.perf_counter() - t_w < min_warm_s):
        step(i)
        i += 1
        if i % 16 == 0:
            torch.cuda.synchronize()
    drain()
    torch.cuda.synchronize()
    # Single GPU: two ways to issue the steps are calibrated after the warm-up and the faster one is used: (a) direct
    # launches (the library chains its kernels with programmatic dependent launch); (b) CUDA-graph replays of n_big
    # consecutive steps.  Multi-GPU steps (NCCL exchange) launch directly.
    use_graph = (world == 1) and not no_graph and not exchange and w.n_bytes < (1 << 30)
    big, per_step_launches = None, None
    n_big = ncopies * max(1, min(steps, 40) // ncopies)      # steps in the graph (whole rounds over the copies)
    l0 = p.info().kernel_launches
    step(0)
    drain()
    per_step_launches = sum(q_.info().kernel_launches for q_ in ctxs) - l0 if not exchange else None
    torch.cuda.synchronize()
    if use_graph:
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):
            big = torch.cuda.CUDAGraph()
            with torch.cuda.graph(big, stream=side):
                for k in range(n_big):
                    step(k)
        torch.cuda.current_stream().wait_stream(side)

    def run_steps(mode, count):
        if mode == "graph_of_steps":
            for _ in range(count // n_big):
                big.replay()
            for k in range(count % n_big):
                step(k, cur_stream)
        else:
            for k in range(count):
                step(k, cur_stream)
        drain()

    def timed(m, count):
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        run_steps(m, count)
        b.record()
        torch.cuda.synchronize()
        return a.elapsed_time(b)

    mode, cal = "direct", None
    if use_graph:
        reps = max(2 * n_big, steps)
        cal = {m: min(timed(m, reps) / reps for _ in range(2)) for m in ("direct", "graph_of_steps")}
        mode = min(cal, key=cal.get)
    launches0 = sum(q_.info().kernel_launches for q_ in ctxs)
    if world > 1:
        dist.barrier()
    ms = timed(mode, steps)                                   # THE timed region: exactly K steps
    if world > 1:
        dist.barrier()
    launches = per_step_launches * steps if mode != "direct" else sum(q_.info().kernel_launches for q_ in ctxs) - launches0
    # further regions of the same steps (not edge-dominated: at least min_region_steps each): median / best / worst
    r_steps = max(steps, min_region_steps)
    per = sorted(timed(mode, r_steps) / r_steps for _ in range(regions)) if (regions and world == 1) else []
    # the hot kernel bracketed by events launch by launch (serialises the launches: latency of an isolated integration)
    for q_ in ctxs:
        q_.set_profiling(True)
    for i in range(min(steps, 50)):
        step(i)
    drain()
    torch.cuda.synchronize()
    hot_ms, hot_launches = 0.0, 0
    for q_ in ctxs:
        ms_q, n_q = q_.get_profile()
        hot_ms, hot_launches = hot_ms + ms_q, hot_launches + n_q
        q_.set_profiling(False)
    hot_per_step = max(1, round(hot_launches / min(steps, 50))) if hot_launches else 1
    # finalize alone (reduce is inside the extract kernels; this is the DFT kernel + the result to the pinned host buffer)
    fin_us = None
    if world == 1 and not exchange:
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(50):
            p.finalize_async(out_pinned)
        b.record()
        torch.cuda.synchronize()
        fin_us = 1e3 * a.elapsed_time(b) / 50
    clocks = sampler.stop() if rank == 0 else None
    big = None
    if world > 1:
        t = torch.tensor([ms], dtype=torch.float64, device=device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    inf = p.info()
    rot = {1: "lut", 2: "generator"}[inf.rotator_in_effect]
    res = {
        "workload": w.name, "n_samples_per_channel": n, "n_channels": C, "n_bins": nb, "bits": w.bits,
        "input_bytes": w.n_bytes, "rotator": rot, "fold_period": int(inf.fold_period), "ms_per_step": ms / steps,
        "value": world * n * C * steps / (ms * 1e-3), "input_gbs": world * w.n_bytes * steps / (ms * 1e-3) / 1e9,
        "stats": {"regions": len(per), "steps_per_region": r_steps, "ms_per_step_median": per[len(per) // 2], "ms_per_step_best": per[0],
                  "ms_per_step_worst": per[-1]} if per else None,
        "gpu_launches": int(launches), "launches_per_step": per_step_launches, "finalize_alone_us": fin_us,
        "launch_mode": {"direct": "direct launches (kernels chained by programmatic dependent launch)",
                        "graph_of_steps": f"cuda_graph: one replay per {n_big} consecutive steps (cycling over the input copies), kernels chained "
                                          "by programmatic dependent launch inside the graph; remainder steps launched directly"}[mode],
        "launch_mode_calibration_us": {k_: 1e3 * v_ for k_, v_ in cal.items()} if cal else None,
        "l2_policy": f"rotating {ncopies} distinct input copies ({ncopies * w.n_bytes / 2**20:.0f} MiB total, >= 2 x the 126 MB L2)"
        if ncopies > 1 else "input larger than 2 x L2",
        "clocks": clocks,
    }
    # calibration: a pure streaming read of the same buffers (no decode, no fold), launched back to back like the steps
    floor_us = None
    if rank == 0:
        for i in range(ncopies):
            p.read_probe(bufs[i % ncopies])
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        cnt = max(min(steps, 50), 2 * ncopies)
        a.record()
        for i in range(cnt):
            p.read_probe(bufs[i % ncopies])
        b.record()
        torch.cuda.synchronize()
        floor_us = 1e3 * a.elapsed_time(b) / cnt
    step_s = 1e-3 * ms / steps / hot_per_step           # per launch of the hot kernel (one per step, unless the segment is cut in pieces)
    wl = w if hot_per_step == 1 else w.scaled(n // hot_per_step)
    res["roofline"] = roofline_of(row_key(idx, rot), wl, step_s, 1e3 * hot_ms / max(hot_launches, 1), floor_us / hot_per_step if floor_us else None,
                                  per_step_launches, pipe_peaks, ktab or {}, rot)
    res["hot_kernel_us"] = step_s * 1e6
    if do_e2e:
        host = bufs[0].cpu().pin_memory()
        e2e_steps = max(1, min(steps, 5 if w.n_bytes > (1 << 30) else steps))
        p.reset(); p.extract_host(host, n); p.finalize()      # warm-up (allocates the staging buffer)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            p.reset()
            p.extract_host(host, n)
            T = p.finalize()
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        if world > 1:
            t = torch.tensor([dt], dtype=torch.float64, device=device)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            dt = float(t.item())
        res["e2e"] = {"value": world * n * C * e2e_steps / dt, "unit": UNIT, "h2d_bytes_per_step": w.n_bytes,
                      "d2h_bytes_per_step": C * nb * 16, "steps": e2e_steps,
                      "api": "pcal_reset + pcal_extract_host (pinned host buffer) + pcal_finalize"}
        del host
    for q_ in ctxs:
        q_.destroy()
    del bufs
    torch.cuda.empty_cache()
    return res, w


ROWS = [(1, None), (2, None), (3, "lut"), (3, "generator"), (4, None), (4, "generator"), (5, None), (8, "lut"), (8, "generator")]   # 8 = the paper's own benchmark shape


def reference_line(args):
    """`--impl reference`: the oracle on the same configuration, a bounded sample of it per step."""
    from paper_2501_05993_b200 import synth
    w = synth.config(args.config)
    probe, cores, _ = time_oracle(w, 1 << 20)
    # a step of about 2 s on every host core, so that K steps + W warm-ups end within a few minutes
    n_sample = int(min(w.n_samples, max(1 << 22, probe * 2.0)))
    n_sample -= n_sample % 128
    for _ in range(max(args.warmup, 1)):
        time_oracle(w, min(n_sample, 1 << 22))
    rate, cores, dt = time_oracle(w, n_sample, steps=args.steps)
    sample = f"first {n_sample} of {w.n_samples} samples per channel of {w.name} per step, O-fold + DFT, {cores} threads"
    return {"metric": METRIC, "value": rate, "unit": UNIT, "impl": "reference", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "n_samples_per_channel": w.n_samples, "sample": sample},
            "cpu_baseline": {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": rate, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}


def parity_report(device):
    """`--parity-report`: achieved error per configuration at FULL size (the table of profiles/r2_parity.md)."""
    from dataclasses import replace
    from paper_2501_05993_b200 import synth
    print("| row | rotator | samples per channel | channels checked | tones compared | max relative error | max phase error (rad) | max error / largest tone |")
    print("|---|---|---|---|---|---|---|---|")
    for idx, rot in ROWS:
        w = synth.config(idx)
        if rot:
            w = replace(w, rotator=rot)
        r = parity_sample(w, device, w.n_samples)
        print(f"| {row_key(idx, r['rotator'])} | {r['rotator']} | {r['samples_per_channel']} | {r['channels']} | {r['tones_compared']} | "
              f"{r['max_rel_err']:.2e} | {r['max_phase_err_rad']:.2e} | {r['max_err_over_largest_tone']:.2e} |", flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=5, help="BASELINE.json config (1-based); default configs[4], the largest single-GPU one")
    ap.add_argument("--impl", default="own", choices=["own", "reference"])
    ap.add_argument("--no-all", action="store_true", help="skip the per-config table")
    ap.add_argument("--samples", type=int, default=0, help="override samples per channel (debug)")
    ap.add_argument("--rotator", default=None, choices=["lut", "generator"], help="force the rotator variant (config 3 runs both)")
    ap.add_argument("--no-graph", action="store_true", help="launch every step directly instead of replaying a CUDA graph")
    ap.add_argument("--force-exchange", action="store_true",
                    help="testing: run the multi-GPU exchange path (NCCL all-gather + rank-order sum) even with one rank")
    ap.add_argument("--quick", action="store_true",
                    help="profiling mode (ncu): exactly W warm-up steps, one timed region, no e2e / cpu_baseline / parity / table")
    ap.add_argument("--parity-report", action="store_true", help="print the full-size parity table (profiles/r2_parity.md) and exit")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    from paper_2501_05993_b200 import synth

    if args.impl == "reference":
        if rank == 0:
            print(json.dumps(reference_line(args)), flush=True)
        return

    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local_rank)
    device = torch.device("cuda", local_rank)
    if args.parity_report:
        parity_report(device)
        return
    if world > 1 or args.force_exchange:
        if "RANK" not in os.environ:
            os.environ.update({"RANK": "0", "WORLD_SIZE": "1", "MASTER_ADDR": "127.0.0.1", "MASTER_PORT": "29533"})
        dist.init_process_group("nccl", device_id=device)
    from paper_2501_05993_b200 import binding as _b
    ktab = load_kernel_table()
    # measured issue-rate ceilings of this GPU: the ALU side of every roofline object
    pipe_peaks = None
    if not args.quick:
        pipe_peaks = {"ffma": _b.pipe_probe(0), "lop3": _b.pipe_probe(1), "imma_k16": _b.pipe_probe(2), "imma_k32": _b.pipe_probe(3)}
    res, w = measure(args.config, args.steps, args.warmup, rank, world, device, n_override=args.samples or None,
                     rotator=args.rotator, no_graph=args.no_graph, exchange=args.force_exchange, do_e2e=not args.quick,
                     min_warm_s=0.0 if args.quick else 0.5, pipe_peaks=pipe_peaks, ktab=ktab, regions=0 if args.quick else 5)
    dtype = {2: "u8 codes -> int32/int64 sums, fp64 rotate + DFT", 8: "int8 -> int32/int64 sums, fp64 rotate + DFT",
             32: "fp32 runs -> fp64"}[res["bits"]]
    line = {"metric": METRIC, "value": res["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": res["ms_per_step"], "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": dtype, "data": "synthetic", "input_gbs": res["input_gbs"],
            "config": {"workload": res["workload"], "n_samples_per_channel": res["n_samples_per_channel"],
                       "n_channels": res["n_channels"], "bits": res["bits"], "n_bins": res["n_bins"],
                       "rotator": res["rotator"], "input_bytes_per_gpu": res["input_bytes"],
                       "parallelism": f"time-sharded x{world}" if world > 1 else "single GPU",
                       "l2": res["l2_policy"], "launch_mode": res["launch_mode"],
                       "launch_mode_calibration_us": res["launch_mode_calibration_us"]},
            "stats": res["stats"], "clocks": res["clocks"], "e2e": res.get("e2e"), "gpu_launches": res["gpu_launches"],
            "launches_per_step": res["launches_per_step"], "finalize_alone_us": res["finalize_alone_us"],
            "roofline": res["roofline"], "hot_kernel_us": res["hot_kernel_us"]}
    if world == 1 and rank == 0 and not args.quick:
        line["pipe_peaks"] = dict(pipe_peaks, unit="thread-instr/s (ffma, lop3), warp-instr/s (imma_k16: m16n8k16 s8, imma_k32: m16n8k32 u8 x s8)",
                                  how="pcal_pipe_probe: 8 independent chains per thread, 8 CTAs x 256 threads per SM, best of 3")
        line["parity"] = parity_sample(w, device, min(w.n_samples, 1 << 24))
        # the oracle as it stands on this box's host cores: ~20 core-seconds on a bounded sample
        probe, cores, _ = time_oracle(w, 1 << 21)
        n_sample = int(min(w.n_samples, max(1 << 22, probe * 1.0)))
        n_sample -= n_sample % 128
        _, cores, dt1 = time_oracle(w, n_sample, steps=1)          # also warms the threads
        reps = max(1, min(50, int(round(1.2 / dt1))))
        rate, cores, dt = time_oracle(w, n_sample, steps=reps)
        line["cpu_baseline"] = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": f"first {n_sample} samples of {w.name}, O-fold + DFT, {reps} x {dt:.2f} s wall on {cores} threads"}
        one = {}
        for idx1 in (1, 2):                                          # a 1-thread figure on configs 1-2
            w1 = synth.config(idx1)
            r1, _, d1 = time_oracle(w1, 1 << 22, steps=1, threads=1)
            one[f"cfg{idx1}"] = {"value": r1, "unit": UNIT, "cores": 1, "sample": f"first {1 << 22} samples of {w1.name}, {d1:.2f} s"}
        line["cpu_baseline"]["one_thread"] = one
        if not args.no_all:
            table = {}
            for idx, rot in ROWS:
                r, wr = measure(idx, 20 if idx == 5 else 200, 3, 0, 1, device, do_e2e=False, rotator=rot, pipe_peaks=pipe_peaks,
                                ktab=ktab, regions=5, min_region_steps=0)
                key = row_key(idx, r["rotator"])
                table[key] = {k: r[k] for k in ("workload", "rotator", "value", "input_gbs", "ms_per_step", "stats", "launches_per_step",
                                                "finalize_alone_us", "launch_mode", "l2_policy", "clocks", "roofline")}
                table[key]["parity"] = parity_sample(wr, device, min(wr.n_samples, 1 << 22))
            line["all_configs"] = table
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1 or args.force_exchange:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
