#!/usr/bin/env python
"""bench.py -- PCal extraction throughput on B200 (contract: see the task statement / DESIGN.md).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config IDX] [--impl reference] [--all]

A *step* is one pass of the whole hot path over one batch: pcal_reset -> pcal_extract (load/demux,
decode, rotate, fold, reduce) -> pcal_finalize (DFT + result to the host).  Default workload:
BASELINE.json configs[1] (single channel, 32 MHz, 2-bit, f_offset 10 kHz, 2^28 samples = 64 MiB).

One JSON line on stdout (rank 0):
  value      whole-job samples/s, inputs resident in HBM, device-timed over K steps (max over ranks)
  e2e        same metric through pcal_extract_host: pinned HOST buffer -> device inside the timed
             region, result read back to the host every step
  roofline   the fused fold (or generator) kernel: algorithmic input bytes / its average launch duration
             over the timed region (CUDA events on the launching stream; launches overlap under PDL)
  cpu_baseline  the CPU oracle timed on this box's host cores on a bounded sample of the workload
`--impl reference` times the oracle (the only "reference implementation" this paper-only task has).
With N > 1 (torchrun) the stream is time-sharded: each rank folds its own 2^28-sample range at its
absolute start index, the bins are exchanged with one NCCL all-gather and summed in rank order
(weak scaling: per-GPU work fixed).
"""
from __future__ import annotations

import argparse
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


def load_traffic(workload: str, rotator: str):
    """dram bytes per launch of the hot kernel from the committed ncu capture (profiles/r1_traffic.csv), or None."""
    path = os.path.join(ROOT, "profiles", "r1_traffic.csv")
    try:
        for line in open(path).read().splitlines()[1:]:
            wl, rot, b = line.split(",")
            if wl == workload and rot == rotator:
                return int(b)
    except Exception:
        pass
    return None


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


def time_oracle(w, n_sample: int, steps: int = 1):
    """The oracle as it stands (O-fold + DFT), on n_sample samples of workload w, all host cores."""
    import numpy as np
    import oracle as orc
    from paper_2501_05993_b200 import synth
    orc.build()
    ws = w.scaled(n_sample)
    buf = synth.generate(ws, "cpu").numpy()
    cores = os.cpu_count() or 1
    fmt = oracle_fmt(orc, ws)
    t0 = time.perf_counter()
    for _ in range(steps):
        for c in range(ws.n_channels):
            orc.extract(buf, fmt, ws.n_channels, c, n_sample, 0, ws.f_s_hz, ws.f_comb_hz, ws.f_offset_hz[c],
                        tabulated=True, threads=cores)
    dt = (time.perf_counter() - t0) / steps
    return n_sample * ws.n_channels / dt, cores, dt


def measure(idx: int, steps: int, warmup: int, rank: int, world: int, device, do_e2e: bool = True,
            rotator: str | None = None, n_override: int | None = None, min_warm_s: float = 0.5,
            no_graph: bool = False, exchange: bool = False):
    """Run config idx on this rank's GPU; returns the measurement dict (device timing is per rank)."""
    import torch
    import torch.distributed as dist
    from dataclasses import replace
    from paper_2501_05993_b200 import binding, synth

    w = synth.config(idx)
    if n_override:
        w = w.scaled(n_override)
    if rotator:
        w = replace(w, rotator=rotator)
    n, C, nb = w.n_samples, w.n_channels, w.n_bins
    # distinct input copies so that every step reads from DRAM, not from the 126 MB L2
    ncopies = 1 if w.n_bytes >= (300 << 20) else min(8, -(-(300 << 20) // w.n_bytes))
    bufs = [synth.generate(replace(w, seed=w.seed + 100 * i + 7 * rank), device) for i in range(ncopies)]
    exchange = exchange or world > 1
    # Multi-GPU: two contexts ("lanes") alternate, so that the all-gather of integration k is in flight
    # (on NCCL's stream) while integration k+1 is being folded and integration k-1 is being finished.
    ctxs = [binding.from_workload(w) for _ in range(2 if exchange else 1)]
    for q_ in ctxs:
        q_.set_input_ready(True)  # inputs are resident in HBM and complete before the timed region starts
    p = ctxs[0]
    out_pinned = torch.empty((C, nb), dtype=torch.complex128).pin_memory()
    lanes = [{"p": q_, "work": None,
              "local": torch.empty(C * nb * 2, dtype=torch.float64, device=device),
              "gathered": torch.empty(world * C * nb * 2, dtype=torch.float64, device=device),
              "out": torch.empty((C, nb), dtype=torch.complex128).pin_memory()} for q_ in ctxs]

    def complete(L):
        """The one exchange step, second half: rank-order sum of the gathered bins, DFT, result to the host."""
        if L["work"] is not None:
            L["work"].wait()                              # the current stream waits for the all-gather
            L["p"].set_folded_sum_dev(L["gathered"], world)
            L["p"].finalize_async(L["out"])
            L["work"] = None

    def drain():
        for L in lanes:
            complete(L)

    buf_ptrs, out_ptr = [b_.data_ptr() for b_ in bufs], out_pinned.data_ptr()
    cur_stream = int(torch.cuda.current_stream().cuda_stream)

    def step(i, stream=None):
        if not exchange:
            # pcal_reset + pcal_extract + pcal_finalize_async in one call; raw addresses, stream handle hoisted
            p.integrate(buf_ptrs[i % ncopies], n, out_ptr, stream=stream)
            return
        L = lanes[i % 2]
        complete(L)                                       # this lane's previous integration, if still open
        L["p"].reset()
        L["p"].set_start_index(rank * n)                  # time shard of rank r starts at r*n
        L["p"].extract(bufs[i % ncopies], n)
        L["p"].get_folded_dev(L["local"])
        L["work"] = dist.all_gather_into_tensor(L["gathered"], L["local"], async_op=True)
        complete(lanes[(i + 1) % 2])                      # finish the other lane under this all-gather

    # clocks are sampled from the start of the warm-up to the end of the timed region (a timed
    # region of K short steps alone can be shorter than one nvidia-smi period); the warm-up runs
    # >= W steps and >= 0.5 s of the same steps, so the samples are taken under the same load
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
    # Single GPU: the step (reset + extract + finalize_async: 3-4 kernels) is launch-bound for the small
    # configs.  Two ways to issue it are calibrated after the warm-up and the faster one is used for the
    # timed region: (a) direct launches -- the library chains its kernels with programmatic dependent
    # launch, so each kernel is scheduled while its predecessor still runs; (b) one CUDA-graph replay per
    # step (each distinct input copy gets its step captured once).  Multi-GPU steps (NCCL exchange)
    # launch directly.
    use_graph = (world == 1) and not no_graph and not exchange
    graphs, per_step_launches = [], None
    n_big = ncopies * max(1, min(steps, 40) // ncopies)      # steps in the big graph (whole rounds over the copies)
    if use_graph:
        side = torch.cuda.Stream()
        side.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(side):
            for k in range(ncopies):
                l0 = p.info().kernel_launches
                g = torch.cuda.CUDAGraph()
                with torch.cuda.graph(g, stream=side):
                    step(k)
                per_step_launches = p.info().kernel_launches - l0
                graphs.append(g)
            big = torch.cuda.CUDAGraph()              # n_big consecutive steps in ONE graph
            with torch.cuda.graph(big, stream=side):
                for k in range(n_big):
                    step(k)
        torch.cuda.current_stream().wait_stream(side)

    def run_steps(mode, count):
        if mode == "graph_per_step":
            for k in range(count):
                graphs[k % ncopies].replay()
        elif mode == "graph_of_steps":
            for _ in range(count // n_big):
                big.replay()
            for k in range(count % n_big):
                step(k, cur_stream)
        else:
            for k in range(count):
                step(k, cur_stream)
        drain()

    mode = "direct"
    if use_graph:
        def timed(m, reps):
            run_steps(m, n_big)
            torch.cuda.synchronize()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record()
            run_steps(m, reps)
            b.record()
            torch.cuda.synchronize()
            return a.elapsed_time(b) / reps
        reps = max(2 * n_big, steps)
        cal = {m: min(timed(m, reps) for _ in range(2)) for m in ("direct", "graph_per_step", "graph_of_steps")}
        mode = min(cal, key=cal.get)
    launches0 = sum(q_.info().kernel_launches for q_ in ctxs)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    run_steps(mode, steps)
    e1.record()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    ms = e0.elapsed_time(e1)
    launches = per_step_launches * steps if use_graph else sum(q_.info().kernel_launches for q_ in ctxs) - launches0
    use_graph = mode != "direct"
    # second pass over the same K steps, launched directly, with the hot kernel bracketed by CUDA
    # events on the launching stream (pcal_set_profiling): the roofline numerator
    for q_ in ctxs:
        q_.set_profiling(True)
    for i in range(steps):
        step(i)
    drain()
    torch.cuda.synchronize()
    hot_ms, hot_launches = 0.0, 0
    for q_ in ctxs:
        ms_q, n_q = q_.get_profile()
        hot_ms, hot_launches = hot_ms + ms_q, hot_launches + n_q
        q_.set_profiling(False)
    clocks = sampler.stop() if rank == 0 else None
    del graphs
    big = None
    if world > 1:
        t = torch.tensor([ms], dtype=torch.float64, device=device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms = float(t.item())
    inf = p.info()
    res = {
        "workload": w.name, "n_samples_per_channel": n, "n_channels": C, "n_bins": nb, "bits": w.bits,
        "input_bytes": w.n_bytes, "rotator": {1: "lut", 2: "generator"}[inf.rotator_in_effect],
        "fold_period": int(inf.fold_period), "ms_per_step": ms / steps,
        "value": world * n * C * steps / (ms * 1e-3),
        "input_gbs": world * w.n_bytes * steps / (ms * 1e-3) / 1e9,
        "hot_kernel_us": 1e3 * hot_ms / max(hot_launches, 1), "hot_kernel_launches": int(hot_launches),
        "gpu_launches": int(launches),
        "launch_mode": {"direct": "direct launches (kernels chained by programmatic dependent launch)",
                        "graph_per_step": "cuda_graph: one graph replay per step (reset + extract + finalize_async captured once per input copy)",
                        "graph_of_steps": f"cuda_graph: one replay per {n_big} consecutive steps (cycling over the input copies), kernels chained "
                                          "by programmatic dependent launch inside the graph; remainder steps launched directly"}[mode],
        "launch_mode_calibration_us": {k_: 1e3 * v_ for k_, v_ in cal.items()} if world == 1 and not no_graph and not exchange else None,
        "l2_policy": f"rotating {ncopies} distinct input copies "
        f"({ncopies * w.n_bytes / 2**20:.0f} MiB total vs 126 MB L2)" if ncopies > 1 else "input larger than L2",
        "clocks": clocks,
    }
    peak, peak_src = load_peaks()
    # calibration: a pure streaming read of the same buffers (no decode, no fold), launched back to back
    # like the steps above (launches may overlap under programmatic dependent launch), timed the same way
    floor_us = None
    if rank == 0:
        for i in range(ncopies):
            p.read_probe(bufs[i % ncopies])
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for i in range(max(steps, 2 * ncopies)):
            p.read_probe(bufs[i % ncopies])
        b.record()
        torch.cuda.synchronize()
        floor_us = 1e3 * a.elapsed_time(b) / max(steps, 2 * ncopies)
    # The dominant kernel's average launch duration over the timed region: consecutive launches overlap
    # (programmatic dependent launch), so it is the region's device time / the kernel's launches in it --
    # an upper bound, the small DFT kernel of every step is inside.  `isolated_kernel_us` is the same kernel
    # bracketed by events launch by launch (which serialises the launches: its latency, not its cost).
    fold_launches = steps * max(1, round(hot_launches / steps)) if hot_launches else steps
    bytes_per_launch = w.n_bytes * steps / fold_launches
    hot_s = 1e-3 * ms / fold_launches
    achieved = bytes_per_launch / hot_s / 1e9
    gen = inf.rotator_in_effect == 2
    res["roofline"] = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s",
                       "frac": achieved / peak, "traffic": None, "peak_source": peak_src,
                       "kernel": "gen_kernel (generator path)" if gen else "fold_*_kernel incl. fused tail (LUT path)",
                       "algorithmic_bytes_per_launch": bytes_per_launch,
                       "avg_launch_us": hot_s * 1e6, "launches_in_timed_region": fold_launches,
                       "isolated_kernel_us": 1e3 * hot_ms / max(hot_launches, 1),
                       "how": "device time of the timed region (CUDA events on the launching stream) / launches of the kernel in it"}
    res["roofline"]["traffic"] = load_traffic(w.name, res["rotator"]) if not n_override else None
    res["hot_kernel_us"], res["hot_kernel_isolated_us"] = hot_s * 1e6, 1e3 * hot_ms / max(hot_launches, 1)
    if floor_us:
        res["roofline"]["read_floor"] = {
            "us": floor_us, "gbs": w.n_bytes / floor_us / 1e3, "frac_of_floor": floor_us / (hot_s * 1e6),
            "what": "pcal_read_probe: pure streaming read of the same buffers (no decode/fold), back-to-back launches timed like the steps"}
    if gen and w.bits == 2:
        # 2-bit generator variant: the work per byte is 4x that of int8.  Reported against HBM like every other
        # row; the issue rate the kernel would need at the HBM rate is given beside it.
        sm_mhz = (clocks or {}).get("sm_max_mhz") or 1965.0
        res["roofline"]["issue_peak_ginstr_s"] = 148 * 4 * 32 * sm_mhz * 1e6 / 1e9
        res["roofline"]["samples_per_s"] = n * C * steps / fold_launches / hot_s
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


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config (1-based); default configs[1]")
    ap.add_argument("--impl", default="own", choices=["own", "reference"])
    ap.add_argument("--no-all", action="store_true", help="skip the short per-config table")
    ap.add_argument("--samples", type=int, default=0, help="override samples per channel (debug)")
    ap.add_argument("--rotator", default=None, choices=["lut", "generator"], help="force the rotator variant (config 3 runs both)")
    ap.add_argument("--no-graph", action="store_true", help="launch every step directly instead of replaying a CUDA graph")
    ap.add_argument("--force-exchange", action="store_true",
                    help="testing: run the multi-GPU exchange path (NCCL all-gather + rank-order sum) even with one rank")
    ap.add_argument("--quick", action="store_true",
                    help="profiling mode (ncu): exactly W warm-up steps, no e2e / cpu_baseline / per-config table")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    from paper_2501_05993_b200 import synth

    if args.impl == "reference":
        if rank != 0:
            return
        w = synth.config(args.config)
        n_sample = 1 << 24
        for _ in range(max(args.warmup, 1)):
            time_oracle(w, 1 << 20)
        rate, cores, dt = time_oracle(w, n_sample, steps=args.steps)
        line = {"metric": METRIC, "value": rate, "unit": UNIT, "impl": "reference", "n_gpus": args.gpus,
                "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
                "config": {"workload": w.name, "sample": f"first {n_sample} samples per step"},
                "cpu_baseline": {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle",
                                 "sample": f"{n_sample} samples of {w.name} per step, O-fold + DFT, {cores} threads"},
                "e2e": {"value": rate, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
                "gpu_launches": 0}
        print(json.dumps(line), flush=True)
        return

    import torch
    import torch.distributed as dist
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local_rank)
    device = torch.device("cuda", local_rank)
    if world > 1 or args.force_exchange:
        if "RANK" not in os.environ:
            os.environ.update({"RANK": "0", "WORLD_SIZE": "1", "MASTER_ADDR": "127.0.0.1", "MASTER_PORT": "29533"})
        dist.init_process_group("nccl", device_id=device)
    res, w = measure(args.config, args.steps, args.warmup, rank, world, device, n_override=args.samples or None,
                     rotator=args.rotator, no_graph=args.no_graph, exchange=args.force_exchange, do_e2e=not args.quick, min_warm_s=0.0 if args.quick else 0.5)
    line = {"metric": METRIC, "value": res["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": res["ms_per_step"], "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None,
            "dtype": "int32/fp64 (integer fold, fp64 rotate+DFT)" if res["rotator"] == "lut" else "fp32 MAC / fp64 accumulate",
            "data": "synthetic", "input_gbs": res["input_gbs"],
            "config": {"workload": res["workload"], "n_samples_per_channel": res["n_samples_per_channel"],
                       "n_channels": res["n_channels"], "bits": res["bits"], "n_bins": res["n_bins"],
                       "rotator": res["rotator"], "input_bytes_per_gpu": res["input_bytes"],
                       "parallelism": f"time-sharded x{world}" if world > 1 else "single GPU",
                       "l2": res["l2_policy"], "launch_mode": res["launch_mode"],
                       "launch_mode_calibration_us": res["launch_mode_calibration_us"]},
            "clocks": res["clocks"], "e2e": res.get("e2e"), "gpu_launches": res["gpu_launches"],
            "roofline": res["roofline"], "hot_kernel_us": res["hot_kernel_us"]}
    if world == 1 and rank == 0 and not args.quick:
        from paper_2501_05993_b200 import binding as _b
        # measured issue-rate ceilings of this GPU; every reported roofline is HBM, these say how far the ALU side is
        line["pipe_peaks"] = {"ffma_thread_instr_per_s": _b.pipe_probe(0), "lop3_thread_instr_per_s": _b.pipe_probe(1),
                              "imma_m16n8k16_s8_warp_instr_per_s": _b.pipe_probe(2),
                              "how": "pcal_pipe_probe: 8 independent chains per thread, 8 CTAs x 256 threads per SM, best of 3"}
        probe, cores, _ = time_oracle(w, 1 << 21)
        n_sample = int(min(w.n_samples, max(1 << 22, probe * 1.0)))
        n_sample -= n_sample % 64
        _, cores, dt1 = time_oracle(w, n_sample, steps=1)          # also warms the threads
        reps = max(1, min(50, int(round(1.2 / dt1))))              # ~1.2 s wall on all cores (~20 core-seconds on 16)
        rate, cores, dt = time_oracle(w, n_sample, steps=reps)
        line["cpu_baseline"] = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle",
                                "sample": f"first {n_sample} samples of {w.name}, O-fold + DFT, {reps} x {dt:.2f} s wall on {cores} threads"}
        if not args.no_all:
            table = {}
            for idx, rot in [(1, None), (2, None), (3, "lut"), (3, "generator"), (4, None), (5, None), (8, None)]:   # 8 = the paper's own benchmark shape
                r, _ = measure(idx, 20 if idx == 5 else 100, 3, 0, 1, device, do_e2e=False, rotator=rot)
                key = ("paper_benchmark_shape" if idx == 8 else f"cfg{idx}") + (f"_{rot}" if rot else "")
                table[key] = {k: r[k] for k in ("workload", "rotator", "value", "input_gbs", "ms_per_step", "hot_kernel_us", "hot_kernel_isolated_us")}
                table[key]["sm_mhz"] = (r.get("clocks") or {}).get("sm_mhz")
                table[key]["roofline_frac"] = r["roofline"]["frac"]
                table[key]["roofline_achieved_gbs"] = r["roofline"]["achieved"]
            line["all_configs"] = table
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1 or args.force_exchange:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
