#!/usr/bin/env python
"""bench.py -- X-engine throughput on synthetic CHIME-shaped frames (BASELINE.json metric), one JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C2|C4|C5|C3] [--impl reference]
                    [--no-sustained] [--no-other-configs] [--no-e2e] [--no-next-rows] [--no-cpu-baseline] [--no-int8-probe] [--no-graph]

A "step" is one pass of the whole hot path over one frame: xcorr_process (TMA stage -> nibble unpack -> tcgen05
int8 MMAs -> epilogue, rows a1..a4) followed by xcorr_read (the packed-triangle epilogue that ends the integration;
BASELINE.json:configs[1] "one integration per frame").  `value` is input Gb/s with the frames already resident in
HBM; `e2e` is the same metric through the streamed C-ABI path (row a5) with page-locked HOST frames and a HOST
result, copies inside the timed region.  Inputs are synthetic (workloads.py) and larger than L2 (256 MiB frames,
two of them alternating), so no flush is needed between iterations.

Two legs.  A B200 runs xengine_kernel at its 1965 MHz boost for a few milliseconds and then sits at the 1 kW power cap near
1.5 GHz, so K steps from a cool part flatter.  The line's `value`, `ms_per_step`, `clocks` and `roofline` therefore come from
exactly K steps timed directly behind a power-steady leg (the same step back to back for >= 2 s, counted in `warmup`); the K
steps from a cool part are kept as `roofline.burst`.  `roofline.peak` is the issue ceiling of the int8 tensor pipe measured in
the same run (bench_support/probe.py; sustained reading for the steady leg, burst reading for the burst leg); 2 x the
measured cuBLAS bf16 rate is beside it as `frac_of_2x_bf16`.  `roofline` also carries what the driver's record must keep:
the added-frame launches (frames added to a running integration, no read in between -- the telescope's steady state,
PAPER.md:99), the long leg's figures (`sustained_*`) and a compact `configs` table of C3 / C4 / C5.  `other_configs` has
their full entries (C3: the 64-frame streamed run of BASELINE.json configs[2] with its H2D-only ceiling; an oracle timing
beside each), `cpu_baseline.one_core` the oracle on one core.

Multi-GPU: the path does not shard ("replicas only"): --gpus N (under torchrun) runs N independent
replicas, one per GPU, no collective on the data path; value = N frames' bits / max-over-ranks time.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time
from pathlib import Path

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

import numpy as np  # noqa: E402

import workloads as wl  # noqa: E402

NOMINAL_INT8_TOPS = 4500.0  # dense int8, B200 nominal (2x the 2.25 PFLOP/s dense bf16 figure)
# dram__bytes_read.sum + dram__bytes_write.sum of ONE xengine_kernel launch, typed in from the committed ncu --set full captures
# (cold caches; profiles/r03_ncu_full_added_frames.md):
# first-frame launch (the step the line times) and a launch ADDED to a running integration (reduce-adds into the slots)
NCU_TRAFFIC_BYTES = {"C2": 277.36e6, "C3": 1465.30e6, "C4": 668.54e6, "C5": 4158.32e6}
NCU_TRAFFIC_BYTES_ADDED = {"C2": 332.92e6, "C3": 1916.14e6, "C4": 951.01e6, "C5": 4234.63e6}
# tcgen05 MMAs (M256 N256 K32, 2 CTAs) xengine_kernel issues per 32-sample K-step of a 256 x 256 super-tile
MMAS_DIAG, MMAS_OFFDIAG = 2, 4


def issued_over_useful(cfg) -> float:
    """int8 ops the kernel issues / useful ops (8 per complex MAC, pairs i <= j only)."""
    nb = -(-cfg.n_inputs // 256)
    return (MMAS_DIAG * nb + MMAS_OFFDIAG * nb * (nb - 1) // 2) * 65536 / (4.0 * cfg.n_pairs)


def load_peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        d = json.loads(p.read_text())
        return {"hbm_gbs": d["hbm_gbs"], "bf16_burst": d["bf16_tflops"], "bf16_sustained": d.get("bf16_tflops_sustained"),
                "source": "measured"}
    return {"hbm_gbs": 6650.0, "bf16_burst": 1590.0, "bf16_sustained": 1400.0, "source": "fallback"}


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.rows.append(ln.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            c = [x.strip() for x in r.split(",")]
            if len(c) < 7:
                continue
            try:
                sm.append(float(c[0])); mx.append(float(c[1])); pw.append(float(c[2]))
            except ValueError:
                continue
            for nm, v in zip(names, c[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": sorted(reasons)}


def oracle_sample_frame(cfg: wl.Config):
    """The bounded sample of `cfg` the oracle is timed on: a few whole channels of one frame (generated outside the timing)."""
    import oracle
    oracle.build()
    cores = oracle.threads()
    n_ch = max(1, min(cfg.n_freq, 8 * cores if cfg.n_inputs <= 256 else 1))
    t_samp = cfg.n_time if cfg.n_inputs <= 512 else min(cfg.n_time, 2048)
    return wl.make_frame(cfg.kind, cfg.n_inputs, n_ch, t_samp, cfg.seed)


def oracle_sample(cfg: wl.Config, fr=None):
    """Time the oracle, as it stands, on a bounded sample of `cfg` (oracle_sample_frame)."""
    import oracle
    if fr is None:
        fr = oracle_sample_frame(cfg)
    cores = oracle.threads()
    t_samp, n_ch = fr.shape[0], fr.shape[1]
    t0 = time.perf_counter()
    oracle.planar(fr)
    dt = time.perf_counter() - t0
    bits = 8.0 * fr.nbytes
    cmacs = n_ch * t_samp * cfg.n_pairs
    return {"value": bits / dt / 1e9, "unit": "Gb/s", "cores": cores, "kind": "oracle",
            "sample": f"oracle.planar (plain C, int64 accumulators, OpenMP) on {n_ch} of {cfg.n_freq} channels x "
                      f"{t_samp} of {cfg.n_time} samples of one {cfg.name} frame (N={cfg.n_inputs}); {dt:.2f} s",
            "cmac_per_s": cmacs / dt, "seconds": dt}


def oracle_one_core(cfg: wl.Config):
    """The oracle, as it stands, on ONE host core: a child process with OMP_NUM_THREADS=1 (the thread count is fixed when the
    OpenMP runtime starts) timing oracle.planar on a few whole channels of one frame; scaled per complex MAC."""
    n_ch = max(1, min(cfg.n_freq, 4 if cfg.n_inputs <= 256 else 1))
    t_samp = cfg.n_time if cfg.n_inputs <= 256 else min(cfg.n_time, 2048)
    env = dict(os.environ, OMP_NUM_THREADS="1")
    try:
        out = subprocess.run([sys.executable, str(ROOT / "bench.py"), "--oracle-sample", f"{cfg.name}:{n_ch}:{t_samp}"], env=env,
                             capture_output=True, text=True, timeout=300, check=True).stdout
        d = json.loads(out.strip().splitlines()[-1])
    except Exception as e:
        return {"error": str(e)[:160]}
    whole = cfg.cmacs_per_frame / d["cmac_per_s"]
    d["whole_frame_seconds_scaled"] = whole
    d["value_scaled"] = 8.0 * cfg.frame_bytes / whole / 1e9
    d["scaling"] = "per complex MAC: whole frame = sample time x (F*T) / (channels*samples of the sample)"
    return d


def oracle_sample_cli(spec: str):
    name, n_ch, t_samp = spec.split(":")
    cfg = wl.CONFIGS[name]
    import oracle
    oracle.build()
    fr = wl.make_frame(cfg.kind, cfg.n_inputs, int(n_ch), int(t_samp), cfg.seed)
    d = oracle_sample(cfg, fr)
    print(json.dumps({k: d[k] for k in ("value", "unit", "cores", "sample", "cmac_per_s", "seconds")}), flush=True)


def measure_next_rows(cfg, x, xb, torch, st, host_frame, peaks, reps: int = 20):
    """NEXT-2 packet assembly and NEXT-1 lost-sample normalisation on the same frame shape: per-kernel CUDA-event times and
    achieved HBM GB/s against the measured copy bandwidth (both are HBM-bound; algorithmic bytes as stated in DESIGN.md)."""
    n, f, t = cfg.n_inputs, cfg.n_freq, cfg.n_time
    fb = wl.sparse_flag_bits(n, f, t, 99)
    pk = wl.packetise(host_frame, fb, 10 ** 12)
    arrived = wl.disturb_packets(pk, 98, p_loss=2e-3, p_dup=1e-3, p_late=5e-3, n_foreign=16)
    n_pk, pbytes = arrived.shape
    pk_dev = [torch.from_numpy(arrived.reshape(-1)).cuda(), torch.from_numpy(arrived.reshape(-1).copy()).cuda()]
    del pk, arrived
    a = xb.Assembler(n, f, t)
    x.norm_enable()
    frame = torch.empty((t, f, n), dtype=torch.uint8, device="cuda")
    flags = torch.empty((t, f, n // 8), dtype=torch.uint8, device="cuda")
    lost = torch.empty(f, dtype=torch.int32, device="cuda")
    counts = torch.empty(4, dtype=torch.int32, device="cuda")
    vis = torch.empty((f, cfg.n_pairs, 2), dtype=torch.float32, device="cuda")
    ev = lambda: torch.cuda.Event(enable_timing=True)
    names = ["assemble_accounted", "process", "read_normalized"]
    times = {k: [] for k in names}
    for _ in range(200):                         # the host-side packet generation let the clocks drop: bring them back up
        x.process(frame, st)
        x.read(vis.view(torch.int32), st)
    evs = []
    for r in range(reps + 3):
        e = [ev() for _ in range(4)]
        with torch.cuda.stream(st):
            e[0].record(st)
            a.assemble(pk_dev[r % 2], n_pk, 10 ** 12, frame, False, lost, counts, stream=st, account_into=x)   # as the streamed path: no flag field
            e[1].record(st)
            x.process(frame, st)
            e[2].record(st)
            x.read_normalized(vis, stream=st)
            e[3].record(st)
        evs.append(e)
    torch.cuda.synchronize()
    for e in evs[3:]:
        for k, nm in enumerate(names):
            times[nm].append(e[k].elapsed_time(e[k + 1]) * 1e3)
    # the same fused call with the optional flag field written as well (callers that want to keep it)
    with_field = []
    evs = []
    for r in range(reps + 3):
        e = [ev() for _ in range(2)]
        with torch.cuda.stream(st):
            e[0].record(st)
            a.assemble(pk_dev[r % 2], n_pk, 10 ** 12, frame, flags, lost, counts, stream=st, account_into=x)
            e[1].record(st)
            x.process(frame, st)
            x.read_normalized(vis, stream=st)
        evs.append(e)
    torch.cuda.synchronize()
    for e in evs[3:]:
        with_field.append(e[0].elapsed_time(e[1]) * 1e3)
    # the two-call form for callers that bring their own flag field: xcorr_assemble, then xcorr_norm_process_dev on its outputs
    sep = {"assemble": [], "norm_process": []}
    evs = []
    for r in range(reps + 3):
        e = [ev() for _ in range(3)]
        with torch.cuda.stream(st):
            e[0].record(st)
            a.assemble(pk_dev[r % 2], n_pk, 10 ** 12, frame, flags, lost, counts, stream=st)
            e[1].record(st)
            x.norm_process_dev(flags, lost, st)
            e[2].record(st)
            x.process(frame, st)
            x.read_normalized(vis, stream=st)
        evs.append(e)
    torch.cuda.synchronize()
    for e in evs[3:]:
        sep["assemble"].append(e[0].elapsed_time(e[1]) * 1e3)
        sep["norm_process"].append(e[1].elapsed_time(e[2]) * 1e3)
    c = counts.cpu().tolist()
    # the same chain end to end from page-locked HOST packet rings: xcorr_stream_submit_packets per frame (H2D copy of the
    # ring, assemble, correlate, flag / loss accounting) and one normalised read into host memory per frame
    pk_host = [p.cpu().pin_memory() for p in pk_dev]
    del pk_dev
    xs = xb.XCorrStream(x, depth=2)
    xs.attach_assembler(a, n_pk)
    vis_host = torch.empty((f, cfg.n_pairs, 2), dtype=torch.float32).pin_memory()
    for k in range(2):
        xs.submit_packets(pk_host[k % 2], n_pk, 10 ** 12)
        xs.read_normalized(vis_host)
    n_pe = 10
    t0 = time.perf_counter()
    for k in range(n_pe):
        xs.submit_packets(pk_host[k % 2], n_pk, 10 ** 12)
        xs.read_normalized(vis_host)
    torch.cuda.synchronize()
    dt_pe = time.perf_counter() - t0
    xs.close()
    a.close()
    us = {k: statistics.mean(v) for k, v in times.items()}
    us_sep = {k: statistics.mean(v) for k, v in sep.items()}
    asm_bytes = n_pk * pbytes + cfg.frame_bytes          # packets in, frame out (no flag field in the fused form as timed)
    flag_bytes = cfg.frame_bytes // 8
    return {
        "what": "packets (arrival order, device resident) -> xcorr_assemble_accounted (assembly + flag / loss accounting in one pass) -> "
                "xcorr_process -> xcorr_read_normalized; per-call CUDA-event means over %d repetitions" % reps,
        "packets": n_pk, "packet_bytes": pbytes, "kept_dup_rejected_lostpos": c, "us": us,
        "us_two_call_form": us_sep, "us_two_call_form_total": sum(us_sep.values()),
        "us_assemble_accounted_with_flag_field": statistics.mean(with_field),
        "assemble_roofline": {"bound": "hbm", "achieved": asm_bytes / (us["assemble_accounted"] * 1e-6) / 1e9, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                              "frac": asm_bytes / (us["assemble_accounted"] * 1e-6) / 1e9 / peaks["hbm_gbs"], "algorithmic_bytes": asm_bytes,
                              "note": "2 kernels in the timed call: packet_claim_kernel + assemble_kernel<true>, no flag field written (as xcorr_stream_submit_packets "
                                      "calls it); us_two_call_form_total is what it replaces (xcorr_assemble with the flag field + xcorr_norm_process_dev)"},
        "flag_count_roofline": {"bound": "hbm", "achieved": flag_bytes / (us_sep["norm_process"] * 1e-6) / 1e9, "peak": peaks["hbm_gbs"],
                                "unit": "GB/s", "frac": flag_bytes / (us_sep["norm_process"] * 1e-6) / 1e9 / peaks["hbm_gbs"],
                                "algorithmic_bytes": flag_bytes,
                                "note": "two-call form only (xcorr_norm_process_dev = flag_count_kernel + lost_add_kernel on a caller-supplied flag "
                                        "field); the packet pipeline no longer runs it"},
        "pipeline_gbps": 8.0 * cfg.frame_bytes / (sum(us.values()) * 1e-6) / 1e9,
        "e2e_packets": {"value": 8.0 * cfg.frame_bytes * n_pe / dt_pe / 1e9, "unit": "Gb/s of frame (sky) data", "steps": n_pe,
                        "ms_per_step": dt_pe / n_pe * 1e3, "h2d_bytes_per_step": n_pk * pbytes, "d2h_bytes_per_step": cfg.output_bytes,
                        "api": "xcorr_stream_submit_packets(pinned host packet ring) + xcorr_stream_read_normalized(pinned host out)"},
    }


def run_reference(args, cfg):
    """--impl reference: the oracle timed on the host cores, bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    # a step is one whole frame of the config through the oracle (C2: about 2.5 s on 16 cores): K up to 40 and W up to 3 are
    # honoured as given, so the driver's --steps 20 --warmup 3 ends within two minutes
    steps, warm = max(1, min(args.steps, 40)), max(0, min(args.warmup, 3))
    fr = oracle_sample_frame(cfg)
    for _ in range(warm):
        oracle_sample(cfg, fr)
    samples = [oracle_sample(cfg, fr) for _ in range(steps)]
    best = samples[-1]
    v = statistics.mean(s["value"] for s in samples)
    ms = statistics.mean(s["seconds"] for s in samples) * 1e3
    line = {
        "impl": "reference", "metric": "xengine_input_gbps", "value": v, "unit": "Gb/s", "n_gpus": args.gpus, "steps": steps,
        "warmup": warm, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int64",
        "data": "synthetic", "config": {"workload": cfg.name, "n_inputs": cfg.n_inputs, "n_freq": cfg.n_freq,
                                        "t_per_frame": cfg.n_time, "note": "each step = a bounded sample, see cpu_baseline.sample"},
        "cpu_baseline": {"value": v, "unit": "Gb/s", "cores": best["cores"], "kind": "oracle", "sample": best["sample"]},
        "e2e": {"value": v, "unit": "Gb/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "cmac_per_s": statistics.mean(s["cmac_per_s"] for s in samples), "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


class Resident:
    """One config with its frames resident in HBM: handle, two distinct device frames, output buffer, stream."""

    def __init__(self, cfg, xb, torch, n_distinct=2):
        self.cfg, self.torch = cfg, torch
        self.host_frames = [cfg.frame(k) for k in range(n_distinct)]
        self.dev_frames = [torch.from_numpy(f).cuda() for f in self.host_frames]
        self.x = xb.XCorr(cfg.n_inputs, cfg.n_freq, cfg.n_time)
        self.x.promise_complete_frames()      # the frames are resident and complete long before any launch (include/xcorr.h)
        self.out_dev = torch.empty((cfg.n_freq, cfg.n_pairs, 2), dtype=torch.int32, device="cuda")
        self.st = torch.cuda.Stream()
        self.n_distinct = n_distinct

    def step(self, k):
        self.x.process(self.dev_frames[k % self.n_distinct], self.st)
        self.x.read(self.out_dev, self.st)

    def timed_steps(self, steps, barrier):
        """K whole steps between two CUDA events on the launching stream -> total ms."""
        torch = self.torch
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        e0.record(self.st)
        for k in range(steps):
            self.step(k)
        e1.record(self.st)
        barrier()
        return e0.elapsed_time(e1)

    def timed_kernels(self, steps, barrier):
        """The same loop with events around every xcorr_process -> list of xengine_kernel durations in ms."""
        torch = self.torch
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        for k in range(steps):
            evs[k][0].record(self.st)
            self.x.process(self.dev_frames[k % self.n_distinct], self.st)
            evs[k][1].record(self.st)
            self.x.read(self.out_dev, self.st)
        barrier()
        return [a.elapsed_time(b) for a, b in evs]

    def timed_added(self, n, barrier):
        """Frames ADDED to a running integration (the kernels "simply add to the output of the last run", no read in
        between): one first frame, then n launches -> (per-launch xengine_kernel ms from events around each launch,
        ms per launch of the same n launches back to back between two events)."""
        torch = self.torch
        self.x.read(self.out_dev, self.st)
        self.x.process(self.dev_frames[0], self.st)                      # first frame of the integration (stores)
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n)]
        for k in range(n):
            evs[k][0].record(self.st)
            self.x.process(self.dev_frames[(k + 1) % self.n_distinct], self.st)
            evs[k][1].record(self.st)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(self.st)
        for k in range(n):
            self.x.process(self.dev_frames[k % self.n_distinct], self.st)
        e1.record(self.st)
        barrier()
        self.x.read(self.out_dev, self.st)
        barrier()
        return [a.elapsed_time(b) for a, b in evs], e0.elapsed_time(e1) / n

    def close(self):
        self.x.close()
        self.dev_frames = self.host_frames = None


def kstats(ms):
    """mean / median / best of a list of per-launch durations (ms)."""
    return {"mean": statistics.mean(ms), "median": statistics.median(ms), "min": min(ms), "launches": len(ms)}


def added_frames_fit(cfg, n):
    """2 n + 1 frames must stay inside the int32 guard of one integration (16,777,215 samples, include/xcorr.h)."""
    return max(4, min(n, (16777215 // cfg.n_time - 1) // 2))


TRAFFIC_SOURCE = {"C2": "profiles/r03_ncu_full_added_frames.md (captured 2026-11-06)", "C3": "profiles/r03_ncu_full_added_frames.md (captured 2026-11-06)",
                  "C4": "profiles/r03_ncu_full_added_frames.md (captured 2026-11-06)", "C5": "profiles/r03_ncu_full_added_frames.md (captured 2026-11-06)"}


def tensor_roofline(cfg, k_ms, peaks, ceiling=None, leg="sustained"):
    """Tensor roofline entries of xengine_kernel for one launch of `cfg` taking k_ms.  `peak` is the issue ceiling of the int8
    tensor pipe measured in this run on this box (bench_support/probe.py: resident operands, nothing but tcgen05.mma kind::i8) --
    its sustained reading for a kernel timed inside a long, power-steady leg, its burst reading for a kernel timed from a cool
    part.  Without the probe (--no-int8-probe) the stand-in is 2 x the measured cuBLAS bf16 rate of MEASURED_PEAKS.json."""
    alg_ops = 8.0 * cfg.cmacs_per_frame              # 4 real MACs = 8 int8 ops per complex MAC, useful pairs i<=j only
    achieved = alg_ops / (k_ms * 1e-3) / 1e12
    bf16 = peaks["bf16_sustained"] if (leg == "sustained" and peaks.get("bf16_sustained")) else peaks["bf16_burst"]
    if ceiling:
        peak = ceiling["sustained_tops" if leg == "sustained" else "burst_tops"]
        source = f"int8 issue ceiling measured in this run ({leg} reading of bench_support/probe.py)"
    else:
        peak = 2.0 * bf16
        source = f"2 x bf16_tflops ({leg}) of MEASURED_PEAKS.json [{peaks['source']}] x the nominal int8:bf16 ratio 4.5:2.25 (no probe in this run)"
    iou = issued_over_useful(cfg)
    return {"bound": "tensor", "kernel": "xengine_kernel (xcorr_process)", "achieved": achieved, "peak": peak, "unit": "TOP/s",
            "frac": achieved / peak, "leg": leg, "peak_source": source,
            "traffic": NCU_TRAFFIC_BYTES.get(cfg.name), "traffic_added_frame": NCU_TRAFFIC_BYTES_ADDED.get(cfg.name),
            "traffic_source": TRAFFIC_SOURCE.get(cfg.name), "frame_bytes": cfg.frame_bytes,
            "kernel_ms": k_ms, "algorithmic_ops_per_launch": alg_ops,
            "frac_of_nominal_4500": achieved / NOMINAL_INT8_TOPS,
            "frac_of_2x_bf16": achieved / (2.0 * bf16), "peak_2x_bf16": 2.0 * bf16,
            "issued_over_useful": iou, "issued_int8_tops": achieved * iou, "frac_issued_of_peak": achieved * iou / peak,
            "hbm_gbs_staging": cfg.frame_bytes / (k_ms * 1e-3) / 1e9, "hbm_peak_gbs": peaks["hbm_gbs"]}


def measure_graph(r, torch, barrier, group=8, seconds=0.4):
    """The paper's remedy for launch latency -- "pre-loaded chains" of GPU operations -- as a CUDA Graph: `group`
    x (xcorr_process, xcorr_read) on the two alternating resident frames captured once (the tensor map is a kernel parameter, so
    each frame needs its own node) and replayed, against the plain launch loop, ABAB in the same thermal state.  Bench-only: no
    ABI change.  -> dict, or {"error": ...} if the capture is refused."""
    import tempfile
    want = torch.empty_like(r.out_dev)
    r.step(0); r.step(1)
    barrier()
    want.copy_(r.out_dev)                                   # result of a step on frame 1: what the graph's last node must leave
    g = torch.cuda.CUDAGraph()
    dot = None
    try:
        g.enable_debug_mode()
    except Exception:
        pass
    with torch.cuda.graph(g, stream=r.st, capture_error_mode="relaxed"):
        for k in range(group):
            r.step(k)
    try:
        with tempfile.TemporaryDirectory() as td:
            g.debug_dump(os.path.join(td, "g.dot"))
            dot = open(os.path.join(td, "g.dot")).read()
    except Exception:
        dot = None
    r.out_dev.zero_()
    with torch.cuda.stream(r.st):
        g.replay()
    barrier()
    exact = bool(torch.equal(r.out_dev, want))

    def plain(n):
        return r.timed_steps(n, barrier) / n

    def replayed(n):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        with torch.cuda.stream(r.st):
            e0.record(r.st)
            for _ in range(n // group):
                g.replay()
            e1.record(r.st)
        barrier()
        return e0.elapsed_time(e1) / (n // group * group)

    n = max(group, int(seconds * 1e3 / plain(200)) // group * group)
    plain(n)                                                # bring the part to the steady state both arms are timed in
    a, b = [], []
    for _ in range(3):
        a.append(plain(n)); b.append(replayed(n))
    out = {"group": group, "steps_per_arm": n, "plain_ms_per_step": statistics.median(a), "graph_ms_per_step": statistics.median(b),
           "gain": statistics.median(a) / statistics.median(b), "plain_all": a, "graph_all": b, "replay_exact": exact,
           "what": "ABAB, 3 rounds of %d steps per arm, medians; one graph = %d x (xcorr_process, xcorr_read) on 2 alternating frames" % (n, group)}
    if dot is not None:
        out["graph_nodes"] = dot.count("KERNEL")
        out["programmatic_edges_in_dot"] = dot.lower().count("programmatic")
    del g
    return out


C3_POOL = 4     # distinct seeded frames the 64-frame streamed run cycles through (1 GiB each, page-locked)


def measure_other_config(name, xb, torch, peaks, ceiling, steps=20, min_seconds=1.0, cpu=True):
    """C4 / C5 (device-resident step) and C3 (device-resident step + the 64-frame streamed run of BASELINE.json configs[2]).
    The step leg runs for at least `min_seconds` (power-steady); the per-launch kernel times are taken straight behind it."""
    cfg = wl.CONFIGS[name]
    r = Resident(cfg, xb, torch)

    def barrier():
        torch.cuda.synchronize()

    for k in range(3):
        r.step(k)
    probe_ms = r.timed_steps(steps, barrier) / steps
    n_steps = max(steps, int(min_seconds * 1e3 / probe_ms))
    total_ms = r.timed_steps(n_steps, barrier)
    kern = r.timed_kernels(max(steps, 20), barrier)
    added, added_b2b = r.timed_added(added_frames_fit(cfg, 24), barrier)
    k_ms = statistics.mean(kern)
    ms = total_ms / n_steps
    out = {"workload": name, "n_inputs": cfg.n_inputs, "n_freq": cfg.n_freq, "t_per_frame": cfg.n_time, "steps": n_steps,
           "ms_per_step": ms, "value_gbps": 8.0 * cfg.frame_bytes / (ms * 1e-3) / 1e9, "cmac_per_s": cfg.cmacs_per_frame / (ms * 1e-3),
           "kernel_ms": k_ms, "kernel_ms_min": min(kern), "kernel_ms_median": statistics.median(kern),
           "added_frame_kernel_ms": kstats(added), "added_frame_back_to_back_ms": added_b2b,
           "added_over_first_median": statistics.median(added) / statistics.median(kern),
           "roofline": tensor_roofline(cfg, k_ms, peaks, ceiling, "sustained")}
    if cpu:
        try:
            c = oracle_sample(cfg)
            out["cpu_oracle"] = {k: c[k] for k in ("value", "unit", "cores", "sample", "cmac_per_s")}
        except Exception as e:
            out["cpu_oracle"] = {"error": str(e)[:160]}
    if cfg.n_frames > 1:
        # BASELINE.json configs[2]: n_frames consecutive frames from pinned host memory, double-buffered H2D overlapped with
        # the correlation, ONE read at the end
        # (BASELINE.json configs[2]: 64 consecutive seeded frames; a pool of C3_POOL distinct seeded frames is cycled, as
        # SURVEY.md section 8(d) allows -- the same pool size tests/test_gpu_parity.py::test_c3_streamed_64_frames checks)
        pool = r.host_frames + [cfg.frame(k) for k in range(len(r.host_frames), C3_POOL)]
        pinned = [torch.from_numpy(f).pin_memory() for f in pool]
        out_host = torch.empty((cfg.n_freq, cfg.n_pairs, 2), dtype=torch.int32).pin_memory()
        s = xb.XCorrStream(r.x, depth=2)
        for k in range(2):
            s.submit(pinned[k % C3_POOL])
        s.read(out_host)
        barrier()
        t0 = time.perf_counter()
        for k in range(cfg.n_frames):
            s.submit(pinned[k % C3_POOL])
        s.read(out_host)
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        hb = torch.empty(cfg.frame_bytes, dtype=torch.uint8, device="cuda")
        torch.cuda.synchronize()
        t1 = time.perf_counter()
        for k in range(4):
            hb.copy_(pinned[k % C3_POOL].view(-1), non_blocking=True)
        torch.cuda.synchronize()
        h2d = 8.0 * 4 * cfg.frame_bytes / (time.perf_counter() - t1) / 1e9
        del hb
        s.close()
        out["streamed"] = {"value": 8.0 * cfg.frame_bytes * cfg.n_frames / dt / 1e9, "unit": "Gb/s", "frames": cfg.n_frames,
                           "pool": C3_POOL, "ms_per_frame": dt / cfg.n_frames * 1e3, "h2d_only_gbps": h2d, "paper_rate_gbps": 819.2,
                           "h2d_bytes_per_frame": cfg.frame_bytes, "d2h_bytes_total": cfg.output_bytes,
                           "api": f"{cfg.n_frames} x xcorr_stream_submit(pinned host frame, pool of {C3_POOL} distinct frames cycled) + one "
                                  "xcorr_stream_read(pinned host out); host wall clock from the first submit to the result in host memory"}
    r.close()
    torch.cuda.empty_cache()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2000)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="C2", choices=sorted(wl.CONFIGS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-next-rows", action="store_true")
    ap.add_argument("--no-int8-probe", action="store_true")
    ap.add_argument("--no-sustained", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true")
    ap.add_argument("--no-graph", action="store_true")
    ap.add_argument("--sustained-seconds", type=float, default=2.0)
    ap.add_argument("--oracle-sample", default=None, help=argparse.SUPPRESS)   # child of oracle_one_core: NAME:channels:samples
    args = ap.parse_args()
    if args.oracle_sample:
        return oracle_sample_cli(args.oracle_sample)
    cfg = wl.CONFIGS[args.config]
    if args.impl == "reference":
        return run_reference(args, cfg)

    import torch
    import paper_1503_06189_b200 as xb
    from bench_support import probe
    from paper_1503_06189_b200 import replicas

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    warm = max(3, args.warmup)
    steps = max(1, args.steps)
    peaks = load_peaks()
    solo = rank == 0 and world == 1

    # ---- synthetic inputs, resident in HBM before the timed region: two distinct frames, alternating
    n_distinct = 2
    r = Resident(cfg, xb, torch, n_distinct)
    x, st, host_frames = r.x, r.st, r.host_frames

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- leg 1, "burst": W warm-up steps on a cool part, then K whole steps and K per-kernel timings.  A B200 runs this kernel
    # at 1965 MHz for a few ms before the power cap (1 kW) pulls the clock down, so this leg flatters; it is reported as `burst`
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.15)            # (the sampler's first reading; before the warm-up so that nothing idles between it and the timed steps)
    for k in range(warm):
        r.step(k)
    barrier()
    burst_total = replicas.max_over_ranks(r.timed_steps(steps, barrier), dist, "cuda")
    burst_kern = r.timed_kernels(max(steps, 20), barrier)
    burst_clocks = sampler.stop()
    burst_ms = burst_total / steps
    bits_per_frame = 8.0 * cfg.frame_bytes

    # ---- the int8 tensor issue ceiling of this box (resident operands, no TMA / unpack / epilogue): burst and >= 4 s sustained
    ceiling = None
    if rank == 0 and not args.no_int8_probe:
        try:
            ceiling = probe.int8_issue_ceiling(pattern=1, sustained_seconds=4.0 if solo else 1.0)
        except Exception as e:
            ceiling = None
            probe_error = str(e)[:160]

    # ---- leg 2, power-steady: the same step back to back for >= sustained_seconds (clocks sampled from here on), and straight
    # behind it, with nothing idling in between, THE timed region of the line: exactly K steps, then the per-kernel timings and
    # the added-frame launches.  `value`, `ms_per_step` and `roofline` come from this leg.
    sustained = None
    warm_total = warm
    if not args.no_sustained:
        n_sus = max(steps, int(args.sustained_seconds * 1e3 / burst_ms))
        warm_total += n_sus // 4 + n_sus
        clk = ClockSampler(local)
        clk.start()
        for k in range(n_sus // 4):                       # bring the part to its steady state first (not timed)
            r.step(k)
        barrier()
        sus_total = replicas.max_over_ranks(r.timed_steps(n_sus, barrier), dist, "cuda")
    else:
        clk = ClockSampler(local)
        clk.start()
    launches0 = x.kernel_launches
    total_ms = r.timed_steps(steps, barrier)
    launches = x.kernel_launches - launches0
    kern_ms = r.timed_kernels(max(steps, 20), barrier)
    added_ms, added_b2b = r.timed_added(added_frames_fit(cfg, max(24, min(steps, 200))), barrier)
    clocks = clk.stop()
    leg = "burst" if args.no_sustained else "sustained"
    clocks["note"] = ("sampled over the power-steady leg (>= %.1f s of back-to-back steps) and the K timed steps that follow it directly"
                      % args.sustained_seconds) if leg == "sustained" else "sampled over the K timed steps only (--no-sustained)"

    total_ms = replicas.max_over_ranks(total_ms, dist, "cuda")
    ms_per_step = total_ms / steps
    value = world * bits_per_frame / (ms_per_step * 1e-3) / 1e9
    cmac_per_s = world * cfg.cmacs_per_frame / (ms_per_step * 1e-3)

    # ---- roofline of the dominant kernel (tensor-bound: a dense int8 contraction) against the measured int8 issue ceiling
    k_ms = statistics.mean(kern_ms)
    roofline = tensor_roofline(cfg, k_ms, peaks, ceiling, leg)
    roofline["kernel_ms_median"] = statistics.median(kern_ms)
    roofline["kernel_ms_min"] = min(kern_ms)
    roofline["kernel_launches_timed"] = len(kern_ms)
    # frames ADDED to a running integration: what the telescope runs 99.6 % of the time (PAPER.md:99, 10 s cadence)
    roofline["added_frame_kernel_ms"] = kstats(added_ms)
    roofline["added_frame_back_to_back_ms"] = added_b2b
    roofline["added_over_first_median"] = statistics.median(added_ms) / statistics.median(kern_ms)
    bk = statistics.mean(burst_kern)
    rb = tensor_roofline(cfg, bk, peaks, ceiling, "burst")
    roofline["burst"] = {"kernel_ms": kstats(burst_kern), "ms_per_step": burst_ms, "value": world * bits_per_frame / (burst_ms * 1e-3) / 1e9,
                         "achieved": rb["achieved"], "peak": rb["peak"], "frac": rb["frac"], "frac_of_nominal_4500": rb["frac_of_nominal_4500"],
                         "frac_of_2x_bf16": rb["frac_of_2x_bf16"], "clocks": burst_clocks,
                         "note": "K steps from a cool part after W = %d warm-up steps: the first milliseconds before the power cap acts" % warm}
    if ceiling:
        roofline["int8_issue_ceiling"] = ceiling
    elif rank == 0 and not args.no_int8_probe:
        roofline["int8_issue_ceiling_error"] = probe_error

    # context: the library's own int8 GEMM on this box in this run (cuBLAS through torch._int_mm, 8192^3, best of 10)
    if rank == 0 and not args.no_int8_probe:
        try:
            ga = torch.randint(-8, 8, (8192, 8192), dtype=torch.int8, device="cuda")
            gb = torch.randint(-8, 8, (8192, 8192), dtype=torch.int8, device="cuda")
            best = None
            for k in range(13):
                g0, g1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                g0.record()
                torch._int_mm(ga, gb)
                g1.record()
                torch.cuda.synchronize()
                if k >= 3:
                    best = g0.elapsed_time(g1) if best is None else min(best, g0.elapsed_time(g1))
            roofline["cublas_int8_gemm_8192_tops_burst"] = 2.0 * 8192 ** 3 / (best * 1e-3) / 1e12
            del ga, gb
        except Exception as e:  # context only
            roofline["cublas_int8_gemm_8192_tops_burst"] = None
            roofline["int8_probe_error"] = str(e)[:120]

    if not args.no_sustained:
        sus_ms = sus_total / n_sus
        step_tops = 8.0 * cfg.cmacs_per_frame / (sus_ms * 1e-3) / 1e12
        sustained = {"steps": n_sus, "seconds": sus_total * 1e-3, "ms_per_step": sus_ms,
                     "value": world * bits_per_frame / (sus_ms * 1e-3) / 1e9, "unit": "Gb/s",
                     "cmac_per_s": world * cfg.cmacs_per_frame / (sus_ms * 1e-3),
                     "step_frac_of_peak": step_tops / roofline["peak"], "step_frac_of_nominal_4500": step_tops / NOMINAL_INT8_TOPS,
                     "note": "the long leg in front of the K timed steps; kernel times of this state are roofline.kernel_ms*"}
        # the driver keeps `roofline`: the long leg's figures go there too
        roofline["sustained_ms_per_step"] = sus_ms
        roofline["sustained_seconds"] = sus_total * 1e-3
        roofline["sustained_kernel_ms"] = k_ms
        roofline["sustained_frac"] = roofline["frac"]
        roofline["sustained_frac_of_nominal"] = roofline["frac_of_nominal_4500"]
        roofline["sustained_step_frac_of_peak"] = step_tops / roofline["peak"]
        roofline["sustained_clocks"] = clocks

    # ---- e2e: streamed C-ABI path, HOST frames in, HOST visibilities out, every step
    e2e = None
    if not args.no_e2e:
        pinned = [torch.from_numpy(f).pin_memory() for f in host_frames]
        out_host = torch.empty((cfg.n_freq, cfg.n_pairs, 2), dtype=torch.int32).pin_memory()
        s = xb.XCorrStream(x, depth=2)
        for k in range(2):
            s.submit(pinned[k % n_distinct]); s.read(out_host)
        barrier()
        if cfg.n_frames > 1:
            # streamed config (C3): n_frames consecutive frames from a pool of pinned host frames, double-buffered H2D
            # overlapped with the correlation, ONE read at the end of the integration (BASELINE.json:configs[2])
            n_e2e = cfg.n_frames
            t0 = time.perf_counter()
            for k in range(n_e2e):
                s.submit(pinned[k % n_distinct])
            s.read(out_host)
            torch.cuda.synchronize()
            dt = time.perf_counter() - t0
            api = (f"{n_e2e} x xcorr_stream_submit(pinned host frame, pool of {n_distinct} distinct frames cycled) + one "
                   "xcorr_stream_read(pinned host out)")
            d2h = cfg.output_bytes / n_e2e
        else:
            # one integration per frame: every step copies its frame in and its visibilities out; the read is enqueued
            # without waiting so that the next frame's H2D copy overlaps it (PCIe is full duplex); two host result buffers
            n_e2e = max(2, min(steps, 20))
            out_hosts = [out_host, torch.empty_like(out_host).pin_memory()]
            t0 = time.perf_counter()
            for k in range(n_e2e):
                s.submit(pinned[k % n_distinct])
                s.read_async(out_hosts[k % 2])
            s.sync()
            torch.cuda.synchronize()
            dt = time.perf_counter() - t0
            api = "per step: xcorr_stream_submit(pinned host frame) + xcorr_stream_read_async(pinned host out); one xcorr_stream_sync at the end"
            d2h = cfg.output_bytes
        dt = replicas.max_over_ranks(dt, dist, "cuda")
        # the PCIe ceiling beside it: the same pinned frames copied host -> device with nothing else running
        hb = torch.empty(cfg.frame_bytes, dtype=torch.uint8, device="cuda")
        torch.cuda.synchronize()
        t1 = time.perf_counter()
        for k in range(4):
            hb.copy_(pinned[k % n_distinct].view(-1), non_blocking=True)
        torch.cuda.synchronize()
        h2d_gbps = 8.0 * 4 * cfg.frame_bytes / (time.perf_counter() - t1) / 1e9
        del hb
        e2e = {"value": world * bits_per_frame * n_e2e / dt / 1e9, "unit": "Gb/s", "h2d_bytes_per_step": cfg.frame_bytes,
               "d2h_bytes_per_step": d2h, "steps": n_e2e, "ms_per_step": dt / n_e2e * 1e3, "api": api,
               "h2d_only_gbps": h2d_gbps, "paper_rate_gbps": 819.2 if cfg.name == "C3" else None}
        s.close()
        del pinned

    # ---- the rows SURVEY.md 8(f) marks "next", same frame shape, timed one by one with CUDA events (not part of `value`)
    next_rows = None
    if solo and not args.no_next_rows and cfg.n_freq % wl.PACKET_F == 0 and cfg.n_time % wl.PACKET_T == 0:
        next_rows = measure_next_rows(cfg, x, xb, torch, st, host_frames[0], peaks)
    # ---- launch granularity: a CUDA Graph of steps against the plain loop (pre-loaded chains)
    if solo and not args.no_graph:
        try:
            roofline["graph"] = measure_graph(r, torch, barrier)
        except Exception as e:
            roofline["graph"] = {"error": str(e)[:200]}
            torch.cuda.synchronize()
    r.close()
    torch.cuda.empty_cache()

    # ---- the other BASELINE.json configs, a few steps each (inputs generated outside the timed regions)
    other = None
    if solo and not args.no_other_configs:
        other = {}
        for name in ("C3", "C4", "C5"):
            if name == cfg.name:
                continue
            try:
                other[name] = measure_other_config(name, xb, torch, peaks, ceiling)
            except Exception as e:      # e.g. not enough pinned host memory for C3 on a small box: say so, keep the line
                other[name] = {"error": str(e)[:200]}

    cpu = None
    if solo and not args.no_cpu_baseline:
        cpu = oracle_sample(cfg)
        cpu = {k: cpu[k] for k in ("value", "unit", "cores", "kind", "sample", "cmac_per_s")}
        cpu["one_core"] = oracle_one_core(cfg)

    if other:
        # compact copy inside `roofline` (the key the driver's record keeps)
        roofline["configs"] = {
            nm: ({"kernel_ms": o["kernel_ms"], "kernel_ms_median": o["kernel_ms_median"], "kernel_ms_min": o["kernel_ms_min"],
                  "ms_per_step": o["ms_per_step"], "frac": o["roofline"]["frac"], "frac_of_nominal": o["roofline"]["frac_of_nominal_4500"],
                  "added_frame_kernel_ms_median": o["added_frame_kernel_ms"]["median"],
                  "added_frame_kernel_ms_min": o["added_frame_kernel_ms"]["min"], "added_over_first_median": o["added_over_first_median"],
                  "streamed_gbps": (o.get("streamed") or {}).get("value"), "h2d_only_gbps": (o.get("streamed") or {}).get("h2d_only_gbps")}
                 if "error" not in o else o)
            for nm, o in other.items()}

    if rank == 0:
        peak = roofline["peak"]
        line = {
            "metric": "xengine_input_gbps", "value": value, "unit": "Gb/s", "n_gpus": world, "steps": steps, "warmup": warm_total,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int8",
            "data": "synthetic",
            "config": {"workload": cfg.name, "n_inputs": cfg.n_inputs, "n_freq": cfg.n_freq, "t_per_frame": cfg.n_time,
                       "frame_bytes": cfg.frame_bytes, "step": "xcorr_process + xcorr_read (one integration per frame)", "options": "xcorr_promise_complete_frames(1)",
                       "l2": f"inputs larger than L2: {n_distinct} distinct {cfg.frame_bytes >> 20} MiB frames alternate",
                       "parallelism": "replicas only" if world > 1 else "1 GPU", "note": cfg.note,
                       "timed_region": ("exactly K steps directly behind a power-steady leg of >= %.1f s of the same steps (counted in `warmup`); "
                                        "the K steps from a cool part are roofline.burst" % args.sustained_seconds) if leg == "sustained"
                                       else "K steps after W warm-up steps (--no-sustained)"},
            "cmac_per_s": cmac_per_s,
            "pct_int8_peak_nominal": 100.0 * 8.0 * cmac_per_s / world / (NOMINAL_INT8_TOPS * 1e12),
            "pct_int8_issue_ceiling_measured": 100.0 * 8.0 * cmac_per_s / world / (peak * 1e12),
            "paper_context": "51.2 Gb/s per 3-GPU server, 819.2 Gb/s over 16 servers (PAPER.md Table I; other hardware)",
            "roofline": roofline, "sustained": sustained, "cpu_baseline": cpu, "e2e": e2e, "other_configs": other,
            "next_rows": next_rows, "gpu_launches": int(launches), "clocks": clocks,
        }
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
