#!/usr/bin/env python
"""bench.py -- X-engine throughput on synthetic CHIME-shaped frames (BASELINE.json metric), one JSON line.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C2|C4|C5|C3] [--impl reference]

A "step" is one pass of the whole hot path over one frame: xcorr_process (TMA stage -> nibble unpack -> tcgen05
int8 MMAs -> epilogue, rows a1..a4) followed by xcorr_read (the packed-triangle epilogue that ends the integration;
BASELINE.json:configs[1] "one integration per frame").  `value` is input Gb/s with the frames already resident in
HBM; `e2e` is the same metric through the streamed C-ABI path (row a5) with page-locked HOST frames and a HOST
result, copies inside the timed region.  Inputs are synthetic (workloads.py) and larger than L2 (256 MiB frames,
two of them alternating), so no flush is needed between iterations.

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
# dram__bytes_read.sum + dram__bytes_write.sum of xengine_kernel<false> for one C2 launch, from the committed
# ncu --set full capture summarised in profiles/ (None until a capture exists)
NCU_TRAFFIC_BYTES = {"C2": 277.2e6}   # profiles/r01_ncu_full_bench_c2.md: 268.49 MB read + 8.66 MB written


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


def oracle_sample(cfg: wl.Config, seconds_hint: float = 12.0):
    """Time the oracle, as it stands, on a bounded sample of `cfg`: a few whole channels of one frame."""
    import oracle
    oracle.build()
    cores = oracle.threads()
    n_ch = max(1, min(cfg.n_freq, 8 * cores if cfg.n_inputs <= 256 else 1))
    t_samp = cfg.n_time if cfg.n_inputs <= 512 else min(cfg.n_time, 2048)
    fr = wl.make_frame(cfg.kind, cfg.n_inputs, n_ch, t_samp, cfg.seed)
    t0 = time.perf_counter()
    oracle.planar(fr)
    dt = time.perf_counter() - t0
    bits = 8.0 * fr.nbytes
    cmacs = n_ch * t_samp * cfg.n_pairs
    return {"value": bits / dt / 1e9, "unit": "Gb/s", "cores": cores, "kind": "oracle",
            "sample": f"oracle.planar (plain C, int64 accumulators, OpenMP) on {n_ch} of {cfg.n_freq} channels x "
                      f"{t_samp} of {cfg.n_time} samples of one {cfg.name} frame (N={cfg.n_inputs}); {dt:.2f} s",
            "cmac_per_s": cmacs / dt, "seconds": dt}


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
    names = ["assemble", "process", "norm_process", "read_normalized"]
    times = {k: [] for k in names}
    for _ in range(200):                         # the host-side packet generation let the clocks drop: bring them back up
        x.process(frame, st)
        x.read(vis.view(torch.int32), st)
    evs = []
    for r in range(reps + 3):
        e = [ev() for _ in range(5)]
        with torch.cuda.stream(st):
            e[0].record(st)
            a.assemble(pk_dev[r % 2], n_pk, 10 ** 12, frame, flags, lost, counts, stream=st)
            e[1].record(st)
            x.process(frame, st)
            e[2].record(st)
            x.norm_process_dev(flags, lost, st)
            e[3].record(st)
            x.read_normalized(vis, stream=st)
            e[4].record(st)
        evs.append(e)
    torch.cuda.synchronize()
    for e in evs[3:]:
        for k, nm in enumerate(names):
            times[nm].append(e[k].elapsed_time(e[k + 1]) * 1e3)
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
    asm_bytes = n_pk * pbytes + cfg.frame_bytes + cfg.frame_bytes // 8
    flag_bytes = cfg.frame_bytes // 8
    return {
        "what": "packets (arrival order, device resident) -> xcorr_assemble -> xcorr_process -> xcorr_norm_process_dev -> "
                "xcorr_read_normalized; per-call CUDA-event means over %d repetitions" % reps,
        "packets": n_pk, "packet_bytes": pbytes, "kept_dup_rejected_lostpos": c, "us": us,
        "assemble_roofline": {"bound": "hbm", "achieved": asm_bytes / (us["assemble"] * 1e-6) / 1e9, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                              "frac": asm_bytes / (us["assemble"] * 1e-6) / 1e9 / peaks["hbm_gbs"], "algorithmic_bytes": asm_bytes,
                              "note": "2 kernels in the timed call: packet_claim_kernel + assemble_kernel"},
        "flag_count_roofline": {"bound": "hbm", "achieved": flag_bytes / (us["norm_process"] * 1e-6) / 1e9, "peak": peaks["hbm_gbs"],
                                "unit": "GB/s", "frac": flag_bytes / (us["norm_process"] * 1e-6) / 1e9 / peaks["hbm_gbs"],
                                "algorithmic_bytes": flag_bytes,
                                "note": "flag_count_kernel + lost_add_kernel; the flag field was just written, so part of it is an L2 hit"},
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
    steps, warm = max(1, min(args.steps, 5)), max(0, min(args.warmup, 1))
    for _ in range(warm):
        oracle_sample(cfg)
    samples = [oracle_sample(cfg) for _ in range(steps)]
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
    args = ap.parse_args()
    cfg = wl.CONFIGS[args.config]
    if args.impl == "reference":
        return run_reference(args, cfg)

    import torch
    import paper_1503_06189_b200 as xb
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

    # ---- synthetic inputs, resident in HBM before the timed region: two distinct frames, alternating
    n_distinct = 2
    host_frames = [cfg.frame(k) for k in range(n_distinct)]
    dev_frames = [torch.from_numpy(f).cuda() for f in host_frames]
    x = xb.XCorr(cfg.n_inputs, cfg.n_freq, cfg.n_time)
    x.promise_complete_frames()      # the frames are resident and complete long before any launch (include/xcorr.h)
    out_dev = torch.empty((cfg.n_freq, cfg.n_pairs, 2), dtype=torch.int32, device="cuda")
    st = torch.cuda.Stream()

    def step(k):
        x.process(dev_frames[k % n_distinct], st)
        x.read(out_dev, st)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for k in range(warm):
        step(k)
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.15)
    # -- timed region 1: K whole steps, CUDA events on the launching stream
    launches0 = x.kernel_launches
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record(st)
    for k in range(steps):
        step(k)
    e1.record(st)
    barrier()
    total_ms = e0.elapsed_time(e1)
    launches = x.kernel_launches - launches0
    # -- timed region 2 (same loop, per-kernel events): duration of the dominant kernel (xengine_kernel = xcorr_process)
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    for k in range(steps):
        evs[k][0].record(st)
        x.process(dev_frames[k % n_distinct], st)
        evs[k][1].record(st)
        x.read(out_dev, st)
    barrier()
    kern_ms = [a.elapsed_time(b) for a, b in evs]
    clocks = sampler.stop()

    total_ms = replicas.max_over_ranks(total_ms, dist, "cuda")
    ms_per_step = total_ms / steps
    bits_per_frame = 8.0 * cfg.frame_bytes
    value = world * bits_per_frame / (ms_per_step * 1e-3) / 1e9
    cmac_per_s = world * cfg.cmacs_per_frame / (ms_per_step * 1e-3)

    # ---- roofline of the dominant kernel (tensor-bound: a dense int8 contraction)
    k_ms = statistics.mean(kern_ms)
    alg_ops = 8.0 * cfg.cmacs_per_frame              # 4 real MACs = 8 int8 ops per complex MAC, useful pairs i<=j only
    achieved = alg_ops / (k_ms * 1e-3) / 1e12
    # int8 = 2 x bf16 (nominal ratio 4.5 : 2.25) x the measured bf16 figure.  The burst figure is used whatever the length
    # of the timed region (the larger denominator, so the smaller fraction); the fraction of the sustained figure is
    # reported beside it because a default run (2000 back-to-back steps) is long enough to be power-capped.
    peak = 2.0 * peaks["bf16_burst"]
    peak_sustained = 2.0 * peaks["bf16_sustained"] if peaks.get("bf16_sustained") else None
    roofline = {
        "bound": "tensor", "kernel": "xengine_kernel (xcorr_process)", "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
        "frac": achieved / peak, "traffic": NCU_TRAFFIC_BYTES.get(cfg.name),
        "peak_source": f"2 x bf16_tflops (burst) of MEASURED_PEAKS.json [{peaks['source']}]; int8:bf16 nominal ratio 4.5:2.25",
        "kernel_ms": k_ms, "kernel_ms_min": min(kern_ms), "algorithmic_ops_per_launch": alg_ops,
        "frac_of_nominal_4500": achieved / NOMINAL_INT8_TOPS,
        "frac_of_sustained_peak": (achieved / peak_sustained) if peak_sustained else None, "peak_sustained": peak_sustained,
        "hbm_gbs_staging": cfg.frame_bytes / (k_ms * 1e-3) / 1e9, "hbm_peak_gbs": peaks["hbm_gbs"],
    }

    # context for the denominator: the library's own int8 GEMM on this box in this run (cuBLAS through torch._int_mm,
    # 8192^3, best of 10 after 3 warm-ups).  Not used for `frac`; shows where a plain int8 contraction lands on this part.
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
            nb = -(-cfg.n_inputs // 256)                       # 256 x 256 super-tiles: 3 MMAs on the diagonal, 4 above it
            issued_over_useful = (3 * nb + 4 * nb * (nb - 1) // 2) * 65536 / (4.0 * cfg.n_pairs)
            roofline["issued_over_useful"] = issued_over_useful
            roofline["issued_int8_tops"] = achieved * issued_over_useful
            del ga, gb
        except Exception as e:  # the probe is context only
            roofline["cublas_int8_gemm_8192_tops_burst"] = None
            roofline["int8_probe_error"] = str(e)[:120]

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

    # ---- the rows SURVEY.md 8(f) marks "next", same frame shape, timed one by one with CUDA events (not part of `value`)
    next_rows = None
    if rank == 0 and world == 1 and not args.no_next_rows and cfg.n_freq % wl.PACKET_F == 0 and cfg.n_time % wl.PACKET_T == 0:
        next_rows = measure_next_rows(cfg, x, xb, torch, st, host_frames[0], peaks)

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = oracle_sample(cfg)
        cpu = {k: cpu[k] for k in ("value", "unit", "cores", "kind", "sample", "cmac_per_s")}

    if rank == 0:
        line = {
            "metric": "xengine_input_gbps", "value": value, "unit": "Gb/s", "n_gpus": world, "steps": steps, "warmup": warm,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int8",
            "data": "synthetic",
            "config": {"workload": cfg.name, "n_inputs": cfg.n_inputs, "n_freq": cfg.n_freq, "t_per_frame": cfg.n_time,
                       "frame_bytes": cfg.frame_bytes, "step": "xcorr_process + xcorr_read (one integration per frame)", "options": "xcorr_promise_complete_frames(1)",
                       "l2": f"inputs larger than L2: {n_distinct} distinct {cfg.frame_bytes >> 20} MiB frames alternate",
                       "parallelism": "replicas only" if world > 1 else "1 GPU", "note": cfg.note},
            "cmac_per_s": cmac_per_s,
            "pct_int8_peak_nominal": 100.0 * 8.0 * cmac_per_s / world / (NOMINAL_INT8_TOPS * 1e12),
            "pct_int8_peak_measured": 100.0 * 8.0 * cmac_per_s / world / (peak * 1e12),
            "paper_context": "51.2 Gb/s per 3-GPU server, 819.2 Gb/s over 16 servers (PAPER.md Table I; other hardware)",
            "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "next_rows": next_rows, "gpu_launches": int(launches), "clocks": clocks,
        }
        print(json.dumps(line), flush=True)
    x.close()
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
