#!/usr/bin/env python
"""bench.py -- 1080p chunk-decode throughput (BASELINE.json metric) through the C ABI, with roofline and CPU baseline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl ours|reference]

A "step" is one ufnvc_chunk_decode call: the whole hot path A1..A9 over one synthetic chunk batch of
BASELINE.json configs[2] (1080p, T = 8; "config 3" in SURVEY.md's 1-based numbering).  Prints ONE JSON line.
Multi-GPU = independent replicas: every rank decodes its own chunks, no collective on the
data path; the only collectives are the timing barrier and the max-over-ranks of the elapsed time.
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

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "1080p decoded frames/s per B200 (T=8 chunks)"
CPU_SAMPLE_HW = (272, 480)        # bounded CPU sample: same layer plan on a 272x480 crop (~1/16 of 1080p)


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm=d["hbm_gbs"], tensor_burst=d["bf16_tflops"], tensor_sustained=d["bf16_tflops_sustained"], src="measured")
    return dict(hbm=6650.0, tensor_burst=1590.0, tensor_sustained=1400.0, src="fallback")


class ClockSampler:
    """nvidia-smi clocks + throttle reasons sampled DURING the timed region (B200_PROFILING.md clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "20"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def __exit__(self, *a):
        if self.proc:
            self.proc.terminate()
            self.th.join(timeout=2)

    def mark(self):
        """Index of the next sample: bench marks the start and the end of the timed region with it."""
        return len(self.rows)

    def summary(self, i0=0, i1=None):
        rows = self.rows[i0:i1] or self.rows          # samples taken DURING the timed region (all, if it was too short)
        sm = [float(r[0]) for r in rows if len(r) >= 7 and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in rows if len(r) >= 7 and r[1].replace(".", "").isdigit()]
        reasons = set()
        for r in rows:
            if len(r) >= 7:
                for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(name)
        return dict(sm_mhz=statistics.median(sm) if sm else None, sm_max_mhz=max(mx) if mx else None,
                    reasons=sorted(reasons), samples=len(sm))


def cpu_oracle_time(cfg_full, steps=1):
    """Time the oracle AS IT STANDS on a bounded sample; return (1080p-equivalent frames/s, description, cores)."""
    import oracle
    from paper_2606_04410_b200 import synth
    cfg = synth.crop_config(cfg_full, *CPU_SAMPLE_HW)
    orc = oracle.Oracle("f64")
    wts, z, u16 = synth.make_weights(cfg), synth.make_z(cfg), synth.make_uniform16(cfg)
    st = oracle.make_stream(orc, cfg, wts, z[0], u16[0])
    ts = []
    for _ in range(steps):
        t0 = time.perf_counter()
        out = oracle.chunk_decode(orc, cfg, wts, z[0], st["bits"], st["sub_off"])
        ts.append(time.perf_counter() - t0)
        assert out["status"] == 0
    scale = (cfg.height * cfg.width) / (cfg_full.height * cfg_full.width)
    fps = cfg.T / statistics.mean(ts) * scale
    desc = (f"oracle (fp64, C+OpenMP) full chunk decode of the {cfg_full.name} layer plan on a {cfg.width}x{cfg.height} crop, "
            f"T={cfg.T}; frames/s scaled by the pixel ratio {scale:.4f} to {cfg_full.width}x{cfg_full.height}")
    return fps, desc, orc.num_threads(), statistics.mean(ts)


def run_reference(args):
    """--impl reference: for this tier the reference arm IS the oracle, timed on the host cores (rank 0 only)."""
    from paper_2606_04410_b200 import synth
    if int(os.environ.get("RANK", "0")) != 0:
        return
    cfg = synth.CONFIGS[args.config] if args.mu_steps == 1 else synth.progressive_config(synth.CONFIGS[args.config])
    ts_fps = []
    for _ in range(args.warmup if args.warmup < 2 else 1):
        cpu_oracle_time(cfg)
    fps, desc, cores, sec = cpu_oracle_time(cfg, steps=max(1, args.steps))
    line = dict(impl="reference", metric=METRIC, value=fps, unit="frames/s", n_gpus=args.gpus, steps=args.steps, warmup=args.warmup,
                ms_per_step=sec * 1e3, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64", data="synthetic",
                config=dict(workload=cfg.name, sample=desc),
                cpu_baseline=dict(value=fps, unit="frames/s", cores=cores, kind="oracle", sample=desc),
                e2e=dict(value=fps, unit="frames/s", h2d_bytes_per_step=0, d2h_bytes_per_step=0))
    print(json.dumps(line))


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2606_04410_b200 import binding, replicas, synth

    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    peaks = load_peaks()

    cfg = synth.CONFIGS[args.config] if args.mu_steps == 1 else synth.progressive_config(synth.CONFIGS[args.config])
    n = cfg.n_chunks
    dec = binding.ChunkDecoder(cfg, device=local)
    dec.load_weights(synth.make_weights(cfg))

    # ---- synthetic inputs, built with the library's own encoder-side fixtures (no oracle on this path) ----
    z_host = synth.make_z(cfg)
    u16 = synth.make_uniform16(cfg)
    z = torch.from_numpy(z_host).to(dev)
    _, _, idx_dev = dec.entropy_params(z)
    idx_host = idx_dev.cpu().numpy()
    parts = []
    for c in range(n):
        sym = dec.symbols_from_uniform(idx_host[c], u16[c])
        parts.append(dec.encode_chunk(idx_host[c], sym))
    bits_host, off_host = binding.concat_streams(parts)
    off_host = off_host.astype(np.int64).astype(np.int32)
    bits, off = torch.from_numpy(bits_host).to(dev), torch.from_numpy(off_host).to(dev)
    frames = dec.new_frames(n)
    stream = torch.cuda.Stream(device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)      # > 126 MB L2

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- device-resident timing: per-step event pairs on the launching stream, L2 flushed between steps ----
    step_ms, stage_us = [], []
    with ClockSampler(local) as clocks:               # started before the warm-up: nvidia-smi takes ~0.2 s to print its first line
        time.sleep(0.3)
        with torch.cuda.stream(stream):
            for _ in range(max(3, args.warmup)):
                dec.chunk_decode(z, bits, off, frames=frames, stream=stream)
        barrier()
        assert dec.get_status() == 0, "bit-stream status"
        i0 = clocks.mark()
        t_wall = time.perf_counter()
        with torch.cuda.stream(stream):
            for _ in range(args.steps):
                flush.zero_()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                stage_us.append(dec.chunk_decode_profiled(z, bits, off, frames, stream=stream))   # syncs the stream at its end
                e1.record(stream)
                e1.synchronize()
                step_ms.append(e0.elapsed_time(e1))
        barrier()
        t_wall = time.perf_counter() - t_wall
        i1 = clocks.mark()
    total_ms = sum(step_ms)
    # A6 / A7 split: a few extra steps AFTER the timed region (two more events per trunk block would cost launch gaps inside it)
    detail_us = []
    with torch.cuda.stream(stream):
        for _ in range(5):
            flush.zero_()
            detail_us.append(dec.chunk_decode_profiled(z, bits, off, frames, stream=stream, detail=True))
    # ---- NEXT-3 (R22): the same chunks from BYTES ONLY (z entropy-decoded on the device first), 10 extra steps ----
    zparts = [dec.encode_z(z_host[c]) for c in range(n)]
    all_bits, all_off = binding.concat_streams([binding.pack_chunk_bytes(zb, zo, pb, po) for (zb, zo), (pb, po) in zip(zparts, parts)])
    ab, ao = torch.from_numpy(all_bits).to(dev), torch.from_numpy(all_off.astype(np.int64).astype(np.int32)).to(dev)
    bytes_ms = []
    with torch.cuda.stream(stream):
        dec.chunk_decode_bytes(ab, ao, n_chunks=n, frames=frames, stream=stream)
        stream.synchronize()
        assert dec.get_status() == 0, "bit-stream status (bytes-only call)"
        bytes_launches = dec.launches_per_call(n)
        for _ in range(10):
            flush.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            dec.chunk_decode_bytes(ab, ao, n_chunks=n, frames=frames, stream=stream)
            e1.record(stream)
            e1.synchronize()
            bytes_ms.append(e0.elapsed_time(e1))
    bytes_in = dict(value=n * cfg.T / (statistics.mean(bytes_ms) / 1e3), unit="frames/s (this rank)", ms_per_step=statistics.mean(bytes_ms),
                    steps=10, z_stream_bytes=int(sum(int(zo[-1]) for _, zo in zparts)), y_stream_bytes=int(sum(int(po[-1]) for _, po in parts)),
                    launches_per_call=bytes_launches, call="ufnvc_chunk_decode_bytes")
    total_ms = replicas.max_over_ranks(total_ms, dev)
    frames_per_step = n * cfg.T
    value = world * frames_per_step * args.steps / (total_ms / 1e3)

    # ---- end to end through the public API with HOST buffers: H2D of z/bits/offsets + decode + D2H of the frames ----
    z_pin, bits_pin, off_pin = (torch.from_numpy(a).pin_memory() for a in (z_host, bits_host, off_host))
    # Two sets of buffers and a copy stream: the D2H of chunk i (199 MB of fp32 frames at 1080p, the dominant cost) overlaps
    # the decode of chunk i+1, as a streaming player would run it.  Every step still pays its own H2D and D2H.
    e2e_steps = max(4, min(args.steps, 20))
    copy_stream = torch.cuda.Stream(device=dev)
    bufs = []
    for _ in range(2):
        bufs.append(dict(frames=dec.new_frames(n), out=torch.empty(frames.shape, dtype=torch.float32).pin_memory(),
                         z=torch.empty_like(z), bits=torch.empty_like(bits), off=torch.empty_like(off),
                         decoded=torch.cuda.Event(), copied=torch.cuda.Event()))

    def e2e_run(k):
        for i in range(k):
            b = bufs[i & 1]
            with torch.cuda.stream(stream):
                stream.wait_event(b["copied"])                       # frames buffer of step i-2 has left the device
                b["z"].copy_(z_pin, non_blocking=True)
                b["bits"].copy_(bits_pin, non_blocking=True)
                b["off"].copy_(off_pin, non_blocking=True)
                dec.chunk_decode(b["z"], b["bits"], b["off"], frames=b["frames"], stream=stream)
                b["decoded"].record(stream)
            with torch.cuda.stream(copy_stream):
                copy_stream.wait_event(b["decoded"])
                b["out"].copy_(b["frames"], non_blocking=True)
                b["copied"].record(copy_stream)
        stream.synchronize()
        copy_stream.synchronize()

    e2e_run(2)
    barrier()
    t0 = time.perf_counter()
    e2e_run(e2e_steps)
    barrier()
    e2e_s = time.perf_counter() - t0
    e2e_s = replicas.max_over_ranks(e2e_s, dev)
    e2e_val = world * frames_per_step * e2e_steps / e2e_s
    assert dec.get_status() == 0 and float(bufs[0]["out"].max()) <= 1.0
    out_pin = bufs[0]["out"]
    h2d = z_pin.numel() * 2 + bits_pin.numel() + off_pin.numel() * 4
    d2h = out_pin.numel() * 4

    if rank != 0:
        return
    # ---- roofline of the dominant kernel: the grouped 3x3 implicit-GEMM conv of A8 (73 % of the chunk's MACs) ----
    P = dec.h * dec.w
    macs_a8 = sum(n * cfg.T * (P << (2 * s)) * 9 * cfg.dec_channels[s] * 4 * cfg.dec_channels[s + 1] for s in range(3))
    a8_us = statistics.mean(s["A8"] for s in stage_us)
    achieved = 2.0 * macs_a8 / (a8_us * 1e-6) / 1e12
    peak = peaks["tensor_sustained"]
    stage_mean = {k: statistics.mean(s[k] for s in stage_us) for k in stage_us[0]}
    stage_mean["A6"] = statistics.mean(s["A6"] for s in detail_us)
    prof = os.path.join(ROOT, "profiles", "r01_traffic.json.txt")
    traffic = json.load(open(prof)).get("a8_dram_bytes_per_launch") if os.path.exists(prof) else None
    roofline = dict(bound="tensor", achieved=achieved, peak=peak, unit="TFLOP/s", frac=achieved / peak, traffic=traffic,
                    kernel="A8 frame-decoder stages 1-3 (3 launches of the implicit-GEMM conv kernel)",
                    peak_source=f"{peaks['src']} bf16 sustained; burst {peaks['tensor_burst']}", stage_us=stage_mean,
                    flops_per_step=2.0 * macs_a8)
    # ---- the other stages against the roofline that bounds each (algorithmic bytes / flops per chunk) ----
    Ct, Ce, B, T = cfg.c_trunk, cfg.c_trunk * cfg.trunk_expand, cfg.n_trunk_blocks, cfg.T
    act = n * T * P * Ct * 2                                                   # one trunk activation tensor, bf16
    nsym = n * cfg.n_symbols
    s3 = n * T * (P << 6) * cfg.dec_channels[3] * 2                            # A9 input, bf16
    out_b = n * T * 3 * cfg.height * cfg.width * 4                             # fp32 frames
    def hbm(name, nbytes, us):
        a = nbytes / (us * 1e-6) / 1e9
        return dict(stage=name, bound="hbm", achieved=a, peak=peaks["hbm"], unit="GB/s", frac=a / peaks["hbm"], bytes=nbytes, us=us)
    def tens(name, flops, us):
        a = flops / (us * 1e-6) / 1e12
        return dict(stage=name, bound="tensor", achieved=a, peak=peak, unit="TFLOP/s", frac=a / peak, flops=flops, us=us)
    a7_us = stage_mean["A6+A7"] - stage_mean["A6"]
    a34 = "A3+A4 rANS decode + dequant (serial-latency bound, reported against HBM as asked)"
    if cfg.mu_steps == 4:
        a34 = "A3+A4 rANS decode + four-step progressive means (prep + 3 tensor-core convs, R21); bytes are the rANS stage's"
    stages = [hbm(a34, nsym * 7 + int(nsym * 0.35), stage_mean["A3+A4"]),
              hbm("A5 cross-frame unfold", n * P * cfg.c_y * 2 + act, stage_mean["A5"])]
    if B:
        stages += [hbm("A6 depthwise 3x3 (all trunk blocks)", B * 2 * act, stage_mean["A6"]),
                   tens("A7 fused trunk MLP (all trunk blocks)", B * 2.0 * n * T * P * 2 * Ct * Ce, a7_us)]
    stages += [tens("A8 frame decoders, stages 1-3", 2.0 * macs_a8, a8_us),
               hbm("A9 last stage + output", s3 + out_b, stage_mean["A9"])]
    roofline["stages"] = stages
    fps_cpu, desc, cores, _ = cpu_oracle_time(cfg)
    line = dict(metric=METRIC, value=value, unit="frames/s", n_gpus=world, steps=args.steps, warmup=max(3, args.warmup),
                ms_per_step=total_ms / args.steps, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="bf16",
                data="synthetic", chunks_per_s=value / cfg.T,
                config=dict(workload=cfg.name, T=cfg.T, frame=f"{cfg.width}x{cfg.height}", chunks_per_step=n,
                            l2="flushed between timed steps (256 MiB memset, untimed)", parallelism=f"replicas x{world}",
                            gmac_per_chunk=cfg.macs_per_chunk() / 1e9),
                clocks=clocks.summary(i0, i1), gpu_launches=dec.launches_per_call(n) * args.steps,
                e2e=dict(value=e2e_val, unit="frames/s", h2d_bytes_per_step=h2d, d2h_bytes_per_step=d2h, steps=e2e_steps,
                         overlap="D2H of step i on a copy stream overlaps the decode of step i+1 (two buffer sets)"),
                roofline=roofline, bytes_in=bytes_in,
                cpu_baseline=dict(value=fps_cpu, unit="frames/s", cores=cores, kind="oracle", sample=desc),
                wall_s_timed_region=t_wall)
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=3, help="SURVEY.md config number 1..5 (3 = 1080p headline)")
    ap.add_argument("--mu-steps", type=int, default=1, choices=[1, 4],
                    help="4: the same workload with the four-step progressive means switched on (SURVEY.md 8f NEXT-1, DESIGN.md R21)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
