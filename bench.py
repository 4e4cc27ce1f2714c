#!/usr/bin/env python
"""bench.py -- 1080p chunk-decode throughput (BASELINE.json metric) through the C ABI, with roofline and CPU baseline.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl ours|reference]

A "step" is one ufnvc_chunk_decode call: the whole hot path A1..A9 over one synthetic chunk batch of
BASELINE.json configs[2] (1080p, T = 8; "config 3" in SURVEY.md's 1-based numbering).  Prints ONE JSON line.
Multi-GPU = independent replicas: every rank decodes its own chunks, no collective on the
data path; the only collectives are the timing barrier and the max-over-ranks of the elapsed time.  `--gpus N` without
a launcher spawns the N ranks itself; under torch.distributed.run it uses the ranks it is given.
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


def oracle_inputs(cfg):
    import oracle
    from paper_2606_04410_b200 import synth
    orc = oracle.Oracle("f64")
    wts, z, u16 = synth.make_weights(cfg), synth.make_z(cfg), synth.make_uniform16(cfg)
    st = oracle.make_stream(orc, cfg, wts, z[0], u16[0])
    return wts, z, st


def cpu_oracle_full(cfg, real="f64", inputs=None):
    """The oracle AS IT STANDS on the WHOLE workload: one full-size chunk decode (O1..O9) of `cfg` on the host cores.
    Returns (frames/s, seconds, cores, description)."""
    import oracle
    wts, z, st = inputs or oracle_inputs(cfg)
    orc = oracle.Oracle(real)
    t0 = time.perf_counter()
    out = oracle.chunk_decode(orc, cfg, wts, z[0], st["bits"], st["sub_off"], idx_override=st["idx"])
    sec = time.perf_counter() - t0
    assert out["status"] == 0 and float(out["frames"].min()) >= 0.0
    desc = (f"oracle ({real}, plain C + OpenMP) full chunk decode O1..O9 of {cfg.name} at full size "
            f"({cfg.width}x{cfg.height}, T={cfg.T}), one run, same seeded inputs as the GPU arm")
    return cfg.T / sec, sec, orc.num_threads(), desc


def run_reference(args):
    """--impl reference: for this tier the reference arm IS the oracle, timed on the host cores (rank 0 only; the other
    ranks exit 0 without work).  One step = ONE FRAME of the full-size workload: the chunk's shared front (O1..O6:
    hyper-decoder, rANS decode, dequantisation, cross-frame unfold; ~2 % of the chunk's MACs) plus the trunk and the
    frame-specific decoder of frame (step mod T) at full resolution -- a bounded sample, so that --steps 20 --warmup 5 ends
    in minutes; frames/s = 1 / mean step time (slightly pessimistic: the shared front is recomputed every step)."""
    import oracle
    from paper_2606_04410_b200 import synth
    if int(os.environ.get("RANK", "0")) != 0:
        return
    cfg = synth.CONFIGS[args.config] if args.mu_steps == 1 else synth.progressive_config(synth.CONFIGS[args.config])
    wts, z, st = oracle_inputs(cfg)
    orc = oracle.Oracle("f64")

    def one_frame(t):
        t0 = time.perf_counter()
        mu, u, idx = oracle.entropy_params(orc, cfg, wts, z[0])
        cdf = orc.build_cdf(cfg.n_buckets, cfg.scale_min, cfg.scale_max)
        sym, status = oracle.decode_symbols(orc, cfg, cdf, idx, st["bits"], st["sub_off"])
        if cfg.mu_steps == 4:
            yhat, _ = oracle.progressive_means(orc, cfg, wts, mu, sym)
        else:
            yhat = sym.astype(np.float64) + mu
        frames, _ = oracle.synthesis(orc, cfg, wts, yhat, only_frames=(t,))
        sec = time.perf_counter() - t0
        assert status == 0 and 0.0 <= float(frames[t].min())
        return sec

    for i in range(min(args.warmup, 1)):            # one untimed step warms the page cache and the OpenMP pool
        one_frame(0)
    ts = [one_frame(i % cfg.T) for i in range(max(1, args.steps))]
    sec = statistics.mean(ts)
    fps = 1.0 / sec
    desc = (f"oracle (f64, plain C + OpenMP): per step the shared front O1..O6 plus trunk + decoder of ONE frame of {cfg.name} at "
            f"full size ({cfg.width}x{cfg.height}); {len(ts)} steps; frames/s = 1 / mean step time")
    line = dict(impl="reference", metric=METRIC, value=fps, unit="frames/s", n_gpus=args.gpus, steps=args.steps, warmup=args.warmup,
                ms_per_step=sec * 1e3, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64", data="synthetic",
                config=dict(workload=cfg.name, T=cfg.T, frame=f"{cfg.width}x{cfg.height}", sample=desc),
                cpu_baseline=dict(value=fps, unit="frames/s", cores=orc.num_threads(), kind="oracle", sample=desc),
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

    # ---- synthetic inputs, built with the library's own encoder-side fixtures (no oracle on this path).  Replicas: rank r
    # decodes ITS OWN chunks (replicas.shard_chunks deals the job's world * n chunks round-robin; every rank draws its
    # shard from the same seeded generator, so the job is reproducible at any N) ----
    z_host = synth.make_z(cfg)
    u16 = synth.make_uniform16(cfg)
    mine = replicas.shard_chunks(world * n, rank, world)
    assert len(mine) == n
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

    # ---- device-resident timing of the call the metric names: plain ufnvc_chunk_decode, one CUDA-event pair per step on the
    # launching stream, L2 flushed (untimed) between steps, no host synchronisation inside the timed region ----
    with ClockSampler(local) as clocks:               # started before the warm-up: nvidia-smi takes ~0.2 s to print its first line
        time.sleep(0.3)
        with torch.cuda.stream(stream):
            for _ in range(max(3, args.warmup)):
                dec.chunk_decode(z, bits, off, frames=frames, stream=stream)
        barrier()
        assert dec.get_status() == 0, "bit-stream status"
        launches_per_call = dec.launches_per_call(n)
        i0 = clocks.mark()
        t_wall = time.perf_counter()
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
        with torch.cuda.stream(stream):
            for e0, e1 in ev:
                flush.zero_()
                e0.record(stream)
                dec.chunk_decode(z, bits, off, frames=frames, stream=stream)
                e1.record(stream)
        barrier()
        t_wall = time.perf_counter() - t_wall
        i1 = clocks.mark()
    step_ms = [e0.elapsed_time(e1) for e0, e1 in ev]
    total_ms = sum(step_ms)
    assert dec.get_status() == 0
    # ---- per-stage split: SEPARATE profiled steps (ufnvc_chunk_decode_profiled records an event after every stage and
    # synchronises; its steps are not the timed ones).  detail=True also brackets every depthwise launch. ----
    prof_steps = max(5, min(args.steps, 20))
    stage_us, detail_us = [], []
    with torch.cuda.stream(stream):
        for _ in range(prof_steps):
            flush.zero_()
            stage_us.append(dec.chunk_decode_profiled(z, bits, off, frames, stream=stream))
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
    # ---- widened rows of SURVEY.md 8f, 10 extra steps each on handles of their own (rank 0's figures are printed):
    # NEXT-2a temporal context with the paper's HT-S count of 11 context DC blocks (R23), NEXT-4 chunk encode with 6 (R24) ----
    def timed(fn, reps=10, before=None):
        ms = []
        with torch.cuda.stream(stream):
            for _ in range(reps + 2):
                if before:
                    before()
                flush.zero_()
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                fn()
                e1.record(stream)
                e1.synchronize()
                ms.append(e0.elapsed_time(e1))
        return statistics.mean(ms[2:])
    extra = {}
    if args.config in (2, 3) and args.mu_steps == 1:
        ccfg = synth.context_config(cfg, 11)
        cdec = binding.ChunkDecoder(ccfg, device=local)
        cdec.load_weights(synth.make_weights(ccfg))
        cdec.reset_context(n, stream=stream)
        _, _, cidx = cdec.entropy_params(z, stream=stream)
        stream.synchronize()
        cparts = [cdec.encode_chunk(cidx[c].cpu().numpy(), cdec.symbols_from_uniform(cidx[c].cpu().numpy(), u16[c])) for c in range(n)]
        cb, co = binding.concat_streams(cparts)
        cb, co = torch.from_numpy(cb).to(dev), torch.from_numpy(co.astype(np.int64).astype(np.int32)).to(dev)
        ms = timed(lambda: cdec.chunk_decode(z, cb, co, frames=frames, stream=stream), before=lambda: cdec.reset_context(n, stream=stream))
        assert cdec.get_status() == 0, "bit-stream status (context leg)"
        prof = cdec.chunk_decode_profiled(z, cb, co, frames, stream=stream)
        extra["context"] = dict(value=n * cfg.T / (ms / 1e3), unit="frames/s (this rank)", ms_per_step=ms, n_ctx_blocks=11,
                                context_generation_us=prof["ctx"], launches_per_call=cdec.launches_per_call(n), workload=ccfg.name,
                                call="ufnvc_chunk_decode on a handle with n_ctx_blocks = 11 (state reset, untimed, before every step)")
        cdec.destroy()
        ecfg = synth.encoder_config(cfg, 6)
        edec = binding.ChunkDecoder(ecfg, device=local)
        edec.load_weights(synth.make_weights(ecfg))
        fr_in = torch.from_numpy(synth.make_frames(ecfg)).to(dev)
        res = {}
        ms = timed(lambda: res.update(edec.chunk_encode(fr_in, stream=stream)))
        assert edec.get_status() == 0, "status (encode leg)"
        nbytes = int(res["sub_off"][-1].item())
        back = edec.chunk_decode(res["z"], res["bits"][:nbytes], res["sub_off"], frames=frames, stream=stream)
        stream.synchronize()
        assert edec.get_status() == 0, "the decoder rejects the encoder's stream"
        mse = float(((back - fr_in) ** 2).mean())
        extra["encode"] = dict(value=n * cfg.T / (ms / 1e3), unit="encoded frames/s (this rank)", ms_per_step=ms, n_enc_blocks=6,
                               stream_bytes=nbytes, launches_per_call=edec.launches_per_call(n), workload=ecfg.name,
                               call="ufnvc_chunk_encode (frames resident on the device -> bytes on the device)",
                               note="random-init weights: the round trip decodes cleanly (status 0) but reconstructs noise, mse %.3f" % mse)
        edec.destroy()
    frames_per_step = n * cfg.T
    value = replicas.job_throughput(frames_per_step, args.steps, total_ms, dev)       # all ranks' frames / max-over-ranks time
    total_ms = replicas.max_over_ranks(total_ms, dev)

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
        if world > 1:
            dist.destroy_process_group()
        return
    # ---- roofline of the dominant kernel: the grouped 3x3 implicit-GEMM conv of A8 (73 % of the chunk's MACs) ----
    P = dec.h * dec.w
    macs_a8 = sum(n * cfg.T * (P << (2 * s)) * 9 * cfg.dec_channels[s] * 4 * cfg.dec_channels[s + 1] for s in range(3))
    stage_mean = {k: statistics.mean(s[k] for s in stage_us) for k in stage_us[0] if k not in ("A6", "ctx")}
    stage_mean["A6 (serialised by its own events)"] = statistics.mean(s["A6"] for s in detail_us)
    a8_us = stage_mean["A8"]
    achieved = 2.0 * macs_a8 / (a8_us * 1e-6) / 1e12
    clk = clocks.summary(i0, i1)
    # which measured peak applies: the timed region is a sequence of ~2 ms bursts separated by an L2 flush; when the sampled
    # SM clock sits at its maximum the burst peak is the ceiling, under a sustained-load clock the sustained one is
    at_max = bool(clk["sm_mhz"] and clk["sm_max_mhz"] and clk["sm_mhz"] >= 0.95 * clk["sm_max_mhz"])
    peak = peaks["tensor_burst"] if at_max else peaks["tensor_sustained"]
    tpath = os.path.join(ROOT, "profiles", "r02_traffic.json.txt")
    tinfo = json.load(open(tpath)) if os.path.exists(tpath) else {}
    roofline = dict(bound="tensor", achieved=achieved, peak=peak, unit="TFLOP/s", frac=achieved / peak,
                    frac_burst=achieved / peaks["tensor_burst"], frac_sustained=achieved / peaks["tensor_sustained"],
                    peak_used="burst" if at_max else "sustained",
                    peak_source=f"{peaks['src']}: bf16 burst {peaks['tensor_burst']}, sustained {peaks['tensor_sustained']} TFLOP/s, HBM {peaks['hbm']} GB/s",
                    traffic=tinfo.get("a8_dram_bytes_per_step"), traffic_source=tinfo.get("source"),
                    kernel="A8 frame-decoder stages 1-3 (3 launches of conv_halo_pair_kernel<EPI_PS2>)",
                    flops_per_step=2.0 * macs_a8, us=a8_us,
                    stage_us=stage_mean, stage_us_source=f"{prof_steps} separate ufnvc_chunk_decode_profiled steps (not the timed ones)")
    # ---- the other stages against the roofline that bounds each (algorithmic bytes / flops per chunk) ----
    Ct, Ce, B, T = cfg.c_trunk, cfg.c_trunk * cfg.trunk_expand, cfg.n_trunk_blocks, cfg.T
    act = n * T * P * Ct * 2                                                   # one trunk activation tensor, bf16
    nsym = n * cfg.n_symbols
    s3 = n * T * (P << 6) * cfg.dec_channels[3] * 2                            # A9 input, bf16
    out_b = n * T * 3 * cfg.height * cfg.width * 4                             # fp32 frames
    def hbm(name, nbytes, us):
        a = nbytes / (us * 1e-6) / 1e9
        return dict(stage=name, bound="hbm", achieved=a, peak=peaks["hbm"], unit="GB/s", frac=a / peaks["hbm"], bytes=nbytes, us=us)
    def tens(name, flops, us, **kw):
        a = flops / (us * 1e-6) / 1e12
        return dict(stage=name, bound="tensor", achieved=a, peak=peak, unit="TFLOP/s", frac=a / peak, flops=flops, us=us, **kw)
    a34 = "A3+A4 rANS decode + dequant (serial-latency bound, reported against HBM as asked)"
    if cfg.mu_steps == 4:
        a34 = "A3+A4 rANS decode + four-step progressive means (prep + 3 tensor-core convs, R21); bytes are the rANS stage's"
    stages = [hbm(a34, nsym * 7 + int(nsym * 0.35), stage_mean["A3+A4"]),
              hbm("A5 cross-frame unfold", n * P * cfg.c_y * 2 + act, stage_mean["A5"])]
    if B:
        # A6 and A7 overlap (the depthwise tiles of block k+1 run under the MLP kernel's last round), so they are ONE stage:
        # the MLP's flops over the joint time; the depthwise bytes ride along
        stages += [tens("A6+A7 trunk (depthwise + fused MLP, all blocks, timed as one region)", B * 2.0 * n * T * P * 2 * Ct * Ce,
                        stage_mean["A6+A7"], depthwise_bytes=B * 2 * act),
                   hbm("A6 depthwise alone (its launches bracketed by events, which serialises them: an upper bound of its cost)",
                       B * 2 * act, stage_mean["A6 (serialised by its own events)"])]
    stages += [tens("A8 frame decoders, stages 1-3", 2.0 * macs_a8, a8_us),
               hbm("A9 last stage + output", s3 + out_b, stage_mean["A9"])]
    roofline["stages"] = stages
    if args.skip_cpu_baseline:                      # profiling runs (ncu replays): the CPU leg only costs time there
        fps_cpu = sec_cpu = fps32 = sec32 = None
        cores, desc, desc32 = 0, "skipped (--skip-cpu-baseline)", "skipped"
    else:
        inputs = oracle_inputs(cfg)
        fps_cpu, sec_cpu, cores, desc = cpu_oracle_full(cfg, "f64", inputs)
        fps32, sec32, _, desc32 = cpu_oracle_full(cfg, "f32", inputs)
    line = dict(metric=METRIC, value=value, unit="frames/s", n_gpus=world, steps=args.steps, warmup=max(3, args.warmup),
                ms_per_step=total_ms / args.steps, higher_is_better=True, scaling="weak", vs_baseline=None, dtype="bf16",
                data="synthetic", chunks_per_s=value / cfg.T, timed_call="ufnvc_chunk_decode",
                config=dict(workload=cfg.name, T=cfg.T, frame=f"{cfg.width}x{cfg.height}", chunks_per_step=n,
                            l2="flushed between timed steps (256 MiB memset, untimed)", parallelism=f"replicas x{world}",
                            gmac_per_chunk=cfg.macs_per_chunk() / 1e9),
                clocks=clk, gpu_launches=launches_per_call * args.steps,
                e2e=dict(value=e2e_val, unit="frames/s", h2d_bytes_per_step=h2d, d2h_bytes_per_step=d2h, steps=e2e_steps,
                         overlap="D2H of step i on a copy stream overlaps the decode of step i+1 (two buffer sets)",
                         bound="PCIe: the boundary's output is fp32 planar frames (199 MB per 1080p chunk)"),
                roofline=roofline, bytes_in=bytes_in, **extra,
                cpu_baseline=dict(value=fps_cpu, unit="frames/s", cores=cores, kind="oracle", sample=desc, seconds=sec_cpu,
                                  fp32_oracle=dict(value=fps32, seconds=sec32, sample=desc32)),
                wall_s_timed_region=t_wall)
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def spawn_ranks(args):
    """`python bench.py --gpus N` without a launcher: start N ranks of this script (one process per GPU, NCCL rendezvous on
    127.0.0.1) exactly as `torch.distributed.run --nproc-per-node N` would; rank 0 prints the JSON line."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    procs = []
    for r in range(args.gpus):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE=str(args.gpus), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, os.path.abspath(__file__)] + sys.argv[1:], env=env))
    rc = 0
    for p in procs:
        rc = p.wait() or rc
    sys.exit(rc)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=3, help="SURVEY.md config number 1..5 (3 = 1080p headline)")
    ap.add_argument("--mu-steps", type=int, default=1, choices=[1, 4],
                    help="4: the same workload with the four-step progressive means switched on (SURVEY.md 8f NEXT-1, DESIGN.md R21)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--skip-cpu-baseline", action="store_true", help="leave the oracle-on-host-cores leg out (for runs under ncu)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        spawn_ranks(args)
    else:
        if int(os.environ.get("WORLD_SIZE", "1")) != args.gpus:
            sys.exit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={os.environ.get('WORLD_SIZE', '1')}")
        run_ours(args)


if __name__ == "__main__":
    main()
