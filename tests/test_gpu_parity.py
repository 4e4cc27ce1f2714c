"""GPU-vs-oracle parity through the C ABI (run with -m gpu on the B200 box).

Tolerances (BASELINE.json north_star): symbols and CDF indices bit-exact when fed the same indices; index mismatch
rate <= 1e-5, only at bucket boundaries; mu within 1e-2 relative (|d mu| <= 1e-2 max(|mu|,1), R13), ln sigma within
1e-2; pixels <= 2e-2 max abs on [0,1] and PSNR >= 45 dB against the oracle's frames.
"""
import dataclasses
import math

import numpy as np
import pytest
import torch

from common import gpu_inputs, nhwc, oracle_case, psnr
from paper_2606_04410_b200 import synth

pytestmark = pytest.mark.gpu

PIX_TOL, PSNR_MIN, IDX_RATE = 2e-2, 45.0, 1e-5

CASES = {
    "cfg1": synth.CONFIGS[1],
    # ragged in every direction: h = 10 (3 substreams, last has 2 rows), w = 14, 160x224 frames cropped to 150x200
    "cfg2-ragged": synth.crop_config(synth.CONFIGS[2], 150, 200),
    "cfg3-crop": synth.crop_config(synth.CONFIGS[3], 272, 480),
    "cfg2": synth.CONFIGS[2],
    # four-step progressive means (NEXT-1, R21) on the same three small workloads
    "cfg1-pmu": synth.progressive_config(synth.CONFIGS[1]),
    "cfg2-ragged-pmu": synth.progressive_config(synth.crop_config(synth.CONFIGS[2], 150, 200)),
    "cfg3-crop-pmu": synth.progressive_config(synth.crop_config(synth.CONFIGS[3], 272, 480)),
}
# narrower trunks: the depthwise kernel is compiled per channel count (64 / 128 / 192 / 256); w = 13 leaves a last column group
# with one valid column, h = 10 a bottom tile with two valid rows
for _ct in (64, 128, 192):
    CASES[f"trunk{_ct}"] = dataclasses.replace(synth.crop_config(synth.CONFIGS[2], 150, 200), T=2, c_trunk=_ct, n_trunk_blocks=2,
                                               dec_channels=(_ct, 64, 64, 32, 3), name=f"cfg2-ragged-trunk{_ct}")
# config 5's layer plan (8 trunk blocks) on a crop, and the low-delay shape T = 1 ("N=1 (single-frame chunk)")
CASES["cfg5-crop"] = synth.crop_config(synth.CONFIGS[5], 272, 480)
CASES["cfg3-crop-T1"] = dataclasses.replace(synth.crop_config(synth.CONFIGS[3], 272, 480), T=1, name="cfg3-crop-T1")


def bf16_bound(want, n_roundings):
    """Bound on the error of a bf16-stored activation tensor ("Tolerances"): a bf16 store keeps 8 significant
    bits, so its relative error is uniform in +-2^-8 (2^e / |x|) <= +-2^-8, rms <= 2^-8 / sqrt 3 of the element; the
    layer gains are ~1 (R11), so after L roundings on the path the error has rms <= sqrt(L) 2^-8 / sqrt 3 * rms(x), and its
    maximum over <= 1e8 elements stays under 6 sigma of the element-wise worst case, sqrt(L) 2^-8 / sqrt 3 * max|x|.
    Returns (rms bound, max bound)."""
    rms = float(np.sqrt(np.mean(np.square(want, dtype=np.float64))))
    amp = float(np.abs(want).max())
    r = math.sqrt(n_roundings) * 2.0 ** -8 / math.sqrt(3.0)
    return r * max(rms, 1e-3), 6.0 * r * max(amp, 1.0)


@pytest.fixture(scope="module")
def decoders():
    from paper_2606_04410_b200 import binding
    cache = {}

    def get(name):
        if name not in cache:
            case = oracle_case(CASES[name])
            dec = binding.ChunkDecoder(case["cfg"])
            dec.load_weights(case["weights"])
            cache[name] = (dec, case)
        return cache[name]
    yield get
    for dec, _ in cache.values():
        dec.destroy()


def bf16_np(t):
    return t.float().cpu().numpy()


@pytest.mark.parametrize("name", ["cfg1", "cfg2-ragged", "cfg3-crop", "cfg2", "cfg1-pmu", "cfg2-ragged-pmu", "cfg3-crop-pmu",
                                  "trunk64", "trunk128", "trunk192", "cfg5-crop", "cfg3-crop-T1"])
def test_chunk_decode_matches_oracle(decoders, name):
    dec, case = decoders(name)
    cfg = case["cfg"]
    z, bits, off = gpu_inputs(case)
    out = dec.chunk_decode_ex(z, bits, off, taps=True)
    torch.cuda.synchronize()
    assert dec.get_status() == 0
    worst = dict(rms=0.0, max=0.0)
    for n, ch in enumerate(case["chunks"]):
        ref, st = ch["out"], ch["stream"]
        # A1 + A2
        idx = out["idx"][n].cpu().numpy()
        mism = idx != nhwc(ref["idx"])
        assert mism.mean() <= IDX_RATE
        if mism.any():     # only at bucket boundaries (R18)
            step = (math.log(cfg.scale_max) - math.log(cfg.scale_min)) / (cfg.n_buckets - 1)
            u = nhwc(ref["u"])[mism]
            frac = (u - math.log(cfg.scale_min)) / step
            assert np.abs(frac - np.floor(frac) - 0.5).max() < 1e-4
        mu_ref = nhwc(ref["mu"])
        assert (np.abs(out["mu"][n].cpu().numpy() - mu_ref) <= 1e-2 * np.maximum(np.abs(mu_ref), 1.0)).all()
        assert np.abs(out["lnscale"][n].cpu().numpy() - nhwc(ref["u"])).max() <= 1e-2
        # A3 + A4: integer work is bit-exact
        assert np.array_equal(out["sym"][n].cpu().numpy(), nhwc(ref["sym"]))
        # yhat = r + mu: r is bit-exact, so yhat inherits mu's tolerance (R13); the tensor-core mean is good to ~3e-5
        d_y = np.abs(out["yhat"][n].cpu().numpy() - nhwc(ref["yhat"]))
        if cfg.mu_steps == 4:
            # progressive means come from bf16 tensor-core convs over [y so far ; mu0]: the north-star bound on mu
            # applies (1e-2 relative, R13); partition 0 still carries the head's mean
            assert (d_y <= 1e-2 * np.maximum(np.abs(mu_ref), 1.0)).all(), d_y.max()
            import oracle
            part0 = nhwc(oracle.partition_index(cfg.c_y, cfg.h, cfg.w)) == 0
            assert d_y[part0].max() <= 1e-4
            print(name, "progressive: max |d yhat| =", d_y.max(), " rms =", float(np.sqrt((d_y ** 2).mean())))
        else:
            assert d_y.max() <= 1e-4
        # A5 .. A8 intermediates: bf16 storage; bound derived from the number of bf16 roundings on the path (bf16_bound):
        # y (1) + F0 (1); per trunk block: depthwise out, hidden, block out (3); one per decoder stage
        taps = ref["taps"]
        wf = 2 if cfg.weight_dtype == 0 else 1        # fp32 blobs: the weights are rounded to bf16 at load too (R19)
        L0 = wf * (2 + (1 if cfg.mu_steps == 4 else 0))
        Lt = L0 + wf * 3 * cfg.n_trunk_blocks
        for t in range(cfg.T):
            for got, want, L in ([(out["f0"][n, t], taps["F0"][t], L0), (out["trunk"][n, t], taps["trunk"][t], Lt)] +
                                 [(out["stage"][s][n, t], taps["stage"][t][s], Lt + wf * (s + 1)) for s in range(3)]):
                w = nhwc(want)
                err = bf16_np(got) - w
                rms_b, max_b = bf16_bound(w, L)
                rms_e, max_e = float(np.sqrt(np.mean(err ** 2))), float(np.abs(err).max())
                worst["rms"] = max(worst["rms"], rms_e / rms_b)
                worst["max"] = max(worst["max"], max_e / max_b)
                assert rms_e <= rms_b and max_e <= max_b, (name, n, t, L, rms_e, rms_b, max_e, max_b)
        # A9: pixels
        f = out["frames"][n].cpu().numpy()
        assert f.shape == ref["frames"].shape and f.min() >= 0.0 and f.max() <= 1.0
        assert np.abs(f - ref["frames"]).max() <= PIX_TOL
        assert psnr(f, ref["frames"]) >= PSNR_MIN
    print(name, "intermediates: worst rms / bound =", round(worst["rms"], 3), " worst max / bound =", round(worst["max"], 3))


def test_plain_entry_point_equals_ex_and_is_deterministic(decoders):
    dec, case = decoders("cfg2-ragged")
    z, bits, off = gpu_inputs(case)
    a = dec.chunk_decode(z, bits, off).clone()
    b = dec.chunk_decode_ex(z, bits, off)["frames"].clone()
    c = dec.chunk_decode(z, bits, off).clone()
    torch.cuda.synchronize()
    assert torch.equal(a, b) and torch.equal(a, c)          # run-to-run bit-identical (R12 ii)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        d = dec.chunk_decode(z, bits, off, stream=s)
    s.synchronize()
    assert torch.equal(a, d)


def test_tail_filling_off_gives_bit_identical_frames(decoders):
    """The trunk's per-tile waits (depthwise tiles start on the MLP kernel's tile counters, dynamic tile claims) only change
    WHEN a tile runs: frames must equal those of whole-grid waits with static striding bit for bit, call after call."""
    from paper_2606_04410_b200 import binding
    dec, case = decoders("cfg3-crop")
    z, bits, off = gpu_inputs(case)
    ref = dec.chunk_decode(z, bits, off).clone()
    plain = binding.ChunkDecoder(case["cfg"], debug_flags=binding.DBG["no_tail_fill"])
    try:
        plain.load_weights(case["weights"])
        a = plain.chunk_decode(z, bits, off).clone()
        torch.cuda.synchronize()
        assert plain.get_status() == 0
        assert torch.equal(a, ref)
        for _ in range(5):                              # tile claims differ from call to call; results must not
            assert torch.equal(dec.chunk_decode(z, bits, off), ref)
    finally:
        plain.destroy()


def test_whole_call_is_cuda_graph_capturable(decoders):
    """ufnvc_chunk_decode only enqueues (no sync, no allocation): the 25-kernel sequence can be captured once in a CUDA
    graph and replayed; the replay's frames equal the direct call's bit for bit."""
    dec, case = decoders("cfg3-crop")
    z, bits, off = gpu_inputs(case)
    ref = dec.chunk_decode(z, bits, off).clone()                 # also the warm-up (function attributes are set here)
    torch.cuda.synchronize()
    frames = dec.new_frames(1)
    s = torch.cuda.Stream()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(s):
        g.capture_begin()
        dec.chunk_decode(z, bits, off, frames=frames, stream=s)
        g.capture_end()
    frames.zero_()
    g.replay()
    torch.cuda.synchronize()
    assert dec.get_status() == 0
    assert torch.equal(frames, ref)


@pytest.mark.parametrize("flag", ["force_generic", "no_pdl", "no_tail_fill", "fp64_head", "no_cta_pairs", "unfused_trunk",
                                  "generic_final", "plain_depthwise", "no_transposed_tiles", "no_quad_clusters"])
def test_every_debug_variant_matches_oracle(decoders, flag):
    """ufnvc_config.debug_flags swaps one kernel (or launch mechanism) for its kept cross-check variant; every kept variant
    is held to the same parity bar as the default path, on the crop of the headline layer plan that reaches every kernel."""
    from paper_2606_04410_b200 import binding
    _, case = decoders("cfg3-crop")
    cfg = case["cfg"]
    dec = binding.ChunkDecoder(cfg, debug_flags=binding.DBG[flag])
    try:
        dec.load_weights(case["weights"])
        z, bits, off = gpu_inputs(case)
        out = dec.chunk_decode_ex(z, bits, off, taps=True)
        torch.cuda.synchronize()
        assert dec.get_status() == 0
        ref = case["chunks"][0]["out"]
        assert np.array_equal(out["sym"][0].cpu().numpy(), nhwc(ref["sym"]))
        assert np.array_equal(out["idx"][0].cpu().numpy(), nhwc(ref["idx"]))
        f = out["frames"][0].cpu().numpy()
        assert np.abs(f - ref["frames"]).max() <= PIX_TOL and psnr(f, ref["frames"]) >= PSNR_MIN
        if flag in ("no_pdl", "no_tail_fill"):          # scheduling only: bit-identical to the default path
            base, _ = decoders("cfg3-crop")
            assert torch.equal(out["frames"], base.chunk_decode(z, bits, off))
        print(flag, "launches:", dec.launches_per_call(1), " max |d pixel| =", float(np.abs(f - ref["frames"]).max()))
    finally:
        dec.destroy()


def test_unknown_debug_flag_is_rejected():
    from paper_2606_04410_b200 import binding
    with pytest.raises(binding.UfnvcError, match="-2"):
        binding.ChunkDecoder(synth.CONFIGS[1], debug_flags=0x400)


@pytest.mark.parametrize("scale", [10.0, 100.0])
def test_hybrid_head_indices_with_scaled_weights(orc, scale):
    """the tensor-core head's fp64 re-decision threshold is an a-priori bound kappa |w row| |x patch| that grows
    with the weights and activations, not a constant calibrated on the synthetic law.  Scale hyper.1's output (and with
    it the head's input) by 10 and 100, re-centre ln sigma so it still spreads over the buckets: the indices must still
    equal the oracle's fp64 decision everywhere."""
    import oracle
    from paper_2606_04410_b200 import binding
    cfg = synth.crop_config(synth.CONFIGS[3], 272, 480)
    wts = dict(synth.make_weights(cfg))
    wts["hyper.1.w"] = synth.round_to_bf16(wts["hyper.1.w"] * np.float32(scale))
    wts["hyper.1.b"] = wts["hyper.1.b"] * np.float32(scale)
    half = cfg.c_y * 16
    w2 = wts["hyper.2.w"].copy()
    w2[half:] = synth.round_to_bf16(w2[half:] * np.float32(0.3 / math.sqrt(scale)))      # sigma spread stays inside the table
    wts["hyper.2.w"] = w2
    z = synth.make_z(cfg)
    mu, u, idx = oracle.entropy_params(orc, cfg, wts, z[0])
    assert 8 < len(np.unique(idx)) and 0.02 < float((np.diff(np.sort(u.ravel())) > 0).mean())
    dec = binding.ChunkDecoder(cfg)
    dec.load_weights(wts)
    _, ls, got = dec.entropy_params(torch.from_numpy(z).cuda())
    torch.cuda.synchronize()
    n_fix = dec.debug_counter(0)
    print(f"scale {scale}: {n_fix} of {idx.size} elements re-decided in fp64; max |d ln sigma| =",
          float(np.abs(ls[0].cpu().numpy() - nhwc(u)).max()))
    assert np.array_equal(got[0].cpu().numpy(), nhwc(idx))
    dec.destroy()


def test_entropy_params_entry_point(decoders):
    dec, case = decoders("cfg3-crop")
    z, _, _ = gpu_inputs(case)
    mu, ls, idx = dec.entropy_params(z)
    torch.cuda.synchronize()
    ref = case["chunks"][0]["out"]
    assert (idx[0].cpu().numpy() != nhwc(ref["idx"])).mean() <= IDX_RATE
    # north_star: mean and scale within 1e-2 relative.  The hybrid head (R12) evaluates both on tensor cores
    # from a 2-term bf16 split (observed error <= 3e-5) and re-decides only the bucket of near-edge elements in fp64.
    assert np.abs(ls[0].cpu().numpy() - nhwc(ref["u"])).max() <= 1e-4
    assert np.abs(mu[0].cpu().numpy() - nhwc(ref["mu"])).max() <= 1e-4


def test_tables_and_encoder_bit_equal_to_oracle(decoders, orc):
    import oracle
    dec, case = decoders("cfg2-ragged")
    cfg = case["cfg"]
    st = case["chunks"][0]["stream"]
    assert np.array_equal(dec.get_cdf(), st["cdf"])                       # two independent table builders (R8)
    idx, u16 = nhwc(st["idx"]), case["u16"][0]
    sym = dec.symbols_from_uniform(idx, u16)
    assert np.array_equal(sym, nhwc(st["sym"]))
    bits, off = dec.encode_chunk(idx, sym)
    assert np.array_equal(off, st["sub_off"]) and np.array_equal(bits, st["bits"])   # two independent encoders
    sym2, status = oracle.decode_symbols(orc, cfg, st["cdf"], st["idx"], bits, off)
    assert status == 0 and np.array_equal(sym2, st["sym"])


def test_teacher_forced_exact_laws_entropy_only(decoders, orc):
    """Entropy-only mode: mu and ln sigma drawn exactly from the stated laws, indices fed to both sides (R3, R12)."""
    import oracle
    dec, case = decoders("cfg3-crop")
    cfg = case["cfg"]
    mu, u = synth.make_exact_law_params(cfg)
    idx_hwc, _ = orc.bucket_index(u[0].astype(np.float64), cfg.n_buckets, cfg.scale_min, cfg.scale_max)
    cdf = orc.build_cdf(cfg.n_buckets, cfg.scale_min, cfg.scale_max)
    sym_hwc = orc.symbols_from_uniform(cdf, idx_hwc, case["u16"][0])
    idx_chw, sym_chw = np.moveaxis(idx_hwc, -1, 0), np.moveaxis(sym_hwc, -1, 0)
    bits, off = oracle.encode_chunk(orc, cfg, cdf, idx_chw, sym_chw)
    z = torch.from_numpy(case["z"]).cuda()
    out = dec.chunk_decode_ex(z, torch.from_numpy(bits).cuda(), torch.from_numpy(off.astype(np.int64)).to(torch.int32).cuda(),
                              idx_override=torch.from_numpy(idx_hwc).cuda(), mu_override=torch.from_numpy(mu[0]).cuda(),
                              taps=True, want_frames=False)
    torch.cuda.synchronize()
    assert dec.get_status() == 0
    assert np.array_equal(out["sym"][0].cpu().numpy(), sym_hwc)
    assert np.array_equal(out["yhat"][0].cpu().numpy(), sym_hwc.astype(np.float32) + mu[0])
    zero_frac = float((sym_hwc == 0).mean())
    assert 0.36 <= zero_frac <= 0.46                                       # P(r=0) ~ 0.41


def test_corrupt_and_truncated_streams_set_status_not_fault(decoders):
    dec, case = decoders("cfg2-ragged")
    z, bits, off = gpu_inputs(case)
    rng = np.random.default_rng(0)
    hdr = 8 * (case["cfg"].lanes_per_substream // 32)
    hits = 0
    for trial in range(12):
        b = bits.clone()
        pos = int(rng.integers(hdr, int(off[1].item())))
        b[pos] ^= 1 << int(rng.integers(0, 8))
        dec.chunk_decode_ex(z, b, off, want_frames=False)
        torch.cuda.synchronize()
        hits += dec.get_status() != 0
    assert hits >= 10
    b = bits.clone()
    b[:hdr] = 0xFF                                                          # garbage header: offsets out of range
    dec.chunk_decode_ex(z, b, off, want_frames=False)
    torch.cuda.synchronize()
    assert dec.get_status() & 4
    off2 = off.clone()
    off2[-1] = off2[-1] // 2 // 4 * 4                                       # truncated last substream
    dec.chunk_decode_ex(z, bits, off2, want_frames=False)
    torch.cuda.synchronize()
    assert dec.get_status() != 0
    dec.chunk_decode_ex(z, bits, off, want_frames=False)                    # and the handle still works
    torch.cuda.synchronize()
    assert dec.get_status() == 0


def test_multi_chunk_low_rate_call():
    """Config-4 shape class on a small frame: 2 independent chunks in one call, T=16, c_y=192 (W=192 lanes), low-rate law."""
    from paper_2606_04410_b200 import binding
    import dataclasses
    cfg = dataclasses.replace(synth.crop_config(synth.CONFIGS[4], 96, 160), n_chunks=2)
    case = oracle_case(cfg)
    dec = binding.ChunkDecoder(cfg)
    dec.load_weights(case["weights"])
    z, bits, off = gpu_inputs(case)
    out = dec.chunk_decode_ex(z, bits, off, taps=True)
    torch.cuda.synchronize()
    assert dec.get_status() == 0
    zero = 0.0
    for n, ch in enumerate(case["chunks"]):
        assert np.array_equal(out["sym"][n].cpu().numpy(), nhwc(ch["out"]["sym"]))
        f = out["frames"][n].cpu().numpy()
        assert np.abs(f - ch["out"]["frames"]).max() <= PIX_TOL and psnr(f, ch["out"]["frames"]) >= PSNR_MIN
        zero += float((ch["out"]["sym"] == 0).mean()) / cfg.n_chunks
    assert zero > 0.5                                                        # low-rate: mostly zero symbols
    assert not torch.equal(out["frames"][0], out["frames"][1])
    dec.destroy()


def test_api_errors(decoders):
    import ctypes as C
    from paper_2606_04410_b200 import binding
    cfg = synth.CONFIGS[1]
    dec = binding.ChunkDecoder(cfg)
    z = torch.zeros((1, cfg.c_z, 1, 1), dtype=torch.int16, device="cuda")
    bits = torch.zeros(64, dtype=torch.uint8, device="cuda")
    off = torch.zeros(2, dtype=torch.int32, device="cuda")
    with pytest.raises(binding.UfnvcError, match="-3"):                      # UFNVC_E_NO_WEIGHTS
        dec.chunk_decode(z, bits, off)
    w = synth.make_weights(cfg)
    blob = binding.pack_weights_blob(w, cfg.weight_dtype)
    bad = np.frombuffer(b"XXXX" + blob[4:], np.uint8)
    assert binding.LIB.ufnvc_load_weights(dec.handle, bad.ctypes.data, bad.size) == -4
    w2 = dict(w); del w2["dec.1.2.w"]
    with pytest.raises(binding.UfnvcError, match="dec.1.2.w"):
        dec.load_weights(w2)
    trunc = np.frombuffer(blob[:len(blob) // 2], np.uint8)
    assert binding.LIB.ufnvc_load_weights(dec.handle, trunc.ctypes.data, trunc.size) == -4
    dec.load_weights(w)
    assert binding.LIB.ufnvc_chunk_decode(dec.handle, 1, None, None, 0, None, None, None) == -1
    assert binding.LIB.ufnvc_chunk_decode(dec.handle, 2, z.data_ptr(), bits.data_ptr(), 64, off.data_ptr(), 1, None) == -1
    dec.destroy()


def test_full_size_1080p_config3_matches_oracle():
    """BASELINE.json configs[2] at FULL size, in the launch configuration bench.py times (plain ufnvc_chunk_decode on
    a side stream): every pixel of all 8 frames against the oracle (894 GMAC in fp64 on the host: ~1-2 minutes)."""
    import json
    import time
    from paper_2606_04410_b200 import binding
    cfg = synth.CONFIGS[3]
    t0 = time.time()
    case = oracle_case(cfg, keep=False)
    t_oracle = time.time() - t0
    dec = binding.ChunkDecoder(cfg)
    dec.load_weights(case["weights"])
    z, bits, off = gpu_inputs(case)
    s = torch.cuda.Stream()
    frames = dec.new_frames(1)
    with torch.cuda.stream(s):
        dec.chunk_decode(z, bits, off, frames=frames, stream=s)
    s.synchronize()
    assert dec.get_status() == 0
    ref = case["chunks"][0]["out"]
    f = frames[0].cpu().numpy()
    err = np.abs(f - ref["frames"])
    res = dict(max_abs=float(err.max()), rms=float(np.sqrt((err ** 2).mean())), psnr=psnr(f, ref["frames"]),
               frame_std=float(ref["frames"].std()), oracle_seconds=t_oracle)
    print("full-size config 3:", json.dumps(res))
    out = dec.chunk_decode_ex(z, bits, off, taps=True, want_frames=False)
    torch.cuda.synchronize()
    assert np.array_equal(out["sym"][0].cpu().numpy(), nhwc(ref["sym"]))          # 1,044,480 symbols bit-exact
    assert (out["idx"][0].cpu().numpy() != nhwc(ref["idx"])).mean() <= IDX_RATE
    assert res["max_abs"] <= PIX_TOL and res["psnr"] >= PSNR_MIN, res
    dec.destroy()


def _entropy_reference(orc, cfg, wts, z_n, u16_n):
    """What the oracle says about the entropy stage of one chunk (O1..O5, seconds even at 4K): stream fixture, decoded
    symbols, y."""
    import oracle
    st = oracle.make_stream(orc, cfg, wts, z_n, u16_n)
    cdf = orc.build_cdf(cfg.n_buckets, cfg.scale_min, cfg.scale_max)
    sym, status = oracle.decode_symbols(orc, cfg, cdf, st["idx"], st["bits"], st["sub_off"])
    assert status == 0 and np.array_equal(sym, st["sym"])
    return st, sym, sym.astype(np.float64) + st["mu"]


def _check_frames(f_gpu, f_ref, what):
    err = np.abs(f_gpu - f_ref)
    res = dict(max_abs=float(err.max()), psnr=psnr(f_gpu, f_ref))
    print(what, res)
    assert res["max_abs"] <= PIX_TOL and res["psnr"] >= PSNR_MIN, (what, res)


def test_full_size_4k_config5_matches_oracle(orc):
    """BASELINE.json configs[4] at FULL size (3840x2160, 8 trunk blocks, 34 substreams of 122,880 symbols, the 136x240
    latent; the stage-3 buffer is 2.1 GB), plain ufnvc_chunk_decode on a side stream as bench.py --config 5 runs it.
    All 4,177,920 symbols and indices against the oracle; the pixels of frames t = 0 and t = 7 (the first and the last
    weight group, the lowest and the highest addresses of every stage buffer) against oracle.synthesis run for those two
    frames only (the T frames are independent after O6; ~480 GMAC of fp64 each)."""
    import oracle
    from paper_2606_04410_b200 import binding
    cfg = synth.CONFIGS[5]
    wts, z, u16 = synth.make_weights(cfg), synth.make_z(cfg), synth.make_uniform16(cfg)
    st, sym, yhat = _entropy_reference(orc, cfg, wts, z[0], u16[0])
    dec = binding.ChunkDecoder(cfg)
    dec.load_weights(wts)
    bits, off = binding.concat_streams([(st["bits"], st["sub_off"])])
    zi = torch.from_numpy(z).cuda()
    bi, oi = torch.from_numpy(bits).cuda(), torch.from_numpy(off.astype(np.int64)).to(torch.int32).cuda()
    s = torch.cuda.Stream()
    frames = dec.new_frames(1)
    with torch.cuda.stream(s):
        dec.chunk_decode(zi, bi, oi, frames=frames, stream=s)
    s.synchronize()
    assert dec.get_status() == 0
    out = dec.chunk_decode_ex(zi, bi, oi, taps=True, want_frames=False)
    torch.cuda.synchronize()
    assert np.array_equal(out["sym"][0].cpu().numpy(), nhwc(sym))
    assert np.array_equal(out["idx"][0].cpu().numpy(), nhwc(st["idx"]))
    assert np.abs(out["yhat"][0].cpu().numpy() - nhwc(yhat)).max() <= 1e-4
    del out
    ref, _ = oracle.synthesis(orc, cfg, wts, yhat, only_frames=(0, cfg.T - 1))
    for t in (0, cfg.T - 1):
        _check_frames(frames[0, t].cpu().numpy(), ref[t], f"config 5 full size, frame {t}:")
    dec.destroy()


def test_full_size_config4_four_chunks_matches_oracle(orc):
    """BASELINE.json configs[3] at FULL size: ONE call decoding 4 independent chunks of T = 16 frames at 1920x1080 with
    c_y = 192 (384 lanes), low-rate law.  The stage-3 buffer holds 64 images x 544 x 960 x 64 bf16 = 4.28 GB (2.14 G
    elements: the range where 32-bit element or byte offsets would wrap).  Symbols and indices of every chunk against the
    oracle; pixels of the first frame of chunk 0 and of the last frame of chunk 3 (lowest / highest addresses), plus one
    frame in the middle (chunk 2, t = 5), against oracle.synthesis run for those frames only."""
    import oracle
    from paper_2606_04410_b200 import binding
    cfg = synth.CONFIGS[4]
    assert cfg.n_chunks == 4 and cfg.T == 16
    wts, z, u16 = synth.make_weights(cfg), synth.make_z(cfg), synth.make_uniform16(cfg)
    refs = [_entropy_reference(orc, cfg, wts, z[n], u16[n]) for n in range(cfg.n_chunks)]
    dec = binding.ChunkDecoder(cfg)
    dec.load_weights(wts)
    bits, off = binding.concat_streams([(st["bits"], st["sub_off"]) for st, _, _ in refs])
    zi = torch.from_numpy(z).cuda()
    bi, oi = torch.from_numpy(bits).cuda(), torch.from_numpy(off.astype(np.int64)).to(torch.int32).cuda()
    s = torch.cuda.Stream()
    frames = dec.new_frames(cfg.n_chunks)
    with torch.cuda.stream(s):
        dec.chunk_decode(zi, bi, oi, frames=frames, stream=s)
    s.synchronize()
    assert dec.get_status() == 0
    out = dec.chunk_decode_ex(zi, bi, oi, taps=True, want_frames=False)
    torch.cuda.synchronize()
    zero = 0.0
    for n, (st, sym, yhat) in enumerate(refs):
        assert np.array_equal(out["sym"][n].cpu().numpy(), nhwc(sym)), n
        assert np.array_equal(out["idx"][n].cpu().numpy(), nhwc(st["idx"])), n
        zero += float((sym == 0).mean()) / cfg.n_chunks
    assert zero > 0.6                                    # BASELINE.json: "~70% zero symbols"
    del out
    for n, t in ((0, 0), (2, 5), (3, cfg.T - 1)):
        ref, _ = oracle.synthesis(orc, cfg, wts, refs[n][2], only_frames=(t,))
        _check_frames(frames[n, t].cpu().numpy(), ref[t], f"config 4 full size, chunk {n} frame {t}:")
    dec.destroy()


def test_200_calls_bit_identical_full_size_config3():
    """The trunk's per-tile counters, dynamic tile claims and relaxed remote mbarrier arrives only change WHEN a tile runs:
    200 back-to-back calls at full 1080p (the launch configuration bench.py times, PDL and tail filling on) must give
    the same frames bit for bit (compared on the device, one checksum-free torch.equal per call)."""
    from paper_2606_04410_b200 import binding
    cfg = synth.CONFIGS[3]
    dec = binding.ChunkDecoder(cfg)
    dec.load_weights(synth.make_weights(cfg))
    z = torch.from_numpy(synth.make_z(cfg)).cuda()
    _, _, idx = dec.entropy_params(z)
    idx_h = idx[0].cpu().numpy()
    sym = dec.symbols_from_uniform(idx_h, synth.make_uniform16(cfg)[0])
    b, o = dec.encode_chunk(idx_h, sym)
    bits, off = torch.from_numpy(b).cuda(), torch.from_numpy(o.astype(np.int64)).to(torch.int32).cuda()
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        ref = dec.chunk_decode(z, bits, off, stream=s).clone()
        frames = dec.new_frames(1)
        bad = 0
        for i in range(200):
            dec.chunk_decode(z, bits, off, frames=frames, stream=s)
            bad += int(not torch.equal(frames, ref))
    s.synchronize()
    assert dec.get_status() == 0 and bad == 0
    dec.destroy()


def test_full_size_progressive_means_match_oracle(orc):
    """NEXT-1 at BASELINE.json configs[2]'s full latent size (128 x 68 x 120 = 1,044,480 elements), entropy stage only
    (the oracle's O1-O5 plus the three mean convs take seconds; the synthesis is covered by the cropped -pmu cases):
    symbols bit-exact, every mean and every y within the north-star bound."""
    import oracle
    from paper_2606_04410_b200 import binding
    cfg = synth.progressive_config(synth.CONFIGS[3])
    wts, z, u16 = synth.make_weights(cfg), synth.make_z(cfg), synth.make_uniform16(cfg)
    st = oracle.make_stream(orc, cfg, wts, z[0], u16[0])
    cdf = orc.build_cdf(cfg.n_buckets, cfg.scale_min, cfg.scale_max)
    sym, status = oracle.decode_symbols(orc, cfg, cdf, st["idx"], st["bits"], st["sub_off"])
    assert status == 0 and np.array_equal(sym, st["sym"])
    yhat, mu = oracle.progressive_means(orc, cfg, wts, st["mu"], sym)
    dec = binding.ChunkDecoder(cfg)
    dec.load_weights(wts)
    bits, off = binding.concat_streams([(st["bits"], st["sub_off"])])
    dev = "cuda"
    out = dec.chunk_decode_ex(torch.from_numpy(z).to(dev), torch.from_numpy(bits).to(dev),
                              torch.from_numpy(off.astype(np.int64)).to(torch.int32).to(dev), taps=True, want_frames=False)
    torch.cuda.synchronize()
    assert dec.get_status() == 0
    assert np.array_equal(out["sym"][0].cpu().numpy(), nhwc(sym))
    mu_ref, y_ref = nhwc(mu), nhwc(yhat)
    bound = 1e-2 * np.maximum(np.abs(mu_ref), 1.0)
    d_mu = np.abs(out["mu"][0].cpu().numpy() - mu_ref)
    d_y = np.abs(out["yhat"][0].cpu().numpy() - y_ref)
    print("full-size progressive: max |d mu| =", d_mu.max(), " max |d y| =", d_y.max(), " rms =", float(np.sqrt((d_y ** 2).mean())))
    assert (d_mu <= bound).all() and (d_y <= bound).all()
    part = nhwc(oracle.partition_index(cfg.c_y, cfg.h, cfg.w))
    for k in range(4):
        assert (part == k).mean() == 0.25
    assert d_mu[part == 0].max() <= 1e-4          # partition 0 keeps the head's mean
    dec.destroy()


# ---- NEXT-3 (R22): the hyper-latent from bytes, and the bytes-only call ----------------------------------
@pytest.mark.parametrize("name", ["cfg1", "cfg2-ragged", "cfg3-crop"])
def test_decode_z_and_bytes_only_call(decoders, orc, name):
    import oracle
    from paper_2606_04410_b200 import binding
    dec, case = decoders(name)
    cfg, wts = case["cfg"], case["weights"]
    cdf = orc.build_cdf(cfg.n_buckets, cfg.scale_min, cfg.scale_max)
    assert np.array_equal(dec.get_z_prior_index(), oracle.z_prior_index(orc, cfg, wts))
    parts_z, parts_all = [], []
    for n, ch in enumerate(case["chunks"]):
        zb, zo = oracle.encode_z(orc, cfg, cdf, wts, case["z"][n])
        zb2, zo2 = dec.encode_z(case["z"][n])                         # the library's own fixture encoder: same bytes
        assert np.array_equal(zb, zb2) and np.array_equal(zo, zo2)
        parts_z.append((zb, zo))
        parts_all.append(oracle.pack_chunk_bytes(zb, zo, ch["stream"]["bits"], ch["stream"]["sub_off"]))
    dev = "cuda"

    def up(a, dt=None):
        t = torch.from_numpy(a.astype(np.int64) if dt is not None else a)
        return (t.to(dt) if dt is not None else t).to(dev)
    bits, off = binding.concat_streams(parts_z)
    z = dec.decode_z(up(bits), up(off, torch.int32), n_chunks=cfg.n_chunks)
    torch.cuda.synchronize()
    assert dec.get_status() == 0
    assert np.array_equal(z.cpu().numpy(), case["z"])                 # integer work: bit-exact
    # bytes in, frames out == the z-in call on the same inputs, bit for bit
    bits, off = binding.concat_streams(parts_all)
    f_bytes = dec.chunk_decode_bytes(up(bits), up(off, torch.int32), n_chunks=cfg.n_chunks)
    torch.cuda.synchronize()
    assert dec.get_status() == 0
    zi, bi, oi = gpu_inputs(case)
    f_z = dec.chunk_decode(zi, bi, oi)
    torch.cuda.synchronize()
    assert torch.equal(f_bytes, f_z)
    ref = case["chunks"][0]["out"]["frames"]
    assert np.abs(f_bytes[0].cpu().numpy() - ref).max() <= PIX_TOL
    # a flipped byte inside the z part, or inside the y part, is reported and never faults
    for where in (int(off[1]) // 2, int(off[dec.n_sub_z]) + 200):
        bad = bits.copy()
        bad[where] ^= 0x77
        dec.chunk_decode_bytes(up(bad), up(off, torch.int32), n_chunks=cfg.n_chunks)
        torch.cuda.synchronize()
        assert dec.get_status() != 0


def test_decode_z_full_size_and_without_prior(orc):
    """Config 3's hyper-latent at full size (64 x 17 x 30, 5 substreams, ragged last one); a blob without zprior.lnscale
    keeps every other entry point working and makes the bytes-only ones fail loudly."""
    import oracle
    from paper_2606_04410_b200 import binding
    cfg = synth.CONFIGS[3]
    wts, z = synth.make_weights(cfg), synth.make_z(cfg)
    cdf = orc.build_cdf(cfg.n_buckets, cfg.scale_min, cfg.scale_max)
    zb, zo = oracle.encode_z(orc, cfg, cdf, wts, z[0])
    dec = binding.ChunkDecoder(cfg)
    dec.load_weights(wts)
    assert dec.n_sub_z == 5 and zo.size == 6
    got = dec.decode_z(torch.from_numpy(zb).cuda(), torch.from_numpy(zo.astype(np.int64)).to(torch.int32).cuda())
    torch.cuda.synchronize()
    assert dec.get_status() == 0 and np.array_equal(got.cpu().numpy(), z)
    dec.load_weights({k: v for k, v in wts.items() if not k.startswith("zprior.")})
    with pytest.raises(binding.UfnvcError):
        dec.decode_z(torch.from_numpy(zb).cuda(), torch.from_numpy(zo.astype(np.int64)).to(torch.int32).cuda())
    mu, ls, idx = dec.entropy_params(torch.from_numpy(z).cuda())       # the z-in path is untouched
    torch.cuda.synchronize()
    assert idx.shape == (1, cfg.h, cfg.w, cfg.c_y)
    dec.destroy()


def test_multi_chunk_progressive_bytes_only_and_graph():
    """The two widened paths together, on a two-chunk call (config 4's layer plan: C_y = 192, T = 16, 384 lanes, cropped):
    mu_steps = 4 with the chunks handed over as bytes only; per-chunk parity against the oracle; the whole call captured
    in a CUDA graph replays bit-identically."""
    import dataclasses
    import oracle
    from paper_2606_04410_b200 import binding
    cfg = synth.progressive_config(dataclasses.replace(synth.crop_config(synth.CONFIGS[4], 96, 160), n_chunks=2))
    case = oracle_case(cfg)
    orc = oracle.Oracle()
    cdf = orc.build_cdf(cfg.n_buckets, cfg.scale_min, cfg.scale_max)
    parts = []
    for n, ch in enumerate(case["chunks"]):
        zb, zo = oracle.encode_z(orc, cfg, cdf, case["weights"], case["z"][n])
        parts.append(oracle.pack_chunk_bytes(zb, zo, ch["stream"]["bits"], ch["stream"]["sub_off"]))
    bits_h, off_h = binding.concat_streams(parts)
    bits = torch.from_numpy(bits_h).cuda()
    off = torch.from_numpy(off_h.astype(np.int64)).to(torch.int32).cuda()
    dec = binding.ChunkDecoder(cfg)
    dec.load_weights(case["weights"])
    ref = dec.chunk_decode_bytes(bits, off, n_chunks=2).clone()
    torch.cuda.synchronize()
    assert dec.get_status() == 0
    for n, ch in enumerate(case["chunks"]):
        f = ref[n].cpu().numpy()
        assert np.abs(f - ch["out"]["frames"]).max() <= PIX_TOL and psnr(f, ch["out"]["frames"]) >= PSNR_MIN
    zi, bi, oi = gpu_inputs(case)
    out = dec.chunk_decode_ex(zi, bi, oi, taps=True)
    torch.cuda.synchronize()
    assert torch.equal(out["frames"], ref)
    for n, ch in enumerate(case["chunks"]):
        assert np.array_equal(out["sym"][n].cpu().numpy(), nhwc(ch["out"]["sym"]))
        mu_ref = nhwc(ch["out"]["mu"])
        assert (np.abs(out["mu"][n].cpu().numpy() - mu_ref) <= 1e-2 * np.maximum(np.abs(mu_ref), 1.0)).all()
    frames = dec.new_frames(2)
    s = torch.cuda.Stream()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(s):
        g.capture_begin()
        dec.chunk_decode_bytes(bits, off, n_chunks=2, frames=frames, stream=s)
        g.capture_end()
    frames.zero_()
    g.replay()
    torch.cuda.synchronize()
    assert dec.get_status() == 0 and torch.equal(frames, ref)
    dec.destroy()


# ---- NEXT-4 (part): GPU rANS encode, byte-identical to the oracle's encoder ----------------------------------------
@pytest.mark.parametrize("name", ["cfg1", "cfg2-ragged", "cfg3-crop", "cfg2"])
def test_gpu_rans_encode_is_byte_identical_to_oracle(decoders, name):
    from paper_2606_04410_b200 import binding
    dec, case = decoders(name)
    cfg = case["cfg"]
    idx = torch.from_numpy(np.stack([nhwc(ch["stream"]["idx"]) for ch in case["chunks"]])).cuda()
    sym = torch.from_numpy(np.stack([nhwc(ch["stream"]["sym"]) for ch in case["chunks"]])).cuda()
    bits, off = dec.encode_chunk_dev(idx, sym)
    torch.cuda.synchronize()
    assert dec.get_status() == 0
    want_bits, want_off = binding.concat_streams([(c["stream"]["bits"], c["stream"]["sub_off"]) for c in case["chunks"]])
    got_off = off.cpu().numpy().astype(np.uint32)
    assert np.array_equal(got_off, want_off)
    assert np.array_equal(bits.cpu().numpy()[:int(got_off[-1])], want_bits)
    # and the library decodes its own stream back (device to device, no host in between)
    zi, _, _ = gpu_inputs(case)
    out = dec.chunk_decode_ex(zi, bits[:int(got_off[-1])], off, taps=True, want_frames=False)
    torch.cuda.synchronize()
    assert dec.get_status() == 0 and torch.equal(out["sym"], sym)
    # error paths: a symbol outside the alphabet, and an output buffer that is too small
    bad = sym.clone()
    bad.view(-1)[5] = 200
    dec.encode_chunk_dev(idx, bad)
    torch.cuda.synchronize()
    assert dec.get_status() != 0
    _, off2 = dec.encode_chunk_dev(idx, sym, cap=64)
    torch.cuda.synchronize()
    assert dec.get_status() != 0 and int(off2[-1]) == int(got_off[-1])


def test_gpu_rans_encode_full_size_1080p(orc):
    """All 1,044,480 symbols of config 3 (17 substreams, 512 lanes): byte-identical to the oracle's encoder, exact-law
    (mu, sigma) maps as in the entropy-only mode; timing printed."""
    import oracle
    from paper_2606_04410_b200 import binding
    cfg = synth.CONFIGS[3]
    _, u = synth.make_exact_law_params(cfg)
    idx_chw, _ = orc.bucket_index(np.moveaxis(u[0], -1, 0), cfg.n_buckets, cfg.scale_min, cfg.scale_max)
    cdf = orc.build_cdf(cfg.n_buckets, cfg.scale_min, cfg.scale_max)
    u16 = synth.make_uniform16(cfg)[0]
    sym_chw = orc.symbols_from_uniform(cdf, idx_chw, np.transpose(u16, (2, 0, 1)))
    want_bits, want_off = oracle.encode_chunk(orc, cfg, cdf, idx_chw, sym_chw)
    dec = binding.ChunkDecoder(cfg)
    idx = torch.from_numpy(nhwc(idx_chw)[None]).cuda()
    sym = torch.from_numpy(nhwc(sym_chw)[None]).cuda()
    bits, off = dec.encode_chunk_dev(idx, sym)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(10):
        bits, off = dec.encode_chunk_dev(idx, sym)
    e1.record()
    e1.synchronize()
    assert dec.get_status() == 0
    got_off = off.cpu().numpy().astype(np.uint32)
    assert np.array_equal(got_off, want_off) and np.array_equal(bits.cpu().numpy()[:int(got_off[-1])], want_bits)
    print("GPU rANS encode, 1080p chunk:", e0.elapsed_time(e1) / 10 * 1e3, "us incl. output allocation;", int(got_off[-1]), "bytes")
    dec.destroy()
