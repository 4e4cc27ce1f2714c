"""Chunk ENCODE on the GPU (R24) against the oracle, through the C ABI.

The encoder takes two integer decisions from floats -- z = round(hyper-encoder(y)) and r = round(y - mu) -- and its y comes
from bf16 tensor-core layers, so the GPU's integers differ from the oracle's at rounding edges (by design: whatever the
encoder picks is what the decoder recovers).  Parity is therefore staged, each stage fed the SAME inputs on both sides:
  1. y (E1..E5) against the oracle's y within the bf16-derived bound;
  2. the hyper-encoder on the GPU's y against the oracle's on that y (fp32 against fp64), z equal except at rounding edges;
  3. r = rint(y - mu) recomputed in numpy from the GPU's own taps: bit-exact;
  4. the bytes: oracle.chunk_encode teacher-forced with the GPU's (y, z) must give the GPU's bit-stream byte for byte
     (prior net indices exact, quantiser exact, rANS encoder exact);
  5. round trip: decoding the GPU's bytes on the GPU returns exactly the coded symbols, and the frames match the oracle's
     decode of the same bytes within the north-star tolerance.
"""
import dataclasses
import math

import numpy as np
import pytest
import torch

import oracle
from common import nhwc, psnr
from paper_2606_04410_b200 import synth

pytestmark = pytest.mark.gpu
PIX_TOL, PSNR_MIN = 2e-2, 45.0


def _case(cfg):
    return cfg, synth.make_weights(cfg), synth.make_frames(cfg)


@pytest.mark.parametrize("name", ["cfg3-crop", "cfg2-ragged", "cfg3-crop-T1", "cfg3-crop-ctx"])
def test_chunk_encode_staged_parity_and_round_trip(orc, name):
    from paper_2606_04410_b200 import binding
    base = {"cfg3-crop": synth.crop_config(synth.CONFIGS[3], 272, 480),
            "cfg2-ragged": synth.crop_config(synth.CONFIGS[2], 150, 200),
            "cfg3-crop-T1": dataclasses.replace(synth.crop_config(synth.CONFIGS[3], 272, 480), T=1, name="cfg3-crop-T1"),
            "cfg3-crop-ctx": synth.context_config(synth.crop_config(synth.CONFIGS[3], 272, 480), 2)}[name]
    cfg, wts, frames = _case(synth.encoder_config(base, 2))
    dec = binding.ChunkDecoder(cfg)
    dec.load_weights(wts)
    ctx = None
    if cfg.n_ctx_blocks:
        # a non-trivial context: what the oracle's decoder hands on after one chunk
        e0 = oracle.chunk_encode(orc, cfg, wts, frames[0])
        ctx = oracle.chunk_decode(orc, cfg, wts, e0["z"], e0["bits"], e0["sub_off"])["ctx_next"]
        dec.set_context(torch.from_numpy(nhwc(ctx).astype(np.float32)[None]).to(torch.bfloat16).cuda())
    out = dec.chunk_encode(torch.from_numpy(frames).cuda(), taps=True)
    torch.cuda.synchronize()
    assert dec.get_status() == 0
    # 1. the latent
    ref = oracle.chunk_encode(orc, cfg, wts, frames[0], ctx=ctx)
    y = out["y"][0].cpu().numpy()
    want = nhwc(ref["y"])
    L = 2 + 1 + 3 * cfg.n_enc_blocks + (1 if cfg.n_ctx_blocks else 0)        # patches, embedding, fold, 3 per block (+ context add)
    r = math.sqrt(L) * 2.0 ** -8 / math.sqrt(3.0)
    d = y - want
    rms_e, rms_b = float(np.sqrt(np.mean(d ** 2))), r * float(np.sqrt(np.mean(want ** 2)))
    max_e, max_b = float(np.abs(d).max()), 6.0 * r * float(np.abs(want).max())
    print(f"{name}: latent rms err / bound = {rms_e / rms_b:.3f}, max err / bound = {max_e / max_b:.3f}")
    assert rms_e <= rms_b and max_e <= max_b
    # 2. hyper-encoder on the GPU's own y
    y_chw = np.moveaxis(y.astype(np.float64), -1, 0)
    z_ref, zf_ref = oracle.hyper_encoder(orc, cfg, wts, y_chw)
    zf = out["zf"][0].cpu().numpy()
    z = out["z"][0].cpu().numpy()
    assert np.abs(zf - zf_ref).max() <= 1e-3 * max(1.0, float(np.abs(zf_ref).max()))
    assert np.array_equal(z, np.clip(np.rint(zf), -127, 127).astype(np.int16))       # the GPU's own rounding rule
    mism = z != z_ref
    assert mism.mean() <= 1e-3 and (np.abs(np.abs(zf_ref[mism] - np.floor(zf_ref[mism])) - 0.5) < 1e-2).all()
    # 3. the quantiser, from the GPU's own taps
    sym = out["sym"][0].cpu().numpy()
    assert np.array_equal(sym, oracle.quantise(y, out["mu"][0].cpu().numpy()))
    # 4. the bytes.  The oracle's encoder teacher-forced with the GPU's y and z: same indices (the prior net's decision is exact);
    # the same residuals except where y - mu sits on a rounding edge (the GPU's tensor-core mean is ~3e-5 from the fp64 one);
    # and, fed the GPU's own (idx, r), the oracle's rANS encoder writes the GPU's bit-stream byte for byte.
    tf = oracle.chunk_encode(orc, cfg, wts, frames[0], ctx=ctx, z_override=z, y_override=y_chw)
    assert np.array_equal(out["idx"][0].cpu().numpy(), nhwc(tf["idx"]))
    flips = sym != nhwc(tf["sym"])
    dref = (y.astype(np.float64) - nhwc(tf["mu"]))[flips]
    assert flips.mean() <= 1e-3 and (np.abs(np.abs(dref - np.floor(dref)) - 0.5) < 1e-3).all()
    cdf = orc.build_cdf(cfg.n_buckets, cfg.scale_min, cfg.scale_max)
    want_bits, want_off = oracle.encode_chunk(orc, cfg, cdf, tf["idx"], np.moveaxis(sym, -1, 0))
    off = out["sub_off"].cpu().numpy().astype(np.uint32)
    assert np.array_equal(off, want_off)
    bits = out["bits"].cpu().numpy()[:int(off[-1])]
    assert np.array_equal(bits, want_bits)
    print(f"{name}: {bits.size} bytes for {cfg.T} frames of {cfg.width}x{cfg.height}; z differs from the fp64 rounding in {int(mism.sum())} of {z.size}, r in {int(flips.sum())} of {sym.size}")
    # 5. round trip on the device
    got = dec.chunk_decode_ex(out["z"], out["bits"][:int(off[-1])], out["sub_off"], taps=True)
    torch.cuda.synchronize()
    assert dec.get_status() == 0
    assert np.array_equal(got["sym"][0].cpu().numpy(), sym)
    ref_dec = oracle.chunk_decode(orc, cfg, wts, z, bits, off, ctx=ctx)
    assert ref_dec["status"] == 0 and np.array_equal(nhwc(ref_dec["sym"]), sym)
    f = got["frames"][0].cpu().numpy()
    assert np.abs(f - ref_dec["frames"]).max() <= PIX_TOL and psnr(f, ref_dec["frames"]) >= PSNR_MIN
    unclipped = np.abs(sym) < 127
    assert np.abs(got["yhat"][0].cpu().numpy() - y)[unclipped].max() <= 0.5 + 1e-3          # |y_hat - y| <= 1/2
    dec.destroy()


def test_colour_conversion_matches_oracle_and_round_trips():
    from paper_2606_04410_b200 import binding
    rng = np.random.default_rng(0)
    rgb = rng.uniform(size=(2, 3, 3, 37, 53)).astype(np.float32)
    x = torch.from_numpy(rgb).cuda()
    yuv = binding.convert_colour(x, True)
    back = binding.convert_colour(yuv, False)
    torch.cuda.synchronize()
    assert np.abs(yuv.cpu().numpy() - oracle.rgb_to_yuv444(rgb)).max() <= 2e-6
    assert np.abs(back.cpu().numpy() - rgb).max() <= 5e-6
    assert np.abs(back.cpu().numpy() - oracle.yuv444_to_rgb(yuv.cpu().numpy().astype(np.float64))).max() <= 2e-6


def test_encode_api_errors():
    from paper_2606_04410_b200 import binding
    base = synth.crop_config(synth.CONFIGS[3], 272, 480)
    dec = binding.ChunkDecoder(base)
    dec.load_weights(synth.make_weights(base))
    with pytest.raises(binding.UfnvcError, match="-2"):            # no encoder in this config
        dec.chunk_encode(torch.zeros((1, base.T, 3, base.height, base.width), device="cuda"))
    dec.destroy()
    cfg = synth.encoder_config(base, 1)
    dec = binding.ChunkDecoder(cfg)
    w = synth.make_weights(cfg)
    w2 = dict(w); del w2["henc.1.w"]
    with pytest.raises(binding.UfnvcError, match="henc.1.w"):
        dec.load_weights(w2)
    dec.load_weights(w)
    out = dec.chunk_encode(torch.from_numpy(synth.make_frames(cfg)).cuda(), cap=64)     # output buffer too small: status, no overrun
    torch.cuda.synchronize()
    assert dec.get_status() != 0
    dec.destroy()
    with pytest.raises(binding.UfnvcError, match="-2"):            # the encoder supports the single-pass mean only
        binding.ChunkDecoder(synth.encoder_config(synth.progressive_config(base), 1))
