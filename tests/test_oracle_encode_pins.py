"""Pins for the oracle's chunk ENCODER and colour interface (R24).

The text fixes: patch embedding to 1/8 resolution, a chunk encoder of DC blocks conditioned on C_i, r = round(y - mu) coded
with sigma, a unified YUV444 interface with BT.709 for RGB.  The layer plan (fold over frames, hyper-encoder) is reading R24.
Pins: the colour matrices against BT.709's published luma coefficients and primaries; space-to-depth against the library's
pixel_unshuffle; every conv step of the plan against explicit gathers / matrix products; the quantiser's defining inequality;
and the encode -> decode round trip (what the decoder recovers is exactly what the encoder coded).  Fidelity to the paper's
trained encoder: parity unpinned.
"""
import dataclasses

import numpy as np
import torch
import torch.nn.functional as F

import oracle
from paper_2606_04410_b200 import synth


def tiny():
    cfg = synth.encoder_config(synth.crop_config(synth.CONFIGS[1], 150, 200), 2)       # H x W = 160 x 224, h = 10, w = 14 (ragged z)
    return cfg, synth.make_weights(cfg), synth.make_frames(cfg)[0]


def test_bt709_closed_forms_and_round_trip():
    px = lambda r, g, b: np.array([r, g, b], np.float64).reshape(3, 1, 1)
    assert np.allclose(oracle.rgb_to_yuv444(px(1, 1, 1)).ravel(), [1.0, 0.5, 0.5])          # white: full luma, neutral chroma
    assert np.allclose(oracle.rgb_to_yuv444(px(0, 0, 0)).ravel(), [0.0, 0.5, 0.5])
    y, cb, cr = oracle.rgb_to_yuv444(px(1, 0, 0)).ravel()                                     # red primary
    assert abs(y - 0.2126) < 1e-15 and abs(cr - 1.0) < 1e-12 and abs(cb - (0.5 - 0.2126 / 1.8556)) < 1e-15
    y, cb, cr = oracle.rgb_to_yuv444(px(0, 0, 1)).ravel()                                     # blue primary
    assert abs(y - 0.0722) < 1e-15 and abs(cb - 1.0) < 1e-12
    assert abs(0.2126 + 0.7152 + 0.0722 - 1.0) < 1e-15                                        # BT.709 luma coefficients
    assert abs(1.8556 - 2 * (1 - 0.0722)) < 1e-12 and abs(1.5748 - 2 * (1 - 0.2126)) < 1e-12  # chroma scalings follow from them
    rgb = np.random.default_rng(0).uniform(size=(2, 3, 5, 7))
    assert np.abs(oracle.yuv444_to_rgb(oracle.rgb_to_yuv444(rgb)) - rgb).max() < 1e-14
    assert oracle.rgb_to_yuv444(rgb).shape == rgb.shape


def test_space_to_depth_against_library_and_inverse(orc):
    rng = np.random.default_rng(1)
    for r in (2, 4, 8):
        x = rng.normal(size=(3, 2 * r, 3 * r))
        s = oracle.space_to_depth(x, r)
        assert s.shape == (3 * r * r, 2, 3)
        for (c, y, xx, i, j) in [(0, 0, 0, 0, 0), (2, 1, 2, r - 1, 1), (1, 0, 1, 1, r - 1)]:
            assert s[(r * i + j) * 3 + c, y, xx] == x[c, r * y + i, r * xx + j]
        # torch.pixel_unshuffle orders channels c r^2 + r i + j (channel-major); ours is position-major
        tu = F.pixel_unshuffle(torch.from_numpy(x)[None], r)[0].numpy().reshape(3, r * r, 2, 3).transpose(1, 0, 2, 3).reshape(3 * r * r, 2, 3)
        assert np.array_equal(s, tu)
        back = F.pixel_shuffle(torch.from_numpy(s.reshape(r * r, 3, 2, 3).transpose(1, 0, 2, 3).reshape(3 * r * r, 2, 3))[None], r)[0].numpy()
        assert np.array_equal(back, x)


def test_quantiser_definition():
    rng = np.random.default_rng(2)
    y = rng.normal(0, 30, size=20000).astype(np.float32)
    mu = rng.normal(0, 1, size=20000).astype(np.float32)
    r = oracle.quantise(y, mu)
    d = y - mu
    inside = np.abs(d) < 127.4
    assert (np.abs(d[inside] - r[inside]) <= 0.5).all()                      # nearest integer
    assert (np.abs(r) <= 127).all() and (r[d > 128] == 127).all() and (r[d < -128] == -127).all()
    assert oracle.quantise(np.float32([0.5, 1.5, 2.5, -0.5, -1.5]), np.zeros(5, np.float32)).tolist() == [0, 2, 2, 0, -2]   # ties to even


def test_patch_embedding_and_fold_by_explicit_gathers(orc):
    cfg, w, frames = tiny()
    g = oracle.geometry(cfg)
    # zero every DC block's W2 and use an identity-like latent head so that y exposes E1/E2 directly
    w = dict(w)
    for k in range(cfg.n_enc_blocks):
        w[f"enc.{k}.pw2.w"] = np.zeros_like(w[f"enc.{k}.pw2.w"]); w[f"enc.{k}.pw2.b"] = np.zeros_like(w[f"enc.{k}.pw2.b"])
    ct = cfg.c_trunk
    w["enc.y.w"] = np.eye(cfg.c_y, ct, dtype=np.float32)[:, :, None, None]; w["enc.y.b"] = np.zeros(cfg.c_y, np.float32)
    y = oracle.encoder_features(orc, cfg, w, frames)
    assert y.shape == (cfg.c_y, g["h"], g["w"])
    x = np.zeros((cfg.T, 3, g["H"], g["W"]))
    x[:, :, :cfg.height, :cfg.width] = frames
    wp, bp = w["enc.patch.w"][:, :, 0, 0].astype(np.float64), w["enc.patch.b"].astype(np.float64)
    wf, bf = w["enc.fold.w"][:, :, 0, 0].astype(np.float64), w["enc.fold.b"].astype(np.float64)
    for (o, ly, lx) in [(0, 0, 0), (3, 9, 13), (cfg.c_y - 1, 4, 7)]:
        acc = bf[o]
        for t in range(cfg.T):
            for i in range(2):
                for j in range(2):
                    y8, x8 = 2 * ly + i, 2 * lx + j                           # the 1/8-resolution pixel
                    patch = np.array([x[t, c, 8 * y8 + a, 8 * x8 + b] for a in range(8) for b in range(8) for c in range(3)])   # (8 a + b) 3 + c
                    f1 = wp @ patch + bp                                      # E1 at that pixel, all C_t channels
                    k0 = t * 4 * ct + (2 * i + j) * ct
                    acc += wf[o, k0:k0 + ct] @ f1
        assert abs(y[o, ly, lx] - acc) < 1e-10
    # frames past the picture edge are zero padding: the bottom-right latent pixel sees partly padded patches and is finite
    assert np.isfinite(y).all()


def test_hyper_encoder_ragged_padding_and_rounding(orc):
    cfg, w, frames = tiny()
    g = oracle.geometry(cfg)
    assert (g["h"], g["h_z"], g["w"], g["w_z"]) == (10, 3, 14, 4)
    rng = np.random.default_rng(3)
    y = rng.normal(0, 8, size=(cfg.c_y, g["h"], g["w"]))
    z, zf = oracle.hyper_encoder(orc, cfg, w, y)
    assert z.shape == (cfg.c_z, 3, 4) and z.dtype == np.int16 and (np.abs(z) <= 127).all()
    assert np.array_equal(z, np.clip(np.rint(zf), -127, 127))
    # the last z row sees latent rows 8, 9 and two rows of ZERO padding: changing nothing but padding-position inputs is impossible,
    # so check instead that y rows >= 8 do not reach z row 1 except through the 3x3 conv's one-pixel halo (z row 0 is untouched)
    y2 = y.copy(); y2[:, 8:, :] += 5.0
    z2, zf2 = oracle.hyper_encoder(orc, cfg, w, y2)
    assert np.array_equal(zf2[:, 0], zf[:, 0]) and not np.array_equal(zf2[:, 2], zf[:, 2])
    # explicit value at one position: a = ReLU(W0 Y4 + b0) per z-pixel, zf = 3x3 conv over a
    yp = np.zeros((cfg.c_y, 12, 16)); yp[:, :10, :14] = y
    a = np.zeros((cfg.c_hyper, 3, 4))
    w0, b0 = w["henc.0.w"][:, :, 0, 0].astype(np.float64), w["henc.0.b"].astype(np.float64)
    for zy in range(3):
        for zx in range(4):
            v = np.array([yp[c, 4 * zy + i, 4 * zx + j] for i in range(4) for j in range(4) for c in range(cfg.c_y)])     # (4 i + j) C_y + c
            a[:, zy, zx] = np.maximum(w0 @ v + b0, 0.0)
    w1, b1 = w["henc.1.w"].astype(np.float64), w["henc.1.b"].astype(np.float64)
    o, zy, zx = 5, 2, 3
    acc = b1[o]
    for dy in range(3):
        for dx in range(3):
            yy, xx = zy + dy - 1, zx + dx - 1
            if 0 <= yy < 3 and 0 <= xx < 4:
                acc += w1[o, :, dy, dx] @ a[:, yy, xx]
    assert abs(zf[o, zy, zx] - acc) < 1e-10


def test_encode_then_decode_round_trip(orc):
    """What the decoder recovers is exactly what the encoder coded: same z -> same indices, symbols bit-exact, status clean,
    and the dequantised latent within half a quantisation step of the encoder's y."""
    cfg, w, frames = tiny()
    e = oracle.chunk_encode(orc, cfg, w, frames)
    assert (np.abs(e["z"]) <= 127).all() and e["sub_off"][-1] == e["bits"].size
    d = oracle.chunk_decode(orc, cfg, w, e["z"], e["bits"], e["sub_off"])
    assert d["status"] == 0 and np.array_equal(d["idx"], e["idx"]) and np.array_equal(d["sym"], e["sym"])
    unclipped = np.abs(e["sym"]) < 127
    assert np.abs(d["yhat"] - e["y"])[unclipped].max() <= 0.5 + 1e-6
    assert d["frames"].shape == (cfg.T, 3, cfg.height, cfg.width)
    # teacher forcing hooks: a foreign z / y is taken as given
    e2 = oracle.chunk_encode(orc, cfg, w, frames, z_override=e["z"], y_override=e["y"])
    assert np.array_equal(e2["bits"], e["bits"])
    # T = 1 (the paper's low-delay shape) goes through the same code
    cfg1 = dataclasses.replace(cfg, T=1)
    w1 = synth.make_weights(cfg1)
    e1 = oracle.chunk_encode(orc, cfg1, w1, frames[:1])
    d1 = oracle.chunk_decode(orc, cfg1, w1, e1["z"], e1["bits"], e1["sub_off"])
    assert d1["status"] == 0 and np.array_equal(d1["sym"], e1["sym"]) and d1["frames"].shape[0] == 1
