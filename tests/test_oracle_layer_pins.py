"""Pins for the oracle's layers (O1, O2, O6-O9) against brute force, closed forms and library routines."""
import math

import numpy as np
import pytest
import torch
import torch.nn.functional as F

import oracle
from paper_2606_04410_b200 import synth


def brute_conv(x, w, b):
    """The definition as 7 nested loops over explicit zero-padded input, float64."""
    co, ci, k, _ = w.shape
    p = (k - 1) // 2
    _, H, W = x.shape
    xp = np.zeros((ci, H + 2 * p, W + 2 * p))
    xp[:, p:p + H, p:p + W] = x
    out = np.zeros((co, H, W))
    for o in range(co):
        for y in range(H):
            for xx in range(W):
                acc = b[o]
                for c in range(ci):
                    for dy in range(k):
                        for dx in range(k):
                            acc += w[o, c, dy, dx] * xp[c, y + dy, xx + dx]
                out[o, y, xx] = acc
    return out


@pytest.mark.parametrize("k,ci,co,H,W", [(3, 3, 4, 5, 7), (3, 2, 3, 1, 1), (1, 5, 6, 4, 3), (3, 1, 2, 2, 9)])
def test_conv_vs_brute_force(orc, k, ci, co, H, W):
    rng = np.random.default_rng(k * 100 + ci)
    x, w, b = rng.normal(size=(ci, H, W)), rng.normal(size=(co, ci, k, k)), rng.normal(size=co)
    assert np.allclose(orc.conv2d(x, w, b), brute_conv(x, w, b), atol=1e-12)


def test_conv_vs_torch_cpu_fp64(orc):
    rng = np.random.default_rng(1)
    x, w, b = rng.normal(size=(6, 11, 13)), rng.normal(size=(8, 6, 3, 3)), rng.normal(size=8)
    ref = F.conv2d(torch.from_numpy(x)[None], torch.from_numpy(w), torch.from_numpy(b), padding=1)[0].numpy()
    assert np.allclose(orc.conv2d(x, w, b), ref, atol=1e-12)       # cross-correlation, not convolution
    w1 = rng.normal(size=(5, 6, 1, 1))
    assert np.allclose(orc.conv2d(x, w1, None), np.einsum("oc,chw->ohw", w1[:, :, 0, 0], x), atol=1e-12)


def test_conv_delta_and_constant_closed_forms(orc):
    rng = np.random.default_rng(2)
    x = rng.normal(size=(3, 6, 5))
    w = np.zeros((3, 3, 3, 3))
    for c in range(3):
        w[c, c, 1, 1] = 1.0
    assert np.array_equal(orc.conv2d(x, w, np.zeros(3)), x)           # delta kernel = identity
    w = np.zeros((1, 1, 3, 3)); w[0, 0, 0, 2] = 1.0                   # tap (dy=0,dx=2) reads in[y-1, x+1]
    y = orc.conv2d(x[:1], w, None)
    assert np.array_equal(y[0, 1:, :-1], x[0, :-1, 1:]) and not y[0, 0].any() and not y[0, :, -1].any()
    ones = orc.conv2d(np.ones((2, 4, 5)), np.ones((1, 2, 3, 3)), np.array([0.5]))
    assert ones[0, 1, 1] == 18.5 and ones[0, 0, 2] == 12.5 and ones[0, 0, 0] == 8.5   # 9, 6, 4 taps x 2 ch


def test_depthwise_is_diagonal_full_conv(orc):
    rng = np.random.default_rng(3)
    C = 5
    x, w, b = rng.normal(size=(C, 7, 6)), rng.normal(size=(C, 1, 3, 3)), rng.normal(size=C)
    full = np.zeros((C, C, 3, 3))
    for c in range(C):
        full[c, c] = w[c, 0]
    assert np.allclose(orc.dwconv3x3(x, w, b), orc.conv2d(x, full, b), atol=1e-13)
    ref = F.conv2d(torch.from_numpy(x)[None], torch.from_numpy(w), torch.from_numpy(b), padding=1, groups=C)[0]
    assert np.allclose(orc.dwconv3x3(x, w, b), ref.numpy(), atol=1e-13)


@pytest.mark.parametrize("r", [2, 4])
def test_pixel_shuffle_formula_bijection_library(orc, r):
    C, H, W = 3, 4, 5
    x = np.arange(C * r * r * H * W, dtype=np.float64).reshape(C * r * r, H, W)      # iota
    y = orc.pixel_shuffle(x, r)
    assert y.shape == (C, H * r, W * r)
    for c, yy, xx, i, j in [(0, 0, 0, 0, 0), (1, 2, 3, 1, 0), (2, 3, 4, r - 1, r - 1), (1, 0, 4, 0, 1)]:
        assert y[c, r * yy + i, r * xx + j] == x[c * r * r + i * r + j, yy, xx]      # R14
    assert sorted(y.ravel()) == sorted(x.ravel())                                    # bijection
    assert np.array_equal(y, F.pixel_shuffle(torch.from_numpy(x)[None], r)[0].numpy())
    inv = F.pixel_unshuffle(torch.from_numpy(y)[None], r)[0].numpy()
    assert np.array_equal(inv, x)


def test_gelu_relu(orc):
    v = np.linspace(-6, 6, 2001)
    g = orc.gelu(v)
    assert g[1000] == 0.0
    assert np.allclose(g - g[::-1], v, atol=1e-14)                    # GELU(v) - GELU(-v) = v
    assert np.allclose(g, F.gelu(torch.from_numpy(v)).numpy(), atol=1e-14)           # erf form, not tanh
    assert abs(orc.gelu(np.array([1.0]))[0] - 0.5 * (1 + math.erf(1 / math.sqrt(2)))) < 1e-15
    assert np.array_equal(orc.relu(np.array([-1.0, 0.0, 2.0])), [0.0, 0.0, 2.0])


def _tiny_inputs():
    cfg = synth.CONFIGS[1]
    return cfg, synth.make_weights(cfg), synth.make_z(cfg), synth.make_uniform16(cfg)


def test_head_split_and_shuffle_by_hand(orc):
    # O2: channel c*16+4i+j of the head conv at z-pixel (y,x) lands at latent (4y+i, 4x+j), channel c;
    # first C_y channels are mu.  Build a head whose output is its own channel index and read it back.
    cfg, wts, z, _ = _tiny_inputs()
    w = {k: v.copy() for k, v in wts.items()}
    w["hyper.2.w"][:] = 0
    w["hyper.2.b"] = np.arange(2 * cfg.c_y * 16) / 1024.0      # exact in fp32
    mu, u, idx = oracle.entropy_params(orc, cfg, w, z[0])
    for c, i, j in [(0, 0, 0), (5, 2, 3), (31, 3, 3)]:
        assert mu[c, i, j] == (c * 16 + 4 * i + j) / 1024.0
        raw = ((cfg.c_y + c) * 16 + 4 * i + j) / 1024.0
        assert u[c, i, j] == min(max(raw, math.log(cfg.scale_min)), math.log(cfg.scale_max))


def test_head_crop_when_latent_is_not_a_multiple_of_4(orc):
    """R2: h_z = ceil(h/4), w_z = ceil(w/4); the head is shuffled x4 to [4 h_z, 4 w_z] and cropped TOP-LEFT to [h, w].
    160x224 padded frame: h = 10, w = 14, h_z = 3, w_z = 4 (shuffled map 12 x 16, two rows and two columns dropped).
    z carries a position code through pass-through convs, the head adds its own channel number, so every element of
    mu / u has a value known by hand: code(zy, zx) + (c 16 + 4 i + j) / 1024 at latent (4 zy + i, 4 zx + j)."""
    cfg = synth.crop_config(synth.CONFIGS[1], 150, 200)
    g = oracle.geometry(cfg)
    assert (g["h"], g["w"], g["h_z"], g["w_z"]) == (10, 14, 3, 4)
    w = {k: np.zeros_like(v) for k, v in synth.make_weights(cfg).items()}
    for name in ("hyper.0.w", "hyper.1.w"):
        w[name][0, 0, 1, 1] = 1.0                                # centre tap, channel 0 -> channel 0
    w["hyper.2.w"][:, 0, 1, 1] = 1.0
    n_head = 2 * cfg.c_y * 16
    w["hyper.2.b"] = np.arange(n_head) / 1024.0
    z = np.zeros((cfg.c_z, 3, 4), np.int16)
    z[0] = np.arange(12).reshape(3, 4)                           # non-negative: ReLU passes it
    mu, u, idx = oracle.entropy_params(orc, cfg, w, z)
    assert mu.shape == (cfg.c_y, 10, 14) and u.shape == mu.shape and idx.shape == mu.shape
    lo, hi = math.log(cfg.scale_min), math.log(cfg.scale_max)
    for c in (0, 7, cfg.c_y - 1):
        for ly in range(10):
            for lx in range(14):
                code = (ly // 4) * 4 + lx // 4
                sub = 4 * (ly % 4) + lx % 4
                assert mu[c, ly, lx] == code + (c * 16 + sub) / 1024.0
                raw = code + ((cfg.c_y + c) * 16 + sub) / 1024.0
                assert u[c, ly, lx] == min(max(raw, lo), hi)
    # the dropped rows / columns are the BOTTOM / RIGHT ones: the last kept row is latent row 9 = (zy 2, i 1)
    assert mu[0, 9, 13] == (2 * 4 + 3) + (4 * 1 + 1) / 1024.0


def test_trunk_block_identity_when_w2_zero(orc):
    cfg = synth.crop_config(synth.CONFIGS[2], 32, 48)
    wts = synth.make_weights(cfg)
    for k in range(cfg.n_trunk_blocks):
        wts[f"trunk.{k}.pw2.w"][:] = 0
        wts[f"trunk.{k}.pw2.b"][:] = 0
    y = np.random.default_rng(0).normal(size=(cfg.c_y, cfg.h, cfg.w))
    _, taps = oracle.synthesis(orc, cfg, wts, y, keep=True)
    assert np.array_equal(taps["trunk"][0], taps["F0"][0])


def test_identical_decoders_give_identical_frames(orc):
    cfg, wts, z, u16 = _tiny_inputs()
    w = dict(wts)
    ct = cfg.c_trunk
    w["xframe.w"] = np.concatenate([wts["xframe.w"][:ct]] * cfg.T)
    w["xframe.b"] = np.concatenate([wts["xframe.b"][:ct]] * cfg.T)
    for s in range(4):
        for t in range(1, cfg.T):
            w[f"dec.{t}.{s}.w"], w[f"dec.{t}.{s}.b"] = w[f"dec.0.{s}.w"], w[f"dec.0.{s}.b"]
    st = oracle.make_stream(orc, cfg, w, z[0], u16[0])
    out = oracle.chunk_decode(orc, cfg, w, z[0], st["bits"], st["sub_off"])
    assert out["status"] == 0 and np.array_equal(out["frames"][0], out["frames"][1])
    out2 = oracle.chunk_decode(orc, cfg, wts, z[0], st["bits"], st["sub_off"])
    assert not np.array_equal(out2["frames"][0], out2["frames"][1])   # distinct weights -> distinct frames


def test_shift_equivariance_interior(orc):
    # fully convolutional synthesis: shifting y by one latent pixel shifts the frame interior by 16 px
    cfg = synth.crop_config(synth.CONFIGS[1], 160, 160)
    wts = synth.make_weights(cfg)
    rng = np.random.default_rng(4)
    y = rng.normal(size=(cfg.c_y, cfg.h, cfg.w))
    y2 = np.zeros_like(y); y2[:, :, 1:] = y[:, :, :-1]
    f1, _ = oracle.synthesis(orc, cfg, wts, y)
    f2, _ = oracle.synthesis(orc, cfg, wts, y2)
    m = 48     # receptive-field margin in pixels: (1 + 1/2 + 1/4 + 1/8 latent px) * 16 < 32, +16 for the shift
    assert np.allclose(f2[:, :, m:-m, m + 16:-m], f1[:, :, m:-m, m:-m - 16], atol=1e-12)


def test_end_to_end_tiny_round_trip_and_fp32_vs_fp64(orc, orc32):
    cfg, wts, z, u16 = _tiny_inputs()
    st = oracle.make_stream(orc, cfg, wts, z[0], u16[0])
    out = oracle.chunk_decode(orc, cfg, wts, z[0], st["bits"], st["sub_off"])
    assert out["status"] == 0 and np.array_equal(out["sym"], st["sym"])
    assert np.array_equal(out["yhat"], st["sym"] + st["mu"])           # O5
    f = out["frames"]
    assert f.shape == (cfg.T, 3, cfg.height, cfg.width) and f.min() >= 0 and f.max() <= 1
    o32 = oracle.chunk_decode(orc32, cfg, wts, z[0], st["bits"], st["sub_off"], idx_override=st["idx"])
    assert np.array_equal(o32["sym"], st["sym"])
    assert np.abs(o32["frames"] - f).max() <= 1e-4                     # bounds the fp32 variant's own error
    assert np.abs(o32["mu"] - st["mu"]).max() <= 1e-4


def test_fp32_oracle_vs_fp64_on_a_config2_crop_with_trunk(orc, orc32):
    """SURVEY.md 8c "fp32 oracle vs an fp64 run of the same loops <= 1e-4 on configs 1-2": the plain-fp32 build that
    BASELINE.json names, against the fp64 build the parity tests use as truth (R12/R24), on config 2's layer
    plan (bf16 weights, 4 trunk blocks, 256 -> 3 decoders) at a 96 x 64 crop.  Indices are teacher-forced (the bucket
    decision is taken in fp64 by definition, R12), so the comparison is about the arithmetic of O5..O9 only."""
    cfg = synth.crop_config(synth.CONFIGS[2], 64, 96)
    wts, z, u16 = synth.make_weights(cfg), synth.make_z(cfg), synth.make_uniform16(cfg)
    st = oracle.make_stream(orc, cfg, wts, z[0], u16[0])
    a = oracle.chunk_decode(orc, cfg, wts, z[0], st["bits"], st["sub_off"], keep=True)
    b = oracle.chunk_decode(orc32, cfg, wts, z[0], st["bits"], st["sub_off"], idx_override=st["idx"], keep=True)
    assert a["status"] == 0 and b["status"] == 0 and np.array_equal(a["sym"], b["sym"])
    assert np.abs(b["mu"] - a["mu"]).max() <= 1e-4
    assert (b["idx"] == a["idx"]).all()
    for t in range(cfg.T):
        assert np.abs(b["taps"]["trunk"][t] - a["taps"]["trunk"][t]).max() <= 1e-4 * max(1.0, np.abs(a["taps"]["trunk"][t]).max())
    assert np.abs(b["frames"] - a["frames"]).max() <= 1e-4
