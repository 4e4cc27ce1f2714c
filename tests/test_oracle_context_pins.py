"""Pins for the oracle's temporal chunk context (SURVEY.md 8f NEXT-2a, R23).

The structure the text fixes: F_i is propagated to form the next context; the chunk decoder and the prior are
conditioned on C_i; context generation is a stack of DC blocks.  What the text leaves open (where C_i enters, the fold)
is reading R23.  The pins check the reading's own formulas against explicit loops and matrix products, the reductions
that must hold whatever the weights are (zero context weights = the context-free path bit for bit; chunk i+1 depends on
chunk i only through C), and the state's data format (bf16-representable).  Fidelity to the paper's trained context net:
parity unpinned (no weights, Fig. 3 is an image).
"""
import dataclasses

import numpy as np
import pytest

import oracle
from paper_2606_04410_b200 import synth


def tiny():
    # config 1's layer plan (no trunk, fp32 weights) on a 96 x 160 frame: h = 6, w = 10, h_z = 2, w_z = 3 (ragged 4 x 4 pooling)
    cfg = synth.context_config(synth.crop_config(synth.CONFIGS[1], 96, 160), 2)
    return cfg, synth.make_weights(cfg), synth.make_z(cfg)[0], synth.make_uniform16(cfg)[0]


def test_context_prior_by_explicit_loops(orc):
    cfg, w, _, _ = tiny()
    g = oracle.geometry(cfg)
    assert (g["h"], g["w"], g["h_z"], g["w_z"]) == (6, 10, 2, 3)
    rng = np.random.default_rng(0)
    ctx = rng.normal(size=(cfg.c_trunk, g["h"], g["w"]))
    q = oracle.context_prior(orc, cfg, w, ctx)
    wp, bp = w["ctx.prior.w"].astype(np.float64), w["ctx.prior.b"].astype(np.float64)
    for (o, zy, zx) in [(0, 0, 0), (5, 1, 2), (cfg.c_hyper - 1, 1, 0), (7, 0, 2)]:
        acc = bp[o]
        for k in range(cfg.c_trunk):
            pool = 0.0
            for i in range(4):
                for j in range(4):
                    y, x = 4 * zy + i, 4 * zx + j
                    if y < g["h"] and x < g["w"]:                 # past the latent's edge: zeros, still divided by 16
                        pool += ctx[k, y, x]
            acc += wp[o, k, 0, 0] * pool / 16.0
        assert abs(q[o, zy, zx] - max(acc, 0.0)) < 1e-12
    # zero context: q = ReLU(b_p) everywhere (closed form)
    q0 = oracle.context_prior(orc, cfg, w, oracle.zero_context(cfg))
    assert np.array_equal(q0, np.broadcast_to(np.maximum(bp, 0.0)[:, None, None], q0.shape))


def test_context_generation_fold_is_a_matrix_product_and_state_is_bf16(orc):
    cfg, w, _, _ = tiny()
    g = oracle.geometry(cfg)
    rng = np.random.default_rng(1)
    feats = [rng.normal(size=(cfg.c_trunk, g["h"], g["w"])) for _ in range(cfg.T)]
    # no DC blocks, identity output conv: C = bf16(fold), and the fold over the T stacked features is one matmul
    cfg0 = dataclasses.replace(cfg, n_ctx_blocks=1)
    w0 = dict(w)
    w0["ctx.0.pw2.w"] = np.zeros_like(w["ctx.0.pw2.w"]); w0["ctx.0.pw2.b"] = np.zeros_like(w["ctx.0.pw2.b"])   # block = identity
    w0["ctx.out.w"] = np.eye(cfg.c_trunk, dtype=np.float32)[:, :, None, None]; w0["ctx.out.b"] = np.zeros(cfg.c_trunk, np.float32)
    c = oracle.context_generation(orc, cfg0, w0, feats)
    stacked = np.concatenate(feats, axis=0).reshape(cfg.T * cfg.c_trunk, -1)
    want = w["ctx.fold.w"][:, :, 0, 0].astype(np.float64) @ stacked + w["ctx.fold.b"].astype(np.float64)[:, None]
    assert np.array_equal(c.reshape(cfg.c_trunk, -1), oracle.round_bf16(want))
    assert not (np.ascontiguousarray(c, np.float32).view(np.uint32) & 0xFFFF).any()       # bf16-representable
    # frame order matters: feature t meets columns [t C_t, (t+1) C_t) of the fold
    c_swapped = oracle.context_generation(orc, cfg0, w0, feats[::-1])
    assert not np.array_equal(c, c_swapped)
    # the full module: a DC block is O7's block (checked in test_oracle_layer_pins); here: blocks with W2 = 0 are identities
    wz = dict(w)
    for k in range(cfg.n_ctx_blocks):
        wz[f"ctx.{k}.pw2.w"] = np.zeros_like(w[f"ctx.{k}.pw2.w"]); wz[f"ctx.{k}.pw2.b"] = np.zeros_like(w[f"ctx.{k}.pw2.b"])
    a = oracle.context_generation(orc, cfg, wz, feats)
    b = oracle.round_bf16(orc.conv2d(want.reshape(cfg.c_trunk, g["h"], g["w"]), w["ctx.out.w"], w["ctx.out.b"]))
    assert np.array_equal(a, b)


def test_round_bf16_is_nearest_even():
    x = np.array([1.0, 1.0 + 2.0 ** -8, 1.0 + 2.0 ** -7, 1.0 + 3 * 2.0 ** -8, -2.5, 0.0, 3.0e-3])
    r = oracle.round_bf16(x)
    assert r[0] == 1.0 and r[1] == 1.0 and r[2] == 1.0 + 2.0 ** -7 and r[3] == 1.0 + 2.0 ** -6     # ties go to the even mantissa
    assert r[4] == -2.5 and r[5] == 0.0 and abs(r[6] - 3.0e-3) <= 3.0e-3 * 2.0 ** -8


def test_zero_context_weights_reduce_to_the_context_free_path(orc):
    """xframe's context columns = 0, prior branch W_p = 0 and b_p = 0  =>  every output of the context-free decode, bit
    for bit (and the context still evolves without influencing anything)."""
    cfg, w, z, u16 = tiny()
    base = dataclasses.replace(cfg, n_ctx_blocks=0)
    wb = {k: v for k, v in w.items() if not k.startswith("ctx.")}
    wb["xframe.w"] = w["xframe.w"][:, :cfg.c_y].copy()
    w0 = dict(w)
    w0["xframe.w"] = w["xframe.w"].copy(); w0["xframe.w"][:, cfg.c_y:] = 0
    w0["ctx.prior.w"] = np.zeros_like(w["ctx.prior.w"]); w0["ctx.prior.b"] = np.zeros_like(w["ctx.prior.b"])
    st = oracle.make_stream(orc, base, wb, z, u16)
    ref = oracle.chunk_decode(orc, base, wb, z, st["bits"], st["sub_off"])
    ctx = np.random.default_rng(2).normal(size=oracle.zero_context(cfg).shape)
    out = oracle.chunk_decode(orc, cfg, w0, z, st["bits"], st["sub_off"], ctx=ctx)
    assert out["status"] == 0
    for k in ("mu", "u", "idx", "sym", "yhat", "frames"):
        assert np.array_equal(out[k], ref[k]), k
    assert "ctx_next" in out and np.abs(out["ctx_next"]).max() > 0


def test_chunk_i_plus_1_depends_on_chunk_i_only_through_the_context(orc):
    cfg, w, z, u16 = tiny()
    zs = [z, np.roll(z, 1, axis=0), np.roll(z, 2, axis=0)]
    ctx, streams = None, []
    for zi in zs:                                            # an encoder's view: each stream is made under the running context
        st = oracle.make_stream(orc, cfg, w, zi, u16, ctx=ctx)
        out = oracle.chunk_decode(orc, cfg, w, zi, st["bits"], st["sub_off"], ctx=ctx)
        streams.append((st["bits"], st["sub_off"]))
        ctx = out["ctx_next"]
    outs = oracle.chunk_decode_sequence(orc, cfg, w, zs, streams)
    assert all(o["status"] == 0 for o in outs)
    assert not outs[0]["ctx"].any() and np.array_equal(outs[1]["ctx"], outs[0]["ctx_next"])
    # chunk 2 decoded on its own from (z_2, bytes_2, C_2) equals chunk 2 of the sequence: nothing else crosses over
    alone = oracle.chunk_decode(orc, cfg, w, zs[2], *streams[2], ctx=outs[2]["ctx"])
    for k in ("idx", "sym", "frames", "ctx_next"):
        assert np.array_equal(alone[k], outs[2][k]), k
    # the context does matter: the same bytes under the zero context decode to something else (different sigma -> the
    # arithmetic decoder desynchronises; the end-state check reports it)
    wrong = oracle.chunk_decode(orc, cfg, w, zs[2], *streams[2], ctx=None)
    assert (wrong["idx"] != outs[2]["idx"]).any()
    assert wrong["status"] != 0 or not np.array_equal(wrong["sym"], outs[2]["sym"])
    # and frames of successive chunks differ although the weights are shared
    assert not np.array_equal(outs[0]["frames"], outs[1]["frames"])


def test_context_stays_bounded_over_a_long_sequence(orc):
    """The synthetic gains (synth.make_weights) must not let the recurrence C -> F -> C blow up: 10 chunks, the context's
    second moment stays O(1)."""
    cfg, w, z, u16 = tiny()
    ctx, m2 = None, []
    for i in range(10):
        zi = np.roll(z, i, axis=0)
        st = oracle.make_stream(orc, cfg, w, zi, u16, ctx=ctx)
        out = oracle.chunk_decode(orc, cfg, w, zi, st["bits"], st["sub_off"], ctx=ctx)
        assert out["status"] == 0
        ctx = out["ctx_next"]
        m2.append(float(np.square(ctx).mean()))
    assert max(m2) < 10.0 and m2[-1] < 2.0 * m2[4] + 1e-9, m2
