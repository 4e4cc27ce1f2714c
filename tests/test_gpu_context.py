"""Temporal chunk context on the GPU (SURVEY.md 8f NEXT-2a, R23) against the oracle, through the C ABI.

Two modes, as for the entropy parameters (R12):
  * teacher-forced context: chunk i is decoded under the ORACLE's C_i (ufnvc_set_context; the state is a bf16 tensor, so
    both sides start from identical numbers): indices and symbols bit-exact, pixels and the new context C_{i+1} within
    the bf16-derived bounds;
  * free-running: the handle carries its own state over three calls.  Its C_i differs from the oracle's by bf16 noise, so
    its indices may differ from the oracle's; the stream of chunk i is therefore encoded with the DEVICE's indices, as
    the real codec does (the encoder runs the decoder's prior net) -- with the oracle's residuals r, so the
    frames stay comparable: symbols bit-exact, pixels within the north-star tolerance.
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
N_CHUNKS = 3


@pytest.fixture(scope="module")
def seq():
    """Oracle sequence of three chunks of ONE video on the 1080p layer plan, 480x272 crop, 2 context DC blocks."""
    cfg = synth.context_config(synth.crop_config(synth.CONFIGS[3], 272, 480), 2)
    orc = oracle.Oracle("f64")
    wts = synth.make_weights(cfg)
    z0, u0 = synth.make_z(cfg)[0], synth.make_uniform16(cfg)[0]
    zs = [np.roll(z0, i, axis=1) for i in range(N_CHUNKS)]
    us = [np.roll(u0, 7 * i, axis=0) for i in range(N_CHUNKS)]
    ctx, chunks = None, []
    for z, u16 in zip(zs, us):
        st = oracle.make_stream(orc, cfg, wts, z, u16, ctx=ctx)
        out = oracle.chunk_decode(orc, cfg, wts, z, st["bits"], st["sub_off"], ctx=ctx, keep=False)
        assert out["status"] == 0 and np.array_equal(out["sym"], st["sym"])
        chunks.append(dict(z=z, stream=st, out=out, ctx=oracle.zero_context(cfg) if ctx is None else ctx))
        ctx = out["ctx_next"]
    return dict(cfg=cfg, weights=wts, chunks=chunks, orc=orc)


def dev(a, dt=None):
    t = torch.from_numpy(np.ascontiguousarray(a))
    return (t.to(dt) if dt is not None else t).cuda()


def ctx_to_dev(ctx_chw):
    return dev(nhwc(ctx_chw).astype(np.float32)[None], torch.bfloat16)       # exact: the oracle's state is bf16-representable


def test_teacher_forced_context_chunk_by_chunk(seq):
    from paper_2606_04410_b200 import binding
    cfg = seq["cfg"]
    dec = binding.ChunkDecoder(cfg)
    dec.load_weights(seq["weights"])
    for i, ch in enumerate(seq["chunks"]):
        st, ref = ch["stream"], ch["out"]
        dec.set_context(ctx_to_dev(ch["ctx"]))
        bits, off = binding.concat_streams([(st["bits"], st["sub_off"])])
        out = dec.chunk_decode_ex(dev(ch["z"][None]), dev(bits), dev(off.astype(np.int64), torch.int32), taps=True)
        torch.cuda.synchronize()
        assert dec.get_status() == 0
        assert np.array_equal(out["idx"][0].cpu().numpy(), nhwc(ref["idx"])), f"chunk {i}: indices"
        assert np.array_equal(out["sym"][0].cpu().numpy(), nhwc(ref["sym"])), f"chunk {i}: symbols"
        assert np.abs(out["mu"][0].cpu().numpy() - nhwc(ref["mu"])).max() <= 1e-4
        f = out["frames"][0].cpu().numpy()
        err = float(np.abs(f - ref["frames"]).max())
        assert err <= PIX_TOL and psnr(f, ref["frames"]) >= PSNR_MIN, (i, err)
        # the new state against the oracle's C_{i+1}: bf16 roundings on the path = y, F0, 3 per trunk block, fold, 3 per
        # context block, the state itself
        got = dec.get_context().float().cpu().numpy()[0]
        want = nhwc(ref["ctx_next"])
        L = 2 + 3 * cfg.n_trunk_blocks + 1 + 3 * cfg.n_ctx_blocks + 1
        r = math.sqrt(L) * 2.0 ** -8 / math.sqrt(3.0)
        d = got - want
        rms_e, rms_b = float(np.sqrt(np.mean(d ** 2))), r * float(np.sqrt(np.mean(want ** 2)))
        max_e, max_b = float(np.abs(d).max()), 6.0 * r * max(1.0, float(np.abs(want).max()))
        print(f"chunk {i}: max |d pixel| = {err:.2e}; context rms err / bound = {rms_e / rms_b:.3f}, max err / bound = {max_e / max_b:.3f}")
        assert rms_e <= rms_b and max_e <= max_b
    dec.destroy()


def test_free_running_sequence_self_consistent(seq):
    from paper_2606_04410_b200 import binding
    cfg, orc = seq["cfg"], seq["orc"]
    dec = binding.ChunkDecoder(cfg)
    dec.load_weights(seq["weights"])
    dec.reset_context()
    flips = []
    for i, ch in enumerate(seq["chunks"]):
        ref = ch["out"]
        z = dev(ch["z"][None])
        _, _, idx_dev = dec.entropy_params(z)                      # the prior net under the handle's OWN context
        idx = idx_dev[0].cpu().numpy()
        flips.append(float((idx != nhwc(ref["idx"])).mean()))
        sym = nhwc(ref["sym"])                                     # the oracle's residuals, coded with the device's scales
        b, o = dec.encode_chunk(idx, sym)
        out = dec.chunk_decode_ex(z, dev(b), dev(o.astype(np.int64), torch.int32), taps=True)
        torch.cuda.synchronize()
        assert dec.get_status() == 0
        assert np.array_equal(out["idx"][0].cpu().numpy(), idx)    # entropy_params and the decode see the same state
        assert np.array_equal(out["sym"][0].cpu().numpy(), sym)
        f = out["frames"][0].cpu().numpy()
        err = float(np.abs(f - ref["frames"]).max())
        print(f"chunk {i}: index differences vs oracle {flips[-1]:.2e}, max |d pixel| = {err:.2e}, psnr = {psnr(f, ref['frames']):.1f}")
        assert err <= PIX_TOL and psnr(f, ref["frames"]) >= PSNR_MIN, (i, err)
    assert flips[0] == 0.0                                         # chunk 0: zero context on both sides
    dec.destroy()


def test_reset_set_get_and_determinism(seq):
    from paper_2606_04410_b200 import binding
    cfg = seq["cfg"]
    dec = binding.ChunkDecoder(cfg)
    dec.load_weights(seq["weights"])
    ch0, ch1 = seq["chunks"][0], seq["chunks"][1]
    assert not dec.get_context().any()                             # a fresh handle holds the zero context
    c1 = ctx_to_dev(ch1["ctx"])
    dec.set_context(c1)
    assert torch.equal(dec.get_context(), c1)
    st = ch1["stream"]
    bits, off = binding.concat_streams([(st["bits"], st["sub_off"])])
    args = (dev(ch1["z"][None]), dev(bits), dev(off.astype(np.int64), torch.int32))
    a = dec.chunk_decode(*args).clone()
    ca = dec.get_context().clone()
    dec.set_context(c1)
    b = dec.chunk_decode(*args).clone()
    torch.cuda.synchronize()
    assert torch.equal(a, b) and torch.equal(ca, dec.get_context())          # run-to-run bit-identical, state included
    # a call that stops after the entropy stage leaves the state alone
    dec.set_context(c1)
    dec.chunk_decode_ex(*args, want_frames=False)
    assert torch.equal(dec.get_context(), c1)
    # under the wrong (zero) context the same bytes do not decode: the status word says so, nothing faults
    dec.reset_context()
    assert not dec.get_context().any()
    dec.chunk_decode(*args)
    torch.cuda.synchronize()
    assert dec.get_status() != 0
    # the whole stateful call is CUDA-graph capturable; replaying it advances the state like a direct call
    dec.set_context(c1)
    frames = dec.new_frames(1)
    s = torch.cuda.Stream()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(s):
        g.capture_begin()
        dec.chunk_decode(*args, frames=frames, stream=s)
        g.capture_end()
    dec.set_context(c1)
    torch.cuda.synchronize()
    g.replay()
    torch.cuda.synchronize()
    assert dec.get_status() == 0 and torch.equal(frames, a) and torch.equal(dec.get_context(), ca)
    dec.destroy()


def test_context_api_errors():
    from paper_2606_04410_b200 import binding
    base = synth.crop_config(synth.CONFIGS[3], 272, 480)
    dec = binding.ChunkDecoder(base)
    dec.load_weights(synth.make_weights(base))
    with pytest.raises(binding.UfnvcError, match="-2"):
        dec.reset_context()                                        # no temporal context in this config
    dec.destroy()
    with pytest.raises(binding.UfnvcError, match="-2"):            # needs c_trunk == 256
        binding.ChunkDecoder(dataclasses.replace(synth.CONFIGS[1], n_ctx_blocks=2))
    cfg = synth.context_config(base, 1)
    dec = binding.ChunkDecoder(cfg)
    w = synth.make_weights(cfg)
    w2 = dict(w); del w2["ctx.out.w"]
    with pytest.raises(binding.UfnvcError, match="ctx.out.w"):
        dec.load_weights(w2)
    dec.destroy()
