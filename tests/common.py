"""Shared helpers for the parity tests: build one seeded case with the oracle, run it through the C ABI."""
import functools

import numpy as np

import oracle
from paper_2606_04410_b200 import synth


@functools.lru_cache(maxsize=8)
def oracle_case(cfg, real="f64", keep=True):
    """Everything the oracle says about `cfg`: stream fixture + full decode, per chunk."""
    orc = oracle.Oracle(real)
    wts = synth.make_weights(cfg)
    z = synth.make_z(cfg)
    u16 = synth.make_uniform16(cfg)
    chunks = []
    for n in range(cfg.n_chunks):
        st = oracle.make_stream(orc, cfg, wts, z[n], u16[n])
        out = oracle.chunk_decode(orc, cfg, wts, z[n], st["bits"], st["sub_off"], keep=keep)
        assert out["status"] == 0 and np.array_equal(out["sym"], st["sym"])
        chunks.append(dict(stream=st, out=out))
    return dict(cfg=cfg, weights=wts, z=z, u16=u16, chunks=chunks)


def nhwc(a_chw):
    return np.ascontiguousarray(np.moveaxis(np.asarray(a_chw), 0, -1))


def psnr(a, b):
    mse = float(np.mean((np.asarray(a, np.float64) - np.asarray(b, np.float64)) ** 2))
    return 99.0 if mse == 0 else 10.0 * np.log10(1.0 / mse)


def gpu_inputs(case):
    """Oracle-encoded streams of all chunks -> device tensors for one ufnvc_chunk_decode call."""
    import torch
    from paper_2606_04410_b200 import binding
    bits, off = binding.concat_streams([(c["stream"]["bits"], c["stream"]["sub_off"]) for c in case["chunks"]])
    dev = "cuda"
    return (torch.from_numpy(case["z"]).to(dev), torch.from_numpy(bits).to(dev), torch.from_numpy(off.astype(np.int64)).to(torch.int32).to(dev))
