"""Pins for the oracle's hyper-latent entropy coding (R22).

decode_z is the already-pinned O4 decoder (tests/test_oracle_entropy_pins.py) with the table chosen per CHANNEL, so
the pins here are about that choice and about the container: hand-computed bucket indices, the index each symbol
of the stream actually used (checked against a scalar decoder written here), the ideal code length of the
factorised prior, round trips at every config's hyper-latent size, and corruption handling.
"""
import dataclasses
import math

import numpy as np
import pytest

import oracle
from paper_2606_04410_b200 import synth


def case(cfg, seed=0):
    w = synth.make_weights(cfg)
    z = synth.make_z(cfg)[0]
    return w, z


def test_prior_index_by_hand(orc):
    """O2's rule on three scales whose bucket is known without arithmetic: the two ends of the table and the level
    value of bucket 32 (ln sigma_k = ln s_min + k (ln s_max - ln s_min) / 63)."""
    cfg = synth.CONFIGS[1]
    lo, hi = math.log(cfg.scale_min), math.log(cfg.scale_max)
    ln = np.array([lo, hi, lo + 32 * (hi - lo) / 63, lo - 1.0, hi + 1.0, lo + 32.4 * (hi - lo) / 63, lo + 32.6 * (hi - lo) / 63])
    idx = oracle.z_prior_index(orc, cfg, {"zprior.lnscale": ln})
    assert idx.tolist() == [0, 63, 32, 0, 63, 32, 33]


@pytest.mark.parametrize("n", [1, 2, 3, 5])
def test_round_trip_every_config_size(orc, n):
    cfg = synth.CONFIGS[n] if n != 5 else synth.crop_config(synth.CONFIGS[5], 1088, 1920)
    w, z = case(cfg)
    cdf = orc.build_cdf(cfg.n_buckets, cfg.scale_min, cfg.scale_max)
    bits, off = oracle.encode_z(orc, cfg, cdf, w, z)
    zg = oracle.z_geometry(cfg)
    assert off.size == zg["n_sub_z"] + 1 and off[0] == 0 and off[-1] == bits.size and not (off % 4).any()
    z2, st = oracle.decode_z(orc, cfg, cdf, w, bits, off)
    assert st == 0 and np.array_equal(z2, z)


def test_code_length_is_the_factorised_prior(orc):
    """The stream is as long as -sum log2 P_c(z) under the per-channel tables, plus the fixed cost of the container
    (a 32-bit final state and at most one more 16-bit word per lane, 8 header bytes per warp-stream)."""
    cfg = synth.CONFIGS[3]
    w, z = case(cfg)
    cdf = orc.build_cdf(cfg.n_buckets, cfg.scale_min, cfg.scale_max)
    bits, off = oracle.encode_z(orc, cfg, cdf, w, z)
    idx_c = oracle.z_prior_index(orc, cfg, w)
    ideal = 0.0
    for c in range(cfg.c_z):
        f = np.diff(cdf[idx_c[c]].astype(np.int64))                   # 255 frequencies, symbol r at position r + 127
        ideal += float(-np.log2(f[z[c].ravel().astype(np.int64) + 127] / 65536.0).sum())
    zg = oracle.z_geometry(cfg)
    lanes = zg["n_sub_z"] * cfg.lanes_per_substream
    assert ideal / 8 <= bits.size <= ideal / 8 + lanes * (4 + 2) + zg["n_sub_z"] * (cfg.lanes_per_substream // 32) * 8 + 64
    # and a WRONG prior costs more: every channel two buckets narrower
    w2 = dict(w); w2["zprior.lnscale"] = w["zprior.lnscale"] - 0.5
    bits2, _ = oracle.encode_z(orc, cfg, cdf, w2, z)
    assert bits2.size > bits.size


def test_table_of_each_symbol_is_its_channel(orc):
    """Decode lane streams with a scalar decoder written here, choosing the table by (stream position mod C_z):
    stream order is (row, col, channel), so position i of a substream belongs to channel i mod C_z."""
    cfg = dataclasses.replace(synth.CONFIGS[1], lanes_per_substream=32)
    w, z = case(cfg)
    w["zprior.lnscale"] = np.linspace(math.log(0.3), math.log(6.0), cfg.c_z).astype(np.float32)   # distinct tables
    cdf = orc.build_cdf(cfg.n_buckets, cfg.scale_min, cfg.scale_max)
    bits, off = oracle.encode_z(orc, cfg, cdf, w, z)
    idx_c = oracle.z_prior_index(orc, cfg, w)
    assert len(set(idx_c.tolist())) > 8
    zg = oracle.z_geometry(cfg)
    assert zg["n_sub_z"] == 1
    n = cfg.c_z * zg["h_z"] * zg["w_z"]
    # container of a substream: per warp-stream (offset, n_words), then 32 states + words
    ws_off, nw = np.frombuffer(bits[:8].tobytes(), np.uint32)
    states = np.frombuffer(bits[ws_off:ws_off + 128].tobytes(), np.uint32).astype(np.int64).copy()
    words = np.frombuffer(bits[ws_off + 128:ws_off + 128 + 2 * nw].tobytes(), np.uint16).astype(np.int64)
    q, got = 0, []
    for i in range(n):
        lane = i % 32
        c = cdf[idx_c[i % cfg.c_z]].astype(np.int64)
        slot = states[lane] & 0xFFFF
        pos = int(np.searchsorted(c, slot, side="right") - 1)
        got.append(pos - 127)
        states[lane] = (c[pos + 1] - c[pos]) * (states[lane] >> 16) + slot - c[pos]
        if i % 32 == 31 or i == n - 1:                                 # renormalise the step's lanes in lane order
            for l in range(i - (i % 32), i + 1):
                if states[l % 32] < (1 << 16):
                    states[l % 32] = (states[l % 32] << 16) | words[q]
                    q += 1
    want = np.transpose(z, (1, 2, 0)).ravel()
    assert got == want.tolist() and q == nw and (states == 1 << 16).all()


def test_corruption_sets_status(orc):
    cfg = synth.CONFIGS[2]
    w, z = case(cfg)
    cdf = orc.build_cdf(cfg.n_buckets, cfg.scale_min, cfg.scale_max)
    bits, off = oracle.encode_z(orc, cfg, cdf, w, z)
    bad = bits.copy(); bad[bits.size // 2] ^= 0x5A
    _, st = oracle.decode_z(orc, cfg, cdf, w, bad, off)
    assert st != 0
    _, st = oracle.decode_z(orc, cfg, cdf, w, bits[:-8], np.minimum(off, bits.size - 8))
    assert st != 0


def test_bytes_only_chunk_equals_the_z_in_call(orc):
    cfg = synth.CONFIGS[1]
    w, z = case(cfg)
    u16 = synth.make_uniform16(cfg)[0]
    cdf = orc.build_cdf(cfg.n_buckets, cfg.scale_min, cfg.scale_max)
    zb, zo = oracle.encode_z(orc, cfg, cdf, w, z)
    ys = oracle.make_stream(orc, cfg, w, z, u16)
    bits, off = oracle.pack_chunk_bytes(zb, zo, ys["bits"], ys["sub_off"])
    assert off.size == oracle.z_geometry(cfg)["n_sub_z"] + oracle.geometry(cfg)["n_sub"] + 1 and off[-1] == bits.size
    a = oracle.chunk_decode_bytes(orc, cfg, w, bits, off)
    b = oracle.chunk_decode(orc, cfg, w, z, ys["bits"], ys["sub_off"])
    assert a["status"] == 0 and np.array_equal(a["z"], z) and np.array_equal(a["sym"], b["sym"])
    assert np.array_equal(a["frames"], b["frames"])
