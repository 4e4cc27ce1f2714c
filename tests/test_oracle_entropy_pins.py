"""Pins for the oracle's entropy model (O2, O3, O4) against things other than itself."""
import math
import os

import numpy as np
import pytest
from scipy.stats import norm

NB, SMIN, SMAX = 64, 0.11, 20.0
GOLD = os.path.join(os.path.dirname(__file__), "golden")


@pytest.fixture(scope="module")
def cdf(orc):
    return orc.build_cdf(NB, SMIN, SMAX)


def test_cdf_invariants(cdf):
    assert cdf.shape == (NB, 256)
    assert (cdf[:, 0] == 0).all() and (cdf[:, 255] == 1 << 16).all()       # sums to 2^16
    freq = np.diff(cdf.astype(np.int64), axis=1)
    assert freq.shape == (NB, 255) and (freq >= 1).all()
    assert (freq.sum(axis=1) == 1 << 16).all()
    assert freq.max() == 65282 and freq.max() < 1 << 16                    # f * 2^16 fits the 32-bit compare (R6)


def test_cdf_golden_sigma_min(cdf):
    for line in open(os.path.join(GOLD, "cdf_sigma_min.txt")):
        if line.startswith("#"):
            continue
        p, c = map(int, line.split())
        assert cdf[0, p] == c


def test_cdf_matches_double_precision_gaussian(cdf):
    # independent route: scipy's normal CDF (not erfc), pmf of the discretised Gaussian with folded tails
    for k in (0, 1, 17, 31, 40, 63):
        sigma = SMIN * (SMAX / SMIN) ** (k / 63)
        edges = np.concatenate([[-np.inf], np.arange(-126.5, 127.0, 1.0), [np.inf]])
        pmf = np.diff(norm.cdf(edges / sigma))
        freq = np.diff(cdf[k].astype(np.int64))
        assert np.abs(freq - 1 - (65536 - 255) * pmf).max() <= 1.0 + 1e-6
        assert (freq == freq[::-1]).all() or np.abs(freq - freq[::-1]).max() <= 1   # symmetric law


def test_bucket_levels_midpoints_clamp(orc):
    lo, hi = math.log(SMIN), math.log(SMAX)
    step = (hi - lo) / 63
    levels = lo + step * np.arange(64)
    idx, uc = orc.bucket_index(levels, NB, SMIN, SMAX)
    assert (idx == np.arange(64)).all()
    # just below / above the hand-computed mid-points (half-up rule, R4)
    mids = lo + step * (np.arange(63) + 0.5)
    assert (orc.bucket_index(mids - 1e-9, NB, SMIN, SMAX)[0] == np.arange(63)).all()
    assert (orc.bucket_index(mids + 1e-9, NB, SMIN, SMAX)[0] == np.arange(1, 64)).all()
    idx, uc = orc.bucket_index(np.array([-50.0, lo - 1e-3, hi + 1e-3, 50.0]), NB, SMIN, SMAX)
    assert list(idx) == [0, 0, 63, 63]
    assert np.allclose(uc, [lo, lo, hi, hi])
    u = np.linspace(lo - 1, hi + 1, 10001)
    assert (np.diff(orc.bucket_index(u, NB, SMIN, SMAX)[0].astype(int)) >= 0).all()   # monotone


def test_inverse_cdf_sampling_brute_force(orc, cdf):
    rng = np.random.default_rng(5)
    idx = rng.integers(0, NB, 4000).astype(np.uint8)
    u16 = rng.integers(0, 1 << 16, 4000).astype(np.uint16)
    sym = orc.symbols_from_uniform(cdf, idx, u16)
    for i in range(0, 4000, 7):
        c = cdf[idx[i]]
        p = int(sym[i]) + 127
        assert c[p] <= u16[i] < c[p + 1]


def _random_case(orc, cdf, n, rng, lo_bucket=0, hi_bucket=NB):
    idx = rng.integers(lo_bucket, hi_bucket, n).astype(np.uint8)
    u16 = rng.integers(0, 1 << 16, n).astype(np.uint16)
    return idx, orc.symbols_from_uniform(cdf, idx, u16)


@pytest.mark.parametrize("W,n", [(32, 1), (32, 5), (32, 32), (32, 512), (64, 1000), (128, 61440), (128, 26624),
                                 (128, 13312), (192, 92160), (512, 4097), (32, 33), (512, 61440), (384, 92160)])
def test_rans_round_trip_end_state_and_size(orc, cdf, W, n):
    rng = np.random.default_rng(n * 31 + W)
    idx, sym = _random_case(orc, cdf, n, rng)
    data = orc.rans_encode_substream(cdf, idx, sym, W)
    out, st = orc.rans_decode_substream(cdf, idx, W, data)
    assert st == 0                                   # every lane back at 2^16 and word pointer == count
    assert np.array_equal(out, sym)
    # size vs information content: payload = 32 state bits per USED lane + 16 per word; an rANS coder that
    # starts at 2^16 spends < 32 extra bits per lane and can not beat the entropy by more than its start slack
    G = W // 32
    hdr = data[:8 * G].view(np.uint32).reshape(G, 2)
    used = min(n, W)
    bits = int(hdr[:, 1].sum()) * 16 + 32 * used
    ideal = orc.ideal_bits(cdf, idx, sym)
    assert ideal - 1e-6 <= bits - 16 * used <= ideal + 16 * used + 1e-6


def test_rans_one_symbol_per_lane_closed_form(orc, cdf):
    # n <= 32, W = 32: each lane codes exactly one symbol from x = 2^16, no renormalisation (2^16 < f 2^16):
    # textbook rANS step C(x,s) = floor(x/f) 2^16 + (x mod f) + c  with x = 2^16.
    rng = np.random.default_rng(2)
    idx, sym = _random_case(orc, cdf, 32, rng)
    data = orc.rans_encode_substream(cdf, idx, sym, 32)
    off, nw = data[:8].view(np.uint32)
    assert nw == 0
    states = data[off:off + 128].view(np.uint32)
    for l in range(32):
        c = cdf[idx[l]].astype(np.int64)
        p = int(sym[l]) + 127
        f = c[p + 1] - c[p]
        assert states[l] == (65536 // f) * 65536 + 65536 % f + c[p]


def test_rans_degenerate_all_zero_at_sigma_min(orc, cdf):
    n = 128 * 300
    idx = np.zeros(n, np.uint8)
    sym = np.zeros(n, np.int16)
    data = orc.rans_encode_substream(cdf, idx, sym, 128)
    out, st = orc.rans_decode_substream(cdf, idx, 128, data)
    assert st == 0 and not out.any()
    # 300 symbols/lane at log2(65536/65282) = 0.0056 bit each = 1.7 bits: no lane ever emits a word
    assert data.size == 8 * 4 + 4 * 128


def test_rans_detects_corruption(orc, cdf):
    rng = np.random.default_rng(9)
    idx, sym = _random_case(orc, cdf, 128 * 64, rng)
    data = orc.rans_encode_substream(cdf, idx, sym, 128)
    bad = 0
    trials = 40
    for t in range(trials):
        d = data.copy()
        pos = int(rng.integers(8 * 4, d.size))
        d[pos] ^= 1 << int(rng.integers(0, 8))
        out, st = orc.rans_decode_substream(cdf, idx, 128, d)
        bad += (st != 0)
    assert bad >= trials - 4          # a flipped bit almost surely breaks the end-state invariant
    out, st = orc.rans_decode_substream(cdf, idx, 128, data[:data.size // 2])
    assert st != 0                    # truncated stream: error status, no crash


def test_rans_lanes_are_independent_streams(orc, cdf):
    # interleave pin: changing the symbols of one warp-stream must leave the other warp-streams' bytes alone,
    # and the per-lane symbol subsequence alone determines that lane's start state.
    rng = np.random.default_rng(11)
    W, n = 64, 64 * 50
    idx, sym = _random_case(orc, cdf, n, rng, 20, 64)
    d0 = orc.rans_encode_substream(cdf, idx, sym, W)
    sym2 = sym.copy().reshape(-1, W)
    idx2 = idx.copy().reshape(-1, W)
    sym2[:, 32:] = _random_case(orc, cdf, n // 2, rng, 20, 64)[1].reshape(-1, 32)[:, :32] * 0
    d1 = orc.rans_encode_substream(cdf, idx2.ravel(), sym2.ravel(), W)
    h0, h1 = d0[:16].view(np.uint32), d1[:16].view(np.uint32)
    assert h0[1] == h1[1]
    n0 = 128 + 2 * int(h0[1])
    assert np.array_equal(d0[h0[0]:h0[0] + n0], d1[h1[0]:h1[0] + n0])


def _scalar_lane_decode(cdf, idx, n, W, data):
    """Textbook scalar rANS decoder (x -> (s, x') with x' = f (x >> 16) + slot - c, renormalise by one 16-bit word while
    x < 2^16), written here with Python ints.  It walks the container warp-stream by warp-stream through ITS OWN header
    entry (byte offset, word count) and inside a warp-stream step by step, lanes in ascending order.  Returns the
    symbols, and per warp-stream (words consumed, words present, all lanes back at 2^16)."""
    G = W // 32
    hdr = np.frombuffer(data[:8 * G].tobytes(), np.uint32).reshape(G, 2)
    steps = -(-n // W)
    sym = np.zeros(n, np.int64)
    info = []
    for g in range(G):
        off, nw = int(hdr[g, 0]), int(hdr[g, 1])
        x = [int(v) for v in np.frombuffer(data[off:off + 128].tobytes(), np.uint32)]
        words = np.frombuffer(data[off + 128:off + 128 + 2 * nw].tobytes(), np.uint16)
        q = 0
        for j in range(steps):
            lanes = [l for l in range(32) if j * W + 32 * g + l < n]
            for l in lanes:
                i = j * W + 32 * g + l
                c = cdf[idx[i]]
                slot = x[l] & 0xFFFF
                p = int(np.searchsorted(c, slot, side="right")) - 1
                sym[i] = p - 127
                x[l] = int(c[p + 1] - c[p]) * (x[l] >> 16) + slot - int(c[p])
            for l in lanes:                      # renormalisation reads the words in ascending lane order
                if x[l] < 1 << 16:
                    x[l] = (x[l] << 16) | int(words[q])
                    q += 1
        info.append((q, nw, all(v == 1 << 16 for v in x)))
    return sym, info


@pytest.mark.parametrize("W,n", [(64, 64 * 37 + 5), (512, 512 * 9 + 300), (384, 384 * 7 + 33)])
def test_rans_multi_warp_stream_container_against_scalar_decoder(orc, cdf, W, n):
    """G > 1 warp-streams: every warp-stream owns header entry g, 32 start states and its own word run.  A per-warp-stream
    offset / count mistake that the encoder mirrors would pass a round trip; it cannot pass a decoder written
    separately that reads each header entry itself, nor the non-overlap and coverage checks on the byte ranges."""
    rng = np.random.default_rng(W + n)
    idx, sym = _random_case(orc, cdf, n, rng)
    data = orc.rans_encode_substream(cdf, idx, sym, W)
    got, info = _scalar_lane_decode(cdf, idx, n, W, data)
    assert np.array_equal(got, sym)
    assert all(q == nw and ended for q, nw, ended in info)
    G = W // 32
    hdr = data[:8 * G].view(np.uint32).reshape(G, 2)
    spans = sorted((int(o), int(o) + 128 + 2 * int(c)) for o, c in hdr)
    assert spans[0][0] == 8 * G and spans[-1][1] <= data.size <= spans[-1][1] + 3      # header, then the runs, then pad
    for (a0, a1), (b0, b1) in zip(spans, spans[1:]):
        assert a1 <= b0 <= a1 + 3 and b0 % 4 == 0                                     # disjoint, 4-byte aligned, no holes
    # the oracle's own decoder agrees (status 0) and so does a decode after shuffling the ORDER of the warp-stream
    # runs inside the container (header entries re-pointed): only the header ties a run to its lanes
    out, st = orc.rans_decode_substream(cdf, idx, W, data)
    assert st == 0 and np.array_equal(out, sym)
    perm = rng.permutation(G)
    parts, new_hdr, pos = [], np.zeros((G, 2), np.uint32), 8 * G
    for g in perm:
        o, c = int(hdr[g, 0]), int(hdr[g, 1])
        run = data[o:o + 128 + 2 * c]
        run = np.concatenate([run, np.zeros((-run.size) % 4, np.uint8)])
        new_hdr[g] = (pos, c)
        parts.append(run)
        pos += run.size
    moved = np.concatenate([new_hdr.view(np.uint8).ravel()] + parts)
    out, st = orc.rans_decode_substream(cdf, idx, W, moved)
    assert st == 0 and np.array_equal(out, sym)


def test_rans_other_warp_streams_bytes_change_only_their_own_run(orc, cdf):
    """Replace the symbols of warp-stream 1 (lanes 32..63) by a DIFFERENT random draw: warp-stream 0's states and words are
    unchanged byte for byte, warp-stream 1's differ, and both decode back."""
    rng = np.random.default_rng(12)
    W, n = 64, 64 * 50
    idx, sym = _random_case(orc, cdf, n, rng, 20, 64)
    d0 = orc.rans_encode_substream(cdf, idx, sym, W)
    sym2 = sym.copy().reshape(-1, W)
    sym2[:, 32:] = orc.symbols_from_uniform(cdf, idx.reshape(-1, W)[:, 32:], rng.integers(0, 1 << 16, (n // W, 32)).astype(np.uint16))
    assert (sym2 != sym.reshape(-1, W)).any()
    d1 = orc.rans_encode_substream(cdf, idx, sym2.ravel(), W)
    h0, h1 = d0[:16].view(np.uint32).reshape(2, 2), d1[:16].view(np.uint32).reshape(2, 2)
    assert h0[0, 1] == h1[0, 1]
    n0 = 128 + 2 * int(h0[0, 1])
    assert np.array_equal(d0[h0[0, 0]:h0[0, 0] + n0], d1[h1[0, 0]:h1[0, 0] + n0])
    r0, r1 = d0[h0[1, 0]:h0[1, 0] + 128 + 2 * int(h0[1, 1])], d1[h1[1, 0]:h1[1, 0] + 128 + 2 * int(h1[1, 1])]
    assert r0.size != r1.size or not np.array_equal(r0, r1)
    out, st = orc.rans_decode_substream(cdf, idx, W, d1)
    assert st == 0 and np.array_equal(out, sym2.ravel())
