"""Pins for the oracle's four-step progressive means (R21).

The paper fixes the STRUCTURE (four partitions; the mean of partition k is estimated from the partitions decoded
before it; the residual of every partition is already there; y = r + mu), not the geometry or the net, so the pins
are: the partition table written out by hand, the dependency structure (what may and may not change when one
residual changes), special cases that collapse to the single-step path or to a constant, and a brute-force
re-evaluation on a tiny case that shares no code with the oracle's conv.
"""
import dataclasses

import numpy as np
import pytest

import oracle
from paper_2606_04410_b200 import synth


def tiny_cfg(c_y=8, h=6, w=8):
    base = synth.progressive_config(synth.CONFIGS[1])
    return dataclasses.replace(base, c_y=c_y, height=h * 16, width=w * 16)


def random_case(cfg, seed):
    rng = np.random.default_rng(seed)
    g = oracle.geometry(cfg)
    wts = {}
    for k in (1, 2, 3):
        wts[f"mu.{k}.w"] = rng.normal(0, 0.1, size=(cfg.c_y, 2 * cfg.c_y, 3, 3))
        wts[f"mu.{k}.b"] = rng.normal(0, 0.1, size=cfg.c_y)
    mu0 = rng.normal(size=(cfg.c_y, g["h"], g["w"]))
    sym = rng.integers(-5, 6, size=(cfg.c_y, g["h"], g["w"])).astype(np.int16)
    return wts, mu0, sym


def test_partition_table_by_hand():
    """R21 for C_y = 4, one 2x2 cell: channel c is its own group, k = (2y + x + c) mod 4."""
    by_hand = np.array([[[0, 1], [2, 3]],      # c = 0
                        [[1, 2], [3, 0]],      # c = 1
                        [[2, 3], [0, 1]],      # c = 2
                        [[3, 0], [1, 2]]])     # c = 3
    assert np.array_equal(oracle.partition_index(4, 2, 2), by_hand)


@pytest.mark.parametrize("c_y,h,w", [(8, 4, 6), (32, 4, 4), (12, 5, 7)])
def test_partition_invariants(c_y, h, w):
    part = oracle.partition_index(c_y, h, w)
    assert part.min() == 0 and part.max() == 3
    cg = c_y // 4
    # quadtree-like: inside one 2x2 cell every channel sees each step once, and at one position the four channel
    # groups sit in four different steps, so every step holds a quarter of every full cell and of every pixel
    for y0 in range(0, h - 1, 2):
        for x0 in range(0, w - 1, 2):
            cell = part[:, y0:y0 + 2, x0:x0 + 2].reshape(c_y, 4)
            assert all(sorted(row) == [0, 1, 2, 3] for row in cell)
    for y in range(h):
        for x in range(w):
            assert sorted(part[::cg, y, x]) == [0, 1, 2, 3]
            assert all(len(set(part[g * cg:(g + 1) * cg, y, x])) == 1 for g in range(4))
    # the pattern has period 2 in both directions
    assert np.array_equal(part[:, 2:, :], part[:, :-2, :]) and np.array_equal(part[:, :, 2:], part[:, :, :-2])


def test_zero_weights_give_the_bias(orc):
    """W_k = 0: mu^k = b_k, so y = r + mu0 on partition 0 and r + b_k[c] on partition k."""
    cfg = tiny_cfg()
    wts, mu0, sym = random_case(cfg, 1)
    for k in (1, 2, 3):
        wts[f"mu.{k}.w"][:] = 0.0
    yhat, mu = oracle.progressive_means(orc, cfg, wts, mu0, sym)
    part = oracle.partition_index(cfg.c_y, *mu0.shape[1:])
    want = np.where(part == 0, mu0, 0.0)
    for k in (1, 2, 3):
        want = np.where(part == k, wts[f"mu.{k}.b"][:, None, None], want)
    assert np.array_equal(mu, want) and np.array_equal(yhat, sym + want)


def test_passing_mu0_through_collapses_to_the_single_step_path(orc):
    """W_k = centre-tap identity on the mu0 half of the input, b = 0: every mean is mu0 and y = r + mu0 (O5)."""
    cfg = tiny_cfg()
    wts, mu0, sym = random_case(cfg, 2)
    for k in (1, 2, 3):
        wts[f"mu.{k}.w"][:] = 0.0
        wts[f"mu.{k}.b"][:] = 0.0
        for c in range(cfg.c_y):
            wts[f"mu.{k}.w"][c, cfg.c_y + c, 1, 1] = 1.0
    yhat, mu = oracle.progressive_means(orc, cfg, wts, mu0, sym)
    assert np.array_equal(mu, mu0) and np.array_equal(yhat, sym + mu0)


def test_input_order_and_mask(orc):
    """Step 1 reads [y so far ; mu0]: a centre tap on input channel j < C_y returns the partition-0 part of r + mu0 of
    channel j and ZERO where channel j is not decoded yet; the same tap at step 2 also sees partition 1."""
    cfg = tiny_cfg()
    wts, mu0, sym = random_case(cfg, 3)
    part = oracle.partition_index(cfg.c_y, *mu0.shape[1:])
    j = 5
    for k in (1, 2, 3):
        wts[f"mu.{k}.w"][:] = 0.0
        wts[f"mu.{k}.b"][:] = 0.0
    wts["mu.1.w"][:, j, 1, 1] = 1.0
    wts["mu.2.w"][:, j, 1, 1] = 1.0
    yhat, mu = oracle.progressive_means(orc, cfg, wts, mu0, sym)
    y0_j = np.where(part[j] == 0, sym[j] + mu0[j], 0.0)
    for c in range(cfg.c_y):
        assert np.array_equal(mu[c][part[c] == 1], y0_j[part[c] == 1])
    # channel j's own partition-1 mean is y0_j there, which is 0 (partition 1 of channel j is not partition 0)
    y01_j = np.where(part[j] == 1, sym[j] + 0.0, y0_j)
    for c in range(cfg.c_y):
        assert np.array_equal(mu[c][part[c] == 2], y01_j[part[c] == 2])
    assert not mu[part == 3].any()                    # step 3 has zero weights and zero bias


def test_dependency_structure(orc):
    """Changing ONE residual of partition k leaves every mean of partitions <= k untouched, and moves the means of
    partition k + j only inside a (2j + 1)^2 window around it (3x3 receptive field per step)."""
    cfg = tiny_cfg(c_y=8, h=10, w=12)
    wts, mu0, sym = random_case(cfg, 4)
    part = oracle.partition_index(cfg.c_y, *mu0.shape[1:])
    _, mu_a = oracle.progressive_means(orc, cfg, wts, mu0, sym)
    for k in range(4):
        c, y, x = next((c, y, x) for c in range(8) for y in (5, 4) for x in (6, 5) if part[c, y, x] == k)
        sym2 = sym.copy()
        sym2[c, y, x] += 3
        yh_b, mu_b = oracle.progressive_means(orc, cfg, wts, mu0, sym2)
        diff = mu_b != mu_a
        assert not diff[part <= k].any()
        for j in range(1, 4 - k):
            d = diff & (part == k + j)
            assert d.any()                                      # random weights: the dependency is really there
            ys, xs = np.nonzero(d.any(axis=0))
            assert np.abs(ys - y).max() <= j and np.abs(xs - x).max() <= j
        assert yh_b[c, y, x] - (sym2[c, y, x] + mu_b[c, y, x]) == 0.0     # y = r + mu everywhere


def test_against_element_wise_brute_force(orc):
    """Re-evaluate the recursion element by element with explicit sums (no conv routine, no masks as arrays)."""
    cfg = tiny_cfg(c_y=4, h=4, w=6)
    wts, mu0, sym = random_case(cfg, 5)
    C, h, w = mu0.shape
    yhat, mu = oracle.progressive_means(orc, cfg, wts, mu0, sym)

    def step_of(c, y, x):
        return (2 * (y % 2) + (x % 2) + (4 * c) // C) % 4

    known = {}                                                   # (c, y, x) -> y value, filled step by step
    for k in range(4):
        new = {}
        for c in range(C):
            for y in range(h):
                for x in range(w):
                    if step_of(c, y, x) != k:
                        continue
                    if k == 0:
                        m = mu0[c, y, x]
                    else:
                        m = wts[f"mu.{k}.b"][c]
                        for ci in range(2 * C):
                            for dy in (-1, 0, 1):
                                for dx in (-1, 0, 1):
                                    yy, xx = y + dy, x + dx
                                    if not (0 <= yy < h and 0 <= xx < w):
                                        continue
                                    v = known.get((ci, yy, xx), 0.0) if ci < C else mu0[ci - C, yy, xx]
                                    m += wts[f"mu.{k}.w"][c, ci, dy + 1, dx + 1] * v
                    assert abs(m - mu[c, y, x]) < 1e-12
                    new[(c, y, x)] = sym[c, y, x] + m
        known.update(new)
    assert all(abs(known[(c, y, x)] - yhat[c, y, x]) < 1e-12 for c in range(C) for y in range(h) for x in range(w))


def test_chunk_decode_uses_the_progressive_means(orc):
    """End to end on the tiny config: mu_steps = 4 changes y exactly as progressive_means says, the symbols and the
    scales do not move (bit-stream operations depend on the scales only)."""
    cfg4 = synth.progressive_config(synth.CONFIGS[1])
    cfg1 = synth.CONFIGS[1]
    w4 = synth.make_weights(cfg4)
    z, u16 = synth.make_z(cfg4)[0], synth.make_uniform16(cfg4)[0]
    st = oracle.make_stream(orc, cfg4, w4, z, u16)
    a = oracle.chunk_decode(orc, cfg1, w4, z, st["bits"], st["sub_off"])
    b = oracle.chunk_decode(orc, cfg4, w4, z, st["bits"], st["sub_off"])
    assert a["status"] == 0 and b["status"] == 0
    assert np.array_equal(a["sym"], b["sym"]) and np.array_equal(a["idx"], b["idx"])
    part = oracle.partition_index(cfg4.c_y, *a["mu"].shape[1:])
    assert np.array_equal(a["yhat"][part == 0], b["yhat"][part == 0])
    yh, mu = oracle.progressive_means(orc, cfg4, w4, a["mu"], a["sym"])
    assert np.array_equal(yh, b["yhat"]) and np.array_equal(mu, b["mu"])
    assert np.abs(b["yhat"] - a["yhat"])[part != 0].max() > 1e-3
