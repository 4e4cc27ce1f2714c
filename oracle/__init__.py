"""ufnvc oracle -- TEST INFRASTRUCTURE ONLY (see ufnvc_oracle.c header).

Plain CPU chunk decode, steps O1..O9 of SURVEY.md section 8(c), following PAPER.md section 3.1 (chunk decoder
+ frame-specific decoders) and section 3.4 (single-step entropy: sigma for everything in one pass,
r = AD(sigma), y = r + mu).  The C file holds the loops; this file strings them together in
the paper's order and keeps every intermediate.  It imports nothing from the product package.

Importers allowed: tests/, __graft_entry__.smoke(), bench.py's cpu_baseline / --impl reference legs.
"""
from __future__ import annotations

import ctypes as C
import math
import os

import numpy as np

from . import build as _build

_LIBS = {}


def _lib(real: str):
    if real not in _LIBS:
        path = _build.lib_path(real)
        if not os.path.exists(path):
            _build.build()
        lib = C.CDLL(path)
        lib.orc_rans_encode_substream.restype = C.c_long
        lib.orc_rans_decode_substream.restype = C.c_int
        lib.orc_ideal_bits.restype = C.c_double
        lib.orc_real_bytes.restype = C.c_int
        _LIBS[real] = lib
    return _LIBS[real]


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


class Oracle:
    """Thin typed wrappers over the C loops.  real = "f64" (default, parity truth) or "f32"."""

    def __init__(self, real: str = "f64"):
        self.real = real
        self.lib = _lib(real)
        self.dt = np.float64 if real == "f64" else np.float32
        assert self.lib.orc_real_bytes() == np.dtype(self.dt).itemsize

    def num_threads(self) -> int:
        return int(self.lib.orc_num_threads())

    def arr(self, a):
        return np.ascontiguousarray(a, dtype=self.dt)

    # ---- layers (planar [C][H][W]) ----
    def conv2d(self, x, w, b):
        x, w = self.arr(x), self.arr(w)
        co, ci, k, _ = w.shape
        assert x.shape[0] == ci and k in (1, 3)
        out = np.empty((co,) + x.shape[1:], self.dt)
        bb = self.arr(b) if b is not None else None
        self.lib.orc_conv2d(_p(x), C.c_int(ci), C.c_int(x.shape[1]), C.c_int(x.shape[2]), _p(w),
                            _p(bb) if bb is not None else None, C.c_int(co), C.c_int(k), _p(out))
        return out

    def dwconv3x3(self, x, w, b):
        x, w = self.arr(x), self.arr(w)
        out = np.empty_like(x)
        bb = self.arr(b) if b is not None else None
        self.lib.orc_dwconv3x3(_p(x), C.c_int(x.shape[0]), C.c_int(x.shape[1]), C.c_int(x.shape[2]), _p(w),
                               _p(bb) if bb is not None else None, _p(out))
        return out

    def pixel_shuffle(self, x, r):
        x = self.arr(x)
        c = x.shape[0] // (r * r)
        assert c * r * r == x.shape[0]
        out = np.empty((c, x.shape[1] * r, x.shape[2] * r), self.dt)
        self.lib.orc_pixel_shuffle(_p(x), C.c_int(c), C.c_int(x.shape[1]), C.c_int(x.shape[2]), C.c_int(r), _p(out))
        return out

    def relu(self, x):
        x = self.arr(x).copy()
        self.lib.orc_relu(_p(x), C.c_size_t(x.size))
        return x

    def gelu(self, x):
        x = self.arr(x).copy()
        self.lib.orc_gelu(_p(x), C.c_size_t(x.size))
        return x

    # ---- entropy model pieces ----
    def build_cdf(self, nb, smin, smax):
        cdf = np.empty((nb, 256), np.uint32)
        self.lib.orc_build_cdf(C.c_int(nb), C.c_double(smin), C.c_double(smax), _p(cdf))
        return cdf

    def bucket_index(self, u, nb, smin, smax):
        u = self.arr(u)
        idx = np.empty(u.shape, np.uint8)
        uc = np.empty_like(u)
        self.lib.orc_bucket_index(_p(u), C.c_size_t(u.size), C.c_int(nb), C.c_double(smin), C.c_double(smax),
                                  _p(idx), _p(uc))
        return idx, uc

    def symbols_from_uniform(self, cdf, idx, u16):
        idx = np.ascontiguousarray(idx, np.uint8)
        u16 = np.ascontiguousarray(u16, np.uint16)
        assert idx.shape == u16.shape
        sym = np.empty(idx.shape, np.int16)
        self.lib.orc_symbols_from_uniform(_p(cdf), _p(idx), _p(u16), C.c_size_t(idx.size), _p(sym))
        return sym

    def rans_encode_substream(self, cdf, idx, sym, W):
        idx = np.ascontiguousarray(idx, np.uint8).ravel()
        sym = np.ascontiguousarray(sym, np.int16).ravel()
        cap = 8 * (W // 32) + (W // 32) * 136 + 2 * sym.size + 64
        out = np.zeros(cap, np.uint8)
        n = self.lib.orc_rans_encode_substream(_p(cdf), _p(idx), _p(sym), C.c_size_t(sym.size), C.c_int(W),
                                               _p(out), C.c_size_t(cap))
        if n < 0:
            raise ValueError(f"rANS encode failed ({n})")
        return out[:n].copy()

    def rans_decode_substream(self, cdf, idx, W, data):
        idx = np.ascontiguousarray(idx, np.uint8).ravel()
        data = np.ascontiguousarray(data, np.uint8)
        sym = np.zeros(idx.size, np.int16)
        st = self.lib.orc_rans_decode_substream(_p(cdf), _p(idx), C.c_size_t(idx.size), C.c_int(W), _p(data),
                                                C.c_size_t(data.size), _p(sym))
        return sym, int(st)

    def ideal_bits(self, cdf, idx, sym):
        idx = np.ascontiguousarray(idx, np.uint8).ravel()
        sym = np.ascontiguousarray(sym, np.int16).ravel()
        return float(self.lib.orc_ideal_bits(_p(cdf), _p(idx), _p(sym), C.c_size_t(sym.size)))


# ---------------------------------------------------------------------------------------------
# geometry (SURVEY.md section 8 notation; R2, R16)
# ---------------------------------------------------------------------------------------------
def geometry(cfg):
    H = -(-cfg.height // 32) * 32
    W = -(-cfg.width // 32) * 32
    h, w = H // 16, W // 16
    return dict(H=H, W=W, h=h, w=w, h_z=-(-h // 4), w_z=-(-w // 4), n_sub=-(-h // cfg.rows_per_substream))


# ---------------------------------------------------------------------------------------------
# the path, in the paper's order
# ---------------------------------------------------------------------------------------------
def round_bf16(a):
    """Nearest-even rounding to bfloat16 (8 significant bits), returned in the input's float type.  The temporal context
    state is DEFINED as a bf16 tensor (R19/R23): this is the one place the oracle applies a storage rounding."""
    u = np.ascontiguousarray(a, dtype=np.float32).view(np.uint32)
    r = ((u >> 16) & 1) + np.uint32(0x7FFF)
    return ((u + r) & np.uint32(0xFFFF0000)).view(np.float32).astype(np.asarray(a).dtype)


def has_context(cfg):
    return getattr(cfg, "n_ctx_blocks", 0) > 0


def zero_context(cfg):
    g = geometry(cfg)
    return np.zeros((cfg.c_trunk, g["h"], g["w"]), np.float64)


def context_prior(orc: Oracle, cfg, weights, ctx):
    """NEXT-2a, reading R23 (the prior input s_i is "derived from hyper-prior z_i and temporal context
    C_i"; how is not in the text).  R23: the context enters the hyper-decoder at the hyper-latent's resolution as
    q = ReLU(W_p pool4(C_i) + b_p), pool4 = mean over the 4 x 4 block of latent pixels under a z-pixel (zeros past the
    latent's edge, always divided by 16), W_p a 1x1 conv C_c -> C_h; s = x2 + q feeds the head conv.
    ctx [C_c][h][w].  Returns q [C_h][h_z][w_z]."""
    g = geometry(cfg)
    c = np.zeros((ctx.shape[0], 4 * g["h_z"], 4 * g["w_z"]), orc.dt)
    c[:, :g["h"], :g["w"]] = ctx
    pool = c.reshape(ctx.shape[0], g["h_z"], 4, g["w_z"], 4).sum(axis=(2, 4)) / 16.0
    return orc.relu(orc.conv2d(pool, weights["ctx.prior.w"], weights["ctx.prior.b"]))


def entropy_params(orc: Oracle, cfg, weights, z, ctx=None):
    """O1 + O2 (one forward pass gives the scale of every element and the mean).
    z: int [C_z][h_z][w_z]; ctx: the temporal chunk context C_i [C_c][h][w] when the config has one (R23).
    Returns mu, u = clamped ln sigma, idx, each [C_y][h][w]."""
    g = geometry(cfg)
    x0 = orc.arr(z)
    x1 = orc.relu(orc.conv2d(x0, weights["hyper.0.w"], weights["hyper.0.b"]))
    x2 = orc.relu(orc.conv2d(x1, weights["hyper.1.w"], weights["hyper.1.b"]))
    if has_context(cfg):
        x2 = x2 + context_prior(orc, cfg, weights, zero_context(cfg) if ctx is None else ctx)     # s_i (R23)
    x3 = orc.conv2d(x2, weights["hyper.2.w"], weights["hyper.2.b"])
    ps = orc.pixel_shuffle(x3, 4)[:, :g["h"], :g["w"]]
    mu = np.ascontiguousarray(ps[:cfg.c_y])
    idx, u = orc.bucket_index(np.ascontiguousarray(ps[cfg.c_y:]), cfg.n_buckets, cfg.scale_min, cfg.scale_max)
    return mu, u, idx


def _stream_order(a_chw, r0, r1):
    """planar [C][h][w] rows [r0,r1) -> stream order (row, col, channel) [R9]."""
    return np.ascontiguousarray(np.transpose(a_chw[:, r0:r1, :], (1, 2, 0))).ravel()


def encode_chunk(orc: Oracle, cfg, cdf, idx, sym):
    """Test-fixture ENCODER (mirror of O4).  idx, sym planar [C_y][h][w].  Returns (bytes, sub_off[n_sub+1])."""
    g = geometry(cfg)
    parts, off = [], [0]
    for s in range(g["n_sub"]):
        r0, r1 = s * cfg.rows_per_substream, min((s + 1) * cfg.rows_per_substream, g["h"])
        b = orc.rans_encode_substream(cdf, _stream_order(idx, r0, r1), _stream_order(sym, r0, r1),
                                      cfg.lanes_per_substream)
        parts.append(b)
        off.append(off[-1] + b.size)
    return np.concatenate(parts), np.asarray(off, np.uint32)


def decode_symbols(orc: Oracle, cfg, cdf, idx, bits, sub_off):
    """O4 (arithmetic decoding of all partitions in one consolidated step, scale only)."""
    g = geometry(cfg)
    sym = np.zeros((cfg.c_y, g["h"], g["w"]), np.int16)
    status = 0
    for s in range(g["n_sub"]):
        r0, r1 = s * cfg.rows_per_substream, min((s + 1) * cfg.rows_per_substream, g["h"])
        ss, st = orc.rans_decode_substream(cdf, _stream_order(idx, r0, r1), cfg.lanes_per_substream,
                                           bits[int(sub_off[s]):int(sub_off[s + 1])])
        sym[:, r0:r1, :] = np.transpose(ss.reshape(r1 - r0, g["w"], cfg.c_y), (2, 0, 1))
        status = status or st
    return sym, status


# ---------------------------------------------------------------------------------------------
# NEXT-3: the hyper-latent's own entropy coding, so that a chunk is bytes only.  Reading R22.
# ---------------------------------------------------------------------------------------------
def z_geometry(cfg):
    g = geometry(cfg)
    return dict(h_z=g["h_z"], w_z=g["w_z"], n_sub_z=-(-g["h_z"] // cfg.rows_per_substream))


def z_prior_index(orc: Oracle, cfg, weights):
    """R22: z has a factorised prior (PAPER.md:125 names z only as "hyper-prior"; the prior's form is not in the
    text): zero-mean Gaussian per channel with one learned ln sigma per channel (`zprior.lnscale` [C_z]), quantised
    with the SAME bucket rule and the SAME tables as y (O2, O3).  Returns uint8 [C_z]."""
    idx, _ = orc.bucket_index(np.asarray(weights["zprior.lnscale"], np.float64), cfg.n_buckets, cfg.scale_min, cfg.scale_max)
    return idx


def _z_stream_idx(cfg, idx_c, r0, r1, w_z):
    return np.ascontiguousarray(np.broadcast_to(idx_c[None, None, :], (r1 - r0, w_z, idx_c.size))).ravel()


def encode_z(orc: Oracle, cfg, cdf, weights, z):
    """Fixture ENCODER for z [C_z][h_z][w_z] (mirror of decode_z): substreams of rows_per_substream rows of the
    hyper-latent, stream order (row, col, channel) as for y [R9].  Returns (bytes, sub_off[n_sub_z + 1])."""
    zg = z_geometry(cfg)
    idx_c = z_prior_index(orc, cfg, weights)
    parts, off = [], [0]
    for s in range(zg["n_sub_z"]):
        r0, r1 = s * cfg.rows_per_substream, min((s + 1) * cfg.rows_per_substream, zg["h_z"])
        b = orc.rans_encode_substream(cdf, _z_stream_idx(cfg, idx_c, r0, r1, zg["w_z"]),
                                      _stream_order(np.asarray(z, np.int16), r0, r1), cfg.lanes_per_substream)
        parts.append(b)
        off.append(off[-1] + b.size)
    return np.concatenate(parts), np.asarray(off, np.uint32)


def decode_z(orc: Oracle, cfg, cdf, weights, bits, sub_off):
    """NEXT-3 / R22: the same arithmetic decoder as O4, the table of every symbol chosen by its CHANNEL alone.
    Returns (z int16 [C_z][h_z][w_z], status)."""
    zg = z_geometry(cfg)
    idx_c = z_prior_index(orc, cfg, weights)
    z = np.zeros((cfg.c_z, zg["h_z"], zg["w_z"]), np.int16)
    status = 0
    for s in range(zg["n_sub_z"]):
        r0, r1 = s * cfg.rows_per_substream, min((s + 1) * cfg.rows_per_substream, zg["h_z"])
        ss, st = orc.rans_decode_substream(cdf, _z_stream_idx(cfg, idx_c, r0, r1, zg["w_z"]), cfg.lanes_per_substream,
                                           bits[int(sub_off[s]):int(sub_off[s + 1])])
        z[:, r0:r1, :] = np.transpose(ss.reshape(r1 - r0, zg["w_z"], cfg.c_z), (2, 0, 1))
        status = status or st
    return z, status


def pack_chunk_bytes(z_bits, z_off, y_bits, y_off):
    """Container of one chunk for the bytes-only call: the z substreams, then the y substreams, one offset table."""
    off = np.concatenate([np.asarray(z_off, np.int64), np.asarray(y_off, np.int64)[1:] + int(z_off[-1])])
    return np.concatenate([z_bits, y_bits]), off.astype(np.uint32)


def chunk_decode_bytes(orc: Oracle, cfg, weights, bits, sub_off, keep=False):
    """One chunk from bytes only: decode z (NEXT-3), then O1..O9 on the rest of the container."""
    zg = z_geometry(cfg)
    cdf = orc.build_cdf(cfg.n_buckets, cfg.scale_min, cfg.scale_max)
    nz = zg["n_sub_z"]
    z, st_z = decode_z(orc, cfg, cdf, weights, bits, sub_off[:nz + 1])
    y0 = int(sub_off[nz])
    out = chunk_decode(orc, cfg, weights, z, bits[y0:], np.asarray(sub_off[nz:], np.int64) - y0, keep=keep)
    out["z"] = z
    out["status"] = out["status"] or st_z
    return out


def partition_index(c_y, h, w):
    """NEXT-1, reading R21 (Fig. 4a, "a quadtree-like partition [36] for y_i is adopted"; PAPER.md:101
    "the quantized latent y_i is divided into four partitions, where each partition's decoding depends on previously
    decoded partitions").  The geometry is not in the text; R21 takes: channels in four equal groups g = floor(4c/C_y),
    positions of a 2x2 cell numbered q = 2 (y mod 2) + (x mod 2), partition k = (q + g) mod 4.
    Returns int [C_y][h][w] with values 0..3."""
    assert c_y % 4 == 0
    k = np.empty((c_y, h, w), np.int64)
    for c in range(c_y):
        g = (4 * c) // c_y
        for y in range(h):
            for x in range(w):
                k[c, y, x] = (2 * (y % 2) + (x % 2) + g) % 4
    return k


def progressive_means(orc: Oracle, cfg, weights, mu0, sym):
    """NEXT-1 (the network "predicts the mean mu^0 for the first partition and the scales for all four
    partitions in a single forward pass"; "We retain the four-step progressive estimation for means
    ... since mean estimation requires no bit-stream interaction, it executes entirely on GPU"; PAPER.md:125:
    y = r + mu).  mu0, sym planar [C_y][h][w]; sym is the residual of EVERY partition, already decoded (O4).
    Step 0: y = r + mu0 on partition 0.  Step k = 1..3 [R21]: mu^k = conv3x3_k([y decoded so far (0 elsewhere) ; mu0]),
    y = r + mu^k on partition k.  Returns (yhat, mu) with mu[c,y,x] = the mean that element used."""
    part = partition_index(cfg.c_y, mu0.shape[1], mu0.shape[2])
    mu0 = orc.arr(mu0)
    r = sym.astype(orc.dt)
    mu = np.where(part == 0, mu0, 0.0).astype(orc.dt)
    yhat = np.where(part == 0, r + mu0, 0.0).astype(orc.dt)
    for k in (1, 2, 3):
        s_in = np.concatenate([yhat, mu0], axis=0)
        mu_k = orc.conv2d(s_in, weights[f"mu.{k}.w"], weights[f"mu.{k}.b"])
        mu = np.where(part == k, mu_k, mu)
        yhat = np.where(part == k, r + mu_k, yhat)
    return yhat, mu


def synthesis(orc: Oracle, cfg, weights, yhat, keep=False, only_frames=None, ctx=None, want_features=False):
    """O6..O9: cross-frame unfold, shared trunk of DC blocks, T frame-specific
    decoders, clamp + crop.  yhat [C_y][h][w].  Returns frames [T][3][height][width] (+ taps).
    only_frames: frame indices to compute (the T frames are independent after O6, "operating in parallel");
    the others are left as NaN -- used by the full-size parity tests of configs 4 and 5 to bound the oracle's time."""
    taps = {}
    if has_context(cfg):
        # R23 ("conditioned on the temporal chunk context C_i"): the chunk decoder's first layer sees the
        # concatenation [y ; C_i]; xframe.w is [T*C_t][C_y + C_c][1][1]
        yhat = np.concatenate([orc.arr(yhat), orc.arr(zero_context(cfg) if ctx is None else ctx)], axis=0)
    if want_features:
        taps["features"] = [None] * cfg.T                                      # F_i, the trunk's output per frame
    f0 = orc.conv2d(yhat, weights["xframe.w"], weights["xframe.b"])            # O6: [T*C_t][h][w]
    frames = np.full((cfg.T, 3, cfg.height, cfg.width), np.nan, orc.dt)
    if keep:
        taps["F0"] = f0.reshape(cfg.T, cfg.c_trunk, *f0.shape[1:]).copy()
        taps["trunk"] = []
        taps["stage"] = [[] for _ in range(cfg.T)]
    for t in (range(cfg.T) if only_frames is None else only_frames):
        x = np.ascontiguousarray(f0[t * cfg.c_trunk:(t + 1) * cfg.c_trunk])
        for k in range(cfg.n_trunk_blocks):                                    # O7, same weights for every t [R15]
            d = orc.dwconv3x3(x, weights[f"trunk.{k}.dw.w"], weights[f"trunk.{k}.dw.b"])
            e = orc.gelu(orc.conv2d(d, weights[f"trunk.{k}.pw1.w"], weights[f"trunk.{k}.pw1.b"]))
            x = x + orc.conv2d(e, weights[f"trunk.{k}.pw2.w"], weights[f"trunk.{k}.pw2.b"])
        if keep:
            taps["trunk"].append(x.copy())           # (indexed by position in only_frames when that is given)
        if want_features:
            taps["features"][t] = x.copy()
        for s in range(4):                                                     # O8 [R10]
            a = orc.conv2d(x, weights[f"dec.{t}.{s}.w"], weights[f"dec.{t}.{s}.b"])
            if s < 3:
                a = orc.gelu(a)
            x = orc.pixel_shuffle(a, 2)
            if keep and s < 3:
                taps["stage"][t].append(x.copy())
        frames[t] = np.clip(x, 0.0, 1.0)[:, :cfg.height, :cfg.width]           # O9 [R16]
    return frames, taps


def context_generation(orc: Oracle, cfg, weights, features):
    """NEXT-2a, reading R23.  PAPER.md:81: the feature F_i "is also propagated to the next chunk to form the next temporal
    context"; PAPER.md:356 (Supp. B): the cross-chunk context generation module is a stack of DC blocks (11 for HT-S).
    R23: C_{i+1} = bf16( conv1x1_out( DCblock^{B_c}( conv1x1_fold( [F_i[0]; ...; F_i[T-1]] ) ) ) ), the fold mixing the T
    per-frame features (T*C_t channels) into one C_c-channel map at latent resolution -- the mirror of the cross-frame
    unfold O6 -- and the DC block being O7's (depthwise 3x3, 1x1 x4, GELU, 1x1, residual).
    features: list of T arrays [C_t][h][w].  Returns C_{i+1} [C_c][h][w], bf16-representable values."""
    x = orc.conv2d(np.concatenate([orc.arr(f) for f in features], axis=0), weights["ctx.fold.w"], weights["ctx.fold.b"])
    for k in range(cfg.n_ctx_blocks):
        d = orc.dwconv3x3(x, weights[f"ctx.{k}.dw.w"], weights[f"ctx.{k}.dw.b"])
        e = orc.gelu(orc.conv2d(d, weights[f"ctx.{k}.pw1.w"], weights[f"ctx.{k}.pw1.b"]))
        x = x + orc.conv2d(e, weights[f"ctx.{k}.pw2.w"], weights[f"ctx.{k}.pw2.b"])
    return round_bf16(orc.conv2d(x, weights["ctx.out.w"], weights["ctx.out.b"]))


def chunk_decode(orc: Oracle, cfg, weights, z, bits, sub_off, idx_override=None, mu_override=None, keep=False, ctx=None):
    """One chunk, O1..O9.  z [C_z][h_z][w_z]; bits uint8; sub_off [n_sub+1] byte offsets into bits.  With a temporal
    context in the config (R23): ctx = C_i (None = the zero context of a sequence's first chunk); the result then
    also carries "ctx_next" = C_{i+1}."""
    mu, u, idx = entropy_params(orc, cfg, weights, z, ctx=ctx)
    if idx_override is not None:
        idx = np.ascontiguousarray(idx_override, np.uint8)
    if mu_override is not None:
        mu = orc.arr(mu_override)
    cdf = orc.build_cdf(cfg.n_buckets, cfg.scale_min, cfg.scale_max)          # O3
    sym, status = decode_symbols(orc, cfg, cdf, idx, bits, sub_off)            # O4
    if getattr(cfg, "mu_steps", 1) == 4:
        yhat, mu = progressive_means(orc, cfg, weights, mu, sym)               # NEXT-1: mu becomes the per-element mean used
    else:
        yhat = sym.astype(orc.dt) + mu                                         # O5
    frames, taps = synthesis(orc, cfg, weights, yhat, keep=keep, ctx=ctx, want_features=has_context(cfg))
    out = dict(mu=mu, u=u, idx=idx, sym=sym, status=status, yhat=yhat, frames=frames, taps=taps)
    if has_context(cfg):
        out["ctx_next"] = context_generation(orc, cfg, weights, taps["features"])
    return out


def chunk_decode_sequence(orc: Oracle, cfg, weights, zs, streams, keep=False):
    """Successive chunks of ONE video ("a sequential chunk-by-chunk coding process"): C_0 = 0, chunk i is
    decoded under C_i and hands C_{i+1} on.  streams[i] = (bits, sub_off).  Returns the list of per-chunk results, each
    with the context it was decoded under ("ctx")."""
    ctx, outs = zero_context(cfg), []
    for z, (bits, sub_off) in zip(zs, streams):
        out = chunk_decode(orc, cfg, weights, z, bits, sub_off, keep=keep, ctx=ctx)
        out["ctx"] = ctx
        outs.append(out)
        ctx = out["ctx_next"]
    return outs


def make_stream(orc: Oracle, cfg, weights, z, u16_hwc, idx_override=None, ctx=None):
    """Fixture: what an encoder would have produced for this z -- run the prior net (O1, O2; under the context C_i when
    the config has one), draw r from the quantised tables by inverse CDF with the given 16-bit uniforms [h][w][C_y]
    (R7), encode (mirror of O4)."""
    mu, u, idx = entropy_params(orc, cfg, weights, z, ctx=ctx)
    if idx_override is not None:
        idx = np.ascontiguousarray(idx_override, np.uint8)
    cdf = orc.build_cdf(cfg.n_buckets, cfg.scale_min, cfg.scale_max)
    sym = orc.symbols_from_uniform(cdf, idx, np.transpose(u16_hwc, (2, 0, 1)))
    bits, sub_off = encode_chunk(orc, cfg, cdf, idx, sym)
    return dict(mu=mu, u=u, idx=idx, sym=sym, bits=bits, sub_off=sub_off, cdf=cdf)


# ---------------------------------------------------------------------------------------------
# NEXT-4: chunk ENCODE, reading R24, and the colour interface of Supp. C.
# ---------------------------------------------------------------------------------------------
def rgb_to_yuv444(rgb):
    """PAPER.md:384 (Supp. C): "a unified YUV444 colorspace that serves as a universal interface ... For both YUV420 and RGB
    videos, they will be converted into YUV444"; the RGB tests use BT.709.  Full-range BT.709 on [0,1] floats:
    Y = 0.2126 R + 0.7152 G + 0.0722 B, Cb = (B - Y) / 1.8556 + 1/2, Cr = (R - Y) / 1.5748 + 1/2.  rgb [..., 3, H, W]."""
    rgb = np.asarray(rgb, np.float64)
    r, g, b = rgb[..., 0, :, :], rgb[..., 1, :, :], rgb[..., 2, :, :]
    y = 0.2126 * r + 0.7152 * g + 0.0722 * b
    return np.stack([y, (b - y) / 1.8556 + 0.5, (r - y) / 1.5748 + 0.5], axis=-3)


def yuv444_to_rgb(yuv):
    """Inverse of rgb_to_yuv444: R = Y + 1.5748 (Cr - 1/2), B = Y + 1.8556 (Cb - 1/2), G = (Y - 0.2126 R - 0.0722 B) / 0.7152."""
    yuv = np.asarray(yuv, np.float64)
    y, cb, cr = yuv[..., 0, :, :], yuv[..., 1, :, :] - 0.5, yuv[..., 2, :, :] - 0.5
    r = y + 1.5748 * cr
    b = y + 1.8556 * cb
    g = (y - 0.2126 * r - 0.0722 * b) / 0.7152
    return np.stack([r, g, b], axis=-3)


def space_to_depth(x, r):
    """[C][H r][W r] -> [r r C][H][W] with channel (r i + j) C + c = x[c, r y + i, r x + j] (the inverse of a pixel shuffle,
    position-major: all channels of sub-position (i, j) are contiguous)."""
    c, hh, ww = x.shape
    assert hh % r == 0 and ww % r == 0
    h, w = hh // r, ww // r
    return np.ascontiguousarray(x.reshape(c, h, r, w, r).transpose(2, 4, 0, 1, 3).reshape(r * r * c, h, w))


def encoder_features(orc: Oracle, cfg, weights, frames, ctx=None):
    """R24, E1..E5 ("transforming it to 1/8 resolution via patch embedding ... conditioned on the temporal chunk
    context C_i, and fed into a chunk encoder ... distill the spatial-temporal information of the entire chunk into a compact
    latent representation y_i"; the chunk encoder is a stack of DC blocks).  The layer plan is the mirror of the
    decode configs: E1 patch embedding = space-to-depth x8 of every frame (zero-padded to the codec's H x W) + 1x1 conv
    192 -> C_t, weights shared over t; E2 = space-to-depth x2 (to the latent's 1/16 resolution) and a 1x1 fold over the T
    frames (T 4 C_t -> C_t); E3 = + 1x1 conv of the context C_i (when the config has one); E4 = B_e DC blocks (O7's block);
    E5 = 1x1 conv C_t -> C_y.  frames [T][3][height][width] in [0,1].  Returns y [C_y][h][w] (unquantised)."""
    g = geometry(cfg)
    x = np.zeros((cfg.T, 3, g["H"], g["W"]), orc.dt)
    x[:, :, :cfg.height, :cfg.width] = frames
    s2 = []
    for t in range(cfg.T):
        p8 = space_to_depth(x[t], 8)                                            # [192][H/8][W/8], channel (8 i + j) 3 + c
        f1 = orc.conv2d(p8, weights["enc.patch.w"], weights["enc.patch.b"])     # E1
        s2.append(space_to_depth(f1, 2))                                        # [4 C_t][h][w]
    feat = orc.conv2d(np.concatenate(s2, axis=0), weights["enc.fold.w"], weights["enc.fold.b"])      # E2
    if has_context(cfg):
        feat = feat + orc.conv2d(orc.arr(zero_context(cfg) if ctx is None else ctx), weights["enc.ctx.w"], weights["enc.ctx.b"])   # E3
    for k in range(cfg.n_enc_blocks):                                           # E4
        d = orc.dwconv3x3(feat, weights[f"enc.{k}.dw.w"], weights[f"enc.{k}.dw.b"])
        e = orc.gelu(orc.conv2d(d, weights[f"enc.{k}.pw1.w"], weights[f"enc.{k}.pw1.b"]))
        feat = feat + orc.conv2d(e, weights[f"enc.{k}.pw2.w"], weights[f"enc.{k}.pw2.b"])
    return orc.conv2d(feat, weights["enc.y.w"], weights["enc.y.b"])             # E5


def hyper_encoder(orc: Oracle, cfg, weights, y):
    """R24, E6: the hyper-latent.  y zero-padded to [4 h_z][4 w_z], space-to-depth x4 -> [16 C_y][h_z][w_z]; ReLU(1x1 conv
    16 C_y -> C_h); 3x3 conv C_h -> C_z; z = clip(rint(.), -127, 127) (the coder's alphabet, R7).  Returns (z int16, zf)."""
    g = geometry(cfg)
    yp = np.zeros((cfg.c_y, 4 * g["h_z"], 4 * g["w_z"]), orc.dt)
    yp[:, :g["h"], :g["w"]] = y
    a = orc.relu(orc.conv2d(space_to_depth(yp, 4), weights["henc.0.w"], weights["henc.0.b"]))
    zf = orc.conv2d(a, weights["henc.1.w"], weights["henc.1.b"])
    return np.clip(np.rint(zf), -127, 127).astype(np.int16), zf


def quantise(y, mu):
    """"After quantization via r_i = round(y_i - mu_i), the result r_i is arithmetically encoded using scale
    sigma_i".  Round half to even, in fp32 -- the precision both sides take this integer decision in -- clipped to the
    coder's alphabet [-127, 127] (R7).  Returns int16."""
    d = np.asarray(y, np.float32) - np.asarray(mu, np.float32)
    return np.clip(np.rint(d), -127, 127).astype(np.int16)


def chunk_encode(orc: Oracle, cfg, weights, frames, ctx=None, z_override=None, y_override=None):
    """One chunk, frames -> bytes (R24): E1..E6, the decoder's own prior net on z, quantisation, the mirror
    of O4.  Only the single-pass mean (mu_steps == 1).  z_override / y_override: teacher forcing for the parity tests (the
    integer decisions z and r depend on floats that differ between implementations at rounding edges).
    Returns dict(y, z, zf, mu, u, idx, sym, bits, sub_off)."""
    assert getattr(cfg, "mu_steps", 1) == 1
    y = encoder_features(orc, cfg, weights, frames, ctx=ctx) if y_override is None else orc.arr(y_override)
    z, zf = hyper_encoder(orc, cfg, weights, y)
    if z_override is not None:
        z = np.asarray(z_override, np.int16)
    mu, u, idx = entropy_params(orc, cfg, weights, z, ctx=ctx)
    sym = quantise(y, mu)
    cdf = orc.build_cdf(cfg.n_buckets, cfg.scale_min, cfg.scale_max)
    bits, sub_off = encode_chunk(orc, cfg, cdf, idx, sym)
    return dict(y=y, z=z, zf=zf, mu=mu, u=u, idx=idx, sym=sym, bits=bits, sub_off=sub_off)
