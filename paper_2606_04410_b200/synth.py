"""Seeded synthetic inputs for the chunk-decode path.

This module is shared by the CUDA path's callers (tests, bench.py) and by the oracle's
callers (tests).  It holds NONE of the method's arithmetic: it only names the five
BASELINE.json workloads and draws raw random numbers (weights, the hyper-latent z, 16-bit
uniforms from which each side derives its own symbols, and exact-law (mu, ln sigma) maps
for the entropy-only mode).  Neither `oracle/` nor `csrc/` imports it.

Stand-in statement: the paper measures on UVG / MCL-JCV / HEVC B-E natural video
 with trained weights; neither is available, so everything below is random
with the shapes of BASELINE.json:configs.
"""
from __future__ import annotations

import dataclasses
import math
import zlib

import numpy as np


@dataclasses.dataclass(frozen=True)
class ChunkConfig:
    """Mirror of `ufnvc_config` (include/ufnvc.h) plus the seed and the input laws."""
    name: str
    seed: int
    T: int
    height: int
    width: int
    c_y: int
    c_z: int
    c_hyper: int
    c_trunk: int
    n_trunk_blocks: int
    trunk_expand: int
    dec_channels: tuple
    n_buckets: int = 64
    scale_min: float = 0.11
    scale_max: float = 20.0
    rows_per_substream: int = 4
    lanes_per_substream: int = 512       # rANS lanes W per substream: 16 warp-streams (R9, speed variant)
    n_chunks: int = 1
    weight_dtype: int = 1          # 0 = fp32, 1 = bf16
    mu_law: str = "normal"         # "normal": N(0,1); "uniform": U(-2,2)
    sigma_hi: float = 20.0         # ln sigma ~ U[ln scale_min, ln sigma_hi] (moment-matched, see make_weights)
    mu_steps: int = 1              # 1: the head's mean serves every element; 4: progressive means (R21)
    n_ctx_blocks: int = 0          # > 0: temporal chunk context (R23) with that many DC blocks in the context generation
    n_enc_blocks: int = 0          # > 0: the blob also carries a chunk ENCODER (R24) with that many DC blocks

    # derived geometry (SURVEY.md section 8 notation)
    @property
    def H(self):  # padded frame height
        return -(-self.height // 32) * 32

    @property
    def W(self):
        return -(-self.width // 32) * 32

    @property
    def h(self):
        return self.H // 16

    @property
    def w(self):
        return self.W // 16

    @property
    def h_z(self):
        return -(-self.h // 4)

    @property
    def w_z(self):
        return -(-self.w // 4)

    @property
    def n_sub(self):
        return -(-self.h // self.rows_per_substream)

    @property
    def n_symbols(self):
        return self.c_y * self.h * self.w

    def macs_per_chunk(self) -> int:
        """Algorithmic multiply-accumulates of one chunk decode."""
        hz, wz, P = self.h_z, self.w_z, self.h * self.w
        m = hz * wz * 9 * (self.c_z * self.c_hyper + self.c_hyper * self.c_hyper
                           + self.c_hyper * 2 * self.c_y * 16)
        if self.mu_steps == 4:
            m += 3 * P * 9 * 2 * self.c_y * self.c_y
        m += P * (self.c_y + (self.c_trunk if self.n_ctx_blocks else 0)) * self.T * self.c_trunk
        if self.n_ctx_blocks:      # prior branch, fold, DC blocks, output conv (R23)
            m += hz * wz * self.c_trunk * self.c_hyper + P * self.T * self.c_trunk * self.c_trunk + P * self.c_trunk * self.c_trunk
            m += self.n_ctx_blocks * P * (9 * self.c_trunk + 2 * self.c_trunk * self.c_trunk * self.trunk_expand)
        m += self.n_trunk_blocks * self.T * P * (9 * self.c_trunk
                                                 + 2 * self.c_trunk * self.c_trunk * self.trunk_expand)
        pix = P
        for s in range(4):
            ci, co = self.dec_channels[s], self.dec_channels[s + 1]
            m += self.T * pix * 9 * ci * 4 * co
            pix *= 4
        return m


_DEC = (256, 192, 128, 64, 3)

CONFIGS = {
    1: ChunkConfig("cfg1-tiny", 0, 2, 64, 64, 32, 16, 32, 64, 0, 4, (64, 48, 32, 16, 3),
                   lanes_per_substream=32, weight_dtype=0, mu_law="uniform"),
    2: ChunkConfig("cfg2-480p", 1, 4, 480, 832, 128, 64, 128, 256, 4, 4, _DEC),
    3: ChunkConfig("cfg3-1080p", 2, 8, 1080, 1920, 128, 64, 128, 256, 6, 4, _DEC),
    4: ChunkConfig("cfg4-1080p-4xT16", 3, 16, 1080, 1920, 192, 64, 128, 256, 6, 4, _DEC,
                   lanes_per_substream=384, n_chunks=4, sigma_hi=2.0),
    5: ChunkConfig("cfg5-4k", 4, 8, 2160, 3840, 128, 64, 128, 256, 8, 4, _DEC),
}


def progressive_config(cfg: ChunkConfig) -> ChunkConfig:
    """Same workload with the four-step progressive means switched on (R21)."""
    return dataclasses.replace(cfg, mu_steps=4, name=cfg.name + "-pmu")


def context_config(cfg: ChunkConfig, n_ctx_blocks: int = 11) -> ChunkConfig:
    """Same workload with the temporal chunk context switched on (R23); 11 DC blocks in
    the cross-chunk context generation is the paper's HT-S count."""
    return dataclasses.replace(cfg, n_ctx_blocks=n_ctx_blocks, name=cfg.name + f"-ctx{n_ctx_blocks}")


def encoder_config(cfg: ChunkConfig, n_enc_blocks: int = 6) -> ChunkConfig:
    """Same workload with the chunk encoder's weights in the blob (R24); 6 DC blocks in the
    chunk encoder is the paper's HT-S count."""
    return dataclasses.replace(cfg, n_enc_blocks=n_enc_blocks, name=cfg.name + f"-enc{n_enc_blocks}")


def make_frames(cfg: ChunkConfig) -> np.ndarray:
    """Synthetic input frames for the encoder, [n_chunks][T][3][height][width] fp32 in [0,1]: smooth low-frequency fields plus a
    little noise, drifting over t (stands in for natural video; only the value range and the smoothness matter here)."""
    rng = _rng(cfg, "frames")
    n, T, H, W = cfg.n_chunks, cfg.T, cfg.height, cfg.width
    gy, gx = np.meshgrid(np.linspace(0, 1, H, dtype=np.float32), np.linspace(0, 1, W, dtype=np.float32), indexing="ij")
    out = np.empty((n, T, 3, H, W), np.float32)
    for i in range(n):
        ph = rng.uniform(0, 2 * np.pi, size=(3, 4)).astype(np.float32)
        fr = rng.uniform(1.0, 6.0, size=(3, 4)).astype(np.float32)
        for t in range(T):
            for c in range(3):
                f = 0.5 + 0.18 * np.sin(2 * np.pi * fr[c, 0] * gx + ph[c, 0] + 0.15 * t) * np.cos(2 * np.pi * fr[c, 1] * gy + ph[c, 1])
                f += 0.12 * np.sin(2 * np.pi * (fr[c, 2] * gx + fr[c, 3] * gy) + ph[c, 2] + 0.1 * t)
                out[i, t, c] = f
        out[i] += rng.normal(0.0, 0.02, size=(T, 3, H, W)).astype(np.float32)
    return np.clip(out, 0.0, 1.0)


def crop_config(cfg: ChunkConfig, height: int, width: int, name: str | None = None) -> ChunkConfig:
    """Same layer plan on a smaller frame (used for bounded CPU-baseline samples and mid-size parity)."""
    return dataclasses.replace(cfg, height=height, width=width,
                               name=name or f"{cfg.name}-crop{width}x{height}")


def round_to_bf16(a: np.ndarray) -> np.ndarray:
    """fp32 array -> nearest-even bf16 value, returned as fp32 (so both sides consume identical weights)."""
    u = np.ascontiguousarray(a, dtype=np.float32).view(np.uint32)
    r = ((u >> 16) & 1) + np.uint32(0x7FFF)
    return ((u + r) & np.uint32(0xFFFF0000)).view(np.float32)


def _rng(cfg: ChunkConfig, tag: str) -> np.random.Generator:
    return np.random.default_rng(np.random.SeedSequence([cfg.seed, zlib.crc32(tag.encode())]))


def _ln_sigma_moments(cfg: ChunkConfig):
    lo, hi = math.log(cfg.scale_min), math.log(cfg.sigma_hi)
    return 0.5 * (lo + hi), (hi - lo) / math.sqrt(12.0)


def _second_moment_yhat(cfg: ChunkConfig) -> float:
    # E[y^2] for y = r + mu, r ~ N(0, sigma^2) rounded, ln sigma uniform: closed form of E[sigma^2].
    lo, hi = cfg.scale_min, cfg.sigma_hi
    e_s2 = (hi * hi - lo * lo) / (2.0 * math.log(hi / lo))
    var_mu = 1.0 if cfg.mu_law == "normal" else 4.0 / 3.0
    # R8 gives every one of the 255 symbols a frequency >= 1/2^16; drawing r from the QUANTISED table (R7) therefore
    # adds sum_r r^2 / 2^16 = 2 * (127*128*255/6) / 65536 = 21.08 to E[r^2] whatever sigma is.
    floor_mass = 2.0 * (127 * 128 * 255 / 6.0) / 65536.0
    return e_s2 + 1.0 / 12.0 + var_mu + floor_mass


def make_weights(cfg: ChunkConfig) -> dict:
    """Canonical-layout weights: conv [C_out][C_in][kh][kw] fp32 (bf16-representable when
    weight_dtype == 1), biases fp32.  Kaiming-normal with analytic gains (R3/R11):
    no data-dependent calibration, so no side has to run the net to make its own inputs."""
    out = {}

    def conv(name, co, ci, k, gain2, bias_std=0.02, bias_mean=0.0):
        rng = _rng(cfg, name)
        fan_in = ci * k * k
        w = rng.normal(0.0, math.sqrt(gain2 / fan_in), size=(co, ci, k, k)).astype(np.float32)
        b = (bias_mean + rng.normal(0.0, bias_std, size=(co,))).astype(np.float32)
        out[name + ".w"] = round_to_bf16(w) if cfg.weight_dtype == 1 else w
        out[name + ".b"] = b

    # hyper-decoder (O1): z ~ round(N(0,4)) so E[z^2] ~ 4.08; ReLU + gain 2 keeps E[x^2] ~ 4.08.
    # `edge`: a 1x1 z map (config 1) sees only the centre tap of each zero-padded 3x3 conv (1/9 of the fan-in), so
    # the gain is raised to keep the variance; larger maps keep the plain gain (borders are then under-dispersed,
    # which only narrows the sigma distribution on small test crops).  Pure geometry, no method arithmetic.
    edge = 1.0 / 9.0 if cfg.h_z * cfg.w_z == 1 else 1.0
    conv("hyper.0", cfg.c_hyper, cfg.c_z, 3, 2.0 / edge)
    conv("hyper.1", cfg.c_hyper, cfg.c_hyper, 3, 2.0 / edge)
    # head: channels after pixel-shuffle x4: [0,C_y) = mu, [C_y,2C_y) = ln sigma.  Pre-shuffle
    # channel o = c*16 + 4i + j  ->  rows [0, 16 C_y) feed mu, the rest feed ln sigma.
    m_u, s_u = _ln_sigma_moments(cfg)
    s_mu = 1.0 if cfg.mu_law == "normal" else 2.0 / math.sqrt(3.0)
    ex2 = 4.08
    name = "hyper.2"
    rng = _rng(cfg, name)
    co, ci = 2 * cfg.c_y * 16, cfg.c_hyper
    w = rng.normal(0.0, 1.0, size=(co, ci, 3, 3)) / math.sqrt(ci * 9 * ex2 * edge)
    half = cfg.c_y * 16
    w[:half] *= s_mu
    w[half:] *= s_u
    b = rng.normal(0.0, 0.02, size=(co,))
    b[half:] += m_u
    w = w.astype(np.float32)
    out[name + ".w"] = round_to_bf16(w) if cfg.weight_dtype == 1 else w
    out[name + ".b"] = b.astype(np.float32)

    # factorised prior of the hyper-latent (NEXT-3, R22): one ln sigma per channel, around the law make_z draws from
    rng = _rng(cfg, "zprior")
    out["zprior.lnscale"] = (math.log(2.0) + rng.uniform(-0.3, 0.3, size=(cfg.c_z,))).astype(np.float32)
    # progressive means (NEXT-1, R21): three 3x3 convs [yhat so far ; mu0] (2 C_y) -> C_y.  Gain so that a mean keeps
    # the law of mu0: the input's second moment is ~ (E[yhat^2] * k/4 + E[mu0^2]) / 2 per channel at step k.
    if cfg.mu_steps == 4:
        var_mu = 1.0 if cfg.mu_law == "normal" else 4.0 / 3.0
        for k in (1, 2, 3):
            ex2_in = 0.5 * (_second_moment_yhat(cfg) * k / 4.0 + var_mu)
            conv(f"mu.{k}", cfg.c_y, 2 * cfg.c_y, 3, var_mu / ex2_in)
    # cross-frame unfold (O6): gain so that E[F0^2] ~ 1.
    conv("xframe", cfg.T * cfg.c_trunk, cfg.c_y, 1, 1.0 / _second_moment_yhat(cfg))
    if cfg.n_ctx_blocks > 0:
        # temporal chunk context (NEXT-2a, R23).  The unfold sees [y ; C_i]: the context columns get their own gain (C has
        # second moment ~2, y ~60) so that each half contributes a comparable share of F0
        cc = cfg.c_trunk
        conv("xframe.ctx", cfg.T * cfg.c_trunk, cc, 1, 0.5 / 2.0)
        out["xframe.w"] = np.concatenate([out["xframe.w"] * np.float32(math.sqrt(0.5)), out.pop("xframe.ctx.w")], axis=1)
        if cfg.weight_dtype == 1:
            out["xframe.w"] = round_to_bf16(out["xframe.w"])
        out.pop("xframe.ctx.b")
        conv("ctx.fold", cc, cfg.T * cfg.c_trunk, 1, 1.0 / 1.5)
        for k in range(cfg.n_ctx_blocks):
            conv(f"ctx.{k}.dw", cc, 1, 3, 1.0)
            conv(f"ctx.{k}.pw1", cc * cfg.trunk_expand, cc, 1, 2.0)
            conv(f"ctx.{k}.pw2", cc, cc * cfg.trunk_expand, 1, 1.0 / cfg.n_ctx_blocks)
        conv("ctx.out", cc, cc, 1, 1.0 / 2.0)
        conv("ctx.prior", cfg.c_hyper, cc, 1, 2.0 * 1.0 / 0.5)       # q = ReLU(W_p pool4(C) + b_p) with E[q^2] ~ 1
    # trunk (O7): shared over t; W2 scaled by 1/B so the residual stream stays O(1).
    ce = cfg.c_trunk * cfg.trunk_expand
    for k in range(cfg.n_trunk_blocks):
        conv(f"trunk.{k}.dw", cfg.c_trunk, 1, 3, 1.0)
        conv(f"trunk.{k}.pw1", ce, cfg.c_trunk, 1, 2.0)
        conv(f"trunk.{k}.pw2", cfg.c_trunk, ce, 1, 1.0 / max(1, cfg.n_trunk_blocks))
    # chunk encoder (NEXT-4, R24): patch embedding, fold over frames, DC blocks, latent head, hyper-encoder.  Gains so that y has
    # the second moment the decoder's cross-frame layer was scaled for and z ~ N(0, 2^2) like make_z.
    if cfg.n_enc_blocks > 0:
        ct = cfg.c_trunk
        conv("enc.patch", ct, 192, 1, 1.0 / 0.3)                    # frames in [0,1]: E[x^2] ~ 0.3
        conv("enc.fold", ct, cfg.T * 4 * ct, 1, 1.0)
        if cfg.n_ctx_blocks > 0:
            conv("enc.ctx", ct, ct, 1, 0.5)
        for k in range(cfg.n_enc_blocks):
            conv(f"enc.{k}.dw", ct, 1, 3, 1.0)
            conv(f"enc.{k}.pw1", ct * cfg.trunk_expand, ct, 1, 2.0)
            conv(f"enc.{k}.pw2", ct, ct * cfg.trunk_expand, 1, 1.0 / cfg.n_enc_blocks)
        conv("enc.y", cfg.c_y, ct, 1, _second_moment_yhat(cfg) / 2.0)
        conv("henc.0", cfg.c_hyper, 16 * cfg.c_y, 1, 2.0 / _second_moment_yhat(cfg))
        conv("henc.1", cfg.c_z, cfg.c_hyper, 3, 4.0)
    # frame-specific decoders (O8): distinct weights per frame index t.
    for t in range(cfg.T):
        for s in range(4):
            ci, co = cfg.dec_channels[s], cfg.dec_channels[s + 1]
            if s < 3:
                conv(f"dec.{t}.{s}", 4 * co, ci, 3, 2.0)
            else:   # linear output stage: mean 0.5, std ~0.2 (input second moment ~1.5)
                conv(f"dec.{t}.{s}", 4 * co, ci, 3, 0.04 / 1.5, bias_std=0.02, bias_mean=0.5)
    return out


def make_z(cfg: ChunkConfig) -> np.ndarray:
    """Hyper-latent z: round(N(0, 2^2)) clipped to +-15, int16 [n_chunks][C_z][h_z][w_z]."""
    rng = _rng(cfg, "z")
    z = np.rint(rng.normal(0.0, 2.0, size=(cfg.n_chunks, cfg.c_z, cfg.h_z, cfg.w_z)))
    return np.clip(z, -15, 15).astype(np.int16)


def make_uniform16(cfg: ChunkConfig) -> np.ndarray:
    """One uniform 16-bit draw per latent element, [n_chunks][h][w][C_y] (stream order).
    Each side turns it into a symbol by inverse-CDF on ITS OWN quantised table (R7)."""
    rng = _rng(cfg, "u16")
    return rng.integers(0, 1 << 16, size=(cfg.n_chunks, cfg.h, cfg.w, cfg.c_y), dtype=np.uint16)


def make_exact_law_params(cfg: ChunkConfig):
    """Entropy-only mode: mu and ln sigma drawn EXACTLY from the laws BASELINE.json states,
    [n_chunks][h][w][C_y] fp32 each."""
    rng = _rng(cfg, "exact")
    shape = (cfg.n_chunks, cfg.h, cfg.w, cfg.c_y)
    if cfg.mu_law == "normal":
        mu = rng.normal(0.0, 1.0, size=shape)
    else:
        mu = rng.uniform(-2.0, 2.0, size=shape)
    u = rng.uniform(math.log(cfg.scale_min), math.log(cfg.sigma_hi), size=shape)
    return mu.astype(np.float32), u.astype(np.float32)
