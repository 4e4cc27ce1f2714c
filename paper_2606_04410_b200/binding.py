"""Thin ctypes binding of libufnvc.so (include/ufnvc.h).  Argument marshalling only: every step of the path runs in
the library's CUDA kernels.  PyTorch is used for device memory and streams, nothing else.

There is no fallback: if the shared library is missing or does not load, importing this module raises.
"""
from __future__ import annotations

import ctypes as C
import os
import struct

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libufnvc.so")


class UfnvcError(RuntimeError):
    pass


class ufnvc_config(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("T", C.c_int32), ("height", C.c_int32), ("width", C.c_int32),
                ("c_y", C.c_int32), ("c_z", C.c_int32), ("c_hyper", C.c_int32), ("c_trunk", C.c_int32),
                ("n_trunk_blocks", C.c_int32), ("trunk_expand", C.c_int32), ("dec_channels", C.c_int32 * 5),
                ("n_buckets", C.c_int32), ("scale_min", C.c_double), ("scale_max", C.c_double),
                ("rows_per_substream", C.c_int32), ("lanes_per_substream", C.c_int32),
                ("max_chunks_per_call", C.c_int32), ("weight_dtype", C.c_int32), ("mu_steps", C.c_int32),
                ("debug_flags", C.c_uint32), ("n_ctx_blocks", C.c_int32), ("n_enc_blocks", C.c_int32)]


class ufnvc_taps(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("mu", C.c_void_p), ("lnscale", C.c_void_p), ("idx", C.c_void_p),
                ("sym", C.c_void_p), ("yhat", C.c_void_p), ("f0", C.c_void_p), ("trunk", C.c_void_p),
                ("stage", C.c_void_p * 3)]


class ufnvc_enc_taps(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("y", C.c_void_p), ("zf", C.c_void_p), ("sym", C.c_void_p), ("mu", C.c_void_p),
                ("idx", C.c_void_p)]


def _load():
    if not os.path.exists(LIB_PATH):
        raise UfnvcError(f"{LIB_PATH} is missing: run `python -m paper_2606_04410_b200.build` "
                         "(__graft_entry__.build()). There is no CPU fallback.")
    lib = C.CDLL(LIB_PATH)
    vp, i, sz = C.c_void_p, C.c_int, C.c_size_t
    sig = {
        "ufnvc_create": (i, [C.POINTER(ufnvc_config), C.POINTER(vp)]),
        "ufnvc_destroy": (i, [vp]),
        "ufnvc_load_weights": (i, [vp, vp, sz]),
        "ufnvc_chunk_decode": (i, [vp, i, vp, vp, sz, vp, vp, vp]),
        "ufnvc_chunk_decode_ex": (i, [vp, i, vp, vp, sz, vp, vp, vp, vp, vp, C.POINTER(ufnvc_taps)]),
        "ufnvc_entropy_params": (i, [vp, i, vp, vp, vp, vp, vp]),
        "ufnvc_get_status": (i, [vp, C.POINTER(C.c_uint32)]),
        "ufnvc_last_error": (C.c_char_p, [vp]),
        "ufnvc_launches_per_call": (i, [vp, i]),
        "ufnvc_chunk_decode_profiled": (i, [vp, i, vp, vp, sz, vp, vp, vp, i, C.POINTER(C.c_float)]),
        "ufnvc_debug_counter": (i, [vp, i, C.POINTER(C.c_uint64)]),
        "ufnvc_get_cdf": (i, [vp, vp]),
        "ufnvc_symbols_from_uniform": (i, [vp, vp, vp, sz, vp]),
        "ufnvc_encode_chunk": (C.c_long, [vp, vp, vp, vp, sz, vp]),
        "ufnvc_decode_z": (i, [vp, i, vp, sz, vp, vp, vp]),
        "ufnvc_chunk_decode_bytes": (i, [vp, i, vp, sz, vp, vp, vp]),
        "ufnvc_get_z_prior_index": (i, [vp, vp]),
        "ufnvc_encode_z": (C.c_long, [vp, vp, vp, sz, vp]),
        "ufnvc_encode_chunk_dev": (i, [vp, i, vp, vp, vp, sz, vp, vp]),
        "ufnvc_encode_chunk_dev_static": (i, [vp, i, vp, vp, vp, sz, vp, vp]),
        "ufnvc_chunk_encode": (i, [vp, i, vp, vp, sz, vp, vp, C.POINTER(ufnvc_enc_taps), vp]),
        "ufnvc_convert_colour": (i, [vp, vp, i, i, i, i, vp]),
        "ufnvc_reset_context": (i, [vp, i, vp]),
        "ufnvc_get_context": (i, [vp, i, vp, vp]),
        "ufnvc_set_context": (i, [vp, i, vp, vp]),
    }
    for name, (res, args) in sig.items():
        fn = getattr(lib, name)
        fn.restype, fn.argtypes = res, args
    return lib


LIB = _load()
EXPORTS = ("ufnvc_create", "ufnvc_destroy", "ufnvc_load_weights", "ufnvc_chunk_decode", "ufnvc_chunk_decode_ex",
           "ufnvc_entropy_params", "ufnvc_get_status", "ufnvc_last_error", "ufnvc_launches_per_call",
           "ufnvc_chunk_decode_profiled", "ufnvc_debug_counter", "ufnvc_get_cdf", "ufnvc_symbols_from_uniform", "ufnvc_encode_chunk",
           "ufnvc_decode_z", "ufnvc_chunk_decode_bytes", "ufnvc_get_z_prior_index", "ufnvc_encode_z", "ufnvc_encode_chunk_dev", "ufnvc_encode_chunk_dev_static",
           "ufnvc_reset_context", "ufnvc_get_context", "ufnvc_set_context", "ufnvc_chunk_encode", "ufnvc_convert_colour")


# ufnvc_config.debug_flags (include/ufnvc.h)
DBG = dict(force_generic=0x01, no_pdl=0x02, no_tail_fill=0x04, fp64_head=0x08, no_cta_pairs=0x10, unfused_trunk=0x20,
           generic_final=0x40, plain_depthwise=0x80, no_transposed_tiles=0x100, no_quad_clusters=0x200)


def make_config(cfg, max_chunks: int | None = None, debug_flags: int = 0) -> ufnvc_config:
    """cfg: any object with the ufnvc_config field names (e.g. synth.ChunkConfig)."""
    c = ufnvc_config()
    c.struct_size = C.sizeof(ufnvc_config)
    for f in ("T", "height", "width", "c_y", "c_z", "c_hyper", "c_trunk", "n_trunk_blocks", "trunk_expand", "n_buckets",
              "scale_min", "scale_max", "rows_per_substream", "lanes_per_substream", "weight_dtype"):
        setattr(c, f, getattr(cfg, f))
    c.dec_channels = (C.c_int32 * 5)(*cfg.dec_channels)
    c.max_chunks_per_call = max_chunks if max_chunks is not None else getattr(cfg, "n_chunks", 1)
    c.mu_steps = getattr(cfg, "mu_steps", 1)
    c.debug_flags = debug_flags
    c.n_ctx_blocks = getattr(cfg, "n_ctx_blocks", 0)
    c.n_enc_blocks = getattr(cfg, "n_enc_blocks", 0)
    return c


def pack_weights_blob(weights: dict, weight_dtype: int) -> bytes:
    """Serialise {name: fp32 ndarray} into the blob format of ufnvc_load_weights (include/ufnvc.h).
    Conv weights ('.w') are stored as bf16 when weight_dtype == 1 (they must already be bf16-representable)."""
    names = sorted(weights)
    head = 16 + 80 * len(names)
    off = (head + 15) // 16 * 16
    entries, chunks = [], []
    for nme in names:
        a = np.ascontiguousarray(weights[nme], dtype=np.float32)
        if weight_dtype == 1 and nme.endswith(".w"):
            u = a.view(np.uint32)
            if (u & 0xFFFF).any():
                raise ValueError(f"{nme}: not bf16-representable")
            data, dt = (u >> 16).astype(np.uint16).tobytes(), 1
        else:
            data, dt = a.tobytes(), 0
        shape = list(a.shape) + [1] * (4 - a.ndim)
        entries.append(struct.pack("<40sII4IQQ", nme.encode(), dt, a.ndim, *shape, off, len(data)))
        pad = (-len(data)) % 16
        chunks.append(data + b"\0" * pad)
        off += len(data) + pad
    blob = b"UFNVCW01" + struct.pack("<II", len(names), 0) + b"".join(entries)
    blob += b"\0" * ((-len(blob)) % 16)
    return blob + b"".join(chunks)


def _ptr(t):
    if t is None:
        return None
    if isinstance(t, torch.Tensor):
        assert t.is_contiguous()
        return C.c_void_p(t.data_ptr())
    assert t.flags["C_CONTIGUOUS"]
    return C.c_void_p(t.ctypes.data)


class ChunkDecoder:
    """One ufnvc_handle.  Methods carry the names of the C entry points they call."""

    def __init__(self, cfg, max_chunks: int | None = None, device: int = 0, debug_flags: int = 0):
        if not torch.cuda.is_available():
            raise UfnvcError("ufnvc needs a CUDA device (sm_100); there is no CPU fallback")
        torch.cuda.set_device(device)
        self.device = torch.device("cuda", device)
        self.cfg = cfg
        self.c = make_config(cfg, max_chunks, debug_flags)
        self.H = -(-cfg.height // 32) * 32
        self.W = -(-cfg.width // 32) * 32
        self.h, self.w = self.H // 16, self.W // 16
        self.h_z, self.w_z = -(-self.h // 4), -(-self.w // 4)
        self.n_sub = -(-self.h // cfg.rows_per_substream)
        self.n_sub_z = -(-self.h_z // cfg.rows_per_substream)
        hp = C.c_void_p()
        rc = LIB.ufnvc_create(C.byref(self.c), C.byref(hp))
        if rc != 0:
            raise UfnvcError(f"ufnvc_create failed: {rc}")
        self.handle = hp

    def _check(self, rc, what):
        if rc < 0:
            raise UfnvcError(f"{what} failed ({rc}): {LIB.ufnvc_last_error(self.handle).decode()}")
        return rc

    def destroy(self):
        if self.handle:
            LIB.ufnvc_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    def load_weights(self, weights: dict):
        blob = pack_weights_blob(weights, self.cfg.weight_dtype)
        buf = np.frombuffer(blob, np.uint8)
        self._check(LIB.ufnvc_load_weights(self.handle, _ptr(buf), len(blob)), "ufnvc_load_weights")

    def _stream(self, stream):
        s = stream if stream is not None else torch.cuda.current_stream()
        return C.c_void_p(s.cuda_stream)

    def new_frames(self, n_chunks=1):
        return torch.empty((n_chunks, self.cfg.T, 3, self.cfg.height, self.cfg.width), dtype=torch.float32, device=self.device)

    def chunk_decode(self, z, bits, sub_off, frames=None, stream=None, n_chunks=None):
        n = n_chunks or z.shape[0]
        frames = frames if frames is not None else self.new_frames(n)
        self._check(LIB.ufnvc_chunk_decode(self.handle, n, _ptr(z), _ptr(bits), bits.numel(), _ptr(sub_off), _ptr(frames),
                                           self._stream(stream)), "ufnvc_chunk_decode")
        return frames

    def chunk_decode_ex(self, z, bits, sub_off, frames=None, stream=None, idx_override=None, mu_override=None,
                        taps=False, want_frames=True):
        n = z.shape[0]
        cfg, dev = self.cfg, self.device
        if want_frames and frames is None:
            frames = self.new_frames(n)
        tp, out = None, {}
        if taps:
            e = (n, self.h, self.w, cfg.c_y)
            out = dict(mu=torch.empty(e, dtype=torch.float32, device=dev), lnscale=torch.empty(e, dtype=torch.float32, device=dev),
                       idx=torch.empty(e, dtype=torch.uint8, device=dev), sym=torch.empty(e, dtype=torch.int16, device=dev),
                       yhat=torch.empty(e, dtype=torch.float32, device=dev))
            if want_frames:
                f = (n, cfg.T, self.h, self.w, cfg.c_trunk)
                out["f0"] = torch.empty(f, dtype=torch.bfloat16, device=dev)
                out["trunk"] = torch.empty(f, dtype=torch.bfloat16, device=dev)
                out["stage"] = [torch.empty((n, cfg.T, self.h << s, self.w << s, cfg.dec_channels[s]), dtype=torch.bfloat16,
                                            device=dev) for s in (1, 2, 3)]
            tp = ufnvc_taps()
            tp.struct_size = C.sizeof(ufnvc_taps)
            for k in ("mu", "lnscale", "idx", "sym", "yhat", "f0", "trunk"):
                if k in out:
                    setattr(tp, k, out[k].data_ptr())
            if "stage" in out:
                tp.stage = (C.c_void_p * 3)(*[t.data_ptr() for t in out["stage"]])
        self._check(LIB.ufnvc_chunk_decode_ex(self.handle, n, _ptr(z), _ptr(bits), bits.numel(), _ptr(sub_off),
                                              _ptr(frames) if want_frames else None, self._stream(stream), _ptr(idx_override),
                                              _ptr(mu_override), C.byref(tp) if tp is not None else None), "ufnvc_chunk_decode_ex")
        out["frames"] = frames
        return out

    # ---- chunk encode (NEXT-4, R24) ----
    def chunk_encode(self, frames, cap=None, taps=False, stream=None):
        """frames: float32 device tensor [n][T][3][height][width] -> dict(bits uint8 [cap], sub_off int32, z int16, + taps)."""
        n, cfg, dev = frames.shape[0], self.cfg, self.device
        G = cfg.lanes_per_substream // 32
        ne = self.h * self.w * cfg.c_y
        cap = cap if cap is not None else n * (2 * ne + self.n_sub * (G * 140 + 16) + 64)
        out = dict(bits=torch.zeros(cap, dtype=torch.uint8, device=dev), sub_off=torch.zeros(n * self.n_sub + 1, dtype=torch.int32, device=dev),
                   z=torch.empty((n, cfg.c_z, self.h_z, self.w_z), dtype=torch.int16, device=dev))
        tp = None
        if taps:
            e = (n, self.h, self.w, cfg.c_y)
            out.update(y=torch.empty(e, dtype=torch.float32, device=dev), zf=torch.empty((n, cfg.c_z, self.h_z, self.w_z), dtype=torch.float32, device=dev),
                       sym=torch.empty(e, dtype=torch.int16, device=dev), mu=torch.empty(e, dtype=torch.float32, device=dev),
                       idx=torch.empty(e, dtype=torch.uint8, device=dev))
            tp = ufnvc_enc_taps()
            tp.struct_size = C.sizeof(ufnvc_enc_taps)
            for k in ("y", "zf", "sym", "mu", "idx"):
                setattr(tp, k, out[k].data_ptr())
        self._check(LIB.ufnvc_chunk_encode(self.handle, n, _ptr(frames), _ptr(out["bits"]), cap, _ptr(out["sub_off"]), _ptr(out["z"]),
                                           C.byref(tp) if tp is not None else None, self._stream(stream)), "ufnvc_chunk_encode")
        return out

    # ---- temporal chunk context (NEXT-2a, R23) ----
    def reset_context(self, n_chunks=1, stream=None):
        self._check(LIB.ufnvc_reset_context(self.handle, n_chunks, self._stream(stream)), "ufnvc_reset_context")

    def get_context(self, n_chunks=1, stream=None):
        ctx = torch.empty((n_chunks, self.h, self.w, self.cfg.c_trunk), dtype=torch.bfloat16, device=self.device)
        self._check(LIB.ufnvc_get_context(self.handle, n_chunks, _ptr(ctx), self._stream(stream)), "ufnvc_get_context")
        return ctx

    def set_context(self, ctx, stream=None):
        assert ctx.dtype == torch.bfloat16 and ctx.shape[1:] == (self.h, self.w, self.cfg.c_trunk)
        self._check(LIB.ufnvc_set_context(self.handle, ctx.shape[0], _ptr(ctx), self._stream(stream)), "ufnvc_set_context")

    # ---- bytes-only entry points (NEXT-3, R22) ----
    def decode_z(self, bits, sub_off, n_chunks=1, stream=None):
        z = torch.empty((n_chunks, self.cfg.c_z, self.h_z, self.w_z), dtype=torch.int16, device=self.device)
        self._check(LIB.ufnvc_decode_z(self.handle, n_chunks, _ptr(bits), bits.numel(), _ptr(sub_off), _ptr(z), self._stream(stream)),
                    "ufnvc_decode_z")
        return z

    def chunk_decode_bytes(self, bits, sub_off, n_chunks=1, frames=None, stream=None):
        frames = frames if frames is not None else self.new_frames(n_chunks)
        self._check(LIB.ufnvc_chunk_decode_bytes(self.handle, n_chunks, _ptr(bits), bits.numel(), _ptr(sub_off), _ptr(frames),
                                                 self._stream(stream)), "ufnvc_chunk_decode_bytes")
        return frames

    def get_z_prior_index(self) -> np.ndarray:
        idx = np.empty(self.cfg.c_z, np.uint8)
        self._check(LIB.ufnvc_get_z_prior_index(self.handle, _ptr(idx)), "ufnvc_get_z_prior_index")
        return idx

    def encode_z(self, z: np.ndarray):
        """z: int16 [c_z][h_z][w_z] host array of ONE chunk -> (bytes uint8, sub_off uint32 [n_sub_z+1])."""
        z = np.ascontiguousarray(z, np.int16)
        G = self.cfg.lanes_per_substream // 32
        cap = 2 * z.size + self.n_sub_z * (G * 140 + 16) + 64
        bits = np.zeros(cap, np.uint8)
        off = np.zeros(self.n_sub_z + 1, np.uint32)
        n = self._check(LIB.ufnvc_encode_z(self.handle, _ptr(z), _ptr(bits), cap, _ptr(off)), "ufnvc_encode_z")
        return bits[:n].copy(), off

    def encode_chunk_dev(self, idx, sym, cap=None, stream=None):
        """GPU rANS encode (NEXT-4): idx uint8, sym int16 device tensors [n][h][w][c_y] -> (bits uint8 [cap], sub_off int32)."""
        n = idx.shape[0]
        G = self.cfg.lanes_per_substream // 32
        cap = cap if cap is not None else n * (2 * idx[0].numel() + self.n_sub * (G * 140 + 16) + 64)
        bits = torch.zeros(cap, dtype=torch.uint8, device=self.device)
        off = torch.zeros(n * self.n_sub + 1, dtype=torch.int32, device=self.device)
        self._check(LIB.ufnvc_encode_chunk_dev(self.handle, n, _ptr(idx), _ptr(sym), _ptr(bits), cap, _ptr(off), self._stream(stream)),
                    "ufnvc_encode_chunk_dev")
        return bits, off

    def encode_chunk_dev_static(self, idx, sym, bits, off, stream=None):
        """ufnvc_encode_chunk_dev_static: the same encode into caller-provided outputs (bits uint8 [cap], off int32 [n * n_sub + 1]);
        neither this wrapper nor the library call allocates device memory.  Calls sharing a GPU must not overlap."""
        self._check(LIB.ufnvc_encode_chunk_dev_static(self.handle, idx.shape[0], _ptr(idx), _ptr(sym), _ptr(bits), bits.numel(), _ptr(off),
                                                      self._stream(stream)), "ufnvc_encode_chunk_dev_static")

    def entropy_params(self, z, stream=None):
        n = z.shape[0]
        e = (n, self.h, self.w, self.cfg.c_y)
        mu = torch.empty(e, dtype=torch.float32, device=self.device)
        ls = torch.empty(e, dtype=torch.float32, device=self.device)
        idx = torch.empty(e, dtype=torch.uint8, device=self.device)
        self._check(LIB.ufnvc_entropy_params(self.handle, n, _ptr(z), _ptr(mu), _ptr(ls), _ptr(idx), self._stream(stream)),
                    "ufnvc_entropy_params")
        return mu, ls, idx

    def get_status(self) -> int:
        v = C.c_uint32(0)
        self._check(LIB.ufnvc_get_status(self.handle, C.byref(v)), "ufnvc_get_status")
        return int(v.value)

    def debug_counter(self, which: int = 0) -> int:
        v = C.c_uint64(0)
        self._check(LIB.ufnvc_debug_counter(self.handle, which, C.byref(v)), "ufnvc_debug_counter")
        return int(v.value)

    def launches_per_call(self, n_chunks=1) -> int:
        return self._check(LIB.ufnvc_launches_per_call(self.handle, n_chunks), "ufnvc_launches_per_call")

    def chunk_decode_profiled(self, z, bits, sub_off, frames, stream=None, detail=False):
        us = (C.c_float * 8)()
        self._check(LIB.ufnvc_chunk_decode_profiled(self.handle, z.shape[0], _ptr(z), _ptr(bits), bits.numel(), _ptr(sub_off),
                                                    _ptr(frames), self._stream(stream), int(detail), us), "ufnvc_chunk_decode_profiled")
        return dict(zip(("A1+A2", "A3+A4", "A5", "A6+A7", "A8", "A9", "A6", "ctx"), [float(x) for x in us]))

    # ---- encoder-side fixtures (host) ----
    def get_cdf(self) -> np.ndarray:
        cdf = np.empty((self.cfg.n_buckets, 256), np.uint32)
        self._check(LIB.ufnvc_get_cdf(self.handle, _ptr(cdf)), "ufnvc_get_cdf")
        return cdf

    def symbols_from_uniform(self, idx: np.ndarray, u16: np.ndarray) -> np.ndarray:
        idx = np.ascontiguousarray(idx, np.uint8)
        u16 = np.ascontiguousarray(u16, np.uint16)
        sym = np.empty(idx.shape, np.int16)
        self._check(LIB.ufnvc_symbols_from_uniform(self.handle, _ptr(idx), _ptr(u16), idx.size, _ptr(sym)),
                    "ufnvc_symbols_from_uniform")
        return sym

    def encode_chunk(self, idx: np.ndarray, sym: np.ndarray):
        """idx, sym: [h][w][c_y] host arrays of ONE chunk -> (bytes uint8, sub_off uint32 [n_sub+1])."""
        idx = np.ascontiguousarray(idx, np.uint8)
        sym = np.ascontiguousarray(sym, np.int16)
        G = self.cfg.lanes_per_substream // 32
        cap = 2 * sym.size + self.n_sub * (G * 140 + 16) + 64
        bits = np.zeros(cap, np.uint8)
        off = np.zeros(self.n_sub + 1, np.uint32)
        n = self._check(LIB.ufnvc_encode_chunk(self.handle, _ptr(idx), _ptr(sym), _ptr(bits), cap, _ptr(off)), "ufnvc_encode_chunk")
        return bits[:n].copy(), off


def convert_colour(x, to_yuv: bool, stream=None):
    """BT.709 full-range RGB <-> YUV444 on a float32 device tensor [..., 3, H, W] (ufnvc_convert_colour); returns a new tensor."""
    assert x.dtype == torch.float32 and x.is_cuda and x.shape[-3] == 3 and x.is_contiguous()
    out = torch.empty_like(x)
    n_img = x.numel() // (3 * x.shape[-2] * x.shape[-1])
    s = stream if stream is not None else torch.cuda.current_stream()
    rc = LIB.ufnvc_convert_colour(_ptr(x), _ptr(out), n_img, x.shape[-2], x.shape[-1], int(to_yuv), C.c_void_p(s.cuda_stream))
    if rc != 0:
        raise UfnvcError(f"ufnvc_convert_colour failed ({rc})")
    return out


def pack_chunk_bytes(z_bits, z_off, y_bits, y_off):
    """One chunk's container for ufnvc_chunk_decode_bytes: z substreams, then y substreams, one offset table."""
    off = np.concatenate([np.asarray(z_off, np.int64), np.asarray(y_off, np.int64)[1:] + int(z_off[-1])])
    return np.concatenate([z_bits, y_bits]), off.astype(np.uint32)


def concat_streams(parts):
    """[(bits, sub_off)] per chunk -> (bits, sub_off[n_chunks*n_sub+1]) for one multi-chunk call."""
    bits, offs, base = [], [np.zeros(1, np.uint32)], 0
    for b, o in parts:
        bits.append(b)
        offs.append((o[1:].astype(np.uint64) + base).astype(np.uint32))
        base += int(o[-1])
    return np.concatenate(bits), np.concatenate(offs)
