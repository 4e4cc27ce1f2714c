"""CPU-only checks of the boundary: the library loads, exports what include/ufnvc.h declares, host logic works."""
import ctypes as C
import dataclasses
import os
import re
import struct

import numpy as np
import pytest
import torch

from paper_2606_04410_b200 import binding, synth

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    src = open(os.path.join(ROOT, "include", "ufnvc.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(ufnvc_[a-z_0-9]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    names = declared_functions()
    assert "ufnvc_create" in names and "ufnvc_chunk_decode" in names and len(names) >= 12
    lib = C.CDLL(binding.LIB_PATH)
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(binding.EXPORTS) == names


def test_config_struct_layout():
    c = binding.make_config(synth.CONFIGS[3])
    assert c.struct_size == C.sizeof(binding.ufnvc_config) == 112
    assert (c.T, c.height, c.width, c.c_y) == (8, 1080, 1920, 128)
    assert list(c.dec_channels) == [256, 192, 128, 64, 3] and c.max_chunks_per_call == 1
    assert binding.make_config(synth.CONFIGS[4]).max_chunks_per_call == 4


def test_geometry_matches_survey_table():
    g = {k: (c.H, c.W, c.h, c.w, c.h_z, c.w_z, c.n_sub, c.n_symbols) for k, c in synth.CONFIGS.items()}
    assert g[1] == (64, 64, 4, 4, 1, 1, 1, 512)
    assert g[2] == (480, 832, 30, 52, 8, 13, 8, 199680)
    assert g[3] == (1088, 1920, 68, 120, 17, 30, 17, 1044480)
    assert g[4][6:] == (17, 1566720)
    assert g[5] == (2176, 3840, 136, 240, 34, 60, 34, 4177920)
    assert abs(synth.CONFIGS[3].macs_per_chunk() / 1e9 - 894.4) < 0.5
    assert abs(synth.CONFIGS[2].macs_per_chunk() / 1e9 - 79.2) < 0.5


def test_blob_round_trip():
    cfg = synth.CONFIGS[1]
    w = synth.make_weights(cfg)
    blob = binding.pack_weights_blob(w, cfg.weight_dtype)
    assert blob[:8] == b"UFNVCW01"
    n = struct.unpack_from("<I", blob, 8)[0]
    assert n == len(w)
    seen = {}
    for i in range(n):
        name, dt, nd, s0, s1, s2, s3, off, nb = struct.unpack_from("<40sII4IQQ", blob, 16 + 80 * i)
        name = name.rstrip(b"\0").decode()
        assert off % 16 == 0 and off + nb <= len(blob)
        a = np.frombuffer(blob, np.float32 if dt == 0 else np.uint16, count=nb // (4 if dt == 0 else 2), offset=off)
        seen[name] = a.reshape([s0, s1, s2, s3][:nd])
    for k, v in w.items():
        assert np.array_equal(seen[k], v)
    cfg2 = synth.crop_config(synth.CONFIGS[2], 64, 64)
    w2 = synth.make_weights(cfg2)
    blob2 = binding.pack_weights_blob(w2, 1)
    assert len(blob2) < sum(v.nbytes for v in w2.values())       # conv weights stored as bf16
    w2["xframe.w"] = w2["xframe.w"] + np.float32(1e-5)
    with pytest.raises(ValueError):
        binding.pack_weights_blob(w2, 1)


def test_concat_streams():
    a = (np.arange(8, dtype=np.uint8), np.array([0, 4, 8], np.uint32))
    b = (np.arange(12, dtype=np.uint8), np.array([0, 8, 12], np.uint32))
    bits, off = binding.concat_streams([a, b])
    assert bits.size == 20 and list(off) == [0, 4, 8, 16, 20]


@pytest.mark.skipif(torch.cuda.is_available(), reason="CPU-box behaviour")
def test_no_gpu_fails_loudly():
    c = binding.make_config(synth.CONFIGS[1])
    h = C.c_void_p()
    assert binding.LIB.ufnvc_create(C.byref(c), C.byref(h)) == -6 and not h.value     # UFNVC_E_CUDA, no handle
    with pytest.raises(binding.UfnvcError):
        binding.ChunkDecoder(synth.CONFIGS[1])
    assert binding.LIB.ufnvc_create(None, None) == -1
    c.struct_size = 4
    assert binding.LIB.ufnvc_create(C.byref(c), C.byref(h)) == -2                       # validated before the device
    assert binding.LIB.ufnvc_last_error(None) == b"null handle"


def test_mu_steps_is_validated_before_the_device():
    """mu_steps (NEXT-1, R21): 1 or 4; 4 needs c_y % 32 == 0 (the mean convs exist on the tensor-core path only)."""
    h = C.c_void_p()
    for steps, c_y, want_bad in ((1, 32, False), (4, 32, False), (2, 32, True), (0, 32, True), (4, 24, True), (4, 128, False)):
        c = binding.make_config(dataclasses.replace(synth.CONFIGS[1], mu_steps=steps, c_y=c_y))
        rc = binding.LIB.ufnvc_create(C.byref(c), C.byref(h))
        if want_bad:
            assert rc == -2, (steps, c_y, rc)                                           # UFNVC_E_BAD_CONFIG
        else:
            assert rc != -2, (steps, c_y, rc)
            if rc == 0:
                binding.LIB.ufnvc_destroy(h)


def test_progressive_weights_and_blob():
    cfg = synth.progressive_config(synth.CONFIGS[2])
    assert cfg.mu_steps == 4 and cfg.name.endswith("-pmu") and synth.CONFIGS[2].mu_steps == 1
    w = synth.make_weights(synth.crop_config(cfg, 64, 64))
    for k in (1, 2, 3):
        assert w[f"mu.{k}.w"].shape == (cfg.c_y, 2 * cfg.c_y, 3, 3) and w[f"mu.{k}.b"].shape == (cfg.c_y,)
        assert np.array_equal(synth.round_to_bf16(w[f"mu.{k}.w"]), w[f"mu.{k}.w"])      # bf16-representable
    assert not any(k.startswith("mu.") for k in synth.make_weights(synth.crop_config(synth.CONFIGS[2], 64, 64)))
    assert cfg.macs_per_chunk() - synth.CONFIGS[2].macs_per_chunk() == 3 * cfg.h * cfg.w * 9 * 2 * cfg.c_y * cfg.c_y
    blob = binding.pack_weights_blob(w, cfg.weight_dtype)
    assert b"mu.3.w" in blob
