"""ufnvc_encode_chunk_dev_static: the GPU rANS encoder with its scratch in a file-scope __device__ array (no cudaMalloc in the
call), checked against ufnvc_encode_chunk_dev -- the existing path, itself byte-identical to the oracle's encoder
(tests/test_gpu_parity.py) -- on two calls in a row.  Byte work: the bar is bit-exact.

Collected last on purpose (the name): the suite runs with pytest -x.  Self-contained: no fixture of another test module, its
own handles, passes alone in a fresh process and after the rest of the suite.
"""
import numpy as np
import pytest
import torch

from paper_2606_04410_b200 import synth

pytestmark = pytest.mark.gpu


def _symbols(cfg, h, w, seed):
    """Seeded (idx, sym) maps for one chunk, channels-last: valid bucket indices and residuals inside the alphabet."""
    rng = np.random.default_rng(seed)
    idx = rng.integers(0, cfg.n_buckets, size=(1, h, w, cfg.c_y), dtype=np.uint8)
    sym = np.clip(np.rint(rng.laplace(scale=1.0 + idx.astype(np.float64) / 8.0)), -127, 127).astype(np.int16)
    return torch.from_numpy(idx).cuda(), torch.from_numpy(sym).cuda()


@pytest.mark.parametrize("name", ["cfg3-crop", "cfg3-1080p"])
def test_static_scratch_encode_matches_allocating_path_on_two_calls_in_a_row(name):
    from paper_2606_04410_b200 import binding
    cfg = synth.crop_config(synth.CONFIGS[3], 272, 480) if name == "cfg3-crop" else synth.CONFIGS[3]
    dec = binding.ChunkDecoder(cfg)                    # (the encoder needs the entropy tables only: no weights)
    try:
        a, b = _symbols(cfg, dec.h, dec.w, 1), _symbols(cfg, dec.h, dec.w, 2)
        G = cfg.lanes_per_substream // 32
        cap = 2 * a[0].numel() + dec.n_sub * (G * 140 + 16) + 64
        # outputs are the caller's: allocated here, before the calls under test
        outs = [(torch.zeros(cap, dtype=torch.uint8, device="cuda"), torch.zeros(dec.n_sub + 1, dtype=torch.int32, device="cuda"))
                for _ in range(3)]
        torch.cuda.synchronize()
        # two calls in a row on the shared array, different inputs; then the first input again over the second call's leftovers.
        # The handle has not run the allocating path yet, so nothing but the static array can be holding the scratch.
        dec.encode_chunk_dev_static(a[0], a[1], *outs[0])
        torch.cuda.synchronize()
        assert dec.get_status() == 0
        free_before = torch.cuda.mem_get_info()[0]
        dec.encode_chunk_dev_static(b[0], b[1], *outs[1])
        dec.encode_chunk_dev_static(a[0], a[1], *outs[2])
        torch.cuda.synchronize()
        assert dec.get_status() == 0
        assert torch.cuda.mem_get_info()[0] == free_before          # no device memory was taken by the calls
        # the existing path
        want = [dec.encode_chunk_dev(*x, cap=cap) for x in (a, b, a)]
        torch.cuda.synchronize()
        assert dec.get_status() == 0
        for (bits, off), (wbits, woff) in zip(outs, want):
            assert torch.equal(off, woff)
            n = int(woff[-1])
            assert n > 0 and torch.equal(bits[:n], wbits[:n])
        assert not torch.equal(outs[0][0], outs[1][0]) and torch.equal(outs[0][0], outs[2][0])
        # status bits behave as on the existing path: a symbol outside the alphabet, an output buffer that is too small
        bad = a[1].clone()
        bad.view(-1)[5] = 200
        dec.encode_chunk_dev_static(a[0], bad, *outs[1])
        torch.cuda.synchronize()
        assert dec.get_status() != 0
        small = torch.zeros(64, dtype=torch.uint8, device="cuda")
        dec.encode_chunk_dev_static(a[0], a[1], small, outs[1][1])
        torch.cuda.synchronize()
        assert dec.get_status() != 0 and int(outs[1][1][-1]) == int(want[0][1][-1])
        # and a clean call after the failed ones is clean again
        dec.encode_chunk_dev_static(b[0], b[1], *outs[0])
        torch.cuda.synchronize()
        assert dec.get_status() == 0 and torch.equal(outs[0][0][:int(want[1][1][-1])], want[1][0][:int(want[1][1][-1])])
    finally:
        dec.destroy()


def test_static_scratch_rejects_a_call_beyond_its_size():
    """Two 1080p chunks need 8.4 MB of scratch: more than UFNVC_STATIC_SCRATCH_BYTES (8 MiB).  Rejected with the byte counts, the
    outputs untouched; one chunk on the same handle still goes through."""
    from paper_2606_04410_b200 import binding
    cfg = synth.CONFIGS[3]
    dec = binding.ChunkDecoder(cfg, max_chunks=2)
    try:
        idx, sym = _symbols(cfg, dec.h, dec.w, 3)
        idx2, sym2 = torch.cat([idx, idx]), torch.cat([sym, sym])
        bits = torch.full((4 * idx2.numel(),), 7, dtype=torch.uint8, device="cuda")
        off = torch.full((2 * dec.n_sub + 1,), -1, dtype=torch.int32, device="cuda")
        with pytest.raises(binding.UfnvcError, match="static array holds 8388608"):
            dec.encode_chunk_dev_static(idx2, sym2, bits, off)
        torch.cuda.synchronize()
        assert int(bits.min()) == 7 and int(off.max()) == -1
        dec.encode_chunk_dev_static(idx, sym, bits, off[:dec.n_sub + 1])
        torch.cuda.synchronize()
        assert dec.get_status() == 0 and int(off[dec.n_sub]) > 0
    finally:
        dec.destroy()
