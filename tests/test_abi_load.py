"""CPU-only: the C-ABI library builds/loads and exports every symbol include/bfsc.h declares;
host-only entry points agree with FORMAT.md. No GPU compute here."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    from paper_1704_00513_b200 import build, binding
    build.build()
    return binding.lib()


def test_exports_match_header(L):
    hdr = open(os.path.join(ROOT, "include", "bfsc.h")).read()
    declared = set(re.findall(r"\b(bfsc_[a-z_0-9]+)\s*\(", hdr))
    assert declared, "no declarations found"
    from paper_1704_00513_b200 import binding
    assert declared == set(binding.EXPORTS)
    for name in declared:
        assert hasattr(L, name), name


def test_bounds_match_format(L, oracle_mod):
    from paper_1704_00513_b200 import binding
    for W in (32, 64):
        for n in (0, 1, 127, 128, 129, 1000, 1 << 20):
            nb = (n + 127) // 128
            pfor = 32 + (4 * (nb + 1) + 15) // 16 * 16 + nb * (16 + 16 * W)
            raw = 32 + (n * W // 8 + 15) // 16 * 16
            assert binding.compress_bound(n, W) == max(pfor, raw)
            assert binding.compress_bound(n, W) >= oracle_mod.compress_bound(n, W)
    assert binding.batch_compress_bound([0, 5, 300], 32) == sum(binding.compress_bound(n, 32) for n in (0, 5, 300))
    assert binding.workspace_bytes(1 << 24, 1, 32) > (1 << 24) // 128 // 64 * 64   # one 64-byte look-back state per 64-block tile
    assert L.bfsc_version() >> 16 == 1 and L.bfsc_version() & 0xffff >= 2


def test_host_arg_validation(L):
    # host-detectable errors are reported without touching the device
    rc = L.bfsc_compress(None, 10, 32, 0, None, 0, None, None, 0, None, None)
    assert rc == 1
    rc = L.bfsc_compress_batch(None, None, 1, 16, 0, None, 0, None, None, 0, None, None)
    assert rc == 1
    rc = L.bfsc_decompress(None, 0, 32, None, 0, None, None, 0, None, None)
    assert rc == 1
    for bad_codec in (0, 3):                       # bfsc_codec: 1 = PFOR, 2 = BP128 (include/bfsc.h)
        assert L.bfsc_compress_codec(bad_codec, None, 0, 32, 0, None, 0, None, None, 0, None, None) == 1
        assert L.bfsc_compress_batch_codec(bad_codec, None, None, 1, 32, 0, None, 0, None, None, 0, None, None) == 1


def test_no_fallback_when_library_missing(monkeypatch):
    from paper_1704_00513_b200 import binding
    monkeypatch.setattr(binding, "_lib", None)
    monkeypatch.setattr(binding, "SO_PATH", "/nonexistent/libbfsc.so")
    with pytest.raises(RuntimeError):
        binding.lib()
