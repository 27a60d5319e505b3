"""ctypes binding of the ORACLE (oracle/bfsc_ref.c) — test infrastructure, not the product.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
import this package. It does not import the CUDA package and shares no code with it.
`build()` compiles bfsc_ref.c with gcc into oracle/libbfsc_ref.so (building the checker is
not using it). All functions take and return numpy arrays on the host.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libbfsc_ref.so")
_SRC = os.path.join(_HERE, "bfsc_ref.c")
_HDR = os.path.join(_HERE, "bfsc_ref.h")
_lib = None

OK, ERR_INVALID_ARG, ERR_DST_TOO_SMALL, ERR_CORRUPT = 0, 1, 2, 3
CODEC_PFOR, CODEC_BP128 = 1, 2          # encoder rule = mode byte of the stream (FORMAT.md §1, §7)
FLAG_RAW_FALLBACK = 0x200               # OR-ed into the rule: RAW when the rule does not shrink the stream (FORMAT.md §8)


class OracleError(RuntimeError):
    def __init__(self, code):
        super().__init__(f"bfsc_ref error {code}")
        self.code = code


def build(force: bool = False) -> str:
    """gcc -O2 -shared; rebuilt when the source is newer than the .so."""
    stale = (not os.path.exists(_SO)
             or os.path.getmtime(_SO) < max(os.path.getmtime(_SRC), os.path.getmtime(_HDR)))
    if force or stale:
        cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-Wall", "-Wextra",
               "-o", _SO, _SRC, "-lpthread"]
        subprocess.run(cmd, check=True, cwd=_HERE)
    return _SO


def lib():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_SO)
        c = ctypes
        vp, sz, i32 = c.c_void_p, c.c_size_t, c.c_int
        L.bfsc_ref_width.restype = i32
        L.bfsc_ref_width.argtypes = [c.c_uint64]
        L.bfsc_ref_block_bytes.restype = sz
        L.bfsc_ref_block_bytes.argtypes = [i32, i32, i32]
        L.bfsc_ref_compress_bound.restype = sz
        L.bfsc_ref_compress_bound.argtypes = [sz, i32]
        L.bfsc_ref_block_deltas.restype = c.c_uint64
        L.bfsc_ref_block_deltas.argtypes = [vp, i32, i32, vp]
        L.bfsc_ref_choose_b.restype = i32
        L.bfsc_ref_choose_b.argtypes = [vp, i32, c.POINTER(i32)]
        L.bfsc_ref_emit_block.restype = sz
        L.bfsc_ref_emit_block.argtypes = [vp, c.c_uint64, i32, i32, vp]
        L.bfsc_ref_compress.restype = i32
        L.bfsc_ref_compress.argtypes = [vp, sz, i32, sz, vp, sz, c.POINTER(sz)]
        L.bfsc_ref_choose_b_bp128.restype = i32
        L.bfsc_ref_choose_b_bp128.argtypes = [vp]
        L.bfsc_ref_compress_codec.restype = i32
        L.bfsc_ref_compress_codec.argtypes = [i32, vp, sz, i32, sz, vp, sz, c.POINTER(sz)]
        L.bfsc_ref_compress_batch_codec.restype = i32
        L.bfsc_ref_compress_batch_codec.argtypes = [i32, vp, vp, sz, i32, sz, vp, sz, vp]
        L.bfsc_ref_decompress.restype = i32
        L.bfsc_ref_decompress.argtypes = [vp, sz, i32, vp, sz, c.POINTER(sz)]
        L.bfsc_ref_compress_batch.restype = i32
        L.bfsc_ref_compress_batch.argtypes = [vp, vp, sz, i32, sz, vp, sz, vp]
        L.bfsc_ref_decompress_batch.restype = i32
        L.bfsc_ref_decompress_batch.argtypes = [vp, vp, sz, i32, vp, sz, vp]
        L.bfsc_ref_compress_batch_mt.restype = i32
        L.bfsc_ref_compress_batch_mt.argtypes = [vp, vp, sz, i32, sz, vp, sz, vp, i32]
        L.bfsc_ref_decompress_batch_mt.restype = i32
        L.bfsc_ref_decompress_batch_mt.argtypes = [vp, vp, sz, i32, vp, sz, vp, i32]
        L.bfsc_ref_compress_bitmap.restype = i32
        L.bfsc_ref_compress_bitmap.argtypes = [i32, vp, sz, c.c_uint64, i32, sz, vp, sz, c.POINTER(sz)]
        L.bfsc_ref_decompress_to_bitmap.restype = i32
        L.bfsc_ref_decompress_to_bitmap.argtypes = [vp, sz, i32, c.c_uint64, vp, sz, c.POINTER(sz)]
        L.bfsc_ref_decompress_to_frontier.restype = i32
        L.bfsc_ref_decompress_to_frontier.argtypes = [vp, sz, i32, c.c_uint64, vp, vp, sz, c.POINTER(sz)]
        L.bfsc_ref_vbitmap_bound.restype = sz
        L.bfsc_ref_vbitmap_bound.argtypes = [sz]
        L.bfsc_ref_compress_vbitmap.restype = i32
        L.bfsc_ref_compress_vbitmap.argtypes = [i32, vp, sz, vp, sz, c.POINTER(sz)]
        L.bfsc_ref_decompress_vbitmap.restype = i32
        L.bfsc_ref_decompress_vbitmap.argtypes = [vp, sz, vp, sz]
        _lib = L
    return _lib


def _W(a: np.ndarray) -> int:
    if a.dtype == np.uint32:
        return 32
    if a.dtype == np.uint64:
        return 64
    raise TypeError(f"ids must be uint32 or uint64, got {a.dtype}")


def _dtype(W: int):
    return {32: np.uint32, 64: np.uint64}[W]


def _p(a: np.ndarray):
    return a.ctypes.data_as(ctypes.c_void_p)


def width(v: int) -> int:
    return lib().bfsc_ref_width(ctypes.c_uint64(v))


def block_bytes(b: int, n_exc: int, W: int) -> int:
    return lib().bfsc_ref_block_bytes(b, n_exc, W)


def compress_bound(n: int, W: int) -> int:
    return lib().bfsc_ref_compress_bound(n, W)


def block_deltas(x: np.ndarray):
    """x: 1..128 IDs of one block -> (base, d[128] as uint64)."""
    x = np.ascontiguousarray(x)
    d = np.zeros(128, dtype=np.uint64)
    base = lib().bfsc_ref_block_deltas(_p(x), len(x), _W(x), _p(d))
    return int(base), d


def choose_b(d: np.ndarray, W: int):
    d = np.ascontiguousarray(d, dtype=np.uint64)
    assert d.shape == (128,)
    n_exc = ctypes.c_int(0)
    b = lib().bfsc_ref_choose_b(_p(d), W, ctypes.byref(n_exc))
    return b, n_exc.value


def choose_b_bp128(d: np.ndarray) -> int:
    d = np.ascontiguousarray(d, dtype=np.uint64)
    assert d.shape == (128,)
    return lib().bfsc_ref_choose_b_bp128(_p(d))


def emit_block(d: np.ndarray, base: int, b: int, W: int) -> bytes:
    d = np.ascontiguousarray(d, dtype=np.uint64)
    out = np.zeros(2304, dtype=np.uint8)
    n = lib().bfsc_ref_emit_block(_p(d), ctypes.c_uint64(base), b, W, _p(out))
    return out[:n].tobytes()


def compress(ids: np.ndarray, raw_threshold_bytes: int = 0, codec: int = CODEC_PFOR) -> np.ndarray:
    ids = np.ascontiguousarray(ids)
    W = _W(ids)
    cap = max(compress_bound(len(ids), W), 32 + (len(ids) * W // 8 + 15) // 16 * 16)
    out = np.empty(cap, dtype=np.uint8)
    nbytes = ctypes.c_size_t(0)
    rc = lib().bfsc_ref_compress_codec(codec, _p(ids), len(ids), W, raw_threshold_bytes, _p(out), cap,
                                       ctypes.byref(nbytes))
    if rc:
        raise OracleError(rc)
    return out[:nbytes.value].copy()


def decompress(stream: np.ndarray, W: int, capacity: int | None = None) -> np.ndarray:
    stream = np.ascontiguousarray(stream, dtype=np.uint8)
    if capacity is None:
        capacity = int.from_bytes(stream[8:16].tobytes(), "little") if len(stream) >= 16 else 0
        capacity = min(capacity, 1 << 34)
    ids = np.empty(capacity, dtype=_dtype(W))
    n = ctypes.c_size_t(0)
    rc = lib().bfsc_ref_decompress(_p(stream), len(stream), W, _p(ids), capacity, ctypes.byref(n))
    if rc:
        raise OracleError(rc)
    return ids[:n.value].copy()


def batch_bound(in_offsets: np.ndarray, W: int) -> int:
    counts = np.diff(np.asarray(in_offsets, dtype=np.uint64)).astype(np.int64)
    return int(sum(max(compress_bound(int(c), W), 32 + (int(c) * W // 8 + 15) // 16 * 16) for c in counts))


def compress_batch(ids: np.ndarray, in_offsets: np.ndarray, raw_threshold_bytes: int = 0, threads: int = 0,
                   codec: int = CODEC_PFOR):
    """-> (out bytes, out_offsets[n_buf+1]); threads > 0 uses the pthread driver (PFOR only)."""
    ids = np.ascontiguousarray(ids)
    W = _W(ids)
    in_offsets = np.ascontiguousarray(in_offsets, dtype=np.uint64)
    n_buf = len(in_offsets) - 1
    counts = np.diff(in_offsets).astype(np.int64)
    nb = (counts + 127) // 128
    bound = 32 + ((4 * (nb + 1) + 15) // 16 * 16) + nb * (16 + 16 * W)
    raw = 32 + (counts * (W // 8) + 15) // 16 * 16
    cap = int(np.maximum(bound, raw).sum()) if n_buf else 0
    out = np.empty(max(cap, 16), dtype=np.uint8)
    out_off = np.zeros(n_buf + 1, dtype=np.uint64)
    if threads > 0:
        assert codec == CODEC_PFOR
        rc = lib().bfsc_ref_compress_batch_mt(_p(ids), _p(in_offsets), n_buf, W, raw_threshold_bytes,
                                              _p(out), cap, _p(out_off), threads)
    else:
        rc = lib().bfsc_ref_compress_batch_codec(codec, _p(ids), _p(in_offsets), n_buf, W, raw_threshold_bytes,
                                                 _p(out), cap, _p(out_off))
    if rc:
        raise OracleError(rc)
    return out[:int(out_off[-1])], out_off


def decompress_batch(stream: np.ndarray, in_offsets: np.ndarray, W: int, capacity: int, threads: int = 0):
    """-> (ids, id_offsets[n_buf+1])."""
    stream = np.ascontiguousarray(stream, dtype=np.uint8)
    in_offsets = np.ascontiguousarray(in_offsets, dtype=np.uint64)
    n_buf = len(in_offsets) - 1
    ids = np.empty(max(capacity, 1), dtype=_dtype(W))
    id_off = np.zeros(n_buf + 1, dtype=np.uint64)
    if threads > 0:
        rc = lib().bfsc_ref_decompress_batch_mt(_p(stream), _p(in_offsets), n_buf, W, _p(ids), capacity,
                                                _p(id_off), threads)
    else:
        rc = lib().bfsc_ref_decompress_batch(_p(stream), _p(in_offsets), n_buf, W, _p(ids), capacity, _p(id_off))
    if rc:
        raise OracleError(rc)
    return ids[:int(id_off[-1])], id_off


def compress_bitmap(bitmap: np.ndarray, n_bits: int, W: int, id_base: int = 0, raw_threshold_bytes: int = 0,
                    codec: int = CODEC_PFOR) -> np.ndarray:
    """bitmap: uint32 words (bit v = bit v % 32 of word v // 32) -> the stream of the IDs id_base + v of its set bits."""
    bitmap = np.ascontiguousarray(bitmap, dtype=np.uint32)
    assert len(bitmap) * 32 >= n_bits
    cap = max(compress_bound(n_bits, W), 32 + (n_bits * W // 8 + 15) // 16 * 16)
    out = np.empty(cap, dtype=np.uint8)
    nbytes = ctypes.c_size_t(0)
    rc = lib().bfsc_ref_compress_bitmap(codec, _p(bitmap), n_bits, ctypes.c_uint64(id_base), W, raw_threshold_bytes,
                                        _p(out), cap, ctypes.byref(nbytes))
    if rc:
        raise OracleError(rc)
    return out[:nbytes.value].copy()


def decompress_to_bitmap(stream: np.ndarray, W: int, bitmap: np.ndarray, n_bits: int, id_base: int = 0) -> int:
    """ORs the decoded IDs into `bitmap` (uint32 words, modified in place); returns the number of IDs decoded."""
    stream = np.ascontiguousarray(stream, dtype=np.uint8)
    assert bitmap.dtype == np.uint32 and bitmap.flags["C_CONTIGUOUS"] and len(bitmap) * 32 >= n_bits
    n = ctypes.c_size_t(0)
    rc = lib().bfsc_ref_decompress_to_bitmap(_p(stream), len(stream), W, ctypes.c_uint64(id_base), _p(bitmap), n_bits,
                                             ctypes.byref(n))
    if rc:
        raise OracleError(rc)
    return n.value


def decompress_to_frontier(stream: np.ndarray, W: int, frontier: np.ndarray, visited: np.ndarray, n_bits: int,
                           id_base: int = 0) -> int:
    """Algorithm 4 lines 10-13 on bitmaps (uint32 words, both modified in place): frontier |= decoded & ~visited,
    visited |= decoded. Returns the number of IDs decoded."""
    stream = np.ascontiguousarray(stream, dtype=np.uint8)
    for b in (frontier, visited):
        assert b.dtype == np.uint32 and b.flags["C_CONTIGUOUS"] and len(b) * 32 >= n_bits
    n = ctypes.c_size_t(0)
    rc = lib().bfsc_ref_decompress_to_frontier(_p(stream), len(stream), W, ctypes.c_uint64(id_base), _p(frontier),
                                               _p(visited), n_bits, ctypes.byref(n))
    if rc:
        raise OracleError(rc)
    return n.value


def vbitmap_bound(n_bits: int) -> int:
    return int(lib().bfsc_ref_vbitmap_bound(n_bits))


def compress_vbitmap(bitmap: np.ndarray, n_bits: int, codec: int = CODEC_PFOR) -> np.ndarray:
    """FORMAT.md §10: bitmap (uint32 words) -> container bytes."""
    bitmap = np.ascontiguousarray(bitmap, dtype=np.uint32)
    cap = vbitmap_bound(n_bits)
    out = np.empty(cap, dtype=np.uint8)
    nb = ctypes.c_size_t(0)
    rc = lib().bfsc_ref_compress_vbitmap(codec, _p(bitmap), n_bits, _p(out), cap, ctypes.byref(nb))
    if rc:
        raise OracleError(rc)
    return out[:nb.value].copy()


def decompress_vbitmap(container: np.ndarray, n_bits: int) -> np.ndarray:
    """-> the bitmap as uint32 words (ceil(n_bits / 32) of them)."""
    container = np.ascontiguousarray(container, dtype=np.uint8)
    bm = np.zeros(max((n_bits + 31) // 32, 1), dtype=np.uint32)
    rc = lib().bfsc_ref_decompress_vbitmap(_p(container), len(container), _p(bm), n_bits)
    if rc:
        raise OracleError(rc)
    return bm[:(n_bits + 31) // 32]

