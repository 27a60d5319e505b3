"""Thin ctypes binding of libbfsc.so (include/bfsc.h). Argument marshalling only: every step
of the path runs in the CUDA kernels. PyTorch supplies device memory and streams.

There is NO CPU fallback: if libbfsc.so is missing or fails to load, `lib()` raises.
Tensors carry the ID bit pattern: torch.int32/uint32 for W=32, torch.int64/uint64 for W=64.
"""
from __future__ import annotations

import ctypes
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
CHECKED = os.environ.get("BFSC_CHECKED", "") == "1"      # the bounds-asserting build (build.py)
SO_PATH = os.path.join(_HERE, "libbfsc_checked.so" if CHECKED else "libbfsc.so")
_lib = None

OK, ERR_INVALID_ARG, ERR_DST_TOO_SMALL, ERR_CORRUPT, ERR_CUDA, ERR_UNSUPPORTED = range(6)
U32, U64 = 32, 64
CODEC_PFOR, CODEC_BP128 = 1, 2          # bfsc_codec (include/bfsc.h)
CODEC_FLAG_EXCLUSIVE = 0x100            # launch flag, OR-ed into the codec (include/bfsc.h)
NOALLOC_MAX_IDS = 1 << 22               # bfsc_compress_noalloc: BFSC_NOALLOC_MAX_IDS (include/bfsc.h)
CODEC_FLAG_RAW_FALLBACK = 0x200         # FORMAT.md §8, OR-ed into the codec of a single-buffer call

EXPORTS = [
    "bfsc_version", "bfsc_compress_bound", "bfsc_batch_compress_bound", "bfsc_workspace_bytes",
    "bfsc_compress", "bfsc_decompress", "bfsc_compress_batch", "bfsc_decompress_batch",
    "bfsc_compress_codec", "bfsc_compress_batch_codec", "bfsc_compress_batch_scatter",
    "bfsc_bitmap_workspace_bytes", "bfsc_compress_bitmap", "bfsc_decompress_to_bitmap", "bfsc_compress_noalloc",
    "bfsc_decompress_to_frontier", "bfsc_decompress_batch_to_frontier",
    "bfsc_vbitmap_bound", "bfsc_vbitmap_workspace_bytes", "bfsc_compress_vbitmap", "bfsc_decompress_vbitmap",
    "bfsc_host_scratch_bytes", "bfsc_compress_host", "bfsc_decompress_host", "bfsc_kernel_launches",
]


class BfscError(RuntimeError):
    def __init__(self, code, where=""):
        super().__init__(f"bfsc error {code} {where}")
        self.code = code


def lib():
    """Loads libbfsc.so (built by paper_1704_00513_b200.build / __graft_entry__.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(SO_PATH):
            raise RuntimeError(f"{SO_PATH} not found: run `python -m paper_1704_00513_b200.build` "
                               "(the CUDA extension is the only implementation; there is no fallback)")
        L = ctypes.CDLL(SO_PATH)
        c = ctypes
        vp, sz, i32 = c.c_void_p, c.c_size_t, c.c_int
        L.bfsc_version.restype = c.c_uint32
        L.bfsc_kernel_launches.restype = c.c_uint64
        L.bfsc_compress_bound.restype = sz
        L.bfsc_compress_bound.argtypes = [sz, i32]
        L.bfsc_batch_compress_bound.restype = sz
        L.bfsc_batch_compress_bound.argtypes = [vp, sz, i32]
        L.bfsc_workspace_bytes.restype = sz
        L.bfsc_workspace_bytes.argtypes = [sz, sz, i32]
        L.bfsc_bitmap_workspace_bytes.restype = sz
        L.bfsc_bitmap_workspace_bytes.argtypes = [sz, i32]
        L.bfsc_compress_bitmap.restype = i32
        L.bfsc_compress_bitmap.argtypes = [i32, vp, sz, c.c_uint64, i32, sz, vp, sz, vp, vp, sz, vp, vp]
        L.bfsc_decompress_to_bitmap.restype = i32
        L.bfsc_decompress_to_bitmap.argtypes = [vp, sz, i32, c.c_uint64, vp, sz, vp, vp, sz, vp, vp]
        L.bfsc_decompress_to_frontier.restype = i32
        L.bfsc_decompress_to_frontier.argtypes = [vp, sz, i32, c.c_uint64, vp, vp, sz, vp, vp, sz, vp, vp]
        L.bfsc_decompress_batch_to_frontier.restype = i32
        L.bfsc_decompress_batch_to_frontier.argtypes = [vp, vp, sz, i32, c.c_uint64, vp, vp, sz, vp, vp, sz, vp, vp]
        L.bfsc_vbitmap_bound.restype = sz
        L.bfsc_vbitmap_bound.argtypes = [sz]
        L.bfsc_vbitmap_workspace_bytes.restype = sz
        L.bfsc_vbitmap_workspace_bytes.argtypes = [sz]
        L.bfsc_compress_vbitmap.restype = i32
        L.bfsc_compress_vbitmap.argtypes = [i32, vp, sz, vp, sz, vp, vp, sz, vp, vp]
        L.bfsc_decompress_vbitmap.restype = i32
        L.bfsc_decompress_vbitmap.argtypes = [vp, sz, vp, sz, vp, sz, vp, vp]
        L.bfsc_host_scratch_bytes.restype = sz
        L.bfsc_host_scratch_bytes.argtypes = [sz, i32]
        L.bfsc_compress.restype = i32
        L.bfsc_compress.argtypes = [vp, sz, i32, sz, vp, sz, vp, vp, sz, vp, vp]
        L.bfsc_compress_noalloc.restype = i32
        L.bfsc_compress_noalloc.argtypes = [vp, sz, i32, sz, vp, sz, vp, vp, vp]
        L.bfsc_compress_codec.restype = i32
        L.bfsc_compress_codec.argtypes = [i32, vp, sz, i32, sz, vp, sz, vp, vp, sz, vp, vp]
        L.bfsc_compress_batch_codec.restype = i32
        L.bfsc_compress_batch_codec.argtypes = [i32, vp, vp, sz, i32, sz, vp, sz, vp, vp, sz, vp, vp]
        L.bfsc_compress_batch_scatter.restype = i32
        L.bfsc_compress_batch_scatter.argtypes = [i32, vp, vp, sz, i32, sz, vp, sz, vp, vp, sz, vp, vp]
        L.bfsc_decompress.restype = i32
        L.bfsc_decompress.argtypes = [vp, sz, i32, vp, sz, vp, vp, sz, vp, vp]
        L.bfsc_compress_batch.restype = i32
        L.bfsc_compress_batch.argtypes = [vp, vp, sz, i32, sz, vp, sz, vp, vp, sz, vp, vp]
        L.bfsc_decompress_batch.restype = i32
        L.bfsc_decompress_batch.argtypes = [vp, vp, sz, i32, vp, sz, vp, vp, sz, vp, vp]
        L.bfsc_compress_host.restype = i32
        L.bfsc_compress_host.argtypes = [vp, sz, i32, sz, vp, sz, vp, vp, sz, vp]
        L.bfsc_decompress_host.restype = i32
        L.bfsc_decompress_host.argtypes = [vp, sz, i32, vp, sz, vp, vp, sz, vp]
        _lib = L
    return _lib


def dtype_of(t: torch.Tensor) -> int:
    if t.dtype in (torch.int32, torch.uint32):
        return U32
    if t.dtype in (torch.int64, torch.uint64):
        return U64
    raise TypeError(f"IDs must be 32- or 64-bit integers, got {t.dtype}")


def _stream() -> int:
    return torch.cuda.current_stream().cuda_stream


def _ptr(t):
    return None if t is None else ctypes.c_void_p(t.data_ptr())


def compress_bound(n_ids: int, W: int) -> int:
    return lib().bfsc_compress_bound(n_ids, W)


def batch_compress_bound(counts, W: int) -> int:
    arr = (ctypes.c_uint64 * len(counts))(*[int(c) for c in counts])
    return lib().bfsc_batch_compress_bound(arr, len(counts), W)


def workspace_bytes(n_ids_total: int, n_buf: int, W: int) -> int:
    return lib().bfsc_workspace_bytes(n_ids_total, n_buf, W)


def bitmap_workspace_bytes(n_bits: int, W: int) -> int:
    return lib().bfsc_bitmap_workspace_bytes(n_bits, W)


def host_scratch_bytes(n_ids: int, W: int) -> int:
    return lib().bfsc_host_scratch_bytes(n_ids, W)


def check_failures():
    """BFSC_CHECKED build only: (violations, first failing source line) of the encode and of the decode kernels so far."""
    out = []
    for name in ("bfsc_debug_checks_encode", "bfsc_debug_checks_decode"):
        buf = (ctypes.c_uint * 2)()
        getattr(lib(), name)(buf)
        out.append((int(buf[0]), int(buf[1])))
    return out


def kernel_launches() -> int:
    return lib().bfsc_kernel_launches()


def _check(rc, where):
    if rc != OK:
        raise BfscError(rc, where)


def compress(d_ids, n_ids, W, raw_threshold_bytes, d_out, d_out_bytes, d_workspace, d_status):
    """bfsc_compress: device tensors in, enqueue only (no sync). d_out: uint8; d_out_bytes:
    int64[1]; d_status: int32[1] (zeroed by the caller)."""
    _check(lib().bfsc_compress(_ptr(d_ids), n_ids, W, raw_threshold_bytes, _ptr(d_out), d_out.numel(),
                               _ptr(d_out_bytes), _ptr(d_workspace), d_workspace.numel(), _ptr(d_status),
                               ctypes.c_void_p(_stream())), "bfsc_compress")


def compress_noalloc(d_ids, n_ids, W, raw_threshold_bytes, d_out, d_out_bytes, d_status):
    """bfsc_compress_noalloc: bfsc_compress with the workspace in the library's own device array (no allocation anywhere;
    n_ids <= NOALLOC_MAX_IDS; calls that overlap on the GPU race on that array)."""
    _check(lib().bfsc_compress_noalloc(_ptr(d_ids), n_ids, W, raw_threshold_bytes, _ptr(d_out), d_out.numel(),
                                       _ptr(d_out_bytes), _ptr(d_status), ctypes.c_void_p(_stream())), "bfsc_compress_noalloc")


def compress_codec(codec, d_ids, n_ids, W, raw_threshold_bytes, d_out, d_out_bytes, d_workspace, d_status):
    """bfsc_compress_codec: bfsc_compress with the encoder rule given (CODEC_PFOR / CODEC_BP128)."""
    _check(lib().bfsc_compress_codec(codec, _ptr(d_ids), n_ids, W, raw_threshold_bytes, _ptr(d_out), d_out.numel(),
                                     _ptr(d_out_bytes), _ptr(d_workspace), d_workspace.numel(), _ptr(d_status),
                                     ctypes.c_void_p(_stream())), "bfsc_compress_codec")


def compress_bitmap(codec, d_bitmap, n_bits, id_base, W, raw_threshold_bytes, d_out, d_out_bytes, d_workspace, d_status):
    """bfsc_compress_bitmap (FORMAT.md §9): d_bitmap int32/uint32 words, bit v = ID id_base + v."""
    _check(lib().bfsc_compress_bitmap(codec, _ptr(d_bitmap), n_bits, id_base, W, raw_threshold_bytes, _ptr(d_out),
                                      d_out.numel(), _ptr(d_out_bytes), _ptr(d_workspace), d_workspace.numel(),
                                      _ptr(d_status), ctypes.c_void_p(_stream())), "bfsc_compress_bitmap")


def decompress_to_bitmap(d_in, in_bytes, W, id_base, d_bitmap, n_bits, d_n_ids, d_workspace, d_status):
    """bfsc_decompress_to_bitmap (FORMAT.md §9): ORs the bits of the stream's IDs into d_bitmap."""
    _check(lib().bfsc_decompress_to_bitmap(_ptr(d_in), in_bytes, W, id_base, _ptr(d_bitmap), n_bits, _ptr(d_n_ids),
                                           _ptr(d_workspace), d_workspace.numel(), _ptr(d_status),
                                           ctypes.c_void_p(_stream())), "bfsc_decompress_to_bitmap")


def decompress_to_frontier(d_in, in_bytes, W, id_base, d_frontier, d_visited, n_bits, d_n_ids, d_workspace, d_status):
    """bfsc_decompress_to_frontier (Algorithm 4 lines 10-13): unvisited decoded IDs -> d_frontier and d_visited."""
    _check(lib().bfsc_decompress_to_frontier(_ptr(d_in), in_bytes, W, id_base, _ptr(d_frontier), _ptr(d_visited), n_bits,
                                             _ptr(d_n_ids), _ptr(d_workspace), d_workspace.numel(), _ptr(d_status),
                                             ctypes.c_void_p(_stream())), "bfsc_decompress_to_frontier")


def decompress_batch_to_frontier(d_in, d_in_offsets, n_buf, W, id_base, d_frontier, d_visited, n_bits, d_n_ids, d_workspace,
                                 d_status):
    _check(lib().bfsc_decompress_batch_to_frontier(_ptr(d_in), _ptr(d_in_offsets), n_buf, W, id_base, _ptr(d_frontier),
                                                   _ptr(d_visited), n_bits, _ptr(d_n_ids), _ptr(d_workspace),
                                                   d_workspace.numel(), _ptr(d_status), ctypes.c_void_p(_stream())),
           "bfsc_decompress_batch_to_frontier")


def vbitmap_bound(n_bits: int) -> int:
    return int(lib().bfsc_vbitmap_bound(n_bits))


def vbitmap_workspace_bytes(n_bits: int) -> int:
    return int(lib().bfsc_vbitmap_workspace_bytes(n_bits))


def compress_vbitmap(codec, d_bitmap, n_bits, d_out, d_out_bytes, d_workspace, d_status):
    _check(lib().bfsc_compress_vbitmap(codec, _ptr(d_bitmap), n_bits, _ptr(d_out), d_out.numel(), _ptr(d_out_bytes),
                                       _ptr(d_workspace), d_workspace.numel(), _ptr(d_status),
                                       ctypes.c_void_p(_stream())), "bfsc_compress_vbitmap")


def decompress_vbitmap(d_in, in_bytes, d_bitmap, n_bits, d_workspace, d_status):
    _check(lib().bfsc_decompress_vbitmap(_ptr(d_in), in_bytes, _ptr(d_bitmap), n_bits, _ptr(d_workspace),
                                         d_workspace.numel(), _ptr(d_status), ctypes.c_void_p(_stream())),
           "bfsc_decompress_vbitmap")


def decompress(d_in, in_bytes, W, d_ids, d_n_ids, d_workspace, d_status):
    _check(lib().bfsc_decompress(_ptr(d_in), in_bytes, W, _ptr(d_ids), d_ids.numel(), _ptr(d_n_ids),
                                 _ptr(d_workspace), d_workspace.numel(), _ptr(d_status),
                                 ctypes.c_void_p(_stream())), "bfsc_decompress")


def compress_batch(d_ids, d_in_offsets, n_buf, W, raw_threshold_bytes, d_out, d_out_offsets, d_workspace, d_status):
    _check(lib().bfsc_compress_batch(_ptr(d_ids), _ptr(d_in_offsets), n_buf, W, raw_threshold_bytes, _ptr(d_out),
                                     d_out.numel(), _ptr(d_out_offsets), _ptr(d_workspace), d_workspace.numel(),
                                     _ptr(d_status), ctypes.c_void_p(_stream())), "bfsc_compress_batch")


def compress_batch_codec(codec, d_ids, d_in_offsets, n_buf, W, raw_threshold_bytes, d_out, d_out_offsets, d_workspace,
                         d_status):
    _check(lib().bfsc_compress_batch_codec(codec, _ptr(d_ids), _ptr(d_in_offsets), n_buf, W, raw_threshold_bytes,
                                           _ptr(d_out), d_out.numel(), _ptr(d_out_offsets), _ptr(d_workspace),
                                           d_workspace.numel(), _ptr(d_status), ctypes.c_void_p(_stream())),
           "bfsc_compress_batch_codec")


def compress_batch_scatter(codec, d_ids, d_in_offsets, n_buf, W, raw_threshold_bytes, d_dst, dst_capacity, d_out_bytes,
                           d_workspace, d_status):
    """d_dst: int64 device tensor of n_buf device addresses (tensor.data_ptr() values; may be peer-mapped)."""
    _check(lib().bfsc_compress_batch_scatter(codec, _ptr(d_ids), _ptr(d_in_offsets), n_buf, W, raw_threshold_bytes,
                                             _ptr(d_dst), dst_capacity, _ptr(d_out_bytes), _ptr(d_workspace),
                                             d_workspace.numel(), _ptr(d_status), ctypes.c_void_p(_stream())),
           "bfsc_compress_batch_scatter")


def decompress_batch(d_in, d_in_offsets, n_buf, W, d_ids, d_id_offsets, d_workspace, d_status):
    _check(lib().bfsc_decompress_batch(_ptr(d_in), _ptr(d_in_offsets), n_buf, W, _ptr(d_ids), d_ids.numel(),
                                       _ptr(d_id_offsets), _ptr(d_workspace), d_workspace.numel(), _ptr(d_status),
                                       ctypes.c_void_p(_stream())), "bfsc_decompress_batch")


def compress_host(h_ids, W, raw_threshold_bytes, h_out, d_scratch) -> int:
    """bfsc_compress_host: (pinned) host tensors in/out; synchronises; returns stream bytes."""
    nbytes = ctypes.c_uint64(0)
    _check(lib().bfsc_compress_host(_ptr(h_ids), h_ids.numel(), W, raw_threshold_bytes, _ptr(h_out), h_out.numel(),
                                    ctypes.byref(nbytes), _ptr(d_scratch), d_scratch.numel(),
                                    ctypes.c_void_p(_stream())), "bfsc_compress_host")
    return nbytes.value


def decompress_host(h_in, in_bytes, W, h_ids, d_scratch) -> int:
    n = ctypes.c_uint64(0)
    _check(lib().bfsc_decompress_host(_ptr(h_in), in_bytes, W, _ptr(h_ids), h_ids.numel(), ctypes.byref(n),
                                      _ptr(d_scratch), d_scratch.numel(), ctypes.c_void_p(_stream())),
           "bfsc_decompress_host")
    return n.value
