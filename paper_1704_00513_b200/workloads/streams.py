"""Synthetic sorted-ID streams (BASELINE.json configs 2 and 5).

Stand-ins for the thesis's extracted frontier buffers (Table 5.3:
29 899 sorted IDs in [1, 65532], i.e. mean gap ~2.2; value range [1..2^24], L782), which
are not available. Everything is seeded (workloads/rng.py) and holds none of the codec's
arithmetic: it only draws gaps and accumulates them.

IDs are returned as torch tensors whose BIT PATTERN is the unsigned ID:
W=32 -> dtype int32 (u32 bits), W=64 -> dtype int64 (u64 bits).
"""
from __future__ import annotations

import math

import torch

from . import rng

# rng stream ids
_S_FIRST, _S_GAP, _S_SEL, _S_OUT, _S_SIZE = 0x10, 0x11, 0x12, 0x13, 0x14


def as_ids(values: torch.Tensor, W: int) -> torch.Tensor:
    """int64 values (already reduced mod 2^W) -> tensor with the ID bit pattern."""
    if W == 32:
        return (values & 0xFFFFFFFF).to(torch.int32) if values.dtype == torch.int64 else values
    return values


def geometric_gaps(seed: int, stream: int, index: torch.Tensor, mean: float) -> torch.Tensor:
    """gaps on support {1,2,...} with the given mean: g = 1 + floor(ln U / ln(1-p)), p = 1/mean.
    mean == 1 -> g == 1 (consecutive IDs)."""
    if mean <= 1.0:
        return torch.ones_like(index)
    u = rng.unit_open_closed(seed, stream, index)
    g = torch.floor(torch.log(u) / math.log1p(-1.0 / mean)).to(torch.int64) + 1
    return g


def gap_stream(n: int, mean: float, seed: int, W: int = 32, outlier_frac: float = 0.0,
               sub: int = 0, device="cpu") -> torch.Tensor:
    """n IDs: first ~ U[0, 2^20), then i.i.d. geometric gaps; with outlier_frac > 0 each gap is
    independently replaced w.p. outlier_frac by U[2^16, 2^24) (config 2c). IDs accumulate
    mod 2^W (u32 streams 2b/2c wrap; legal, deltas are modular)."""
    if n == 0:
        return as_ids(torch.zeros(0, dtype=torch.int64, device=device), W)
    idx = torch.arange(n, dtype=torch.int64, device=device)
    first = int(rng.mix_scalar(seed, _S_FIRST + 16 * sub, 0) >> 32) % (1 << 20)
    g = geometric_gaps(seed, _S_GAP + 16 * sub, idx, mean)
    if outlier_frac > 0.0:
        sel = rng.below(seed, _S_SEL + 16 * sub, idx, 1_000_000) < int(outlier_frac * 1_000_000)
        big = (1 << 16) + rng.below(seed, _S_OUT + 16 * sub, idx, (1 << 24) - (1 << 16))
        g = torch.where(sel, big, g)
    g[0] = first
    vals = torch.cumsum(g, 0)
    if W == 32:
        vals = vals & 0xFFFFFFFF
    return as_ids(vals, W)


def batch_of_streams(counts: torch.Tensor, mean: float, seed: int, W: int = 32, device="cpu"):
    """Concatenation of len(counts) independent gap streams (buffer i has counts[i] IDs, its own
    first value ~ U[0, 2^20)). Returns (ids, in_offsets[n_buf+1] int64 element offsets)."""
    counts = counts.to(torch.int64).to(device)
    n_buf = counts.numel()
    off = torch.zeros(n_buf + 1, dtype=torch.int64, device=device)
    off[1:] = torch.cumsum(counts, 0)
    n = int(off[-1].item())
    if n == 0:
        return as_ids(torch.zeros(0, dtype=torch.int64, device=device), W), off
    idx = torch.arange(n, dtype=torch.int64, device=device)
    g = geometric_gaps(seed, _S_GAP, idx, mean)
    firsts = rng.below(seed, _S_FIRST, torch.arange(n_buf, dtype=torch.int64, device=device), 1 << 20)
    nonempty = counts > 0
    g[off[:-1][nonempty]] = firsts[nonempty]
    c = torch.cumsum(g, 0)
    # subtract everything accumulated before each buffer's first element
    start_c = torch.zeros(n_buf, dtype=torch.int64, device=device)
    starts = off[:-1][nonempty]
    start_c[nonempty] = c[starts] - g[starts]
    buf_of = torch.repeat_interleave(torch.arange(n_buf, device=device), counts)
    vals = c - start_c[buf_of]
    if W == 32:
        vals = vals & 0xFFFFFFFF
    return as_ids(vals, W), off


def log_uniform_counts(n_buf: int, lo_bytes_log2: int, hi_bytes_log2: int, W: int, seed: int) -> torch.Tensor:
    """config 5 batch: raw sizes 2^U[lo,hi] bytes rounded down to a whole ID."""
    u = rng.unit_open_closed(seed, _S_SIZE, torch.arange(n_buf, dtype=torch.int64))
    size = torch.floor(torch.exp2(lo_bytes_log2 + (hi_bytes_log2 - lo_bytes_log2) * u)).to(torch.int64)
    return size // (W // 8)


def split_mod(frontier: torch.Tensor, parts: int):
    """config 1: destination = v mod parts; IDs stay global. frontier: sorted int64 values.
    Returns (values reordered buffer by buffer, in_offsets)."""
    chunks = [frontier[frontier % parts == q] for q in range(parts)]
    off = torch.zeros(parts + 1, dtype=torch.int64, device=frontier.device)
    off[1:] = torch.cumsum(torch.tensor([c.numel() for c in chunks], dtype=torch.int64), 0).to(frontier.device)
    return (torch.cat(chunks) if chunks else frontier), off


def split_block(frontier: torch.Tensor, parts: int, n_vertices: int):
    """configs 3/4: contiguous vertex-range owner = v div (N/parts); buffers are contiguous
    slices of the sorted frontier. Returns (frontier, in_offsets)."""
    bounds = torch.arange(parts + 1, dtype=torch.int64, device=frontier.device) * (n_vertices // parts)
    bounds[-1] = n_vertices
    off = torch.searchsorted(frontier, bounds, right=False)
    off[-1] = frontier.numel()
    return frontier, off.to(torch.int64)


_S_BIT, _S_JUNK = 0x15, 0x16


def frontier_bitmap(n_bits: int, density: float, seed: int, run: int = 1) -> torch.Tensor:
    """A frontier bitmap (32-bit words): int32 words, whole 16-byte groups. Cells of `run` consecutive
    bits are set together w.p. `density` (run > 1: clustered frontiers); bits at positions >= n_bits of the padded
    words are random junk the codec must ignore (FORMAT.md §9). density 0 / 1: empty / full."""
    words = (n_bits + 31) // 32
    padded = max(4, (words + 3) // 4 * 4)
    pos = torch.arange(padded * 32, dtype=torch.int64)
    if density >= 1.0:
        bits = torch.ones_like(pos, dtype=torch.bool)
    elif density <= 0.0:
        bits = torch.zeros_like(pos, dtype=torch.bool)
    else:
        bits = rng.below(seed, _S_BIT, pos // run, 1_000_000) < int(density * 1_000_000)
    junk = rng.below(seed, _S_JUNK, pos, 2) == 1
    bits = torch.where(pos < n_bits, bits, junk)
    w = (bits.view(padded, 32).to(torch.int64) << torch.arange(32, dtype=torch.int64)).sum(1)
    return (w & 0xFFFFFFFF).to(torch.uint32).view(torch.int32)
