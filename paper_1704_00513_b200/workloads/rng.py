"""Counter-based integer RNG used by every synthetic workload.

`mix(seed, stream, index)` -> 64 random bits, a pure function of its three integer
arguments, evaluated with wrapping int64 tensor arithmetic so that CPU and CUDA tensors
give identical bits. The finaliser is the published splitmix64 bit mixer restated here;
nothing in this module is part of the codec (no deltas, widths, packing).
"""
from __future__ import annotations

import torch


def _s64(c: int) -> int:
    """Python int (u64 bit pattern) -> the int64 with the same bits."""
    c &= (1 << 64) - 1
    return c - (1 << 64) if c >= (1 << 63) else c


_C_SEED = _s64(0x9E3779B97F4A7C15)
_C_STREAM = _s64(0xD1B54A32D192ED03)
_C_INDEX = _s64(0x2545F4914F6CDD1D)
_M1 = _s64(0xBF58476D1CE4E5B9)
_M2 = _s64(0x94D049BB133111EB)


def lsr(x: torch.Tensor, s: int) -> torch.Tensor:
    """logical shift right of an int64 bit pattern"""
    return (x >> s) & ((1 << (64 - s)) - 1)


def mix(seed: int, stream: int, index: torch.Tensor) -> torch.Tensor:
    """index: int64 tensor -> int64 tensor holding 64 random bits per element."""
    base = _s64(seed * 0x9E3779B97F4A7C15 + (stream + 1) * 0xD1B54A32D192ED03)
    z = index * _C_INDEX + base
    z = (z ^ lsr(z, 30)) * _M1
    z = (z ^ lsr(z, 27)) * _M2
    z = z ^ lsr(z, 31)
    # second round decorrelates consecutive indices of nearby streams
    z = (z + _C_SEED) * _M1
    z = z ^ lsr(z, 29)
    return z


def mix_scalar(seed: int, stream: int, index: int) -> int:
    """the same function for one index, as an unsigned python int"""
    z = mix(seed, stream, torch.tensor([index], dtype=torch.int64))
    return int(z.item()) & ((1 << 64) - 1)


def u32(seed: int, stream: int, index: torch.Tensor) -> torch.Tensor:
    """top 32 bits as a non-negative int64"""
    return lsr(mix(seed, stream, index), 32)


def below(seed: int, stream: int, index: torch.Tensor, bound: int) -> torch.Tensor:
    """uniform integer in [0, bound) (bound < 2^31; modulo bias < 2^-32 * bound, irrelevant here)"""
    return lsr(mix(seed, stream, index), 32) % bound


def unit_open_closed(seed: int, stream: int, index: torch.Tensor) -> torch.Tensor:
    """uniform float64 in (0, 1]: ((u >> 11) + 1) * 2^-53"""
    return (lsr(mix(seed, stream, index), 11) + 1).to(torch.float64) * (2.0 ** -53)
