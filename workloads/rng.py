"""Counter-based random numbers for the synthetic PWA workloads.

Every number is a pure function of (seed, stream, plane, index), so a sample can be generated in
chunks of any size, in any order, on the CPU or on a GPU, and always comes out the same
(SURVEY.md §8(d) "RNG").  The generator is the SplitMix64 finaliser applied to a 64-bit counter;
it is written with torch int64 ops only (two's-complement wrap-around on every backend) so one
implementation serves the CPU tests and the on-device generation of the full-size configs.

This module holds no likelihood arithmetic.  It is shared by the oracle's tests and by the CUDA
path's tests/bench as the single source of input arrays.
"""
from __future__ import annotations

import math

import torch

_MASK64 = (1 << 64) - 1


def _s64(u: int) -> int:
    """Unsigned 64-bit constant -> the signed Python int with the same bit pattern."""
    u &= _MASK64
    return u - (1 << 64) if u >= (1 << 63) else u


_GOLDEN = _s64(0x9E3779B97F4A7C15)
_C1 = _s64(0xBF58476D1CE4E5B9)
_C2 = _s64(0x94D049BB133111EB)


def _lsr(x: torch.Tensor, k: int) -> torch.Tensor:
    """Logical shift right of int64 bit patterns (torch's >> is arithmetic)."""
    return (x >> k) & ((1 << (64 - k)) - 1)


def splitmix64(x: torch.Tensor) -> torch.Tensor:
    """SplitMix64 output function on int64 bit patterns (Steele, Lea, Flood 2014)."""
    z = x + _GOLDEN
    z = (z ^ _lsr(z, 30)) * _C1
    z = (z ^ _lsr(z, 27)) * _C2
    return z ^ _lsr(z, 31)


def splitmix64_int(x: int) -> int:
    """The same function on Python ints (unsigned semantics) - used for keys and for testing."""
    z = (x + 0x9E3779B97F4A7C15) & _MASK64
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _MASK64
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _MASK64
    return z ^ (z >> 31)


def stream_key(seed: int, stream: int, plane: int = 0, draw: int = 0) -> int:
    """64-bit key of one (seed, stream, plane, draw) sequence; `draw` separates the several
    uniforms one variate needs (e.g. the two of Box-Muller)."""
    k = splitmix64_int(seed & _MASK64)
    k = splitmix64_int(k ^ ((stream * 0x100000001B3) & _MASK64))
    k = splitmix64_int(k ^ ((plane * 0xD6E8FEB86659FD93) & _MASK64))
    k = splitmix64_int(k ^ ((draw * 0xCA5A826395121157) & _MASK64))
    return k


def bits(key: int, start: int, count: int, device="cpu") -> torch.Tensor:
    """`count` 64-bit patterns for indices start..start+count-1 of the sequence `key`."""
    idx = torch.arange(start, start + count, dtype=torch.int64, device=device)
    return splitmix64(idx * _GOLDEN + _s64(key))


def uniform01(key: int, start: int, count: int, device="cpu") -> torch.Tensor:
    """fp64 uniforms in the open interval (0, 1): (top 53 bits + 1/2) * 2^-53."""
    b = _lsr(bits(key, start, count, device), 11)
    return (b.to(torch.float64) + 0.5) * (1.0 / 9007199254740992.0)


def uniform(key: int, start: int, count: int, lo: float, hi: float, device="cpu") -> torch.Tensor:
    return lo + (hi - lo) * uniform01(key, start, count, device)


def normal_pair(seed: int, stream: int, plane: int, start: int, count: int, device="cpu"):
    """Two independent N(0,1) fp64 sequences (Box-Muller on two uniform sequences)."""
    u1 = uniform01(stream_key(seed, stream, plane, 0), start, count, device)
    u2 = uniform01(stream_key(seed, stream, plane, 1), start, count, device)
    rad = torch.sqrt(-2.0 * torch.log(u1))
    ang = (2.0 * math.pi) * u2
    return rad * torch.cos(ang), rad * torch.sin(ang)
