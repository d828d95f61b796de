"""Counter-based random numbers for the synthetic generator.

Every draw is a pure function of (seed, stream, element index), so a tensor can be produced in
chunks, on the CPU or on a GPU, and come out the same up to the last-bit differences of the
device's log/cos.  None of the gridding arithmetic lives here.
"""
import math

import torch

_M64 = (1 << 64) - 1


def _i64(x: int) -> int:
    """Python int (mod 2^64) -> the int64 with the same bit pattern."""
    x &= _M64
    return x - (1 << 64) if x >= (1 << 63) else x


_K_SEED = _i64(0x9E3779B97F4A7C15)
_K_STREAM = _i64(0xD1B54A32D192ED03)
_K_MIX1 = _i64(0xBF58476D1CE4E5B9)
_K_MIX2 = _i64(0x94D049BB133111EB)


def _lsr(x: torch.Tensor, s: int) -> torch.Tensor:
    """Logical shift right of an int64 tensor (torch's >> is arithmetic)."""
    return (x >> s) & ((1 << (64 - s)) - 1)


def hash64(seed: int, stream: int, idx: torch.Tensor) -> torch.Tensor:
    """splitmix64 finaliser of a counter built from (seed, stream, idx); int64 in, int64 out."""
    x = idx.to(torch.int64) + _i64(seed * 0x9E3779B97F4A7C15 + (stream + 1) * 0xD1B54A32D192ED03)
    x = (x ^ _lsr(x, 30)) * _K_MIX1
    x = (x ^ _lsr(x, 27)) * _K_MIX2
    return x ^ _lsr(x, 31)


def uniform(seed: int, stream: int, idx: torch.Tensor) -> torch.Tensor:
    """U(0,1) in fp64, never exactly 0 or 1 (53 random bits, centred)."""
    bits = _lsr(hash64(seed, stream, idx), 11)
    return (bits.to(torch.float64) + 0.5) * (1.0 / 9007199254740992.0)


def normal(seed: int, stream: int, idx: torch.Tensor) -> torch.Tensor:
    """N(0,1) in fp64 by Box-Muller from two independent streams."""
    u1 = uniform(seed, 2 * stream + 1000, idx)
    u2 = uniform(seed, 2 * stream + 1001, idx)
    return torch.sqrt(-2.0 * torch.log(u1)) * torch.cos((2.0 * math.pi) * u2)
