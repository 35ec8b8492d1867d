"""Seeded synthetic inputs (the ONLY module the CUDA path's callers and the oracle's callers share).

It holds none of the method's arithmetic: no mask, no softmax, no block rule -- only a
counter-based generator of bf16 values and the seeded shape recipes of BASELINE.json's configs
(DESIGN.md "Input recipe").  It imports neither the binding nor the oracle.

Why counter-based: the value of K/V/Q element (stream, layer, session, position, head, dim) is a
pure function of the seed and those coordinates, so
  * the GPU side can generate a whole history on the device (no multi-GB host copies), and
  * a test can regenerate, on the CPU, exactly the rows of the few sessions it samples,
and both get the SAME bf16 bits: every step is integer arithmetic on int64 tensors (exact on CPU
and CUDA), one exact int->float32 conversion (|x| < 2^24), one IEEE float32 multiply by a constant,
optional exact-in-fp32 outlier scaling, and one round-to-nearest-even to bf16.

Distribution: Irwin-Hall sum of 8 uniform bytes, centred and scaled to unit variance -- a
stand-in for the N(0,1) BASELINE.json names (support +-4.9 sigma, excess kurtosis -0.15).
"""
from __future__ import annotations

import math

import torch

_M32 = 0xFFFFFFFF
_MUL = 0x45D9F3B          # < 2^27: (x < 2^32) * _MUL < 2^59 fits int64 exactly
_GOLD = 0x9E3779B1        # < 2^32: times (e+1) <= 2^16 fits int64 exactly
STREAM_K, STREAM_V, STREAM_Q = 1, 2, 3

# std of a sum of 8 independent uniform bytes: sqrt(8 * (256^2 - 1) / 12)
_IH_STD = math.sqrt(8.0 * (256.0 ** 2 - 1.0) / 12.0)
_IH_MEAN = 8 * 255 // 2   # 1020, exact


def _hash32(x: torch.Tensor) -> torch.Tensor:
    """32-bit integer mixer on int64 tensors holding values in [0, 2^32)."""
    x = (((x >> 16) ^ x) * _MUL) & _M32
    x = (((x >> 16) ^ x) * _MUL) & _M32
    return (x >> 16) ^ x


def _byte_sum(x: torch.Tensor) -> torch.Tensor:
    return (x & 0xFF) + ((x >> 8) & 0xFF) + ((x >> 16) & 0xFF) + ((x >> 24) & 0xFF)


def rows(seed: int, stream: int, layer: int, sessions: torch.Tensor, positions: torch.Tensor,
         n_heads: int, head_dim: int, outlier_channels: torch.Tensor | None = None,
         outlier_scale: float = 1.0) -> torch.Tensor:
    """bf16 [n, n_heads, head_dim]: row i is the (stream, layer) vector of session sessions[i] at
    absolute position positions[i].  Runs on sessions.device (CPU or CUDA), bit-identical on both.

    outlier_channels: int64 indices into the flattened (head, dim) axis whose values are
    multiplied by outlier_scale (config 4's "1% outlier channels scaled 20x")."""
    dev = sessions.device
    sessions = sessions.to(torch.int64)
    positions = positions.to(torch.int64)
    h = _hash32(torch.tensor((seed & _M32), dtype=torch.int64, device=dev))
    h = _hash32(h ^ ((stream & 0xFF) | ((layer & 0xFFFF) << 8)))
    h = _hash32((h + sessions) & _M32)                          # [n]
    h = _hash32((h + (positions & _M32)) & _M32)                # [n]
    h = _hash32(h ^ ((positions >> 32) & _M32))
    e = torch.arange(1, n_heads * head_dim + 1, dtype=torch.int64, device=dev)
    x = (h[:, None] + e[None, :] * _GOLD) & _M32                # [n, H*D]
    a = _hash32(x)
    b = _hash32(a ^ 0x85EBCA6B)
    s = _byte_sum(a) + _byte_sum(b) - _IH_MEAN                  # exact integer, |s| <= 1020
    val = s.to(torch.float32) * torch.tensor(1.0 / _IH_STD, dtype=torch.float32, device=dev)
    if outlier_channels is not None and outlier_channels.numel() > 0:
        mult = torch.ones(n_heads * head_dim, dtype=torch.float32, device=dev)
        mult[outlier_channels.to(dev)] = outlier_scale
        val = val * mult[None, :]
    return val.to(torch.bfloat16).reshape(-1, n_heads, head_dim)


def to_u16(t: torch.Tensor):
    """bf16 tensor -> numpy uint16 bit patterns (what the oracle consumes)."""
    return t.detach().cpu().contiguous().view(torch.int16).numpy().view("uint16")
