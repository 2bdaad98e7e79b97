"""Counter-based synthetic tensor generator (input data only; see synth/__init__.py).

Recipe: element e of tensor number `tid` is

    x   = (tid << 40) + e                      (64-bit counter, e < 2**40)
    h   = mix64(x + MASTER)                    (SplitMix64 finaliser, exact integer arithmetic)
    u   = ((h >> 11) + 0.5) * 2**-53           (uniform in (0, 1), exact in fp64)
    z   = sqrt(2) * erfinv(2u - 1)             (inverse-CDF normal, fp64)
    out = round_dtype(scale * z)

It is deliberately NOT the method's generator (Philox4x32-10 + Box-Muller, which
the oracle and the CUDA kernel each implement on their own): a different hash and
a different uniform->normal transform, so nothing of the method is shared.

Everything is written with torch ops that exist on CPU and CUDA alike, so the
40.8 GB weight set of the full-depth configs can be produced on the device while
the oracle produces the same values on the host.  Integer steps are exact; the
fp64 erfinv may differ between host and device by a few ulp, which can flip a
bf16 rounding only for a value within ~1e-15 (relative) of a rounding boundary.
`tensor_checksum` (sum of bit patterns mod 2**63) is compared host vs device by
the tests before any parity verdict.
"""
from __future__ import annotations

import math

import torch

MASTER = 0x5EED0000_2606_1900 & 0x7FFF_FFFF_FFFF_FFFF
_M1 = 0xBF58476D1CE4E5B9
_M2 = 0x94D049BB133111EB


def _s64(v: int) -> int:
    """Two's-complement reinterpretation of a 64-bit pattern as a Python int that fits int64."""
    v &= 0xFFFF_FFFF_FFFF_FFFF
    return v - (1 << 64) if v >= (1 << 63) else v


def _lsr(x: torch.Tensor, n: int) -> torch.Tensor:
    """Logical shift right on int64 (torch's >> is arithmetic)."""
    return (x >> n) & ((1 << (64 - n)) - 1)


def _mix64(x: torch.Tensor) -> torch.Tensor:
    x = x ^ _lsr(x, 30)
    x = x * _s64(_M1)          # wraps mod 2**64 on CPU and CUDA alike
    x = x ^ _lsr(x, 27)
    x = x * _s64(_M2)
    x = x ^ _lsr(x, 31)
    return x


def hash_normal(tid: int, numel: int, scale: float, dtype: torch.dtype,
                device: str | torch.device = "cpu", chunk: int = 1 << 24) -> torch.Tensor:
    """Flat tensor of `numel` values scale*N(0,1), rounded once to `dtype` (RNE)."""
    assert 0 <= tid < (1 << 22) and 0 <= numel < (1 << 40)
    out = torch.empty(numel, dtype=dtype, device=device)
    base = (tid << 40) + MASTER
    for lo in range(0, numel, chunk):
        hi = min(numel, lo + chunk)
        e = torch.arange(lo, hi, dtype=torch.int64, device=device)
        h = _mix64(e + _s64(base))
        u = (_lsr(h, 11).to(torch.float64) + 0.5) * (2.0 ** -53)
        z = math.sqrt(2.0) * torch.special.erfinv(2.0 * u - 1.0)
        out[lo:hi] = (scale * z).to(dtype)
    return out


def round_to(x: torch.Tensor, dtype: torch.dtype) -> torch.Tensor:
    """Round-to-nearest-even to `dtype` (reading S13)."""
    return x.to(dtype)


def tensor_checksum(x: torch.Tensor) -> int:
    """Order-independent checksum of the raw bit patterns (mod 2**63)."""
    flat = x.reshape(-1)
    if flat.dtype == torch.bfloat16 or flat.dtype == torch.float16:
        bits = flat.view(torch.int16).to(torch.int64) & 0xFFFF
    elif flat.dtype == torch.float32:
        bits = flat.view(torch.int32).to(torch.int64) & 0xFFFF_FFFF
    elif flat.dtype == torch.float64:
        bits = flat.view(torch.int64) & 0x7FFF_FFFF_FFFF_FFFF
    else:
        raise TypeError(flat.dtype)
    idx = torch.arange(bits.numel(), dtype=torch.int64, device=bits.device) % 65521 + 1
    return int(((bits * idx).sum().item()) & 0x7FFF_FFFF_FFFF_FFFF)
