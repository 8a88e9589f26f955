"""splitmix64 counter stream -> uniform doubles in [0,1), as torch ops so that large fields can be drawn on any device.

u_n = (mix(seed + (n+1)*GOLDEN) >> 11) * 2^-53 , n = 0,1,2,...  (counter based: element n needs no earlier element).
torch has no full uint64 arithmetic; int64 multiplication/addition wrap modulo 2^64 exactly like uint64, and the
logical right shifts are emulated by masking the sign-extended bits.
"""
import torch


def _i64(x: int) -> int:
    """Reinterpret an unsigned 64-bit constant as a signed one."""
    x &= (1 << 64) - 1
    return x - (1 << 64) if x >= (1 << 63) else x


_GOLDEN = _i64(0x9E3779B97F4A7C15)
_M1 = _i64(0xBF58476D1CE4E5B9)
_M2 = _i64(0x94D049BB133111EB)


def _lsr(x: torch.Tensor, k: int) -> torch.Tensor:
    return (x >> k) & ((1 << (64 - k)) - 1)


def splitmix64_uniform(seed: int, start: int, count: int, device="cpu", stride: int = 1) -> torch.Tensor:
    """Elements start, start+stride, ... (count of them) of the stream of `seed`, float64 in [0,1)."""
    n = torch.arange(count, dtype=torch.int64, device=device) * stride + (start + 1)
    z = n * _GOLDEN + _i64(seed)
    z = (z ^ _lsr(z, 30)) * _M1
    z = (z ^ _lsr(z, 27)) * _M2
    z = z ^ _lsr(z, 31)
    return _lsr(z, 11).to(torch.float64) * (1.0 / 9007199254740992.0)
