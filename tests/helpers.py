"""Test-side helpers: bf16 <-> numpy bit patterns.  No method arithmetic."""
import numpy as np
import torch


def bf16_bits(x) -> np.ndarray:
    """float array-like -> uint16 bf16 bit patterns (round-to-nearest-even, via torch)."""
    t = torch.as_tensor(np.asarray(x, dtype=np.float64)).to(torch.float32).to(torch.bfloat16)
    return t.view(torch.int16).numpy().view(np.uint16).copy()


def bits_of(t: torch.Tensor) -> np.ndarray:
    """bf16 torch tensor (any device) -> uint16 numpy bit patterns."""
    assert t.dtype == torch.bfloat16
    return t.detach().cpu().contiguous().view(torch.int16).numpy().view(np.uint16).copy()


def bits_to_f64(b: np.ndarray) -> np.ndarray:
    """uint16 bf16 bit patterns -> float64 (exact)."""
    u = b.astype(np.uint32) << 16
    return u.view(np.float32).astype(np.float64)


def exact_bf16(x) -> bool:
    x = np.asarray(x, dtype=np.float64)
    return bool(np.all(bits_to_f64(bf16_bits(x)) == x))
