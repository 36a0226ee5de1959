"""Test-side helpers (no method arithmetic shared with either implementation)."""
from __future__ import annotations

import numpy as np
import torch


def bf16_bits(x) -> np.ndarray:
    """float array -> bf16 bit patterns (uint16), round-to-nearest-even (torch's cast)."""
    t = torch.as_tensor(np.asarray(x, dtype=np.float32)).to(torch.bfloat16)
    return t.view(torch.int16).numpy().view(np.uint16).copy()


def bits_to_f64(bits: np.ndarray) -> np.ndarray:
    return (bits.astype(np.uint32) << 16).view(np.float32).astype(np.float64)


def torch_bits(t: torch.Tensor) -> np.ndarray:
    """torch bf16 tensor (any device) -> numpy uint16 bits on the host."""
    return t.detach().cpu().contiguous().view(torch.int16).numpy().view(np.uint16).copy()
