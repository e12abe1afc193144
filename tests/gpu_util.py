"""Helpers for the ``-m gpu`` parity tests: move seeded host arrays to the device bit for bit and
back.  No arithmetic of the method lives here."""
import numpy as np
import torch

DEV = "cuda:0"


def to_dev(a: np.ndarray) -> torch.Tensor:
    """numpy array (uint16 bf16 bit patterns, uint32 or float32) -> device tensor with the same bits."""
    a = np.ascontiguousarray(a)
    if a.dtype == np.uint16:
        return torch.from_numpy(a.view(np.int16)).to(DEV)
    if a.dtype == np.uint32:
        return torch.from_numpy(a.view(np.int32)).to(DEV)
    if a.dtype == np.float32:
        return torch.from_numpy(a).to(DEV)
    raise TypeError(a.dtype)


def to_host(t: torch.Tensor) -> np.ndarray:
    """device tensor -> numpy array with the same bits (int16 -> uint16, int32 -> uint32)."""
    a = t.detach().cpu().numpy()
    if a.dtype == np.int16:
        return a.view(np.uint16)
    if a.dtype == np.int32:
        return a.view(np.uint32)
    return a


def bf16_bits_to_f64(bits: np.ndarray) -> np.ndarray:
    return (bits.astype(np.uint32) << np.uint32(16)).view(np.float32).astype(np.float64)


def nan_fill_(t: torch.Tensor) -> torch.Tensor:
    """Fill an int16 (bf16 bits) tensor with the quiet-NaN pattern 0x7fc0."""
    return t.fill_(0x7FC0)
