"""Shared helpers for the GPU parity tests: torch <-> numpy marshalling for the oracle and
small instance builders.  No arithmetic of the method."""
from __future__ import annotations

import numpy as np
import torch


def bf16_bits(t: torch.Tensor) -> np.ndarray:
    """bf16 tensor -> uint16 bit patterns on host."""
    return t.detach().cpu().contiguous().view(torch.int16).numpy().view(np.uint16)


def to_np(t):
    return None if t is None else t.detach().cpu().numpy()


def ws_tensor(nbytes: int, device="cuda") -> torch.Tensor:
    return torch.empty(max(nbytes, 256), dtype=torch.uint8, device=device)
