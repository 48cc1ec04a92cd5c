"""Seeded synthetic inputs for the split-MLP hot path.

This module serves both the CUDA path and the oracle (tests hand the SAME arrays to each). It holds
none of the method's arithmetic: it only draws numbers and rounds them once to the storage dtype.

Recipe (BASELINE.json configs):
  X, dY ~ N(0, 1);  W1, W2, b1, b2 ~ N(0, std 0.02); dense, no structure.
  Element ``i`` of tensor stream ``sid`` under ``seed`` is a pure function of (seed, sid, i):
  a counter-based 64-bit mix (splitmix64 finaliser) gives two 32-bit uniforms, Box-Muller in fp64
  gives one standard normal.  No library RNG is involved, so the inputs never change with a
  numpy/torch version.  Values are then rounded ONCE (round-to-nearest-even) to the storage dtype
  (bf16 or fp32); both the GPU and the oracle see exactly those stored values.

The paper names no dataset (PAPER.md:199 uses minGPT models; throughput does not depend on token
content), so these tensors stand in for its activations/weights with GPT-style init.
"""
from __future__ import annotations

import dataclasses

import numpy as np
import torch

# Per-tensor stream ids (fixed; part of the recipe).
STREAM_X, STREAM_W1, STREAM_B1, STREAM_W2, STREAM_B2, STREAM_DY = 1, 2, 3, 4, 5, 6

_MASK64 = (1 << 64) - 1
_GOLDEN = 0x9E3779B97F4A7C15
_M1 = 0xBF58476D1CE4E5B9
_M2 = 0x94D049BB133111EB


def _s64(v: int) -> int:
    """Two's-complement reinterpretation of a 64-bit pattern as a signed Python int (torch has no uint64 math)."""
    v &= _MASK64
    return v - (1 << 64) if v >> 63 else v


def _mix64_int(z: int) -> int:
    """splitmix64 finaliser on one Python int (64-bit wrapping)."""
    z = ((z ^ (z >> 30)) * _M1) & _MASK64
    z = ((z ^ (z >> 27)) * _M2) & _MASK64
    return z ^ (z >> 31)


def _lsr(z: torch.Tensor, s: int) -> torch.Tensor:
    """Logical shift right of 64-bit patterns held in an int64 tensor."""
    return (z >> s) & ((1 << (64 - s)) - 1)


def _mix64(z: torch.Tensor) -> torch.Tensor:
    """splitmix64 finaliser on 64-bit patterns held in an int64 tensor (wrapping multiply)."""
    z = (z ^ _lsr(z, 30)) * _s64(_M1)
    z = (z ^ _lsr(z, 27)) * _s64(_M2)
    return z ^ _lsr(z, 31)


def _key(seed: int, sid: int) -> int:
    k = _mix64_int(((seed & _MASK64) * _GOLDEN + sid) & _MASK64)
    return _mix64_int((k + _GOLDEN) & _MASK64)


def standard_normal_t(seed: int, sid: int, start: int, count: int) -> torch.Tensor:
    """fp64 standard normals (torch CPU tensor) for flat indices [start, start+count) of stream (seed, sid)."""
    idx = torch.arange(start, start + count, dtype=torch.int64)
    bits = _mix64(idx * _s64(_GOLDEN) + _s64(_key(seed, sid)))
    u1 = (_lsr(bits, 32).to(torch.float64) + 0.5) * (1.0 / 4294967296.0)
    u2 = ((bits & 0xFFFFFFFF).to(torch.float64) + 0.5) * (1.0 / 4294967296.0)
    return torch.sqrt(-2.0 * torch.log(u1)) * torch.cos((2.0 * np.pi) * u2)


def standard_normal(seed: int, sid: int, start: int, count: int) -> np.ndarray:
    return standard_normal_t(seed, sid, start, count).numpy()


def normal_tensor(seed: int, sid: int, shape, std: float, dtype: torch.dtype,
                  chunk: int = 1 << 22, pin: bool = False) -> torch.Tensor:
    """CPU tensor of ``shape`` ~ N(0, std), rounded once (RNE) to ``dtype`` (torch.float32/bfloat16).

    The generator is counter-based, so the result does not depend on the chunk size or thread count."""
    n = int(np.prod(shape))
    out = torch.empty(n, dtype=dtype, pin_memory=pin)
    for s in range(0, n, chunk):
        c = min(chunk, n - s)
        out[s:s + c] = (standard_normal_t(seed, sid, s, c) * std).to(torch.float32).to(dtype)
    return out.reshape(*shape)


@dataclasses.dataclass
class MlpInputs:
    """One MLP operator's tensors, stored values (CPU).  Layout: row-major, W is [in x out]."""
    X: torch.Tensor    # [T, h]
    W1: torch.Tensor   # [h, f]
    b1: torch.Tensor   # [f]
    W2: torch.Tensor   # [f, h]
    b2: torch.Tensor   # [h]
    dY: torch.Tensor   # [T, h]

    def as_f64(self) -> dict:
        """Exact widening of the stored values to fp64 numpy (what the oracle consumes)."""
        return {k: getattr(self, k).to(torch.float64).numpy() for k in ("X", "W1", "b1", "W2", "b2", "dY")}

    def to(self, device) -> "MlpInputs":
        return MlpInputs(*[getattr(self, k).to(device) for k in ("X", "W1", "b1", "W2", "b2", "dY")])


def mlp_inputs(tokens: int, hidden: int, ffn: int, dtype: torch.dtype, seed: int = 0,
               w_std: float = 0.02, pin: bool = False) -> MlpInputs:
    """The recipe above for one operator.  ``seed`` selects the operator (C5: seed = layer index)."""
    return MlpInputs(
        X=normal_tensor(seed, STREAM_X, (tokens, hidden), 1.0, dtype, pin=pin),
        W1=normal_tensor(seed, STREAM_W1, (hidden, ffn), w_std, dtype, pin=pin),
        b1=normal_tensor(seed, STREAM_B1, (ffn,), w_std, dtype, pin=pin),
        W2=normal_tensor(seed, STREAM_W2, (ffn, hidden), w_std, dtype, pin=pin),
        b2=normal_tensor(seed, STREAM_B2, (hidden,), w_std, dtype, pin=pin),
        dY=normal_tensor(seed, STREAM_DY, (tokens, hidden), 1.0, dtype, pin=pin),
    )


@dataclasses.dataclass
class LinearInputs:
    """One Linear operator's tensors (attention projection), stored values (CPU).  W is [in x out]."""
    X: torch.Tensor    # [T, in]
    W: torch.Tensor    # [in, out]
    b: torch.Tensor    # [out]
    dY: torch.Tensor   # [T, out]

    def as_f64(self) -> dict:
        return {k: getattr(self, k).to(torch.float64).numpy() for k in ("X", "W", "b", "dY")}

    def to(self, device) -> "LinearInputs":
        return LinearInputs(*[getattr(self, k).to(device) for k in ("X", "W", "b", "dY")])


def linear_inputs(tokens: int, in_features: int, out_features: int, dtype: torch.dtype, seed: int = 0,
                  w_std: float = 0.02) -> LinearInputs:
    """Same recipe and stream ids as the MLP's first Linear: X, dY ~ N(0, 1); W, b ~ N(0, std 0.02)."""
    return LinearInputs(
        X=normal_tensor(seed, STREAM_X, (tokens, in_features), 1.0, dtype),
        W=normal_tensor(seed, STREAM_W1, (in_features, out_features), w_std, dtype),
        b=normal_tensor(seed, STREAM_B1, (out_features,), w_std, dtype),
        dY=normal_tensor(seed, STREAM_DY, (tokens, out_features), 1.0, dtype),
    )


# BASELINE.json configs, by short name.  k lists are the split counts each config is run at.
CONFIGS = {
    "C1": dict(tokens=512, hidden=256, ffn=1024, dtype="f32", ks=(4,), seed=0),
    "C2": dict(tokens=8192, hidden=1024, ffn=4096, dtype="bf16", ks=(1, 2, 4, 8), seed=0),
    "C3": dict(tokens=32768, hidden=4096, ffn=16384, dtype="bf16", ks=(1, 4, 16), seed=0),
    "C4": dict(tokens=8192, hidden=8192, ffn=32768, dtype="bf16", ks=(1, 2, 4, 8, 16, 32), seed=0),
    "C5": dict(tokens=16384, hidden=2048, ffn=8192, dtype="bf16", ks=None, seed=0, layers=24,
               act_cap_bytes=24 << 30),
}


def torch_dtype(name: str) -> torch.dtype:
    return {"f32": torch.float32, "bf16": torch.bfloat16}[name]
