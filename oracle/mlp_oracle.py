"""fp64 CPU oracle for the split-MLP hot path.  TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import this file.  It shares no code with the CUDA path (``paper_2305_09940_b200/csrc``) and
imports nothing from that package.

What it computes.  OSDP's operator splitting (§3.3 "Operator Splitting") processes a
huge operator slice by slice and "all computation results are summed as the final output": the split
is an execution schedule, not an approximation, so the result it must reach has a plain definition —
the UNSPLIT transformer MLP operator, forward and backward.  That definition is written out below in
fp64 (readings S1-S6 in DESIGN.md):

    1. Z  = X W1 + 1 b1^T          (T x f)      6. dH = dY W2^T               (T x f)
    2. H  = gelu(Z)                             7. dZ = dH (.) gelu'(Z)
    3. Y  = H W2 + 1 b2^T          (T x h)      8. db1 = sum_t dZ[t, :]
    4. db2 = sum_t dY[t, :]                     9. dW1 = X^T dZ               (h x f)
    5. dW2 = H^T dY                (f x h)     10. dX  = dZ W1^T              (T x h)

    gelu(z)  = 1/2 z (1 + tanh u),  u = c (z + a z^3),  c = sqrt(2/pi),  a = 0.044715   (reading S2)
    gelu'(z) = 1/2 (1 + tanh u) + 1/2 z (1 - tanh^2 u) c (1 + 3 a z^2)

Weights are [in x out] ("first dimension of the operator" is the contraction axis).
Inputs are the STORED values (already rounded to bf16/fp32) widened exactly to fp64; no intermediate
rounding is applied.  Library primitive used as a step: numpy ``@`` (fp64 matmul).  No blocking, fusion
or reordering.

Pins (tests/test_oracle_pins.py): brute-force scalar loops at 4x8x16; central finite differences;
torch fp64 autograd (independent derivation of steps 4-10); torch's own tanh-GeLU; closed-form
values/identities/limits of gelu and gelu'; special cases (W2 = 0, large b1); split == unsplit.
Parity status: pinned (no "parity unpinned" function in this file).  The paper's own Fig. 7/8 curves
are images and cannot be compared: those stay unpinned against the paper.
"""
from __future__ import annotations

import math

import numpy as np

GELU_C = math.sqrt(2.0 / math.pi)   # 0.7978845608028654
GELU_A = 0.044715


def gelu(z: np.ndarray) -> np.ndarray:
    """tanh-approximate GeLU (reading S2)."""
    u = GELU_C * (z + GELU_A * z * z * z)
    return 0.5 * z * (1.0 + np.tanh(u))


def gelu_prime(z: np.ndarray) -> np.ndarray:
    """d gelu / dz."""
    u = GELU_C * (z + GELU_A * z * z * z)
    t = np.tanh(u)
    return 0.5 * (1.0 + t) + 0.5 * z * (1.0 - t * t) * GELU_C * (1.0 + 3.0 * GELU_A * z * z)


def mlp_forward(X, W1, b1, W2, b2):
    """Steps 1-3.  Returns (Y, Z, H), all fp64."""
    Z = X @ W1 + b1[None, :]
    H = gelu(Z)
    Y = H @ W2 + b2[None, :]
    return Y, Z, H


def mlp_backward(X, W1, b1, W2, dY):
    """Steps 4-10 (Z, H recomputed from the inputs: the backward takes no saved activations).

    Returns dict(dX, dW1, db1, dW2, db2), all fp64.  b2 does not enter the backward (reading S4).
    """
    Z = X @ W1 + b1[None, :]
    H = gelu(Z)
    db2 = dY.sum(axis=0)
    dW2 = H.T @ dY
    dH = dY @ W2.T
    dZ = dH * gelu_prime(Z)
    db1 = dZ.sum(axis=0)
    dW1 = X.T @ dZ
    dX = dZ @ W1.T
    return dict(dX=dX, dW1=dW1, db1=db1, dW2=dW2, db2=db2)


def mlp_forward_backward(X, W1, b1, W2, b2, dY):
    """Whole path, unsplit: dict(Y, dX, dW1, db1, dW2, db2)."""
    Y, _, _ = mlp_forward(X, W1, b1, W2, b2)
    out = mlp_backward(X, W1, b1, W2, dY)
    out["Y"] = Y
    return out


# ----------------------------------------------------------------------------------------------
# The split schedule itself, in fp64 ("the computation of each slice is executed
# sequentially ... all computation results are summed as the final output").  Token-axis reading
# (S1).  Used only to pin "split == unsplit"; ragged slices follow reading S7:
# slice s = rows [floor(s T / k), floor((s+1) T / k)).
# ----------------------------------------------------------------------------------------------
def slice_bounds(T: int, k: int):
    return [((s * T) // k, ((s + 1) * T) // k) for s in range(k)]


def mlp_forward_backward_split(X, W1, b1, W2, b2, dY, k: int):
    T = X.shape[0]
    Y = np.empty((T, W2.shape[1]))
    dX = np.empty_like(X)
    dW1 = np.zeros_like(W1)
    dW2 = np.zeros_like(W2)
    db1 = np.zeros_like(b1)
    db2 = np.zeros_like(b2)
    for lo, hi in slice_bounds(T, k):
        Ys, _, _ = mlp_forward(X[lo:hi], W1, b1, W2, b2)
        Y[lo:hi] = Ys
        g = mlp_backward(X[lo:hi], W1, b1, W2, dY[lo:hi])
        dX[lo:hi] = g["dX"]
        dW1 += g["dW1"]
        dW2 += g["dW2"]
        db1 += g["db1"]
        db2 += g["db2"]
    return dict(Y=Y, dX=dX, dW1=dW1, db1=db1, dW2=dW2, db2=db2)


def matmul_contraction_split(X, W, granularity: int):
    """The paper-literal split of ONE MatMul (Fig. 4): the last dimension of the input
    and the first dimension of the operator are partitioned into ``granularity`` slices, the slices
    are computed one after another, and the partial results are summed."""
    K = X.shape[1]
    out = np.zeros((X.shape[0], W.shape[1]))
    for lo, hi in slice_bounds(K, granularity):
        out += X[:, lo:hi] @ W[lo:hi, :]
    return out


def ffn_slice_bounds(f: int, k: int, unit: int):
    """Slices of the ffn axis in whole ``unit``-column groups (unit = 16 bytes of storage elements):
    slice s = columns [floor(s U / k) unit, floor((s + 1) U / k) unit) with U = f / unit."""
    U = f // unit
    return [((s * U) // k * unit, ((s + 1) * U) // k * unit) for s in range(k)]


def mlp_forward_backward_ffn_split(X, W1, b1, W2, b2, dY, k: int, unit: int = 8):
    """The paper-literal split applied to the MLP pair, in fp64: Linear2's contraction
    axis (= Linear1's output axis) is cut into k slices, the slices are computed one after another and
    the partial products of Y and of dX are summed; each slice writes its own rows of dW2 and columns
    of dW1 / db1.  Used only to pin "ffn split == unsplit"."""
    T, f = X.shape[0], W1.shape[1]
    Y = np.zeros((T, W2.shape[1]))
    dX = np.zeros_like(X)
    dW1 = np.empty_like(W1)
    dW2 = np.empty_like(W2)
    db1 = np.empty_like(b1)
    for lo, hi in ffn_slice_bounds(f, k, unit):
        Zs = X @ W1[:, lo:hi] + b1[None, lo:hi]
        Hs = gelu(Zs)
        Y += Hs @ W2[lo:hi, :]
        dZs = (dY @ W2[lo:hi, :].T) * gelu_prime(Zs)
        dW2[lo:hi, :] = Hs.T @ dY
        dW1[:, lo:hi] = X.T @ dZs
        db1[lo:hi] = dZs.sum(axis=0)
        dX += dZs @ W1[:, lo:hi].T
    Y += b2[None, :]
    return dict(Y=Y, dX=dX, dW1=dW1, db1=db1, dW2=dW2, db2=dY.sum(axis=0))


# ----------------------------------------------------------------------------------------------
# Sampled oracle for the large configs (SURVEY.md §8(c) "GPU vs oracle"): the SAME definition,
# restricted to a subset of token rows or of ffn columns.  Every output tensor is covered:
#   rows t  ->  Y[t, :], dX[t, :]          (4 h f MACs each)
#   cols j  ->  dW2[j, :], dW1[:, j], db1[j]   (4 T h MACs each)
#   db2 in full.
# ----------------------------------------------------------------------------------------------
def sampled_rows(X, W1, b1, W2, b2, dY, rows):
    rows = np.asarray(rows)
    Zr = X[rows] @ W1 + b1[None, :]
    Hr = gelu(Zr)
    Yr = Hr @ W2 + b2[None, :]
    dHr = dY[rows] @ W2.T
    dZr = dHr * gelu_prime(Zr)
    dXr = dZr @ W1.T
    return dict(Y=Yr, dX=dXr)


def sampled_cols(X, W1, b1, W2, dY, cols):
    cols = np.asarray(cols)
    Zc = X @ W1[:, cols] + b1[None, cols]        # T x c
    Hc = gelu(Zc)
    dW2c = Hc.T @ dY                             # c x h   = dW2[cols, :]
    dHc = dY @ W2[cols, :].T                     # T x c
    dZc = dHc * gelu_prime(Zc)
    db1c = dZc.sum(axis=0)                       # c       = db1[cols]
    dW1c = X.T @ dZc                             # h x c   = dW1[:, cols]
    return dict(dW2_rows=dW2c, dW1_cols=dW1c, db1=db1c)


def db2_full(dY):
    return dY.sum(axis=0)


# ----------------------------------------------------------------------------------------------
# Brute force (pure-Python scalar loops; tiny shapes only) — used by the pins, kept here so the
# loops can be read against steps 1-10 by eye.
# ----------------------------------------------------------------------------------------------
def _gelu_scalar(z: float) -> float:
    return 0.5 * z * (1.0 + math.tanh(GELU_C * (z + GELU_A * z ** 3)))


def brute_force_forward(X, W1, b1, W2, b2):
    T, h = len(X), len(X[0])
    f = len(b1)
    Y = [[0.0] * h for _ in range(T)]
    for t in range(T):
        Hrow = []
        for j in range(f):
            z = b1[j]
            for i in range(h):
                z += X[t][i] * W1[i][j]
            Hrow.append(_gelu_scalar(z))
        for o in range(h):
            y = b2[o]
            for j in range(f):
                y += Hrow[j] * W2[j][o]
            Y[t][o] = y
    return Y
