"""fp64 CPU oracle for the split Linear operator (attention projections).  TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s baseline legs may import this file.  It shares no
code with the CUDA path (``paper_2305_09940_b200/csrc``) and imports nothing from that package.

What it computes.  The paper's models have two operators per layer, an attention block and an MLP block (Table 1,
PAPER.md:191-195: Operator Num = 2 x Layer Num + 2); the MatMuls of the attention block are plain Linear operators
(minGPT's c_attn: hidden -> 3 hidden, c_proj: hidden -> hidden).  Operator splitting (PAPER.md:165,
section 3.3) partitions "the last dimension of the input data and the first dimension of the operator" into slices,
computes the slices one after another and sums the results: an execution schedule, not an approximation, so the result
it must reach is the UNSPLIT operator, written out here in fp64:

    forward :  Y  = X W + 1 b^T                 X [T x in], W [in x out] (weights are [in x out]), b [out]
    backward:  dX = dY W^T          [T x in]
               dW = X^T dY          [in x out]
               db = sum_t dY[t, :]  [out]

Inputs are the STORED values (already rounded to bf16/fp32) widened exactly to fp64; no intermediate rounding.
Library primitive used as a step: numpy ``@``.  The two schedules (contraction-axis slices, the paper's own; token
slices) are written out below only to pin "split == unsplit".

Pins (tests/test_linear_oracle.py): pure-Python scalar loops at 3 x 5 x 4; central finite differences of
L = sum(Y * dY) per parameter; torch fp64 autograd; special cases (W = 0 => Y = b broadcast, dX = 0; X = e_i picks a
row of W); consistency with oracle/mlp_oracle.py (an MLP whose second Linear is this operator); split == unsplit to
1e-13 for both axes.  Parity status: pinned.
"""
from __future__ import annotations

import numpy as np


def linear_forward(X, W, b=None):
    Y = X @ W
    if b is not None:
        Y = Y + b[None, :]
    return Y


def linear_backward(X, W, dY):
    """dict(dX, dW, db)."""
    return dict(dX=dY @ W.T, dW=X.T @ dY, db=dY.sum(axis=0))


def linear_forward_backward(X, W, b, dY):
    out = linear_backward(X, W, dY)
    out["Y"] = linear_forward(X, W, b)
    return out


def slice_bounds(n: int, k: int, unit: int = 1):
    """k slices of an axis of n elements in whole groups of ``unit``: slice s = [floor(s U / k) unit, floor((s+1) U / k) unit),
    U = n / unit (unit = 1 for token rows; 16 bytes of storage elements for the contraction axis)."""
    U = n // unit
    return [((s * U) // k * unit, ((s + 1) * U) // k * unit) for s in range(k)]


def linear_forward_backward_contraction_split(X, W, b, dY, k: int, unit: int = 8):
    """The paper-literal split (Fig. 4): slice s owns input features [lo, hi); partial products of Y are
    summed; dX[:, lo:hi] and dW[lo:hi, :] belong to one slice each."""
    Y = np.zeros((X.shape[0], W.shape[1]))
    dX = np.empty_like(X)
    dW = np.empty_like(W)
    for lo, hi in slice_bounds(X.shape[1], k, unit):
        Y += X[:, lo:hi] @ W[lo:hi, :]
        dX[:, lo:hi] = dY @ W[lo:hi, :].T
        dW[lo:hi, :] = X[:, lo:hi].T @ dY
    if b is not None:
        Y += b[None, :]
    return dict(Y=Y, dX=dX, dW=dW, db=dY.sum(axis=0))


def linear_forward_backward_token_split(X, W, b, dY, k: int):
    """Token slices (the north_star's axis): rows [floor(s T / k), floor((s+1) T / k)); dW and db are summed over slices."""
    T = X.shape[0]
    Y = np.empty((T, W.shape[1]))
    dX = np.empty_like(X)
    dW = np.zeros_like(W)
    db = np.zeros(W.shape[1])
    for lo, hi in slice_bounds(T, k):
        Y[lo:hi] = linear_forward(X[lo:hi], W, b)
        g = linear_backward(X[lo:hi], W, dY[lo:hi])
        dX[lo:hi] = g["dX"]
        dW += g["dW"]
        db += g["db"]
    return dict(Y=Y, dX=dX, dW=dW, db=db)


# Sampled restriction for full-size checks: rows t -> Y[t, :], dX[t, :]; columns j of the OUTPUT axis -> dW[:, j], db[j].
def sampled_rows(X, W, b, dY, rows):
    rows = np.asarray(rows)
    Y = X[rows] @ W + (b[None, :] if b is not None else 0.0)
    return dict(Y=Y, dX=dY[rows] @ W.T)


def sampled_cols(X, dY, cols):
    cols = np.asarray(cols)
    return dict(dW_cols=X.T @ dY[:, cols], db=dY[:, cols].sum(axis=0))


def brute_force(X, W, b, dY):
    """Pure-Python scalar loops (tiny shapes only), to be read against the four formulas by eye."""
    T, n_in, n_out = len(X), len(W), len(W[0])
    Y = [[(b[o] if b is not None else 0.0) + sum(X[t][i] * W[i][o] for i in range(n_in)) for o in range(n_out)] for t in range(T)]
    dX = [[sum(dY[t][o] * W[i][o] for o in range(n_out)) for i in range(n_in)] for t in range(T)]
    dW = [[sum(X[t][i] * dY[t][o] for t in range(T)) for o in range(n_out)] for i in range(n_in)]
    db = [sum(dY[t][o] for t in range(T)) for o in range(n_out)]
    return dict(Y=Y, dX=dX, dW=dW, db=db)
