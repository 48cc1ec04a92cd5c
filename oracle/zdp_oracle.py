"""fp64 CPU oracle of the ZDP (sharded) execution of the ffn-axis split MLP.  TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s baseline legs may import this file.  It shares no
code with the CUDA path (``paper_2305_09940_b200/csrc``) and imports nothing from that package.

What it computes.  ZDP mode (section 2 "Zero Redundancy Data Parallel"): the model states of an operator
are sharded over the N data-parallel ranks; the parameters are all-gathered before the forward and again before the
backward, and the gradients are reduce-scattered - three collectives per operator instead of DP's two.
Operator splitting cuts the operator into k slices processed one after another, so that only
size(MatMul) / slice_granularity of gathered parameters exists at a time.  Every rank owns its own token batch (data
parallelism); the result the schedule must reach has a plain definition:

    Y_r, dX_r            = the UNSPLIT MLP (oracle/mlp_oracle.py) on rank r's tokens with the whole weights
    dW1, db1, dW2, db2   = the SUM over ranks of the unsplit MLP's gradients, of which rank r keeps its shard

The schedule below follows the paper step by step with an explicit ``comm`` object whose two methods are the two
collectives the paper names (ring all-gather and reduce-scatter); ``LocalComm`` runs all ranks in one
process (list in, list out), a torch.distributed (gloo) communicator with the same two methods is used by the
multi-process test.

Shard layout, slice s = ffn columns [lo_s, hi_s) in whole (N x unit)-column groups so that every
rank's piece is whole 16-byte units:
    W1[:, lo:hi]  -> rank r holds ROWS   [r h/N, (r+1) h/N)   of the [h x fs] slice   (gather = concatenate rows)
    b1[lo:hi]     -> rank r holds elements [r fs/N, (r+1) fs/N)
    W2[lo:hi, :]  -> rank r holds ROWS   [r fs/N, (r+1) fs/N) of the [fs x h] slice
    b2            -> rank r holds elements [r h/N, (r+1) h/N)
Gradients use the same layout.

Pins (tests/test_zdp.py): sharded schedule == unsplit oracle to 1e-13 for N in {1, 2, 4}, k in {1, 2, 3, 4}; shard /
unshard round trip; bytes moved per rank = 3 (N-1)/N S ("3(N-1) communication steps" of S/N each);
gathered bytes alive at a time <= 2 slices (size / slice_granularity, double-buffered).
Parity status: pinned.
"""
from __future__ import annotations

import numpy as np

from oracle import mlp_oracle as M


def slice_bounds(f: int, k: int, N: int, unit: int):
    """ffn slices in whole groups of N * unit columns: slice s = [floor(s G / k), floor((s+1) G / k)) * N * unit."""
    g = N * unit
    G = f // g
    return [((s * G) // k * g, ((s + 1) * G) // k * g) for s in range(k)]


def shard_params(W1, b1, W2, b2, k: int, N: int, unit: int):
    """Per rank: list over slices of (W1 piece, b1 piece, W2 piece), plus the b2 piece."""
    h = W1.shape[0]
    out = []
    for r in range(N):
        slices = []
        for lo, hi in slice_bounds(W1.shape[1], k, N, unit):
            fs = hi - lo
            slices.append((W1[r * h // N:(r + 1) * h // N, lo:hi].copy(), b1[lo + r * fs // N: lo + (r + 1) * fs // N].copy(),
                           W2[lo + r * fs // N: lo + (r + 1) * fs // N, :].copy()))
        out.append(dict(slices=slices, b2=b2[r * h // N:(r + 1) * h // N].copy()))
    return out


def unshard_grads(shards, h: int, f: int, k: int, N: int, unit: int):
    """Inverse of the layout for gradient shards: dict(dW1, db1, dW2, db2) whole."""
    dW1, db1, dW2, db2 = np.zeros((h, f)), np.zeros(f), np.zeros((f, h)), np.zeros(h)
    for r, sh in enumerate(shards):
        for (lo, hi), (g1, gb, g2) in zip(slice_bounds(f, k, N, unit), sh["slices"]):
            fs = hi - lo
            dW1[r * h // N:(r + 1) * h // N, lo:hi] = g1
            db1[lo + r * fs // N: lo + (r + 1) * fs // N] = gb
            dW2[lo + r * fs // N: lo + (r + 1) * fs // N, :] = g2
        db2[r * h // N:(r + 1) * h // N] = sh["b2"]
    return dict(dW1=dW1, db1=db1, dW2=dW2, db2=db2)


class LocalComm:
    """All N ranks in one process: each collective takes the list of every rank's send buffer and returns the list of
    every rank's result.  Counts the bytes each rank receives (ring algorithms: (N-1)/N of the gathered / reduced size)."""

    def __init__(self, N: int, bytes_per_elem: int = 1):
        self.N, self.e = N, bytes_per_elem
        self.recv_elems = 0
        self.calls = []

    def all_gather(self, pieces, axis=0):
        full = np.concatenate(pieces, axis=axis)
        self.recv_elems += full.size * (self.N - 1) // self.N
        self.calls.append(("all_gather", full.size))
        return [full.copy() for _ in range(self.N)]

    def reduce_scatter(self, fulls, axis=0):
        tot = sum(fulls)
        self.recv_elems += tot.size * (self.N - 1) // self.N
        self.calls.append(("reduce_scatter", tot.size))
        return [p.copy() for p in np.split(tot, self.N, axis=axis)]


def zdp_forward_backward(Xs, dYs, shards, k: int, N: int, unit: int, comm: LocalComm):
    """Xs, dYs: per-rank token batches; shards: shard_params(...).  Returns (per-rank dict(Y, dX), per-rank gradient
    shards in the layout of shard_params, max gathered parameter elements alive at a time)."""
    h = Xs[0].shape[1]
    f = sum(sl[1].size for sl in shards[0]["slices"]) * N
    bounds = slice_bounds(f, k, N, unit)
    # ---- forward: gather slice s, compute, release ("released serially")
    Y = [np.zeros((X.shape[0], h)) for X in Xs]
    alive_max = 0
    for s, (lo, hi) in enumerate(bounds):
        W1s = comm.all_gather([sh["slices"][s][0] for sh in shards], axis=0)      # first all-gather
        b1s = comm.all_gather([sh["slices"][s][1] for sh in shards], axis=0)
        W2s = comm.all_gather([sh["slices"][s][2] for sh in shards], axis=0)
        alive_max = max(alive_max, W1s[0].size + b1s[0].size + W2s[0].size)
        for r in range(N):
            Y[r] += M.gelu(Xs[r] @ W1s[r] + b1s[r][None, :]) @ W2s[r]           # partial products summed
    b2 = comm.all_gather([sh["b2"] for sh in shards], axis=0)
    for r in range(N):
        Y[r] += b2[r][None, :]
    # ---- backward: gather again, compute, reduce-scatter the slice's gradients
    dX = [np.zeros_like(X) for X in Xs]
    gshards = [dict(slices=[], b2=None) for _ in range(N)]
    for s, (lo, hi) in enumerate(bounds):
        W1s = comm.all_gather([sh["slices"][s][0] for sh in shards], axis=0)      # second all-gather
        b1s = comm.all_gather([sh["slices"][s][1] for sh in shards], axis=0)
        W2s = comm.all_gather([sh["slices"][s][2] for sh in shards], axis=0)
        g1, gb, g2 = [], [], []
        for r in range(N):
            Z = Xs[r] @ W1s[r] + b1s[r][None, :]
            H = M.gelu(Z)
            dZ = (dYs[r] @ W2s[r].T) * M.gelu_prime(Z)
            g2.append(H.T @ dYs[r])
            g1.append(Xs[r].T @ dZ)
            gb.append(dZ.sum(axis=0))
            dX[r] += dZ @ W1s[r].T
        r1, rb, r2 = comm.reduce_scatter(g1, axis=0), comm.reduce_scatter(gb, axis=0), comm.reduce_scatter(g2, axis=0)
        for r in range(N):
            gshards[r]["slices"].append((r1[r], rb[r], r2[r]))
    rb2 = comm.reduce_scatter([dY.sum(axis=0) for dY in dYs], axis=0)
    for r in range(N):
        gshards[r]["b2"] = rb2[r]
    return [dict(Y=Y[r], dX=dX[r]) for r in range(N)], gshards, alive_max
