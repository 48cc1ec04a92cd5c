"""ZDP (sharded) execution of the ffn-axis split MLP: pins of oracle/zdp_oracle.py against the
unsplit oracle and the paper's communication law; host logic of the library's shard layout and schedule; a world_size-2
gloo run of the same schedule.  CPU only."""
import os
import subprocess
import sys

import numpy as np
import pytest

from oracle import mlp_oracle as M
from oracle import zdp_oracle as Z

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _problem(N, T=6, h=8, f=32, seed=0):
    rng = np.random.default_rng(seed)
    W1, b1 = 0.3 * rng.standard_normal((h, f)), 0.1 * rng.standard_normal(f)
    W2, b2 = 0.3 * rng.standard_normal((f, h)), 0.1 * rng.standard_normal(h)
    Xs = [rng.standard_normal((T + r, h)) for r in range(N)]          # ranks may hold different numbers of tokens
    dYs = [rng.standard_normal((T + r, h)) for r in range(N)]
    return W1, b1, W2, b2, Xs, dYs


@pytest.mark.parametrize("N,k,unit", [(1, 1, 8), (1, 3, 4), (2, 1, 4), (2, 2, 4), (2, 4, 2), (4, 2, 2), (4, 3, 1)])
def test_oracle_sharded_schedule_equals_unsplit_mlp(N, k, unit):
    W1, b1, W2, b2, Xs, dYs = _problem(N, h=8, f=48)
    shards = Z.shard_params(W1, b1, W2, b2, k, N, unit)
    comm = Z.LocalComm(N)
    outs, gsh, alive = Z.zdp_forward_backward(Xs, dYs, shards, k, N, unit, comm)
    refs = [M.mlp_forward_backward(Xs[r], W1, b1, W2, b2, dYs[r]) for r in range(N)]
    for r in range(N):
        np.testing.assert_allclose(outs[r]["Y"], refs[r]["Y"], rtol=1e-13, atol=1e-13)
        np.testing.assert_allclose(outs[r]["dX"], refs[r]["dX"], rtol=1e-13, atol=1e-13)
    got = Z.unshard_grads(gsh, 8, 48, k, N, unit)
    for name in ("dW1", "db1", "dW2", "db2"):                          # data parallelism: gradients are summed over ranks
        np.testing.assert_allclose(got[name], sum(ref[name] for ref in refs), rtol=1e-12, atol=1e-13)
    # ZDP = three collectives (two all-gathers, one reduce-scatter) of S (N-1)/N each; b2 does not enter
    # the backward (reading S4), so it is gathered once: two collectives
    S = W1.size + b1.size + W2.size
    assert comm.recv_elems == (3 * S + 2 * b2.size) * (N - 1) // N
    # gathered size / slice_granularity (slices are whole N * unit column groups, so the widest slice)
    widest = max(hi - lo for lo, hi in Z.slice_bounds(48, k, N, unit))
    assert alive == widest * (2 * 8 + 1)


def test_oracle_shard_layout_round_trip_and_slice_bounds():
    W1, b1, W2, b2, _, _ = _problem(1, h=8, f=64, seed=3)
    for N, k, unit in ((2, 3, 4), (4, 2, 2), (1, 5, 8)):
        sh = Z.shard_params(W1, b1, W2, b2, k, N, unit)
        back = Z.unshard_grads(sh, 8, 64, k, N, unit)                  # gradients use the parameters' layout
        for got, ref in ((back["dW1"], W1), (back["db1"], b1), (back["dW2"], W2), (back["db2"], b2)):
            np.testing.assert_array_equal(got, ref)
        per_rank = sum(a.size + b.size + c.size for a, b, c in sh[0]["slices"]) + sh[0]["b2"].size
        assert per_rank * N == W1.size + b1.size + W2.size + b2.size   # model states / N
        bounds = Z.slice_bounds(64, k, N, unit)
        assert bounds[0][0] == 0 and bounds[-1][1] == 64
        assert all(a[1] == b[0] for a, b in zip(bounds, bounds[1:]))
        assert all((hi - lo) % (N * unit) == 0 for lo, hi in bounds)
