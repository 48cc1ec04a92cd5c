"""Pins of oracle/linear_oracle.py (the Linear operator of the attention block) against things
other than itself: scalar loops, finite differences, torch autograd, special cases, the MLP oracle.  CPU only."""
import numpy as np
import pytest
import torch

from oracle import linear_oracle as L
from oracle import mlp_oracle as M


def _rand(T, n_in, n_out, seed=0):
    rng = np.random.default_rng(seed)
    return (rng.standard_normal((T, n_in)), 0.3 * rng.standard_normal((n_in, n_out)), 0.3 * rng.standard_normal(n_out),
            rng.standard_normal((T, n_out)))


def test_matches_scalar_loops():
    X, W, b, dY = _rand(3, 5, 4)
    ref = L.brute_force(X.tolist(), W.tolist(), b.tolist(), dY.tolist())
    got = L.linear_forward_backward(X, W, b, dY)
    for name in ("Y", "dX", "dW", "db"):
        np.testing.assert_allclose(got[name], np.array(ref[name]), rtol=1e-13, atol=1e-13)
    # a transposed operand or a swapped X / dY would change shapes or values: check shapes explicitly
    assert got["Y"].shape == (3, 4) and got["dX"].shape == (3, 5) and got["dW"].shape == (5, 4) and got["db"].shape == (4,)


def test_matches_torch_autograd_fp64():
    X, W, b, dY = _rand(7, 6, 9, seed=1)
    tX, tW, tb = (torch.tensor(a, requires_grad=True) for a in (X, W, b))
    tY = tX @ tW + tb
    tY.backward(torch.tensor(dY))
    got = L.linear_forward_backward(X, W, b, dY)
    np.testing.assert_allclose(got["Y"], tY.detach().numpy(), rtol=1e-13, atol=1e-13)
    np.testing.assert_allclose(got["dX"], tX.grad.numpy(), rtol=1e-13, atol=1e-13)
    np.testing.assert_allclose(got["dW"], tW.grad.numpy(), rtol=1e-13, atol=1e-13)
    np.testing.assert_allclose(got["db"], tb.grad.numpy(), rtol=1e-13, atol=1e-13)


@pytest.mark.parametrize("which", ["X", "W", "b"])
def test_finite_differences(which):
    X, W, b, dY = _rand(4, 5, 3, seed=2)
    g = L.linear_backward(X, W, dY)
    rng = np.random.default_rng(9)
    p = {"X": X, "W": W, "b": b}[which]
    v = rng.standard_normal(p.shape)
    eps = 1e-6

    def loss(sign):
        q = {"X": X, "W": W, "b": b}
        q[which] = p + sign * eps * v
        return float((L.linear_forward(q["X"], q["W"], q["b"]) * dY).sum())

    fd = (loss(+1) - loss(-1)) / (2 * eps)
    an = float(({"X": g["dX"], "W": g["dW"], "b": g["db"]}[which] * v).sum())
    assert abs(fd - an) <= 1e-7 * max(1.0, abs(an))


def test_special_cases():
    X, W, b, dY = _rand(5, 4, 6, seed=3)
    out = L.linear_forward_backward(X, np.zeros_like(W), b, dY)
    np.testing.assert_array_equal(out["Y"], np.broadcast_to(b, (5, 6)))
    np.testing.assert_array_equal(out["dX"], np.zeros_like(X))
    np.testing.assert_allclose(out["dW"], X.T @ dY, rtol=1e-13)               # dW does not depend on W
    E = np.eye(4)
    np.testing.assert_allclose(L.linear_forward(E, W, None), W, rtol=0, atol=0)   # X = identity picks the rows of W
    np.testing.assert_array_equal(L.linear_backward(E, W, np.eye(4, 6))["dX"], W[:, :4].T)   # dY = e_o picks a column of W
    np.testing.assert_array_equal(L.linear_forward(X, W, None) + b[None, :], L.linear_forward(X, W, b))


def test_consistent_with_the_mlp_oracle():
    """The MLP's second Linear is this operator applied to H: Y, dH, dW2, db2 must agree with oracle/mlp_oracle.py."""
    rng = np.random.default_rng(4)
    T, h, f = 6, 8, 16
    X, W1, b1 = rng.standard_normal((T, h)), 0.3 * rng.standard_normal((h, f)), 0.1 * rng.standard_normal(f)
    W2, b2, dY = 0.3 * rng.standard_normal((f, h)), 0.1 * rng.standard_normal(h), rng.standard_normal((T, h))
    ref = M.mlp_forward_backward(X, W1, b1, W2, b2, dY)
    _, Z, H = M.mlp_forward(X, W1, b1, W2, b2)
    lin = L.linear_forward_backward(H, W2, b2, dY)
    np.testing.assert_allclose(lin["Y"], ref["Y"], rtol=1e-13, atol=1e-13)
    np.testing.assert_allclose(lin["dW"], ref["dW2"], rtol=1e-13, atol=1e-13)
    np.testing.assert_allclose(lin["db"], ref["db2"], rtol=1e-13, atol=1e-13)
    first = L.linear_backward(X, W1, lin["dX"] * M.gelu_prime(Z))              # chain rule through the first Linear
    np.testing.assert_allclose(first["dX"], ref["dX"], rtol=1e-12, atol=1e-13)
    np.testing.assert_allclose(first["dW"], ref["dW1"], rtol=1e-12, atol=1e-13)
    np.testing.assert_allclose(first["db"], ref["db1"], rtol=1e-12, atol=1e-13)


@pytest.mark.parametrize("k", [1, 2, 3, 4, 7])
def test_split_equals_unsplit_both_axes(k):
    """'all computation results are summed as the final output'."""
    X, W, b, dY = _rand(14, 56, 24, seed=5)
    ref = L.linear_forward_backward(X, W, b, dY)
    for got in (L.linear_forward_backward_contraction_split(X, W, b, dY, k, unit=8),
                L.linear_forward_backward_token_split(X, W, b, dY, k)):
        for name in ("Y", "dX", "dW", "db"):
            np.testing.assert_allclose(got[name], ref[name], rtol=1e-13, atol=1e-13)
    assert L.slice_bounds(56, k, 8)[0][0] == 0 and L.slice_bounds(56, k, 8)[-1][1] == 56
    assert all(lo % 8 == 0 and hi % 8 == 0 for lo, hi in L.slice_bounds(56, k, 8))


def test_sampled_restrictions():
    X, W, b, dY = _rand(9, 8, 12, seed=6)
    ref = L.linear_forward_backward(X, W, b, dY)
    r = L.sampled_rows(X, W, b, dY, [0, 4, 8])
    np.testing.assert_allclose(r["Y"], ref["Y"][[0, 4, 8]], rtol=1e-13)
    np.testing.assert_allclose(r["dX"], ref["dX"][[0, 4, 8]], rtol=1e-13)
    c = L.sampled_cols(X, dY, [1, 11])
    np.testing.assert_allclose(c["dW_cols"], ref["dW"][:, [1, 11]], rtol=1e-13)
    np.testing.assert_allclose(c["db"], ref["db"][[1, 11]], rtol=1e-13)
