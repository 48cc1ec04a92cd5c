"""Pins for oracle/mlp_oracle.py: the oracle is checked against things other than itself.

Each pin is chosen so that a plausible mistake (dropped term, wrong sign/index, transposed operand)
fails at least one of them.  CPU only.
"""
import math
import os

import numpy as np
import pytest
import torch

from oracle import mlp_oracle as O

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _rand(shape, seed, scale=1.0):
    return np.random.default_rng(seed).standard_normal(shape) * scale


def _tiny(T=4, h=8, f=16, seed=0, wscale=0.5):
    return dict(X=_rand((T, h), seed), W1=_rand((h, f), seed + 1, wscale), b1=_rand((f,), seed + 2, wscale),
                W2=_rand((f, h), seed + 3, wscale), b2=_rand((h,), seed + 4, wscale), dY=_rand((T, h), seed + 5))


# ---------------------------------------------------------------- GeLU
def test_gelu_golden_values():
    """Values from tests/golden/gelu_values.txt."""
    fn = {"gelu": O.gelu, "gelu_prime": O.gelu_prime}
    n = 0
    for line in open(os.path.join(GOLDEN, "gelu_values.txt")):
        if line.startswith("#") or not line.strip():
            continue
        name, z, v = line.split()
        assert abs(float(fn[name](np.array(float(z)))) - float(v)) < 5e-15, (name, z)
        n += 1
    assert n == 6


def test_gelu_identities_and_limits():
    z = np.linspace(-12, 12, 4801)
    assert np.allclose(O.gelu(z) - O.gelu(-z), z, rtol=0, atol=1e-14)          # odd part is z/2
    assert np.allclose(O.gelu_prime(z) + O.gelu_prime(-z), 1.0, rtol=0, atol=1e-14)
    assert O.gelu(np.array(0.0)) == 0.0 and O.gelu_prime(np.array(0.0)) == 0.5
    assert abs(O.gelu(np.array(30.0)) - 30.0) < 1e-12 and abs(O.gelu_prime(np.array(30.0)) - 1.0) < 1e-12
    assert abs(O.gelu(np.array(-30.0))) < 1e-12 and abs(O.gelu_prime(np.array(-30.0))) < 1e-12
    assert abs(O.GELU_C - 0.7978845608028654) < 1e-16 and O.GELU_A == 0.044715


def test_gelu_matches_torch_tanh_gelu_and_is_close_to_erf_gelu():
    z = torch.linspace(-8, 8, 3201, dtype=torch.float64, requires_grad=True)
    g = torch.nn.functional.gelu(z, approximate="tanh")
    g.sum().backward()
    assert np.allclose(O.gelu(z.detach().numpy()), g.detach().numpy(), rtol=0, atol=1e-14)
    assert np.allclose(O.gelu_prime(z.detach().numpy()), z.grad.numpy(), rtol=0, atol=1e-13)
    # the tanh form approximates x*Phi(x) to within ~5e-4 everywhere (Hendrycks & Gimpel)
    exact = torch.nn.functional.gelu(z.detach()).numpy()
    assert np.max(np.abs(O.gelu(z.detach().numpy()) - exact)) < 1e-3


def test_gelu_prime_is_derivative_of_gelu():
    z = np.linspace(-6, 6, 1201)
    e = 1e-6
    fd = (O.gelu(z + e) - O.gelu(z - e)) / (2 * e)
    assert np.max(np.abs(fd - O.gelu_prime(z))) < 1e-9


# ---------------------------------------------------------------- forward
def test_forward_brute_force_4x8x16():
    d = _tiny()
    Y, _, _ = O.mlp_forward(d["X"], d["W1"], d["b1"], d["W2"], d["b2"])
    Yb = O.brute_force_forward(d["X"].tolist(), d["W1"].tolist(), d["b1"].tolist(), d["W2"].tolist(),
                               d["b2"].tolist())
    assert np.max(np.abs(Y - np.array(Yb))) < 1e-13


def test_forward_special_cases():
    d = _tiny(T=5, h=6, f=12, seed=10)
    Y, _, _ = O.mlp_forward(d["X"], d["W1"], d["b1"], np.zeros_like(d["W2"]), d["b2"])
    assert np.array_equal(Y, np.broadcast_to(d["b2"], Y.shape))                 # W2 = 0 => Y = b2
    big = d["b1"] + 40.0                                                         # gelu -> identity
    Y, _, _ = O.mlp_forward(d["X"], d["W1"] * 0.1, big, d["W2"], d["b2"])
    lin = (d["X"] @ (d["W1"] * 0.1) + big) @ d["W2"] + d["b2"]
    assert np.allclose(Y, lin, rtol=1e-12, atol=1e-10)


def test_forward_matches_torch():
    d = _tiny(T=7, h=12, f=20, seed=3)
    t = {k: torch.from_numpy(v) for k, v in d.items()}
    Yt = torch.nn.functional.gelu(t["X"] @ t["W1"] + t["b1"], approximate="tanh") @ t["W2"] + t["b2"]
    Y, _, _ = O.mlp_forward(d["X"], d["W1"], d["b1"], d["W2"], d["b2"])
    assert np.allclose(Y, Yt.numpy(), rtol=1e-13, atol=1e-13)


# ---------------------------------------------------------------- backward
def test_backward_matches_torch_autograd():
    """Independent derivation: reverse-mode autodiff of L = sum(Y * dY) vs the oracle's hand-written steps."""
    d = _tiny(T=9, h=10, f=24, seed=7)
    t = {k: torch.from_numpy(v).clone().requires_grad_(k != "dY") for k, v in d.items()}
    Y = torch.nn.functional.gelu(t["X"] @ t["W1"] + t["b1"], approximate="tanh") @ t["W2"] + t["b2"]
    (Y * t["dY"]).sum().backward()
    g = O.mlp_backward(d["X"], d["W1"], d["b1"], d["W2"], d["dY"])
    for name, key in (("dX", "X"), ("dW1", "W1"), ("db1", "b1"), ("dW2", "W2"), ("db2", "b2")):
        assert g[name].shape == d[key].shape
        assert np.allclose(g[name], t[key].grad.numpy(), rtol=1e-12, atol=1e-12), name


@pytest.mark.parametrize("param", ["X", "W1", "b1", "W2", "b2"])
def test_backward_finite_differences(param):
    """(L(theta + e v) - L(theta - e v)) / 2e = <grad, v>,  L = sum(Y * dY)."""
    d = _tiny(T=4, h=8, f=16, seed=21)
    g = O.mlp_forward_backward(**d)
    grad = {"X": g["dX"], "W1": g["dW1"], "b1": g["db1"], "W2": g["dW2"], "b2": g["db2"]}[param]
    v = _rand(d[param].shape, 99)
    e = 1e-6

    def L(sign):
        dd = dict(d)
        dd[param] = d[param] + sign * e * v
        Y, _, _ = O.mlp_forward(dd["X"], dd["W1"], dd["b1"], dd["W2"], dd["b2"])
        return float((Y * d["dY"]).sum())

    fd = (L(+1) - L(-1)) / (2 * e)
    assert abs(fd - float((grad * v).sum())) < 1e-7 * max(1.0, abs(fd))


def test_backward_special_cases():
    d = _tiny(T=6, h=8, f=16, seed=5)
    g = O.mlp_backward(d["X"], d["W1"], d["b1"], d["W2"], d["dY"])
    assert np.allclose(g["db2"], np.array([sum(d["dY"][:, j]) for j in range(8)]), rtol=0, atol=1e-14)
    g0 = O.mlp_backward(d["X"], d["W1"], d["b1"], np.zeros_like(d["W2"]), d["dY"])
    assert not g0["dW1"].any() and not g0["db1"].any() and not g0["dX"].any()     # W2 = 0
    g2 = O.mlp_backward(d["X"], d["W1"], d["b1"], d["W2"], 2.0 * d["dY"])          # linear in dY
    for kname in g:
        assert np.allclose(g2[kname], 2.0 * g[kname], rtol=1e-14, atol=0)


# ---------------------------------------------------------------- splitting
@pytest.mark.parametrize("k", [1, 2, 3, 4, 7, 16])
def test_split_equals_unsplit(k):
    d = _tiny(T=32, h=8, f=16, seed=11)
    ref = O.mlp_forward_backward(**d)
    got = O.mlp_forward_backward_split(**d, k=k)
    for name in ref:
        scale = np.max(np.abs(ref[name]))
        assert np.max(np.abs(ref[name] - got[name])) <= 1e-13 * scale, name


def test_slice_bounds_partition():
    for T, k in ((32, 4), (33, 4), (5, 5), (7, 3), (100, 16)):
        b = O.slice_bounds(T, k)
        assert b[0][0] == 0 and b[-1][1] == T and all(b[i][1] == b[i + 1][0] for i in range(k - 1))
        assert max(hi - lo for lo, hi in b) == -(-T // k)


@pytest.mark.parametrize("g", [1, 2, 4, 16])
def test_paper_literal_contraction_split(g):
    """'all computation results are summed as the final output'."""
    X, W = _rand((6, 32), 1), _rand((32, 10), 2)
    ref = np.array([[sum(X[i, k] * W[k, j] for k in range(32)) for j in range(10)] for i in range(6)])
    assert np.allclose(O.matmul_contraction_split(X, W, g), ref, rtol=1e-13, atol=1e-13)


@pytest.mark.parametrize("k,unit", [(1, 8), (2, 8), (3, 8), (5, 8), (6, 8), (4, 4), (12, 4)])
def test_ffn_split_equals_unsplit(k, unit):
    """The paper-literal split of the MLP pair along ffn: summed partial products == unsplit."""
    d = _tiny(T=12, h=8, f=48, seed=12)
    ref = O.mlp_forward_backward(**d)
    got = O.mlp_forward_backward_ffn_split(**d, k=k, unit=unit)
    for name in ref:
        scale = np.max(np.abs(ref[name]))
        assert np.max(np.abs(ref[name] - got[name])) <= 1e-13 * scale, name


def test_ffn_slice_bounds_partition_in_whole_units():
    for f, k, unit in ((48, 5, 8), (520, 3, 8), (1032, 4, 8), (68, 4, 4), (8, 1, 8), (64, 8, 8)):
        b = O.ffn_slice_bounds(f, k, unit)
        assert b[0][0] == 0 and b[-1][1] == f and all(b[i][1] == b[i + 1][0] for i in range(k - 1))
        assert all(lo % unit == 0 and hi % unit == 0 and hi > lo for lo, hi in b)
        assert max(hi - lo for lo, hi in b) == -(-(f // unit) // k) * unit


# ---------------------------------------------------------------- sampled oracle == full oracle
def test_sampled_oracle_is_a_restriction_of_the_full_one():
    d = _tiny(T=20, h=8, f=24, seed=13)
    ref = O.mlp_forward_backward(**d)
    rows = [0, 3, 19]
    cols = [0, 5, 23]
    r = O.sampled_rows(d["X"], d["W1"], d["b1"], d["W2"], d["b2"], d["dY"], rows)
    c = O.sampled_cols(d["X"], d["W1"], d["b1"], d["W2"], d["dY"], cols)
    assert np.allclose(r["Y"], ref["Y"][rows], rtol=1e-13, atol=1e-13)
    assert np.allclose(r["dX"], ref["dX"][rows], rtol=1e-13, atol=1e-13)
    assert np.allclose(c["dW2_rows"], ref["dW2"][cols, :], rtol=1e-13, atol=1e-13)
    assert np.allclose(c["dW1_cols"], ref["dW1"][:, cols], rtol=1e-13, atol=1e-13)
    assert np.allclose(c["db1"], ref["db1"][cols], rtol=1e-13, atol=1e-13)
    assert np.allclose(O.db2_full(d["dY"]), ref["db2"], rtol=1e-14, atol=1e-14)


# ---------------------------------------------------------------- input generator
def test_inputs_are_seeded_and_distributed_as_stated():
    from paper_2305_09940_b200 import inputs as I
    a = I.standard_normal(0, I.STREAM_X, 0, 200000)
    b = I.standard_normal(0, I.STREAM_X, 0, 200000)
    assert np.array_equal(a, b)
    assert np.array_equal(a[1000:1010], I.standard_normal(0, I.STREAM_X, 1000, 10))   # counter-based
    assert not np.array_equal(a, I.standard_normal(1, I.STREAM_X, 0, 200000))
    assert not np.array_equal(a, I.standard_normal(0, I.STREAM_DY, 0, 200000))
    assert abs(a.mean()) < 0.01 and abs(a.std() - 1.0) < 0.01
    assert abs(np.mean(a ** 4) - 3.0) < 0.1                                           # normal kurtosis
    w = I.normal_tensor(0, I.STREAM_W1, (256, 1024), 0.02, torch.bfloat16)
    assert w.dtype == torch.bfloat16 and abs(float(w.float().std()) - 0.02) < 5e-4
    m = I.mlp_inputs(16, 8, 32, torch.bfloat16, seed=3)
    f64 = m.as_f64()
    assert f64["W1"].shape == (8, 32) and f64["W2"].shape == (32, 8) and f64["X"].dtype == np.float64
    # stored values survive the widening exactly
    assert torch.equal(torch.from_numpy(f64["X"]).to(torch.bfloat16), m.X)
