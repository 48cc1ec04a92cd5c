"""Parity of the split Linear operator (attention projections) through the C ABI against
oracle/linear_oracle.py.  GPU only.  Bar: max|gpu - ref| <= tol * max|ref| per output tensor, tol = 2e-2 (bf16) / 1e-4
(fp32), as for the MLP."""
import numpy as np
import pytest
import torch

from oracle import linear_oracle as L
from paper_2305_09940_b200 import inputs as I

pytestmark = pytest.mark.gpu
TOL = {torch.bfloat16: 2e-2, torch.float32: 1e-4}


def rel_err(got, ref):
    scale = float(np.max(np.abs(ref)))
    return float(np.max(np.abs(got - ref))) / (scale if scale > 0 else 1.0)


def run_gpu(lib, inp, dtype, k, axis, has_bias=True):
    T, n_in = inp.X.shape
    n_out = inp.W.shape[1]
    d = inp.to("cuda")
    op = lib.SplitLinear(T, n_in, n_out, dtype, k, axis=axis, has_bias=has_bias)
    Y = op.forward(d.X, d.W, d.b if has_bias else None)
    g = op.backward(d.X, d.W, d.dY)
    torch.cuda.synchronize()
    out = {"Y": Y, "dX": g["dX"], "dW": g["dW"]}
    if has_bias:
        out["db"] = g["db"]
    return {n: t.to(torch.float64).cpu().numpy() for n, t in out.items()}


def check(got, ref, tol, what):
    errs = {n: rel_err(got[n], ref[n]) for n in got}
    bad = {n: e for n, e in errs.items() if not (e <= tol)}
    assert not bad, f"{what}: rel err over {tol}: {bad} (all {errs})"


# attention-projection shapes of a minGPT layer: QKV hidden -> 3 hidden, output projection hidden -> hidden
@pytest.mark.parametrize("axis", ["contraction", "tokens"])
@pytest.mark.parametrize("T,h,mult,k", [(1024, 512, 3, 1), (1024, 512, 3, 4), (2048, 256, 1, 2), (777, 264, 3, 3),
                                        (300, 136, 1, 5), (64, 8, 3, 1)])
def test_bf16_attention_projection_shapes_match_oracle(lib, axis, T, h, mult, k):
    if axis == "contraction" and k > h // 8:
        k = h // 8
    inp = I.linear_inputs(T, h, mult * h, torch.bfloat16, seed=11)
    x = inp.as_f64()
    ref = L.linear_forward_backward(x["X"], x["W"], x["b"], x["dY"])
    check(run_gpu(lib, inp, torch.bfloat16, k, axis), ref, 2e-2, f"linear bf16 {T}x{h}x{mult * h} k={k} {axis}")


@pytest.mark.parametrize("axis", ["contraction", "tokens"])
def test_fp32_matches_oracle_and_is_split_invariant(lib, axis):
    inp = I.linear_inputs(200, 64, 192, torch.float32, seed=12)
    x = inp.as_f64()
    ref = L.linear_forward_backward(x["X"], x["W"], x["b"], x["dY"])
    outs = {k: run_gpu(lib, inp, torch.float32, k, axis) for k in (1, 2, 4, 7)}
    for k, got in outs.items():
        check(got, ref, 1e-4, f"linear fp32 k={k} {axis}")
        for n in got:
            assert rel_err(got[n], outs[1][n]) <= 1e-5, (k, n)


def test_no_bias_variant_and_null_workspace(lib):
    inp = I.linear_inputs(512, 128, 384, torch.bfloat16, seed=13)
    x = inp.as_f64()
    ref = L.linear_forward_backward(x["X"], x["W"], None, x["dY"])
    for axis in ("contraction", "tokens"):
        got = run_gpu(lib, inp, torch.bfloat16, 2, axis, has_bias=False)
        assert "db" not in got
        check(got, {n: ref[n] for n in got}, 2e-2, f"no-bias {axis}")
    desc = lib.make_linear_desc(512, 128, 384, torch.bfloat16, 1, lib.OSDP_SPLIT_TOKENS, has_bias=False)
    assert lib.osdp_split_linear_workspace_bytes(desc, lib.OSDP_FWD) == 0
    assert lib.osdp_split_linear_workspace_bytes(desc, lib.OSDP_BWD) == 0
    d = inp.to("cuda")
    Y = torch.empty(512, 384, dtype=torch.bfloat16, device="cuda")
    lib.osdp_split_linear_forward(desc, d.X, d.W, None, Y, None)          # no workspace needed, none given
    torch.cuda.synchronize()
    assert rel_err(Y.double().cpu().numpy(), ref["Y"]) <= 2e-2


def test_contraction_split_results_that_belong_to_one_slice_do_not_depend_on_k(lib):
    """dX columns and dW rows are written by exactly one slice: bit-identical for every k; Y differs only by fp32
    re-association of the slice sums."""
    inp = I.linear_inputs(640, 256, 768, torch.bfloat16, seed=14)
    outs = {k: run_gpu(lib, inp, torch.bfloat16, k, "contraction") for k in (1, 2, 4, 32)}
    for k in (2, 4, 32):
        assert np.array_equal(outs[k]["dX"], outs[1]["dX"]) and np.array_equal(outs[k]["dW"], outs[1]["dW"])
        assert np.array_equal(outs[k]["db"], outs[1]["db"])
        assert rel_err(outs[k]["Y"], outs[1]["Y"]) <= 1e-2


def test_token_split_rows_do_not_depend_on_k_and_runs_are_reproducible(lib):
    inp = I.linear_inputs(640, 256, 768, torch.bfloat16, seed=15)
    outs = {k: run_gpu(lib, inp, torch.bfloat16, k, "tokens") for k in (1, 2, 5)}
    for k in (2, 5):
        assert np.array_equal(outs[k]["Y"], outs[1]["Y"]) and np.array_equal(outs[k]["dX"], outs[1]["dX"])
    again = run_gpu(lib, inp, torch.bfloat16, 5, "tokens")
    for n in again:
        assert np.array_equal(again[n], outs[5][n]), n


def test_linear_error_codes(lib):
    T, i, o = 64, 64, 128
    inp = I.linear_inputs(T, i, o, torch.bfloat16, seed=1).to("cuda")
    Y = torch.empty(T, o, dtype=torch.bfloat16, device="cuda")
    ws = torch.empty(1 << 20, dtype=torch.uint8, device="cuda")
    mk = lambda **kw: lib.make_linear_desc(kw.get("T", T), kw.get("i", i), kw.get("o", o), kw.get("dt", torch.bfloat16),
                                           kw.get("k", 2), kw.get("axis", lib.OSDP_SPLIT_CONTRACTION), kw.get("bias", True))
    f = lib.osdp_split_linear_forward
    assert f(mk(), inp.X, inp.W, inp.b, Y, ws, check=False) == lib.OSDP_OK
    assert f(mk(k=0), inp.X, inp.W, inp.b, Y, ws, check=False) == lib.OSDP_ERR_K
    assert f(mk(k=9), inp.X, inp.W, inp.b, Y, ws, check=False) == lib.OSDP_ERR_K            # > in / 8 units
    assert f(mk(k=65, axis=lib.OSDP_SPLIT_TOKENS), inp.X, inp.W, inp.b, Y, ws, check=False) == lib.OSDP_ERR_K
    assert f(mk(axis=7), inp.X, inp.W, inp.b, Y, ws, check=False) == lib.OSDP_ERR_ARG
    assert f(mk(dt=5), inp.X, inp.W, inp.b, Y, ws, check=False) == lib.OSDP_ERR_DTYPE
    assert f(mk(), inp.X, inp.W, None, Y, ws, check=False) == lib.OSDP_ERR_NULL             # has_bias but no b
    assert f(mk(), inp.X, inp.W, inp.b, Y, ws, workspace_bytes=64, check=False) == lib.OSDP_ERR_WORKSPACE
    assert f(mk(), inp.X, inp.W, inp.b, Y, None, check=False) == lib.OSDP_ERR_WORKSPACE     # k = 2 needs the accumulator
    assert f(mk(), inp.X.data_ptr() + 2, inp.W, inp.b, Y, ws, check=False) == lib.OSDP_ERR_ALIGN
    assert f(mk(), inp.X.float(), inp.W, inp.b, Y, ws, check=False) == lib.OSDP_ERR_DTYPE   # binding: dtype mismatch
    assert f(mk(i=i + 8), inp.X, inp.W, inp.b, Y, ws, check=False) == lib.OSDP_ERR_SHAPE    # binding: element count
    assert lib.osdp_split_linear_workspace_bytes(mk(i=12), lib.OSDP_FWD, check=False) == -lib.OSDP_ERR_SHAPE
