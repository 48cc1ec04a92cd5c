"""Full-size parity (BASELINE.json configs C3, C4, C5) in the launch configuration bench.py times, on sampled
outputs the oracle computes one by one (SURVEY.md §8(c) "sampled oracle"), and peak device bytes against the
cost model (north_star: within 5 %).  GPU only (-m gpu)."""
import numpy as np
import pytest
import torch

from oracle import mlp_oracle as O
from oracle import plan_oracle as P
from paper_2305_09940_b200 import inputs as I

pytestmark = pytest.mark.gpu
TOL = 2e-2


def rel(got, ref):
    s = float(np.max(np.abs(ref)))
    return float(np.max(np.abs(got - ref))) / (s if s > 0 else 1.0)


def sample_indices(T, k, f, seed=0, every_tile=False):
    rng = np.random.default_rng(seed)
    b = O.slice_bounds(T, k)
    rows = {0, T - 1, b[0][1] - 1, b[-1][0], b[k // 2][0], b[k // 2][1] - 1}       # first/last rows of slices
    rows |= set(int(r) for r in rng.integers(0, T, 6))
    cols = {0, f - 1, 255, 256} | set(int(c) for c in rng.integers(0, f, 4))         # across n-tile edges
    if every_tile:
        # one token row in every 512-row block (every m-tile of the token-major GEMMs A1-A4, A7, whichever slice and wave
        # it falls in) and one ffn column in every 256-column block (every n-tile of A1/A3/A4, every m-tile of dW2 = A5
        # and every n-tile of dW1 = A6); a sampled row covers all of Y / dX along hidden, a sampled column all of
        # dW2[j, :] and dW1[:, j], so every output tile of every GEMM of every wave has a checked element
        rows |= {min(T - 1, r0 + int(rng.integers(0, 512))) for r0 in range(0, T, 512)}
        cols |= {min(f - 1, c0 + int(rng.integers(0, 256))) for c0 in range(0, f, 256)}
    return sorted(rows), sorted(cols)


def check_sampled(lib, inp, x64, ks, what, refs=None, axis="tokens", every_tile=False):
    T, h = inp.X.shape
    f = inp.W1.shape[1]
    d = inp.to("cuda")
    cache = {}
    for k in ks:
        rows, cols = sample_indices(T, k, f, every_tile=every_tile)
        if axis == "ffn":      # first/last columns of ffn slices as well
            fb = O.ffn_slice_bounds(f, k, 8)
            cols = sorted(set(cols) | {fb[0][1] - 1, fb[-1][0], fb[k // 2][0], fb[k // 2][1] - 1})
        key = (tuple(rows), tuple(cols))
        if key not in cache:
            cache[key] = (O.sampled_rows(x64["X"], x64["W1"], x64["b1"], x64["W2"], x64["b2"], x64["dY"], rows),
                          O.sampled_cols(x64["X"], x64["W1"], x64["b1"], x64["W2"], x64["dY"], cols),
                          O.db2_full(x64["dY"]))
        r, c, db2 = cache[key]
        op = lib.SplitMlp(T, h, f, torch.bfloat16, k, axis=axis)
        Y = op.forward(d.X, d.W1, d.b1, d.W2, d.b2)
        g = op.backward(d.X, d.W1, d.b1, d.W2, d.dY)
        torch.cuda.synchronize()
        ri, ci = torch.tensor(rows, device="cuda"), torch.tensor(cols, device="cuda")
        got = {"Y": Y[ri].double().cpu().numpy(), "dX": g["dX"][ri].double().cpu().numpy(),
               "dW2": g["dW2"][ci].double().cpu().numpy(), "dW1": g["dW1"][:, ci].double().cpu().numpy(),
               "db1": g["db1"][ci].double().cpu().numpy(), "db2": g["db2"].double().cpu().numpy()}
        ref = {"Y": r["Y"], "dX": r["dX"], "dW2": c["dW2_rows"], "dW1": c["dW1_cols"], "db1": c["db1"], "db2": db2}
        errs = {n: rel(got[n], ref[n]) for n in ref}
        assert all(e <= TOL for e in errs.values()), f"{what} k={k}: {errs}"
        # properties that hold at any size: nothing non-finite anywhere in the full outputs
        for t in (Y, *g.values()):
            assert bool(torch.isfinite(t).all())
        del op, Y, g
        torch.cuda.empty_cache()


def test_c3_sampled_oracle_k_1_4_16(lib):
    c = I.CONFIGS["C3"]
    inp = I.mlp_inputs(c["tokens"], c["hidden"], c["ffn"], torch.bfloat16, seed=c["seed"])
    check_sampled(lib, inp, inp.as_f64(), c["ks"], "C3", every_tile=True)


def test_c4_sampled_oracle_bench_config_and_extremes(lib):
    c = I.CONFIGS["C4"]
    inp = I.mlp_inputs(c["tokens"], c["hidden"], c["ffn"], torch.bfloat16, seed=c["seed"])
    check_sampled(lib, inp, inp.as_f64(), (4, 1, 32), "C4", every_tile=True)          # k = 4 is what bench.py times


def test_c4_ffn_split_sampled_oracle(lib):
    """The ffn-axis (paper-literal) split at the gigantic-operator config, unsplit and at the two extremes bench.py reports."""
    c = I.CONFIGS["C4"]
    inp = I.mlp_inputs(c["tokens"], c["hidden"], c["ffn"], torch.bfloat16, seed=c["seed"])
    check_sampled(lib, inp, inp.as_f64(), (4, 32), "C4 ffn split", axis="ffn")


def test_large_token_count_offsets_beyond_2_gib(lib):
    """Maximum-size edge: tokens x ffn = 2^30 elements, so every [T x f] workspace tensor is 2 GiB and byte offsets
    inside it pass 2^31; rows at the far end and columns across tile edges are checked against the sampled oracle,
    for both split axes (unsplit and split)."""
    T, h, f = 262144, 1024, 4096
    inp = I.mlp_inputs(T, h, f, torch.bfloat16, seed=3)
    x64 = inp.as_f64()
    check_sampled(lib, inp, x64, (1, 3), "2^30-element intermediate")
    check_sampled(lib, inp, x64, (2,), "2^30-element intermediate, ffn split", axis="ffn")


@pytest.mark.parametrize("cfg,k", [("C4", 4), ("C3", 4), ("C5", 2)])
def test_token_downscaled_full_oracle(lib, cfg, k):
    """Full oracle on a token-downscaled copy (T/8) of each large config: every output element
    checked, for the token split and the ffn-axis split."""
    c = I.CONFIGS[cfg]
    T = c["tokens"] // 8
    inp = I.mlp_inputs(T, c["hidden"], c["ffn"], torch.bfloat16, seed=3)
    ref = O.mlp_forward_backward(**inp.as_f64())
    d = inp.to("cuda")
    for axis in ("tokens", "ffn"):
        op = lib.SplitMlp(T, c["hidden"], c["ffn"], torch.bfloat16, k, axis=axis)
        out = {"Y": op.forward(d.X, d.W1, d.b1, d.W2, d.b2)}
        out.update(op.backward(d.X, d.W1, d.b1, d.W2, d.dY))
        torch.cuda.synchronize()
        errs = {n: rel(out[n].double().cpu().numpy(), ref[n]) for n in ref}
        assert all(e <= TOL for e in errs.values()), (cfg, axis, errs)
        del op, out
        torch.cuda.empty_cache()


def test_c5_stack_planned_k_teacher_forced(lib):
    """24-layer chain, per-layer k from osdp_plan under the 24 GiB activation cap (pure-sum accounting at
    8 B per T x f element, SURVEY.md §8 note), forward through all layers then backward; parity per layer,
    teacher-forced on the GPU's own bf16 X_l and dY_l (reading S13), on sampled outputs of ALL 24 layers."""
    c = I.CONFIGS["C5"]
    T, h, f, L = c["tokens"], c["hidden"], c["ffn"], c["layers"]
    desc1 = lib.make_desc(T, h, f, torch.bfloat16, 1)
    # planner-only record in the paper's accounting: activations summed over layers, 8 B per T x f element
    ops = []
    for _ in range(L):
        oc = lib.osdp_mlp_op_cost(desc1, lib.OSDP_BWD)
        oc.model_bytes = (2 * h * f + f + h) * 2                     # weights only; grads/optimizer outside the cap
        oc.extra_fixed = 0
        oc.extra_transient = 0
        oc.extra_summed = 8 * T * f                                  # Z, H, dH, dZ in bf16, unfused autograd view
        oc.act_bytes = T * h * 2                                     # saved layer input
        oc.gamma = 3.0e-3
        oc.delta = 1.0e-4
        ops.append(oc)
    cap = c["act_cap_bytes"]
    dev = lib.osdp_device(1, 0.0, 0.0, cap)
    st, ks, modes, sec, peak = lib.osdp_plan(ops, dev, 1, [1, 2, 4, 8, 16, 32])
    assert st == lib.OSDP_OK and peak <= cap and set(modes) == {0}
    assert any(k > 1 for k in ks), "the 24 GiB cap must bind under pure-sum accounting"
    pops = [P.OpCost(S=o.S, model=o.model_bytes, act=o.act_bytes, extra_summed=o.extra_summed, gamma=o.gamma,
                     delta=o.delta) for o in ops]
    mem, ps = P.plan_memory_time(pops, modes, ks, 1, P.Device(N=1, mem_limit=cap))
    assert mem == peak and ps == round(sec * 1e12)

    # run the chain on the GPU with the planned k per layer
    Ws = [I.mlp_inputs(1, h, f, torch.bfloat16, seed=l) for l in range(L)]      # weights/biases of layer l (seed = l)
    X0 = I.normal_tensor(0, I.STREAM_X, (T, h), 1.0, torch.bfloat16)
    dYL = I.normal_tensor(0, I.STREAM_DY, (T, h), 1.0, torch.bfloat16)
    dev_w = [(w.W1.cuda(), w.b1.cuda(), w.W2.cuda(), w.b2.cuda()) for w in Ws]
    Xs = [X0.cuda()]
    opsl = [lib.SplitMlp(T, h, f, torch.bfloat16, ks[l]) for l in range(L)]
    for l in range(L):
        W1, b1, W2, b2 = dev_w[l]
        Xs.append(opsl[l].forward(Xs[l], W1, b1, W2, b2))
    dY = dYL.cuda()
    checked = set(range(L))
    rows, cols = sample_indices(T, 4, f, seed=5)
    ri, ci = torch.tensor(rows, device="cuda"), torch.tensor(cols, device="cuda")
    for l in reversed(range(L)):
        W1, b1, W2, b2 = dev_w[l]
        g = opsl[l].backward(Xs[l], W1, b1, W2, dY)
        torch.cuda.synchronize()
        assert all(bool(torch.isfinite(t).all()) for t in g.values())
        if l in checked:
            x64 = dict(X=Xs[l].double().cpu().numpy(), W1=W1.double().cpu().numpy(), b1=b1.double().cpu().numpy(),
                       W2=W2.double().cpu().numpy(), b2=b2.double().cpu().numpy(), dY=dY.double().cpu().numpy())
            r = O.sampled_rows(x64["X"], x64["W1"], x64["b1"], x64["W2"], x64["b2"], x64["dY"], rows)
            cc = O.sampled_cols(x64["X"], x64["W1"], x64["b1"], x64["W2"], x64["dY"], cols)
            errs = {"Y": rel(Xs[l + 1][ri].double().cpu().numpy(), r["Y"]),
                    "dX": rel(g["dX"][ri].double().cpu().numpy(), r["dX"]),
                    "dW2": rel(g["dW2"][ci].double().cpu().numpy(), cc["dW2_rows"]),
                    "dW1": rel(g["dW1"][:, ci].double().cpu().numpy(), cc["dW1_cols"]),
                    "db1": rel(g["db1"][ci].double().cpu().numpy(), cc["db1"]),
                    "db2": rel(g["db2"].double().cpu().numpy(), O.db2_full(x64["dY"]))}
            assert all(e <= TOL for e in errs.values()), f"C5 layer {l} k={ks[l]}: {errs}"
        dY = g["dX"]


@pytest.mark.parametrize("cfg,ks", [("C1", (1, 4)), ("C2", (1, 2, 4, 8)), ("C4", (1, 4, 32))])
def test_peak_bytes_within_5pct_of_cost_model(lib, cfg, ks):
    import bench
    c = I.CONFIGS[cfg]
    for k in ks:
        pk = bench.measure_peak_bytes(lib, c, k)
        for name in ("fwd", "bwd"):
            m, model = pk[name]["measured"], pk[name]["model"]
            assert abs(m - model) <= 0.05 * model, (cfg, k, name, pk)
            e = 4 if c["dtype"] == "f32" else 2
            want = P.mlp_workspace_bytes(c["tokens"], c["hidden"], c["ffn"], e, k, name == "bwd")   # PAPER.md:167 size / k
            bound = want // 32 + 32 * c["hidden"] * 4 + (192 << 10)          # DESIGN.md reading W1: the library's own scratch
            assert 0 <= pk[name]["workspace"] - want <= bound, (cfg, k, name, pk[name]["workspace"], want)


@pytest.mark.parametrize("cfg,ks", [("C4", (1, 4, 32)), ("C2", (2, 8))])
def test_ffn_split_peak_bytes_within_5pct_of_cost_model(lib, cfg, ks):
    """Peak device bytes of the ffn-axis split: caller tensors + [T x ceil(f/k)] slice buffers + the fp32 [T x h]
    accumulator (k > 1) + scratch, against osdp_ffn_split_mlp_op_cost + osdp_cost_eval."""
    import bench
    c = I.CONFIGS[cfg]
    T, h, f = c["tokens"], c["hidden"], c["ffn"]
    for k in ks:
        pk = bench.measure_peak_bytes(lib, c, k, axis="ffn")
        for name in ("fwd", "bwd"):
            m, model = pk[name]["measured"], pk[name]["model"]
            assert abs(m - model) <= 0.05 * model, (cfg, k, name, pk)
            fs = -(-(f // 8) // k) * 8
            bufs = (2 if name == "bwd" else 1) * ((T * fs * 2 + 255) // 256 * 256)
            acc = 0 if k == 1 else (T * h * 4 + 255) // 256 * 256
            # + the library's own scratch (reading W1): db1 band partials of one slice, db2 partials, sync words
            bound = bufs // 32 + 32 * h * 4 + (192 << 10)
            assert 0 <= pk[name]["workspace"] - (bufs + acc) <= bound, (cfg, k, name, pk[name]["workspace"], bufs + acc)

