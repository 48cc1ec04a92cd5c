"""Parity of the CUDA path (through the C ABI) against the fp64 oracle.  GPU only (-m gpu).

Bar (BASELINE.json north_star): per output tensor, max|gpu - ref| <= tol * max|ref| with tol = 2e-2 for bf16
storage / fp32 accumulation and 1e-4 for the fp32 config; split-invariance across k <= 1e-5 relative (fp32).
"""
import numpy as np
import pytest
import torch

from oracle import mlp_oracle as O
from paper_2305_09940_b200 import inputs as I

pytestmark = pytest.mark.gpu

TOL = {torch.bfloat16: 2e-2, torch.float32: 1e-4}
NAMES = ("Y", "dX", "dW1", "db1", "dW2", "db2")


def run_gpu(lib, inp, k, dtype):
    """One forward + backward through the C ABI; returns dict of CPU fp64 numpy outputs."""
    T, h = inp.X.shape
    f = inp.W1.shape[1]
    d = inp.to("cuda")
    op = lib.SplitMlp(T, h, f, dtype, k)
    Y = op.forward(d.X, d.W1, d.b1, d.W2, d.b2)
    g = op.backward(d.X, d.W1, d.b1, d.W2, d.dY)
    torch.cuda.synchronize()
    out = {"Y": Y}
    out.update(g)
    return {n: out[n].to(torch.float64).cpu().numpy() for n in NAMES}


def rel_err(got, ref):
    scale = float(np.max(np.abs(ref)))
    return float(np.max(np.abs(got - ref))) / (scale if scale > 0 else 1.0)


def check(got, ref, tol, what=""):
    errs = {n: rel_err(got[n], ref[n]) for n in NAMES}
    bad = {n: e for n, e in errs.items() if not (e <= tol)}
    assert not bad, f"{what}: rel err over tol {tol}: {bad} (all: {errs})"
    return errs


# ------------------------------------------------------------------ C1: fp32 config, full oracle
def test_c1_fp32_k4_matches_oracle_and_is_split_invariant(lib):
    c = I.CONFIGS["C1"]
    inp = I.mlp_inputs(c["tokens"], c["hidden"], c["ffn"], torch.float32, seed=c["seed"])
    ref = O.mlp_forward_backward(**inp.as_f64())
    outs = {k: run_gpu(lib, inp, k, torch.float32) for k in (1, 2, 4, 8, 3)}
    for k, got in outs.items():
        check(got, ref, 1e-4, f"C1 k={k}")
    for k, got in outs.items():
        for n in NAMES:
            assert rel_err(got[n], outs[1][n]) <= 1e-5, (k, n)
    for k in (2, 4, 8):                      # same per-row arithmetic for every k
        assert np.array_equal(outs[k]["Y"], outs[1]["Y"]) and np.array_equal(outs[k]["dX"], outs[1]["dX"])


# ------------------------------------------------------------------ small bf16 cases: several tiles + ragged tails
@pytest.mark.parametrize("T,h,f,k", [
    (256, 256, 512, 1),       # exact tiles
    (384, 128, 512, 2),
    (333, 136, 520, 3),       # ragged everywhere: T % k != 0, h, f not multiples of 64/128/256
    (130, 72, 264, 1),
    (1000, 320, 1032, 4),
    (64, 8, 8, 4),            # minimum hidden/ffn
    (5, 64, 128, 5),          # one token per slice (k = T)
    (1, 16, 24, 1),           # a single token
])
def test_bf16_small_shapes_match_oracle(lib, T, h, f, k):
    inp = I.mlp_inputs(T, h, f, torch.bfloat16, seed=7)
    ref = O.mlp_forward_backward(**inp.as_f64())
    check(run_gpu(lib, inp, k, torch.bfloat16), ref, 2e-2, f"bf16 {T}x{h}x{f} k={k}")


@pytest.mark.parametrize("T,h,f,k", [(333, 136, 520, 3), (64, 8, 12, 4), (7, 4, 4, 7)])
def test_fp32_small_shapes_match_oracle(lib, T, h, f, k):
    inp = I.mlp_inputs(T, h, f, torch.float32, seed=8)
    ref = O.mlp_forward_backward(**inp.as_f64())
    check(run_gpu(lib, inp, k, torch.float32), ref, 1e-4, f"f32 {T}x{h}x{f} k={k}")


def test_bf16_large_weights_stress_gelu_range(lib):
    """W std 0.2 instead of 0.02 pushes |Z| to ~10: both GeLU tails and the steep middle are exercised."""
    inp = I.mlp_inputs(512, 256, 1024, torch.bfloat16, seed=11, w_std=0.2)
    ref = O.mlp_forward_backward(**inp.as_f64())
    check(run_gpu(lib, inp, 2, torch.bfloat16), ref, 2e-2, "bf16 wide")


# ------------------------------------------------------------------ every tile shape of the bf16 GEMM on small shapes
@pytest.fixture
def force_big_tiles(lib):
    """512 x 256 pair tiles (MT = 2) for every launch, whatever K and the tile count: the default build takes them
    only for long-K GEMMs that fill the machine (full-size tests), so the ragged small shapes would never see them."""
    keys = (lib.OSDP_TUNE_MT2_MIN_K, lib.OSDP_TUNE_MT2_MIN_TILES, lib.OSDP_TUNE_WAVE_SYNC, lib.OSDP_TUNE_BAND_MIB,
            lib.OSDP_TUNE_CLUSTER_MIN_TILES, lib.OSDP_TUNE_SLICE_KERNEL_MAX_TILES)
    old = {k: lib.osdp_get_tuning(k) for k in keys}
    lib.osdp_set_tuning(lib.OSDP_TUNE_MT2_MIN_K, 1)
    lib.osdp_set_tuning(lib.OSDP_TUNE_MT2_MIN_TILES, 1)
    lib.osdp_set_tuning(lib.OSDP_TUNE_SLICE_KERNEL_MAX_TILES, 0)   # small slices would take the one-kernel-per-slice path
    yield
    for k, v in old.items():
        lib.osdp_set_tuning(k, v)


@pytest.mark.parametrize("T,h,f,k", [
    (512, 256, 512, 1),       # exact 512 x 256 tiles
    (333, 136, 520, 3),       # ragged everywhere
    (1000, 320, 1032, 2),     # partial second M-half, partial last tile
    (130, 72, 264, 1),        # less than one M-half
    (5, 64, 128, 5),
])
def test_bf16_big_tiles_match_oracle(lib, force_big_tiles, T, h, f, k):
    inp = I.mlp_inputs(T, h, f, torch.bfloat16, seed=9)
    ref = O.mlp_forward_backward(**inp.as_f64())
    check(run_gpu(lib, inp, k, torch.bfloat16), ref, 2e-2, f"bf16 MT=2 {T}x{h}x{f} k={k}")


@pytest.mark.parametrize("T,h,f,k", [(333, 136, 520, 3), (1000, 320, 1032, 2), (130, 72, 264, 1), (512, 256, 768, 1)])
@pytest.mark.parametrize("big", [False, True])
def test_bf16_multicast_clusters_match_oracle(lib, force_big_tiles, T, h, f, k, big):
    """4-CTA clusters (two CTA pairs sharing their A rows through TMA multicast) on ragged shapes, including odd
    tile counts where one pair of a cluster has no tile of its own."""
    lib.osdp_set_tuning(lib.OSDP_TUNE_CLUSTER_MIN_TILES, 1)
    if not big:
        lib.osdp_set_tuning(lib.OSDP_TUNE_MT2_MIN_K, 1 << 40)
    inp = I.mlp_inputs(T, h, f, torch.bfloat16, seed=16)
    ref = O.mlp_forward_backward(**inp.as_f64())
    check(run_gpu(lib, inp, k, torch.bfloat16), ref, 2e-2, f"bf16 clusters MT={2 if big else 1} {T}x{h}x{f} k={k}")


def test_bf16_tile_shapes_and_wave_sync_agree_bitwise(lib, force_big_tiles):
    """One owner CTA per output element and ascending-k accumulation in every configuration: tile shape, raster
    band and wave sync change the schedule, not a single bit of the result.  Shape: more 512 x 256 tiles than CTA
    pairs in the big GEMMs (several waves, so the wave sync really waits), ragged edges."""
    T, h, f = 5200, 1288, 5144
    inp = I.mlp_inputs(T, h, f, torch.bfloat16, seed=10)
    outs = []
    for min_k, sync, band, cluster in ((1, 1, 0, 0), (1, 0, 32, 0), (1, 4, 32, 0), (1, 1, 1, 0), (1 << 40, 1, 0, 0),
                                       (1, 1, 32, 1), (1 << 40, 1, 32, 1)):        # last two: 4-CTA multicast clusters
        # band 0 = the default square-wave raster, > 0 = round 1's L2-budget bands
        lib.osdp_set_tuning(lib.OSDP_TUNE_MT2_MIN_K, min_k)
        lib.osdp_set_tuning(lib.OSDP_TUNE_WAVE_SYNC, sync)
        lib.osdp_set_tuning(lib.OSDP_TUNE_BAND_MIB, band)
        lib.osdp_set_tuning(lib.OSDP_TUNE_CLUSTER_MIN_TILES, cluster)
        outs.append(run_gpu(lib, inp, 2, torch.bfloat16))
    for o in outs[1:]:
        for n in NAMES:
            assert np.array_equal(o[n], outs[0][n]), n
    check(outs[0], O.mlp_forward_backward(**inp.as_f64()), 2e-2, "bf16 MT=2 several waves")


def test_two_streams_with_wave_sync_do_not_deadlock(lib, force_big_tiles):
    """Two multi-wave MT = 2 launches in flight on different streams can each hold SMs the other one's missing CTAs
    need; the wave sync must give up instead of waiting for ever, and the results must not change."""
    T, h, f = 5200, 1288, 5144
    inps = [I.mlp_inputs(T, h, f, torch.bfloat16, seed=s) for s in (20, 21)]
    want = [run_gpu(lib, inp, 1, torch.bfloat16) for inp in inps]
    devs = [inp.to("cuda") for inp in inps]
    ops = [lib.SplitMlp(T, h, f, torch.bfloat16, 1) for _ in inps]
    streams = [torch.cuda.Stream() for _ in inps]
    torch.cuda.synchronize()
    outs = [None, None]
    for _ in range(3):
        for i, (d, op, st) in enumerate(zip(devs, ops, streams)):
            with torch.cuda.stream(st):
                Y = op.forward(d.X, d.W1, d.b1, d.W2, d.b2, stream=st)
                g = op.backward(d.X, d.W1, d.b1, d.W2, d.dY, stream=st)
            outs[i] = dict(Y=Y, **g)
    torch.cuda.synchronize()
    for o, w in zip(outs, want):
        for n in NAMES:
            assert np.array_equal(o[n].double().cpu().numpy(), w[n]), n


def test_forward_backward_can_be_captured_in_a_cuda_graph(lib):
    """The library only enqueues on the caller's stream (no allocation, no synchronisation), so after one warm-up call
    (which caches function attributes and the driver entry point) a whole step can be stream-captured and replayed;
    launch-bound small operators gain from that."""
    T, h, f, k = 1000, 320, 1032, 4
    inp = I.mlp_inputs(T, h, f, torch.bfloat16, seed=15)
    want = {ax: (run_gpu if ax == "tokens" else run_gpu_ffn)(lib, inp, k, torch.bfloat16) for ax in ("tokens", "ffn")}
    d = inp.to("cuda")
    for axis in ("tokens", "ffn"):
        op = lib.SplitMlp(T, h, f, torch.bfloat16, k, axis=axis)
        Y = torch.empty_like(d.X)
        g = dict(dX=torch.empty_like(d.X), dW1=torch.empty(h, f, device="cuda"), db1=torch.empty(f, device="cuda"),
                 dW2=torch.empty(f, h, device="cuda"), db2=torch.empty(h, device="cuda"))
        s = torch.cuda.Stream()
        s.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(s):
            op.forward(d.X, d.W1, d.b1, d.W2, d.b2, Y=Y, stream=s)                 # warm-up outside the capture
            op.backward(d.X, d.W1, d.b1, d.W2, d.dY, out=g, stream=s)
            s.synchronize()
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph, stream=s):
                op.forward(d.X, d.W1, d.b1, d.W2, d.b2, Y=Y, stream=s)
                op.backward(d.X, d.W1, d.b1, d.W2, d.dY, out=g, stream=s)
        for t in (Y, *g.values()):
            t.fill_(7.0)
        graph.replay()
        graph.replay()
        torch.cuda.synchronize()
        got = dict(Y=Y, **g)
        for n in NAMES:
            assert np.array_equal(got[n].double().cpu().numpy(), want[axis][n]), (axis, n)


@pytest.fixture
def per_gemm_launches(lib):
    """The launch-per-GEMM path for small slices too (by default they run as one kernel per slice,
    tests/test_gpu_slice_kernel.py)."""
    old = lib.osdp_get_tuning(lib.OSDP_TUNE_SLICE_KERNEL_MAX_TILES)
    lib.osdp_set_tuning(lib.OSDP_TUNE_SLICE_KERNEL_MAX_TILES, 0)
    yield
    lib.osdp_set_tuning(lib.OSDP_TUNE_SLICE_KERNEL_MAX_TILES, old)


def test_trace_records_every_launch_with_its_step(lib, per_gemm_launches):
    """osdp_trace_*: one (step id, milliseconds) entry per kernel launch, in launch order, both split axes."""
    T, h, f, k = 600, 128, 512, 3
    d = I.mlp_inputs(T, h, f, torch.bfloat16, seed=17).to("cuda")
    # step 8 = column sums: db2 takes two launches once per call (partials of dY, fixed-order sum); db1 one per slice
    # (the band partials come out of the A4 epilogue, only their fixed-order sum is a launch)
    for axis, fwd_steps, bwd_steps in (("tokens", [1, 2] * k, [8, 8] + [3, 4, 5, 8, 6, 7] * k),
                                       ("ffn", [1, 2] * k + [10], [3, 4, 5, 8, 8, 8, 6, 7] + [3, 4, 5, 8, 6, 7] * (k - 1) + [10])):
        op = lib.SplitMlp(T, h, f, torch.bfloat16, k, axis=axis)
        op.forward(d.X, d.W1, d.b1, d.W2, d.b2)                      # warm-up, untraced
        lib.osdp_trace_enable(True)
        op.forward(d.X, d.W1, d.b1, d.W2, d.b2)
        n_fwd = lib.osdp_last_launch_count()
        op.backward(d.X, d.W1, d.b1, d.W2, d.dY)
        n_bwd = lib.osdp_last_launch_count()
        tr = lib.osdp_trace_read()
        lib.osdp_trace_enable(False)
        assert [s for s, _ in tr] == fwd_steps + bwd_steps and (n_fwd, n_bwd) == (len(fwd_steps), len(bwd_steps)), axis
        assert all(0.0 < ms < 50.0 for _, ms in tr)
        assert lib.osdp_trace_read() == []                           # reading clears the trace
    assert "GEMM1" in lib.osdp_step_name(1) and "column sums" in lib.osdp_step_name(8)
    assert "accumulator" in lib.osdp_step_name(10) and lib.osdp_step_name(99) == "unknown"


def test_tuning_rejects_bad_arguments(lib):
    assert lib.osdp_set_tuning(99, 1, check=False) == lib.OSDP_ERR_ARG
    assert lib.osdp_set_tuning(lib.OSDP_TUNE_WAVE_SYNC, -1, check=False) == lib.OSDP_ERR_ARG
    assert lib.osdp_set_tuning(lib.OSDP_TUNE_MT2_MIN_K, 0, check=False) == lib.OSDP_ERR_ARG
    assert lib.osdp_set_tuning(lib.OSDP_TUNE_BAND_MIB, -1, check=False) == lib.OSDP_ERR_ARG
    assert lib.osdp_get_tuning(99) == -1
    assert lib.osdp_get_tuning(lib.OSDP_TUNE_MT2_MIN_K) == 4096 and lib.osdp_get_tuning(lib.OSDP_TUNE_WAVE_SYNC) == 1


# ------------------------------------------------------------------ ffn-axis (paper-literal) split
def run_gpu_ffn(lib, inp, k, dtype):
    T, h = inp.X.shape
    f = inp.W1.shape[1]
    d = inp.to("cuda")
    op = lib.SplitMlp(T, h, f, dtype, k, axis="ffn")
    Y = op.forward(d.X, d.W1, d.b1, d.W2, d.b2)
    g = op.backward(d.X, d.W1, d.b1, d.W2, d.dY)
    torch.cuda.synchronize()
    out = {"Y": Y}
    out.update(g)
    return {n: out[n].to(torch.float64).cpu().numpy() for n in NAMES}


@pytest.mark.parametrize("T,h,f,k", [
    (256, 256, 512, 1),
    (256, 256, 512, 2),
    (333, 136, 520, 3),       # ragged everywhere; 65 column units over 3 slices (176, 168, 176 columns)
    (1000, 320, 1032, 4),
    (130, 72, 264, 33),       # one 8-column unit per slice (k = ffn / 8)
    (64, 8, 8, 1),
    (1, 16, 24, 3),
])
def test_bf16_ffn_split_matches_oracle(lib, T, h, f, k):
    inp = I.mlp_inputs(T, h, f, torch.bfloat16, seed=13)
    ref = O.mlp_forward_backward(**inp.as_f64())
    check(run_gpu_ffn(lib, inp, k, torch.bfloat16), ref, 2e-2, f"bf16 ffn split {T}x{h}x{f} k={k}")


def test_bf16_ffn_split_big_tiles_match_oracle(lib, force_big_tiles):
    inp = I.mlp_inputs(1000, 320, 1032, torch.bfloat16, seed=14)
    ref = O.mlp_forward_backward(**inp.as_f64())
    check(run_gpu_ffn(lib, inp, 3, torch.bfloat16), ref, 2e-2, "bf16 ffn split MT=2")


def test_fp32_ffn_split_matches_oracle_and_is_split_invariant(lib):
    c = I.CONFIGS["C1"]
    inp = I.mlp_inputs(c["tokens"], c["hidden"], c["ffn"], torch.float32, seed=c["seed"])
    ref = O.mlp_forward_backward(**inp.as_f64())
    outs = {k: run_gpu_ffn(lib, inp, k, torch.float32) for k in (1, 2, 4, 3, 256)}
    for k, got in outs.items():
        check(got, ref, 1e-4, f"C1 ffn split k={k}")
        for n in NAMES:
            assert rel_err(got[n], outs[1][n]) <= 1e-5, (k, n)
        for n in ("dW1", "db1", "dW2", "db2"):          # slices own disjoint parts of the weight gradients
            assert np.array_equal(got[n], outs[1][n]), (k, n)


def test_c2_ffn_split_matches_oracle_and_weight_grads_are_bit_identical_across_k(lib, c2):
    inp, ref = c2
    outs = {k: run_gpu_ffn(lib, inp, k, torch.bfloat16) for k in (1, 2, 4, 8)}
    for k, got in outs.items():
        check(got, ref, 2e-2, f"C2 ffn split k={k}")
        for n in ("dW1", "db1", "dW2", "db2"):
            assert np.array_equal(got[n], outs[1][n]), (k, n)
    again = run_gpu_ffn(lib, inp, 8, torch.bfloat16)
    for n in NAMES:
        assert np.array_equal(again[n], outs[8][n]), n      # deterministic run to run


def test_ffn_split_error_codes_and_workspace(lib):
    T, h, f = 64, 64, 128
    inp = I.mlp_inputs(T, h, f, torch.bfloat16, seed=1).to("cuda")
    desc = lib.make_desc(T, h, f, torch.bfloat16, 4)
    fwd, bwd = (lib.osdp_ffn_split_mlp_workspace_bytes(desc, p) for p in (lib.OSDP_FWD, lib.OSDP_BWD))
    # bwd: two slice buffers, the fp32 dX accumulator, db1 band partials (T / 32 rows x 32 columns) and db2 partials (32 x h)
    # (+ at most 128 KiB of tile counter / flag words of the one-kernel-per-slice path and their 256 B padding)
    assert 0 <= fwd - (T * 32 * 2 + T * h * 4) <= 129 << 10
    assert 0 <= bwd - (2 * T * 32 * 2 + T * h * 4 + (T // 32) * 32 * 4 + 32 * h * 4) <= 129 << 10
    assert 0 <= lib.osdp_ffn_split_mlp_workspace_bytes(lib.make_desc(T, h, f, torch.bfloat16, 1), lib.OSDP_FWD) - T * f * 2 <= 129 << 10
    assert lib.osdp_ffn_split_mlp_workspace_bytes(lib.make_desc(T, h, f, torch.bfloat16, f // 8 + 1), lib.OSDP_FWD) == 0
    ws = torch.empty(bwd, dtype=torch.uint8, device="cuda")
    Y = torch.full_like(inp.X, 3.0)
    args = (inp.X, inp.W1, inp.b1, inp.W2, inp.b2, Y, ws)
    assert lib.osdp_ffn_split_mlp_forward(desc, *args, check=False) == lib.OSDP_OK
    assert lib.osdp_ffn_split_mlp_forward(lib.make_desc(T, h, f, torch.bfloat16, T + 1), *args, check=False) == lib.OSDP_ERR_K
    assert lib.osdp_ffn_split_mlp_forward(lib.make_desc(T, h, f, torch.bfloat16, 16), *args, check=False) == lib.OSDP_OK
    assert lib.osdp_ffn_split_mlp_forward(lib.make_desc(T, h, f, torch.bfloat16, 0), *args, check=False) == lib.OSDP_ERR_K
    assert lib.osdp_ffn_split_mlp_forward(desc, None, *args[1:], check=False) == lib.OSDP_ERR_NULL
    assert lib.osdp_ffn_split_mlp_forward(desc, *args[:6], ws, workspace_bytes=64, check=False) == lib.OSDP_ERR_WORKSPACE
    assert lib.osdp_last_launch_count() == 0


# ------------------------------------------------------------------ C2: full oracle at every k
@pytest.fixture(scope="module")
def c2():
    c = I.CONFIGS["C2"]
    inp = I.mlp_inputs(c["tokens"], c["hidden"], c["ffn"], torch.bfloat16, seed=c["seed"])
    return inp, O.mlp_forward_backward(**inp.as_f64())


@pytest.mark.parametrize("k", [1, 2, 4, 8])
def test_c2_bf16_matches_oracle(lib, c2, k):
    inp, ref = c2
    check(run_gpu(lib, inp, k, torch.bfloat16), ref, 2e-2, f"C2 k={k}")


def test_c2_rows_are_bit_identical_across_k_and_runs(lib, c2):
    inp, _ = c2
    a, b, c = run_gpu(lib, inp, 1, torch.bfloat16), run_gpu(lib, inp, 8, torch.bfloat16), run_gpu(lib, inp, 8, torch.bfloat16)
    assert np.array_equal(a["Y"], b["Y"]) and np.array_equal(a["dX"], b["dX"])      # reading S12
    for n in NAMES:
        assert np.array_equal(b[n], c[n]), n                                          # deterministic run to run


# ------------------------------------------------------------------ errors and edge cases of the boundary
def test_error_codes(lib):
    T, h, f = 64, 64, 128
    inp = I.mlp_inputs(T, h, f, torch.bfloat16, seed=1).to("cuda")
    desc = lib.make_desc(T, h, f, torch.bfloat16, 2)
    ws = torch.empty(lib.osdp_split_mlp_workspace_bytes(desc, lib.OSDP_BWD), dtype=torch.uint8, device="cuda")
    Y = torch.full_like(inp.X, 3.0)
    args = (inp.X, inp.W1, inp.b1, inp.W2, inp.b2, Y, ws)
    assert lib.osdp_split_mlp_forward(desc, *args, check=False) == lib.OSDP_OK
    assert lib.osdp_split_mlp_forward(desc, None, *args[1:], check=False) == lib.OSDP_ERR_NULL
    assert lib.osdp_split_mlp_forward(lib.make_desc(T, h, f, torch.bfloat16, 0), *args, check=False) == lib.OSDP_ERR_K
    assert lib.osdp_split_mlp_forward(lib.make_desc(T, h, f, torch.bfloat16, T + 1), *args, check=False) == lib.OSDP_ERR_K
    assert lib.osdp_split_mlp_forward(lib.make_desc(T, h + 4, f, torch.bfloat16, 1), *args, check=False) == lib.OSDP_ERR_SHAPE
    assert lib.osdp_split_mlp_forward(lib.make_desc(T, h, f, 5, 1), *args, check=False) == lib.OSDP_ERR_DTYPE
    Y.fill_(3.0)
    torch.cuda.synchronize()
    assert lib.osdp_split_mlp_forward(desc, *args[:6], ws, workspace_bytes=16, check=False) == lib.OSDP_ERR_WORKSPACE
    assert lib.osdp_split_mlp_forward(desc, *args[:6], ws.data_ptr() + 16, workspace_bytes=ws.numel() - 16,
                                      check=False) == lib.OSDP_ERR_WORKSPACE
    assert lib.osdp_split_mlp_forward(desc, inp.X.data_ptr() + 2, *args[1:], check=False) == lib.OSDP_ERR_ALIGN
    torch.cuda.synchronize()
    assert bool((Y == 3.0).all())                      # outputs untouched on error
    with pytest.raises(lib.OsdpError):
        lib.osdp_split_mlp_backward(desc, inp.X, inp.W1, inp.b1, inp.W2, None, None, Y, None, None, None, None, ws)
    assert lib.osdp_last_launch_count() == 0


def test_backward_overwrites_and_accepts_null_b2(lib, per_gemm_launches):
    """Reading S11 (overwrite, not accumulate) and S4 (b2 unused)."""
    T, h, f = 200, 64, 256
    inp = I.mlp_inputs(T, h, f, torch.bfloat16, seed=2)
    ref = O.mlp_forward_backward(**inp.as_f64())
    d = inp.to("cuda")
    op = lib.SplitMlp(T, h, f, torch.bfloat16, 3)
    out = dict(dX=torch.full_like(d.X, 9.0), dW1=torch.full((h, f), 9.0, device="cuda"),
               db1=torch.full((f,), 9.0, device="cuda"), dW2=torch.full((f, h), 9.0, device="cuda"),
               db2=torch.full((h,), 9.0, device="cuda"))
    op.backward(d.X, d.W1, d.b1, d.W2, d.dY, out=out)
    op.backward(d.X, d.W1, d.b1, d.W2, d.dY, out=out)      # second call must not accumulate into the first
    torch.cuda.synchronize()
    for n in ("dX", "dW1", "db1", "dW2", "db2"):
        assert rel_err(out[n].double().cpu().numpy(), ref[n]) <= 2e-2, n
    assert lib.osdp_last_launch_count() == 2 + 3 * 6      # db2 (2 launches per call) + k slices x (5 GEMMs + the db1 sum)


def test_runs_on_a_side_stream(lib):
    T, h, f = 256, 128, 512
    inp = I.mlp_inputs(T, h, f, torch.bfloat16, seed=4)
    ref = O.mlp_forward_backward(**inp.as_f64())
    d = inp.to("cuda")
    op = lib.SplitMlp(T, h, f, torch.bfloat16, 2)
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        Y = op.forward(d.X, d.W1, d.b1, d.W2, d.b2, stream=s)
    s.synchronize()
    assert rel_err(Y.double().cpu().numpy(), ref["Y"]) <= 2e-2


@pytest.mark.parametrize("dtype,T,h,f,k", [(torch.bfloat16, 333, 136, 520, 3), (torch.bfloat16, 260, 72, 264, 2),
                                           (torch.float32, 100, 36, 68, 4)])
def test_no_out_of_bounds_writes_guard_bands(lib, dtype, T, h, f, k):
    """compute-sanitizer is closed on this pool, so out-of-bounds stores are caught with guard bands: every
    output and the workspace sit between 4 KiB bands of 0xA5 that must come back untouched (ragged shapes, so
    partial tiles clip on every edge)."""
    G = 4096
    e = 2 if dtype == torch.bfloat16 else 4
    desc = lib.make_desc(T, h, f, dtype, k)
    sizes = {"Y": T * h * e, "dX": T * h * e, "dW1": h * f * 4, "db1": f * 4, "dW2": f * h * 4, "db2": h * 4,
             "ws": lib.osdp_split_mlp_workspace_bytes(desc, lib.OSDP_BWD)}
    offs, total = {}, G
    for n, sz in sizes.items():
        offs[n] = total
        total += (sz + 255) // 256 * 256 + G
    arena = torch.full((total,), 0xA5, dtype=torch.uint8, device="cuda")
    view = lambda n, dt, shape: arena[offs[n]: offs[n] + sizes[n]].view(dt).view(*shape)
    inp = I.mlp_inputs(T, h, f, dtype, seed=5)
    ref = O.mlp_forward_backward(**inp.as_f64())
    d = inp.to("cuda")
    Y, dX = view("Y", dtype, (T, h)), view("dX", dtype, (T, h))
    dW1, db1 = view("dW1", torch.float32, (h, f)), view("db1", torch.float32, (f,))
    dW2, db2 = view("dW2", torch.float32, (f, h)), view("db2", torch.float32, (h,))
    ws = arena[offs["ws"]: offs["ws"] + sizes["ws"]]
    lib.osdp_split_mlp_forward(desc, d.X, d.W1, d.b1, d.W2, d.b2, Y, ws)
    lib.osdp_split_mlp_backward(desc, d.X, d.W1, d.b1, d.W2, d.b2, d.dY, dX, dW1, db1, dW2, db2, ws)
    torch.cuda.synchronize()
    mask = torch.ones(total, dtype=torch.bool, device="cuda")
    for n, sz in sizes.items():
        mask[offs[n]: offs[n] + sz] = False
    assert bool((arena[mask] == 0xA5).all()), "a kernel wrote outside its output/workspace"
    got = dict(Y=Y, dX=dX, dW1=dW1, db1=db1, dW2=dW2, db2=db2)
    tol = TOL[dtype]
    for n in NAMES:
        assert rel_err(got[n].double().cpu().numpy(), ref[n]) <= tol, n


@pytest.mark.parametrize("T,h,f,k", [
    (1100, 3840, 264, 1),     # dX: 5 x 15 = 75 tiles of 256 columns on 74 pairs -> 192-column tiles (5 x 20 = 100, two waves of 0.75)
    (1100, 3848, 264, 2),     # the same with a ragged last column tile and ragged row tiles
    (2048, 8192, 512, 4),     # the headline's dX tile grid per slice (512 rows, 8192 columns)
    (700, 2440, 136, 1),      # a width whose last 64-column chunk is 16 / 48 columns wide
])
def test_dx_tile_width_balancing_is_bitwise_neutral(lib, per_gemm_launches, T, h, f, k):
    """OSDP_TUNE_BALANCE_N: the dX GEMM may take 240 / 224 / 208 / 192-column tiles to fill its last wave; every output
    element still has one owner and ascending-k accumulation, so nothing changes but the time."""
    inp = I.mlp_inputs(T, h, f, torch.bfloat16, seed=41)
    assert lib.osdp_get_tuning(lib.OSDP_TUNE_BALANCE_N) == 1
    got = run_gpu(lib, inp, k, torch.bfloat16)
    lib.osdp_set_tuning(lib.OSDP_TUNE_BALANCE_N, 0)
    try:
        want = run_gpu(lib, inp, k, torch.bfloat16)
    finally:
        lib.osdp_set_tuning(lib.OSDP_TUNE_BALANCE_N, 1)
    for n in NAMES:
        assert np.array_equal(got[n], want[n]), n
    if T * h <= 1100 * 3848:
        check(got, O.mlp_forward_backward(**inp.as_f64()), 2e-2, f"balanced dX {T}x{h}x{f}")
