"""The one-kernel-per-slice path of the token split (csrc/slice_sm100.cuh, OSDP_TUNE_SLICE_KERNEL_MAX_TILES): parity
with the fp64 oracle, bit-identity with the launch-per-GEMM path, concurrency on 2 and on 24 streams, CUDA-graph capture, two graphs replayed
side by side.
GPU only (-m gpu)."""
import numpy as np
import pytest
import torch

from oracle import mlp_oracle as O
from paper_2305_09940_b200 import inputs as I

pytestmark = pytest.mark.gpu

NAMES = ("Y", "dX", "dW1", "db1", "dW2", "db2")


def run_gpu(lib, inp, k, stream=None):
    T, h = inp.X.shape
    f = inp.W1.shape[1]
    d = inp.to("cuda")
    op = lib.SplitMlp(T, h, f, torch.bfloat16, k)
    Y = op.forward(d.X, d.W1, d.b1, d.W2, d.b2)
    g = op.backward(d.X, d.W1, d.b1, d.W2, d.dY)
    torch.cuda.synchronize()
    out = {"Y": Y}
    out.update(g)
    return {n: out[n].to(torch.float64).cpu().numpy() for n in NAMES}


def rel_err(got, ref):
    scale = float(np.max(np.abs(ref)))
    return float(np.max(np.abs(got - ref))) / (scale if scale > 0 else 1.0)


@pytest.fixture
def slice_kernel(lib):
    """Slice kernel for every eligible shape (the default threshold only takes small slices)."""
    keys = (lib.OSDP_TUNE_SLICE_KERNEL_MAX_TILES, lib.OSDP_TUNE_SLICE_KERNEL_FFN_MAX_TILES)
    old = [lib.osdp_get_tuning(k) for k in keys]
    for k in keys:
        lib.osdp_set_tuning(k, 1 << 20)
    yield
    for k, v in zip(keys, old):
        lib.osdp_set_tuning(k, v)


def per_gemm(lib, fn):
    keys = (lib.OSDP_TUNE_SLICE_KERNEL_MAX_TILES, lib.OSDP_TUNE_SLICE_KERNEL_FFN_MAX_TILES)
    old = [lib.osdp_get_tuning(k) for k in keys]
    for k in keys:
        lib.osdp_set_tuning(k, 0)
    try:
        return fn()
    finally:
        for k, v in zip(keys, old):
            lib.osdp_set_tuning(k, v)


@pytest.mark.parametrize("T,h,f,k", [
    (256, 256, 512, 1),       # exact tiles, one tile row
    (384, 128, 512, 2),
    (333, 136, 520, 3),       # ragged everywhere
    (130, 72, 264, 1),
    (1000, 320, 1032, 4),
    (64, 8, 8, 4),            # minimum hidden / ffn
    (5, 64, 128, 5),          # one token per slice
    (1, 16, 24, 1),
    (1536, 1024, 2048, 2),    # several tile rows and columns: every dependency kind spans several tiles
    (2100, 520, 1288, 3),     # the same, ragged; hidden wider than 256: 128-column tiles for A2 / A7
])
def test_slice_kernel_matches_oracle_and_the_per_gemm_path_bitwise(lib, slice_kernel, T, h, f, k):
    inp = I.mlp_inputs(T, h, f, torch.bfloat16, seed=31)
    ref = O.mlp_forward_backward(**inp.as_f64())
    got = run_gpu(lib, inp, k)
    n_fwd_bwd = lib.osdp_last_launch_count()
    errs = {n: rel_err(got[n], ref[n]) for n in NAMES}
    assert all(e <= 2e-2 for e in errs.values()), errs
    assert n_fwd_bwd == 2 + k, "backward = db2 (two launches) + one slice kernel per slice"
    want = per_gemm(lib, lambda: run_gpu(lib, inp, k))
    for n in NAMES:
        assert np.array_equal(got[n], want[n]), f"{n}: slice kernel and launch-per-GEMM path differ"


def test_slice_kernel_is_reproducible_and_rows_do_not_depend_on_k(lib, slice_kernel):
    inp = I.mlp_inputs(2048, 512, 1024, torch.bfloat16, seed=32)
    a = run_gpu(lib, inp, 4)
    b = run_gpu(lib, inp, 4)
    c = run_gpu(lib, inp, 8)
    for n in NAMES:
        assert np.array_equal(a[n], b[n]), n
    assert np.array_equal(a["Y"], c["Y"]) and np.array_equal(a["dX"], c["dX"]) and np.array_equal(a["db2"], c["db2"])


def test_two_streams_of_slice_kernels_do_not_deadlock(lib, slice_kernel):
    """Two slice kernels in flight on different streams can each hold SMs the other's missing CTAs would use; tiles are
    claimed dynamically by the CTAs that run, so neither launch ever waits for a CTA that is not resident."""
    T, h, f, k = 4096, 1024, 4096, 2
    inps = [I.mlp_inputs(T, h, f, torch.bfloat16, seed=s) for s in (40, 41)]
    want = [run_gpu(lib, inp, k) for inp in inps]
    devs = [inp.to("cuda") for inp in inps]
    ops = [lib.SplitMlp(T, h, f, torch.bfloat16, k) for _ in inps]
    streams = [torch.cuda.Stream() for _ in inps]
    torch.cuda.synchronize()
    outs = [None, None]
    for _ in range(4):
        for i, (d, op, st) in enumerate(zip(devs, ops, streams)):
            with torch.cuda.stream(st):
                Y = op.forward(d.X, d.W1, d.b1, d.W2, d.b2, stream=st)
                g = op.backward(d.X, d.W1, d.b1, d.W2, d.dY, stream=st)
            outs[i] = dict(Y=Y, **g)
    torch.cuda.synchronize()
    for o, w in zip(outs, want):
        for n in NAMES:
            assert np.array_equal(o[n].double().cpu().numpy(), w[n]), n


def test_slice_kernel_step_can_be_captured_in_a_cuda_graph(lib, slice_kernel):
    T, h, f, k = 1000, 320, 1032, 4
    inp = I.mlp_inputs(T, h, f, torch.bfloat16, seed=33)
    want = run_gpu(lib, inp, k)
    d = inp.to("cuda")
    op = lib.SplitMlp(T, h, f, torch.bfloat16, k)
    Y = torch.empty_like(d.X)
    g = dict(dX=torch.empty_like(d.X), dW1=torch.empty(h, f, device="cuda"), db1=torch.empty(f, device="cuda"),
             dW2=torch.empty(f, h, device="cuda"), db2=torch.empty(h, device="cuda"))
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        op.forward(d.X, d.W1, d.b1, d.W2, d.b2, Y=Y, stream=s)
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
        assert np.array_equal(got[n].double().cpu().numpy(), want[n]), n


def test_24_calls_in_flight_on_24_streams_each_with_its_own_workspace(lib):
    """The tile counter and flags of a call sit in ITS workspace (round 2: 16 static blocks handed out round-robin, so a
    17th call in flight shared a live call's tile counter).  24 operators, 24 streams, three rounds without a host
    synchronisation in between: every call gives the bits of the same call made alone."""
    T, h, f, k, n = 1024, 256, 1024, 4, 24
    inps = [I.mlp_inputs(T, h, f, torch.bfloat16, seed=s) for s in (50, 51, 52)]
    want = [run_gpu(lib, inp, k) for inp in inps]
    assert lib.osdp_last_launch_count() == 2 + k                     # the backward ran as one kernel per slice
    devs = [inp.to("cuda") for inp in inps]
    ops = [lib.SplitMlp(T, h, f, torch.bfloat16, k) for _ in range(n)]
    streams = [torch.cuda.Stream() for _ in range(n)]
    torch.cuda.synchronize()
    outs = [None] * n
    for _ in range(3):
        for i, (op, st) in enumerate(zip(ops, streams)):
            d = devs[i % 3]
            with torch.cuda.stream(st):
                Y = op.forward(d.X, d.W1, d.b1, d.W2, d.b2, stream=st)
                g = op.backward(d.X, d.W1, d.b1, d.W2, d.dY, stream=st)
            outs[i] = dict(Y=Y, **g)
    torch.cuda.synchronize()
    for i, o in enumerate(outs):
        for name in NAMES:
            assert np.array_equal(o[name].double().cpu().numpy(), want[i % 3][name]), (i, name)


def test_two_captured_graphs_replayed_side_by_side_with_eager_calls(lib):
    """Two captured steps (each operator with its own workspace, so its own counter and flags are what the graph holds)
    replayed at the same time on two streams while a third stream makes eager calls: all three give the serial bits."""
    T, h, f, k = 1000, 320, 1032, 4
    inps = [I.mlp_inputs(T, h, f, torch.bfloat16, seed=s) for s in (53, 54, 55)]
    want = [run_gpu(lib, inp, k) for inp in inps]
    devs = [inp.to("cuda") for inp in inps]
    ops = [lib.SplitMlp(T, h, f, torch.bfloat16, k) for _ in inps]
    streams = [torch.cuda.Stream() for _ in inps]
    outs = [dict(Y=torch.empty_like(d.X), dX=torch.empty_like(d.X), dW1=torch.empty(h, f, device="cuda"),
                 db1=torch.empty(f, device="cuda"), dW2=torch.empty(f, h, device="cuda"), db2=torch.empty(h, device="cuda"))
            for d in devs]

    def step(i):
        d, o, s = devs[i], outs[i], streams[i]
        ops[i].forward(d.X, d.W1, d.b1, d.W2, d.b2, Y=o["Y"], stream=s)
        ops[i].backward(d.X, d.W1, d.b1, d.W2, d.dY, out={n: o[n] for n in NAMES if n != "Y"}, stream=s)

    graphs = []
    for i in (0, 1):
        s = streams[i]
        s.wait_stream(torch.cuda.current_stream())
        with torch.cuda.stream(s):
            step(i)                                                   # warm-up outside the capture
            s.synchronize()
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph, stream=s):
                step(i)
        graphs.append(graph)
    for o in outs:
        for t in o.values():
            t.fill_(7.0)
    torch.cuda.synchronize()
    for _ in range(6):
        for i in (0, 1):
            with torch.cuda.stream(streams[i]):
                graphs[i].replay()
        with torch.cuda.stream(streams[2]):
            step(2)
    torch.cuda.synchronize()
    for i, o in enumerate(outs):
        for name in NAMES:
            assert np.array_equal(o[name].double().cpu().numpy(), want[i][name]), (i, name)


def test_default_threshold_takes_small_slices_only(lib):
    """Default OSDP_TUNE_SLICE_KERNEL_MAX_TILES = 128 tiles of the [T_s x ffn] GEMMs: small slices run as one kernel per
    slice, large ones keep one launch per GEMM."""
    assert lib.osdp_get_tuning(lib.OSDP_TUNE_SLICE_KERNEL_MAX_TILES) == 128
    for (T, h, f, k), per_slice in (((2048, 256, 1024, 2), 1), ((8192, 512, 4096, 1), 6)):
        d = I.mlp_inputs(T, h, f, torch.bfloat16, seed=36).to("cuda")
        op = lib.SplitMlp(T, h, f, torch.bfloat16, k)
        op.backward(d.X, d.W1, d.b1, d.W2, d.dY)
        torch.cuda.synchronize()
        assert lib.osdp_last_launch_count() == 2 + k * per_slice, (T, h, f, k)


def test_slice_kernel_trace_and_fallback(lib, slice_kernel):
    """One traced launch per slice (steps 21 / 22); fp32 and over-sized calls keep the launch-per-GEMM path."""
    T, h, f, k = 600, 128, 512, 3
    d = I.mlp_inputs(T, h, f, torch.bfloat16, seed=34).to("cuda")
    op = lib.SplitMlp(T, h, f, torch.bfloat16, k)
    op.forward(d.X, d.W1, d.b1, d.W2, d.b2)
    lib.osdp_trace_enable(True)
    op.forward(d.X, d.W1, d.b1, d.W2, d.b2)
    op.backward(d.X, d.W1, d.b1, d.W2, d.dY)
    tr = lib.osdp_trace_read()
    lib.osdp_trace_enable(False)
    assert [s for s, _ in tr] == [21] * k + [8, 8] + [22] * k
    assert "slice kernel" in lib.osdp_step_name(21) and "slice kernel" in lib.osdp_step_name(22)
    d32 = I.mlp_inputs(96, 32, 64, torch.float32, seed=35).to("cuda")
    op32 = lib.SplitMlp(96, 32, 64, torch.float32, 2)
    op32.forward(d32.X, d32.W1, d32.b1, d32.W2, d32.b2)
    assert lib.osdp_last_launch_count() == 2 * 2               # fp32: one launch per GEMM


def test_many_tiny_slices_pipeline_and_single_buffer_forward(lib, slice_kernel):
    """k = 64 slices of 24 tokens: 64 forward launches that alternate the two H_s buffers without waiting for each other
    (late programmatic wait), 64 backward launches with their own flags; and the forward with its own minimum workspace
    (one H_s buffer: slices strictly in sequence) gives the same bits."""
    T, h, f, k = 1536, 264, 520, 64
    inp = I.mlp_inputs(T, h, f, torch.bfloat16, seed=37)
    ref = O.mlp_forward_backward(**inp.as_f64())
    got = run_gpu(lib, inp, k)
    errs = {n: rel_err(got[n], ref[n]) for n in NAMES}
    assert all(e <= 2e-2 for e in errs.values()), errs
    want = per_gemm(lib, lambda: run_gpu(lib, inp, k))
    for n in NAMES:
        assert np.array_equal(got[n], want[n]), n
    d = inp.to("cuda")
    desc = lib.make_desc(T, h, f, torch.bfloat16, k)
    nbytes = lib.osdp_split_mlp_workspace_bytes(desc, lib.OSDP_FWD)
    ws = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
    for _ in range(3):                                          # back to back: the next call's first slice waits for this one
        Y = torch.empty_like(d.X)
        lib.osdp_split_mlp_forward(desc, d.X, d.W1, d.b1, d.W2, d.b2, Y, ws, workspace_bytes=nbytes)
    torch.cuda.synchronize()
    assert lib.osdp_last_launch_count() == k
    assert np.array_equal(Y.double().cpu().numpy(), got["Y"])


def test_back_to_back_steps_reuse_buffers_safely(lib, slice_kernel):
    """Forward, backward, forward, ... on one stream with one workspace: the pipelined forward of step i + 1 must not
    touch the buffers the backward of step i still reads (the first slice of every call waits for everything before it)."""
    T, h, f, k = 2048, 512, 2048, 4
    inp = I.mlp_inputs(T, h, f, torch.bfloat16, seed=38)
    want = run_gpu(lib, inp, k)
    d = inp.to("cuda")
    op = lib.SplitMlp(T, h, f, torch.bfloat16, k)
    outs = []
    for _ in range(6):
        Y = op.forward(d.X, d.W1, d.b1, d.W2, d.b2)
        g = op.backward(d.X, d.W1, d.b1, d.W2, d.dY)
        outs.append(dict(Y=Y, **g))
    torch.cuda.synchronize()
    for o in outs:
        for n in NAMES:
            assert np.array_equal(o[n].double().cpu().numpy(), want[n]), n


def run_gpu_ffn(lib, inp, k):
    T, h = inp.X.shape
    f = inp.W1.shape[1]
    d = inp.to("cuda")
    op = lib.SplitMlp(T, h, f, torch.bfloat16, k, axis="ffn")
    Y = op.forward(d.X, d.W1, d.b1, d.W2, d.b2)
    g = op.backward(d.X, d.W1, d.b1, d.W2, d.dY)
    torch.cuda.synchronize()
    out = {"Y": Y}
    out.update(g)
    return {n: out[n].to(torch.float64).cpu().numpy() for n in NAMES}


@pytest.mark.parametrize("T,h,f,k", [
    (256, 256, 512, 1),
    (333, 136, 520, 3),       # ragged everywhere, ragged ffn slices
    (1000, 320, 1032, 4),
    (1536, 1024, 2048, 2),    # several tile rows and columns
    (2100, 520, 1288, 5),
    (640, 64, 4096, 16),      # many narrow ffn slices
])
def test_ffn_split_slice_kernel_matches_oracle_and_the_per_gemm_path_bitwise(lib, slice_kernel, T, h, f, k):
    """The paper-literal ffn-axis split through the same kernel: A1 -> A2 (Y accumulated in fp32 by reduce-add), and
    (A3 + A4) -> A7 (dX accumulated) | A5 | A6 with the slice's own dW / db1 parts written once."""
    inp = I.mlp_inputs(T, h, f, torch.bfloat16, seed=39)
    ref = O.mlp_forward_backward(**inp.as_f64())
    got = run_gpu_ffn(lib, inp, k)
    n_bwd = lib.osdp_last_launch_count()
    errs = {n: rel_err(got[n], ref[n]) for n in NAMES}
    assert all(e <= 2e-2 for e in errs.values()), errs
    assert n_bwd == 2 + k + (1 if k > 1 else 0), "db2 (two launches) + one kernel per slice (+ accumulator -> dX)"
    want = per_gemm(lib, lambda: run_gpu_ffn(lib, inp, k))
    for n in NAMES:
        assert np.array_equal(got[n], want[n]), f"{n}: slice kernel and launch-per-GEMM path differ"
