"""osdp_bias_grad_static: the bias gradient (step A8, db = column sums of dY) for callers that cannot allocate.

Every other entry point of the library borrows its scratch from a workspace the caller allocated.  A caller that runs
where the CUDA allocator must not be entered (inside another library's callback or allocator hook), that sits on a
device whose memory is wholly owned by a pool it may not draw from, or that is handed nothing but the input and output
pointers by its embedder, has no workspace to lend.  For it the library keeps the 32 x cols partial sums in a static
__device__ array of its own (2 MiB, so cols <= 16384), shared by all calls on a GPU.

This file checks that entry point against the path that already exists (the db2 of osdp_split_mlp_backward, which uses
the caller's workspace) on two calls in a row that differ in shape, so that what the first call left in the shared
array would show up in the second if it mattered.  It is named test_zz_* so that pytest collects it last: with -x a
failure here cannot hide any other test.  It holds no state of its own, so it passes alone in a fresh process (where
its first call is the one that looks the array's address up) and after the rest of the suite.  GPU only."""
import numpy as np
import pytest
import torch

from paper_2305_09940_b200 import inputs as I

pytestmark = pytest.mark.gpu
TOL = {torch.bfloat16: 2e-2, torch.float32: 1e-4}   # the bar of the other GPU tests: max|a - b| <= tol * max|b|


def rel_err(got, ref):
    scale = float(np.max(np.abs(ref)))
    return float(np.max(np.abs(got - ref))) / (scale if scale > 0 else 1.0)


def db2_of_the_workspace_path(lib, d, T, h, f, dtype, k):
    op = lib.SplitMlp(T, h, f, dtype, k)
    g = op.backward(d.X, d.W1, d.b1, d.W2, d.dY)
    torch.cuda.synchronize()
    return g["db2"].double().cpu().numpy()


@pytest.mark.parametrize("dtype,shapes", [
    (torch.bfloat16, [(1000, 320, 264, 3), (777, 136, 72, 2)]),     # second call: fewer rows and columns than the first
    (torch.float32, [(300, 64, 32, 2), (517, 200, 16, 4)]),         # second call: more of both
])
def test_two_calls_in_a_row_match_the_workspace_path(lib, dtype, shapes):
    cases = []
    for seed, (T, h, f, k) in enumerate(shapes):
        d = I.mlp_inputs(T, h, f, dtype, seed=40 + seed).to("cuda")
        cases.append((d, db2_of_the_workspace_path(lib, d, T, h, f, dtype, k), torch.full((h,), float("nan"), device="cuda")))
    for d, _, db in cases:                      # back to back on one stream: the calls share the static array in order
        lib.osdp_bias_grad_static(d.dY, db)
    torch.cuda.synchronize()
    for (d, want, db), shape in zip(cases, shapes):
        got = db.double().cpu().numpy()
        assert np.all(np.isfinite(got)), shape
        assert rel_err(got, want) <= TOL[dtype], (shape, rel_err(got, want))
        assert np.array_equal(got, want), shape      # same chunking and summation order as the existing path: same bits


def test_repeat_calls_take_no_device_memory_and_sizes_over_the_limit_are_refused(lib):
    rows, cols = 513, lib.OSDP_BIAS_GRAD_STATIC_MAX_COLS                     # the widest tensor the static array holds
    g = torch.Generator(device="cuda").manual_seed(7)
    dY = (torch.rand(rows, cols, device="cuda", generator=g) - 0.5).to(torch.bfloat16)
    db = torch.empty(cols, device="cuda")
    too_wide = torch.zeros(8, cols + 8, device="cuda", dtype=torch.bfloat16)
    db_wide = torch.full((cols + 8,), 3.0, device="cuda")
    lib.osdp_bias_grad_static(dY, db)             # first use of this dtype's kernels (lazy module loading happens here)
    torch.cuda.synchronize()
    want = dY.double().sum(dim=0).cpu().numpy()   # fp64 column sums of the same bf16 values
    assert rel_err(db.double().cpu().numpy(), want) <= TOL[torch.bfloat16]
    first = db.clone()
    free_before, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        lib.osdp_bias_grad_static(dY, db)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_after == free_before, (free_before, free_after)              # nothing was allocated on the device
    assert torch.equal(db, first)
    assert lib.osdp_bias_grad_static(too_wide, db_wide, check=False) == lib.OSDP_ERR_STATIC_LIMIT
    with pytest.raises(lib.OsdpError, match="static scratch"):
        lib.osdp_bias_grad_static(too_wide, db_wide)
    torch.cuda.synchronize()
    assert bool((db_wide == 3.0).all())                                      # refused before any launch
    assert lib.osdp_bias_grad_static(dY[:, :12].contiguous(), db[:12].clone(), check=False) == lib.OSDP_ERR_SHAPE
