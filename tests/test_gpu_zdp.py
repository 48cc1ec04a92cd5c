"""ZDP weight-slice gathering on ONE GPU (world = 1: the collectives degenerate to device copies), through the C ABI with
two streams, against the fp64 MLP oracle.  GPU only.  N > 1 is covered on CPU (tests/test_zdp.py); no multi-GPU box
is available to this build."""
import numpy as np
import pytest
import torch

from oracle import mlp_oracle as O
from paper_2305_09940_b200 import inputs as I

pytestmark = pytest.mark.gpu
NAMES = ("Y", "dX", "dW1", "db1", "dW2", "db2")


def rel_err(got, ref):
    scale = float(np.max(np.abs(ref)))
    return float(np.max(np.abs(got - ref))) / (scale if scale > 0 else 1.0)


def run_zdp(lib, inp, dtype, k, two_streams=True):
    T, h = inp.X.shape
    f = inp.W1.shape[1]
    d = inp.to("cuda")
    desc = lib.make_zdp_desc(T, h, f, dtype, k, 1, 0)
    shard = lib.zdp_shard(desc, d.W1, d.b1, d.W2, d.b2)
    ws = torch.empty(max(lib.osdp_zdp_ffn_split_mlp_workspace_bytes(desc, p) for p in (lib.OSDP_FWD, lib.OSDP_BWD)),
                     dtype=torch.uint8, device="cuda")
    Y, dX = torch.empty_like(d.X), torch.empty_like(d.X)
    gshard = torch.full((shard.numel(),), float("nan"), dtype=torch.float32, device="cuda")
    comm_stream = torch.cuda.Stream() if two_streams else None
    lib.osdp_zdp_ffn_split_mlp_forward(desc, shard, d.X, Y, ws, comm_stream=comm_stream)
    lib.osdp_zdp_ffn_split_mlp_backward(desc, shard, d.X, d.dY, dX, gshard, ws, comm_stream=comm_stream)
    torch.cuda.synchronize()
    dW1, db1, dW2, db2 = lib.zdp_unshard(desc, [gshard])
    out = dict(Y=Y, dX=dX, dW1=dW1, db1=db1, dW2=dW2, db2=db2)
    return {n: out[n].to(torch.float64).cpu().numpy() for n in NAMES}


@pytest.mark.parametrize("T,h,f,k,two", [(512, 256, 1024, 1, True), (512, 256, 1024, 4, True), (300, 136, 520, 3, True),
                                         (384, 128, 512, 2, False), (1000, 320, 1032, 5, True)])
def test_bf16_zdp_world1_matches_oracle(lib, T, h, f, k, two):
    inp = I.mlp_inputs(T, h, f, torch.bfloat16, seed=21)
    ref = O.mlp_forward_backward(**inp.as_f64())
    got = run_zdp(lib, inp, torch.bfloat16, k, two)
    errs = {n: rel_err(got[n], ref[n]) for n in NAMES}
    assert all(e <= 2e-2 for e in errs.values()), errs


def test_fp32_zdp_world1_matches_oracle_and_the_in_place_ffn_split(lib):
    T, h, f, k = 96, 32, 64, 4
    inp = I.mlp_inputs(T, h, f, torch.float32, seed=22)
    ref = O.mlp_forward_backward(**inp.as_f64())
    got = run_zdp(lib, inp, torch.float32, k)
    for n in NAMES:
        assert rel_err(got[n], ref[n]) <= 1e-4, n
    # same slices, same kernels as osdp_ffn_split_mlp_* on weights sliced in place: bit-identical results
    d = inp.to("cuda")
    op = lib.SplitMlp(T, h, f, torch.float32, k, axis="ffn")
    Y = op.forward(d.X, d.W1, d.b1, d.W2, d.b2)
    g = op.backward(d.X, d.W1, d.b1, d.W2, d.dY)
    torch.cuda.synchronize()
    assert np.array_equal(Y.double().cpu().numpy(), got["Y"]) and np.array_equal(g["dX"].double().cpu().numpy(), got["dX"])
    for n in ("dW1", "db1", "dW2", "db2"):
        assert np.array_equal(g[n].double().cpu().numpy(), got[n]), n


def test_zdp_is_graph_capturable_and_repeatable(lib):
    """Back-to-back calls reuse the gathered buffers: the second call's gathers must wait for the first call's GEMMs."""
    T, h, f, k = 512, 256, 2048, 4
    inp = I.mlp_inputs(T, h, f, torch.bfloat16, seed=23)
    first = run_zdp(lib, inp, torch.bfloat16, k)
    d = inp.to("cuda")
    desc = lib.make_zdp_desc(T, h, f, torch.bfloat16, k, 1, 0)
    shard = lib.zdp_shard(desc, d.W1, d.b1, d.W2, d.b2)
    shard2 = lib.zdp_shard(desc, d.W1 * 2, d.b1, d.W2, d.b2)
    ws = torch.empty(lib.osdp_zdp_ffn_split_mlp_workspace_bytes(desc, lib.OSDP_BWD) + lib.osdp_zdp_ffn_split_mlp_workspace_bytes(desc, lib.OSDP_FWD),
                     dtype=torch.uint8, device="cuda")
    Ya, Yb = torch.empty_like(d.X), torch.empty_like(d.X)
    cs = torch.cuda.Stream()
    for _ in range(5):      # alternate two different parameter shards through the same workspace, no host sync in between
        lib.osdp_zdp_ffn_split_mlp_forward(desc, shard2, d.X, Yb, ws, comm_stream=cs)
        lib.osdp_zdp_ffn_split_mlp_forward(desc, shard, d.X, Ya, ws, comm_stream=cs)
    torch.cuda.synchronize()
    assert np.array_equal(Ya.double().cpu().numpy(), first["Y"])
    assert not np.array_equal(Yb.double().cpu().numpy(), first["Y"])


def test_zdp_error_codes(lib):
    T, h, f = 64, 64, 128
    inp = I.mlp_inputs(T, h, f, torch.bfloat16, seed=1).to("cuda")
    desc = lib.make_zdp_desc(T, h, f, torch.bfloat16, 2, 1, 0)
    shard = lib.zdp_shard(desc, inp.W1, inp.b1, inp.W2, inp.b2)
    ws = torch.empty(lib.osdp_zdp_ffn_split_mlp_workspace_bytes(desc, lib.OSDP_FWD), dtype=torch.uint8, device="cuda")
    Y = torch.empty_like(inp.X)
    assert lib.osdp_zdp_ffn_split_mlp_forward(desc, shard, inp.X, Y, ws, check=False) == lib.OSDP_OK
    assert lib.osdp_zdp_ffn_split_mlp_forward(desc, shard, inp.X, Y, ws[:1024], check=False) == lib.OSDP_ERR_WORKSPACE
    two = lib.make_zdp_desc(T, h, f, torch.bfloat16, 2, 2, 0)
    assert lib.osdp_zdp_ffn_split_mlp_forward(two, shard, inp.X, Y, ws, check=False) == lib.OSDP_ERR_NULL   # N > 1 needs comm
    assert lib.osdp_zdp_ffn_split_mlp_forward(desc, None, inp.X, Y, ws, check=False) == lib.OSDP_ERR_NULL


NCCL_WORKER = r'''
import os, sys, json
sys.path.insert(0, %r)
import numpy as np, torch, torch.distributed as dist
from oracle import mlp_oracle as O
from paper_2305_09940_b200 import binding as lib, inputs as I
torch.cuda.set_device(0)
dist.init_process_group("nccl", device_id=torch.device("cuda", 0))
T, h, f, k = 384, 128, 1024, 4
inp = I.mlp_inputs(T, h, f, torch.bfloat16, seed=31)
ref = O.mlp_forward_backward(**inp.as_f64())
d = inp.to("cuda")
desc = lib.make_zdp_desc(T, h, f, torch.bfloat16, k, dist.get_world_size(), dist.get_rank())
shard = lib.zdp_shard(desc, d.W1, d.b1, d.W2, d.b2)
ws = torch.empty(max(lib.osdp_zdp_ffn_split_mlp_workspace_bytes(desc, p) for p in (0, 1)), dtype=torch.uint8, device="cuda")
Y, dX = torch.empty_like(d.X), torch.empty_like(d.X)
g = torch.full((shard.numel(),), float("nan"), dtype=torch.float32, device="cuda")
comm = lib.TorchDistComm()
cs = torch.cuda.Stream()
for _ in range(2):
    lib.osdp_zdp_ffn_split_mlp_forward(desc, shard, d.X, Y, ws, comm=comm, comm_stream=cs)
    lib.osdp_zdp_ffn_split_mlp_backward(desc, shard, d.X, d.dY, dX, g, ws, comm=comm, comm_stream=cs)
torch.cuda.synchronize()
assert comm.error is None, comm.error
dW1, db1, dW2, db2 = lib.zdp_unshard(desc, [g])
out = dict(Y=Y, dX=dX, dW1=dW1, db1=db1, dW2=dW2, db2=db2)
errs = {n: float(np.max(np.abs(out[n].double().cpu().numpy() - ref[n])) / np.max(np.abs(ref[n]))) for n in ref}
print(json.dumps(errs))
dist.destroy_process_group()
''' % __import__("os").path.dirname(__import__("os").path.dirname(__import__("os").path.abspath(__file__)))


def test_zdp_through_nccl_collectives_single_rank(tmp_path):
    """The collectives really go through the caller-supplied osdp_comm callbacks (binding.TorchDistComm: NCCL all-gather /
    reduce-scatter enqueued on the library's comm stream) - with the one GPU this build has, a single-rank group."""
    import json
    import os
    import socket
    import subprocess
    import sys
    script = tmp_path / "zdp_nccl_worker.py"
    script.write_text(NCCL_WORKER)
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    env = dict(os.environ, WORLD_SIZE="1", RANK="0", LOCAL_RANK="0", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    p = subprocess.run([sys.executable, str(script)], env=env, capture_output=True, text=True, timeout=600)
    assert p.returncode == 0, p.stderr[-3000:]
    errs = json.loads(p.stdout.strip().splitlines()[-1])
    assert all(e <= 2e-2 for e in errs.values()), errs
