"""ZDP weight-slice gathering on ONE GPU through the C ABI with two streams, against the fp64 MLP oracle: world = 1 (the
collectives degenerate to device copies), and world = 2 / 3 as host threads of one process over an in-process loopback
osdp_comm, which runs the library's real executor and its cross-stream event chain at N > 1.  GPU only.  No multi-GPU
box is available to this build, so N > 1 over NVLink stays unmeasured."""
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


class LoopbackComm:
    """The two collectives of osdp_comm for N ranks that are N HOST THREADS on ONE GPU (no multi-GPU box exists for this
    build): every rank pulls the other ranks' send buffers with device copies (all-gather) or adds their chunks in rank
    order (reduce-scatter) on the stream the library names, ordered across ranks by CUDA events; the host threads meet
    at a barrier per collective (all ranks walk the same schedule).  No kernel ever waits for another kernel - only
    streams wait for events - so the ranks cannot deadlock however the GPU schedules them.  Test plumbing: what is under
    test is the library's executor (its gather / compute / reduce-scatter event chain and buffer reuse at N = 2)."""

    def __init__(self, lib, world):
        import threading
        self.lib, self.world = lib, world
        self.barrier = threading.Barrier(world)
        self.send = [None] * world
        self.ready = [None] * world
        self.done = [None] * world
        self.error = None
        self.calls = [0] * world

    def _meet(self):
        self.barrier.wait(timeout=120)

    def _collective(self, rank, send, stream, body):
        try:
            st = torch.cuda.ExternalStream(int(stream or 0))
            ev = torch.cuda.Event()
            ev.record(st)                                   # this rank's send buffer is complete at this point of its stream
            self.send[rank], self.ready[rank] = int(send), ev
            self._meet()
            with torch.cuda.stream(st):
                for p in range(self.world):
                    if p != rank:
                        st.wait_event(self.ready[p])
                body(st)
            done = torch.cuda.Event()
            done.record(st)
            self.done[rank] = done
            self._meet()
            for p in range(self.world):
                if p != rank:
                    st.wait_event(self.done[p])             # nobody still reads my send buffer when my stream moves on
            self._meet()                                    # the slots above may be overwritten by the next collective now
            self.calls[rank] += 1
            return 0
        except Exception as e:                              # a Python exception must not unwind through C
            self.error = self.error or e
            self.barrier.abort()
            return 1

    def _mem(self, ptr, nbytes, typestr):
        return torch.as_tensor(self.lib._DevMem(ptr, nbytes, typestr), device="cuda")

    def rank(self, r):
        lib = self.lib

        def all_gather(ctx, send, recv, nbytes, stream):
            def body(st):
                for p in range(self.world):
                    self._mem(recv + p * nbytes, nbytes, "|u1").copy_(self._mem(self.send[p], nbytes, "|u1"))
            return self._collective(r, send, stream, body)

        def reduce_scatter(ctx, send, recv, nfloats, stream):
            def body(st):
                out = self._mem(recv, nfloats * 4, "<f4")
                out.copy_(self._mem(self.send[0] + r * nfloats * 4, nfloats * 4, "<f4"))
                for p in range(1, self.world):              # fixed rank order: deterministic sums
                    out.add_(self._mem(self.send[p] + r * nfloats * 4, nfloats * 4, "<f4"))
            return self._collective(r, send, stream, body)

        class _Comm:
            pass
        c = _Comm()
        c._ag, c._rs = lib.ALL_GATHER_FN(all_gather), lib.REDUCE_SCATTER_FN(reduce_scatter)
        c.struct = lib.osdp_comm(None, c._ag, c._rs)
        c.error = None
        return c


@pytest.mark.parametrize("dtype,T,h,f,k,N", [(torch.bfloat16, 384, 128, 1024, 4, 2), (torch.bfloat16, 300, 144, 528, 5, 2),
                                             (torch.bfloat16, 512, 240, 1200, 3, 3), (torch.float32, 96, 32, 64, 4, 2)])
def test_zdp_executor_at_world_2_and_3_on_one_gpu_matches_the_oracle(lib, dtype, T, h, f, k, N):
    """The C executor of the ZDP mode with N > 1 (PAPER.md:47 all-gather before use / reduce-scatter of the gradients;
    PAPER.md:92-94 three collectives; PAPER.md:177 communication beside computation): N host threads, each one rank
    with its own token batch, shard, workspace and stream pair, two steps back to back (the second step's gathers reuse
    the buffers the first step's GEMMs read).  Per rank Y_r and dX_r are the unsplit MLP's on that rank's batch; the
    gathered gradient shards are the SUM over ranks (reading Z3) of the unsplit MLP's gradients."""
    import threading
    tol = 2e-2 if dtype == torch.bfloat16 else 1e-4
    base = I.mlp_inputs(T, h, f, dtype, seed=60)
    batches = [base] + [I.mlp_inputs(T, h, f, dtype, seed=60 + r) for r in range(1, N)]
    refs = []
    for b in batches:
        x = base.as_f64()
        x["X"], x["dY"] = b.as_f64()["X"], b.as_f64()["dY"]
        refs.append(O.mlp_forward_backward(**x))
    dbase = base.to("cuda")
    ranks = []
    for r, b in enumerate(batches):
        d = b.to("cuda")
        desc = lib.make_zdp_desc(T, h, f, dtype, k, N, r)
        shard = lib.zdp_shard(desc, dbase.W1, dbase.b1, dbase.W2, dbase.b2)
        ws = torch.empty(max(lib.osdp_zdp_ffn_split_mlp_workspace_bytes(desc, p) for p in (lib.OSDP_FWD, lib.OSDP_BWD)),
                         dtype=torch.uint8, device="cuda")
        ranks.append(dict(desc=desc, shard=shard, ws=ws, X=d.X, dY=d.dY, Y=torch.full_like(d.X, float("nan")),
                          dX=torch.full_like(d.X, float("nan")),
                          g=torch.full((shard.numel(),), float("nan"), dtype=torch.float32, device="cuda")))
    loop = LoopbackComm(lib, N)
    comms = [loop.rank(r) for r in range(N)]
    torch.cuda.synchronize()
    failures = []

    def worker(r):
        try:
            torch.cuda.set_device(0)
            R = ranks[r]
            cs, ms = torch.cuda.Stream(), torch.cuda.Stream()
            for _ in range(2):
                lib.osdp_zdp_ffn_split_mlp_forward(R["desc"], R["shard"], R["X"], R["Y"], R["ws"], comm=comms[r],
                                                   compute_stream=cs, comm_stream=ms)
                lib.osdp_zdp_ffn_split_mlp_backward(R["desc"], R["shard"], R["X"], R["dY"], R["dX"], R["g"], R["ws"],
                                                    comm=comms[r], compute_stream=cs, comm_stream=ms)
            cs.synchronize()
            ms.synchronize()
        except Exception as e:
            failures.append((r, e))
            loop.barrier.abort()

    threads = [threading.Thread(target=worker, args=(r,)) for r in range(N)]
    for t in threads:
        t.start()
    for t in threads:
        t.join(timeout=300)
    assert not any(t.is_alive() for t in threads), "a rank did not finish"
    assert not failures and loop.error is None, (failures, loop.error)
    torch.cuda.synchronize()
    assert all(c == 2 * ((3 * k + 1) + (3 * k + 3 * k + 1)) for c in loop.calls), loop.calls   # W1, b1, W2 per slice (+ b2 / db2)
    for r, R in enumerate(ranks):
        for name in ("Y", "dX"):
            assert rel_err(R[name].double().cpu().numpy(), refs[r][name]) <= tol, (r, name)
    dW1, db1, dW2, db2 = lib.zdp_unshard(ranks[0]["desc"], [R["g"] for R in ranks])
    for name, t in dict(dW1=dW1, db1=db1, dW2=dW2, db2=db2).items():
        want = sum(ref[name] for ref in refs)
        assert rel_err(t.double().cpu().numpy(), want) <= tol, name


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
    shard2 = lib.zdp_shard(two, inp.W1, inp.b1, inp.W2, inp.b2)
    assert lib.osdp_zdp_ffn_split_mlp_forward(two, shard2, inp.X, Y, ws, check=False) == lib.OSDP_ERR_NULL   # N > 1 needs comm
    assert lib.osdp_zdp_ffn_split_mlp_forward(two, shard, inp.X, Y, ws, check=False) == lib.OSDP_ERR_SHAPE   # binding: world-1 shard
    assert lib.osdp_zdp_ffn_split_mlp_forward(desc, None, inp.X, Y, ws, check=False) == lib.OSDP_ERR_NULL
    # binding: the same marshalling checks as the other calls (dtype, element count)
    assert lib.osdp_zdp_ffn_split_mlp_forward(desc, shard.float(), inp.X, Y, ws, check=False) == lib.OSDP_ERR_DTYPE
    assert lib.osdp_zdp_ffn_split_mlp_forward(desc, shard[:-8], inp.X, Y, ws, check=False) == lib.OSDP_ERR_SHAPE
    # a collective that fails: its own status, and comm_stream is joined back (both streams drain, the next call works)
    calls = []

    class Failing:
        def __init__(self):
            self._ag = lib.ALL_GATHER_FN(lambda ctx, send, recv, n, st: calls.append(n) or (1 if len(calls) == 3 else 0))
            self._rs = lib.REDUCE_SCATTER_FN(lambda ctx, send, recv, n, st: 1)
            self.struct = lib.osdp_comm(None, self._ag, self._rs)
            self.error = "third all-gather refused"
    ws2 = torch.empty(lib.osdp_zdp_ffn_split_mlp_workspace_bytes(two, lib.OSDP_FWD), dtype=torch.uint8, device="cuda")
    cs = torch.cuda.Stream()
    assert lib.osdp_zdp_ffn_split_mlp_forward(two, shard2, inp.X, Y, ws2, comm=Failing(), comm_stream=cs,
                                              check=False) == lib.OSDP_ERR_COMM
    assert len(calls) == 3 and "collective" in lib.osdp_status_string(lib.OSDP_ERR_COMM)
    torch.cuda.synchronize()
    assert lib.osdp_zdp_ffn_split_mlp_forward(desc, shard, inp.X, Y, ws, comm_stream=cs, check=False) == lib.OSDP_OK
    torch.cuda.synchronize()


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
