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


# ------------------------------------------------------------------ library host logic (no GPU): layout, schedule, bytes
def test_library_shard_layout_matches_the_oracles(lib):
    import torch
    for N, k, h, f, dt, unit in ((2, 2, 16, 64, torch.float32, 4), (4, 3, 32, 192, torch.bfloat16, 8), (1, 1, 8, 8, torch.bfloat16, 8)):
        rng = np.random.default_rng(1)
        W1, b1, W2, b2 = rng.standard_normal((h, f)), rng.standard_normal(f), rng.standard_normal((f, h)), rng.standard_normal(h)
        ref = Z.shard_params(W1, b1, W2, b2, k, N, unit)
        tW1, tb1, tW2, tb2 = (torch.tensor(a) for a in (W1, b1, W2, b2))
        desc = lib.make_zdp_desc(5, h, f, dt, k, N, 0)
        got_bounds = [(lib.osdp_zdp_slice_layout(desc, s).lo, lib.osdp_zdp_slice_layout(desc, s).hi) for s in range(k)]
        assert got_bounds == Z.slice_bounds(f, k, N, unit)
        shards = []
        for r in range(N):
            sh = lib.zdp_shard(desc, tW1, tb1, tW2, tb2, rank=r)
            shards.append(sh)
            flat = np.concatenate([np.concatenate([a.reshape(-1), b, c.reshape(-1)]) for a, b, c in ref[r]["slices"]] + [ref[r]["b2"]])
            np.testing.assert_array_equal(sh.numpy(), flat)                  # the library's offsets == the oracle's layout
            assert sh.numel() == lib.osdp_zdp_shard_elems(desc) == (2 * h * f + f + h) // N
        back = lib.zdp_unshard(desc, shards)
        for got, want in zip(back, (W1, b1, W2, b2)):
            np.testing.assert_array_equal(got.numpy(), want)


def test_library_schedule_follows_the_paper(lib):
    """PAPER.md:47 / :92-94: two all-gathers (one per pass) and one reduce-scatter of the parameters; PAPER.md:165:
    slices in order; at most two gathered slices exist (double buffering); the gather of
    slice s + 1 is enqueued before the computation of slice s so that it overlaps."""
    import torch
    N, k, h, f, e = 4, 5, 64, 640, 2
    desc = lib.make_zdp_desc(128, h, f, torch.bfloat16, k, N, 2)
    fwd, bwd = lib.osdp_zdp_schedule(desc, lib.OSDP_FWD), lib.osdp_zdp_schedule(desc, lib.OSDP_BWD)
    G, Cc, R = lib.OSDP_ZDP_GATHER, lib.OSDP_ZDP_COMPUTE, lib.OSDP_ZDP_REDUCE_SCATTER
    for sched, has_rs in ((fwd, False), (bwd, True)):
        comp = [s for op, s, *_ in sched if op == Cc]
        assert comp == list(range(k))                                            # sequential slices
        pos = {(op, s): i for i, (op, s, *_) in enumerate(sched)}
        for s in range(k):
            assert pos[(G, s)] < pos[(Cc, s)]
            if s + 1 < k:
                assert pos[(G, s + 1)] < pos[(Cc, s)]                            # prefetch of the next slice
            if s + 2 < k:
                assert pos[(G, s + 2)] > pos[(Cc, s)]                            # only two gathered buffers
            if has_rs:
                assert pos[(Cc, s)] < pos[(R, s)] and (s + 2 >= k or pos[(R, s)] < pos[(Cc, s + 2)])
        for op, s, buf, on_comm, nbytes in sched:
            assert on_comm == (0 if op == Cc else 1)
            if s < k:
                assert buf == s % 2
    S = (2 * h * f + f + h) * e
    gathered_fwd = sum(b for op, s, _, _, b in fwd if op == G)
    gathered_bwd = sum(b for op, s, _, _, b in bwd if op == G)
    scattered = sum(b for op, s, _, _, b in bwd if op == R)
    assert gathered_fwd * N == S and gathered_bwd * N == S - h * e               # b2 is not needed in the backward (S4)
    assert scattered * N == (2 * h * f + f + h) * 4                              # fp32 gradients
    # received bytes per rank = (N - 1) x contributed bytes: the (alpha, beta) model's 3 (N - 1) steps of S / N
    dev = lib.osdp_device(N, 0.0, 1.0, 1 << 62)
    c = lib.osdp_zdp_ffn_split_mlp_op_cost(desc, lib.OSDP_BWD)
    _, _, t_zdp = lib.osdp_cost_eval(c, lib.OSDP_ZDP, k, 0, dev)
    assert t_zdp == pytest.approx(3 * (N - 1) * S / N)
    assert (gathered_fwd + gathered_bwd) * (N - 1) + scattered * (N - 1) * e // 4 == pytest.approx(t_zdp, rel=h * e * 4 / S)


@pytest.mark.parametrize("T,h,f,N", [(512, 256, 2048, 8), (300, 264, 2112, 3), (128, 64, 1024, 2), (64, 32, 96, 1),
                                     (8192, 8192, 32768, 8)])
def test_library_zdp_cost_factors_never_underestimate_the_workspace(lib, T, h, f, N):
    """extra_fixed + ceil(extra_transient / k) >= osdp_zdp_ffn_split_mlp_workspace_bytes for every (N, k), odd k
    included (slices are whole groups of N x 16 bytes of columns, so the widest slice exceeds f / k), both dtypes, both
    passes - otherwise osdp_plan could accept a ZDP plan whose workspace does not fit M_limit.  And not by more than one
    group of columns + the accumulator at k = 1 + padding.  Round 2 under-estimated by up to 7.6 % (T = 512, h = 256,
    f = 2048, N = 8, k = 7, backward)."""
    import torch
    for dtype, e in ((torch.bfloat16, 2), (torch.float32, 4)):
        unit = 16 // e
        groups = f // (N * unit)
        for k in (1, 2, 3, 5, 7, 8, 11, groups):
            if k > groups:
                continue
            desc = lib.make_zdp_desc(T, h, f, dtype, k, N, 0)
            for pass_ in (lib.OSDP_FWD, lib.OSDP_BWD):
                ws = lib.osdp_zdp_ffn_split_mlp_workspace_bytes(desc, pass_)
                c = lib.osdp_zdp_ffn_split_mlp_op_cost(desc, pass_)
                est = c.extra_fixed + -(-c.extra_transient // k)
                per_col = c.extra_transient // f
                assert est >= ws, (dtype, k, pass_, est, ws)
                assert est - ws <= N * unit * per_col + 24 * 256 + (T * h * 4 + 256 if k == 1 else 0), (dtype, k, pass_, est, ws)


def test_library_zdp_workspace_holds_two_gathered_slices_and_shrinks_with_k(lib):
    import torch
    T, h, f, N, e = 256, 256, 4096, 8, 2
    prev = None
    for k in (1, 2, 4, 8):
        desc = lib.make_zdp_desc(T, h, f, torch.bfloat16, k, N, 0)
        fs = f // k
        slice_params = (2 * h * fs + fs) * e
        fw = lib.osdp_zdp_ffn_split_mlp_workspace_bytes(desc, lib.OSDP_FWD)
        bw = lib.osdp_zdp_ffn_split_mlp_workspace_bytes(desc, lib.OSDP_BWD)
        acc = 0 if k == 1 else T * h * 4
        assert 0 <= fw - (2 * slice_params + h * e + T * fs * e + acc) <= 8 * 256
        scratch = (T // 32) * fs * 4 + 32 * h * 4                      # db1 band partials of one slice + db2 partials
        assert 0 <= bw - (2 * slice_params + 2 * slice_params * 2 + h * 4 + 2 * T * fs * e + acc + scratch) <= 16 * 256
        c = lib.osdp_zdp_ffn_split_mlp_op_cost(desc, lib.OSDP_FWD)
        dev = lib.osdp_device(N, 0.0, 0.0, 1 << 62)
        p, tr, _ = lib.osdp_cost_eval(c, lib.OSDP_ZDP, k, 1, dev)
        model = p + tr - c.act_bytes                                    # model-state shard + workspace, as the cost model sees it
        shard = -(-c.model_bytes // N)
        # the cost model predicts the workspace from above: never less (the planner's M_limit check relies on it), and
        # no more than one group of N x 8 columns of slice tensors + padding (+ the accumulator it also charges at k = 1)
        slack = N * 8 * (2 * (2 * h + 1) * e + T * e) + 24 * 256 + (T * h * 4 if k == 1 else 0)
        assert 0 <= (model - shard) - fw <= slack, (k, model - shard, fw)
        if prev is not None:
            assert fw < prev                                             # size / slice_granularity
        prev = fw
    with pytest.raises(lib.OsdpError):
        lib.osdp_zdp_shard_elems(lib.make_zdp_desc(T, 100, f, torch.bfloat16, 1, 8, 0))       # h % (N unit) != 0
    with pytest.raises(lib.OsdpError):
        lib.osdp_zdp_shard_elems(lib.make_zdp_desc(T, h, f, torch.bfloat16, 1, 8, 8))         # rank out of range
    with pytest.raises(lib.OsdpError):
        lib.osdp_zdp_shard_elems(lib.make_zdp_desc(T, h, f, torch.bfloat16, f // 64 + 1, 8, 0))   # k > groups


# ------------------------------------------------------------------ world_size 2 on CPU (gloo): the library's schedule
# and layout executed in fp64 with real collectives equals the unsplit MLP
WORKER = r'''
import sys, json
sys.path.insert(0, %r)
import numpy as np, torch, torch.distributed as dist
from paper_2305_09940_b200 import binding as lib, dist as D, inputs as I
from oracle import mlp_oracle as M
world, rank, _ = D.init("gloo")
T, h, f, k = 12 + 4 * rank, 16, 96, 3                 # ranks hold different numbers of tokens
dt = torch.float32
full = I.mlp_inputs(4, h, f, dt, seed=0)              # the same weights on every rank (seed 0)
mine = I.mlp_inputs(T, h, f, dt, seed=100 + rank)     # this rank's tokens
W1, b1, W2, b2 = (t.double() for t in (full.W1, full.b1, full.W2, full.b2))
X, dY = mine.X.double(), mine.dY.double()
desc = lib.make_zdp_desc(T, h, f, dt, k, world, rank)
shard = lib.zdp_shard(desc, W1, b1, W2, b2)
G, C, R = lib.OSDP_ZDP_GATHER, lib.OSDP_ZDP_COMPUTE, lib.OSDP_ZDP_REDUCE_SCATTER
recv_bytes = 0
def gather(off, n):
    global recv_bytes
    out = torch.empty(n * world, dtype=torch.float64)
    dist.all_gather_into_tensor(out, shard[off:off + n].contiguous())
    recv_bytes += n * (world - 1) * 4
    return out
def reduce_scatter(fullbuf):
    global recv_bytes
    t = fullbuf.contiguous().reshape(-1).clone()
    dist.all_reduce(t)                                # gloo has no reduce_scatter: all-reduce, keep this rank's chunk
    n = t.numel() // world
    recv_bytes += n * (world - 1) * 4
    return t[rank * n:(rank + 1) * n]
def run(pass_):
    bufs, out = {}, {}
    Y = torch.zeros(T, h, dtype=torch.float64); dX = torch.zeros(T, h, dtype=torch.float64)
    gshard = torch.zeros_like(shard); stage = {}
    b2g = None
    for op, s, buf, on_comm, nbytes in lib.osdp_zdp_schedule(desc, pass_):
        sl = lib.osdp_zdp_slice_layout(desc, s)
        fs = sl.hi - sl.lo
        if op == G and s == k:
            b2g = gather(sl.b1_off, sl.b1_elems)
        elif op == G:
            bufs[buf] = (gather(sl.w1_off, sl.w1_elems).reshape(h, fs), gather(sl.b1_off, sl.b1_elems),
                         gather(sl.w2_off, sl.w2_elems).reshape(fs, h))
            assert nbytes == (sl.w1_elems + sl.b1_elems + sl.w2_elems) * 4
        elif op == C:
            W1s, b1s, W2s = bufs[buf]
            Z = X @ W1s + b1s[None, :]
            H = torch.from_numpy(M.gelu(Z.numpy()))
            if pass_ == lib.OSDP_FWD:
                Y += H @ W2s
            else:
                dZ = (dY @ W2s.T) * torch.from_numpy(M.gelu_prime(Z.numpy()))
                stage[buf] = (X.T @ dZ, dZ.sum(0), H.T @ dY)
                dX += dZ @ W1s.T
                if s == 0:
                    stage["db2"] = dY.sum(0)
        else:
            if s == k:
                gshard[sl.b1_off:sl.b1_off + sl.b1_elems] = reduce_scatter(stage["db2"])
            else:
                g1, gb, g2 = stage[buf]
                gshard[sl.w1_off:sl.w1_off + sl.w1_elems] = reduce_scatter(g1)
                gshard[sl.b1_off:sl.b1_off + sl.b1_elems] = reduce_scatter(gb)
                gshard[sl.w2_off:sl.w2_off + sl.w2_elems] = reduce_scatter(g2)
    if pass_ == lib.OSDP_FWD:
        return Y + b2g[None, :]
    return dX, gshard
Y = run(lib.OSDP_FWD)
dX, gshard = run(lib.OSDP_BWD)
ref = M.mlp_forward_backward(X.numpy(), W1.numpy(), b1.numpy(), W2.numpy(), b2.numpy(), dY.numpy())
errY = float(np.max(np.abs(Y.numpy() - ref["Y"]))); errdX = float(np.max(np.abs(dX.numpy() - ref["dX"])))
# gradients: gather every rank's shard and every rank's reference gradient sum
shards = [torch.empty_like(gshard) for _ in range(world)]
dist.all_gather(shards, gshard)
tot = {}
for name in ("dW1", "db1", "dW2", "db2"):
    t = torch.from_numpy(ref[name]).clone(); dist.all_reduce(t); tot[name] = t
gW1, gb1, gW2, gb2 = lib.zdp_unshard(desc, shards)
errg = max(float((a - tot[n]).abs().max()) for a, n in ((gW1, "dW1"), (gb1, "db1"), (gW2, "dW2"), (gb2, "db2")))
S = (2 * h * f + f + h) * 4
print(json.dumps({"rank": rank, "errY": errY, "errdX": errdX, "errg": errg, "recv_bytes": recv_bytes,
                  "expect_bytes": (3 * S - h * 4) * (world - 1) // world}))
D.finalize()
''' % ROOT


def test_two_rank_gloo_run_of_the_library_schedule(tmp_path):
    import json
    import socket
    script = tmp_path / "zdp_worker.py"
    script.write_text(WORKER)
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    procs = []
    for r in range(2):
        env = dict(os.environ, WORLD_SIZE="2", RANK=str(r), LOCAL_RANK=str(r), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), CUDA_VISIBLE_DEVICES="")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    for p in procs:
        o, e = p.communicate(timeout=300)
        assert p.returncode == 0, e[-3000:]
        res = json.loads(o.strip().splitlines()[-1])
        assert res["errY"] <= 1e-12 and res["errdX"] <= 1e-12 and res["errg"] <= 1e-11, res
        assert res["recv_bytes"] == res["expect_bytes"], res            # 3 collectives of S (N-1)/N (b2: two)
