"""N > 1 host logic on CPU: world_size 2, gloo backend (no GPU, no collective on the data path)."""
import os
import socket
import subprocess
import sys
import textwrap

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = textwrap.dedent("""
    import sys, json
    sys.path.insert(0, %r)
    import torch
    from paper_2305_09940_b200 import dist as D, inputs as I
    world, rank, local = D.init("gloo")
    assert world == 2
    # each rank draws its own token batch; weights differ per seed too (independent replicas)
    x = I.normal_tensor(D.rank_seed(0, rank), I.STREAM_X, (8, 8), 1.0, torch.float32)
    D.barrier()
    ms_local = 10.0 if rank == 0 else 12.5          # rank 1 is the slow one
    value, ms = D.whole_job_throughput(ms_local, 1e9)
    print(json.dumps({"rank": rank, "value": value, "ms": ms, "x0": float(x[0, 0])}))
    D.finalize()
""") % ROOT


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_two_rank_replica_aggregation(tmp_path):
    import json
    script = tmp_path / "worker.py"
    script.write_text(WORKER)
    port = _free_port()
    procs = []
    for r in range(2):
        env = dict(os.environ, WORLD_SIZE="2", RANK=str(r), LOCAL_RANK=str(r), MASTER_ADDR="127.0.0.1",
                   MASTER_PORT=str(port), CUDA_VISIBLE_DEVICES="")
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    outs = []
    for p in procs:
        o, e = p.communicate(timeout=240)
        assert p.returncode == 0, e[-2000:]
        outs.append(json.loads(o.strip().splitlines()[-1]))
    for o in outs:
        assert o["ms"] == 12.5                              # max over ranks
        assert abs(o["value"] - 2 * 1e9 / 12.5e-3) < 1e-3    # whole-job units/s
    assert outs[0]["x0"] != outs[1]["x0"]                    # different token batches per rank


def test_single_process_defaults():
    from paper_2305_09940_b200 import dist as D
    assert D.env_world() == (1, 0, 0) or "WORLD_SIZE" in os.environ
    assert D.max_over_ranks(3.5) == 3.5
    v, ms = D.whole_job_throughput(2.0, 10.0)
    assert ms == 2.0 and v == 10.0 / 2e-3
    assert D.rank_seed(5, 3) == 8
