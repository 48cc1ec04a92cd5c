"""Host-side logic of bench.py that needs no GPU: the cost-model fit, the oracle sample size, the reference arm's line."""
import json
import math
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_fit_gamma_delta_recovers_a_linear_cost_model():
    """T(k) = gamma + (k - 1) delta (reading P2): exact data gives the parameters back, residual 0."""
    import bench
    gamma, delta = 22.0, 1.25      # ms
    table = [{"k": k, "ms_per_step": gamma + (k - 1) * delta} for k in (1, 2, 4, 8, 16, 32)]
    fit = bench.fit_gamma_delta(table)
    assert math.isclose(fit["gamma_s"], gamma * 1e-3, rel_tol=1e-12)
    assert math.isclose(fit["delta_s"], delta * 1e-3, rel_tol=1e-12)
    assert fit["max_rel_residual"] < 1e-12
    # a convex curve: the residual reports the misfit instead of hiding it
    table[-1]["ms_per_step"] *= 1.5
    assert bench.fit_gamma_delta(table)["max_rel_residual"] > 0.05
    assert bench.fit_gamma_delta([{"k": 4, "ms_per_step": 1.0}]) is None          # no k = 1 point: nothing to fit


def test_oracle_sample_is_bounded_and_a_power_of_two():
    import bench
    for h, f in ((256, 1024), (1024, 4096), (8192, 32768), (12288, 49152)):
        t = bench.oracle_sample_tokens(h, f)
        assert 8 <= t <= 4096 and t & (t - 1) == 0
        assert 14.0 * t * h * f <= 2.5e12 or t == 8


def test_executed_flops_counts_the_slice_recompute():
    import bench
    T, h, f = 8192, 8192, 32768
    assert bench.executed_flops(T, h, f) == 14.0 * T * h * f           # 4 fwd + 8 bwd + 2 recompute of Z


def test_reference_arm_prints_one_json_line_on_cpu():
    """`bench.py --impl reference` times the oracle on host cores and needs no GPU (C1 is small enough for a test)."""
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--config", "C1", "--k", "4",
                        "--steps", "1", "--warmup", "0"], capture_output=True, text=True, timeout=300, cwd=ROOT)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [ln for ln in r.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["cpu_baseline"]["kind"] == "oracle" and d["value"] > 0
    assert d["e2e"]["h2d_bytes_per_step"] == 0 and d["gpu_launches"] == 0 and d["vs_baseline"] is None


def test_gemms_per_traced_launch_cover_the_slice_kernel_steps():
    """The trace step ids of the one-kernel-per-slice path carry 2 (forward) and 5 (backward) GEMMs of 2 T_s h f flops each;
    the per-GEMM steps A1-A7 one.  bench.py divides by these for the per-launch TFLOP/s and the roofline fraction."""
    import bench
    assert bench.GEMMS_PER_LAUNCH[21] == 2 and bench.GEMMS_PER_LAUNCH[22] == 5
    assert all(bench.GEMMS_PER_LAUNCH[s] == 1 for s in range(1, 8))
    assert 8 not in bench.GEMMS_PER_LAUNCH and 10 not in bench.GEMMS_PER_LAUNCH      # column sums, accumulator -> output
    # a whole step = k x (2 + 5) GEMMs = 14 T h f
    T, h, f, k = 8192, 1024, 4096, 8
    assert k * (bench.GEMMS_PER_LAUNCH[21] + bench.GEMMS_PER_LAUNCH[22]) * 2.0 * (T // k) * h * f == bench.executed_flops(T, h, f)
