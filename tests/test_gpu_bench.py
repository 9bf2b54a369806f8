"""-m gpu: bench.py's B200 arm end to end on the tiny workload -- the JSON contract, and the N > 1 code path
(baseline sharding, grid all-reduce inside the timed step, max-over-ranks timing) with two ranks that share the one
device of the box and talk over gloo (NCCL wants one device per rank; the kernels of the two ranks never wait on
one another)."""
import json
import os
import socket
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
KEYS = ("metric", "value", "unit", "n_gpus", "steps", "warmup", "ms_per_step", "higher_is_better", "scaling", "vs_baseline",
        "dtype", "data", "config", "clocks", "e2e", "gpu_launches", "roofline")


def _line(out):
    assert out.returncode == 0, out.stderr[-3000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, out.stdout[-2000:]
    return json.loads(lines[0])


def test_one_rank_line_has_the_contract_keys():
    out = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--workload", "tiny", "--steps", "3", "--warmup", "3"],
                         capture_output=True, text=True, timeout=900, cwd=ROOT)
    d = _line(out)
    for k in KEYS + ("cpu_baseline",):
        assert k in d, k
    assert d["n_gpus"] == 1 and d["scaling"] == "weak" and d["gpu_launches"] == 3 * 5 and d["value"] > 0
    r = d["roofline"]
    assert r["bound"] == "alu" and 0 < r["frac"] < 1.2 and len(r["kernels"]) == 5
    assert {k["stage"] for k in r["kernels"]} == {"gridder", "degridder", "subgrid_fft", "adder", "splitter_ifft"}
    assert r["measured_mix_peak"]["tflops"] > 10
    assert d["e2e"]["h2d_bytes_per_step"] > 0 and d["e2e"]["d2h_bytes_per_step"] > 0
    assert d["detail"]["collective"] is None


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_two_ranks_shard_one_workload_and_reduce_the_grid():
    env = dict(os.environ, IDG_BENCH_DIST_BACKEND="gloo", IDG_BENCH_SINGLE_DEVICE="1")
    out = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                          "--master-addr", "127.0.0.1", "--master-port", str(_free_port()), os.path.join(ROOT, "bench.py"),
                          "--gpus", "2", "--workload", "tiny", "--steps", "3", "--warmup", "3"],
                         capture_output=True, text=True, timeout=900, cwd=ROOT, env=env)
    d = _line(out)
    for k in KEYS:
        assert k in d, k
    assert d["n_gpus"] == 2 and d["scaling"] == "strong" and "cpu_baseline" not in d
    assert d["detail"]["n_vis_total"] == 28 * 32 * 4                      # ONE workload: all of configs[0], once
    assert d["detail"]["n_vis_rank0"] == 14 * 32 * 4                      # rank 0 owns half the baselines
    c = d["detail"]["collective"]
    assert c["bytes"] == 8 * 4 * 256 * 256 and c["ms"] > 0
    assert d["detail"]["stage_ms"]["allreduce_grid"] > 0
    assert "2 ranks" in d["config"]["parallelism"]


def test_mma_rate_probe_reports_the_measured_floor():
    """idg_bench_mma_rate (csrc/mmabench.cu): the M128 x N x K16 MMA with A in tensor memory runs at M N / 256 cycles
    from N = 64 up and at ~9 cycles for N = 16, whatever the number of CTAs per SM (profiles/r02_experiments.md
    section 7); loose bounds, the probe is a measurement aid."""
    from paper_1909_07226_b200 import binding as idg
    c16 = idg.idg_bench_mma_rate(16, 1)
    c16x4 = idg.idg_bench_mma_rate(16, 4)
    c256 = idg.idg_bench_mma_rate(256, 1)
    assert 4.0 < c16 < 16.0 and 4.0 < c16x4 < 16.0
    assert 100.0 < c256 < 160.0
    with pytest.raises(idg.IdgError):
        idg.idg_bench_mma_rate(32, 1)
