"""-m gpu: the N > 1 flow of bench.py, launched the way the driver launches it (torch.distributed.run, one process
per rank, rendezvous on 127.0.0.1).  The GPU box of the tests has ONE GPU, so both ranks share it and reduce their
timings over gloo (`--dist-backend gloo`): what is checked is the flow -- shards, barriers, max over ranks, ONE JSON
line from rank 0 -- not a throughput.  The ranks' kernels never wait on one another (streams shard with no
collective)."""
import json
import os
import socket
import subprocess
import sys

import pytest

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


@pytest.mark.parametrize("workload", ["C1_u32", "C3_draw"])
def test_bench_two_ranks_print_one_line_with_the_whole_job_value(workload):
    torch = pytest.importorskip("torch")
    if not torch.cuda.is_available():
        pytest.fail("-m gpu tests need a CUDA device")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port()), os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "3", "--warmup", "3",
           "--workload", workload, "--dist-backend", "gloo", "--e2e-steps", "1"]
    r = subprocess.run(cmd, cwd=ROOT, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, r.stdout[-2000:]  # rank 0 alone prints
    d = json.loads(lines[0])
    assert d["n_gpus"] == 2 and d["scaling"] == "weak" and d["value"] > 0 and d["steps"] == 3
    assert d["config"]["workload"] == workload and d["config"]["parallelism"] == "streams x2"
    assert d["e2e"]["value"] > 0 and d["gpu_launches"] >= 3
    assert "cpu_baseline" not in d and "configs" not in d  # rank 0 at N = 1 only
    assert len(lines[0]) < 4096
