"""bench.py's multi-rank flow (torchrun, barrier, max over ranks, rank 0 prints ONE line) on a single GPU: two ranks
share the GPU, the process group is gloo (ACM_DIST_BACKEND) because NCCL refuses two ranks on one device.  The replicas
are independent -- no kernel waits on another rank -- so sharing the GPU is safe; the numbers are not a measurement."""
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


def _torchrun(extra, nproc=2):
    env = dict(os.environ, ACM_DIST_BACKEND="gloo")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={nproc}", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port()), os.path.join(ROOT, "bench.py"), "--gpus", str(nproc), "--steps", "4", "--warmup", "3",
           "--no-cpu-baseline"] + extra
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=900, cwd=ROOT, env=env)
    assert out.returncode == 0, out.stderr[-3000:]
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1, out.stdout[-2000:]
    return json.loads(lines[0])


def test_two_replica_ranks_print_one_line():
    d = _torchrun(["--config", "1"])
    assert d["n_gpus"] == 2 and d["scaling"] == "weak" and d["steps"] == 4 and d["warmup"] == 20
    assert d["config"]["parallelism"] == "replicas only"
    assert d["value"] > 0 and d["value_min"] <= d["value"] <= d["value_max"]
    assert d["gpu_launches"] == 8 and d["roofline"]["bound"] == "hbm" and "cpu_baseline" not in d and "also" not in d
    assert d["e2e"]["value"] > 0 and d["config"]["finite"]


def test_two_slab_ranks_over_gloo_fail_loudly():
    """--decompose moves halo planes with torch.distributed P2P on CUDA tensors, which gloo does not offer: the run gets
    through the slab set-up, initialisation and plan (the code both backends share) and must then fail loudly at the
    first exchange -- no hang, no JSON line (the NCCL transport needs two GPUs: test_gpu_slab_ipc.py::test_two_gpus_over_nccl)."""
    env = dict(os.environ, ACM_DIST_BACKEND="gloo")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2", "--master-addr", "127.0.0.1",
           "--master-port", str(_free_port()), os.path.join(ROOT, "bench.py"), "--gpus", "2", "--steps", "2", "--warmup", "1",
           "--no-cpu-baseline", "--config", "1", "--decompose"]
    out = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT, env=env)
    lines = [l for l in out.stdout.splitlines() if l.startswith("{")]
    assert out.returncode != 0 and not lines
    assert "refresh_halos" in out.stderr and "batch_isend_irecv" in out.stderr      # it got as far as the first exchange
