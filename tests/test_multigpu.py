"""The multi-GPU paths on real processes and GPUs (NEXT-4): launched with torch.distributed.run,
one rank per GPU over NCCL.  Skipped unless two CUDA devices are visible (the build box and the 1-GPU test box have
fewer); the exchange arithmetic itself is covered on CPU by tests/test_multirank_host.py (gloo, world size 2) and the
kernels behind it by test_view_parallel_two_emulated_ranks / test_blocked_blocks_dealt_over_two_ranks on one GPU."""
import os
import socket
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
pytestmark = pytest.mark.gpu


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    return port


def test_view_parallel_and_block_replicas_on_two_gpus_over_nccl():
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two CUDA devices")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
           "--master-addr", "127.0.0.1", "--master-port", str(_free_port()),
           os.path.join(ROOT, "tests", "_multigpu_worker.py")]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=900, cwd=ROOT)
    assert r.returncode == 0, r.stdout[-2000:] + r.stderr[-4000:]
    assert "rank 0 ok" in r.stdout and "rank 1 ok" in r.stdout
